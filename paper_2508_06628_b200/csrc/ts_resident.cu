/* ts_resident.cu -- system-resident engine (placeholder until the kernel lands). */
#include "ts_internal.cuh"

bool resident_supported(const ts_state *st) { (void)st; return false; }
ts_status resident_md(ts_state *st, const MdConst &c, int n_steps, unsigned want, cudaStream_t q)
{
    (void)st; (void)c; (void)n_steps; (void)want; (void)q;
    return TS_ERR_UNSUPPORTED;
}
