/*
 * ts_step.cu -- stepping entry points of the C ABI (include/ts.h): ts_build_neighbors,
 * ts_compute_forces, ts_md_step, ts_fire_step, ts_poll, ts_converged_mask, ts_swap_systems,
 * ts_get_neighbors and the small accessors.  Host code only: it sequences kernels on the
 * caller's stream; the skin check and the rebuild decision stay on the device.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "ts_internal.cuh"

static ts_status check_launch(ts_state *st)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        ts_set_error(st, "kernel launch failed: %s", cudaGetErrorString(e));
        return TS_ERR_CUDA;
    }
    return TS_OK;
}

#define NEED_STATE(st)                                  \
    do {                                                \
        if (!(st)) return TS_ERR_INVALID_ARG;           \
        if ((st)->seen_flags) return TS_ERR_STICKY;     \
    } while (0)

void ts_whole_batch_mode(ts_state *st)
{
    if (st->list_mixed) { st->list_built = false; st->forces_current = false; st->list_mixed = false; }
    st->d.mixed = 0;
}

/* list for the current positions: forced build the first time, skin-checked afterwards */
static void ensure_list(ts_state *st, cudaStream_t q)
{
    if (!st->list_built) {
        launch_build(st, true, q);
    } else {
        launch_import(st, q);
        launch_build(st, false, q);
    }
}

extern "C" ts_status ts_build_neighbors(ts_state *st, void *stream)
{
    NEED_STATE(st);
    launch_build(st, true, (cudaStream_t)stream);
    return check_launch(st);
}

extern "C" ts_status ts_compute_forces(ts_state *st, uint32_t want, void *stream)
{
    NEED_STATE(st);
    cudaStream_t q = (cudaStream_t)stream;
    st->last_engine = 0;
    ts_whole_batch_mode(st);
    ensure_list(st, q);
    launch_pair(st, want & 3u, false, q);
    if (want & TS_WANT_ENERGY) launch_kinetic(st, q);
    st->forces_current = true;
    return check_launch(st);
}

extern "C" ts_status ts_md_step(ts_state *st, const ts_md_params *p, int32_t n_steps, uint32_t want, void *stream)
{
    NEED_STATE(st);
    if (!p || n_steps < 0 || (p->integrator != TS_NVE && p->integrator != TS_BAOAB) || !(p->dt > 0.0))
        return TS_ERR_INVALID_ARG;
    if (p->integrator == TS_BAOAB && (!(p->friction >= 0.0) || !(p->temperature >= 0.0))) return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    MdConst c;
    c.integrator = p->integrator;
    c.dt = p->dt; c.hdt = 0.5 * p->dt;
    c.c1 = exp(-p->friction * p->dt);
    c.c2 = sqrt(1.0 - c.c1 * c.c1);
    c.kT = st->d.kB * p->temperature;
    c.key0 = (unsigned)(p->seed & 0xffffffffull); c.key1 = (unsigned)(p->seed >> 32);
    want = (want & 3u) | TS_WANT_ENERGY;
    /* Engine dispatch.  The resident engine steps every system it can hold, size class by size class; the general engine
     * steps the others NEXT to it on a stream of its own (mixed dispatch of a ragged batch), or the whole batch when the
     * resident engine is switched off or does not apply at all. */
    const int n_general = st->engine == 1 ? resident_general_count(st) : st->d.S;
    const bool use_resident = n_general < st->d.S, mixed = use_resident && n_general > 0;
    if (use_resident) {
        ts_status rc = resident_md(st, c, n_steps, want, q);
        if (rc != TS_OK) return rc;
        if (!mixed) {
            st->steps_done += n_steps;
            st->forces_current = true;
            st->list_built = false;          /* the general engine's list no longer matches the positions */
            st->list_mixed = false;
            return TS_OK;
        }
    } else {
        st->last_engine = 0;
    }
    cudaStream_t g = q;
    if (mixed) {
        if (!st->list_mixed) { st->list_built = false; st->forces_current = false; st->list_mixed = true; }
        st->d.mixed = 1;
        g = resident_fork_general(st, q);
    } else {
        ts_whole_batch_mode(st);
    }
    if (!st->forces_current || !st->list_built || n_steps == 0) {   /* no list of its own yet (e.g. the resident engine ran before) */
        ensure_list(st, g);
        launch_pair(st, n_steps == 0 ? want : 0u, false, g);
        if (n_steps == 0) launch_kinetic(st, g);
        st->forces_current = true;
    }
    for (int n = 0; n < n_steps; ++n) {
        bool last = n == n_steps - 1;
        launch_md_pre(st, c, g);
        launch_build(st, false, g);
        launch_pair(st, last ? want : 0u, false, g);
        launch_md_post(st, c, last, g);
    }
    if (mixed) {
        resident_join_general(st, q);
        st->d.mixed = 0;
    }
    st->steps_done += n_steps;
    return check_launch(st);
}

extern "C" ts_status ts_fire_step(ts_state *st, const ts_fire_params *p, int32_t n_steps, void *stream)
{
    NEED_STATE(st);
    if (!p || n_steps < 0 || !(p->dt_start > 0.0) || !(p->dt_max > 0.0) || !(p->f_max > 0.0)) return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    if (st->engine == 1 && resident_supported(st)) {
        ts_status rc = resident_fire(st, *p, n_steps, q);
        if (rc != TS_ERR_UNSUPPORTED) {
            if (rc == TS_OK) { st->steps_done += n_steps; st->forces_current = true; st->list_built = false; st->list_mixed = false; }
            return rc;
        }
    }
    st->last_engine = 0;
    ts_whole_batch_mode(st);
    launch_fire_init(st, *p, q);
    ensure_list(st, q);
    launch_pair(st, TS_WANT_ENERGY, true, q);
    launch_fire_check0(st, *p, q);
    for (int n = 0; n < n_steps; ++n) {
        launch_fire_pre(st, *p, q);
        launch_build(st, false, q);
        launch_pair(st, TS_WANT_ENERGY, true, q);
        launch_fire_post(st, *p, q);
    }
    st->forces_current = true;
    st->steps_done += n_steps;
    return check_launch(st);
}

extern "C" ts_status ts_poll(ts_state *st, ts_report *out, void *stream)
{
    if (!st || !out) return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    launch_fire_count(st, q);
    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    DevStatus hs;
    int cnt[2];
    TS_CUDA_OK(st, cudaMemcpy(&hs, st->d.status, sizeof hs, cudaMemcpyDeviceToHost));
    TS_CUDA_OK(st, cudaMemcpy(cnt, st->d.scratch + 2 * (size_t)st->d.S + 2, sizeof cnt, cudaMemcpyDeviceToHost));
    memset(out, 0, sizeof *out);
    out->flags = hs.flags;
    out->n_rebuilds = (int32_t)hs.n_rebuilds;
    const unsigned long long rnnz = hs.res_nnz[st->res_nnz_slot & 1];
    out->nnz = st->last_engine == 1 ? (int64_t)rnnz : st->last_engine == 2 ? (int64_t)(rnnz + hs.nnz) : (int64_t)hs.nnz;
    out->resident_rebuilds = (int64_t)hs.res_rebuilds;
    out->engine = st->last_engine;
    out->nnz_capacity = st->d.nbr_cap;
    out->steps_done = st->steps_done;
    out->n_converged = cnt[0];
    out->n_failed = cnt[1];
    out->max_neighbors = (int32_t)hs.max_nbr;
    out->list_valid = (int32_t)(hs.list_valid && st->list_built);
    st->seen_flags = hs.flags;
    if (hs.flags) ts_set_error(st, "device status flags 0x%x (1 overflow, 2 shift range, 4 non-finite, 8 bad cell)", hs.flags);
    return TS_OK;
}

extern "C" ts_status ts_clear_error(ts_state *st, void *stream)
{
    if (!st) return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    TS_CUDA_OK(st, cudaMemsetAsync(&st->d.status->flags, 0, sizeof(unsigned), q));
    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    st->seen_flags = 0;
    st->list_built = false;
    st->forces_current = false;
    st->err[0] = 0;
    return TS_OK;
}

extern "C" ts_status ts_converged_mask(ts_state *st, uint8_t *mask, int32_t *status, int32_t *fire_steps, void *stream)
{
    if (!st) return TS_ERR_INVALID_ARG;
    int S = st->d.S;
    TS_CUDA_OK(st, cudaStreamSynchronize((cudaStream_t)stream));
    std::vector<int> hs((size_t)S);
    TS_CUDA_OK(st, cudaMemcpy(hs.data(), st->d.f_status, sizeof(int) * (size_t)S, cudaMemcpyDeviceToHost));
    for (int s = 0; s < S; ++s) {
        if (mask) mask[s] = hs[(size_t)s] == TS_FIRE_CONVERGED ? 1 : 0;
        if (status) status[s] = hs[(size_t)s];
    }
    if (fire_steps) TS_CUDA_OK(st, cudaMemcpy(fire_steps, st->d.f_nsteps, sizeof(int) * (size_t)S, cudaMemcpyDeviceToHost));
    return TS_OK;
}

extern "C" ts_status ts_fire_status_async(ts_state *st, int32_t *status, int32_t *fire_steps, void *stream)
{
    if (!st) return TS_ERR_INVALID_ARG;
    const size_t bytes = sizeof(int) * (size_t)st->d.S;
    cudaStream_t q = (cudaStream_t)stream;
    if (status) TS_CUDA_OK(st, cudaMemcpyAsync(status, st->d.f_status, bytes, cudaMemcpyDeviceToHost, q));
    if (fire_steps) TS_CUDA_OK(st, cudaMemcpyAsync(fire_steps, st->d.f_nsteps, bytes, cudaMemcpyDeviceToHost, q));
    return TS_OK;
}

extern "C" ts_status ts_swap_systems(ts_state *st, const int32_t *slots, int32_t n, const ts_state_desc *fresh, void *stream)
{
    NEED_STATE(st);
    if (n == 0) return TS_OK;
    int S = st->d.S;
    if (!slots || !fresh || n < 0 || n > S || !fresh->pos || fresh->dtype != st->d.dtype || fresh->n_systems != n)
        return TS_ERR_INVALID_ARG;
    cudaStream_t q = (cudaStream_t)stream;
    std::vector<int> up(2 * (size_t)n);
    std::vector<char> seen((size_t)S, 0);
    long long off = 0;
    for (int k = 0; k < n; ++k) {
        int s = slots[k];
        if (s < 0 || s >= S || seen[(size_t)s]) return TS_ERR_INVALID_ARG;
        seen[(size_t)s] = 1;
        up[(size_t)k] = s;
        up[(size_t)n + k] = (int)off;
        off += st->h_sysoff[s + 1] - st->h_sysoff[s];
    }
    if (off != fresh->n_atoms) return TS_ERR_INVALID_ARG;
    TS_CUDA_OK(st, cudaMemcpyAsync(st->d.scratch, up.data(), sizeof(int) * up.size(), cudaMemcpyHostToDevice, q));
    launch_swap(st, n, fresh, q);
    std::vector<char> hcell;
    if (fresh->cell) {
        launch_geometry(st, 0, n, st->d.scratch, q);
        hcell.resize((size_t)n * 9 * (st->d.dtype == TS_F32 ? 4 : 8));
        TS_CUDA_OK(st, cudaMemcpyAsync(hcell.data(), fresh->cell, hcell.size(), cudaMemcpyDeviceToHost, q));
    }
    st->list_built = false;
    st->forces_current = false;
    /* the upload buffer must outlive the copy */
    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    if (fresh->cell) resident_after_swap(st, slots, n, hcell.data());   /* keeps the launch plan when the new cells fit it */
    return check_launch(st);
}

extern "C" ts_status ts_get_neighbors(ts_state *st, int64_t *off, int32_t *j, int8_t *shift, int64_t cap, void *stream)
{
    if (!st || !off) return TS_ERR_INVALID_ARG;
    if (!st->list_built) return TS_ERR_STALE_NBR;
    const DevState &d = st->d;
    long long N = d.N;
    int S = d.S;
    TS_CUDA_OK(st, cudaStreamSynchronize((cudaStream_t)stream));
    std::vector<int> cnt((size_t)N), wrap((size_t)N);
    std::vector<long long> noff((size_t)N), len((size_t)S), base((size_t)S + 1);
    TS_CUDA_OK(st, cudaMemcpy(cnt.data(), d.nbr_cnt, 4 * (size_t)N, cudaMemcpyDeviceToHost));
    TS_CUDA_OK(st, cudaMemcpy(wrap.data(), d.atom_wrap, 4 * (size_t)N, cudaMemcpyDeviceToHost));
    TS_CUDA_OK(st, cudaMemcpy(noff.data(), d.nbr_off, 8 * (size_t)N, cudaMemcpyDeviceToHost));
    TS_CUDA_OK(st, cudaMemcpy(len.data(), d.nbr_len, 8 * (size_t)S, cudaMemcpyDeviceToHost));
    TS_CUDA_OK(st, cudaMemcpy(base.data(), d.nbr_base, 8 * (size_t)(S + 1), cudaMemcpyDeviceToHost));
    for (int s = 0; s < S; ++s)
        if (len[(size_t)s] < 0) return TS_ERR_NBR_OVERFLOW;
    off[0] = 0;
    for (long long i = 0; i < N; ++i) off[i + 1] = off[i] + cnt[(size_t)i];
    if (!j && !shift) return TS_OK;
    if (off[N] > cap) return TS_ERR_WORKSPACE_TOO_SMALL;
    std::vector<unsigned> seg;
    for (int s = 0; s < S; ++s) {
        long long L = len[(size_t)s];
        if (L == 0) continue;
        seg.resize((size_t)L);
        TS_CUDA_OK(st, cudaMemcpy(seg.data(), d.nbr + base[(size_t)s], 4 * (size_t)L, cudaMemcpyDeviceToHost));
        int a0 = st->h_sysoff[s], a1 = st->h_sysoff[s + 1];
        for (int i = a0; i < a1; ++i) {
            const unsigned *row = seg.data() + (noff[(size_t)i] - base[(size_t)s]);
            int wi0 = (signed char)(wrap[(size_t)i] & 0xff), wi1 = (signed char)((wrap[(size_t)i] >> 8) & 0xff),
                wi2 = (signed char)((wrap[(size_t)i] >> 16) & 0xff);
            for (int k = 0; k < cnt[(size_t)i]; ++k) {
                unsigned e = row[k];
                int lj = (int)(e & TS_J_MASK);
                int gj = a0 + lj;
                int s0 = (int)((e >> 17) & 31u) - 16, s1 = (int)((e >> 22) & 31u) - 16, s2 = (int)(e >> 27) - 16;
                int wj0 = (signed char)(wrap[(size_t)gj] & 0xff), wj1 = (signed char)((wrap[(size_t)gj] >> 8) & 0xff),
                    wj2 = (signed char)((wrap[(size_t)gj] >> 16) & 0xff);
                int64_t o = off[i] + k;
                if (j) j[o] = gj;
                if (shift) {
                    /* stored positions: x_j - x_i + S.h with S = S_stencil - wrap_j + wrap_i (R6) */
                    shift[3 * o + 0] = (int8_t)(s0 - wj0 + wi0);
                    shift[3 * o + 1] = (int8_t)(s1 - wj1 + wi1);
                    shift[3 * o + 2] = (int8_t)(s2 - wj2 + wi2);
                }
            }
        }
    }
    return TS_OK;
}

extern "C" ts_status ts_set_system_steps(ts_state *st, const uint64_t *steps, void *stream)
{
    if (!st || !steps) return TS_ERR_INVALID_ARG;
    TS_CUDA_OK(st, cudaStreamSynchronize((cudaStream_t)stream));
    TS_CUDA_OK(st, cudaMemcpy(st->d.sys_step, steps, 8 * (size_t)st->d.S, cudaMemcpyHostToDevice));
    return TS_OK;
}

extern "C" ts_status ts_get_system_steps(ts_state *st, uint64_t *steps, void *stream)
{
    if (!st || !steps) return TS_ERR_INVALID_ARG;
    TS_CUDA_OK(st, cudaStreamSynchronize((cudaStream_t)stream));
    TS_CUDA_OK(st, cudaMemcpy(steps, st->d.sys_step, 8 * (size_t)st->d.S, cudaMemcpyDeviceToHost));
    return TS_OK;
}

extern "C" ts_status ts_set_engine(ts_state *st, int32_t engine)
{
    if (!st || engine < 0 || engine > 1) return TS_ERR_INVALID_ARG;
    st->engine = engine;
    return TS_OK;
}

extern "C" ts_status ts_invalidate(ts_state *st)
{
    if (!st) return TS_ERR_INVALID_ARG;
    st->forces_current = false;
    st->res_saved_ok = false;             /* the resident engine's saved lists were built for other positions */
    return TS_OK;
}

extern "C" int64_t ts_launch_count(const ts_state *st) { return st ? st->launches : 0; }

extern "C" const char *ts_status_string(ts_status s)
{
    switch (s) {
    case TS_OK: return "ok";
    case TS_ERR_INVALID_ARG: return "invalid argument";
    case TS_ERR_CUDA: return "CUDA error";
    case TS_ERR_WORKSPACE_TOO_SMALL: return "workspace or output buffer too small";
    case TS_ERR_NBR_OVERFLOW: return "neighbour list capacity overflow";
    case TS_ERR_STALE_NBR: return "no neighbour list has been built";
    case TS_ERR_NONFINITE: return "non-finite force";
    case TS_ERR_UNSUPPORTED: return "unsupported";
    case TS_ERR_STICKY: return "device error flags are set (ts_poll, ts_clear_error)";
    default: return "unknown status";
    }
}

extern "C" const char *ts_last_error(const ts_state *st) { return st ? st->err : ""; }
