/*
 * ts_graph.cu -- the batched graph builder as a service to an external energies / forces / stress
 * provider (SURVEY.md 8(f) NEXT-2; PAPER.md:56 "ModelInterface", :112 "graph construction"):
 *   ts_export_edges          the current Verlet list as a dense device-side edge list (i, j, S)
 *   ts_export_edges_static   the same with its scratch in a file-scope device array (no workspace region, no allocation)
 *   ts_md_step_external      one MD step split around a force evaluation the caller does
 *   ts_fire_step_external    the same for FIRE
 * The integrators are the general engine's kernels, unchanged; only the pair kernel is replaced by
 * whatever the caller runs on `stream` between the two halves.
 */
#include <math.h>
#include <string.h>

#include <mutex>

#include "ts_internal.cuh"

/* first edge of every system: exclusive scan of the pairs in use (one block; S is small next to N) */
__global__ void k_edge_base(DevState d, long long *edge_base /* [S+1] */, long long *n_edges)
{
    __shared__ long long part[256];
    const int S = d.S, per = (S + 255) / 256;
    const int s0 = threadIdx.x * per, s1 = min(S, s0 + per);
    long long sum = 0;
    for (int s = s0; s < s1; ++s) sum += d.nbr_len[s] > 0 ? d.nbr_len[s] : 0;
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long run = 0;
        for (int t = 0; t < 256; ++t) { const long long v = part[t]; part[t] = run; run += v; }
        edge_base[S] = run;
        *n_edges = run;
    }
    __syncthreads();
    long long run = part[threadIdx.x];
    for (int s = s0; s < s1; ++s) { edge_base[s] = run; run += d.nbr_len[s] > 0 ? d.nbr_len[s] : 0; }
}

/* eight lanes per atom copy its row: edge = first edge of the system + place of the row in the system's segment */
template <typename T>
__global__ void k_edge_fill(DevState d, const long long *edge_base, long long *ei, long long *ej, T *eS, long long cap)
{
    const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 3;
    const int l = threadIdx.x & 7;
    if (i >= d.N) return;
    const int s = d.sysidx[i];
    if (d.nbr_len[s] < 0) return;                      /* overflowed segment: flagged, exports nothing */
    const int a0 = d.sysoff[s];
    const long long row = d.nbr_off[i];
    const long long e0 = edge_base[s] + (row - d.nbr_base[s]);
    const int cnt = d.nbr_cnt[i];
    int wi0, wi1, wi2;
    ts_unpack_wrap(d.atom_wrap[i], wi0, wi1, wi2);
    for (int k = l; k < cnt; k += 8) {
        const long long e = e0 + k;
        if (e >= cap) break;
        const unsigned p = d.nbr[row + k];
        const int gj = a0 + (int)(p & TS_J_MASK);
        int s0, s1, s2, wj0, wj1, wj2;
        ts_unpack_shift(p, s0, s1, s2);
        ts_unpack_wrap(d.atom_wrap[gj], wj0, wj1, wj2);
        ei[e] = i; ej[e] = gj;
        /* stored positions: x_j - x_i + S.h with S = S_stencil - wrap_j + wrap_i (R6) */
        eS[3 * e + 0] = (T)(s0 - wj0 + wi0); eS[3 * e + 1] = (T)(s1 - wj1 + wi1); eS[3 * e + 2] = (T)(s2 - wj2 + wi2);
    }
}

static void ensure_list_graph(ts_state *st, cudaStream_t q)
{
    ts_whole_batch_mode(st);
    if (!st->list_built) launch_build(st, true, q);
    else { launch_import(st, q); launch_build(st, false, q); }
}

extern "C" ts_status ts_export_edges(ts_state *st, int64_t *edge_i, int64_t *edge_j, void *edge_shift, int64_t cap,
                                     int64_t *n_edges, void *stream)
{
    if (!st || !edge_i || !edge_j || !edge_shift || !n_edges || cap < 0) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    cudaStream_t q = (cudaStream_t)stream;
    ensure_list_graph(st, q);
    const DevState &d = st->d;
    long long *edge_base = (long long *)d.cell_count;      /* [S+1] int64 in a region the next build rewrites: (N+S+1) ints */
    if ((size_t)(d.S + 1) * 8 > (size_t)(st->N_cap + st->S_cap + 1) * 4) return TS_ERR_UNSUPPORTED;
    k_edge_base<<<1, 256, 0, q>>>(d, edge_base, (long long *)n_edges);
    const unsigned nb = (unsigned)((d.N * 8 + 255) / 256);
    if (d.dtype == TS_F32) k_edge_fill<float><<<nb, 256, 0, q>>>(d, edge_base, (long long *)edge_i, (long long *)edge_j, (float *)edge_shift, cap);
    else k_edge_fill<double><<<nb, 256, 0, q>>>(d, edge_base, (long long *)edge_i, (long long *)edge_j, (double *)edge_shift, cap);
    st->launches += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ts_set_error(st, "edge export failed: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    return TS_OK;
}

/* ------------------------------------------------------------------ edge export without workspace scratch
 * ts_export_edges keeps its [S + 1] exclusive scan of the edge counts in a workspace region the next list build
 * rewrites.  The variant below keeps it in a file-scope device array instead, for callers that must not allocate and
 * whose workspace region is in use: every GPU that loads the library holds the array (131,080 bytes) until exit.
 * In host code `g_edge_scan` is only a stand-in for the symbol, not a device address: the address the kernels get is
 * looked up with cudaGetSymbolAddress once per device, with that device current.                                     */
#define TS_STATIC_EDGE_MAX_SYSTEMS 16384
#define TS_STATIC_MAX_DEVICES 64
static __device__ __align__(256) long long g_edge_scan[TS_STATIC_EDGE_MAX_SYSTEMS + 1];

static std::mutex g_edge_scan_lock;
static long long *g_edge_scan_addr[TS_STATIC_MAX_DEVICES];      /* device address of g_edge_scan, by device ordinal */

/* address of the array on the CURRENT device (looked up on the first call for that device); nullptr + *err on failure */
static long long *edge_scan_address(cudaError_t *err)
{
    int dev = -1;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= TS_STATIC_MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> hold(g_edge_scan_lock);
    if (!g_edge_scan_addr[dev]) {
        long long *p = nullptr;
        *err = cudaGetSymbolAddress((void **)&p, g_edge_scan);
        if (*err != cudaSuccess) return nullptr;
        g_edge_scan_addr[dev] = p;
    }
    return g_edge_scan_addr[dev];
}

extern "C" ts_status ts_static_scratch_setup(int64_t *max_systems)
{
    if (max_systems) *max_systems = TS_STATIC_EDGE_MAX_SYSTEMS;
    cudaError_t e = cudaSuccess;
    return edge_scan_address(&e) ? TS_OK : TS_ERR_CUDA;
}

extern "C" ts_status ts_export_edges_static(ts_state *st, int64_t *edge_i, int64_t *edge_j, void *edge_shift, int64_t cap,
                                            int64_t *n_edges, void *stream)
{
    if (!st || !edge_i || !edge_j || !edge_shift || !n_edges || cap < 0) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    if (st->d.S > TS_STATIC_EDGE_MAX_SYSTEMS) {
        ts_set_error(st, "ts_export_edges_static: %d systems, the static scratch array holds at most %d (use ts_export_edges)",
                     st->d.S, TS_STATIC_EDGE_MAX_SYSTEMS);
        return TS_ERR_WORKSPACE_TOO_SMALL;
    }
    cudaError_t e = cudaSuccess;
    long long *edge_base = edge_scan_address(&e);
    if (!edge_base) { ts_set_error(st, "address of the static scratch array: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    cudaStream_t q = (cudaStream_t)stream;
    ensure_list_graph(st, q);
    const DevState &d = st->d;
    /* the array keeps what the last call left: k_edge_base rewrites entries 0 .. S before k_edge_fill reads them, and
     * nothing is accumulated into it, so nothing has to be cleared */
    k_edge_base<<<1, 256, 0, q>>>(d, edge_base, (long long *)n_edges);
    const unsigned nb = (unsigned)((d.N * 8 + 255) / 256);
    if (d.dtype == TS_F32) k_edge_fill<float><<<nb, 256, 0, q>>>(d, edge_base, (long long *)edge_i, (long long *)edge_j, (float *)edge_shift, cap);
    else k_edge_fill<double><<<nb, 256, 0, q>>>(d, edge_base, (long long *)edge_i, (long long *)edge_j, (double *)edge_shift, cap);
    st->launches += 2;
    e = cudaGetLastError();
    if (e != cudaSuccess) { ts_set_error(st, "edge export failed: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    return TS_OK;
}

static MdConst md_const(const ts_state *st, const ts_md_params *p)
{
    MdConst c;
    c.integrator = p->integrator;
    c.dt = p->dt; c.hdt = 0.5 * p->dt;
    c.c1 = exp(-p->friction * p->dt);
    c.c2 = sqrt(1.0 - c.c1 * c.c1);
    c.kT = st->d.kB * p->temperature;
    c.key0 = (unsigned)(p->seed & 0xffffffffull); c.key1 = (unsigned)(p->seed >> 32);
    return c;
}

extern "C" ts_status ts_md_step_external(ts_state *st, const ts_md_params *p, int32_t phase, void *stream)
{
    if (!st || !p || (p->integrator != TS_NVE && p->integrator != TS_BAOAB) || !(p->dt > 0.0)) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    cudaStream_t q = (cudaStream_t)stream;
    const MdConst c = md_const(st, p);
    st->last_engine = 0;
    switch (phase) {
    case TS_PHASE_INIT:                                   /* list for the current positions; the caller then computes F(x) */
        ensure_list_graph(st, q);
        break;
    case TS_PHASE_PRE:                                    /* B A (O A) with the caller's forces, skin check, rebuild if due */
        launch_md_pre(st, c, q);
        launch_build(st, false, q);
        break;
    case TS_PHASE_POST:                                   /* B with the caller's forces at the new positions, kinetic energy */
        launch_md_post(st, c, true, q);
        st->steps_done += 1;
        st->forces_current = true;
        break;
    default:
        return TS_ERR_INVALID_ARG;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ts_set_error(st, "kernel launch failed: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    return TS_OK;
}

extern "C" ts_status ts_fire_step_external(ts_state *st, const ts_fire_params *p, int32_t phase, void *stream)
{
    if (!st || !p || !(p->dt_start > 0.0) || !(p->dt_max > 0.0) || !(p->f_max > 0.0)) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    cudaStream_t q = (cudaStream_t)stream;
    st->last_engine = 0;
    switch (phase) {
    case TS_PHASE_INIT:                                   /* fresh systems: v = 0, dt_start, alpha_start; list for the current positions */
        launch_fire_init(st, *p, q);
        ensure_list_graph(st, q);
        break;
    case TS_PHASE_CHECK0:                                 /* after the caller's first force evaluation: the 0-step convergence test */
        launch_fire_check0(st, *p, q);
        st->forces_current = true;
        break;
    case TS_PHASE_PRE:
        launch_fire_pre(st, *p, q);
        launch_build(st, false, q);
        break;
    case TS_PHASE_POST:                                   /* second half kick, the four reductions, the FIRE state machine */
        launch_fire_post(st, *p, q);
        st->steps_done += 1;
        st->forces_current = true;
        break;
    default:
        return TS_ERR_INVALID_ARG;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ts_set_error(st, "kernel launch failed: %s", cudaGetErrorString(e)); return TS_ERR_CUDA; }
    return TS_OK;
}
