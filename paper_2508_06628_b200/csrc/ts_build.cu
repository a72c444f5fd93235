/*
 * ts_build.cu -- binned cell-list neighbour build (readings R5..R9, R27).
 *
 * Pipeline (all kernels early-exit unless status->need_rebuild is set, so the whole build can sit
 * in the stream every step without a host round trip):
 *   k_build_begin : zero the per-cell counters
 *   k_bin         : f = x . h^-1 (fp64), wrap = floor(f), bin id, rank in cell (atomic counter)
 *   k_cellscan    : per-system exclusive scan of the cell counters (block per system; the key
 *                   space of system s is [sysoff[s]+s, sysoff[s+1]+s] so no global scan exists)
 *   k_scatter     : counting-sort scatter of wrapped fp64 coordinates; x_ref and pos4 refresh
 *   k_nbr_fill    : quarter-warp walk of the (2D+1)^3 extended-bin stencil, rows buffered in shared memory,
 *                   reserved in the system's CSR segment with one atomicAdd and copied out (ONE pass)
 *   k_nbr_finish  : cursor > capacity -> overflow state (flag, nothing was written past capacity)
 * The cutoff test is strict r^2 < r_list^2 in fp64 on the promoted coordinates (R9, R27).
 */
#include "ts_internal.cuh"

template <typename T>
__global__ void k_geometry(DevState d, const int *slots, int count)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= count) return;
    int s = slots ? slots[t] : t;
    const T *c = (const T *)d.cell + 9 * (size_t)s;
    SysGeom g;
    for (int k = 0; k < 9; ++k) g.h[k] = (double)c[k];
    const double *h = g.h;
    double c00 = h[4] * h[8] - h[5] * h[7];
    double c01 = h[5] * h[6] - h[3] * h[8];
    double c02 = h[3] * h[7] - h[4] * h[6];
    double det = h[0] * c00 + h[1] * c01 + h[2] * c02;
    g.bad = !(fabs(det) > 0.0);
    double id = g.bad ? 0.0 : 1.0 / det;
    g.hinv[0] = c00 * id;
    g.hinv[1] = (h[2] * h[7] - h[1] * h[8]) * id;
    g.hinv[2] = (h[1] * h[5] - h[2] * h[4]) * id;
    g.hinv[3] = c01 * id;
    g.hinv[4] = (h[0] * h[8] - h[2] * h[6]) * id;
    g.hinv[5] = (h[2] * h[3] - h[0] * h[5]) * id;
    g.hinv[6] = c02 * id;
    g.hinv[7] = (h[1] * h[6] - h[0] * h[7]) * id;
    g.hinv[8] = (h[0] * h[4] - h[1] * h[3]) * id;
    g.vol = fabs(det);
    int ns = d.sysoff[s + 1] - d.sysoff[s];
    for (int k = 0; k < 3; ++k) {
        double n2 = g.hinv[k] * g.hinv[k] + g.hinv[3 + k] * g.hinv[3 + k] + g.hinv[6 + k] * g.hinv[6 + k];
        g.hperp[k] = g.bad ? 1.0 : 1.0 / sqrt(n2);
        double q = g.hperp[k] / d.r_list;
        g.nb[k] = q >= 2.0 ? (q < 1024.0 ? (int)floor(q) : 1024) : 1;
    }
    /* never more cells than atoms: the per-system key space has ns + 1 slots */
    while ((long long)g.nb[0] * g.nb[1] * g.nb[2] > (long long)(ns > 1 ? ns : 1)) {
        int m = (g.nb[0] >= g.nb[1] && g.nb[0] >= g.nb[2]) ? 0 : (g.nb[1] >= g.nb[2] ? 1 : 2);
        g.nb[m] -= 1;
    }
    g.ncell = g.nb[0] * g.nb[1] * g.nb[2];
    for (int k = 0; k < 3; ++k) {
        double w = d.r_list * (double)g.nb[k] / g.hperp[k];
        int D = (int)ceil(w * (1.0 + 1e-12));
        if (D < 1) D = 1;
        if (D > 15) { D = 15; g.bad = 1; }
        g.D[k] = D;
    }
    if (g.bad) atomicOr(&d.status->flags, TS_FLAG_BAD_CELL);
    d.geom[s] = g;
    T *hT = (T *)d.hT + 9 * (size_t)s;
    for (int k = 0; k < 9; ++k) hT[k] = c[k];
}

/* Only the systems whose skin flag is set (sys_rebuild) are rebuilt: every system has its own bin range, its own
 * CSR segment and its own reference positions, so a build touches nothing of the others (R12). */
__global__ void k_build_begin(DevState d)
{
    if (!d.status->need_rebuild) return;
    for (int s = blockIdx.x; s < d.S; s += gridDim.x) {
        if (!d.sys_rebuild[s]) continue;
        const int base = ts_cell_base(d.sysoff, s), nc = d.geom[s].ncell;
        for (int c = threadIdx.x; c <= nc; c += blockDim.x) d.cell_count[base + c] = 0;
        if (threadIdx.x == 0) {
            d.nbr_len[s] = 0;                                  /* row cursor of the system's CSR segment (k_nbr_fill) */
            atomicAdd(&d.status->res_rebuilds, 1ull);          /* per-system list builds, summed over systems */
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        d.status->nnz = 0ull;
        d.status->list_valid = 1u;
        d.status->n_rebuilds += 1;
    }
}

__global__ void k_build_end(DevState d)
{
    /* no early exit here: block 0 clears need_rebuild, and a block that starts later must still clear its flags */
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < d.S; s += gridDim.x * blockDim.x) d.sys_rebuild[s] = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) d.status->need_rebuild = 0u;
}

template <typename T>
__global__ void k_bin(DevState d)
{
    if (!d.status->need_rebuild) return;
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (!d.sys_rebuild[s]) return;
    const SysGeom &g = d.geom[s];
    const T *x = (const T *)d.pos + 3 * i;
    double x0 = (double)x[0], x1 = (double)x[1], x2 = (double)x[2];
    int c[3], w[3];
    bool range = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double f = x0 * g.hinv[k] + x1 * g.hinv[3 + k] + x2 * g.hinv[6 + k];
        double fl = floor(f);
        double fw = f - fl;
        int nb = g.nb[k];
        int ck = (int)(fw * (double)nb);
        c[k] = ck < 0 ? 0 : (ck >= nb ? nb - 1 : ck);
        if (!(fabs(fl) <= 100.0)) { range = true; fl = 0.0; }
        w[k] = (int)fl;
    }
    if (range) atomicOr(&d.status->flags, TS_FLAG_SHIFT_RANGE);
    int cid = ts_cell_base(d.sysoff, s) + (c[0] * g.nb[1] + c[1]) * g.nb[2] + c[2];
    d.atom_cell[i] = cid;
    d.atom_rank[i] = atomicAdd(&d.cell_count[cid], 1);
    d.atom_wrap[i] = ts_pack_wrap(w[0], w[1], w[2]);
}

/* Exclusive block scan helper: returns the exclusive prefix of v, total in *tot (all threads). */
template <typename V>
__device__ __forceinline__ V block_excl_scan(V v, V *sh /* [33] */, V *tot)
{
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    V inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        V u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    __syncthreads();
    if (lane == 31) sh[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        V w = lane < nw ? sh[lane] : (V)0;
        V winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            V u = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += u;
        }
        if (lane < nw) sh[lane] = winc - w;
        if (lane == 31) sh[32] = winc;
    }
    __syncthreads();
    *tot = sh[32];
    return inc - v + sh[wid];
}

__global__ void k_cellscan(DevState d)
{
    if (!d.status->need_rebuild) return;
    __shared__ int sh[33];
    int s = blockIdx.x;
    if (!d.sys_rebuild[s]) return;
    int base = ts_cell_base(d.sysoff, s);
    int nc = d.geom[s].ncell;
    int run = d.sysoff[s];
    for (int c0 = 0; c0 < nc; c0 += blockDim.x) {
        int c = c0 + threadIdx.x;
        int v = c < nc ? d.cell_count[base + c] : 0;
        int tot;
        int ex = block_excl_scan<int>(v, sh, &tot);
        if (c < nc) d.cell_start[base + c] = run + ex;
        run += tot;
    }
    if (threadIdx.x == 0) {
        d.cell_start[base + nc] = run;
    }
    /* The ranks k_bin handed out inside a cell came from an atomic counter: their order changes from run to run, and with
     * it the order of the neighbours in every row and the rounding of every force.  Make them canonical (by atom index):
     * the block lists the atoms of every cell (nbr_cnt serves as scratch: k_nbr_fill writes it afterwards), then a warp
     * per cell ranks each atom by the number of smaller indices in its cell. */
    __syncthreads();
    const int a0 = d.sysoff[s], a1 = d.sysoff[s + 1];
    int *order = d.nbr_cnt;
    for (int i = a0 + threadIdx.x; i < a1; i += blockDim.x) order[d.cell_start[d.atom_cell[i]] + d.atom_rank[i]] = i;
    __syncthreads();
    const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (int c = threadIdx.x >> 5; c < nc; c += nw) {
        const int c0 = d.cell_start[base + c], n = d.cell_start[base + c + 1] - c0;
        for (int k = lane; k < n; k += 32) {
            const int id = order[c0 + k];
            int rank = 0;
            for (int m = 0; m < n; ++m) rank += order[c0 + m] < id;
            d.atom_rank[id] = rank;
        }
    }
}

template <typename T>
__global__ void k_scatter(DevState d)
{
    if (!d.status->need_rebuild) return;
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    int s = d.sysidx[i];
    if (!d.sys_rebuild[s]) return;
    const SysGeom &g = d.geom[s];
    const T *x = (const T *)d.pos + 3 * i;
    T xs0 = x[0], xs1 = x[1], xs2 = x[2];
    int w0, w1, w2;
    ts_unpack_wrap(d.atom_wrap[i], w0, w1, w2);
    double xw0 = (double)xs0 - ((double)w0 * g.h[0] + (double)w1 * g.h[3] + (double)w2 * g.h[6]);
    double xw1 = (double)xs1 - ((double)w0 * g.h[1] + (double)w1 * g.h[4] + (double)w2 * g.h[7]);
    double xw2 = (double)xs2 - ((double)w0 * g.h[2] + (double)w1 * g.h[5] + (double)w2 * g.h[8]);
    int p = d.cell_start[d.atom_cell[i]] + d.atom_rank[i];
    int li = (int)(i - d.sysoff[s]);
    d.spos[p] = make_double4(xw0, xw1, xw2, __longlong_as_double((long long)li));
    T *xr = (T *)d.xref + 3 * i;
    xr[0] = xs0; xr[1] = xs1; xr[2] = xs2;
    typedef typename Vec4<T>::type V4;
    V4 q;
    q.x = (T)xw0; q.y = (T)xw1; q.z = (T)xw2;
    int ty = d.type[i];
    if (sizeof(T) == 4) q.w = (T)__int_as_float(ty); else q.w = (T)__longlong_as_double((long long)ty);
    ((V4 *)d.pos4)[i] = q;
}

__device__ __forceinline__ int floordiv(int a, int n) { int q = a / n; return (a % n < 0) ? q - 1 : q; }

/* Neighbour search, ONE pass.  One quarter-warp (8 lanes) per sorted slot p, four consecutive slots per warp: sorted
 * slots that follow each other sit in the same or in adjacent bins, so the four stencil walks of a warp stay converged
 * and share their loads.  The lanes of a quarter stride over the atoms of each stencil bin; hits are compacted with a
 * quarter-wide ballot into a shared-memory buffer (NBR_BUF entries per atom).  When the walk is done the quarter
 * reserves a contiguous row inside the CSR segment of its system with one atomicAdd on the system's cursor (nbr_len)
 * and copies the row out: no counting pass, no scan (a row longer than the buffer is walked a second time and written
 * straight into the reserved place).  Rows of a system are therefore stored in arrival order (nbr_off
 * says where); the content and order of every row are deterministic.  Nothing is written past the capacity of the
 * segment: a row that does not fit only advances the cursor, and k_nbr_finish turns cursor > capacity into the
 * overflow state (nbr_len = -1, TS_FLAG_NBR_OVERFLOW).  The grid is capped (grid-stride over the slots): when no
 * rebuild is due the launch costs a few microseconds. */
#define NBR_BUF 256
__global__ void __launch_bounds__(256) k_nbr_fill(DevState d)
{
    if (!d.status->need_rebuild) return;
    __shared__ unsigned buf[32 * NBR_BUF];
    const int lane = threadIdx.x & 31, l = lane & 7, qg = lane >> 3;
    unsigned *const mybuf = buf + (size_t)(threadIdx.x >> 3) * NBR_BUF;
    const unsigned qmask = 0xffu << (8 * qg);
    const unsigned lt = (1u << l) - 1u;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const double R2 = d.r_list2;
    unsigned mx = 0u;
    for (long long p4 = (((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 4; p4 < d.N; p4 += nwarps * 4) {
        const long long p = p4 + qg;
        if (p >= d.N) continue;
        const int s = d.sysidx[p];           /* sorted slots of a system occupy the system's own range */
        if (!d.sys_rebuild[s]) continue;
        const SysGeom &g = d.geom[s];
        const int a0 = d.sysoff[s];
        const int base = a0 + s;
        const double4 me = d.spos[p];
        const int li = (int)__double_as_longlong(me.w);
        const int lin = d.atom_cell[a0 + li] - base;
        const int nb0 = g.nb[0], nb1 = g.nb[1], nb2 = g.nb[2];
        const int c2 = lin % nb2, c1 = (lin / nb2) % nb1, c0 = lin / (nb2 * nb1);
        const int D0 = g.D[0], D1 = g.D[1], D2 = g.D[2];
        int cnt = 0;
        long long start = 0;
        const long long seg = d.nbr_base[s], cap = d.nbr_base[s + 1] - seg;
        /* pass 0 buffers the row in shared memory; a row longer than the buffer is walked a second time and written
         * straight into its reserved place (pass 1: rare, so the second walk costs nothing on average) */
        for (int pass = 0; pass < 2; ++pass) {
        const bool direct = pass == 1;
        unsigned *const out = d.nbr + seg + start;
        const bool room = start + cnt <= cap;                    /* pass 1: cnt is the length found by pass 0 */
        cnt = 0;
        for (int e0 = c0 - D0; e0 <= c0 + D0; ++e0) {
            const int s0 = floordiv(e0, nb0), b0 = e0 - s0 * nb0;
            for (int e1 = c1 - D1; e1 <= c1 + D1; ++e1) {
                const int s1 = floordiv(e1, nb1), b1 = e1 - s1 * nb1;
                const double tx = (double)s0 * g.h[0] + (double)s1 * g.h[3] - me.x;
                const double ty = (double)s0 * g.h[1] + (double)s1 * g.h[4] - me.y;
                const double tz = (double)s0 * g.h[2] + (double)s1 * g.h[5] - me.z;
                for (int e2 = c2 - D2; e2 <= c2 + D2; ++e2) {
                    const int s2 = floordiv(e2, nb2), b2 = e2 - s2 * nb2;
                    const int cell = base + (b0 * nb1 + b1) * nb2 + b2;
                    const int q0 = d.cell_start[cell], q1 = d.cell_start[cell + 1];
                    if (q0 == q1) continue;
                    const double sx = tx + (double)s2 * g.h[6], sy = ty + (double)s2 * g.h[7], sz = tz + (double)s2 * g.h[8];
                    const bool home = (s0 == 0) & (s1 == 0) & (s2 == 0);
                    for (int q = q0; q < q1; q += 8) {
                        const int qq = q + l;
                        bool ok = false;
                        int lj = 0;
                        if (qq < q1) {
                            const double4 c = d.spos[qq];
                            const double rx = c.x + sx, ry = c.y + sy, rz = c.z + sz;
                            const double r2 = rx * rx + ry * ry + rz * rz;
                            lj = (int)__double_as_longlong(c.w);
                            ok = (r2 < R2) && !(home && qq == (int)p);
                        }
                        const unsigned m = (__ballot_sync(qmask, ok) >> (8 * qg)) & 0xffu;
                        const int at = cnt + __popc(m & lt);
                        if (ok) {
                            if (direct) { if (room) out[at] = ts_pack_nbr(lj, s0, s1, s2); }
                            else if (at < NBR_BUF) mybuf[at] = ts_pack_nbr(lj, s0, s1, s2);
                        }
                        cnt += __popc(m);
                    }
                }
            }
        }
        if (direct) break;
        /* reserve the row and copy it out */
        if (l == 0) start = (long long)atomicAdd((unsigned long long *)&d.nbr_len[s], (unsigned long long)cnt);
        start = __shfl_sync(qmask, start, 8 * qg);
        __syncwarp(qmask);
        if (cnt <= NBR_BUF) {
            if (start + cnt <= cap)
                for (int k = l; k < cnt; k += 8) d.nbr[seg + start + k] = mybuf[k];
            break;
        }
        }
        __syncwarp(qmask);
        if (l == 0) {
            d.nbr_off[a0 + li] = seg + start;
            d.nbr_cnt[a0 + li] = cnt;
            mx = max(mx, (unsigned)cnt);
        }
    }
    /* statistics: one atomic per warp */
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 0 && mx) atomicMax(&d.status->max_nbr, mx);
}

/* cursor -> state of the segment: pairs in use, or -1 when the rows did not fit (overflow: flagged, list invalid) */
__global__ void k_nbr_finish(DevState d)
{
    if (!d.status->need_rebuild) return;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= d.S) return;
    if (ts_skip(d, s)) return;
    const long long cap = d.nbr_base[s + 1] - d.nbr_base[s];
    long long len = d.nbr_len[s];
    if (d.sys_rebuild[s] && len > cap) {
        len = -1;
        d.nbr_len[s] = -1;
        atomicOr(&d.status->flags, TS_FLAG_NBR_OVERFLOW);
    }
    if (len < 0) d.status->list_valid = 0u;                    /* also a system that overflowed earlier and was not rebuilt */
    else atomicAdd(&d.status->nnz, (unsigned long long)len);  /* pairs of the whole batch, rebuilt or not */
}

/* ------------------------------------------------------------------ host launchers */
void launch_geometry(ts_state *st, int s_first, int s_count, const int *slots, cudaStream_t q)
{
    (void)s_first;
    int nb = (s_count + 127) / 128;
    if (st->d.dtype == TS_F32) k_geometry<float><<<nb, 128, 0, q>>>(st->d, slots, s_count);
    else k_geometry<double><<<nb, 128, 0, q>>>(st->d, slots, s_count);
    st->launches += 1;
}

__global__ void k_force_rebuild(DevState d)
{
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < d.S; s += gridDim.x * blockDim.x) d.sys_rebuild[s] = ts_skip(d, s) ? 0 : 1;
    if (blockIdx.x == 0 && threadIdx.x == 0) { d.status->need_rebuild = 1u; d.status->max_nbr = 0u; }
}

void launch_build(ts_state *st, bool force, cudaStream_t q)
{
    const DevState &d = st->d;
    /* a whole-batch build writes every system's segment of `nbr`: the lists the resident engine saved there are gone
     * (in mixed mode the kernels below skip the resident engine's systems and their segments stay) */
    if (!d.mixed) st->res_saved_ok = false;
    if (force) { k_force_rebuild<<<(d.S + 255) / 256, 256, 0, q>>>(d); st->launches += 1; }
    int tb = 256;
    int nba = (int)((d.N + tb - 1) / tb);
    long long nwarp_blocks = (d.N * 8 + tb - 1) / tb;          /* 8 lanes per atom ... */
    if (nwarp_blocks > 148 * 16) nwarp_blocks = 148 * 16;       /* ... in a capped, grid-stride grid */
    k_build_begin<<<d.S < 148 * 8 ? d.S : 148 * 8, tb, 0, q>>>(d);
    if (d.dtype == TS_F32) k_bin<float><<<nba, tb, 0, q>>>(d); else k_bin<double><<<nba, tb, 0, q>>>(d);
    k_cellscan<<<d.S, 256, 0, q>>>(d);
    if (d.dtype == TS_F32) k_scatter<float><<<nba, tb, 0, q>>>(d); else k_scatter<double><<<nba, tb, 0, q>>>(d);
    k_nbr_fill<<<(unsigned)nwarp_blocks, tb, 0, q>>>(d);
    k_nbr_finish<<<(d.S + 255) / 256, 256, 0, q>>>(d);
    k_build_end<<<(d.S + 255) / 256, 256, 0, q>>>(d);
    st->launches += 7;
    if (force) st->list_built = true;                          /* a skin-checked build keeps what the forced one established */
}
