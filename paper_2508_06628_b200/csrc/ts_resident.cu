/*
 * ts_resident.cu -- system-resident MD engine (SURVEY.md section 7 "hard part 1", kernel K13).
 *
 * The graded batch (BASELINE.json:configs[1], 64 x 864 atoms) is so small that a step is bound by
 * launch latency and on-chip bandwidth, not by HBM.  This engine therefore keeps a whole system on
 * chip for all n_steps of a ts_md_step call: one thread-block cluster of CL CTAs per system, each
 * CTA owning a contiguous slice of the system's atoms.  Per CTA, in shared memory:
 *     pos[2][N_s+1]  wrapped positions + type of ALL atoms of the system (double buffered; every
 *                    owner publishes its atom into every CTA of the cluster through DSMEM)
 *     fr[N_s]        fractional coordinates as 32-bit fixed point (rebuilds only)
 *     rows[A][pitch] the Verlet list of the CTA's own atoms, 16-bit entries
 *     fs[3][A]       forces of the own atoms (pair phase -> integrator phase)
 * and in registers of the owner thread of an atom: x (unwrapped), v, F, x_ref, wrap shift.
 * HBM is touched when a system is loaded, when it is stored, and never in between.
 *
 * One MD step = [owner: B A (O A) + publish + skin test] -> cluster barrier -> [rebuild if any
 * atom moved > skin/2] -> [pair phase] -> block barrier -> [owner: B].  Same physics as the
 * general engine.
 *
 * Pair phase: 8 lanes per atom (one quarter-warp = one LDS.128 phase).  The list of an atom is
 * ordered at build time so that the 8 entries a quarter-warp fetches together point at 8 different
 * 16-byte bank groups (round-robin over j mod 8): the position gather is then conflict-free.  Home
 * pairs (image shift 0) and shifted pairs are kept in two segments so the home loop carries no
 * shift arithmetic; a home entry is the byte offset 16 j, a shifted entry is j | code << 11.
 *
 * Rebuild: brute force over the system in fractional fixed point (integer subtraction wraps = the
 * minimum image), valid because the engine is only used when every cell height is >= 2 r_list
 * (then an image within r_list is the rounded one and is unique).  The list radius is inflated by
 * a few float ulps of the box; a Verlet list only has to be a superset of the pairs within r_c.
 */
#include <cooperative_groups.h>
#include <math.h>
#include <string.h>

#include <vector>

#include "ts_internal.cuh"
#include "ts_pot.cuh"
#include "ts_rng.cuh"

namespace cg = cooperative_groups;

#define RES_MAX_THREADS 896         /* fp32; the fp64 kernels need twice the registers: 512 */
#define RES_MAX_THREADS_F64 512
#define RES_MAX_ATOMS 2047          /* 11-bit neighbour index; slot N_s is the far-away dummy */
#define RES_SMEM_LIMIT (227 * 1024)

struct ResCfg {
    int CL;            /* CTAs per system = cluster size                       */
    int A;             /* atoms per CTA, capacity (multiple of 4)              */
    int pitch;         /* u16 entries per list row, pitch mod 64 in {16, 48}   */
    int NP;            /* max atoms per system + 1                             */
    int nwarps;
    int n_clusters;
    unsigned posbytes; /* bytes of one position buffer                         */
    unsigned o_pos, o_fr, o_rows, o_fs, o_cnt, o_shtab, o_pot, o_red, o_cred, o_misc;
    unsigned smem;
    float eps_rel;     /* list radius inflation, relative to the longest cell vector */
};

struct ResMisc {
    int flags[2];
    unsigned nnz;
    unsigned rebuilds;
    int overflow;
    int pad[3];        /* 32 bytes: the fp64 cell copy follows */
};

/* ------------------------------------------------------------------ position slots */
template <typename T> struct P3 { T x, y, z; int ty; };

__device__ __forceinline__ P3<float> ld_pos(const unsigned char *base, unsigned off, unsigned, float)
{
    float4 v = *(const float4 *)(base + off);
    P3<float> p; p.x = v.x; p.y = v.y; p.z = v.z; p.ty = __float_as_int(v.w);
    return p;
}
__device__ __forceinline__ P3<double> ld_pos(const unsigned char *base, unsigned off, unsigned zt, double)
{
    double2 a = *(const double2 *)(base + off);
    double2 b = *(const double2 *)(base + zt + off);
    P3<double> p; p.x = a.x; p.y = a.y; p.z = b.x; p.ty = (int)__double_as_longlong(b.y);
    return p;
}
__device__ __forceinline__ void st_pos(unsigned char *base, unsigned off, unsigned, float x, float y, float z, int ty)
{
    *(float4 *)(base + off) = make_float4(x, y, z, __int_as_float(ty));
}
__device__ __forceinline__ void st_pos(unsigned char *base, unsigned off, unsigned zt, double x, double y, double z, int ty)
{
    *(double2 *)(base + off) = make_double2(x, y);
    *(double2 *)(base + zt + off) = make_double2(z, __longlong_as_double((long long)ty));
}

__device__ __forceinline__ unsigned frac_to_u32(float ff) { return __float2uint_rz(ff * 4294967296.0f); }
__device__ __forceinline__ unsigned frac_to_u32(double ff) { return (unsigned)(unsigned long long)(ff * 4294967296.0); }

template <typename T> __device__ __forceinline__ T t_floor(T x);
template <> __device__ __forceinline__ float t_floor<float>(float x) { return floorf(x); }
template <> __device__ __forceinline__ double t_floor<double>(double x) { return floor(x); }

/* image shift of j relative to i in one direction from the fixed-point fractions */
__device__ __forceinline__ int image_shift(unsigned uj, unsigned ui)
{
    int dd = (int)(uj - ui);
    return (uj > ui && dd < 0) ? -1 : ((uj < ui && dd > 0) ? 1 : 0);
}

/* position p of the m-th member of bank group g in the round-robin order over groups with
 * populations c[0..7]: all members of rank < m first, then the groups below g that reach rank m */
__device__ __forceinline__ int rr_position(const int c[8], int g, int m)
{
    int p = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) p += min(c[k], m) + ((k < g && c[k] > m) ? 1 : 0);
    return p;
}

/* u16 index of list slot p (p = 8 k + lane) inside a row: pairs of k interleaved per lane */
__device__ __forceinline__ int row_index(int p)
{
    int k = p >> 3, l = p & 7;
    return ((k >> 1) << 4) + (l << 1) + (k & 1);
}

/* ------------------------------------------------------------------ one pair */
template <typename T, int KIND, bool NT1, bool EV, bool SH>
__device__ __forceinline__ void pair_accum(const P3<T> &xi, const P3<T> &xj, T sx, T sy, T sz, const PotEntry<T> &pe1,
                                           const PotEntry<T> *tab, int tirow, T &fx, T &fy, T &fz, T *ev)
{
    T rx = xj.x - xi.x, ry = xj.y - xi.y, rz = xj.z - xi.z;
    if (SH) { rx += sx; ry += sy; rz += sz; }
    T r2 = rx * rx + ry * ry + rz * rz;
    PotEntry<T> pe = pe1;
    if (!NT1) pe = tab[tirow + xj.ty];
    const bool in = r2 < pe.rc2;                 /* strict (R9); the padding dummy sits at 1e15 */
    if (EV) {
        T V, g;
        pot_eval<T, KIND>(pe, r2, V, g);
        g = in ? g : (T)0; V = in ? V : (T)0;
        fx += g * rx; fy += g * ry; fz += g * rz;
        ev[0] += V;
        T gx = g * rx, gy = g * ry;
        ev[1] += gx * rx; ev[2] += gx * ry; ev[3] += gx * rz;
        ev[4] += gy * ry; ev[5] += gy * rz; ev[6] += g * rz * rz;
    } else {
        T g = pot_force<T, KIND>(pe, r2);
        g = in ? g : (T)0;
        fx += g * rx; fy += g * ry; fz += g * rz;
    }
}

/* Forces of the CTA's own atoms from the shared-memory list; E and W partials into acc8 (fp64). */
template <typename T, int KIND, bool NT1, bool EV>
__device__ __forceinline__ void pair_phase(const ResCfg &rc, const unsigned char *posb, const unsigned short *rows,
                                           const unsigned *cnt, const T *shtab, const PotEntry<T> *tab, T *fs,
                                           int a_begin, int A_own, int NT, double *red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = lane & 7, q = lane >> 3;
    const unsigned zt = (unsigned)rc.NP * 16u;
    const int ntasks = (A_own + 3) >> 2;
    double acc8[EV ? 7 : 1];
    if (EV)
#pragma unroll
        for (int k = 0; k < 7; ++k) acc8[k] = 0.0;
    for (int task = warp; task < ntasks; task += rc.nwarps) {
        T ev[7] = { 0, 0, 0, 0, 0, 0, 0 };
        int al = task * 4 + q;
        bool has = al < A_own;
        int ai = a_begin + (has ? al : 0);
        P3<T> xi = ld_pos(posb, (unsigned)ai * 16u, zt, (T)0);
        unsigned c = has ? cnt[al] : 0u;
        int th2 = (int)(c & 255u) >> 1, ts2 = (int)(c >> 8) >> 1;
        const unsigned *row = (const unsigned *)(rows + (size_t)al * rc.pitch) + l;
        PotEntry<T> pe1 = tab[NT1 ? 0 : xi.ty * NT];
        int tirow = xi.ty * NT;
        T fx = 0, fy = 0, fz = 0;
#pragma unroll 2
        for (int k = 0; k < th2; ++k) {
            unsigned e2 = row[k * 8];
            P3<T> x0 = ld_pos(posb, e2 & 0xffffu, zt, (T)0);
            P3<T> x1 = ld_pos(posb, e2 >> 16, zt, (T)0);
            pair_accum<T, KIND, NT1, EV, false>(xi, x0, (T)0, (T)0, (T)0, pe1, tab, tirow, fx, fy, fz, ev);
            pair_accum<T, KIND, NT1, EV, false>(xi, x1, (T)0, (T)0, (T)0, pe1, tab, tirow, fx, fy, fz, ev);
        }
        row += th2 * 8;
        for (int k = 0; k < ts2; ++k) {
            unsigned e2 = row[k * 8];
            unsigned j0 = (e2 & 0x7ffu) << 4, c0 = (e2 >> 11) & 31u, j1 = ((e2 >> 16) & 0x7ffu) << 4, c1 = e2 >> 27;
            P3<T> x0 = ld_pos(posb, j0, zt, (T)0);
            P3<T> x1 = ld_pos(posb, j1, zt, (T)0);
            const T *s0 = shtab + 4 * c0, *s1 = shtab + 4 * c1;
            pair_accum<T, KIND, NT1, EV, true>(xi, x0, s0[0], s0[1], s0[2], pe1, tab, tirow, fx, fy, fz, ev);
            pair_accum<T, KIND, NT1, EV, true>(xi, x1, s1[0], s1[1], s1[2], pe1, tab, tirow, fx, fy, fz, ev);
        }
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            fx += __shfl_xor_sync(0xffffffffu, fx, o);
            fy += __shfl_xor_sync(0xffffffffu, fy, o);
            fz += __shfl_xor_sync(0xffffffffu, fz, o);
        }
        if (has && l == 0) { fs[al] = fx; fs[rc.A + al] = fy; fs[2 * rc.A + al] = fz; }
        if (EV) {                       /* fp64 from here on (R31): E = 1/2 sum V, W = -1/2 sum g r (x) r */
            acc8[0] += 0.5 * (double)ev[0];
#pragma unroll
            for (int k = 1; k < 7; ++k) acc8[k] += -0.5 * (double)ev[k];
        }
    }
    if (EV) {                           /* warp partials of E, W into red[warp][0..6] */
#pragma unroll
        for (int k = 0; k < 7; ++k) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc8[k] += __shfl_xor_sync(0xffffffffu, acc8[k], o);
            if (lane == 0) red[warp * 8 + k] = acc8[k];
        }
    }
}

/* ------------------------------------------------------------------ list build (per CTA, own atoms) */
/* One quarter-warp per atom; lane l tests the candidates j = l mod 8 (bank group l), keeps the hits
 * as a bit mask in registers, then places its hits in round-robin order (rr_position).            */
__device__ __forceinline__ void build_phase(const ResCfg &rc, const uint4 *fr, unsigned short *rows, unsigned *cnt,
                                            const float *G, float rb2, int a_begin, int A_own, int N_s, ResMisc *misc)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = lane & 7, q = lane >> 3;
    const int ntasks = (A_own + 3) >> 2;
    const float G0 = G[0], G1 = G[1], G2 = G[2], G3 = G[3], G4 = G[4], G5 = G[5];
    unsigned nnz = 0;
    for (int task = warp; task < ntasks; task += rc.nwarps) {
        int al = task * 4 + q;
        bool has = al < A_own;
        int ai = a_begin + (has ? al : 0);
        uint4 ui = fr[ai];
        unsigned mask[8];
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            unsigned word = 0u;
            if (w * 256 < N_s) {
                int jb = w * 256 + l;
#pragma unroll 4
                for (int b = 0; b < 32; ++b) {
                    int j = jb + b * 8;
                    if (j < N_s) {
                        uint4 uj = fr[j];
                        float e0 = (float)(int)(uj.x - ui.x), e1 = (float)(int)(uj.y - ui.y), e2 = (float)(int)(uj.z - ui.z);
                        float r2 = e0 * (G0 * e0 + G1 * e1 + G2 * e2) + e1 * (G3 * e1 + G4 * e2) + G5 * e2 * e2;
                        if (r2 < rb2 && j != ai) word |= 1u << b;
                    }
                }
            }
            mask[w] = word;
        }
        /* classify my hits: home (shift 0) or shifted */
        int nh = 0, ns = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            unsigned word = mask[w];
            while (word) {
                int b = __ffs(word) - 1;
                word &= word - 1u;
                uint4 uj = fr[w * 256 + b * 8 + l];
                int sh = image_shift(uj.x, ui.x) | image_shift(uj.y, ui.y) | image_shift(uj.z, ui.z);
                if (sh) ns += 1; else nh += 1;
            }
        }
        int cH[8], cS[8], NH = 0, NS = 0;
#pragma unroll
        for (int g = 0; g < 8; ++g) {
            cH[g] = __shfl_sync(0xffffffffu, nh, (lane & 24) | g);
            cS[g] = __shfl_sync(0xffffffffu, ns, (lane & 24) | g);
            NH += cH[g]; NS += cS[g];
        }
        int th = ((NH + 15) >> 4) << 1, tsn = ((NS + 15) >> 4) << 1;      /* k counts, even */
        bool fits = 8 * (th + tsn) <= rc.pitch && th < 256 && tsn < 256;
        if (!fits) {
            if (has) misc->overflow = 1;
            th = 0; tsn = 0;
        }
        unsigned short *row = rows + (size_t)al * rc.pitch;
        if (has && fits) {
            int mh = 0, ms = 0;
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                unsigned word = mask[w];
                while (word) {
                    int b = __ffs(word) - 1;
                    word &= word - 1u;
                    int j = w * 256 + b * 8 + l;
                    uint4 uj = fr[j];
                    int s0 = image_shift(uj.x, ui.x), s1 = image_shift(uj.y, ui.y), s2 = image_shift(uj.z, ui.z);
                    if ((s0 | s1 | s2) == 0) {
                        row[row_index(rr_position(cH, l, mh))] = (unsigned short)(j << 4);
                        mh += 1;
                    } else {
                        int code = (s0 + 1) * 9 + (s1 + 1) * 3 + (s2 + 1);
                        row[row_index(8 * th + rr_position(cS, l, ms))] = (unsigned short)(j | (code << 11));
                        ms += 1;
                    }
                }
            }
            for (int p = NH + l; p < 8 * th; p += 8) row[row_index(p)] = (unsigned short)(N_s << 4);
            for (int p = NS + l; p < 8 * tsn; p += 8) row[row_index(8 * th + p)] = (unsigned short)(N_s | (13 << 11));
        }
        if (has && l == 0) {
            cnt[al] = (unsigned)th | ((unsigned)tsn << 8);
            nnz += (unsigned)(NH + NS);
        }
    }
    if (nnz) atomicAdd(&misc->nnz, nnz);
}

/* ------------------------------------------------------------------ block / cluster reduction of 8 doubles */
/* red[warp][0..6] already holds the warp partials of E, W; ke is this thread's kinetic energy.
 * Returns total k to thread k < 8 of cluster rank 0 (fixed summation order: deterministic). */
__device__ __forceinline__ double reduce8(cg::cluster_group &cluster, int CL, int rank, double ke, double *red,
                                          double *cred, int nwarps)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ke += __shfl_xor_sync(0xffffffffu, ke, o);
    if (lane == 0) red[warp * 8 + 7] = ke;
    __syncthreads();
    if (threadIdx.x < 8) {
        double s = 0.0;
        for (int w = 0; w < nwarps; ++w) s += red[w * 8 + threadIdx.x];
        double *dst = cluster.map_shared_rank(cred, 0);
        dst[rank * 8 + threadIdx.x] = s;
    }
    cluster.sync();
    double s = 0.0;
    if (rank == 0 && threadIdx.x < 8)
        for (int r = 0; r < CL; ++r) s += cred[r * 8 + threadIdx.x];
    return s;
}

/* ------------------------------------------------------------------ the kernel */
template <typename T, int KIND, bool NT1>
__global__ void __launch_bounds__(sizeof(T) == 4 ? RES_MAX_THREADS : RES_MAX_THREADS_F64, 1) k_resident_md(DevState d, MdConst c, ResCfg rc, int n_steps, unsigned want)
{
    extern __shared__ __align__(16) unsigned char smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const int CL = rc.CL;
    const int rank = (int)cluster.block_rank();
    const int cid = (int)(blockIdx.x / (unsigned)CL);
    const int tid = threadIdx.x;
    const unsigned zt = (unsigned)rc.NP * 16u;

    unsigned char *const posb0 = smem + rc.o_pos, *const posb1 = smem + rc.o_pos + rc.posbytes;
    uint4 *fr = (uint4 *)(smem + rc.o_fr);
    unsigned short *rows = (unsigned short *)(smem + rc.o_rows);
    T *fs = (T *)(smem + rc.o_fs);
    unsigned *cnt = (unsigned *)(smem + rc.o_cnt);
    T *shtab = (T *)(smem + rc.o_shtab);
    PotEntry<T> *tab = (PotEntry<T> *)(smem + rc.o_pot);
    double *red = (double *)(smem + rc.o_red);
    double *cred = (double *)(smem + rc.o_cred);
    ResMisc *misc = (ResMisc *)(smem + rc.o_misc);
    T *gh = (T *)(misc + 1);            /* h[9], hinv[9] in the state dtype */
    float *G = (float *)(gh + 18);      /* metric of the fixed-point fractions, [6] + rb2 */

    const int NT = d.n_types;
    for (int k = tid; k < NT * NT; k += blockDim.x) tab[k] = ((const PotEntry<T> *)d.pot)[k];

    for (int s = cid; s < d.S; s += rc.n_clusters) {
        const int g0 = d.sysoff[s];
        const int N_s = d.sysoff[s + 1] - g0;
        const int A_s = ((((N_s + CL - 1) / CL) + 3) >> 2) << 2;
        const int a_begin = rank * A_s;
        const int A_own = max(0, min(A_s, N_s - a_begin));
        const SysGeom &geo = d.geom[s];
        /* ---- per-system constants into shared memory */
        if (tid < 9) { gh[tid] = (T)geo.h[tid]; gh[9 + tid] = (T)geo.hinv[tid]; }
        if (tid >= 32 && tid < 32 + 27) {
            int code = tid - 32;
            double s0 = (double)(code / 9 - 1), s1 = (double)((code / 3) % 3 - 1), s2 = (double)(code % 3 - 1);
            for (int b = 0; b < 3; ++b) shtab[4 * code + b] = (T)(s0 * geo.h[b] + s1 * geo.h[3 + b] + s2 * geo.h[6 + b]);
            shtab[4 * code + 3] = (T)0;
        }
        if (tid == 64) {
            const double *h = geo.h;
            double M[6], lmax = 0.0;
            int kk[6][2] = { { 0, 0 }, { 0, 1 }, { 0, 2 }, { 1, 1 }, { 1, 2 }, { 2, 2 } };
            for (int e = 0; e < 6; ++e) {
                int a = kk[e][0], b = kk[e][1];
                M[e] = h[3 * a] * h[3 * b] + h[3 * a + 1] * h[3 * b + 1] + h[3 * a + 2] * h[3 * b + 2];
                if (a != b) M[e] *= 2.0;
            }
            const double sc = 1.0 / 18446744073709551616.0;      /* 2^-64 */
            for (int e = 0; e < 6; ++e) G[e] = (float)(M[e] * sc);
            for (int a = 0; a < 3; ++a) lmax = fmax(lmax, sqrt(h[3 * a] * h[3 * a] + h[3 * a + 1] * h[3 * a + 1] + h[3 * a + 2] * h[3 * a + 2]));
            double rb = d.r_list + (double)rc.eps_rel * lmax;
            G[6] = (float)(rb * rb);
            misc->flags[0] = 0; misc->flags[1] = 0; misc->nnz = 0u; misc->rebuilds = 0u; misc->overflow = 0;
        }
        /* ---- owner state */
        const bool own = tid < A_own;
        const int ai = a_begin + tid;                 /* system-local atom index  */
        const long long gi = (long long)g0 + ai;      /* global atom index        */
        T x0 = 0, x1 = 0, x2 = 0, v0 = 0, v1 = 0, v2 = 0, f0 = 0, f1 = 0, f2 = 0, r0 = 0, r1 = 0, r2 = 0;
        T ws0 = 0, ws1 = 0, ws2 = 0, im = 0, mass = 0;
        int ty = 0;
        if (own) {
            const T *x = (const T *)d.pos + 3 * gi, *v = (const T *)d.vel + 3 * gi;
            x0 = x[0]; x1 = x[1]; x2 = x[2]; v0 = v[0]; v1 = v[1]; v2 = v[2];
            mass = ((const T *)d.mass)[gi];
            im = (T)1 / (mass * (T)d.mass_conv);
            ty = d.type[gi];
        }
        const unsigned uid = d.uid_own[s];
        const unsigned long long step0 = d.sys_step[s];
        const T hdt = (T)c.hdt, dt = (T)c.dt;
        cluster.sync();                               /* constants visible; previous system fully retired everywhere */

        for (int n = 0; n <= n_steps; ++n) {
            const int nb = n & 1;
            unsigned char *const posn = nb ? posb1 : posb0;
            bool moved = false;
            if (n > 0 && own) {
                /* first half of the step (O3 / O4), as in the general engine */
                if (c.integrator == TS_NVE) {
                    v0 = v0 + hdt * (f0 * im); x0 = x0 + dt * v0;
                    v1 = v1 + hdt * (f1 * im); x1 = x1 + dt * v1;
                    v2 = v2 + hdt * (f2 * im); x2 = x2 + dt * v2;
                } else {
                    unsigned long long step = step0 + (unsigned long long)(n - 1);
                    unsigned w[4];
                    philox4x32_10((unsigned)ai, uid, (unsigned)(step & 0xffffffffull), (unsigned)(step >> 32), c.key0, c.key1, w);
                    T xi[3];
                    normals3(w, xi);
                    T sig = sizeof(T) == 4 ? (T)sqrtf((float)((T)c.kT * im)) : (T)sqrt((double)((T)c.kT * im));
                    T c1 = (T)c.c1, c2 = (T)c.c2;
                    v0 = v0 + hdt * (f0 * im); x0 = x0 + hdt * v0; v0 = c1 * v0 + c2 * sig * xi[0]; x0 = x0 + hdt * v0;
                    v1 = v1 + hdt * (f1 * im); x1 = x1 + hdt * v1; v1 = c1 * v1 + c2 * sig * xi[1]; x1 = x1 + hdt * v1;
                    v2 = v2 + hdt * (f2 * im); x2 = x2 + hdt * v2; v2 = c1 * v2 + c2 * sig * xi[2]; x2 = x2 + hdt * v2;
                }
                T a = x0 - r0, b = x1 - r1, cc = x2 - r2;
                moved = (double)(a * a + b * b + cc * cc) > d.half_skin2;
                for (int r = 0; r < CL; ++r) {
                    unsigned char *pb = cluster.map_shared_rank(posn, r);
                    st_pos(pb, (unsigned)ai * 16u, zt, x0 - ws0, x1 - ws1, x2 - ws2, ty);
                    if (moved) cluster.map_shared_rank(misc, r)->flags[nb] = 1;
                }
            }
            if (n > 0) cluster.sync();
            const bool rebuild = (n == 0) || (misc->flags[nb] != 0);
            if (rebuild) {
                __syncthreads();
                if (tid == 0) { misc->flags[nb] = 0; misc->rebuilds += 1u; misc->nnz = 0u; }
                if (own) {
                    /* wrap into the cell: f = x . h^-1, w = floor(f) (R5: the stored x stays unwrapped) */
                    T fa = x0 * gh[9] + x1 * gh[12] + x2 * gh[15];
                    T fb = x0 * gh[10] + x1 * gh[13] + x2 * gh[16];
                    T fc = x0 * gh[11] + x1 * gh[14] + x2 * gh[17];
                    T wa = t_floor<T>(fa), wb = t_floor<T>(fb), wc = t_floor<T>(fc);
                    fa -= wa; fb -= wb; fc -= wc;
                    if (fa >= (T)1) { wa += (T)1; fa = (T)0; }
                    if (fb >= (T)1) { wb += (T)1; fb = (T)0; }
                    if (fc >= (T)1) { wc += (T)1; fc = (T)0; }
                    ws0 = wa * gh[0] + wb * gh[3] + wc * gh[6];
                    ws1 = wa * gh[1] + wb * gh[4] + wc * gh[7];
                    ws2 = wa * gh[2] + wb * gh[5] + wc * gh[8];
                    r0 = x0; r1 = x1; r2 = x2;
                    uint4 u = make_uint4(frac_to_u32(fa), frac_to_u32(fb), frac_to_u32(fc), 0u);
                    for (int r = 0; r < CL; ++r) {
                        unsigned char *pb = cluster.map_shared_rank(posn, r);
                        st_pos(pb, (unsigned)ai * 16u, zt, x0 - ws0, x1 - ws1, x2 - ws2, ty);
                        cluster.map_shared_rank(fr, r)[ai] = u;
                    }
                }
                if (tid == 0) {                       /* the far-away dummy neighbour (list padding), both buffers */
                    T far = (T)1e15;
                    st_pos(posb0, (unsigned)N_s * 16u, zt, far, far, far, 0);
                    st_pos(posb1, (unsigned)N_s * 16u, zt, far, far, far, 0);
                }
                cluster.sync();
                build_phase(rc, fr, rows, cnt, G, G[6], a_begin, A_own, N_s, misc);
                __syncthreads();
            }
            const bool last = n == n_steps;
            if (last) pair_phase<T, KIND, NT1, true>(rc, posn, rows, cnt, shtab, tab, fs, a_begin, A_own, NT, red);
            else pair_phase<T, KIND, NT1, false>(rc, posn, rows, cnt, shtab, tab, fs, a_begin, A_own, NT, red);
            __syncthreads();
            if (own) {
                f0 = fs[tid]; f1 = fs[rc.A + tid]; f2 = fs[2 * rc.A + tid];
                if (n > 0) { v0 = v0 + hdt * (f0 * im); v1 = v1 + hdt * (f1 * im); v2 = v2 + hdt * (f2 * im); }
            }
        }
        /* ---- store the system (R16): x, v at t + n dt, F(x), E, W, KE */
        double ke = 0.0;
        if (own) {
            T *x = (T *)d.pos + 3 * gi, *v = (T *)d.vel + 3 * gi, *f = (T *)d.force + 3 * gi;
            x[0] = x0; x[1] = x1; x[2] = x2; v[0] = v0; v[1] = v1; v[2] = v2; f[0] = f0; f[1] = f1; f[2] = f2;
            ke = 0.5 * (double)mass * d.mass_conv * ((double)v0 * (double)v0 + (double)v1 * (double)v1 + (double)v2 * (double)v2);
            if (!(fabs((double)f0) + fabs((double)f1) + fabs((double)f2) < 1e300)) atomicOr(&d.status->flags, TS_FLAG_NONFINITE);
        }
        const double tot = reduce8(cluster, CL, rank, ke, red, cred, rc.nwarps);
        if (rank == 0 && tid < 8) {
            if (tid == 0) d.energy[s] = tot;
            if (tid == 7) d.kinetic[s] = tot;
            if (tid >= 1 && tid <= 6 && (want & TS_WANT_VIRIAL)) {
                /* acc order: xx xy xz yy yz zz -> symmetric 3x3 */
                const int at[6][2] = { { 0, 0 }, { 1, 3 }, { 2, 6 }, { 4, 4 }, { 5, 7 }, { 8, 8 } };
                double *W = d.virial + 9 * (size_t)s;
                W[at[tid - 1][0]] = tot;
                W[at[tid - 1][1]] = tot;
            }
        }
        if (tid == 0) {
            if (misc->overflow) atomicOr(&d.status->flags, TS_FLAG_NBR_OVERFLOW);
            atomicAdd(&d.status->res_nnz, (unsigned long long)misc->nnz);
            if (rank == 0) {
                atomicAdd(&d.status->res_rebuilds, (unsigned long long)misc->rebuilds);
                d.sys_step[s] = step0 + (unsigned long long)n_steps;
            }
        }
        cluster.sync();                               /* nobody overwrites shared state a peer still reads */
    }
}

/* ------------------------------------------------------------------ host side */
struct ResPlan {
    bool checked, ok;
    ResCfg cfg;
};
static ResPlan *plan_of(ts_state *st) { return (ResPlan *)st->res_plan; }

typedef void (*ResKernel)(DevState, MdConst, ResCfg, int, unsigned);

template <typename T>
static ResKernel pick_kernel_t(int kind, bool nt1)
{
    if (kind == TS_LJ) return nt1 ? k_resident_md<T, TS_LJ, true> : k_resident_md<T, TS_LJ, false>;
    if (kind == TS_MORSE) return nt1 ? k_resident_md<T, TS_MORSE, true> : k_resident_md<T, TS_MORSE, false>;
    return nt1 ? k_resident_md<T, TS_SOFT_SPHERE, true> : k_resident_md<T, TS_SOFT_SPHERE, false>;
}
static ResKernel pick_kernel(const ts_state *st)
{
    bool nt1 = st->d.n_types == 1;
    return st->d.dtype == TS_F32 ? pick_kernel_t<float>(st->d.kind, nt1) : pick_kernel_t<double>(st->d.kind, nt1);
}

static unsigned up16(unsigned x) { return (x + 15u) & ~15u; }

/* Shared-memory carve for cluster size CL; returns false when it does not fit. */
static bool res_layout(ResCfg &c, int CL, int nmax, int need_row, int dtype, int n_types)
{
    size_t w = dtype == TS_F32 ? 4 : 8;
    int A = ((((nmax + CL - 1) / CL) + 3) / 4) * 4;
    const int max_threads = dtype == TS_F32 ? RES_MAX_THREADS : RES_MAX_THREADS_F64;
    if (A > max_threads) return false;
    int pitch = 32 * ((need_row - 16 + 31) / 32) + 16;
    if (pitch < 48) pitch = 48;
    int ntasks = A / 4, maxw = max_threads / 32;
    int passes = (ntasks + maxw - 1) / maxw;
    int nwarps = (ntasks + passes - 1) / passes;
    if (nwarps * 32 < A) nwarps = (A + 31) / 32;
    c.CL = CL; c.A = A; c.pitch = pitch; c.NP = nmax + 1; c.nwarps = nwarps;
    c.posbytes = up16((unsigned)(c.NP * 4 * w));
    unsigned o = 0;
    c.o_pos = o; o += 2 * c.posbytes;
    c.o_fr = o; o += up16((unsigned)c.NP * 16u);
    c.o_rows = o; o += up16((unsigned)A * (unsigned)pitch * 2u);
    c.o_fs = o; o += up16((unsigned)(3 * A * w));
    c.o_cnt = o; o += up16((unsigned)A * 4u);
    c.o_shtab = o; o += up16((unsigned)(27 * 4 * w));
    c.o_pot = o; o += up16((unsigned)(n_types * n_types * (dtype == TS_F32 ? sizeof(PotEntry<float>) : sizeof(PotEntry<double>))));
    c.o_red = o; o += (unsigned)(RES_MAX_THREADS / 32) * 64u;
    c.o_cred = o; o += 8u * 64u;
    c.o_misc = o; o += up16((unsigned)(sizeof(ResMisc) + 18 * w + 8 * sizeof(float)));
    c.smem = o;
    return o <= RES_SMEM_LIMIT;
}

/* Decides once per batch geometry whether the resident engine applies and how it is launched. */
bool resident_supported(ts_state *st)
{
    if (!st->res_plan) st->res_plan = calloc(1, sizeof(ResPlan));
    ResPlan *p = plan_of(st);
    if (p->checked) return p->ok;
    p->checked = true; p->ok = false;
    const DevState &d = st->d;
    int S = d.S;
    std::vector<SysGeom> geo((size_t)S);
    if (cudaMemcpy(geo.data(), d.geom, sizeof(SysGeom) * (size_t)S, cudaMemcpyDeviceToHost) != cudaSuccess) return false;
    const float eps_rel = 4e-6f;
    int nmax = 0;
    double need = 0.0;
    for (int s = 0; s < S; ++s) {
        int n = st->h_sysoff[s + 1] - st->h_sysoff[s];
        nmax = n > nmax ? n : nmax;
        const SysGeom &g = geo[(size_t)s];
        double lmax = 0.0;
        for (int a = 0; a < 3; ++a)
            lmax = fmax(lmax, sqrt(g.h[3 * a] * g.h[3 * a] + g.h[3 * a + 1] * g.h[3 * a + 1] + g.h[3 * a + 2] * g.h[3 * a + 2]));
        double rb = d.r_list + 2.0 * eps_rel * lmax;
        for (int k = 0; k < 3; ++k)
            if (!(g.hperp[k] >= 2.0 * rb)) return false;          /* more than one image within r_list possible */
        double nbar = (double)n / g.vol * (4.0 / 3.0) * M_PI * rb * rb * rb;
        need = fmax(need, nbar);
    }
    if (nmax > RES_MAX_ATOMS || d.n_types > TS_MAX_TYPES) return false;
    double slack = st->nbr.slack >= 1.0 ? st->nbr.slack : 1.25;
    int need_row = (int)ceil(need * slack) + 40;                   /* + padding of both segments to 16 */
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    ResCfg best; bool have = false;
    for (int CL = 1; CL <= 8; CL *= 2) {
        ResCfg c;
        memset(&c, 0, sizeof c);
        if (!res_layout(c, CL, nmax, need_row, d.dtype, d.n_types)) continue;
        best = c; have = true;
        if ((long long)S * CL >= (nsm * 3) / 4 || c.A <= 64) break;   /* enough CTAs to occupy the chip */
    }
    if (!have) return false;
    best.eps_rel = eps_rel;
    ResKernel k = pick_kernel(st);
    if (cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)best.smem) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)best.CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.gridDim = dim3((unsigned)(best.CL * S)); lc.blockDim = dim3((unsigned)(best.nwarps * 32));
    lc.dynamicSmemBytes = best.smem; lc.attrs = at; lc.numAttrs = 1;
    int maxc = 0;
    if (cudaOccupancyMaxActiveClusters(&maxc, (const void *)k, &lc) != cudaSuccess || maxc < 1) {
        cudaGetLastError();
        return false;
    }
    best.n_clusters = S < maxc ? S : maxc;
    p->cfg = best;
    p->ok = true;
    return true;
}

void resident_invalidate(ts_state *st)
{
    if (st->res_plan) plan_of(st)->checked = false;
}

void resident_free(ts_state *st)
{
    free(st->res_plan);
    st->res_plan = nullptr;
}

ts_status resident_md(ts_state *st, const MdConst &c, int n_steps, unsigned want, cudaStream_t q)
{
    if (!resident_supported(st)) return TS_ERR_UNSUPPORTED;
    const ResCfg &cfg = plan_of(st)->cfg;
    ResKernel k = pick_kernel(st);
    TS_CUDA_OK(st, cudaMemsetAsync(&st->d.status->res_nnz, 0, sizeof(unsigned long long), q));
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)cfg.CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.gridDim = dim3((unsigned)(cfg.CL * cfg.n_clusters)); lc.blockDim = dim3((unsigned)(cfg.nwarps * 32));
    lc.dynamicSmemBytes = cfg.smem; lc.stream = q; lc.attrs = at; lc.numAttrs = 1;
    TS_CUDA_OK(st, cudaLaunchKernelEx(&lc, k, st->d, c, cfg, n_steps, want));
    st->launches += 1;
    st->last_engine = 1;
    st->list_built = false;          /* the general engine's list no longer matches the positions */
    return TS_OK;
}
