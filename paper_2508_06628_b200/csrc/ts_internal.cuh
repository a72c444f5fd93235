/*
 * ts_internal.cuh -- structures shared by the translation units of libts (CUDA path only; the
 * oracle under oracle/ shares nothing with this tree).
 *
 * Data layout in HBM:
 *   boundary arrays (caller-owned): pos/vel/force [N,3], mass [N], type [N], system_idx [N],
 *                                   cell [S,3,3], energy [S], virial [S,9], kinetic [S]
 *   workspace (caller-owned blob, carved by ts_layout):
 *     per system : sysoff, SysGeom (fp64 cell, inverse, heights, bin grid, stencil half-widths),
 *                  hT (cell in the state dtype), nbr_base / nbr_len (CSR segment of the system),
 *                  FIRE scalars, step counter
 *     per atom   : pos4 (x~,y~,z~,type) gather array, spos (bin-sorted wrapped fp64 coordinates +
 *                  local index), xref (positions at the last build), cell id / rank / wrap,
 *                  nbr_cnt, nbr_off
 *     per pair   : packed uint32 neighbour entry = local j (17 bits) | 3 x 5-bit biased shift
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "ts.h"

#define TS_MAX_TYPES 8
#define TS_J_BITS 17
#define TS_J_MASK 0x1FFFFu
#define TS_MAX_SYS_ATOMS (1 << TS_J_BITS)

struct SysGeom {
    double h[9];      /* rows = lattice vectors                         */
    double hinv[9];   /* f_k = sum_b x_b hinv[3b+k]                      */
    double hperp[3];  /* distance between lattice planes k               */
    double vol;
    int nb[3];        /* bins per axis                                   */
    int D[3];         /* stencil half-width in bins (R8)                 */
    int ncell;
    int bad;
};

template <typename T>
struct PotEntry {
    T p0, p1, p2, rc2, vshift;
    T c0, c1, c2;     /* precomputed: LJ 4 eps s^12, 4 eps s^6 ; Morse 2 D alpha ; soft eps/alpha, eps/sigma, 1/sigma */
};

struct DevStatus {
    unsigned int flags;         /* TS_FLAG_* sticky                                  */
    unsigned int need_rebuild;  /* set by the skin check, cleared after a build      */
    unsigned int n_rebuilds;
    unsigned int max_nbr;
    unsigned long long nnz;
    unsigned int list_valid;
    unsigned int pad;
    unsigned long long res_nnz[2];    /* resident engine: pairs in the lists at the end of the last call; two slots used in
                                       * turn: a call adds into one and clears the other for the next call (no memset launch) */
    unsigned long long res_rebuilds;  /* per-system list builds, summed over systems (both engines)      */
};

/* Everything a kernel needs, passed by value (well under the 4 KB parameter limit). */
struct DevState {
    long long N;
    int S;
    int dtype;
    int kind, n_types, shift_energy;
    double mass_conv, kB;
    double r_list, r_list2, half_skin2;
    /* boundary */
    void *pos, *vel, *force;
    const void *mass;
    const int *type;
    const int *sysidx;
    const void *cell;
    double *energy, *virial, *kinetic;
    const unsigned int *uid;
    /* workspace: per system */
    int *sysoff;                 /* [S+1]                              */
    SysGeom *geom;               /* [S]                                */
    void *hT;                    /* [S,9] cell in state dtype          */
    long long *nbr_base;         /* [S+1] first pair slot of a system  */
    long long *nbr_len;          /* [S]  pairs in use, -1 = overflow   */
    double *f_dt, *f_alpha;      /* [S] FIRE                           */
    int *f_npos, *f_nsteps, *f_status;
    double *f_acc;               /* [S,4] fmax2, P, vv, ff             */
    int *sys_active;             /* [S] 1 = atoms of the system move   */
    int *sys_rebuild;            /* [S] 1 = an atom of the system moved > skin/2: its list is rebuilt at the next build (R12) */
    unsigned long long *sys_step;/* [S] per-system step counter (R18)  */
    unsigned int *uid_own;       /* [S] persistent ids (copy or iota)  */
    int *sys_engine;             /* [S] 1 = stepped by the system-resident engine (mixed dispatch of a ragged batch) */
    int *res_list;               /* [S] the resident engine's systems, size class after size class */
    int *res_saved;              /* [S] 1 = the resident engine's list of the system (rows, task words, image table, x_ref / wrap)
                                  * lies in the system's own segment of `nbr` and matches its stored positions */
    double *red_slots;           /* [(N / 4 + S + 2)][8] partial sums of the general engine's per-system reductions (ts_sys_store) */
    int mixed;                   /* 1: this launch sequence of the general engine skips the systems with sys_engine = 1 */
    /* workspace: per atom */
    void *pos4;                  /* [N] float4 / double4 (x~,y~,z~,type) */
    double4 *spos;               /* [N] sorted wrapped coords + local idx */
    void *xref;                  /* [N,3] state dtype                  */
    int *cell_count, *cell_start;/* [N+S+1]                            */
    int *atom_cell, *atom_rank, *atom_wrap; /* [N]                     */
    int *nbr_cnt;                /* [N]                                */
    long long *nbr_off;          /* [N]                                */
    /* workspace: per pair */
    unsigned int *nbr;           /* [cap]                              */
    long long nbr_cap;
    void *pot;                   /* PotEntry<T> [n_types^2]            */
    DevStatus *status;
    int *scratch;                /* small upload area (swap lists)     */
};

struct ts_state {
    DevState d;
    ts_state_desc desc;
    ts_nbr_params nbr;
    int *h_sysoff;               /* host copy [S+1]                    */
    long long N_cap;             /* atoms / systems the state was created with: the capacity ts_repack_systems fills */
    int S_cap;
    bool list_built;             /* a build has been enqueued and no swap since */
    bool forces_current;
    int res_nnz_slot;            /* slot of DevStatus.res_nnz the last resident launch added into */
    bool res_saved_ok;           /* nothing has happened since the last resident launch that invalidates res_saved for the
                                  * whole batch (a general-engine build, positions written from outside, a new plan) */
    bool list_mixed;             /* the general engine's list covers only the systems the resident engine does not step */
    int engine;
    int last_engine;             /* engine that ran the last stepping call */
    void *res_plan;              /* resident engine launch plan (ts_resident.cu) */
    long long launches;
    long long steps_done;
    unsigned int seen_flags;     /* last flags seen by ts_poll         */
    char err[256];
};

/* ------------------------------------------------------------------ workspace carving */
struct TsLayout {
    size_t total;
    size_t sysoff, geom, hT, nbr_base, nbr_len, f_dt, f_alpha, f_npos, f_nsteps, f_status, f_acc,
        sys_active, sys_rebuild, sys_step, uid_own, sys_engine, res_list, res_saved, red_slots, pos4, spos, xref, cell_count, cell_start, atom_cell,
        atom_rank, atom_wrap, nbr_cnt, nbr_off, nbr, pot, status, scratch;
};
TsLayout ts_layout(long long N, int S, long long nbr_cap, int dtype, int n_types);

/* ------------------------------------------------------------------ launchers (host) */
#define TS_CUDA_OK(st, call)                                                              \
    do {                                                                                  \
        cudaError_t e__ = (call);                                                         \
        if (e__ != cudaSuccess) {                                                         \
            ts_set_error((st), "CUDA error %s at %s:%d", cudaGetErrorString(e__), __FILE__, __LINE__); \
            return TS_ERR_CUDA;                                                           \
        }                                                                                 \
    } while (0)
void ts_set_error(ts_state *st, const char *fmt, ...);

/* ts_api.cu */
long long ts_system_pair_capacity(long long n, double vol, double r_list, double slack);
/* ts_step.cu: the general engine is about to work on the WHOLE batch: a list built for a mixed dispatch is stale */
void ts_whole_batch_mode(ts_state *st);
/* ts_build.cu */
void launch_geometry(ts_state *st, int s_first, int s_count, const int *slots, cudaStream_t q);
void launch_build(ts_state *st, bool force, cudaStream_t q);
/* ts_pair.cu */
void launch_pair(ts_state *st, unsigned want, bool masked, cudaStream_t q);
/* ts_integrate.cu */
struct MdConst { int integrator; double dt, hdt, c1, c2, kT; unsigned int key0, key1; };
void launch_import(ts_state *st, cudaStream_t q);   /* pos -> pos4 + skin check */
void launch_md_pre(ts_state *st, const MdConst &c, cudaStream_t q);
void launch_md_post(ts_state *st, const MdConst &c, bool want_ke, cudaStream_t q);
void launch_kinetic(ts_state *st, cudaStream_t q);
void launch_fire_init(ts_state *st, const ts_fire_params &p, cudaStream_t q);
void launch_fire_check0(ts_state *st, const ts_fire_params &p, cudaStream_t q);
void launch_fire_pre(ts_state *st, const ts_fire_params &p, cudaStream_t q);
void launch_fire_post(ts_state *st, const ts_fire_params &p, cudaStream_t q);
void launch_fire_count(ts_state *st, cudaStream_t q);
void launch_swap(ts_state *st, int n, const ts_state_desc *fresh, cudaStream_t q);
/* ts_resident.cu */
bool resident_supported(ts_state *st);
int resident_general_count(ts_state *st);
cudaStream_t resident_fork_general(ts_state *st, cudaStream_t q);
void resident_join_general(ts_state *st, cudaStream_t q);
void resident_invalidate(ts_state *st);
void resident_after_swap(ts_state *st, const int32_t *slots, int n, const void *cells_host);
void resident_free(ts_state *st);
ts_status resident_md(ts_state *st, const MdConst &c, int n_steps, unsigned want, cudaStream_t q);
ts_status resident_fire(ts_state *st, const ts_fire_params &fp, int n_steps, cudaStream_t q);

/* ------------------------------------------------------------------ device helpers */
template <typename T> struct Vec4;
template <> struct Vec4<float> { typedef float4 type; };
template <> struct Vec4<double> { typedef double4 type; };

__device__ __forceinline__ int ts_cell_base(const int *sysoff, int s) { return sysoff[s] + s; }
/* mixed dispatch: the system belongs to the resident engine, the general engine's kernels leave it alone */
__device__ __forceinline__ bool ts_skip(const DevState &d, int s) { return d.mixed && d.sys_engine[s]; }

/* Per-system sums of the general engine, bitwise reproducible from run to run (fp64 atomics would add in arrival order),
 * in two kernels and without fences.  The producing kernel's threads cover the atoms in order, LANES lanes per atom, so
 * the warps that hold atoms of system s are w_first(s) .. w_last(s).  ts_sys_store: every warp reduces the lanes of each
 * system it holds in a fixed tree and stores the partial in slot (warp + s) of red_slots -- a warp that straddles k
 * systems writes k slots, and warp + s is unique and increasing.  ts_sys_total (a kernel launched after the producer, one
 * warp per system): the lanes stride the slots of the system in slot order, then a fixed tree.  key: system of the lane's
 * atom, -1 for lanes that contribute nothing (all atoms of a system contribute or none do); every lane of the warp calls. */
template <int NQ, int LANES>
__device__ __forceinline__ void ts_sys_store(const DevState &d, int key, const double (&acc)[NQ])
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const long long warp = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    unsigned remaining = __ballot_sync(FULL, key >= 0);
    while (remaining) {
        const int sl = __shfl_sync(FULL, key, __ffs(remaining) - 1);
        const bool mine = key == sl;
        double v[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            v[q] = mine ? acc[q] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(FULL, v[q], o);
        }
        if (lane == 0) {
            double *slot = d.red_slots + 8 * (size_t)(warp + sl);
#pragma unroll
            for (int q = 0; q < NQ; ++q) slot[q] = v[q];
        }
        remaining &= ~__ballot_sync(FULL, mine);
    }
}

/* totals of system s from the slots a kernel with `lanes` lanes per atom stored; the result is in every lane */
template <int NQ>
__device__ __forceinline__ void ts_sys_total(const DevState &d, int s, int lanes, double (&tot)[NQ])
{
    const int lane = threadIdx.x & 31;
    const long long w_first = ((long long)d.sysoff[s] * lanes) >> 5, w_last = ((long long)d.sysoff[s + 1] * lanes - 1) >> 5;
    const int n = (int)(w_last - w_first + 1);
    const double *base = d.red_slots + 8 * (size_t)(w_first + s);
#pragma unroll
    for (int q = 0; q < NQ; ++q) tot[q] = 0.0;
    for (int k = lane; k < n; k += 32)
#pragma unroll
        for (int q = 0; q < NQ; ++q) tot[q] += base[8 * (size_t)k + q];
#pragma unroll
    for (int q = 0; q < NQ; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot[q] += __shfl_xor_sync(0xffffffffu, tot[q], o);
}

__device__ __forceinline__ unsigned int ts_pack_nbr(int j, int s0, int s1, int s2)
{
    return (unsigned)j | ((unsigned)(s0 + 16) << 17) | ((unsigned)(s1 + 16) << 22) | ((unsigned)(s2 + 16) << 27);
}
__device__ __forceinline__ void ts_unpack_shift(unsigned int e, int &s0, int &s1, int &s2)
{
    s0 = (int)((e >> 17) & 31u) - 16;
    s1 = (int)((e >> 22) & 31u) - 16;
    s2 = (int)(e >> 27) - 16;
}
__device__ __forceinline__ int ts_pack_wrap(int w0, int w1, int w2)
{
    return (w0 & 0xff) | ((w1 & 0xff) << 8) | ((w2 & 0xff) << 16);
}
__device__ __forceinline__ void ts_unpack_wrap(int p, int &w0, int &w1, int &w2)
{
    w0 = (int)(signed char)(p & 0xff);
    w1 = (int)(signed char)((p >> 8) & 0xff);
    w2 = (int)(signed char)((p >> 16) & 0xff);
}
