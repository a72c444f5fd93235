/*
 * ts_resident.cu -- system-resident MD and FIRE engine (SURVEY.md section 7 "hard part 1", kernel K13).
 *
 * The graded batch (BASELINE.json:configs[1], 64 x 864 atoms) is so small that a step is bound by
 * launch latency and on-chip bandwidth, not by HBM.  This engine therefore keeps a whole system on
 * chip for all n_steps of a ts_md_step / ts_fire_step call: one thread-block cluster of CL CTAs per
 * system, each CTA owning a contiguous slice of the system's atoms.  Per CTA, in shared memory:
 *     pos[NS]        position slots (16 B: wrapped x, y, z + type; fp64: two planes).  HOME slots of
 *                    ALL atoms of the system (a hashed permutation of the atom order, hslot), eight
 *                    far-away dummies (list padding, one per 16-byte bank group) and the GHOST
 *                    slots: every periodic image of an atom that can lie within r_list of the cell
 *                    owns a slot holding x + S.h, in the bank group of its atom.  An owner writes the
 *                    home slot and the images of its atom locally and sends the home slot to the
 *                    other CTAs of the cluster through DSMEM; every CTA regenerates the images of
 *                    the other CTAs' atoms locally each step (peer_pass).
 *     fr[N_s]        fractional coordinates as 32-bit fixed point (rebuilds only; aliased onto the
 *                    ghost slots, which are dead between the cluster barrier of a rebuild and the
 *                    ghost refresh that ends it)
 *     gtab[N_s]      first ghost slot, active axes and image signs of every atom
 *     rows           the Verlet list of the CTA's own atoms: 14-bit entries = slot number of the
 *                    neighbour, in trips of 16 entries per atom (see "list layout").  Thanks to the
 *                    ghosts EVERY pair is a plain difference of two slots: no image arithmetic in the
 *                    pair loop.  One COLUMN per bank group (build_phase).
 *     fs[3][A]       forces of the own atoms (pair phase -> integrator phase)
 *     own state      fp32: x (unwrapped) | 1/m, v, x_ref | wrap shift of the own atoms as three
 *                    4-vectors per atom (the 72 registers of a thread belong to the pair loop);
 *                    fp64: the same in registers of the owner thread
 * HBM is touched when a system is loaded, when it is stored, and never in between.
 *
 * One MD step = [owner: B A (O A) + skin test; spare threads draw the Langevin kicks of the next
 * step] -> wait(peers done reading; split-phase cluster barrier, no fence) -> [home slots to the
 * other CTAs with st.async: they complete transaction bytes on the receiving CTA's mbarrier, the
 * skin flag rides in the slot's type word; own home slot and images locally] -> wait on the own
 * mbarrier -> [images of the others' atoms] -> [rebuild if any atom moved > skin/2, then all images
 * again] -> [pair phase] -> arrive(done reading) -> block barrier -> [owner: B].  FIRE mode
 * (template flag): per-system dt, the four reductions and the state machine after every step,
 * finished systems skipped untouched.  Same physics as the general engine (SURVEY O2..O6, R5, R9,
 * R12, R16, R18, R21, R22).
 *
 * Pair phase: tasks of eight atoms per warp, four lanes per atom; the two atoms of a quarter-warp
 * gather from eight different 16-byte bank groups in every step ("list layout").  The builder's
 * lane l tests the slots = l mod 8, so its hits all live in bank group l and fill column l of the
 * atom's list: a gather is served by one shared-memory wavefront per quarter-warp unless a group
 * overflowed its column.  The fp32 Lennard-Jones force-only loop uses Blackwell's packed
 * FFMA2/FMUL2 (f32x2) on pairs of entries and gathers two entries ahead of the arithmetic.
 *
 * Rebuild: brute force over the system in fractional fixed point (integer subtraction wraps = the
 * minimum image), valid because the engine is only used when every cell height is >= 2 r_list
 * (then an image within r_list is the rounded one and is unique).  The list radius is inflated by
 * a few float ulps of the box; a Verlet list only has to be a superset of the pairs within r_c.
 */
#include <cooperative_groups.h>
#include <math.h>
#include <string.h>
#include <stdio.h>
#include <stdlib.h>

#include <vector>

#include "ts_internal.cuh"
#include "ts_pot.cuh"
#include "ts_rng.cuh"

namespace cg = cooperative_groups;

#define RES_MAX_THREADS 896         /* fp32; the fp64 kernels need twice the registers: 512 */
#define RES_MAX_THREADS_F64 512
#define RES_MAX_ATOMS 2048          /* builder hit masks cover 8 x 256 candidates */
#define RES_MAX_SLOTS 16376         /* list entries are 16-bit slot numbers; shared memory is the real limit */
#define RES_SMEM_LIMIT (227 * 1024)

struct ResCfg {
    int CL;            /* CTAs per system = cluster size                       */
    int A;             /* atoms per CTA, capacity (multiple of 4)              */
    int pitch;         /* u16 entries per list row, a multiple of 32           */
    int NS;            /* position slots per CTA: atoms + dummies + ghosts     */
    int nwarps;
    int n_clusters;
    unsigned o_pos, o_fr, o_gtab, o_rows, o_fs, o_own, o_meta, o_noise, o_pot, o_red, o_cred, o_misc, o_fire, o_mbar;
    unsigned smem;
    int nnz_slot;      /* slot of DevStatus.res_nnz this launch adds into (the other one is cleared for the next launch) */
    int noise_helpers; /* the kick buffers of the noise helpers exist (they are left out when they do not fit) */
    float eps_rel;     /* list radius inflation, relative to the longest cell vector */
    const int *syslist; /* device: the systems this launch steps (one size class of the batch); NULL = 0 .. n_list - 1 */
    int n_list;
    int dump_sys;      /* list export (ts_get_resident_neighbors): the one system whose list is dumped, -1 = normal run */
    unsigned char *dump;  /* device: per CTA rank [rows | tmeta | gtab | wrap shift of the own atoms] */
    unsigned dump_cta_bytes;
};

struct ResMisc {
    int unused[2];
    unsigned nnz;
    unsigned rebuilds;
    int overflow;
    int pad[3];        /* 32 bytes: the cell copy follows */
};

/* optional phase timers (build with -DTS_RES_TIMING; debugging only): cycles of warp 0 of every CTA */
#ifdef TS_RES_TIMING
__device__ unsigned long long g_res_prof[16];
__device__ unsigned long long g_res_wprof[64];   /* [0..31] pair-phase cycles per warp, [32..63] trips per warp */
#define TICK(k) do { if (threadIdx.x == 0) { long long t__ = clock64(); prof_acc[k] += t__ - prof_t; prof_t = t__; } } while (0)
#else
#define TICK(k) do { } while (0)
#endif

/* "this CTA has finished READING the positions of the step": nothing was written, so no release fence is needed
 * (the loads completed before their values were consumed); the matching wait still acquires */
__device__ __forceinline__ void cl_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

/* ------------------------------------------------------------------ mbarrier for the per-step position exchange
 * Every CTA owns one FULL mbarrier.  The owners of the cluster send the home slots with st.async, which completes
 * transaction bytes on the RECEIVING CTA's barrier; a CTA waits on its own barrier only: no cluster-wide barrier
 * with a GPU-scope release fence (MEMBAR.ALL.GPU + CCTL.IVALL) on the critical path of a step.  The write-after-
 * read side (peers have finished reading the old slots) stays on the split-phase cluster barrier, whose arrive
 * needs no fence. */
__device__ __forceinline__ void mb_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mb_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mb_wait(unsigned bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ unsigned map_cluster(unsigned saddr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_async_pos(unsigned dst, unsigned bar, unsigned, float x, float y, float z, int ty)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];"
                 :: "r"(dst), "f"(x), "f"(y), "f"(z), "f"(__int_as_float(ty)), "r"(bar) : "memory");
}
__device__ __forceinline__ void st_async_pos(unsigned dst, unsigned bar, unsigned zt, double x, double y, double z, int ty)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 :: "r"(dst), "d"(x), "d"(y), "r"(bar) : "memory");
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 :: "r"(dst + zt), "d"(z), "d"(__longlong_as_double((long long)ty)), "r"(bar) : "memory");
}
#define MOVED_BIT 0x40000000              /* in the type word of a home slot: its atom moved more than skin / 2 */

/* ------------------------------------------------------------------ position slots */
template <typename T> struct P3 { T x, y, z; int ty; };
template <typename T> struct __align__(16) Q4 { T a, b, c, d; };
__device__ __forceinline__ float bits_to(int v, float) { return __int_as_float(v); }
__device__ __forceinline__ double bits_to(int v, double) { return __longlong_as_double((long long)v); }
__device__ __forceinline__ int bits_from(float v) { return __float_as_int(v); }
__device__ __forceinline__ int bits_from(double v) { return (int)__double_as_longlong(v); }

__device__ __forceinline__ P3<float> ld_pos(const unsigned char *base, unsigned off, unsigned, float)
{
    float4 v = *(const float4 *)(base + off);
    P3<float> p; p.x = v.x; p.y = v.y; p.z = v.z; p.ty = __float_as_int(v.w) & 0xff;        /* bit 30: MOVED_BIT */
    return p;
}
__device__ __forceinline__ P3<double> ld_pos(const unsigned char *base, unsigned off, unsigned zt, double)
{
    double2 a = *(const double2 *)(base + off);
    double2 b = *(const double2 *)(base + zt + off);
    P3<double> p; p.x = a.x; p.y = a.y; p.z = b.x; p.ty = (int)__double_as_longlong(b.y) & 0xff;
    return p;
}
__device__ __forceinline__ int ld_tyword(const unsigned char *base, unsigned off, unsigned, float) { return *(const int *)(base + off + 12u); }
__device__ __forceinline__ int ld_tyword(const unsigned char *base, unsigned off, unsigned zt, double) { return *(const int *)(base + zt + off + 8u); }
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

/* Home slot of atom j.  The bank group of a slot is slot mod 8; atoms that follow each other in a
 * regular pattern (a lattice written cell by cell) would load the groups of a neighbour list very
 * unevenly, so every block of eight atoms is rotated by a hash of the block number.  The last block
 * is not rotated: the unused slots stay the ones >= N_s.  Everything built from the positions (fr,
 * gtab, the rows) lives in SLOT space; only the owner of an atom knows its index. */
__device__ __forceinline__ int hslot(int j, int N8)
{
    const unsigned b = (unsigned)j >> 3;
    const unsigned h = (int)b == (N8 >> 3) - 1 ? 0u : (b * 0x9E3779B1u) >> 29;
    return (j & ~7) | (int)(((unsigned)j + h) & 7u);
}

/* ------------------------------------------------------------------ ghosts
 * gtab entry of an atom: first ghost slot (16 bits) | active axes (3 bits) << 16 | image signs
 * (bit = 1: the image sits at +h_k) << 19.  The images of an atom are the non-empty subsets m of
 * its active axes, in increasing m; image number r lives in slot base + 8 r (same bank group as
 * the atom).  Owners publish only the HOME slot of their atom through DSMEM; every CTA then
 * regenerates all ghost slots locally from its home slots (ghost_pass, one thread per atom): DSMEM
 * carries 16 bytes per atom and peer instead of 16 bytes per image.                               */

/* the owner writes the home slot of its atom into every CTA of the cluster */
template <typename T>
__device__ __forceinline__ void publish_home(cg::cluster_group &cluster, int CL, unsigned char *posb, unsigned zt, int ai,
                                             T px, T py, T pz, int ty)
{
    for (int r = 0; r < CL; ++r) st_pos(cluster.map_shared_rank(posb, r), (unsigned)ai * 16u, zt, px, py, pz, ty);
}

/* the images of one atom: gtab entry e, home position (px, py, pz); image number r lives in slot base + 8 r */
template <typename T>
__device__ __forceinline__ void ghost_write(unsigned char *posb, unsigned zt, unsigned e, const T *gh, T px, T py, T pz, int ty)
{
    const unsigned act = (e >> 16) & 7u;
    if (act == 0u) return;
    T a[3][3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const T sgn = ((e >> (19 + k)) & 1u) ? (T)1 : (T)-1;
#pragma unroll
        for (int b = 0; b < 3; ++b) a[k][b] = sgn * gh[3 * k + b];
    }
    /* q[m] = p + sum_{k in m} a_k, built incrementally: q[m] = q[m without its top axis] + a_top */
    T q[8][3] = { { px, py, pz } };
    unsigned off = (e & 0xffffu) * 16u;
#pragma unroll
    for (int m = 1; m < 8; ++m) {
        const int top = m >= 4 ? 2 : (m >= 2 ? 1 : 0);
        const int rest = m & ~(1 << top);
#pragma unroll
        for (int b = 0; b < 3; ++b) q[m][b] = q[rest][b] + a[top][b];
        if ((m & ~act) == 0u) {
            st_pos(posb, off, zt, q[m][0], q[m][1], q[m][2], ty);
            off += 128u;
        }
    }
}

/* every CTA refreshes the images of every atom of the system from the home slots (after a rebuild) */
template <typename T>
__device__ __forceinline__ void ghost_pass(unsigned char *posb, unsigned zt, const unsigned *gtab, const T *gh, int N_s)
{
    for (int j = threadIdx.x; j < N_s; j += (int)blockDim.x) {
        const unsigned e = gtab[j];
        if (((e >> 16) & 7u) == 0u) continue;
        const P3<T> p = ld_pos(posb, (unsigned)j * 16u, zt, (T)0);
        ghost_write<T>(posb, zt, e, gh, p.x, p.y, p.z, p.ty);
    }
}

/* the new home positions of the other CTAs' atoms have arrived in the slot array (st.async): refresh their images and
 * collect the owners' skin flags (R12), which travel in the type word.  [sb0, sb0 + sbw) are the CTA's own slots. */
template <typename T>
__device__ __forceinline__ bool peer_pass(unsigned char *posb, unsigned zt, const unsigned *gtab, const T *gh, int sb0, int sbw,
                                          int n_peer_slots, int N_s)
{
    bool moved = false;
    for (int k = threadIdx.x; k < n_peer_slots; k += (int)blockDim.x) {
        const int hs = k < sb0 ? k : k + sbw;
        if (hs >= N_s) continue;                 /* the unused slots of the last block */
        moved |= (ld_tyword(posb, (unsigned)hs * 16u, zt, (T)0) & MOVED_BIT) != 0;
        const unsigned e = gtab[hs];
        if (((e >> 16) & 7u) == 0u) continue;
        const P3<T> p = ld_pos(posb, (unsigned)hs * 16u, zt, (T)0);
        ghost_write<T>(posb, zt, e, gh, p.x, p.y, p.z, p.ty);
    }
    return moved;
}

/* ------------------------------------------------------------------ one pair (generic path) */
template <typename T, int KIND, bool NT1, bool EV>
__device__ __forceinline__ void pair_accum(const P3<T> &xi, const P3<T> &xj, const PotEntry<T> &pe1, const PotEntry<T> *tab,
                                           int tirow, T &fx, T &fy, T &fz, T *ev)
{
    T rx = xj.x - xi.x, ry = xj.y - xi.y, rz = xj.z - xi.z;
    T r2 = rx * rx + ry * ry + rz * rz;
    PotEntry<T> pe = pe1;
    if (!NT1) pe = tab[tirow + xj.ty];
    const bool in = r2 < pe.rc2;                 /* strict (R9); the padding dummies sit at 1e15 */
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

/* ------------------------------------------------------------------ packed fp32 helpers (FFMA2 / FMUL2) */
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

/* ------------------------------------------------------------------ shared-space addressing
 * Addresses are shared-window addresses of THIS CTA (cvta: they carry the CTA's rank inside its cluster in bits 24+;
 * an address without it is illegal on every CTA but rank 0).  The loads are volatile so that the gathers of the next
 * trip stay ahead of the arithmetic of the current one. */
extern __shared__ __align__(16) unsigned char ts_smem[];
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float4 lds128(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds64(unsigned a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ unsigned lds32(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
/* position slot at shared-space address a (fp64: second plane zt bytes further) */
__device__ __forceinline__ P3<float> ld_pos_sa(unsigned a, unsigned, float)
{
    const float4 v = lds128(a);
    P3<float> p; p.x = v.x; p.y = v.y; p.z = v.z; p.ty = __float_as_int(v.w) & 0xff;
    return p;
}
__device__ __forceinline__ P3<double> ld_pos_sa(unsigned a, unsigned zt, double)
{
    double2 u, w;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(u.x), "=d"(u.y) : "r"(a));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(w.x), "=d"(w.y) : "r"(a + zt));
    P3<double> p; p.x = u.x; p.y = u.y; p.z = w.x; p.ty = (int)__double_as_longlong(w.y) & 0xff;
    return p;
}

/* one packed step of the fp32 Lennard-Jones force loop: the two pairs (xi, pa) and (xi, pb) */
__device__ __forceinline__ void lj_pair2(const float4 &pa, const float4 &pb, float xix, float xiy, float xiz, float rc2,
                                         f32x2 C12, f32x2 C6, f32x2 &FX, f32x2 &FY, f32x2 &FZ)
{
    const f32x2 RX = pk2(pa.x - xix, pb.x - xix), RY = pk2(pa.y - xiy, pb.y - xiy), RZ = pk2(pa.z - xiz, pb.z - xiz);
    f32x2 R2 = mul2(RX, RX);
    R2 = fma2(RY, RY, R2);
    R2 = fma2(RZ, RZ, R2);
    float r2a, r2b;
    upk2(R2, r2a, r2b);
    float ia, ib;
    /* volatile: keeps the arithmetic of a pair behind the (volatile) gathers issued before it in program order, so
     * that the gathers of the next two entries are in flight while this pair is computed */
    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(ia) : "f"(r2a));
    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(ib) : "f"(r2b));
    const float ma = r2a < rc2 ? 1.0f : 0.0f, mb = r2b < rc2 ? 1.0f : 0.0f;   /* strict (R9) */
    const f32x2 I = mul2(pk2(ia, ib), pk2(ma, mb));
    const f32x2 I2 = mul2(I, I);
    const f32x2 I6 = mul2(I2, I);
    const f32x2 P = fma2(I6, C12, C6);
    const f32x2 G = mul2(mul2(I6, I), P);              /* g = V'(r)/r = ir2 ir6 (6 c1 - 12 c0 ir6) */
    FX = fma2(G, RX, FX);
    FY = fma2(G, RY, FY);
    FZ = fma2(G, RZ, FZ);
}

/* the same for the fp32 Morse force loop: g = V'(r)/r = 2 D alpha (1 - e) e / r, e = exp(-alpha (r - r0)) as one ex2
 * (NA = -alpha log2 e, AR = alpha r0 log2 e), 1 / r as one rsqrt */
__device__ __forceinline__ void morse_pair2(const float4 &pa, const float4 &pb, float xix, float xiy, float xiz, float rc2,
                                            f32x2 NA, f32x2 AR, f32x2 C0, f32x2 &FX, f32x2 &FY, f32x2 &FZ)
{
    const f32x2 RX = pk2(pa.x - xix, pb.x - xix), RY = pk2(pa.y - xiy, pb.y - xiy), RZ = pk2(pa.z - xiz, pb.z - xiz);
    f32x2 R2 = mul2(RX, RX);
    R2 = fma2(RY, RY, R2);
    R2 = fma2(RZ, RZ, R2);
    float r2a, r2b;
    upk2(R2, r2a, r2b);
    float ia, ib;
    asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(ia) : "f"(r2a));      /* volatile: see lj_pair2 */
    asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(ib) : "f"(r2b));
    const float ma = r2a < rc2 ? 1.0f : 0.0f, mb = r2b < rc2 ? 1.0f : 0.0f;   /* strict (R9) */
    const f32x2 IR = pk2(ia, ib);
    const f32x2 X = fma2(mul2(R2, IR), NA, AR);        /* -alpha (r - r0) log2 e */
    float xa, xb, ea, eb;
    upk2(X, xa, xb);
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ea) : "f"(xa));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(eb) : "f"(xb));
    const f32x2 E = pk2(ea, eb);
    const f32x2 OM = fma2(E, pk2(-1.0f, -1.0f), pk2(1.0f, 1.0f));
    const f32x2 G = mul2(mul2(mul2(C0, pk2(ma, mb)), OM), mul2(E, IR));
    FX = fma2(G, RX, FX);
    FY = fma2(G, RY, FY);
    FZ = fma2(G, RZ, FZ);
}

/* one packed step of the fast loops: KIND selects the potential; A, B, C are its three packed constants */
template <int KIND>
__device__ __forceinline__ void fast_pair2(const float4 &pa, const float4 &pb, float xix, float xiy, float xiz, float rc2,
                                           f32x2 A, f32x2 B, f32x2 C, f32x2 &FX, f32x2 &FY, f32x2 &FZ)
{
    if (KIND == TS_LJ) lj_pair2(pa, pb, xix, xiy, xiz, rc2, A, B, FX, FY, FZ);
    else morse_pair2(pa, pb, xix, xiy, xiz, rc2, A, B, C, FX, FY, FZ);
}

/* ------------------------------------------------------------------ list layout
 * A TASK is eight consecutive own atoms, served by one warp: four lanes per atom (lane = 4 a + l4, a = atom of the
 * task, l4 = lane of the atom).  The list of an atom has eight COLUMNS, one per 16-byte bank group of the slot array
 * (column c holds neighbours whose slot number is c modulo 8), and R rows; lane l4 reads the columns l4 and l4 + 4.
 * The list of a task is a sequence of TRIPS of 256 bytes: lane (a, l4) owns the 64-bit word at a * 32 + l4 * 8, which
 * holds four entries, gathered in the order k = 0..3:
 *     k = 0: row 2 t,     column l4 + 4 p        k = 1: row 2 t,     column l4 + 4 (1 - p)
 *     k = 2: row 2 t + 1, column l4 + 4 p        k = 3: row 2 t + 1, column l4 + 4 (1 - p)        p = a & 1
 * so that the eight lanes of a quarter-warp (two atoms of opposite parity) gather from eight different bank groups in
 * every step: one shared-memory wavefront per quarter-warp unless a group overflowed its column (build_phase).
 * An entry is the number of a position slot (14 bits): k = 0, 2 sit in bits 0..13 of the two 32-bit halves, k = 1, 3
 * in bits 18..31, bits 14..17 are zero, so that the shared-memory address of an odd entry is one instruction (base +
 * (word >> 14): LEA.HI) and of an even one two (mask; base + 16 x: IMAD).  tmeta[8 task + a] = home slot of the atom |
 * trips << 14 (the trip count is the same for the eight atoms of a task). */
#define ENT_MASK 0x3fffu
__device__ __forceinline__ unsigned ent_even(unsigned w, unsigned base)
{
    unsigned a;
    asm("mad.lo.u32 %0, %1, 16, %2;" : "=r"(a) : "r"(w & ENT_MASK), "r"(base));
    return a;
}
__device__ __forceinline__ unsigned ent_odd(unsigned w, unsigned base) { return base + (w >> 14); }

/* sum over the four lanes of an atom of three values in three shuffles: lane 0 ends with fx, 1 fy, 2 fz (3: zero) */
template <typename T>
__device__ __forceinline__ T reduce3_4(T fx, T fy, T fz, int l4)
{
    const bool h = (l4 & 2) != 0, o = (l4 & 1) != 0;
    const T r0 = __shfl_xor_sync(0xffffffffu, h ? fx : fz, 2);
    const T r1 = __shfl_xor_sync(0xffffffffu, fy, 2);
    const T a = (h ? fz : fx) + r0;               /* lanes 0-1: fx of lanes {l, l ^ 2}; lanes 2-3: fz */
    const T b = h ? (T)0 : fy + r1;               /* lanes 0-1: fy */
    const T r2 = __shfl_xor_sync(0xffffffffu, o ? a : b, 1);
    return (o ? b : a) + r2;
}

/* Forces of the CTA's own atoms from the shared-memory list; EV: energy and virial partials accumulate in fp64 (R31)
 * and end as warp partials in red.  FAST = fp32 Lennard-Jones or Morse, one type, forces only: two entries share packed f32x2
 * operations, and the positions of the next two entries are gathered while the current two are computed. */
template <typename T, int KIND, bool NT1, bool EV>
__device__ __forceinline__ void pair_phase(const ResCfg &rc, unsigned pos_sa, unsigned rows_sa, const unsigned *tmeta,
                                           const PotEntry<T> *tab, T *fs, int A_own, int NT, double *red)
{
    double acc[EV ? 7 : 1];
    if (EV)
#pragma unroll
        for (int k = 0; k < 7; ++k) acc[k] = 0.0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l4 = lane & 3, a8 = lane >> 2;
    const unsigned zt = (unsigned)rc.NS * 16u;
    const int ntasks = (A_own + 7) >> 3;
    constexpr bool FAST = (sizeof(T) == 4) && (KIND == TS_LJ || KIND == TS_MORSE) && NT1 && !EV;
    const unsigned task_stride = (unsigned)rc.pitch * 16u;
    const unsigned lane_off = (unsigned)lane * 8u;
    const PotEntry<T> pe1 = tab[0];
    /* packed constants of the fast loops.  LJ: -12 c0, 6 c1.  Morse: -alpha log2 e, alpha r0 log2 e, 2 D alpha */
    const float rc2f = (float)pe1.rc2;
    const float ka = KIND == TS_LJ ? -12.0f * (float)pe1.c0 : -1.4426950408889634f * (float)pe1.p1;
    const float kb = KIND == TS_LJ ? 6.0f * (float)pe1.c1 : 1.4426950408889634f * (float)pe1.p1 * (float)pe1.p2;
    const float kc = (float)pe1.c0;
    for (int task = warp; task < ntasks; task += rc.nwarps) {
        const int al = task * 8 + a8;
        const unsigned meta = tmeta[al];
        const int nt = (int)(meta >> 14);
        const unsigned xa = pos_sa + ((meta & ENT_MASK) << 4);
        const bool has = al < A_own;
        const unsigned ra = rows_sa + (unsigned)task * task_stride + lane_off;
        T fx = 0, fy = 0, fz = 0;
        T ev[7] = { 0, 0, 0, 0, 0, 0, 0 };
        if (FAST) {
            const float4 xi4 = lds128(xa);
            const float xix = xi4.x, xiy = xi4.y, xiz = xi4.z;
            const f32x2 KA = pk2(ka, ka), KB = pk2(kb, kb), KC = pk2(kc, kc);
            f32x2 FX = pk2(0.f, 0.f), FY = FX, FZ = FX;
            if (nt > 0) {
                uint2 w = lds64(ra);
                float4 p0 = lds128(ent_even(w.x, pos_sa)), p1 = lds128(ent_odd(w.x, pos_sa));
                for (int t = 1; t < nt; ++t) {
                    const float4 q0 = lds128(ent_even(w.y, pos_sa)), q1 = lds128(ent_odd(w.y, pos_sa));
                    w = lds64(ra + (unsigned)t * 256u);
                    fast_pair2<KIND>(p0, p1, xix, xiy, xiz, rc2f, KA, KB, KC, FX, FY, FZ);
                    p0 = lds128(ent_even(w.x, pos_sa)); p1 = lds128(ent_odd(w.x, pos_sa));
                    fast_pair2<KIND>(q0, q1, xix, xiy, xiz, rc2f, KA, KB, KC, FX, FY, FZ);
                }
                const float4 q0 = lds128(ent_even(w.y, pos_sa)), q1 = lds128(ent_odd(w.y, pos_sa));
                fast_pair2<KIND>(p0, p1, xix, xiy, xiz, rc2f, KA, KB, KC, FX, FY, FZ);
                fast_pair2<KIND>(q0, q1, xix, xiy, xiz, rc2f, KA, KB, KC, FX, FY, FZ);
            }
            float a, b;
            upk2(FX, a, b); fx = (T)(a + b);
            upk2(FY, a, b); fy = (T)(a + b);
            upk2(FZ, a, b); fz = (T)(a + b);
        } else {
            const P3<T> xi = ld_pos_sa(xa, zt, (T)0);
            const PotEntry<T> pei = NT1 ? pe1 : tab[xi.ty * NT];
            const int tirow = xi.ty * NT;
            for (int t = 0; t < nt; ++t) {
                const uint2 w = lds64(ra + (unsigned)t * 256u);
                const P3<T> x0 = ld_pos_sa(ent_even(w.x, pos_sa), zt, (T)0);
                const P3<T> x1 = ld_pos_sa(ent_odd(w.x, pos_sa), zt, (T)0);
                const P3<T> x2 = ld_pos_sa(ent_even(w.y, pos_sa), zt, (T)0);
                const P3<T> x3 = ld_pos_sa(ent_odd(w.y, pos_sa), zt, (T)0);
                pair_accum<T, KIND, NT1, EV>(xi, x0, pei, tab, tirow, fx, fy, fz, ev);
                pair_accum<T, KIND, NT1, EV>(xi, x1, pei, tab, tirow, fx, fy, fz, ev);
                pair_accum<T, KIND, NT1, EV>(xi, x2, pei, tab, tirow, fx, fy, fz, ev);
                pair_accum<T, KIND, NT1, EV>(xi, x3, pei, tab, tirow, fx, fy, fz, ev);
            }
        }
        const T v = reduce3_4<T>(fx, fy, fz, l4);
        if (has && l4 < 3) fs[l4 * rc.A + al] = v;
        if (EV && has) {                /* fp64 from here on (R31): E = 1/2 sum V, W = -1/2 sum g r (x) r */
            acc[0] += 0.5 * (double)ev[0];
#pragma unroll
            for (int k = 1; k < 7; ++k) acc[k] += -0.5 * (double)ev[k];
        }
    }
    if (EV) {                           /* warp partials of E, W into red[warp][0..6] */
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            double a = acc[k];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
            if (lane == 0) red[warp * 8 + k] = a;
        }
    }
}

/* ------------------------------------------------------------------ ghost table (identical in every CTA) */
/* thr[k] = fixed-point fraction within which an atom is close enough to a face to need an image */
__device__ __forceinline__ void ghost_table(const ResCfg &rc, const uint4 *fr, unsigned *gtab, const unsigned *thr, int N_s,
                                            int NSB, ResMisc *misc)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = threadIdx.x; j < N_s; j += blockDim.x) {
        const uint4 u = fr[j];
        const unsigned uu[3] = { u.x, u.y, u.z };
        unsigned act = 0u, sg = 0u;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const bool lo = uu[k] < thr[k], hi = uu[k] > ~thr[k];
            act |= (unsigned)(lo || hi) << k;
            sg |= (unsigned)(uu[k] < 0x80000000u) << k;
        }
        gtab[j] = (act << 16) | (sg << 19) | ((1u << __popc(act)) - 1u);          /* low bits: image count for now */
    }
    __syncthreads();
    if (warp < 8) {                               /* warp g scans the atoms j = g mod 8: slots stay in bank group g */
        const int g = warp;
        unsigned run = 0u;
        for (int j0 = g; j0 < N_s; j0 += 256) {
            const int j = j0 + 8 * lane;
            const unsigned e = j < N_s ? gtab[j] : 0u;
            const unsigned c = e & 0xffffu;
            unsigned inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned v = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += v;
            }
            const unsigned slot = (unsigned)NSB + 8u * (run + inc - c) + (unsigned)g;
            if (j < N_s) gtab[j] = (e & 0xffff0000u) | (slot & 0xffffu);
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0 && (unsigned)NSB + 8u * run + 8u > (unsigned)rc.NS) misc->overflow = 1;   /* more images than planned */
    }
    __syncthreads();
    /* flagged overflow: no atom gets an image (and build_phase leaves every row empty) */
    if (misc->overflow)
        for (int j = threadIdx.x; j < N_s; j += blockDim.x) gtab[j] = 0u;
    __syncthreads();
}

/* ------------------------------------------------------------------ list build (per CTA, own atoms) */
/* One quarter-warp per atom; lane l tests the candidates j = 8 t + l (bank group l) and keeps the
 * hits as bit t of a mask in registers.  Two candidates per loop trip share packed f32x2 ops.  The
 * fractions fr[] are padded to a multiple of 16 atoms, so the loop carries no bounds checks; the
 * bits of j >= N_s and of j == i are cleared afterwards.                                          */
__device__ __forceinline__ unsigned wrap_bit(unsigned uj, unsigned ui)
{
    /* bit 31 = 1 when the minimum image of j relative to i along this axis is not the home image:
     * borrow(uj - ui) xor sign(uj - ui), one LOP3 */
    const unsigned dd = uj - ui;
    return (((~uj & ui) | (~(uj ^ ui) & dd)) ^ dd) >> 31;
}

/* shared-memory accesses of the build by 32-bit shared-window address (no generic address arithmetic in the loops) */
__device__ __forceinline__ uint4 lds_u4(unsigned a)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_u16(unsigned a, unsigned v) { asm volatile("st.shared.u16 [%0], %1;" :: "r"(a), "h"((unsigned short)v) : "memory"); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 pk2u(unsigned a, unsigned b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(a), "r"(b));
    return r;
}
/* u = u_j - u_i + 2^31 (the minimum-image difference of two 32-bit fractions, offset to unsigned) -> the bits of the
 * float 2^23 + (u >> 9): one funnel shift places the top 23 bits under the exponent of 2^23 (0x4B000000 = 0x96 << 23).
 * Subtracting 2^23 + 2^22 leaves floor(d / 512), d the signed difference: no integer-to-float conversion (a quarter-rate
 * instruction: six of them were the limit of the test loop) */
__device__ __forceinline__ unsigned frac_diff_bits(unsigned u) { return __funnelshift_r(u, 0x96u, 9); }

/* all ones when a < b, else zero */
__device__ __forceinline__ unsigned set_lt(float a, float b)
{
    unsigned r;
    asm("set.lt.u32.f32 %0, %1, %2;" : "=r"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ unsigned lds_u8(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
/* bit 31 = 1 when the minimum image of j relative to i along this axis is not the home image (wrap_bit without the shift) */
__device__ __forceinline__ unsigned wrap_msb(unsigned uj, unsigned ui)
{
    const unsigned dd = uj - ui;
    return ((~uj & ui) | (~(uj ^ ui) & dd)) ^ dd;
}
/* entry (act << 3 | mm) of the image-rank table: 8 x the rank of the subset mm among the non-empty subsets of act */
__device__ __forceinline__ unsigned char image_rank8(int idx)
{
    const unsigned act = (unsigned)idx >> 3, mm = (unsigned)idx & 7u;
    if (mm == 0u || (mm & ~act)) return 0x80;
    const unsigned a0 = act & 1u, a1 = (act >> 1) & 1u;
    return (unsigned char)(8u * ((mm & 1u) + (((mm >> 1) & 1u) << a0) + ((mm >> 2) << (a0 + a1)) - 1u));
}

template <bool ORTHO>
__device__ __noinline__ void build_phase(const ResCfg &rc, uint4 *fr, const unsigned *gtab, unsigned short *rows,
                                            unsigned *tmeta, const float *G, float rb2, int a_begin, int A_own, int N_s,
                                            int N8, ResMisc *misc, unsigned rank_sa)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = lane & 7, q = lane >> 3;
    const int ntasks = (A_own + 7) >> 3;          /* tasks of the pair phase: eight atoms, built four at a time */
    /* metric of the fraction differences (units of 2^-23 of the cell): xx, 2xy, 2xz, yy, 2yz, zz.  Orthogonal cell
     * vectors: the slots of the off-diagonal terms carry l_k = sqrt(G_kk) in G0, G3, G5 and -C l_k in G1, G2, G4 */
    const bool ortho = ORTHO;
    const float CF = 12582912.f;                                    /* C = 2^23 + 2^22 */
    const float l0 = sqrtf(G[0]), l1 = sqrtf(G[3]), l2 = sqrtf(G[5]);
    const f32x2 G0 = ortho ? pk2(l0, l0) : pk2(G[0], G[0]), G1 = ortho ? pk2(-CF * l0, -CF * l0) : pk2(G[1], G[1]);
    const f32x2 G2 = ortho ? pk2(-CF * l1, -CF * l1) : pk2(G[2], G[2]), G3 = ortho ? pk2(l1, l1) : pk2(G[3], G[3]);
    const f32x2 G4 = ortho ? pk2(-CF * l2, -CF * l2) : pk2(G[4], G[4]), G5 = ortho ? pk2(l2, l2) : pk2(G[5], G[5]);
    const f32x2 NC = pk2(-CF, -CF);
    const bool ovf = misc->overflow != 0;         /* ghost slots exhausted: leave every row empty (flagged) */
    const int T = (N_s + 7) >> 3;                 /* candidates per lane */
    const int W = (T + 31) >> 5;                  /* mask words per lane */
    const unsigned fr_sa = smem_u32(fr), rows_sa = smem_u32(rows);
    const unsigned cand_sa = fr_sa + (unsigned)l * 16u;             /* candidate t of lane l: cand_sa + 128 t */
    /* the gtab entry of every atom rides in the spare word of its fraction: one load per hit in the placement */
    for (int j = threadIdx.x; j < N_s; j += blockDim.x) {
        const unsigned e = gtab[j];
        ((unsigned *)fr)[4 * j + 3] = (e & 0xffffu) | (((e >> 16) & 7u) << 19);   /* first image slot | active axes << 19 */
    }
    __syncthreads();
    unsigned nnz = 0;
    for (int task = warp; task < ntasks; task += rc.nwarps) {
      int Rh0 = 0, Rh1 = 0, ai0 = 0;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        const int a8 = half * 4 + q;                            /* atom of the task */
        const int al = task * 8 + a8;
        const bool has = al < A_own;
        const int ai = hslot(a_begin + (has ? al : 0), N8);     /* slot of the atom: the build works in slot space */
        const uint4 ui = lds_u4(fr_sa + (unsigned)ai * 16u);
        const unsigned ox = ui.x + 0x80000000u, oy = ui.y + 0x80000000u, oz = ui.z + 0x80000000u;
        unsigned mask[8];
        int mine = 0;
#ifdef TS_RES_TIMING
        long long bt0 = clock64();
#endif
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            unsigned word = 0u;
            if (w < W) {
                const unsigned cw = cand_sa + (unsigned)w * 4096u;
                const int nb = min(32, T - w * 32);                 /* uniform */
#pragma unroll 4
                for (int b = 0; b < nb; b += 2) {
                    const uint4 ua = lds_u4(cw + (unsigned)b * 128u), ub = lds_u4(cw + (unsigned)b * 128u + 128u);
                    const f32x2 F0 = pk2u(frac_diff_bits(ua.x - ox), frac_diff_bits(ub.x - ox));
                    const f32x2 F1 = pk2u(frac_diff_bits(ua.y - oy), frac_diff_bits(ub.y - oy));
                    const f32x2 F2 = pk2u(frac_diff_bits(ua.z - oz), frac_diff_bits(ub.z - oz));
                    f32x2 R;
                    if (ORTHO) {
                        /* orthogonal cell vectors: Cartesian components l_k (F_k - C) straight from the bits, the offset
                         * folded into the product (its rounding shifts every difference vector by the same < 1e-7 L) */
                        const f32x2 Y0 = fma2(F0, G0, G1), Y1 = fma2(F1, G3, G2), Y2 = fma2(F2, G5, G4);
                        R = mul2(Y0, Y0);
                        R = fma2(Y1, Y1, R);
                        R = fma2(Y2, Y2, R);
                    } else {
                        const f32x2 E0 = add2(F0, NC), E1 = add2(F1, NC), E2 = add2(F2, NC);
                        f32x2 A0 = mul2(G0, E0);
                        A0 = fma2(G1, E1, A0);
                        A0 = fma2(G2, E2, A0);
                        f32x2 A1 = mul2(G3, E1);
                        A1 = fma2(G4, E2, A1);
                        R = mul2(mul2(G5, E2), E2);
                        R = fma2(E1, A1, R);
                        R = fma2(E0, A0, R);
                    }
                    float ra, rb;
                    upk2(R, ra, rb);
                    /* the hit bits enter at the top and move down: candidate 0 of the word ends up in bit 0 */
                    word = __funnelshift_r(word, set_lt(ra, rb2), 1);
                    word = __funnelshift_r(word, set_lt(rb, rb2), 1);
                }
                if (nb < 31) word >>= 32 - ((nb + 1) & ~1);        /* the loop tests candidates in pairs */
                /* candidates past the end of the system (padding) and the atom itself */
                const int tmax = (N_s - l + 7) >> 3;                /* lane l owns t < tmax */
                const int keep = tmax - w * 32;
                if (keep < 32) word &= keep <= 0 ? 0u : ((1u << keep) - 1u);
                if ((ai & 7) == l && (ai >> 8) == w) word &= ~(1u << ((ai >> 3) & 31));
                if (!has) word = 0u;
            }
            mask[w] = word;
            mine += __popc(word);
        }
#ifdef TS_RES_TIMING
        if (threadIdx.x == 0) { long long t = clock64(); atomicAdd(&g_res_prof[12], (unsigned long long)(t - bt0)); bt0 = t; }
#endif
        /* entries of the lanes below (exclusive prefix inside the quarter-warp) and of the whole atom */
        int inc = mine;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o, 8);
            if (l >= o) inc += v;
        }
        const int NT = __shfl_sync(0xffffffffu, inc, 7, 8);
        int R = ((NT + 15) >> 4) << 1;                                /* rows: whole trips of 16 entries */
        R = max(R, __shfl_xor_sync(0xffffffffu, R, 8));
        R = max(R, __shfl_xor_sync(0xffffffffu, R, 16));              /* the four atoms of a half task place into the same rows */
        const bool fits = 8 * R <= rc.pitch && !ovf;
        if (!fits) {
            if (lane == 0) misc->overflow = 1;
            R = 0;
        }
        /* u16 halves of the trip words of this atom (see "list layout"): row r of column c lives at
         * base + (r / 2) * 128 + (c & 3) * 4 + (r & 1) * 2 + ((c >> 2) ^ p), p = parity of the atom in its task;
         * the odd half holds the entry << 2 (bits 18..31 of the word) */
        const int par = a8 & 1;
        const unsigned rowB_sa = rows_sa + 2u * ((unsigned)task * (unsigned)rc.pitch * 8u + (unsigned)a8 * 16u);
#define CELL_SA(r, c) (rowB_sa + 2u * (unsigned)(((r) >> 1) * 128 + ((c) & 3) * 4 + ((r) & 1) * 2 + (((c) >> 2) ^ par)))
#define ENT(slot, c) ((unsigned)(slot) << (((((c) >> 2) ^ par)) << 1))
        if (fits) {
            /* Placement.  The pair loop reads R rows of eight entries; entry (row, column) is read by lane
             * `column`, and one shared-memory wavefront serves a row when its eight bank groups differ.  Lane l
             * holds the hits of bank group l: its first R hits fill column l from the top (column = bank
             * group, so those never collide), the rest of the column is padded with the far-away dummy of group l.
             * A group with more than R hits overflows: those hits take the free cells of the other columns in
             * column-major order, where they collide with their own group's column once each -- the minimum. */
            const int o_l = max(0, mine - R), f_l = max(0, R - mine);
            int io = o_l, jf = f_l;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                const int vo = __shfl_up_sync(0xffffffffu, io, o, 8), vf = __shfl_up_sync(0xffffffffu, jf, o, 8);
                if (l >= o) { io += vo; jf += vf; }
            }
            const int O = __shfl_sync(0xffffffffu, io, 7, 8);             /* overflow entries of the atom */
            const int F_l = jf - f_l;                                     /* free cells in the columns below l */
            const int recv = min(max(O - F_l, 0), f_l);                   /* overflow entries that land in column l */
            int u = io - o_l;                                             /* number of my first overflow entry */
            /* slot of the neighbour whose fraction lies at shared address ja, as seen from atom i: its home slot, or the
             * slot of the image the minimum-image convention selects (bit k of mm: the pair wraps along axis k) */
            auto slot_of = [&](unsigned ja, unsigned j) -> unsigned {
                const uint4 uj = lds_u4(ja);
                /* mm = wrap bits of z, y, x: three funnel shifts collect the three top bits */
                const unsigned mm = __funnelshift_l(wrap_msb(uj.x, ui.x), __funnelshift_l(wrap_msb(uj.y, ui.y), wrap_msb(uj.z, ui.z) >> 31, 1), 1);
                unsigned slot = j;
                if (mm) {
                    /* uj.w = first image slot | active axes << 19: the byte table gives 8 x the rank of the subset mm among
                     * the non-empty subsets of the active axes (0x80: not a subset -- cannot happen, see ghost_table) */
                    const unsigned r8 = lds_u8(rank_sa + (uj.w >> 16) + mm);
                    if (r8 & 0x80u) misc->overflow = 1;
                    slot = (uj.w & 0xffffu) + r8;
                }
                return slot;
            };
            /* pass 1: the first R hits of the lane go down its own column -- the common case, kept lean */
            const unsigned cmul = 1u << ((((l >> 2) ^ par)) << 1);        /* the odd half holds the entry << 2 */
            unsigned cell = CELL_SA(0, l), dlt = 4u;
            int left = R;
#pragma unroll
            for (int w = 0; w < 8; ++w) {
                unsigned word = mask[w];
                const unsigned cw = cand_sa + (unsigned)w * 4096u, jw = (unsigned)(w * 256 + l);
                while (word && left) {
                    const unsigned b = (unsigned)__ffs(word) - 1u;
                    word &= word - 1u;
                    sts_u16(cell, slot_of(cw + b * 128u, jw + b * 8u) * cmul);
                    cell += dlt;                                       /* row m + 1 of the column: + 4, + 252, + 4, ... bytes */
                    dlt = 256u - dlt;
                    --left;
                }
                mask[w] = word;
            }
            /* pass 2: the overflow hits (what is left in the masks) take the free cells, column-major */
            int cq[8];                                                    /* populations of the eight bank groups of the atom */
#pragma unroll
            for (int c = 0; c < 8; ++c) cq[c] = __shfl_sync(0xffffffffu, mine, c, 8);
#pragma unroll 1
            for (int w = 0; w < W; ++w) {
                unsigned word = mask[0];
#pragma unroll
                for (int k = 1; k < 8; ++k) word = w == k ? mask[k] : word;
                const unsigned cw = cand_sa + (unsigned)w * 4096u, jw = (unsigned)(w * 256 + l);
                while (word) {
                    const unsigned b = (unsigned)__ffs(word) - 1u;
                    word &= word - 1u;
                    const unsigned slot = slot_of(cw + b * 128u, jw + b * 8u);
                    int P = 0, Fc = 0, pcol = 0;
#pragma unroll
                    for (int c = 0; c < 8; ++c) {                      /* columns whose free cells all come before cell u */
                        P += R - min(R, cq[c]);
                        if (P <= u) { pcol = c + 1; Fc = P; }
                    }
                    int cc = 0;
#pragma unroll
                    for (int c = 0; c < 8; ++c) cc = pcol == c ? cq[c] : cc;
                    const int prow = cc + (u - Fc);
                    ++u;
                    sts_u16(CELL_SA(prow, pcol), ENT(slot, pcol));
                }
            }
            /* padding of my column below my own hits and the overflow entries it received */
            for (int r = min(mine, R) + recv; r < R; ++r) sts_u16(CELL_SA(r, l), ENT(N8 + l, l));
        }
#ifdef TS_RES_TIMING
        if (threadIdx.x == 0) { long long t = clock64(); atomicAdd(&g_res_prof[13], (unsigned long long)(t - bt0)); bt0 = t; }
#endif
        if (half == 0) { Rh0 = R; ai0 = has ? ai : N8; } else Rh1 = R;
        if (has) nnz += (unsigned)mine;
        if (half == 1) {
            /* the eight atoms of the task share the trip count: the shorter half is padded with dummies */
            const int Rm = max(Rh0, Rh1);
            unsigned short *row0 = rows + (size_t)task * rc.pitch * 8 + q * 16;
            const int par0 = q & 1;
            for (int r = Rh0; r < Rm; ++r)
                row0[(r >> 1) * 128 + (l & 3) * 4 + (r & 1) * 2 + ((l >> 2) ^ par0)] = (unsigned short)((unsigned)(N8 + l) << (((l >> 2) ^ par0) << 1));
            for (int r = Rh1; r < Rm; ++r) sts_u16(CELL_SA(r, l), ENT(N8 + l, l));
            if (l == 0) {
                tmeta[task * 8 + q] = (unsigned)ai0 | ((unsigned)(Rm >> 1) << 14);
                tmeta[task * 8 + 4 + q] = (unsigned)(has ? ai : N8) | ((unsigned)(Rm >> 1) << 14);
            }
        }
#undef CELL_SA
#undef ENT
      }
    }
    nnz = __reduce_add_sync(0xffffffffu, nnz);
    if (lane == 0 && nnz) atomicAdd(&misc->nnz, nnz);
}

/* ------------------------------------------------------------------ the list across calls
 * At the end of a call every CTA copies what it needs to go on without a rebuild -- task words, x_ref | wrap shift of its
 * own atoms, the image table, and the trips of the rows that are in use -- into its share of the system's own segment
 * of the general engine's pair array (the resident engine's systems do not use it), and the next call that finds
 * res_saved[s] = 1 copies it back instead of building the list (a 10-step call of an in-flight FIRE run spends more
 * than a third of its time in that build).  The flag is 1 only when every CTA of the cluster had room; it is cleared
 * by the swap kernel for a replaced system and by the host for the whole batch whenever something else wrote the pair
 * array or the positions (ts_internal.cuh: res_saved_ok).                                                            */
struct SavedHead { unsigned trips, ntasks, nnz, pad; };

template <typename T>
__device__ __forceinline__ unsigned char *saved_base(const DevState &d, const ResCfg &rc, int s, int rank, size_t &share)
{
    const long long b0 = d.nbr_base[s], b1 = d.nbr_base[s + 1];
    share = ((size_t)(b1 - b0) * 4u / (size_t)rc.CL) & ~(size_t)15;
    return (unsigned char *)(d.nbr + b0) + (size_t)rank * share;
}

/* scan[t] = trips of the tasks before t (scan: ntasks + 1 words of scratch); returns the total */
__device__ __forceinline__ unsigned trip_scan(const unsigned *tmeta, int ntasks, unsigned *scan)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned run = 0u;
        for (int t = 0; t < ntasks; ++t) { scan[t] = run; run += tmeta[8 * t] >> 14; }
        scan[ntasks] = run;
    }
    __syncthreads();
    return scan[ntasks];
}

/* (plain arguments, no references to the kernel's parameter structs: those would move to local memory) */
template <typename T>
__device__ __forceinline__ void save_list(unsigned char *base, size_t share, int *flag, int A, int pitch, int nwarps, int N_s,
                                       int A_own, const unsigned short *rows, const unsigned *tmeta, const unsigned *gtab,
                                       const Q4<T> *oref, Q4<T> Rr, unsigned nnz, bool overflow, unsigned *scan)
{
    const int ntasks = (A_own + 7) >> 3;
    const unsigned total = trip_scan(tmeta, ntasks, scan);
    const size_t o_meta = sizeof(SavedHead), o_ref = o_meta + 4u * (size_t)A, o_gtab = o_ref + sizeof(Q4<T>) * (size_t)A;
    const size_t o_rows = o_gtab + 4u * (size_t)((N_s + 3) & ~3);
    if (overflow || o_rows + 256u * (size_t)total > share) {      /* no room (or no list): the next call builds it */
        if (threadIdx.x == 0) *flag = 0;
        return;
    }
    if (threadIdx.x == 0) {
        SavedHead h;
        h.trips = total; h.ntasks = (unsigned)ntasks; h.nnz = nnz; h.pad = 0u;
        *(SavedHead *)base = h;
    }
    unsigned *gm = (unsigned *)(base + o_meta), *gg = (unsigned *)(base + o_gtab);
    for (int k = threadIdx.x; k < 8 * ntasks; k += blockDim.x) gm[k] = tmeta[k];
    for (int k = threadIdx.x; k < N_s; k += blockDim.x) gg[k] = gtab[k];
    if ((int)threadIdx.x < A_own) ((Q4<T> *)(base + o_ref))[threadIdx.x] = sizeof(T) == 4 ? oref[threadIdx.x] : Rr;
    const int lane = threadIdx.x & 31;
    for (int t = threadIdx.x >> 5; t < ntasks; t += nwarps) {
        const uint4 *src = (const uint4 *)(rows + (size_t)t * pitch * 8);
        uint4 *dst = (uint4 *)(base + o_rows + 256u * (size_t)scan[t]);
        const int n16 = (int)(scan[t + 1] - scan[t]) * 16;
        for (int k = lane; k < n16; k += 32) dst[k] = src[k];
    }
}

/* the reverse; the own atoms' x_ref | wrap shift go to oref (fp32) or come back in the return value (fp64) */
template <typename T>
__device__ __forceinline__ Q4<T> restore_list(const unsigned char *base, int A, int pitch, int nwarps, int N_s, int A_own,
                                           unsigned short *rows, unsigned *tmeta, unsigned *gtab, Q4<T> *oref,
                                           ResMisc *misc, unsigned *scan)
{
    const int ntasks = (A_own + 7) >> 3;
    const size_t o_meta = sizeof(SavedHead), o_ref = o_meta + 4u * (size_t)A, o_gtab = o_ref + sizeof(Q4<T>) * (size_t)A;
    const size_t o_rows = o_gtab + 4u * (size_t)((N_s + 3) & ~3);
    const unsigned *gm = (const unsigned *)(base + o_meta), *gg = (const unsigned *)(base + o_gtab);
    for (int k = threadIdx.x; k < 8 * ntasks; k += blockDim.x) tmeta[k] = gm[k];
    for (int k = threadIdx.x; k < N_s; k += blockDim.x) gtab[k] = gg[k];
    Q4<T> R;
    R.a = R.b = R.c = R.d = 0;
    if ((int)threadIdx.x < A_own) {
        R = ((const Q4<T> *)(base + o_ref))[threadIdx.x];
        if (sizeof(T) == 4) oref[threadIdx.x] = R;
    }
    if (threadIdx.x == 0) { misc->nnz = ((const SavedHead *)base)->nnz; misc->overflow = 0; }
    trip_scan(tmeta, ntasks, scan);
    const int lane = threadIdx.x & 31;
    for (int t = threadIdx.x >> 5; t < ntasks; t += nwarps) {
        uint4 *dst = (uint4 *)(rows + (size_t)t * pitch * 8);
        const uint4 *src = (const uint4 *)(base + o_rows + 256u * (size_t)scan[t]);
        const int n16 = (int)(scan[t + 1] - scan[t]) * 16;
        for (int k = lane; k < n16; k += 32) dst[k] = src[k];
    }
    __syncthreads();
    return R;
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

/* ------------------------------------------------------------------ FIRE inside the resident engine (O6, R21, R22)
 * The per-system FIRE state lives in shared memory, replicated in every CTA of the cluster: each CTA runs the same
 * state machine on the same (bitwise identical) reduced values, so no state is ever sent. */
struct FireSm {
    double dt, alpha;
    int npos, nsteps, status, pad;
    double acc[4];     /* max |F_i|^2, P = F.v, v.v, F.F of the system */
};

/* max / sums over the system in fixed order: warp shuffle -> per-warp slots -> per-CTA -> every CTA of the cluster */
__device__ __forceinline__ void fire_reduce(cg::cluster_group &cluster, int CL, int rank, double f2, double P, double vv,
                                            double *red, double *cred, int nwarps, double out[4])
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double mx = f2, ff = f2;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        P += __shfl_xor_sync(0xffffffffu, P, o);
        vv += __shfl_xor_sync(0xffffffffu, vv, o);
        ff += __shfl_xor_sync(0xffffffffu, ff, o);
    }
    if (lane == 0) { red[warp * 8 + 0] = mx; red[warp * 8 + 1] = P; red[warp * 8 + 2] = vv; red[warp * 8 + 3] = ff; }
    __syncthreads();
    if (threadIdx.x < 4) {
        double a = red[threadIdx.x];
        for (int w = 1; w < nwarps; ++w) a = threadIdx.x == 0 ? fmax(a, red[w * 8]) : a + red[w * 8 + threadIdx.x];
        for (int r = 0; r < CL; ++r) cluster.map_shared_rank(cred, r)[rank * 8 + threadIdx.x] = a;
    }
    if (CL > 1) cluster.sync(); else __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        double a = cred[k];
        for (int r = 1; r < CL; ++r) a = k == 0 ? fmax(a, cred[r * 8 + k]) : a + cred[r * 8 + k];
        out[k] = a;
    }
    if (CL > 1) cluster.sync(); else __syncthreads();          /* cred may be rewritten by the next reduction */
}

/* ------------------------------------------------------------------ the kernel */
template <typename T, int KIND, bool NT1, bool FIRE, bool DUMP = false>
__global__ void __launch_bounds__(sizeof(T) == 4 ? RES_MAX_THREADS : RES_MAX_THREADS_F64, 1) k_resident_md(DevState d, MdConst c, ResCfg rc, int n_steps, unsigned want, ts_fire_params fp)
{
    unsigned char *const smem = ts_smem;
    cg::cluster_group cluster = cg::this_cluster();
    const int CL = rc.CL;
    const int rank = (int)cluster.block_rank();
    const int cid = (int)(blockIdx.x / (unsigned)CL);
    const int tid = threadIdx.x;
    const unsigned zt = (unsigned)rc.NS * 16u;
    constexpr unsigned SB = 4u * (unsigned)sizeof(T);          /* bytes of a home slot */

    unsigned char *const posb = smem + rc.o_pos;
    uint4 *fr = (uint4 *)(smem + rc.o_fr);
    unsigned *gtab = (unsigned *)(smem + rc.o_gtab);
    unsigned short *rows = (unsigned short *)(smem + rc.o_rows);
    T *fs = (T *)(smem + rc.o_fs);
    unsigned *tmeta = (unsigned *)(smem + rc.o_meta);
    T *noise = (T *)(smem + rc.o_noise);  /* [3][A] Langevin kicks of the own atoms for the next step */
    /* state of the own atoms, one 4-vector each, between the owner phases.  fp32: in shared memory -- at 72 registers
     * per thread (864 threads) the registers belong to the pair loop, whose gathers must stay one trip ahead of its
     * arithmetic.  fp64 (512 threads, 128 registers): in registers (Xr, Vr, Rr), the slots are twice as large */
    constexpr bool OWN_SMEM = sizeof(T) == 4;
    Q4<T> *ox = (Q4<T> *)(smem + rc.o_own);   /* [A] x (unwrapped), 1 / (m mass_conv)                                 */
    Q4<T> *ov = ox + rc.A;                    /* [A] v                                                                */
    Q4<T> *oref = ov + rc.A;                  /* [A] x at the last build (skin test), packed wrap shift (wa, wb, wc)   */
    PotEntry<T> *tab = (PotEntry<T> *)(smem + rc.o_pot);
    double *red = (double *)(smem + rc.o_red);
    double *cred = (double *)(smem + rc.o_cred);
    ResMisc *misc = (ResMisc *)(smem + rc.o_misc);
    T *gh = (T *)(misc + 1);            /* h[9], hinv[9] in the state dtype */
    float *G = (float *)(gh + 18);      /* metric of the fixed-point fractions, [6] + rb2 */
    unsigned *thr = (unsigned *)(G + 8);/* ghost thresholds [3] */
    FireSm *fsm = (FireSm *)(smem + rc.o_fire);
    double *fred = (double *)(fsm + 1);   /* per-warp scratch of fire_reduce, [nwarps][8] */

    const unsigned mb_full = smem_u32(smem + rc.o_mbar);
    const unsigned pos_sa = smem_u32(posb);
    const unsigned rows_sa = smem_u32(rows);
    unsigned full_parity = 0u;
    if (tid == 0) {
        mb_init(mb_full, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int NT = d.n_types;
    for (int k = tid; k < NT * NT; k += blockDim.x) tab[k] = ((const PotEntry<T> *)d.pot)[k];
    if (blockIdx.x == 0 && tid == 0 && !DUMP) d.status->res_nnz[rc.nnz_slot ^ 1] = 0ull;
    __shared__ unsigned char s_rank[64];          /* image-rank table of the list build */
    if (tid < 64) s_rank[tid] = image_rank8(tid);

    for (int ks = cid; ks < rc.n_list; ks += rc.n_clusters) {
        const int s = rc.syslist ? rc.syslist[ks] : ks;
        const int g0 = d.sysoff[s];
        const int N_s = d.sysoff[s + 1] - g0;
        const int N8 = (N_s + 7) & ~7;
        if (DUMP && s != rc.dump_sys) continue;
        const int A_s = ((((N_s + CL - 1) / CL) + 7) >> 3) << 3;   /* whole blocks of eight slots per CTA */
        const int a_begin = rank * A_s;
        const int A_own = max(0, min(A_s, N_s - a_begin));
        const int sb0 = min(a_begin, N8), sbw = min(a_begin + A_s, N8) - sb0;   /* the CTA's own slots [sb0, sb0 + sbw) */
        const int n_peer_slots = N8 - sbw;            /* slots of the other CTAs */
        const unsigned peer_bytes = (unsigned)(N_s - A_own) * SB;
        const SysGeom &geo = d.geom[s];
        int fstat0 = 0;
        if (FIRE) {                                    /* finished systems stay bit-unchanged (R22) */
            fstat0 = d.f_status[s];
            if (fstat0 == TS_FIRE_CONVERGED || fstat0 == TS_FIRE_FAILED) continue;
        }
        /* ---- per-system constants into shared memory */
        if (tid < 9) { gh[tid] = (T)geo.h[tid]; gh[9 + tid] = (T)geo.hinv[tid]; }
        if (tid == 64) {
            const double *h = geo.h;
            double M[6], lmax = 0.0;
            int kk[6][2] = { { 0, 0 }, { 0, 1 }, { 0, 2 }, { 1, 1 }, { 1, 2 }, { 2, 2 } };
            for (int e = 0; e < 6; ++e) {
                int a = kk[e][0], b = kk[e][1];
                M[e] = h[3 * a] * h[3 * b] + h[3 * a + 1] * h[3 * b + 1] + h[3 * a + 2] * h[3 * b + 2];
                if (a != b) M[e] *= 2.0;
            }
            const double sc = 1.0 / 70368744177664.0;            /* 2^-46: the build measures fractions in units of 2^-23 */
            for (int e = 0; e < 6; ++e) G[e] = (float)(M[e] * sc);
            for (int a = 0; a < 3; ++a) lmax = fmax(lmax, sqrt(h[3 * a] * h[3 * a] + h[3 * a + 1] * h[3 * a + 1] + h[3 * a + 2] * h[3 * a + 2]));
            const double rb = d.r_list + (double)rc.eps_rel * lmax;
            G[6] = (float)(rb * rb);
            for (int k = 0; k < 3; ++k) {       /* a pair within rb that wraps along k has u_j within rb / h_perp of a face */
                double rho = (rb + 2.0 * (double)rc.eps_rel * lmax) / geo.hperp[k] + 1e-6;
                thr[k] = rho >= 0.5 ? 0x80000000u : (unsigned)(rho * 4294967296.0);
            }
            misc->nnz = 0u; misc->rebuilds = 0u; misc->overflow = 0;
            if (FIRE) {
                const bool fresh = fstat0 == TS_FIRE_FRESH;
                fsm->dt = fresh ? fp.dt_start : d.f_dt[s];
                fsm->alpha = fresh ? fp.alpha_start : d.f_alpha[s];
                fsm->npos = fresh ? 0 : d.f_npos[s];
                fsm->nsteps = fresh ? 0 : d.f_nsteps[s];
                fsm->status = TS_FIRE_RUNNING;
            }
        }
        /* ---- owner state */
        const bool own = tid < A_own;
        const int ai = a_begin + tid;                 /* system-local atom index  */
        const int hs = hslot(ai, N8);                 /* its home slot            */
        const long long gi = (long long)g0 + ai;      /* global atom index        */
        int ty = 0;
        Q4<T> Xr, Vr, Rr;
        Xr.a = Xr.b = Xr.c = Xr.d = 0; Vr = Xr; Rr = Xr;
        if (own) {
            const T *x = (const T *)d.pos + 3 * gi, *v = (const T *)d.vel + 3 * gi;
            Q4<T> X, V;
            X.a = x[0]; X.b = x[1]; X.c = x[2]; V.a = v[0]; V.b = v[1]; V.c = v[2]; V.d = 0;
            X.d = (T)1 / (((const T *)d.mass)[gi] * (T)d.mass_conv);
            ty = d.type[gi];
            if (FIRE && fstat0 == TS_FIRE_FRESH) { V.a = 0; V.b = 0; V.c = 0; }
            if (OWN_SMEM) { ox[tid] = X; ov[tid] = V; } else { Xr = X; Vr = V; }
        }
        const unsigned uid = d.uid_own[s];
        const unsigned long long step0 = d.sys_step[s];
        /* Langevin noise (O4, O5): when the block has a spare thread for every own atom, thread blockDim - A_own + k draws
         * the kick c2 sqrt(kT / m) xi of atom k for step n + 1 while the owners integrate step n: the Philox rounds and the
         * Box-Muller transform are more than half of the owners' dependent instruction chain */
        const bool noise_helpers = !FIRE && rc.noise_helpers && c.integrator == TS_BAOAB && (int)blockDim.x >= 2 * A_own;
        const int hk = tid - ((int)blockDim.x - A_own);          /* helper of own atom hk */
        T hsig = 0;
        if (noise_helpers && hk >= 0) {
            const T hm = (T)1 / (((const T *)d.mass)[g0 + a_begin + hk] * (T)d.mass_conv);
            hsig = (T)c.c2 * (sizeof(T) == 4 ? (T)sqrtf((float)((T)c.kT * hm)) : (T)sqrt((double)((T)c.kT * hm)));
        }
        T hdt = (T)c.hdt, dt = (T)c.dt;
        int n_done = 0;                               /* steps taken by this system in this call */
        bool have_ev = false;                         /* the last pair pass also produced E (and W) */
        cluster.sync();                               /* constants visible; previous system fully retired everywhere */

        /* the list the last call left for these positions (every CTA of the cluster reads the same flag) */
        bool restored = false;
#ifdef TS_RES_TIMING
        long long rt0 = clock64();
#endif
        if (!DUMP && d.res_saved[s]) {
            size_t share;
            const unsigned char *sbase = saved_base<T>(d, rc, s, rank, share);
            const Q4<T> R = restore_list<T>(sbase, rc.A, rc.pitch, rc.nwarps, N_s, A_own, rows, tmeta, gtab, oref, misc, (unsigned *)red);
            if (own) {
                /* home slots of all atoms in every CTA, with the wrap shift of the build that made the list */
                if (!OWN_SMEM) Rr = R;
                const Q4<T> X = OWN_SMEM ? ox[tid] : Xr;
                const int wpack = bits_from(R.d);
                const T wa = (T)(signed char)(wpack & 0xff), wb = (T)(signed char)((wpack >> 8) & 0xff), wc = (T)(signed char)((wpack >> 16) & 0xff);
                publish_home<T>(cluster, CL, posb, zt, hs, X.a - (wa * gh[0] + wb * gh[3] + wc * gh[6]),
                                X.b - (wa * gh[1] + wb * gh[4] + wc * gh[7]), X.c - (wa * gh[2] + wb * gh[5] + wc * gh[8]), ty);
            }
            if (tid < 8) {
                const T far = (T)1e15;
                st_pos(posb, (unsigned)(N8 + tid) * 16u, zt, far, far, far, 0);
            }
            cluster.sync();
            ghost_pass<T>(posb, zt, gtab, gh, N_s);
            __syncthreads();
            restored = true;
        }
#ifdef TS_RES_TIMING
        if (tid == 0) atomicAdd(&g_res_prof[12], (unsigned long long)(clock64() - rt0));
#endif
#ifdef TS_RES_TIMING
        long long prof_acc[12] = { 0 }, prof_t = clock64();
#endif
        for (int n = 0; n <= n_steps; ++n) {
            bool rebuild = n == 0 && !restored;
            const bool last = n == n_steps;
            if (FIRE && n > 0) {
                if (fsm->nsteps >= fp.max_steps) {     /* reported as failed, never counted (R24) */
                    __syncthreads();
                    if (tid == 0) fsm->status = TS_FIRE_FAILED;
                    break;
                }
                dt = (T)fsm->dt; hdt = (T)0.5 * dt;
            }
            T kick0 = 0, kick1 = 0, kick2 = 0;
            const bool draws = noise_helpers && hk >= 0 && n < n_steps;
            if (draws) {                                               /* the kicks of step n + 1, stored once the owners have read those of step n */
                const unsigned long long step = step0 + (unsigned long long)n;
                unsigned w[4];
                philox4x32_10((unsigned)(a_begin + hk), uid, (unsigned)(step & 0xffffffffull), (unsigned)(step >> 32), c.key0, c.key1, w);
                T xi[3];
                normals3(w, xi);
                kick0 = hsig * xi[0]; kick1 = hsig * xi[1]; kick2 = hsig * xi[2];
            }
            if (n > 0) {
                bool moved = false;
                if (tid == 0 && peer_bytes) mb_expect_tx(mb_full, peer_bytes);   /* this step's home slots of the other CTAs */
                T x0 = 0, x1 = 0, x2 = 0;
                int wpack = 0;
                if (own) {
                    const T f0 = fs[tid], f1 = fs[rc.A + tid], f2 = fs[2 * rc.A + tid];
                    const Q4<T> X = OWN_SMEM ? ox[tid] : Xr, V = OWN_SMEM ? ov[tid] : Vr, R = OWN_SMEM ? oref[tid] : Rr;
                    const T im = X.d;
                    T v0 = V.a, v1 = V.b, v2 = V.c;
                    x0 = X.a; x1 = X.b; x2 = X.c;
                    /* first half of the step (O3 / O4), as in the general engine */
                    if (FIRE || c.integrator == TS_NVE) {
                        v0 = v0 + hdt * (f0 * im); x0 = x0 + dt * v0;
                        v1 = v1 + hdt * (f1 * im); x1 = x1 + dt * v1;
                        v2 = v2 + hdt * (f2 * im); x2 = x2 + dt * v2;
                    } else if (noise_helpers) {
                        const T *nz = noise + tid;
                        const T c1 = (T)c.c1, k0 = nz[0], k1 = nz[rc.A], k2 = nz[2 * rc.A];
                        v0 = v0 + hdt * (f0 * im); x0 = x0 + hdt * v0; v0 = c1 * v0 + k0; x0 = x0 + hdt * v0;
                        v1 = v1 + hdt * (f1 * im); x1 = x1 + hdt * v1; v1 = c1 * v1 + k1; x1 = x1 + hdt * v1;
                        v2 = v2 + hdt * (f2 * im); x2 = x2 + hdt * v2; v2 = c1 * v2 + k2; x2 = x2 + hdt * v2;
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
                    Q4<T> Xn, Vn;
                    Xn.a = x0; Xn.b = x1; Xn.c = x2; Xn.d = im; Vn.a = v0; Vn.b = v1; Vn.c = v2; Vn.d = 0;
                    if (OWN_SMEM) { ox[tid] = Xn; ov[tid] = Vn; } else { Xr = Xn; Vr = Vn; }
                    T a = x0 - R.a, b = x1 - R.b, cc = x2 - R.c;
                    moved = (double)(a * a + b * b + cc * cc) > d.half_skin2;
                    wpack = bits_from(R.d);
                }
                TICK(1);
                if (!FIRE && CL > 1) cl_wait();       /* every CTA of the cluster has finished reading the old positions (FIRE: fire_reduce's barriers) */
                TICK(2);
                if (own) {
                    /* the new home slot: into the other CTAs' slot arrays with st.async, which completes transaction bytes
                     * on the RECEIVING CTA's mbarrier (the skin flag travels in the type word); into the own slot array
                     * directly, together with the images of the atom */
                    /* the wrap shift of the last build, from its integer coefficients with the expression of the build */
                    const T wa = (T)(signed char)(wpack & 0xff), wb = (T)(signed char)((wpack >> 8) & 0xff), wc = (T)(signed char)((wpack >> 16) & 0xff);
                    const T px = x0 - (wa * gh[0] + wb * gh[3] + wc * gh[6]);
                    const T py = x1 - (wa * gh[1] + wb * gh[4] + wc * gh[7]);
                    const T pz = x2 - (wa * gh[2] + wb * gh[5] + wc * gh[8]);
                    const int tyw = ty | (moved ? MOVED_BIT : 0);
                    for (int r = 0; r < CL; ++r)
                        if (r != rank)
                            st_async_pos(map_cluster(pos_sa + (unsigned)hs * 16u, (unsigned)r), map_cluster(mb_full, (unsigned)r), zt, px, py, pz, tyw);
                    st_pos(posb, (unsigned)hs * 16u, zt, px, py, pz, ty);
                    ghost_write<T>(posb, zt, gtab[hs], gh, px, py, pz, ty);
                }
                TICK(0);
                if (peer_bytes) {                     /* all home slots of the others have arrived in THIS CTA */
                    mb_wait(mb_full, full_parity);
                    full_parity ^= 1u;
                }
                TICK(3);
                /* images of the others' new home positions and their skin flags; own home and image slots complete */
                moved |= peer_pass<T>(posb, zt, gtab, gh, sb0, sbw, n_peer_slots, N_s);
                rebuild = __syncthreads_or(moved ? 1 : 0) != 0;
                TICK(4);
            }
            if (draws) { noise[hk] = kick0; noise[rc.A + hk] = kick1; noise[2 * rc.A + hk] = kick2; }
            if (rebuild) {
                /* every CTA of the cluster takes this branch in the same step (the flags travel with the home slots);
                 * nobody may still be reading its home / ghost slots when the re-wrapped slots and fr arrive */
                cluster.sync();
                if (tid == 0) { misc->rebuilds += 1u; misc->nnz = 0u; }
                if (own) {
                    /* wrap into the cell: f = x . h^-1, w = floor(f) (R5: the stored x stays unwrapped) */
                    const Q4<T> X = OWN_SMEM ? ox[tid] : Xr;
                    const T x0 = X.a, x1 = X.b, x2 = X.c;
                    T fa = x0 * gh[9] + x1 * gh[12] + x2 * gh[15];
                    T fb = x0 * gh[10] + x1 * gh[13] + x2 * gh[16];
                    T fc = x0 * gh[11] + x1 * gh[14] + x2 * gh[17];
                    T wa = t_floor<T>(fa), wb = t_floor<T>(fb), wc = t_floor<T>(fc);
                    fa -= wa; fb -= wb; fc -= wc;
                    if (fa >= (T)1) { wa += (T)1; fa = (T)0; }
                    if (fb >= (T)1) { wb += (T)1; fb = (T)0; }
                    if (fc >= (T)1) { wc += (T)1; fc = (T)0; }
                    const T ws0 = wa * gh[0] + wb * gh[3] + wc * gh[6];
                    const T ws1 = wa * gh[1] + wb * gh[4] + wc * gh[7];
                    const T ws2 = wa * gh[2] + wb * gh[5] + wc * gh[8];
                    /* |w| < 128, or the system is flagged: an atom that far outside its cell has left any sensible trajectory */
                    if (!(fabs((double)wa) < 127.5 && fabs((double)wb) < 127.5 && fabs((double)wc) < 127.5)) atomicOr(&d.status->flags, TS_FLAG_SHIFT_RANGE);
                    Q4<T> R;
                    R.a = x0; R.b = x1; R.c = x2;
                    R.d = bits_to(((int)wa & 0xff) | (((int)wb & 0xff) << 8) | (((int)wc & 0xff) << 16), (T)0);
                    if (OWN_SMEM) oref[tid] = R; else Rr = R;
                    const uint4 u = make_uint4(frac_to_u32(fa), frac_to_u32(fb), frac_to_u32(fc), 0u);
                    for (int r = 0; r < CL; ++r) cluster.map_shared_rank(fr, r)[hs] = u;
                    publish_home<T>(cluster, CL, posb, zt, hs, x0 - ws0, x1 - ws1, x2 - ws2, ty);
                }
                if (tid < 8) {                        /* the far-away dummy neighbours (list padding), one per bank group */
                    const T far = (T)1e15;
                    st_pos(posb, (unsigned)(N8 + tid) * 16u, zt, far, far, far, 0);
                }
                cluster.sync();                       /* fractions and home slots complete in every CTA */
                TICK(5);
                ghost_table(rc, fr, gtab, thr, N_s, N8 + 8, misc);
                TICK(6);
                if (G[1] == 0.f && G[2] == 0.f && G[4] == 0.f) build_phase<true>(rc, fr, gtab, rows, tmeta, G, G[6], a_begin, A_own, N_s, N8, misc, smem_u32(s_rank));
                else build_phase<false>(rc, fr, gtab, rows, tmeta, G, G[6], a_begin, A_own, N_s, N8, misc, smem_u32(s_rank));
                __syncthreads();
                TICK(7);
                ghost_pass<T>(posb, zt, gtab, gh, N_s);          /* images again: the rebuild re-wrapped the home slots */
                __syncthreads();
                TICK(8);
            }
            if (DUMP) {
                /* list export: the list this engine would step with for the current positions goes to global memory
                 * as it lies in shared memory (the host decodes it); nothing of the state is changed */
                unsigned char *out = rc.dump + (size_t)rank * rc.dump_cta_bytes;
                const unsigned nrow = (unsigned)rc.A * (unsigned)rc.pitch * 2u / 4u;
                for (unsigned k = tid; k < nrow; k += blockDim.x) ((unsigned *)out)[k] = ((const unsigned *)rows)[k];
                unsigned *om = (unsigned *)out + nrow;
                for (int k = tid; k < rc.A; k += blockDim.x) om[k] = tmeta[k];
                for (int k = tid; k < N8; k += blockDim.x) om[rc.A + k] = k < N_s ? gtab[k] : 0u;
                if (own) om[rc.A + RES_MAX_ATOMS + 1 + tid] = (unsigned)bits_from(OWN_SMEM ? oref[tid].d : Rr.d);
                break;
            }
#ifdef TS_RES_TIMING
            const long long wt0 = clock64();
#endif
            if (last) pair_phase<T, KIND, NT1, true>(rc, pos_sa, rows_sa, tmeta, tab, fs, A_own, NT, red);
            else pair_phase<T, KIND, NT1, false>(rc, pos_sa, rows_sa, tmeta, tab, fs, A_own, NT, red);
#ifdef TS_RES_TIMING
            if ((tid & 31) == 0) {
                atomicAdd(&g_res_wprof[tid >> 5], (unsigned long long)(clock64() - wt0));
                unsigned tr = 0;
                for (int task = tid >> 5; task < (A_own + 7) / 8; task += rc.nwarps) tr += tmeta[task * 8] >> 14;
                atomicAdd(&g_res_wprof[32 + (tid >> 5)], (unsigned long long)tr);
            }
#endif
            have_ev = last;
            TICK(9);
            if (!FIRE && CL > 1) cl_arrive_relaxed(); /* this CTA no longer reads the positions of step n */
            __syncthreads();
            TICK(10);
            T f0 = 0, f1 = 0, f2 = 0, v0 = 0, v1 = 0, v2 = 0;
            if (own && (FIRE || n > 0)) {
                f0 = fs[tid]; f1 = fs[rc.A + tid]; f2 = fs[2 * rc.A + tid];
                const Q4<T> V = OWN_SMEM ? ov[tid] : Vr;
                v0 = V.a; v1 = V.b; v2 = V.c;
                if (n > 0) {
                    const T im = OWN_SMEM ? ox[tid].d : Xr.d;
                    v0 = v0 + hdt * (f0 * im); v1 = v1 + hdt * (f1 * im); v2 = v2 + hdt * (f2 * im);
                    if (!FIRE) { Q4<T> Vn; Vn.a = v0; Vn.b = v1; Vn.c = v2; Vn.d = 0; if (OWN_SMEM) ov[tid] = Vn; else Vr = Vn; }
                }
            }
            if (n > 0) n_done = n;
            if (FIRE) {
                /* the four per-system reductions, then the FIRE state machine (identical in every CTA) */
                double fsq = 0.0, P = 0.0, vv = 0.0;
                if (own) {
                    fsq = (double)f0 * (double)f0 + (double)f1 * (double)f1 + (double)f2 * (double)f2;
                    P = (double)f0 * (double)v0 + (double)f1 * (double)v1 + (double)f2 * (double)v2;
                    vv = (double)v0 * (double)v0 + (double)v1 * (double)v1 + (double)v2 * (double)v2;
                }
                double a[4];
                fire_reduce(cluster, CL, rank, fsq, P, vv, fred, cred, rc.nwarps, a);
                const bool conv = sqrt(a[0]) < fp.f_max;
                if (n == 0) {                         /* fresh system: the 0-step convergence test */
                    if (conv && fstat0 == TS_FIRE_FRESH) { if (tid == 0) fsm->status = TS_FIRE_CONVERGED; break; }
                } else {
                    const double al = fsm->alpha;     /* mixing uses alpha before its update (R21) */
                    if (!conv) {
                        if (a[1] > 0.0) {
                            const double fn = sqrt(a[3]), vn = sqrt(a[2]);
                            if (fn > 0.0 && own) {
                                const T cf = (T)(al * (vn / fn)), om = (T)(1.0 - al);
                                v0 = om * v0 + cf * f0; v1 = om * v1 + cf * f1; v2 = om * v2 + cf * f2;
                            }
                        } else if (own) { v0 = 0; v1 = 0; v2 = 0; }
                    }
                    if (own) { Q4<T> Vn; Vn.a = v0; Vn.b = v1; Vn.c = v2; Vn.d = 0; if (OWN_SMEM) ov[tid] = Vn; else Vr = Vn; }
                    __syncthreads();                  /* everybody has read the state of this step */
                    if (tid == 0) {
                        fsm->nsteps += 1;
                        if (conv) fsm->status = TS_FIRE_CONVERGED;
                        else if (a[1] > 0.0) {
                            const int np = fsm->npos + 1;
                            fsm->npos = np;
                            if (np > fp.n_min) {
                                const double nd = fsm->dt * fp.f_inc;
                                fsm->dt = nd < fp.dt_max ? nd : fp.dt_max;
                                fsm->alpha = fsm->alpha * fp.f_alpha;
                            }
                        } else {
                            fsm->dt = fsm->dt * fp.f_dec;
                            fsm->alpha = fp.alpha_start;
                            fsm->npos = 0;
                        }
                    }
                    __syncthreads();
                    if (conv) break;                  /* frozen at the first step whose new forces satisfy the criterion */
                }
            }
        }
        if (!FIRE && CL > 1 && !DUMP) cl_wait();   /* pairs the last arrive */
        if (FIRE && !have_ev && !DUMP) {                       /* stopped before the last pass: E of the final positions */
            pair_phase<T, KIND, NT1, true>(rc, pos_sa, rows_sa, tmeta, tab, fs, A_own, NT, red);
            __syncthreads();
        }
#ifdef TS_RES_TIMING
        if (tid == 0) for (int k = 0; k < 12; ++k) atomicAdd(&g_res_prof[k], (unsigned long long)prof_acc[k]);
#endif
        if (DUMP) { cluster.sync(); continue; }
        /* ---- store the system (R16): x, v at t + n dt, F(x), E, W, KE */
        double ke = 0.0;
        if (own) {
            T *x = (T *)d.pos + 3 * gi, *v = (T *)d.vel + 3 * gi, *f = (T *)d.force + 3 * gi;
            const T f0 = fs[tid], f1 = fs[rc.A + tid], f2 = fs[2 * rc.A + tid];
            const Q4<T> X = OWN_SMEM ? ox[tid] : Xr, V = OWN_SMEM ? ov[tid] : Vr;
            const T x0 = X.a, x1 = X.b, x2 = X.c, v0 = V.a, v1 = V.b, v2 = V.c;
            x[0] = x0; x[1] = x1; x[2] = x2; v[0] = v0; v[1] = v1; v[2] = v2; f[0] = f0; f[1] = f1; f[2] = f2;
            ke = 0.5 * (double)((const T *)d.mass)[gi] * d.mass_conv * ((double)v0 * (double)v0 + (double)v1 * (double)v1 + (double)v2 * (double)v2);
            if (!(fabs((double)f0) + fabs((double)f1) + fabs((double)f2) < 1e300)) atomicOr(&d.status->flags, TS_FLAG_NONFINITE);
        }
        if (rank == 0 && tid == 0) d.res_saved[s] = 1;   /* a CTA without room for its part clears it after the barrier in reduce8 */
        const double tot = reduce8(cluster, CL, rank, ke, red, cred, rc.nwarps);
        if (rank == 0 && tid < 8) {
            if (tid == 0) d.energy[s] = tot;
            if (tid == 7 && !FIRE) d.kinetic[s] = tot;
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
            atomicAdd(&d.status->res_nnz[rc.nnz_slot], (unsigned long long)misc->nnz);
            if (rank == 0) {
                atomicAdd(&d.status->res_rebuilds, (unsigned long long)misc->rebuilds);
                d.sys_step[s] = step0 + (unsigned long long)(FIRE ? n_done : n_steps);
                if (FIRE) {
                    d.f_dt[s] = fsm->dt; d.f_alpha[s] = fsm->alpha; d.f_npos[s] = fsm->npos; d.f_nsteps[s] = fsm->nsteps;
                    d.f_status[s] = fsm->status;
                    d.sys_active[s] = fsm->status == TS_FIRE_RUNNING ? 1 : 0;
                }
            }
        }
        {
#ifdef TS_RES_TIMING
            long long st0 = clock64();
#endif
            size_t share;
            unsigned char *sbase = saved_base<T>(d, rc, s, rank, share);
            save_list<T>(sbase, share, d.res_saved + s, rc.A, rc.pitch, rc.nwarps, N_s, A_own, rows, tmeta, gtab, oref, Rr, misc->nnz,
                         misc->overflow != 0, (unsigned *)red);
#ifdef TS_RES_TIMING
            __syncthreads();
            if (tid == 0) atomicAdd(&g_res_prof[13], (unsigned long long)(clock64() - st0));
#endif
        }
        cluster.sync();                               /* nobody overwrites shared state a peer still reads */
    }
}

/* ------------------------------------------------------------------ host side */
/* A ragged batch is stepped in up to four SIZE CLASSES (<= 256, <= 512, <= 1024, <= 2048 atoms), each with its own
 * launch shape and its own launch, side by side on their own streams; systems the engine cannot hold (a cell height
 * below 2 r_list, too many atoms, no shape that fits shared memory) stay with the general engine, which then runs
 * next to the resident launches on a stream of its own (ts_step.cu). */
#define RES_MAX_CLASSES 4
struct ResClass {
    ResCfg cfg;
    int fire_clusters;     /* clusters in flight of the FIRE kernel (0 = not asked yet) */
    int n, list_off;       /* systems of the class: d.res_list[list_off .. list_off + n) */
};
struct ResPlan {
    bool checked;
    int n_classes, n_general;
    ResClass cls[RES_MAX_CLASSES];
    int *cls_of_sys;       /* host [S]: class of every system, -1 = general engine */
    bool streams;
    cudaStream_t aux[RES_MAX_CLASSES + 1];
    cudaEvent_t ev_start, ev_done[RES_MAX_CLASSES + 1];
};
static ResPlan *plan_of(ts_state *st) { return (ResPlan *)st->res_plan; }

typedef void (*ResKernel)(DevState, MdConst, ResCfg, int, unsigned, ts_fire_params);

template <typename T, bool FIRE>
static ResKernel pick_kernel_t(int kind, bool nt1)
{
    if (kind == TS_LJ) return nt1 ? k_resident_md<T, TS_LJ, true, FIRE> : k_resident_md<T, TS_LJ, false, FIRE>;
    if (kind == TS_MORSE) return nt1 ? k_resident_md<T, TS_MORSE, true, FIRE> : k_resident_md<T, TS_MORSE, false, FIRE>;
    return nt1 ? k_resident_md<T, TS_SOFT_SPHERE, true, FIRE> : k_resident_md<T, TS_SOFT_SPHERE, false, FIRE>;
}
static ResKernel pick_kernel(const ts_state *st, bool fire = false)
{
    bool nt1 = st->d.n_types == 1;
    if (fire) return st->d.dtype == TS_F32 ? pick_kernel_t<float, true>(st->d.kind, nt1) : pick_kernel_t<double, true>(st->d.kind, nt1);
    return st->d.dtype == TS_F32 ? pick_kernel_t<float, false>(st->d.kind, nt1) : pick_kernel_t<double, false>(st->d.kind, nt1);
}

static unsigned up16(unsigned x) { return (x + 15u) & ~15u; }

/* Shared-memory carve for cluster size CL; returns false when it does not fit. */
static bool res_layout_n(ResCfg &c, int CL, int nmax, int need_row, int need_slots, int dtype, int n_types, int thread_div, int with_noise)
{
    size_t w = dtype == TS_F32 ? 4 : 8;
    int A = ((((nmax + CL - 1) / CL) + 7) / 8) * 8;              /* whole blocks of eight slots per CTA */
    int max_threads = (dtype == TS_F32 ? RES_MAX_THREADS : RES_MAX_THREADS_F64) / thread_div;
    if (getenv("TS_RES_MAXT")) max_threads = atoi(getenv("TS_RES_MAXT"));
    if (A > max_threads) return false;
    int pitch = 16 * ((need_row + 15) / 16);                     /* whole trips of 16 entries */
    int ntasks = A / 4, maxw = max_threads / 32;
    int passes = (ntasks + maxw - 1) / maxw;
    int nwarps = (ntasks + passes - 1) / passes;
    if (nwarps * 32 < A) nwarps = (A + 31) / 32;
    if (nwarps < 8) nwarps = 8;                                   /* ghost_table scans with eight warps */
    c.CL = CL; c.A = A; c.pitch = pitch; c.NS = need_slots; c.nwarps = nwarps;
    unsigned o = 0;
    c.o_pos = o; o += up16((unsigned)(c.NS * 4 * w));
    /* fr (rebuilds only; padded: the builder tests two candidates per trip) lives INSIDE the ghost part of the first
     * position plane: a rebuild runs between the cluster barrier of a step and the ghost refresh that follows it,
     * when no ghost slot is live; need_slots >= 2 N8 + 32 keeps it inside the array */
    c.o_fr = c.o_pos + (unsigned)(((nmax + 7) & ~7) + 8) * 16u;
    c.o_gtab = o; o += up16((unsigned)nmax * 4u);
    c.o_rows = o; o += up16((unsigned)A * (unsigned)pitch * 2u);
    c.o_fs = o; o += up16((unsigned)(3 * A * w));
    c.o_own = o; o += dtype == TS_F32 ? up16((unsigned)(12 * A * w)) : 0u;   /* fp32: x | 1/m, v, x_ref | wrap shift of the own atoms */
    c.o_meta = o; o += up16((unsigned)A * 4u);                    /* one word per atom slot of a task */
    c.noise_helpers = with_noise;
    c.o_noise = o; o += with_noise ? up16((unsigned)(3 * A * w)) : 0u;   /* Langevin kicks of the own atoms for the next step */
    c.o_pot = o; o += up16((unsigned)(n_types * n_types * (dtype == TS_F32 ? sizeof(PotEntry<float>) : sizeof(PotEntry<double>))));
    c.o_red = o; o += (unsigned)(RES_MAX_THREADS / 32) * 64u;
    c.o_cred = o; o += 8u * 64u;
    c.o_misc = o; o += up16((unsigned)(sizeof(ResMisc) + 18 * w + 8 * sizeof(float) + 4 * sizeof(unsigned)));
    c.o_fire = o; o += up16((unsigned)(sizeof(FireSm) + (RES_MAX_THREADS / 32) * 64u));
    c.o_mbar = o; o += 16u;                                       /* FULL mbarrier of the position exchange */
    c.smem = o;
    return o <= RES_SMEM_LIMIT;
}

/* with the kick buffers of the noise helpers when they fit, else without */
static bool res_layout(ResCfg &c, int CL, int nmax, int need_row, int need_slots, int dtype, int n_types, int thread_div = 1)
{
    if (res_layout_n(c, CL, nmax, need_row, need_slots, dtype, n_types, thread_div, 1)) return true;
    return res_layout_n(c, CL, nmax, need_row, need_slots, dtype, n_types, thread_div, 0);
}

/* what one system asks of a launch shape */
struct SysNeed { bool eligible; double nbar, slots; };

static SysNeed system_need(const DevState &d, const SysGeom &g, int n, float eps_rel)
{
    SysNeed r = { false, 0.0, 0.0 };
    if (n > RES_MAX_ATOMS) return r;
    double lmax = 0.0;
    for (int a = 0; a < 3; ++a)
        lmax = fmax(lmax, sqrt(g.h[3 * a] * g.h[3 * a] + g.h[3 * a + 1] * g.h[3 * a + 1] + g.h[3 * a + 2] * g.h[3 * a + 2]));
    const double rb = d.r_list + 4.0 * eps_rel * lmax;
    double images = 1.0, images2 = 1.0;                       /* E[c + 1], E[(c + 1)^2] of the image count c of an atom */
    for (int k = 0; k < 3; ++k) {
        if (!(g.hperp[k] >= 2.0 * rb)) return r;              /* more than one image within r_list possible */
        const double pk = fmin(1.0, 2.0 * rb / g.hperp[k]);   /* an atom is within rb of a face of axis k */
        images *= 1.0 + pk;
        images2 *= 1.0 + 3.0 * pk;
    }
    r.eligible = true;
    r.nbar = (double)n / g.vol * (4.0 / 3.0) * M_PI * rb * rb * rb;
    /* atoms + dummies + ghosts.  The ghosts of a bank group occupy one of eight interleaved slot sequences, so the
     * array needs 8 x the fullest group: mean + z sigma of a sum of n / 8 independent image counts, + 8 per group.
     * z = 6: 4 sigma overflowed a few of the 10^6 group fills of a 10^4-system liquid batch; a lattice written cell
     * by cell deviates systematically by ~2.5 sigma (measured on configs[1]).  An overflow is always detected and
     * flagged (TS_FLAG_NBR_OVERFLOW), never silent. */
    const double mean_c = images - 1.0, var_c = fmax(0.0, (images2 - 2.0 * images + 1.0) - mean_c * mean_c);
    const double sd_g = sqrt(var_c * n / 8.0);
    r.slots = ((n + 7) & ~7) + 8 + 8.0 * ceil(mean_c * n / 8.0 + 6.0 * sd_g + 8.0);
    return r;
}

/* launch shape of one size class: S systems of at most nmax atoms, `need` neighbours per atom, need_slots position slots */
static bool plan_class(ts_state *st, int S, int nmax, double need, double need_slots, float eps_rel, ResCfg &best_out)
{
    const DevState &d = st->d;
    double slack = st->nbr.slack >= 1.0 ? st->nbr.slack : 1.25;
    int need_row = (int)ceil(need * slack);
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    ResKernel k = pick_kernel(st);
    const char *force_cl = getenv("TS_RES_CL");
    /* launch shape for a given slot count: smallest cluster that fits and fills the chip; cost ~ waves x per-CTA work */
    auto plan = [&](double slots, int need_row, ResCfg &out, int &maxc_out, double &cost) -> bool {
        int ns = (((int)ceil(slots) + 7) / 8) * 8;
        if (getenv("TS_RES_NS")) ns = atoi(getenv("TS_RES_NS"));
        if (ns > RES_MAX_SLOTS) ns = RES_MAX_SLOTS & ~7;
        if (ns < 2 * ((nmax + 7) & ~7) + 32) ns = 2 * ((nmax + 7) & ~7) + 32;     /* room for fr inside the ghost part */
        bool have = false;
        for (int CL = 1; CL <= 8; CL *= 2) {
            ResCfg c;
            memset(&c, 0, sizeof c);
            if (force_cl && atoi(force_cl) != CL) continue;
            if (!res_layout(c, CL, nmax, need_row, ns, d.dtype, d.n_types)) continue;
            out = c; have = true;
            if ((long long)S * CL >= (nsm * 3) / 4 || c.A <= 64) break;   /* enough CTAs to occupy the chip */
        }
        if (!have) return false;
        if (cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)out.smem) != cudaSuccess) {
            cudaGetLastError();
            return false;
        }
        cudaLaunchConfig_t lc;
        memset(&lc, 0, sizeof lc);
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)out.CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        lc.gridDim = dim3((unsigned)(out.CL * S)); lc.blockDim = dim3((unsigned)(out.nwarps * 32));
        lc.dynamicSmemBytes = out.smem; lc.attrs = at; lc.numAttrs = 1;
        int maxc = 0;
        if (cudaOccupancyMaxActiveClusters(&maxc, (const void *)k, &lc) != cudaSuccess || maxc < 1) {
            cudaGetLastError();
            return false;
        }
        /* many more systems than clusters in flight, and the atoms of a CTA fit half the threads: a half-size block
         * lets two CTAs share an SM (registers were the limit), which hides the barrier latencies of small systems */
        if (S >= 2 * maxc && !getenv("TS_RES_MAXT")) {
            ResCfg h;
            memset(&h, 0, sizeof h);
            if (res_layout(h, out.CL, nmax, need_row, ns, d.dtype, d.n_types, 2) && h.nwarps < out.nwarps) {
                lc.blockDim = dim3((unsigned)(h.nwarps * 32));
                lc.dynamicSmemBytes = h.smem;
                int maxc2 = 0;
                if (cudaOccupancyMaxActiveClusters(&maxc2, (const void *)k, &lc) == cudaSuccess && maxc2 >= (3 * maxc) / 2) {
                    out = h;
                    maxc = maxc2;
                } else {
                    cudaGetLastError();
                }
            }
        }
        maxc_out = maxc;
        const int live = S < maxc ? S : maxc;
        cost = (double)((S + live - 1) / live) * ((double)out.A + 40.0 * out.CL);
        return true;
    };
    /* Row capacity.  slack x the mean count is enough for a crystal or an equilibrium liquid; a configuration with
     * ideal-gas density fluctuations (cfg4's uniformly random starting points) has Poisson counts: mean + 6 sqrt(mean)
     * + 8.  The Poisson capacity is taken whenever it does not make the launch shape costlier (cluster size, waves);
     * either way a row overflow is detected and flagged, never silent. */
    const int need_row_p = (int)ceil(fmax(need * slack, need + 6.0 * sqrt(need) + 8.0));
    ResCfg best, alt;
    int maxc = 0, maxc_p = 0;
    double cost = 0.0, cost_p = 0.0;
    const bool ok0 = plan(need_slots, need_row, best, maxc, cost), okp = plan(need_slots, need_row_p, alt, maxc_p, cost_p);
    if (!ok0 && !okp) return false;
    if (okp && (!ok0 || cost_p <= 1.05 * cost)) { best = alt; maxc = maxc_p; }
    best.eps_rel = eps_rel;
    if (getenv("TS_RES_VERBOSE"))
        fprintf(stderr, "[ts resident] CL %d A %d pitch %d NS %d warps %d smem %u clusters %d of %d systems (<= %d atoms)\n", best.CL,
                best.A, best.pitch, best.NS, best.nwarps, best.smem, S < maxc ? S : maxc, S, nmax);
    best.n_clusters = S < maxc ? S : maxc;
    best_out = best;
    return true;
}

/* Decides once per batch geometry which systems the resident engine steps, in which size classes and launch shapes.
 * Reads the cell geometry back (synchronises). */
static ResPlan *resident_plan(ts_state *st)
{
    if (!st->res_plan) st->res_plan = calloc(1, sizeof(ResPlan));
    ResPlan *p = plan_of(st);
    if (p->checked) return p;
    p->checked = true; p->n_classes = 0; p->n_general = st->d.S;
    st->res_saved_ok = false;                /* a new plan: other launch shapes, the saved lists do not fit them */
    const DevState &d = st->d;
    const int S = d.S;
    free(p->cls_of_sys);
    p->cls_of_sys = (int *)malloc(sizeof(int) * (size_t)S);
    for (int s = 0; s < S; ++s) p->cls_of_sys[s] = -1;
    if (d.n_types > TS_MAX_TYPES) return p;
    std::vector<SysGeom> geo((size_t)S);
    if (cudaMemcpy(geo.data(), d.geom, sizeof(SysGeom) * (size_t)S, cudaMemcpyDeviceToHost) != cudaSuccess) return p;
    const float eps_rel = 4e-6f;
    const int bound[RES_MAX_CLASSES] = { 256, 512, 1024, RES_MAX_ATOMS };
    std::vector<int> cls_of((size_t)S, -1), engine((size_t)S, 0), list;
    std::vector<SysNeed> need((size_t)S);
    int count[RES_MAX_CLASSES] = { 0, 0, 0, 0 };
    for (int s = 0; s < S; ++s) {
        const int n = st->h_sysoff[s + 1] - st->h_sysoff[s];
        need[(size_t)s] = system_need(d, geo[(size_t)s], n, eps_rel);
        if (!need[(size_t)s].eligible) continue;
        int c = 0;
        while (n > bound[c]) ++c;
        cls_of[(size_t)s] = c;
        count[c] += 1;
    }
    /* a class too small to fill even a few SMs joins the next larger one (its systems run in that shape) */
    for (int c = 0; c + 1 < RES_MAX_CLASSES; ++c)
        if (count[c] > 0 && count[c] < 8 && count[c + 1] > 0) {
            for (int s = 0; s < S; ++s) if (cls_of[(size_t)s] == c) cls_of[(size_t)s] = c + 1;
            count[c + 1] += count[c]; count[c] = 0;
        }
    unsigned max_smem = 0;
    for (int c = 0; c < RES_MAX_CLASSES; ++c) {
        if (!count[c]) continue;
        int nmax = 0;
        double nb = 0.0, slots = 0.0;
        for (int s = 0; s < S; ++s)
            if (cls_of[(size_t)s] == c) {
                const int n = st->h_sysoff[s + 1] - st->h_sysoff[s];
                nmax = n > nmax ? n : nmax;
                nb = fmax(nb, need[(size_t)s].nbar); slots = fmax(slots, need[(size_t)s].slots);
            }
        ResClass &k = p->cls[p->n_classes];
        memset(&k, 0, sizeof k);
        if (!plan_class(st, count[c], nmax, nb, slots, eps_rel, k.cfg)) continue;       /* its systems stay with the general engine */
        k.n = count[c]; k.list_off = (int)list.size();
        for (int s = 0; s < S; ++s)
            if (cls_of[(size_t)s] == c) { list.push_back(s); engine[(size_t)s] = 1; p->cls_of_sys[s] = p->n_classes; }
        k.cfg.syslist = d.res_list + k.list_off;
        k.cfg.n_list = k.n;
        max_smem = k.cfg.smem > max_smem ? k.cfg.smem : max_smem;
        p->n_classes += 1;
    }
    p->n_general = S - (int)list.size();
    if (p->n_classes) {
        if (cudaMemcpy(d.res_list, list.data(), sizeof(int) * list.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(d.sys_engine, engine.data(), sizeof(int) * (size_t)S, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaFuncSetAttribute((const void *)pick_kernel(st), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem) != cudaSuccess ||
            cudaFuncSetAttribute((const void *)pick_kernel(st, true), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_smem) != cudaSuccess) {
            cudaGetLastError();
            p->n_classes = 0; p->n_general = S;
            for (int s = 0; s < S; ++s) p->cls_of_sys[s] = -1;
        }
    }
    if (getenv("TS_RES_VERBOSE"))
        fprintf(stderr, "[ts resident] %d size class(es), %d of %d systems with the general engine\n", p->n_classes, p->n_general, S);
    return p;
}

/* the resident engine steps the WHOLE batch (what ts_fire_step and the list export ask) */
bool resident_supported(ts_state *st)
{
    ResPlan *p = resident_plan(st);
    return p->n_classes > 0 && p->n_general == 0;
}

/* systems the general engine has to step next to the resident launches (0: none; S: the resident engine does not apply) */
int resident_general_count(ts_state *st) { return resident_plan(st)->n_general; }

void resident_invalidate(ts_state *st)
{
    if (st->res_plan) plan_of(st)->checked = false;
    st->res_saved_ok = false;
}

/* An equal-size swap brought new cells (HOST copy, [n, 9] in the state dtype) into `slots`: the plan stays when every
 * new system still fits the launch shape of its slot's class (eligible, neighbours per row, position slots), so that an
 * in-flight run does not re-plan (a device read and occupancy queries) at every swap. */
void resident_after_swap(ts_state *st, const int32_t *slots, int n, const void *cells_host)
{
    if (!st->res_plan || !plan_of(st)->checked) return;
    ResPlan *p = plan_of(st);
    const DevState &d = st->d;
    const double slack = st->nbr.slack >= 1.0 ? st->nbr.slack : 1.25;
    for (int k = 0; k < n; ++k) {
        const int s = slots[k], c = p->cls_of_sys ? p->cls_of_sys[s] : -1;
        SysGeom g;
        for (int e = 0; e < 9; ++e)
            g.h[e] = d.dtype == TS_F32 ? (double)((const float *)cells_host)[9 * (size_t)k + e] : ((const double *)cells_host)[9 * (size_t)k + e];
        const double *h = g.h;
        const double c00 = h[4] * h[8] - h[5] * h[7], c01 = h[5] * h[6] - h[3] * h[8], c02 = h[3] * h[7] - h[4] * h[6];
        const double det = h[0] * c00 + h[1] * c01 + h[2] * c02;
        if (!(fabs(det) > 0.0)) { p->checked = false; st->res_saved_ok = false; return; }
        const double id = 1.0 / det;
        const double hinv[9] = { c00 * id, (h[2] * h[7] - h[1] * h[8]) * id, (h[1] * h[5] - h[2] * h[4]) * id,
                                 c01 * id, (h[0] * h[8] - h[2] * h[6]) * id, (h[2] * h[3] - h[0] * h[5]) * id,
                                 c02 * id, (h[1] * h[6] - h[0] * h[7]) * id, (h[0] * h[4] - h[1] * h[3]) * id };
        g.vol = fabs(det);
        for (int a = 0; a < 3; ++a) g.hperp[a] = 1.0 / sqrt(hinv[a] * hinv[a] + hinv[3 + a] * hinv[3 + a] + hinv[6 + a] * hinv[6 + a]);
        const int natoms = st->h_sysoff[s + 1] - st->h_sysoff[s];
        const SysNeed need = system_need(d, g, natoms, 4e-6f);
        bool fits = c >= 0 ? need.eligible : !need.eligible;            /* a general-engine slot stays one only if it still has to */
        if (c >= 0 && fits) {
            const ResCfg &cfg = p->cls[c].cfg;
            fits = (int)ceil(need.nbar * slack) <= cfg.pitch && need.slots <= (double)cfg.NS;
        }
        if (!fits) { p->checked = false; st->res_saved_ok = false; return; }
    }
}

void resident_free(ts_state *st)
{
    if (st->res_plan) {
        ResPlan *p = plan_of(st);
        if (p->streams) {
            for (int k = 0; k <= RES_MAX_CLASSES; ++k) { cudaStreamDestroy(p->aux[k]); cudaEventDestroy(p->ev_done[k]); }
            cudaEventDestroy(p->ev_start);
        }
        free(p->cls_of_sys);
    }
    free(st->res_plan);
    st->res_plan = nullptr;
}

static bool plan_streams(ResPlan *p)
{
    if (p->streams) return true;
    for (int k = 0; k <= RES_MAX_CLASSES; ++k)
        if (cudaStreamCreateWithFlags(&p->aux[k], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&p->ev_done[k], cudaEventDisableTiming) != cudaSuccess) return false;
    if (cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming) != cudaSuccess) return false;
    p->streams = true;
    return true;
}

/* The stream the general engine uses next to the resident launches of this call (fork from q), and the join. */
cudaStream_t resident_fork_general(ts_state *st, cudaStream_t q)
{
    ResPlan *p = resident_plan(st);
    if (!plan_streams(p)) return q;
    cudaEventRecord(p->ev_start, q);
    cudaStreamWaitEvent(p->aux[RES_MAX_CLASSES], p->ev_start, 0);
    return p->aux[RES_MAX_CLASSES];
}
void resident_join_general(ts_state *st, cudaStream_t q)
{
    ResPlan *p = resident_plan(st);
    if (!p->streams) return;
    cudaEventRecord(p->ev_done[RES_MAX_CLASSES], p->aux[RES_MAX_CLASSES]);
    cudaStreamWaitEvent(q, p->ev_done[RES_MAX_CLASSES], 0);
}

/* one launch per size class: the first on the caller's stream, the others on their own streams, joined at the end */
static ts_status launch_classes(ts_state *st, bool fire, const MdConst &c, int n_steps, unsigned want, const ts_fire_params &fp,
                                cudaStream_t q)
{
    ResPlan *p = resident_plan(st);
    if (p->n_classes < 1) return TS_ERR_UNSUPPORTED;
    if (p->n_classes > 1 && !plan_streams(p)) return TS_ERR_CUDA;
    ResKernel k = pick_kernel(st, fire);
    st->res_nnz_slot ^= 1;                    /* this call adds into the slot the last call cleared */
    /* saved lists: valid per system (res_saved) unless something invalidated them for the whole batch since the last launch */
    if (!st->res_saved_ok) TS_CUDA_OK(st, cudaMemsetAsync(st->d.res_saved, 0, sizeof(int) * (size_t)st->d.S, q));
    st->res_saved_ok = true;
    if (p->n_classes > 1) TS_CUDA_OK(st, cudaEventRecord(p->ev_start, q));
    for (int ci = 0; ci < p->n_classes; ++ci) {
        ResClass &cl = p->cls[ci];
        ResCfg cfg = cl.cfg;
        cfg.nnz_slot = st->res_nnz_slot & 1;
        cudaStream_t sq = ci == 0 ? q : p->aux[ci];
        if (ci > 0) TS_CUDA_OK(st, cudaStreamWaitEvent(sq, p->ev_start, 0));
        cudaLaunchConfig_t lc;
        memset(&lc, 0, sizeof lc);
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)cfg.CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        lc.blockDim = dim3((unsigned)(cfg.nwarps * 32));
        lc.dynamicSmemBytes = cfg.smem; lc.stream = sq; lc.attrs = at; lc.numAttrs = 1;
        if (fire) {
            if (cl.fire_clusters == 0) {               /* the FIRE variant has its own register count and occupancy */
                lc.gridDim = dim3((unsigned)(cfg.CL * cl.n));
                int maxc = 0;
                if (cudaOccupancyMaxActiveClusters(&maxc, (const void *)k, &lc) != cudaSuccess || maxc < 1) {
                    cudaGetLastError();
                    return TS_ERR_UNSUPPORTED;
                }
                cl.fire_clusters = cl.n < maxc ? cl.n : maxc;
            }
            cfg.n_clusters = cl.fire_clusters;
        }
        lc.gridDim = dim3((unsigned)(cfg.CL * cfg.n_clusters));
        TS_CUDA_OK(st, cudaLaunchKernelEx(&lc, k, st->d, c, cfg, n_steps, want, fp));
        st->launches += 1;
        if (ci > 0) {
            TS_CUDA_OK(st, cudaEventRecord(p->ev_done[ci], sq));
            TS_CUDA_OK(st, cudaStreamWaitEvent(q, p->ev_done[ci], 0));
        }
    }
    st->last_engine = p->n_general ? 2 : 1;
    return TS_OK;
}

/* the resident share of an MD call: every size class; the general engine steps the other systems (ts_step.cu) */
ts_status resident_md(ts_state *st, const MdConst &c, int n_steps, unsigned want, cudaStream_t q)
{
    ts_fire_params nofire;
    memset(&nofire, 0, sizeof nofire);
    return launch_classes(st, false, c, n_steps, want, nofire, q);
}

/* FIRE relaxation inside the resident engine: the same kernel in FIRE mode (per-system dt, the four reductions and
 * the state machine after every step, finished systems skipped bit-unchanged); whole batches only. */
ts_status resident_fire(ts_state *st, const ts_fire_params &fp, int n_steps, cudaStream_t q)
{
    if (!resident_supported(st)) return TS_ERR_UNSUPPORTED;
    MdConst c;
    memset(&c, 0, sizeof c);
    c.integrator = TS_NVE;
    return launch_classes(st, true, c, n_steps, (unsigned)TS_WANT_ENERGY, fp, q);
}

/* ------------------------------------------------------------------ list export (ts.h: ts_get_resident_neighbors)
 * Runs the engine's own rebuild for the current positions of one system and decodes the list on the host: the list
 * the benched engine steps with becomes checkable against the oracle's pair set (it is a SUPERSET list: radius
 * r_list + eps_rel x the longest cell edge, in fixed-point fractions). */
extern "C" ts_status ts_get_resident_neighbors(ts_state *st, int32_t system, int64_t *off, int32_t *j_out, int8_t *shift,
                                               int64_t cap, int64_t *nnz, void *stream)
{
    if (!st || !off || !nnz || system < 0 || system >= st->d.S) return TS_ERR_INVALID_ARG;
    if (st->seen_flags) return TS_ERR_STICKY;
    ResPlan *pl = resident_plan(st);
    if (pl->cls_of_sys[system] < 0) return TS_ERR_UNSUPPORTED;
    cudaStream_t q = (cudaStream_t)stream;
    ResCfg cfg = pl->cls[pl->cls_of_sys[system]].cfg;
    cfg.syslist = nullptr; cfg.n_list = st->d.S;
    const int a0 = st->h_sysoff[system], N_s = st->h_sysoff[system + 1] - a0, N8 = (N_s + 7) & ~7, CL = cfg.CL;
    const size_t nrow = (size_t)cfg.A * cfg.pitch * 2 / 4;
    const size_t cta_words = nrow + (size_t)cfg.A + RES_MAX_ATOMS + 1 + (size_t)cfg.A;
    if (cta_words * 4 * CL > (size_t)st->d.nbr_cap * 4) return TS_ERR_WORKSPACE_TOO_SMALL;   /* the pair region is the dump area */
    cfg.dump = (unsigned char *)st->d.nbr;
    cfg.dump_sys = system;
    cfg.dump_cta_bytes = (unsigned)(cta_words * 4);
    cfg.n_clusters = 1;
    st->list_built = false;                                 /* the general engine's list lived there */
    st->res_saved_ok = false;                               /* and so did the saved lists of the resident engine */
    ResKernel k = st->d.dtype == TS_F32 ? (ResKernel)k_resident_md<float, TS_LJ, false, false, true>
                                        : (ResKernel)k_resident_md<double, TS_LJ, false, false, true>;   /* the build does not depend on the potential */
    if (cudaFuncSetAttribute((const void *)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem) != cudaSuccess) {
        cudaGetLastError();
        return TS_ERR_CUDA;
    }
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.gridDim = dim3((unsigned)CL); lc.blockDim = dim3((unsigned)(cfg.nwarps * 32));
    lc.dynamicSmemBytes = cfg.smem; lc.stream = q; lc.attrs = at; lc.numAttrs = 1;
    MdConst c;
    memset(&c, 0, sizeof c);
    c.integrator = TS_NVE; c.dt = 1.0; c.hdt = 0.5;
    ts_fire_params nofire;
    memset(&nofire, 0, sizeof nofire);
    DevState dd = st->d;
    /* the kernel walks systems cid, cid + n_clusters, ...: start the one cluster at `system` by shifting the batch view */
    TS_CUDA_OK(st, cudaLaunchKernelEx(&lc, k, dd, c, cfg, 0, 0u, nofire));
    st->launches += 1;
    std::vector<unsigned> buf(cta_words * (size_t)CL);
    TS_CUDA_OK(st, cudaStreamSynchronize(q));
    TS_CUDA_OK(st, cudaMemcpy(buf.data(), st->d.nbr, buf.size() * 4, cudaMemcpyDeviceToHost));
    const int A_s = ((((N_s + CL - 1) / CL) + 7) >> 3) << 3;
    auto unhash = [&](int t) {
        const unsigned b = (unsigned)t >> 3;
        const unsigned h = (int)b == (N8 >> 3) - 1 ? 0u : (b * 0x9E3779B1u) >> 29;
        return (t & ~7) | (int)(((unsigned)t - h) & 7u);
    };
    /* ghost slot -> (slot of the atom, image subset, signs); wrap shift of every atom */
    const unsigned *g0 = buf.data() + nrow + cfg.A;          /* gtab as rank 0 built it (identical in every CTA) */
    std::vector<int> gsrc((size_t)cfg.NS, -1), gm((size_t)cfg.NS, 0), gsg((size_t)cfg.NS, 0);
    for (int t = 0; t < N_s; ++t) {
        const unsigned e = g0[t], act = (e >> 16) & 7u, sg = (e >> 19) & 7u;
        unsigned slot = e & 0xffffu;
        for (unsigned m = 1; m < 8; ++m)
            if ((m & ~act) == 0u) {
                if (slot < (unsigned)cfg.NS) { gsrc[slot] = t; gm[slot] = (int)m; gsg[slot] = (int)sg; }
                slot += 8u;
            }
    }
    std::vector<int> wpack((size_t)N_s, 0);
    for (int r = 0; r < CL; ++r)
        for (int al = 0; al < A_s && r * A_s + al < N_s; ++al)
            wpack[(size_t)(r * A_s + al)] = (int)buf[(size_t)r * cta_words + nrow + cfg.A + RES_MAX_ATOMS + 1 + al];
    auto wk = [&](int atom, int k) { return (int)(signed char)((wpack[(size_t)atom] >> (8 * k)) & 0xff); };
    int64_t n = 0;
    off[0] = 0;
    for (int i = 0; i < N_s; ++i) {
        const int r = i / A_s, al = i - r * A_s, task = al >> 3, a8 = al & 7;
        const unsigned *cta = buf.data() + (size_t)r * cta_words;
        const unsigned meta = cta[nrow + al];
        const int nt = (int)(meta >> 14);
        for (int t = 0; t < nt; ++t)
            for (int l4 = 0; l4 < 4; ++l4)
                for (int kk = 0; kk < 4; ++kk) {
                    const unsigned word = cta[((size_t)task * cfg.pitch * 16 + (size_t)t * 256 + a8 * 32 + l4 * 8 + (kk >> 1) * 4) / 4];
                    const int slot = (int)((kk & 1) ? word >> 18 : word & 0x3fffu);
                    if (slot >= N8 && slot < N8 + 8) continue;                /* padding dummy */
                    int src = slot, S[3] = { 0, 0, 0 };
                    if (slot >= N8 + 8) {
                        src = slot < cfg.NS ? gsrc[(size_t)slot] : -1;
                        if (src < 0) return TS_ERR_INVALID_ARG;                /* an entry that names no slot: cannot happen */
                        for (int c3 = 0; c3 < 3; ++c3)
                            if ((gm[(size_t)slot] >> c3) & 1) S[c3] = ((gsg[(size_t)slot] >> c3) & 1) ? 1 : -1;
                    }
                    const int jj = unhash(src);
                    if (j_out && shift) {
                        if (n >= cap) return TS_ERR_WORKSPACE_TOO_SMALL;
                        j_out[n] = a0 + jj;
                        /* stored positions: x_j - x_i + S.h with S = S_image - wrap_j + wrap_i (R6) */
                        for (int c3 = 0; c3 < 3; ++c3) shift[3 * n + c3] = (int8_t)(S[c3] - wk(jj, c3) + wk(i, c3));
                    }
                    ++n;
                }
        off[i + 1] = n;
    }
    *nnz = n;
    return TS_OK;
}

/* debugging aid (only with -DTS_RES_TIMING): summed cycles per phase of warp 0 over all CTAs, then reset */
extern "C" int ts_debug_resident_profile(unsigned long long *out16)
{
#ifdef TS_RES_TIMING
    unsigned long long z[16] = { 0 };
    if (cudaMemcpyFromSymbol(out16, g_res_prof, sizeof z) != cudaSuccess) return 1;
    cudaMemcpyToSymbol(g_res_prof, z, sizeof z);
    if (getenv("TS_RES_WPROF")) {
        unsigned long long w[64], zz[64] = { 0 };
        cudaMemcpyFromSymbol(w, g_res_wprof, sizeof w);
        cudaMemcpyToSymbol(g_res_wprof, zz, sizeof zz);
        for (int k = 0; k < 32; ++k) fprintf(stderr, "warp %2d pair cycles %llu trips %llu\n", k, w[k], w[32 + k]);
    }
    return 0;
#else
    (void)out16;
    return 2;
#endif
}
