/*
 * ts_pair.cu -- pair-potential kernel over the CSR Verlet list.
 *
 *   F_i = sum_{(i,j,S)} V'(r) r/|r|,  r = x~_j - x~_i + S.h      (r points i -> j)
 *   E_s = 1/2 sum V(r) (shifted by V(rc) when shift_energy),  W_s = -1/2 sum V'(r) (r (x) r)/r
 * Pairs with r^2 >= rc^2 that sit in the Verlet shell contribute exactly 0 (R9).
 *
 * Mapping: LPA = 8 lanes per atom read the atom's CSR row in 32-byte pieces (coalesced sector
 * reads), gather x~_j as one float4 / double4 from the pos4 array (L1/L2 resident per system),
 * xor-shuffle over the 8 lanes, then the per-system sums of E and W in fp64 in a fixed order
 * (ts_sys_store: one partial per warp and system; k_sum_ev, launched next, adds them in slot
 * order): bitwise reproducible from run to run, no floating-point atomics.
 */
#include "ts_internal.cuh"
#include "ts_pot.cuh"

#define LPA 8

template <typename T>
__device__ __forceinline__ int type_of(const typename Vec4<T>::type &q)
{
    if (sizeof(T) == 4) return __float_as_int((float)q.w);
    return (int)__double_as_longlong((double)q.w);
}

/* EV = 0: forces only; 1: + energy (FIRE: the virial accumulators would cost 12 registers of occupancy); 2: + virial */
template <typename T, int KIND, int EV>
__global__ void __launch_bounds__(256, 3) k_pair(DevState d, int masked)
{
    typedef typename Vec4<T>::type V4;
    const unsigned FULL = 0xffffffffu;
    long long gid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long i = gid / LPA;
    int sub = threadIdx.x & (LPA - 1);
    bool valid = i < d.N;
    int s = valid ? d.sysidx[i] : -1;
    bool act = valid && !(masked && !d.sys_active[s]) && !ts_skip(d, s) && d.nbr_len[s] >= 0;
    const V4 *pos4 = (const V4 *)d.pos4;
    const PotEntry<T> *tab = (const PotEntry<T> *)d.pot;
    int nt = d.n_types;
    T fx = 0, fy = 0, fz = 0, e = 0, w0 = 0, w1 = 0, w2 = 0, w3 = 0, w4 = 0, w5 = 0;
    if (act) {
        const T *h = (const T *)d.hT + 9 * (size_t)s;
        T h0 = __ldg(h), h1 = __ldg(h + 1), h2 = __ldg(h + 2), h3 = __ldg(h + 3), h4 = __ldg(h + 4),
          h5 = __ldg(h + 5), h6 = __ldg(h + 6), h7 = __ldg(h + 7), h8 = __ldg(h + 8);
        V4 xi = pos4[i];
        int ti = type_of<T>(xi);
        int a0 = d.sysoff[s];
        const unsigned *row = d.nbr + d.nbr_off[i];
        int cnt = d.nbr_cnt[i];
        PotEntry<T> pe = tab[ti * nt];
#pragma unroll 2
        for (int k = sub; k < cnt; k += LPA) {
            unsigned en = __ldg(row + k);
            int j = (int)(en & TS_J_MASK);
            int s0, s1, s2;
            ts_unpack_shift(en, s0, s1, s2);
            V4 xj = pos4[a0 + j];
            T f0 = (T)s0, f1 = (T)s1, f2 = (T)s2;
            T rx = (xj.x - xi.x) + (f0 * h0 + f1 * h3 + f2 * h6);
            T ry = (xj.y - xi.y) + (f0 * h1 + f1 * h4 + f2 * h7);
            T rz = (xj.z - xi.z) + (f0 * h2 + f1 * h5 + f2 * h8);
            T r2 = rx * rx + ry * ry + rz * rz;
            if (nt > 1) pe = tab[ti * nt + type_of<T>(xj)];
            const bool in = r2 < pe.rc2;     /* pairs in the Verlet shell contribute exactly 0 (R9) */
            if (EV) {
                T V, g;
                pot_eval<T, KIND>(pe, r2, V, g);
                g = in ? g : (T)0; V = in ? V : (T)0;
                fx += g * rx; fy += g * ry; fz += g * rz;
                e += V;
                if (EV == 2) {
                    T gx = g * rx, gy = g * ry;
                    w0 += gx * rx; w1 += gx * ry; w2 += gx * rz;
                    w3 += gy * ry; w4 += gy * rz; w5 += g * rz * rz;
                }
            } else {
                T g = pot_force<T, KIND>(pe, r2);
                g = in ? g : (T)0;
                fx += g * rx; fy += g * ry; fz += g * rz;
            }
        }
    }
#pragma unroll
    for (int o = 1; o < LPA; o <<= 1) {
        fx += __shfl_xor_sync(FULL, fx, o);
        fy += __shfl_xor_sync(FULL, fy, o);
        fz += __shfl_xor_sync(FULL, fz, o);
    }
    if (act && sub == 0) {
        T *f = (T *)d.force + 3 * i;
        f[0] = fx; f[1] = fy; f[2] = fz;
        if (!(fabs((double)fx) + fabs((double)fy) + fabs((double)fz) < 1e300))
            atomicOr(&d.status->flags, TS_FLAG_NONFINITE);
    }
    if (EV) {
        /* fp64 from here on (R31): E = 1/2 sum V, W = -1/2 sum g r (x) r */
        constexpr int NQ = EV == 2 ? 7 : 1;
        double acc[7] = { 0.5 * (double)e, -0.5 * (double)w0, -0.5 * (double)w1, -0.5 * (double)w2,
                          -0.5 * (double)w3, -0.5 * (double)w4, -0.5 * (double)w5 };
        /* the eight lanes of an atom first (fixed tree), then the per-system partials in fixed order (ts_sys_store): the
         * results do not depend on which warp finishes first */
#pragma unroll
        for (int q = 0; q < NQ; ++q)
#pragma unroll
            for (int o = 1; o < LPA; o <<= 1) acc[q] += __shfl_xor_sync(FULL, acc[q], o);
        double part[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) part[q] = sub == 0 ? acc[q] : 0.0;
        ts_sys_store<NQ, LPA>(d, act ? s : -1, part);            /* k_sum_ev adds the slots of every system */
    }
}

/* E / W of the systems k_pair has just evaluated: one warp per system adds the partials k_pair stored, in slot order */
__global__ void k_sum_ev(DevState d, int masked, unsigned want)
{
    const int s = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5);
    if (s >= d.S) return;
    if (masked && !d.sys_active[s]) return;
    if (ts_skip(d, s)) return;
    if (d.nbr_len[s] < 0) return;
    const int lane = threadIdx.x & 31;
    if ((want & TS_WANT_VIRIAL) && d.virial) {
        double tot[7];
        ts_sys_total<7>(d, s, LPA, tot);
        if (lane == 0) {
            d.energy[s] = tot[0];
            double *W = d.virial + 9 * (size_t)s;
            W[0] = tot[1]; W[1] = tot[2]; W[2] = tot[3];
            W[3] = tot[2]; W[4] = tot[4]; W[5] = tot[5];
            W[6] = tot[3]; W[7] = tot[5]; W[8] = tot[6];
        }
    } else {
        double tot[1];
        ts_sys_total<1>(d, s, LPA, tot);
        if (lane == 0) d.energy[s] = tot[0];
    }
}

template <typename T, int KIND>
static void launch_pair_k(ts_state *st, unsigned want, bool masked, cudaStream_t q)
{
    DevState d = st->d;
    long long nthreads = d.N * LPA;
    unsigned nb = (unsigned)((nthreads + 255) / 256);
    if (want) {
        if (!(want & TS_WANT_VIRIAL)) d.virial = nullptr;
        if (d.virial) k_pair<T, KIND, 2><<<nb, 256, 0, q>>>(d, masked ? 1 : 0);
        else k_pair<T, KIND, 1><<<nb, 256, 0, q>>>(d, masked ? 1 : 0);
        k_sum_ev<<<(d.S + 3) / 4, 128, 0, q>>>(d, masked ? 1 : 0, want);
        st->launches += 2;
    } else {
        k_pair<T, KIND, 0><<<nb, 256, 0, q>>>(d, masked ? 1 : 0);
        st->launches += 1;
    }
}

void launch_pair(ts_state *st, unsigned want, bool masked, cudaStream_t q)
{
    int kind = st->d.kind;
    if (st->d.dtype == TS_F32) {
        if (kind == TS_LJ) launch_pair_k<float, TS_LJ>(st, want, masked, q);
        else if (kind == TS_MORSE) launch_pair_k<float, TS_MORSE>(st, want, masked, q);
        else launch_pair_k<float, TS_SOFT_SPHERE>(st, want, masked, q);
    } else {
        if (kind == TS_LJ) launch_pair_k<double, TS_LJ>(st, want, masked, q);
        else if (kind == TS_MORSE) launch_pair_k<double, TS_MORSE>(st, want, masked, q);
        else launch_pair_k<double, TS_SOFT_SPHERE>(st, want, masked, q);
    }
}
