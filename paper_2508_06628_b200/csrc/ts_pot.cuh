/*
 * ts_pot.cuh -- pair-potential arithmetic shared by the two stepping engines of libts (CUDA path
 * only): V (energy-shifted) and g = V'(r)/r for LJ / Morse / soft sphere.
 */
#pragma once
#include "ts_internal.cuh"

template <typename T> __device__ __forceinline__ T t_exp(T x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return __expf(x); }   /* ex2.approx: ~2 ulp on |x| < 10, inside the fp32 tolerances */
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }
template <typename T> __device__ __forceinline__ T t_pow(T x, T a);
template <> __device__ __forceinline__ float t_pow<float>(float x, float a) { return powf(x, a); }
template <> __device__ __forceinline__ double t_pow<double>(double x, double a) { return pow(x, a); }
template <typename T> __device__ __forceinline__ T t_sqrt(T x);
template <> __device__ __forceinline__ float t_sqrt<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double t_sqrt<double>(double x) { return sqrt(x); }

/* 1/x and 1/sqrt(x): one MUFU on the fp32 path (about 1 ulp, far inside the fp32 tolerances of
 * BASELINE.json:north_star); fp64: IEEE divide for 1/x, the <= 1 ulp library rsqrt for 1/sqrt(x) (the fp64
 * tolerances, 1e-12 relative on E and 1e-10 absolute on F, leave four orders of magnitude of room). */
template <typename T> __device__ __forceinline__ T t_rcp(T x);
template <> __device__ __forceinline__ float t_rcp<float>(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
template <> __device__ __forceinline__ double t_rcp<double>(double x) { return 1.0 / x; }
template <typename T> __device__ __forceinline__ T t_rsqrt(T x);
template <> __device__ __forceinline__ float t_rsqrt<float>(float x) { return rsqrtf(x); }
template <> __device__ __forceinline__ double t_rsqrt<double>(double x) { return rsqrt(x); }   /* CUDA math rsqrt: <= 1 ulp, no IEEE divide */

/* V (shifted) and g = V'(r)/r.  Branch-free for LJ and Morse: the caller masks r^2 >= rc^2. */
template <typename T, int KIND>
__device__ __forceinline__ void pot_eval(const PotEntry<T> &pe, T r2, T &V, T &g)
{
    if (KIND == TS_LJ) {
        T ir2 = t_rcp<T>(r2);
        T ir6 = ir2 * ir2 * ir2;
        T a = pe.c0 * ir6 * ir6, b = pe.c1 * ir6;
        V = (a - b) - pe.vshift;
        g = ((T)6 * b - (T)12 * a) * ir2;
    } else if (KIND == TS_MORSE) {
        T ir = t_rsqrt<T>(r2);
        T r = r2 * ir;
        T e = t_exp<T>(-pe.p1 * (r - pe.p2));
        T om = (T)1 - e;
        V = pe.p0 * (om * om - (T)1) - pe.vshift;
        g = pe.c0 * om * e * ir;
    } else {
        T ir = t_rsqrt<T>(r2);
        T r = r2 * ir;
        T u = (T)1 - r * pe.c2;
        if (u <= (T)0) { V = (T)0; g = (T)0; return; }
        T um1;                       /* u^(alpha-1) */
        T al = pe.p2;
        if (al == (T)2) um1 = u;
        else if (al == (T)1) um1 = (T)1;
        else if (al == (T)3) um1 = u * u;
        else um1 = t_pow<T>(u, al - (T)1);
        V = pe.c0 * um1 * u - pe.vshift;
        g = -pe.c1 * um1 * ir;
    }
}

/* force-only variant of the LJ arithmetic (no energy): g = ir2 ir6 (6 c1 - 12 c0 ir6) */
template <typename T, int KIND>
__device__ __forceinline__ T pot_force(const PotEntry<T> &pe, T r2)
{
    if (KIND == TS_LJ) {
        T ir2 = t_rcp<T>(r2);
        T ir6 = ir2 * ir2 * ir2;
        return (ir6 * ir2) * ((T)6 * pe.c1 - ((T)12 * pe.c0) * ir6);
    } else {
        T V, g;
        pot_eval<T, KIND>(pe, r2, V, g);
        return g;
    }
}
