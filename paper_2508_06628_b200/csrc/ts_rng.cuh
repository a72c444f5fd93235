/*
 * ts_rng.cuh -- counter-based Philox4x32-10 and the Box-Muller normals of the Langevin O-step
 * (SURVEY.md 8(c) O5, R18, R19), shared by the two stepping engines of libts (CUDA path only).
 */
#pragma once
#include <cuda_runtime.h>

/* ------------------------------------------------------------------ Philox4x32-10 (O5) */
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3,
                                              unsigned k0, unsigned k1, unsigned out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__device__ __forceinline__ void normals3(const unsigned w[4], double xi[3])
{
    const double s = 1.0 / 4294967296.0;
    double u0 = ((double)w[0] + 0.5) * s, u1 = ((double)w[1] + 0.5) * s;
    double u2 = ((double)w[2] + 0.5) * s, u3 = ((double)w[3] + 0.5) * s;
    double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
    double sn, cs, sn2, cs2;
    sincospi(2.0 * u1, &sn, &cs);
    sincospi(2.0 * u3, &sn2, &cs2);
    xi[0] = r0 * cs; xi[1] = r0 * sn; xi[2] = r1 * cs2;
}
/* fp32 runs (R19: log / sin / cos may be evaluated in fp32): the hardware approximations (MUFU.LG2, MUFU.SQRT,
 * MUFU.SIN / COS on an argument reduced to [-pi, pi)) -- absolute error ~1e-6 on a unit normal, far below the fp32
 * rounding of the velocity update it feeds; no trajectory parity is asked of fp32 runs. */
__device__ __forceinline__ void normals3(const unsigned w[4], float xi[3])
{
    const float s = 2.3283064365386963e-10f;
    const float u0 = ((float)w[0] + 0.5f) * s, u1 = ((float)w[1] + 0.5f) * s;
    const float u2 = ((float)w[2] + 0.5f) * s, u3 = ((float)w[3] + 0.5f) * s;
    float r0, r1;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r0) : "f"(-1.3862943611198906f * __log2f(u0)));   /* -2 ln u = -2 ln2 lg2 u */
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r1) : "f"(-1.3862943611198906f * __log2f(u2)));
    const float t1 = fmaf(6.283185307179586f, u1, -3.141592653589793f);                      /* cos(t + pi) = -cos t */
    const float t3 = fmaf(6.283185307179586f, u3, -3.141592653589793f);
    xi[0] = -r0 * __cosf(t1); xi[1] = -r0 * __sinf(t1); xi[2] = -r1 * __cosf(t3);
}
