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
__device__ __forceinline__ void normals3(const unsigned w[4], float xi[3])
{
    const float s = 2.3283064365386963e-10f;
    float u0 = ((float)w[0] + 0.5f) * s, u1 = ((float)w[1] + 0.5f) * s;
    float u2 = ((float)w[2] + 0.5f) * s, u3 = ((float)w[3] + 0.5f) * s;
    float r0 = sqrtf(-2.0f * logf(u0)), r1 = sqrtf(-2.0f * logf(u2));
    float sn, cs, sn2, cs2;
    sincospif(2.0f * u1, &sn, &cs);
    sincospif(2.0f * u3, &sn2, &cs2);
    xi[0] = r0 * cs; xi[1] = r0 * sn; xi[2] = r1 * cs2;
}

