// CC_LADDER_ALGO_SIMPLE: a slow, scalar-FMA device path kept as an on-GPU cross-check of the fused kernel
// (it is NOT a fallback: the default path never routes here).  It follows the paper's own order for a chunk of
// (a,b) pairs: build the integral slab into a workspace chunk, contract it with t.
#pragma once
#include "ladder_common.cuh"

namespace ccl {

// Vc[p][c][d] = sum_P L[P,a_p,c] L[P,b_p,d] for the pairs p in [pair0, pair0+npairs)   (Eq. 5)
__global__ void simple_eri_chunk(const double *__restrict__ L, double *__restrict__ Vc, int v, int x, long long pair0,
                                 int npairs)
{
    const long long vv = (long long)v * v;
    const long long total = (long long)npairs * vv;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long pl = e / vv;
        const int c = (int)((e % vv) / v), d = (int)(e % v);
        const long long pair = pair0 + pl;
        const int a = (int)(pair / v), b = (int)(pair % v);
        double s = 0.0;
        for (int P = 0; P < x; ++P)
            s = fma(L[((size_t)P * v + a) * v + c], L[((size_t)P * v + b) * v + d], s);
        Vc[e] = s;
    }
}

// R[ij][a_p][b_p] += sum_cd t[ij][c][d] Vc[p][c][d]; one warp per (ij, p)                (Eq. 6)
__global__ void simple_contract_chunk(const double *__restrict__ t, const double *__restrict__ Vc, double *__restrict__ R,
                                      long long oo, int v, long long pair0, int npairs)
{
    const long long vv = (long long)v * v;
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long w = warp; w < oo * npairs; w += nwarps) {
        const long long ij = w / npairs;
        const long long pl = w % npairs;
        const double *tp = t + (size_t)ij * vv;
        const double *vp = Vc + (size_t)pl * vv;
        double s = 0.0;
        for (long long k = lane; k < vv; k += 32) s = fma(tp[k], vp[k], s);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if (lane == 0) R[(size_t)ij * vv + (size_t)(pair0 + pl)] += s;
    }
}

}  // namespace ccl
