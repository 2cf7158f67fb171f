// Steps a0 and a5 of the hot path in split (t+/t-) mode (reading 10; not in the paper, north_star):
//   a0  pack     T+[ij,c,d] = t[ij,c,d] + t[ij,d,c],   T-[ij,c,d] = t[ij,c,d] - t[ij,d,c]      (full v x v squares)
//   a5  unpack   R[ij,a,b] += W+[ij,a,b] + W-[ij,a,b]           where blk(a) <= blk(b)
//                R[ij,a,b] += W+[ij,b,a] - W-[ij,b,a]           where blk(a) >  blk(b)          (blk = index / TAB)
// W+- are what the fused kernel accumulated for the block pairs A <= B (R+ and R- of reading 10).  Both kernels are
// HBM-bound tiled transposes: 32 x 32 tiles through shared memory, every global access coalesced.
#pragma once
#include "ladder_common.cuh"

namespace ccl {

constexpr int kTT = 32;   // transpose tile edge

__global__ void __launch_bounds__(256) split_pack_kernel(const double *__restrict__ t, double *__restrict__ Tp,
                                                         double *__restrict__ Tm, long long oo, int v)
{
    __shared__ double tr[kTT][kTT + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
    const int c0 = blockIdx.y * kTT, d0 = blockIdx.x * kTT;
    const size_t vv = (size_t)v * v;
    for (long long ij = blockIdx.z; ij < oo; ij += gridDim.z) {
        const double *m = t + (size_t)ij * vv;
        // tr[dl][cl] = t[d0+dl][c0+cl]  (rows of the mirrored tile, read coalesced along c)
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {
            const int d = d0 + r, c = c0 + tx;
            tr[r][tx] = (d < v && c < v) ? m[(size_t)d * v + c] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {
            const int c = c0 + r, d = d0 + tx;
            if (c < v && d < v) {
                const double tcd = m[(size_t)c * v + d], tdc = tr[tx][r];
                Tp[(size_t)ij * vv + (size_t)c * v + d] = tcd + tdc;
                Tm[(size_t)ij * vv + (size_t)c * v + d] = tcd - tdc;
            }
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) split_unpack_kernel(const double *__restrict__ Wp, const double *__restrict__ Wm,
                                                           double *__restrict__ R, long long oo, int v, int tab)
{
    __shared__ double sp[kTT][kTT + 1], sm[kTT][kTT + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int ta = blockIdx.y, tb = blockIdx.x;          // output tile: rows a in ta, columns b in tb
    const int a0 = ta * kTT, b0 = tb * kTT;
    const size_t vv = (size_t)v * v;
    for (long long ij = blockIdx.z; ij < oo; ij += gridDim.z) {
        const double *wp = Wp + (size_t)ij * vv, *wm = Wm + (size_t)ij * vv;
        double *r = R + (size_t)ij * vv;
        if (ta < tb) {            // every element has blk(a) < blk(b): direct
#pragma unroll
            for (int rr = ty; rr < kTT; rr += 8) {
                const int a = a0 + rr, b = b0 + tx;
                if (a < v && b < v) r[(size_t)a * v + b] += wp[(size_t)a * v + b] + wm[(size_t)a * v + b];
            }
        } else {
            // mirrored source tile W[b][a] (rows b in tb, columns a in ta), read coalesced along a, used transposed.
            // For ta == tb the same tile also serves the direct elements.
#pragma unroll
            for (int rr = ty; rr < kTT; rr += 8) {
                const int b = b0 + rr, a = a0 + tx;
                const bool ok = (b < v && a < v);
                sp[rr][tx] = ok ? wp[(size_t)b * v + a] : 0.0;
                sm[rr][tx] = ok ? wm[(size_t)b * v + a] : 0.0;
            }
            __syncthreads();
#pragma unroll
            for (int rr = ty; rr < kTT; rr += 8) {
                const int a = a0 + rr, b = b0 + tx;
                if (a < v && b < v) {
                    double add;
                    if (a / tab <= b / tab)
                        add = wp[(size_t)a * v + b] + wm[(size_t)a * v + b];     // direct (diagonal tiles only)
                    else
                        add = sp[tx][rr] - sm[tx][rr];                             // R+ - R- of the pair (b, a)
                    r[(size_t)a * v + b] += add;
                }
            }
            __syncthreads();
        }
    }
}

// Precondition check of the 8-fold-symmetry mode (CC_LADDER_OPT_SYMM_L): counts the elements with
// L[P][a][c] != L[P][c][a] (a < c).  32 x 32 tiles through shared memory so that both reads are coalesced.
__global__ void __launch_bounds__(256) symm_check_kernel(const double *__restrict__ L, int x, int v,
                                                         unsigned long long *__restrict__ count)
{
    __shared__ double tr[kTT][kTT + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int a0 = blockIdx.y * kTT, c0 = blockIdx.x * kTT;
    if (blockIdx.y > blockIdx.x) return;                  // upper block triangle only (whole block exits together)
    const size_t vv = (size_t)v * v;
    unsigned long long bad = 0;
    for (int P = blockIdx.z; P < x; P += gridDim.z) {
        const double *m = L + (size_t)P * vv;
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {               // tr[cl][al] = L[c0+cl][a0+al]
            const int c = c0 + r, a = a0 + tx;
            tr[r][tx] = (c < v && a < v) ? m[(size_t)c * v + a] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {
            const int a = a0 + r, c = c0 + tx;
            if (a < v && c < v && a < c && m[(size_t)a * v + c] != tr[tx][r]) ++bad;
        }
        __syncthreads();
    }
    if (bad) atomicAdd(count, bad);
}

}  // namespace ccl
