// Steps a0 and a5 of the hot path in split (t+/t-) mode (reading 10; not in the paper, north_star), on PACKED
// TRIANGLES: per (i,j) the upper triangle c <= d, row-major, every row aligned for 128-bit copies
// (tri_base / tri_size in ladder_common.cuh: element (c,d) at tri_base(c) + d, nt = tri_size(v) ~ v^2/2 doubles):
//   a0  pack     T+[ij][(c,d)] = t[ij,c,d] + t[ij,d,c] (c < d),  = t[ij,c,c] (c == d);   T-[ij][(c,d)] = t[ij,c,d] - t[ij,d,c]
//                (zeros left of the diagonal and in the padding; the same pass zeroes W+ and W-)
//   a5  unpack   R[ij,a,b] += W+[(a,b)] + W-[(a,b)],  R[ij,b,a] += W+[(a,b)] - W-[(a,b)]  (a < b),  R[ij,a,a] += W+[(a,a)]
// T+- rows are nt doubles; W+- rows carry 8 extra doubles at the end (the "sink": the fused kernel sends what lies
// outside the triangle's slots there instead of predicating its reductions).
// The paper's own storage (iajb != 0): t[i][c][j][d] in, R[i][a][j][b] out -- the (i,j) matrix then starts at
// i*(v*o*v) + j*v and its rows are o*v apart; the packed workspace is the same.  The exchange variant (Eq. 7)
// is the ladder of t with c and d swapped, i.e. the same T+ and the negated T-: unpack with wsign = -1.
// Both kernels are HBM-bound tiled transposes: 32 x 32 tiles through shared memory, every global access coalesced.
#pragma once
#include "ladder_common.cuh"

namespace ccl {

constexpr int kTT = 32;   // transpose tile edge (a multiple of 4: a row's slot starts on a tile-column boundary or inside the
                          // diagonal tile)

// offset of the (i,j) matrix and stride of its rows in the boundary storage [i][j][c][d] / the paper's [i][c][j][d]
__device__ __forceinline__ void ij_matrix(long long ij, int o, int v, int iajb, size_t &base, size_t &rstride)
{
    if (!iajb) {
        base = (size_t)ij * v * v;
        rstride = (size_t)v;
    } else {
        const long long i = ij / o, j = ij - i * o;
        base = (size_t)i * v * o * v + (size_t)j * v;
        rstride = (size_t)o * v;
    }
}

// grid: (tile column td, tile row tc <= td, ij); tiles below the block diagonal exit at once
__global__ void __launch_bounds__(256) split_pack_kernel(const double *__restrict__ t, double *__restrict__ Tp,
                                                         double *__restrict__ Tm, double *__restrict__ Wp,
                                                         double *__restrict__ Wm, long long oo, int v, int o, int iajb)
{
    __shared__ double tr[kTT][kTT + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
    if (blockIdx.y > blockIdx.x) return;
    const int c0 = blockIdx.y * kTT, d0 = blockIdx.x * kTT;
    const long long v4 = tri_v4(v);
    const size_t nt = (size_t)tri_size(v);
    for (long long ij = blockIdx.z; ij < oo; ij += gridDim.z) {
        size_t base, rst;
        ij_matrix(ij, o, v, iajb, base, rst);
        const double *m = t + base;
        // tr[dl][cl] = t[d0+dl][c0+cl]  (rows of the mirrored tile, read coalesced along c)
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {
            const int d = d0 + r, c = c0 + tx;
            tr[r][tx] = (d < v && c < v) ? m[(size_t)d * rst + c] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int r = ty; r < kTT; r += 8) {
            const int c = c0 + r, d = d0 + tx;
            if (c < v && d < v4 && d >= (c & ~3)) {          // inside row c's slot (zeros left of the diagonal / in the padding)
                double sp = 0.0, sm = 0.0;
                if (d < v && c <= d) {
                    const double tcd = m[(size_t)c * rst + d], tdc = tr[tx][r];
                    sp = (c == d) ? tcd : tcd + tdc;
                    sm = tcd - tdc;                           // 0 on the diagonal
                }
                const size_t k = (size_t)(tri_base(c, v4) + d);
                Tp[(size_t)ij * nt + k] = sp;
                Tm[(size_t)ij * nt + k] = sm;
                Wp[(size_t)ij * (nt + 8) + k] = 0.0;
                Wm[(size_t)ij * (nt + 8) + k] = 0.0;
            }
        }
        if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x < 8) {      // the sinks start at zero too (hygiene: they
            Wp[(size_t)ij * (nt + 8) + nt + threadIdx.x] = 0.0;            // accumulate values that are never read)
            Wm[(size_t)ij * (nt + 8) + nt + threadIdx.x] = 0.0;
        }
        __syncthreads();
    }
}

// grid: (tile column tb, tile row ta <= tb, ij)
__global__ void __launch_bounds__(256) split_unpack_kernel(const double *__restrict__ Wp, const double *__restrict__ Wm,
                                                           double *__restrict__ R, long long oo, int v, int o, int iajb,
                                                           double wsign)
{
    __shared__ double sd[kTT][kTT + 1];     // sd[al][bl] = W+ - W- of the pair (a0+al, b0+bl), a < b: what R[b][a] receives
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (blockIdx.y > blockIdx.x) return;
    const int a0 = blockIdx.y * kTT, b0 = blockIdx.x * kTT;
    const long long v4 = tri_v4(v);
    const size_t nt = (size_t)tri_size(v);
    for (long long ij = blockIdx.z; ij < oo; ij += gridDim.z) {
        const double *wp = Wp + (size_t)ij * (nt + 8), *wm = Wm + (size_t)ij * (nt + 8);
        size_t base, rst;
        ij_matrix(ij, o, v, iajb, base, rst);
        double *r = R + base;
#pragma unroll
        for (int rr = ty; rr < kTT; rr += 8) {            // direct half: rows a, columns b, coalesced along b
            const int a = a0 + rr, b = b0 + tx;
            double diff = 0.0;
            if (a < v && b < v && a <= b) {
                const size_t k = (size_t)(tri_base(a, v4) + b);
                const double p = wp[k];
                const double q = (a < b) ? wsign * wm[k] : 0.0;
                r[(size_t)a * rst + b] += p + q;
                diff = p - q;
            }
            sd[rr][tx] = diff;
        }
        __syncthreads();
#pragma unroll
        for (int rr = ty; rr < kTT; rr += 8) {            // mirrored half: rows b, columns a, coalesced along a
            const int b = b0 + rr, a = a0 + tx;
            if (a < v && b < v && a < b) r[(size_t)b * rst + a] += sd[tx][rr];
        }
        __syncthreads();
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
