// Fused Cholesky vvvv ladder kernel for sm_100a (steps a1-a5 of the hot path).
//
// One persistent CTA per SM walks a list of tiles (A-block, B-block, C-block, D-block).  Per tile:
//   GEMM-1  V[(a,c),(b,d)] = sum_P L[P,a,c] L[P,b,d]            (Eq. 5)   DMMA, K = nchol,
//           operands staged by cp.async through a 4-deep shared-memory ring, accumulators in registers;
//   regroup the accumulators are scattered to shared memory as Vs[(c,d)][(a,b)]
//   GEMM-2  R[(ij),(a,b)] += sum_(c,d) t[(ij),(c,d)] Vs[(c,d)][(a,b)]                  (Eq. 6)
//           DMMA, M = nocc^2 streamed in chunks of 64 rows through a 2-deep ring, K = the tile's (c,d) pairs;
//   accumulate: each 64-row chunk's partial sums leave the SM as red.global.add.f64    ("+=").
// The (ac|bd) tile lives only in registers and shared memory; nothing of size v^4 touches HBM.
#pragma once
#include "ladder_common.cuh"

namespace ccl {

struct FusedParams {
    const double *L;   // [x][v][v]
    const double *t;   // [o*o][v][v]
    double *R;         // [o*o][v][v]
    int o, v, x;
    long long oo;          // o*o
    int nA, nB, nC, nD;    // number of blocks along a, b, c, d
    long long n_ab_blk;    // nA*nB
    long long n_cd_blk;    // nC*nD
    long long n_tiles;     // n_ab_blk*n_cd_blk
    int supertile;         // L2 super-tile edge (in blocks)
};

// Maps the linear tile index to (ab block, cd block): super-rows of `S` ab-blocks; inside a super-row, super-columns
// of `S` cd-blocks; inside a super-tile ab-major.  ~S*S consecutive tiles (= the CTAs in flight) then share S
// R blocks and S t blocks, which stay L2-resident.
__device__ __forceinline__ void decode_tile(const FusedParams &p, long long T, long long &ab, long long &cd)
{
    const long long S = p.supertile;
    const long long per_sr = S * p.n_cd_blk;
    const long long sr = T / per_sr;
    const long long rem = T - sr * per_sr;
    const long long rows = (p.n_ab_blk - sr * S) < S ? (p.n_ab_blk - sr * S) : S;
    const long long sc = rem / (rows * S);
    const long long rem2 = rem - sc * rows * S;
    const long long w = (p.n_cd_blk - sc * S) < S ? (p.n_cd_blk - sc * S) : S;
    const long long abl = rem2 / w;
    ab = sr * S + abl;
    cd = sc * S + (rem2 - abl * w);
}

template <int TA_, int TB_, int TC_, int TD_>
struct FusedCfg {
    static constexpr int TA = TA_, TB = TB_, TC = TC_, TD = TD_;
    static constexpr int M1 = TA * TC;          // GEMM-1 tile rows  (a,c)
    static constexpr int N1 = TB * TD;          // GEMM-1 tile cols  (b,d)
    static constexpr int NAB = TA * TB;         // (a,b) pairs per tile = GEMM-2 N
    static constexpr int NCD = TC * TD;         // (c,d) pairs per tile = GEMM-2 K
    static constexpr int THREADS = 256;
    static constexpr int KC = 16;               // Cholesky vectors per GEMM-1 stage
    static constexpr int PX = M1 + 4;           // pitch of a staged L row (== 4 mod 16 doubles: conflict-free)
    static constexpr int PY = N1 + 4;
    static constexpr int G1_STAGE = KC * (PX + PY);
    static constexpr int G1_STAGES = 4;
    static constexpr int PV = NAB + 4;          // pitch of Vs[(c,d)][(a,b)]
    static constexpr int V_DOUBLES = NCD * PV;
    static constexpr int MC = 64;               // ij rows per GEMM-2 chunk
    static constexpr int KS = 64;               // (c,d) pairs per staged t slab
    static constexpr int NKS = NCD / KS;
    static constexpr int PT = KS + 4;
    static constexpr int T_STAGE = MC * PT;
    static constexpr int REGION0 = (V_DOUBLES > G1_STAGES * G1_STAGE) ? V_DOUBLES : G1_STAGES * G1_STAGE;
    static constexpr int SMEM_BYTES = (REGION0 + 2 * T_STAGE) * 8;
    // warp tiling: 8 warps, 2 along M x 4 along N in both GEMMs
    static constexpr int MI1 = M1 / 2 / 8, NI1 = N1 / 4 / 8;        // 8 x 4 fragments
    static constexpr int MI2 = MC / 2 / 8, NI2 = NAB / 4 / 8;       // 4 x (4 or 2) fragments
    static_assert(M1 == 128 && N1 == 128, "GEMM-1 tile is 128 x 128");
    static_assert(NCD % KS == 0 && NAB % 32 == 0, "tile shape");
    static_assert(TC % 2 == 0 && TD % 2 == 0, "16-byte copies need even block widths");
    static_assert(TB % 8 == 0, "an 8-wide output fragment must stay inside one row of R");
};

template <class C, bool ALIGN2>
__device__ __forceinline__ void g1_load_stage(const FusedParams &p, double *stage, int kc, int a0, int b0, int c0,
                                              int d0, int tid)
{
    double *Xs = stage;
    double *Ys = stage + C::KC * C::PX;
    const size_t v = (size_t)p.v;
    if (ALIGN2) {
        constexpr int XCH = C::KC * C::TA * C::TC / 2;
        static_assert(XCH % C::THREADS == 0, "loader shape");
#pragma unroll
        for (int it = 0; it < XCH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int cc = id % (C::TC / 2);
            const int al = (id / (C::TC / 2)) % C::TA;
            const int Pl = id / (C::TC / 2 * C::TA);
            const int P = kc * C::KC + Pl, a = a0 + al, c = c0 + 2 * cc;
            const bool ok = (P < p.x) && (a < p.v) && (c < p.v);
            const double *src = ok ? p.L + ((size_t)P * v + a) * v + c : p.L;
            cp_async_16(smem_u32(Xs + Pl * C::PX + al * C::TC + 2 * cc), src, ok);
        }
        constexpr int YCH = C::KC * C::TB * C::TD / 2;
        static_assert(YCH % C::THREADS == 0, "loader shape");
#pragma unroll
        for (int it = 0; it < YCH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int dd = id % (C::TD / 2);
            const int bl = (id / (C::TD / 2)) % C::TB;
            const int Pl = id / (C::TD / 2 * C::TB);
            const int P = kc * C::KC + Pl, b = b0 + bl, d = d0 + 2 * dd;
            const bool ok = (P < p.x) && (b < p.v) && (d < p.v);
            const double *src = ok ? p.L + ((size_t)P * v + b) * v + d : p.L;
            cp_async_16(smem_u32(Ys + Pl * C::PY + bl * C::TD + 2 * dd), src, ok);
        }
    } else {
        constexpr int XCH = C::KC * C::TA * C::TC;
        static_assert(XCH % C::THREADS == 0, "loader shape");
#pragma unroll 4
        for (int it = 0; it < XCH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int cc = id % C::TC;
            const int al = (id / C::TC) % C::TA;
            const int Pl = id / (C::TC * C::TA);
            const int P = kc * C::KC + Pl, a = a0 + al, c = c0 + cc;
            const bool ok = (P < p.x) && (a < p.v) && (c < p.v);
            const double *src = ok ? p.L + ((size_t)P * v + a) * v + c : p.L;
            cp_async_8(smem_u32(Xs + Pl * C::PX + al * C::TC + cc), src, ok);
        }
        constexpr int YCH = C::KC * C::TB * C::TD;
        static_assert(YCH % C::THREADS == 0, "loader shape");
#pragma unroll 4
        for (int it = 0; it < YCH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int dd = id % C::TD;
            const int bl = (id / C::TD) % C::TB;
            const int Pl = id / (C::TD * C::TB);
            const int P = kc * C::KC + Pl, b = b0 + bl, d = d0 + dd;
            const bool ok = (P < p.x) && (b < p.v) && (d < p.v);
            const double *src = ok ? p.L + ((size_t)P * v + b) * v + d : p.L;
            cp_async_8(smem_u32(Ys + Pl * C::PY + bl * C::TD + dd), src, ok);
        }
    }
}

// One staged slab of t: rows ij in [chunk*MC, +MC), (c,d) pairs k in [ksi*KS, +KS) of the tile.
template <class C, bool ALIGN2>
__device__ __forceinline__ void t_load_stage(const FusedParams &p, double *Ts, long long chunk, int ksi, int c0, int d0,
                                             int tid)
{
    const size_t v = (size_t)p.v;
    const size_t vv = v * v;
    if (ALIGN2) {
        constexpr int CH = C::MC * C::KS / 2;
        static_assert(CH % C::THREADS == 0, "loader shape");
#pragma unroll
        for (int it = 0; it < CH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int ch = id % (C::KS / 2);
            const int rl = id / (C::KS / 2);
            const int k = ksi * C::KS + 2 * ch;
            const int c = c0 + k / C::TD, d = d0 + k % C::TD;
            const long long ij = chunk * C::MC + rl;
            const bool ok = (ij < p.oo) && (c < p.v) && (d < p.v);
            const double *src = ok ? p.t + (size_t)ij * vv + (size_t)c * v + d : p.t;
            cp_async_16(smem_u32(Ts + rl * C::PT + 2 * ch), src, ok);
        }
    } else {
        constexpr int CH = C::MC * C::KS;
        static_assert(CH % C::THREADS == 0, "loader shape");
#pragma unroll 4
        for (int it = 0; it < CH / C::THREADS; ++it) {
            const int id = tid + it * C::THREADS;
            const int kl = id % C::KS;
            const int rl = id / C::KS;
            const int k = ksi * C::KS + kl;
            const int c = c0 + k / C::TD, d = d0 + k % C::TD;
            const long long ij = chunk * C::MC + rl;
            const bool ok = (ij < p.oo) && (c < p.v) && (d < p.v);
            const double *src = ok ? p.t + (size_t)ij * vv + (size_t)c * v + d : p.t;
            cp_async_8(smem_u32(Ts + rl * C::PT + kl), src, ok);
        }
    }
}

template <class C, bool ALIGN2>
__global__ void __launch_bounds__(C::THREADS, 1) ladder_fused_kernel(const FusedParams p)
{
    extern __shared__ __align__(16) double smem[];
    double *region0 = smem;                    // GEMM-1 stage ring, then the Vs tile
    double *tbuf = smem + C::REGION0;          // two t stages

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp & 1, wn = warp >> 1;

    const int nk = (p.x + C::KC - 1) / C::KC;
    const long long nchunks = (p.oo + C::MC - 1) / C::MC;
    const long long nstages2 = nchunks * C::NKS;

    for (long long T = blockIdx.x; T < p.n_tiles; T += gridDim.x) {
        long long ab_blk, cd_blk;
        decode_tile(p, T, ab_blk, cd_blk);
        const int a0 = (int)(ab_blk / p.nB) * C::TA, b0 = (int)(ab_blk % p.nB) * C::TB;
        const int c0 = (int)(cd_blk / p.nD) * C::TC, d0 = (int)(cd_blk % p.nD) * C::TD;

        // ------------------------------------------------------------------ GEMM-1: (ac|bd) tile, K = nchol
        double acc1[C::MI1][C::NI1][2];
#pragma unroll
        for (int i = 0; i < C::MI1; ++i)
#pragma unroll
            for (int j = 0; j < C::NI1; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;

#pragma unroll
        for (int s = 0; s < C::G1_STAGES - 1; ++s) {
            if (s < nk) g1_load_stage<C, ALIGN2>(p, region0 + s * C::G1_STAGE, s, a0, b0, c0, d0, tid);
            cp_async_commit();
        }
        for (int kc = 0; kc < nk; ++kc) {
            cp_async_wait<C::G1_STAGES - 2>();
            __syncthreads();
            {
                const int nxt = kc + C::G1_STAGES - 1;
                if (nxt < nk)
                    g1_load_stage<C, ALIGN2>(p, region0 + (nxt % C::G1_STAGES) * C::G1_STAGE, nxt, a0, b0, c0, d0, tid);
                cp_async_commit();
            }
            const double *Xs = region0 + (kc % C::G1_STAGES) * C::G1_STAGE + wm * (C::M1 / 2) + g;
            const double *Ys = region0 + (kc % C::G1_STAGES) * C::G1_STAGE + C::KC * C::PX + wn * (C::N1 / 4) + g;
#pragma unroll
            for (int kk = 0; kk < C::KC / 4; ++kk) {
                double af[C::MI1], bf[C::NI1];
#pragma unroll
                for (int i = 0; i < C::MI1; ++i) af[i] = Xs[(kk * 4 + q) * C::PX + i * 8];
#pragma unroll
                for (int j = 0; j < C::NI1; ++j) bf[j] = Ys[(kk * 4 + q) * C::PY + j * 8];
#pragma unroll
                for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                    for (int j = 0; j < C::NI1; ++j) dmma_8x8x4(acc1[i][j][0], acc1[i][j][1], af[i], bf[j]);
            }
        }
        cp_async_wait<0>();
        __syncthreads();   // every warp is done with the stage ring: region0 may become Vs

        // ------------------------------------------------------------------ regroup (ac)(bd) -> Vs[(cd)][(ab)]
        {
            double *Vs = region0;
#pragma unroll
            for (int i = 0; i < C::MI1; ++i) {
                const int m = wm * (C::M1 / 2) + i * 8 + g;
                const int al = m / C::TC, cl = m % C::TC;
#pragma unroll
                for (int j = 0; j < C::NI1; ++j)
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        const int n = wn * (C::N1 / 4) + j * 8 + 2 * q + r;
                        const int bl = n / C::TD, dl = n % C::TD;
                        Vs[(cl * C::TD + dl) * C::PV + al * C::TB + bl] = acc1[i][j][r];
                    }
            }
        }
        // first two t slabs (their latency overlaps the regroup stores)
        t_load_stage<C, ALIGN2>(p, tbuf, 0, 0, c0, d0, tid);
        cp_async_commit();
        if (nstages2 > 1) t_load_stage<C, ALIGN2>(p, tbuf + C::T_STAGE, 1 / C::NKS, 1 % C::NKS, c0, d0, tid);
        cp_async_commit();

        // ------------------------------------------------------------------ GEMM-2: R[(ij),(ab)] += t . Vs
        double acc2[C::MI2][C::NI2][2];
#pragma unroll
        for (int i = 0; i < C::MI2; ++i)
#pragma unroll
            for (int j = 0; j < C::NI2; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;

        for (long long s = 0; s < nstages2; ++s) {
            cp_async_wait<1>();
            __syncthreads();   // slab s landed (and, for s == 0, Vs is complete)
            const int ksi = (int)(s % C::NKS);
            const double *Ts = tbuf + (s & 1) * C::T_STAGE + (wm * (C::MC / 2) + g) * C::PT + q;
            const double *Vs = region0 + (ksi * C::KS + q) * C::PV + wn * (C::NAB / 4) + g;
#pragma unroll 4
            for (int k4 = 0; k4 < C::KS / 4; ++k4) {
                double af[C::MI2], bf[C::NI2];
#pragma unroll
                for (int i = 0; i < C::MI2; ++i) af[i] = Ts[i * 8 * C::PT + k4 * 4];
#pragma unroll
                for (int j = 0; j < C::NI2; ++j) bf[j] = Vs[k4 * 4 * C::PV + j * 8];
#pragma unroll
                for (int i = 0; i < C::MI2; ++i)
#pragma unroll
                    for (int j = 0; j < C::NI2; ++j) dmma_8x8x4(acc2[i][j][0], acc2[i][j][1], af[i], bf[j]);
            }
            if (ksi == C::NKS - 1) {
                // accumulate this chunk's partial sums into R (fire-and-forget L2 reductions)
                const long long chunk = s / C::NKS;
#pragma unroll
                for (int i = 0; i < C::MI2; ++i) {
                    const long long ij = chunk * C::MC + wm * (C::MC / 2) + i * 8 + g;
#pragma unroll
                    for (int j = 0; j < C::NI2; ++j) {
                        const int n = wn * (C::NAB / 4) + j * 8 + 2 * q;
                        const int a = a0 + n / C::TB, b = b0 + n % C::TB;
                        if (ij < p.oo && a < p.v) {
                            double *dst = p.R + ((size_t)ij * p.v + a) * (size_t)p.v + b;
                            if (b < p.v) red_add_f64(dst, acc2[i][j][0]);
                            if (b + 1 < p.v) red_add_f64(dst + 1, acc2[i][j][1]);
                        }
                        acc2[i][j][0] = acc2[i][j][1] = 0.0;
                    }
                }
            }
            __syncthreads();   // everyone is done reading slab s: its buffer can be refilled
            if (s + 2 < nstages2)
                t_load_stage<C, ALIGN2>(p, tbuf + (s & 1) * C::T_STAGE, (s + 2) / C::NKS, (int)((s + 2) % C::NKS), c0, d0,
                                        tid);
            cp_async_commit();
        }
        cp_async_wait<0>();
        // the last __syncthreads above also protects region0 (Vs) against the next tile's stage loads
    }
}

}  // namespace ccl
