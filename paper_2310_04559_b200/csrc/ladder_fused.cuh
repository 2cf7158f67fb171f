// Fused Cholesky vvvv ladder kernel for sm_100a (steps a1-a5 of the hot path).
//
// One persistent CTA per SM walks a list of tiles (A-block, B-block, C-block, D-block).  Per tile:
//   GEMM-1  V[(a,c),(b,d)] = sum_P L[P,a,c] L[P,b,d]            (Eq. 5)   DMMA, K = nchol,
//           operands staged by cp.async through a 4-deep shared-memory ring, accumulators in registers;
//   regroup the accumulators are stored to shared memory as Vs[(a,b)][(c,d)]
//   GEMM-2  R[(ij),(a,b)] += sum_(c,d) t[(ij),(c,d)] Vs[(a,b)][(c,d)]                  (Eq. 6)
//           DMMA, M = nocc^2 streamed in chunks of 64 rows, K = the tile's (c,d) pairs in slabs of 32 through a
//           4-slot ring whose "slab landed" flags are mbarriers fed by cp.async (no CTA-wide barrier per slab);
//   accumulate: each 64-row chunk's partial sums leave the SM as red.global.add.f64    ("+=").
// The (ac|bd) tile lives only in registers and shared memory; nothing of size v^4 touches HBM.
//
// All global->shared copies are issued from inside the DMMA loops (one or two cp.async per k-step, addresses
// advanced incrementally), so the copy engine work hides under the tensor pipe instead of forming its own phase.
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
    // split (t+/t-) mode only: n_ab_blk / n_cd_blk count block PAIRS (A <= B), (C <= D) of the square partitions;
    // CTA rank 0 of a pair contracts V+ with t (= T+ = t_cd + t_dc) into R (= W+), rank 1 V- with tm (= T-) into Rm (= W-).
    const double *tm;
    double *Rm;
};

// Index u in [0, n(n+1)/2) of the row-major upper triangle -> (r, c), r <= c.
__device__ __forceinline__ void decode_upper(long long u, int n, int &r, int &c)
{
    const double nn = 2.0 * n + 1.0;
    int rr = (int)((nn - sqrt(nn * nn - 8.0 * (double)u)) * 0.5);
    if (rr < 0) rr = 0;
    if (rr > n - 1) rr = n - 1;
    auto start = [&](long long x) { return x * n - x * (x - 1) / 2; };
    while (rr > 0 && start(rr) > u) --rr;
    while (rr + 1 < n && start(rr + 1) <= u) ++rr;
    r = rr;
    c = rr + (int)(u - start(rr));
}

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
    static constexpr int PV = NCD + 4;          // pitch of Vs[(a,b)][(c,d)]
    static constexpr int V_DOUBLES = NAB * PV;
    static constexpr int MC = 64;               // ij rows per GEMM-2 chunk
    static constexpr int KS = 32;               // (c,d) pairs per staged t slab
    static constexpr int NKS = NCD / KS;
    static constexpr int PT = KS + 4;
    static constexpr int T_STAGE = MC * PT;
    static constexpr int T_STAGES = 4;
    static constexpr int REGION0 = (V_DOUBLES > G1_STAGES * G1_STAGE) ? V_DOUBLES : G1_STAGES * G1_STAGE;
    static constexpr int SMEM_BYTES = (REGION0 + T_STAGES * T_STAGE) * 8 + T_STAGES * 8;   // + mbarriers
    // warp tiling: 8 warps.  GEMM-1: 2 (M) x 4 (N) with wm = warp>>2; GEMM-2: 2 (M) x 4 (N) with wn = warp>>1.
    static constexpr int MI1 = M1 / 2 / 8, NI1 = N1 / 4 / 8;        // 8 x 4 fragments
    static constexpr int MI2 = MC / 2 / 8, NI2 = NAB / 4 / 8;       // 4 x (4 or 2) fragments
    // per-thread copy shapes (16-byte chunks)
    static constexpr int XCH = KC * M1 / 2 / THREADS;               // 4 chunks of X per thread per stage
    static constexpr int YCH = KC * N1 / 2 / THREADS;               // 4 chunks of Y
    static constexpr int TCH = MC * KS / 2 / THREADS;               // 4 chunks of t
    static_assert(M1 == 128 && N1 == 128, "GEMM-1 tile is 128 x 128");
    static_assert(NCD % KS == 0 && NAB % 32 == 0, "tile shape");
    static_assert(TC % 2 == 0 && TD % 2 == 0, "16-byte copies need even block widths");
    static_assert(TB % 8 == 0 && TD % 4 == 0, "fragment shapes");
    static_assert(XCH == KC / 4 && YCH == KC / 4, "one X and one Y chunk per k-step");
    static_assert(TCH < KS / 4, "t chunks are issued in the first k-steps of the previous slab");
    static_assert(T_STAGES >= 3, "prefetch distance 1 without 'slot free' barriers needs >= 3 slots");
};

template <class C, bool ALIGN2, bool SPLIT>
__global__ void __launch_bounds__(C::THREADS, 1) ladder_fused_kernel(const FusedParams p)
{
    static_assert(!SPLIT || (C::TA == C::TB && C::TC == C::TD), "split mode needs square block partitions");
    const uint32_t rank = SPLIT ? cluster_ctarank() : 0u;     // split: 0 builds (ac|bd), 1 builds (ad|bc)
    const long long tile_first = SPLIT ? (long long)(blockIdx.x >> 1) : (long long)blockIdx.x;
    const long long tile_step = SPLIT ? (long long)(gridDim.x >> 1) : (long long)gridDim.x;
    const double *const t_in = (SPLIT && rank) ? p.tm : p.t;
    double *const r_out = (SPLIT && rank) ? p.Rm : p.R;
    extern __shared__ __align__(16) double smem[];
    double *region0 = smem;                    // GEMM-1 stage ring, then the Vs tile
    double *tbuf = smem + C::REGION0;          // t slab ring
    const uint32_t region0_u32 = smem_u32(region0);
    const uint32_t tbuf_u32 = smem_u32(tbuf);
    const uint32_t bars_u32 = tbuf_u32 + (uint32_t)(C::T_STAGES * C::T_STAGE * 8);   // "t slab landed" mbarriers
    if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < C::T_STAGES; ++i) mbar_init(bars_u32 + 8u * i, C::THREADS);
    }
    __syncthreads();
    int ld_slot = 0, use_slot = 0;     // t ring: next slot to fill / to consume (identical in every thread)
    uint32_t use_phase = 0;

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm1 = warp >> 2, wn1 = warp & 3;     // GEMM-1 warp grid (every SM sub-partition holds wm1 = 0 and 1)
    const int wm2 = warp & 1, wn2 = warp >> 1;     // GEMM-2 warp grid (every sub-partition holds wn2 = s and s+2)

    const size_t v = (size_t)p.v, vv = v * v;
    const int nk = (p.x + C::KC - 1) / C::KC;
    const long long nchunks = (p.oo + C::MC - 1) / C::MC;
    const long long nstages2 = nchunks * C::NKS;

    // ---- per-thread copy roles (fixed for the whole kernel) -----------------------------------------------------
    // GEMM-1 stage: X rows (P_l, a_l) of TC doubles, Y rows (P_l, b_l) of TD doubles.  With 16-byte chunks a
    // thread owns one (a_l, c-chunk) and one (b_l, d-chunk) position and the P_l rows tid/64 + 4*it, it = 0..3.
    // (8-byte mode, odd v: the same positions, two adjacent doubles copied separately.)
    const int x_cc = tid % (C::TC / 2), x_al = (tid / (C::TC / 2)) % C::TA, x_pl = tid / (C::TC / 2 * C::TA);
    const int y_dd = tid % (C::TD / 2), y_bl = (tid / (C::TD / 2)) % C::TB, y_pl = tid / (C::TD / 2 * C::TB);
    static_assert(C::TC / 2 * C::TA == 64 && C::TD / 2 * C::TB == 64, "64 chunks per staged P row");
    const uint32_t x_dst = (uint32_t)((x_pl * C::PX + x_al * C::TC + 2 * x_cc) * 8);
    const uint32_t y_dst = (uint32_t)((C::KC * C::PX + y_pl * C::PY + y_bl * C::TD + 2 * y_dd) * 8);
    // t slab: rows r_l = tid/16 + 16*it, chunk ch = tid%16 -> k_l = 2*ch
    const int t_ch = tid % (C::KS / 2), t_rl = tid / (C::KS / 2);
    const uint32_t t_dst = (uint32_t)((t_rl * C::PT + 2 * t_ch) * 8);

    for (long long T = tile_first; T < p.n_tiles; T += tile_step) {
        long long ab_blk, cd_blk;
        decode_tile(p, T, ab_blk, cd_blk);
        int a0, b0, c0, d0;
        bool diag_cd = false;
        if (SPLIT) {
            int A, B, Cb, D;
            decode_upper(ab_blk, p.nA, A, B);
            decode_upper(cd_blk, p.nC, Cb, D);
            a0 = A * C::TA, b0 = B * C::TB, c0 = Cb * C::TC, d0 = D * C::TD;
            diag_cd = (Cb == D);
        } else {
            a0 = (int)(ab_blk / p.nB) * C::TA, b0 = (int)(ab_blk % p.nB) * C::TB;
            c0 = (int)(cd_blk / p.nD) * C::TC, d0 = (int)(cd_blk % p.nD) * C::TD;
        }

        // ------------------------------------------------------------------ GEMM-1: (ac|bd) tile, K = nchol
        // rows of the tile are (ra, c) and columns (rb, d): (a, b) on rank 0; on rank 1 of a split pair (b, a), which
        // makes its tile G[(b,c),(a,d)] = (bc|ad) = (ad|bc), the exchange partner of (ac|bd).
        const int ra0 = rank ? b0 : a0, rb0 = rank ? a0 : b0;
        const int xa = ra0 + x_al, xc = c0 + 2 * x_cc, yb = rb0 + y_bl, yd = d0 + 2 * y_dd;
        const bool x_ok0 = (xa < p.v) && (xc < p.v), x_ok1 = (xa < p.v) && (xc + 1 < p.v);
        const bool y_ok0 = (yb < p.v) && (yd < p.v), y_ok1 = (yb < p.v) && (yd + 1 < p.v);
        const double *x_src = p.L + (x_ok0 ? ((size_t)x_pl * v + xa) * v + xc : 0);   // advanced by KC*vv per stage
        const double *y_src = p.L + (y_ok0 ? ((size_t)y_pl * v + yb) * v + yd : 0);
        int ld_kc = 0;                                                                  // next stage to load

        auto g1_issue = [&](int it) {   // chunk `it` (P row x_pl + 4*it) of stage ld_kc
            const int P = ld_kc * C::KC + 4 * it;
            const uint32_t sb = region0_u32 + (uint32_t)((ld_kc % C::G1_STAGES) * C::G1_STAGE * 8) +
                                (uint32_t)(4 * it * C::PX * 8);
            const bool px = (P + x_pl) < p.x, py = (P + y_pl) < p.x;
            if (ALIGN2) {
                cp_async_16(sb + x_dst, x_src + (size_t)(4 * it) * vv, px && x_ok0);
                cp_async_16(sb + y_dst, y_src + (size_t)(4 * it) * vv, py && y_ok0);
            } else {
                cp_async_8(sb + x_dst, x_src + (size_t)(4 * it) * vv, px && x_ok0);
                cp_async_8(sb + x_dst + 8, x_src + (size_t)(4 * it) * vv + 1, px && x_ok1);
                cp_async_8(sb + y_dst, y_src + (size_t)(4 * it) * vv, py && y_ok0);
                cp_async_8(sb + y_dst + 8, y_src + (size_t)(4 * it) * vv + 1, py && y_ok1);
            }
        };
        auto g1_advance = [&]() {
            ++ld_kc;
            if (x_ok0) x_src += (size_t)C::KC * vv;
            if (y_ok0) y_src += (size_t)C::KC * vv;
        };

        double acc1[C::MI1][C::NI1][2];
#pragma unroll
        for (int i = 0; i < C::MI1; ++i)
#pragma unroll
            for (int j = 0; j < C::NI1; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;

#pragma unroll
        for (int s = 0; s < C::G1_STAGES - 1; ++s) {
            if (s < nk) {
#pragma unroll
                for (int it = 0; it < C::XCH; ++it) g1_issue(it);
                g1_advance();
            }
            cp_async_commit();
        }
        for (int kc = 0; kc < nk; ++kc) {
            cp_async_wait<C::G1_STAGES - 2>();
            __syncthreads();   // stage kc landed; every warp is done with stage kc-1, whose buffer is refilled below
            const bool more = ld_kc < nk;
            const double *Xs = region0 + (kc % C::G1_STAGES) * C::G1_STAGE + wm1 * (C::M1 / 2) + g;
            const double *Ys = region0 + (kc % C::G1_STAGES) * C::G1_STAGE + C::KC * C::PX + wn1 * (C::N1 / 4) + g;
#pragma unroll
            for (int kk = 0; kk < C::KC / 4; ++kk) {
                double af[C::MI1], bf[C::NI1];
#pragma unroll
                for (int i = 0; i < C::MI1; ++i) af[i] = Xs[(kk * 4 + q) * C::PX + i * 8];
#pragma unroll
                for (int j = 0; j < C::NI1; ++j) bf[j] = Ys[(kk * 4 + q) * C::PY + j * 8];
                if (more) g1_issue(kk);
#pragma unroll
                for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                    for (int j = 0; j < C::NI1; ++j) dmma_8x8x4(acc1[i][j][0], acc1[i][j][1], af[i], bf[j]);
            }
            if (more) g1_advance();
            cp_async_commit();
        }
        cp_async_wait<0>();
        __syncthreads();   // every warp is done with the stage ring: region0 may become Vs

        // ------------------------------------------------------------------ t slab copy roles for this tile
        // slab s = chunk*NKS + ksi covers rows [chunk*MC, +MC) and pairs k in [ksi*KS, +KS): k = c_l*TD + d_l.
        const int tk = 2 * t_ch;                                     // k_l of this thread's chunk
        const int t_d = d0 + tk % C::TD;                              // d is the same in every slab (KS % TD == 0)
        const bool t_dok0 = t_d < p.v, t_dok1 = t_d + 1 < p.v;
        static_assert(C::KS % C::TD == 0, "slab covers whole d rows");
        const int t_cbase = c0 + tk / C::TD;                          // c of slab ksi: t_cbase + ksi*(KS/TD)
        const double *t_src = t_in + (size_t)t_rl * vv + (size_t)(t_cbase < p.v ? t_cbase : 0) * v + (t_dok0 ? t_d : 0);
        long long ld_s = 0;                                           // next slab of this tile to load
        int ld_ksi = 0;
        long long ld_row = t_rl;                                      // first row this thread copies in slab ld_s

        auto t_issue = [&](int it) {   // rows ld_row + 16*it of slab ld_s, into ring slot ld_slot
            const uint32_t sb = tbuf_u32 + (uint32_t)(ld_slot * C::T_STAGE * 8) +
                                (uint32_t)(it * (C::THREADS / (C::KS / 2)) * C::PT * 8);
            const bool rok = (ld_row + it * (C::THREADS / (C::KS / 2))) < p.oo;
            const bool cok = (t_cbase + ld_ksi * (C::KS / C::TD)) < p.v;
            const double *src = t_src + (size_t)(it * (C::THREADS / (C::KS / 2))) * vv;
            if (ALIGN2) {
                cp_async_16(sb + t_dst, (rok && cok && t_dok0) ? src : t_in, rok && cok && t_dok0);
            } else {
                cp_async_8(sb + t_dst, (rok && cok && t_dok0) ? src : t_in, rok && cok && t_dok0);
                cp_async_8(sb + t_dst + 8, (rok && cok && t_dok1) ? src + 1 : t_in, rok && cok && t_dok1);
            }
        };
        auto t_advance = [&]() {   // signal "my part of the slab is in flight" and move to the next slab
            cp_async_mbar_arrive(bars_u32 + 8u * ld_slot);
            ld_slot = (ld_slot + 1) % C::T_STAGES;
            ++ld_s;
            if (++ld_ksi == C::NKS) {
                ld_ksi = 0;
                ld_row += C::MC;
                t_src += (size_t)C::MC * vv - (size_t)(C::NKS - 1) * (C::KS / C::TD) * v;
            } else {
                t_src += (size_t)(C::KS / C::TD) * v;
            }
        };

        // slab 0: its latency overlaps the regroup stores
#pragma unroll
        for (int it = 0; it < C::TCH; ++it) t_issue(it);
        t_advance();

        // ------------------------------------------------------------------ regroup (ac)(bd) -> Vs[(ab)][(cd)]
        // A lane's accumulator pair sits at tile row m = (ra_l, c_l) and columns n, n+1 = (rb_l, d_l), (rb_l, d_l+1):
        // two adjacent (c,d) pairs of one (a,b) pair, i.e. one 16-byte store into Vs[(a_l,b_l)][(c_l,d_l)].
        auto vs_pos = [&](int i, int j) {
            const int m = wm1 * (C::M1 / 2) + i * 8 + g;
            const int n = wn1 * (C::N1 / 4) + j * 8 + 2 * q;
            const int ral = m / C::TC, cl = m % C::TC, rbl = n / C::TD, dl = n % C::TD;
            const int al = rank ? rbl : ral, bl = rank ? ral : rbl;
            return (al * C::TB + bl) * C::PV + cl * C::TD + dl;
        };
        if (!SPLIT) {
#pragma unroll
            for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                for (int j = 0; j < C::NI1; ++j)
                    *reinterpret_cast<double2 *>(region0 + vs_pos(i, j)) = make_double2(acc1[i][j][0], acc1[i][j][1]);
        } else {
            // V+ = w/2 [(ac|bd) + (ad|bc)] on rank 0, V- = w/2 [(ac|bd) - (ad|bc)] on rank 1, w = 1/2 on diagonal (C == D)
            // block pairs (they hold every (c,d) pair twice), else 1  (reading 10).
            // Each CTA writes its tile into the partner's Vs, then folds the partner's tile into its own registers.
            cluster_sync_all();   // the partner is done with its stage ring too: its region0 may be written
            const uint32_t peer = map_to_cta(region0_u32, rank ^ 1u);
#pragma unroll
            for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                for (int j = 0; j < C::NI1; ++j)
                    st_cluster_f64x2(peer + (uint32_t)(vs_pos(i, j) * 8), acc1[i][j][0], acc1[i][j][1]);
            cluster_sync_all();   // both tiles have landed
            const double sc = diag_cd ? 0.25 : 0.5;
            const double sg = rank ? -sc : sc;      // rank 1: sc * (partner - own)
#pragma unroll
            for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                for (int j = 0; j < C::NI1; ++j) {
                    double2 *ptr = reinterpret_cast<double2 *>(region0 + vs_pos(i, j));
                    const double2 o = *ptr;
                    *ptr = make_double2(sc * o.x + sg * acc1[i][j][0], sc * o.y + sg * acc1[i][j][1]);
                }
        }
        __syncthreads();   // Vs complete

        // ------------------------------------------------------------------ GEMM-2: R[(ij),(ab)] += t . Vs^T
        // Column n of an 8-wide output fragment is the (a,b) pair n0 + pi(n), pi = [0,6,1,7,2,4,3,5]: the lane's first
        // accumulator then sits at pair n0 + q and the second at n0 + [6,7,4,5][q], so every red instruction of a warp
        // covers 8 rows x one full 32-byte sector, while the B-fragment rows n0 + pi(g) stay bank-conflict-free.
        const int pig = (g & 1) ? (4 + (((g >> 1) + 2) & 3)) : (g >> 1);          // pi(g)
        const int sq = (q < 2) ? (6 + q) : (2 + q);                            // pair offset of the second accumulator
        double *r_ptr[C::NI2];
        bool r_ok0[C::NI2], r_ok1[C::NI2];
        const bool interior = (a0 + C::TA <= p.v) && (b0 + C::TB <= p.v);
#pragma unroll
        for (int j = 0; j < C::NI2; ++j) {
            const int n = wn2 * (C::NAB / 4) + j * 8;
            const int a = a0 + n / C::TB, b = b0 + n % C::TB;     // n % TB is 0 or 8: the fragment stays in one row of R
            r_ok0[j] = (a < p.v) && (b + q < p.v);
            r_ok1[j] = (a < p.v) && (b + sq < p.v);
            r_ptr[j] = r_out + ((a < p.v) ? (size_t)a * v : 0) + (r_ok0[j] ? b + q : 0) + (size_t)(wm2 * (C::MC / 2) + g) * vv;
        }
        long long row0 = wm2 * (C::MC / 2) + g;      // row of fragment i = 0 in the current chunk

        double acc2[C::MI2][C::NI2][2];
#pragma unroll
        for (int i = 0; i < C::MI2; ++i)
#pragma unroll
            for (int j = 0; j < C::NI2; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;

        int ksi = 0;
        for (long long s = 0; s < nstages2; ++s) {
            // Slab s is consumed from ring slot use_slot once every thread's copies have landed.  Slab s+1 is issued
            // during the first k-steps below into the next slot; a thread can only get here after every thread has
            // issued slab s, i.e. is at least in slab s-1, so with >= 3 slots no slot is overwritten while in use.
            mbar_wait(bars_u32 + 8u * use_slot, use_phase);
            const bool more = ld_s < nstages2;
            const double *Ts = tbuf + use_slot * C::T_STAGE + (wm2 * (C::MC / 2) + g) * C::PT + q;
            const double *Vs = region0 + (wn2 * (C::NAB / 4) + pig) * C::PV + ksi * C::KS + q;
#pragma unroll
            for (int k4 = 0; k4 < C::KS / 4; ++k4) {
                double af[C::MI2], bf[C::NI2];
#pragma unroll
                for (int i = 0; i < C::MI2; ++i) af[i] = Ts[i * 8 * C::PT + k4 * 4];
#pragma unroll
                for (int j = 0; j < C::NI2; ++j) bf[j] = Vs[j * 8 * C::PV + k4 * 4];
                if (k4 < C::TCH && more) t_issue(k4);
                if (k4 == C::TCH && more) t_advance();
#pragma unroll
                for (int i = 0; i < C::MI2; ++i)
#pragma unroll
                    for (int j = 0; j < C::NI2; ++j) dmma_8x8x4(acc2[i][j][0], acc2[i][j][1], af[i], bf[j]);
            }
            if (++use_slot == C::T_STAGES) { use_slot = 0; use_phase ^= 1u; }
            if (++ksi == C::NKS) {
                ksi = 0;
                // accumulate this chunk's partial sums into R (fire-and-forget L2 reductions)
                if (interior && row0 - g + (C::MC / 2) <= p.oo) {   // warp-uniform
#pragma unroll
                    for (int i = 0; i < C::MI2; ++i)
#pragma unroll
                        for (int j = 0; j < C::NI2; ++j) {
                            double *dst = r_ptr[j] + (size_t)(i * 8) * vv;
                            red_add_f64(dst, acc2[i][j][0]);
                            red_add_f64(dst + (sq - q), acc2[i][j][1]);
                            acc2[i][j][0] = acc2[i][j][1] = 0.0;
                        }
                } else {
#pragma unroll
                    for (int i = 0; i < C::MI2; ++i) {
                        const bool rok = (row0 + i * 8) < p.oo;
#pragma unroll
                        for (int j = 0; j < C::NI2; ++j) {
                            double *dst = r_ptr[j] + (size_t)(i * 8) * vv;
                            if (rok && r_ok0[j]) red_add_f64(dst, acc2[i][j][0]);
                            if (rok && r_ok1[j]) red_add_f64(dst + (sq - q), acc2[i][j][1]);
                            acc2[i][j][0] = acc2[i][j][1] = 0.0;
                        }
                    }
                }
                row0 += C::MC;
#pragma unroll
                for (int j = 0; j < C::NI2; ++j) r_ptr[j] += (size_t)C::MC * vv;
            }
        }
        __syncthreads();   // Vs (region0) and the t ring are dead: the next tile may overwrite them
    }
}

}  // namespace ccl
