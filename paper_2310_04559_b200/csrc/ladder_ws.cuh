// Warp-specialised fused Cholesky vvvv ladder kernel for sm_100a (steps a1-a5 of the hot path).
//
// One persistent CTA per SM: 8 consumer warps (all the DMMA work, 232 registers each after setmaxnreg) + one producer
// warpgroup (all global->shared copies, 40 registers): every SM sub-partition holds two consumers and one producer.
// Per tile (A-block, B-block, C-block, D-block):
//   GEMM-1  G[(a,c),(b,d)] = sum_P L[P,a,c] L[P,b,d]                  (Eq. 5)   DMMA, K = nchol,
//           operands staged by the producer's cp.async through a ring of "full"/"empty" mbarriers;
//   regroup accumulators -> shared memory as Vs[(a,b)][(c,d)]
//   GEMM-2  R[(ij),(a,b)] += sum_(c,d) t[(ij),(c,d)] Vs[(a,b)][(c,d)]                        (Eq. 6)
//           DMMA, M = nocc^2 streamed in chunks of 64 rows, K = the tile's (c,d) pairs in slabs through a second ring;
//   accumulate: each chunk's partial sums leave the SM as red.global.add.f64 ("+="), issued a few at a
//           time from inside the next chunk's first K slab so that the reductions overlap the DMMA stream.
// The (ac|bd) tile lives only in registers and shared memory; nothing of size v^4 touches HBM.
//
// The tile shape <TA,TB,TC,TD> is a template parameter with few constraints (TA*TC % 16 == 0, TB*TD % 32 == 0,
// TA*TB % 32 == 0, TC and TD even), so the plan can pick block edges that divide nvirt (12 for 300 and 420) instead
// of padding every dimension to 8 or 16.
#pragma once
#include <type_traits>
#include <utility>

#include "ladder_common.cuh"

namespace ccl {

struct FusedParams {
    // GEMM-1 operands: X[P][r][c] at X + P*xps + r*xrs + c (r < nr), Y[P][s][d] at Y + P*yps + s*yrs + d (s < ns);
    // c, d < v.  The ladder is X = Y = L, nr = ns = v, xps = yps = v*v, xrs = yrs = v  (Eq. 6); the
    // occupied-virtual family takes rectangular blocks of Cholesky vectors (Eqs. 8-9).
    const double *X, *Y;
    long long xps, xrs, yps, yrs;
    int nr, ns;
    const double *t;   // [o*o][v][v]
    double *R;         // [o*o][nr][ns]
    int o, v, x;
    long long oo;          // o*o
    long long rs;          // nr*ns: row stride of R in the [i][j][r][s] storage
    int nA, nB, nC, nD;    // number of blocks along a, b, c, d
    long long n_ab_blk;    // nA*nB            (split: block pairs A <= B)
    long long n_cd_blk;    // nC*nD            (split: block pairs C <= D)
    long long n_tiles;     // n_ab_blk*n_cd_blk
    int SA, SB, SC, SD;    // L2 super-tile: SA x SB x SC x SD blocks are in flight together (full mode)
    int supertile;         // split mode: super-tile edge in (pair) blocks
    int idx32;             // every product of the tile decode fits 32 bits (host-checked)
    long long ovv;         // IAJB layout: stride of i in t[i][c][j][d] = v*o*v
    long long ovv_out;     // IAJB layout: stride of i in R[i][r][j][s] = nr*o*ns
    int exchange;          // full mode, square tile shapes only: build (ad|bc) instead of (ac|bd)  (Eq. 7)
    // split (t+/t-) mode only: CTA rank 0 of a pair contracts V+ with t (= T+, packed triangles of tri_nt doubles per
    // (i,j), element (c,d) at tri_base(c) + d) into R (= W+, rows of rs = tri_nt + 8 doubles, the last 8 a sink), rank 1
    // V- with tm (= T-) into Rm (= W-), same layouts.
    const double *tm;
    double *Rm;
    long long tri_nt, tri_v4;
    // Dynamic tile scheduler (full mode): a device counter, zero at launch, from which every CTA draws its next tile
    // index; nullptr = static round-robin (tile = blockIdx.x + k * gridDim.x).
    unsigned long long *tile_counter;
};

// Offset of row (i,j) of the (ij) x (rs) output matrix R.  Boundary layout [i][j][r][s]: row * nr*ns.  The paper's own
// storage (t_new[i,a,j,b]; IAJB = true): i * (nr*o*ns) + j * ns, and the stride of the slow index r
// becomes o*ns instead of ns.
template <bool IAJB>
__device__ __forceinline__ size_t row_offset(const FusedParams &p, long long row, size_t rs)
{
    if (!IAJB) return (size_t)row * rs;
    const unsigned r = (unsigned)row, i = r / (unsigned)p.o, j = r - i * (unsigned)p.o;
    return (size_t)i * (size_t)p.ovv_out + (size_t)j * (size_t)p.ns;
}

// Index u in [0, n(n+1)/2) of the upper triangle (r <= c) of an n x n block grid, enumerated in bands of H rows:
// band g holds the rows [gH, gH+h), h = min(H, n - gH); inside a band the columns c = gH .. n-1 in order, and for
// each column its (at most h) rows r <= c.  Away from the diagonal, H*W consecutive indices are an H x W rectangle of
// blocks, which is what keeps the L slabs of the tiles in flight few (a row-major triangle would give a 1 x HW strip).
__host__ __device__ __forceinline__ void decode_banded(long long u, int n, int H, int &r, int &c)
{
    int g0 = 0;      // first row of the band
    for (;;) {
        const int h = (n - g0) < H ? (n - g0) : H;
        const long long cnt = (long long)h * (h + 1) / 2 + (long long)h * (n - g0 - h);
        if (u < cnt || g0 + h >= n) {
            const long long tri = (long long)h * (h + 1) / 2;
            if (u < tri) {                       // the band's diagonal corner: columns g0 .. g0+h-1
                int j = 0;
                while ((long long)(j + 1) * (j + 2) / 2 <= u) ++j;
                c = g0 + j;
                r = g0 + (int)(u - (long long)j * (j + 1) / 2);
            } else {
                const long long w = u - tri;
                c = g0 + h + (int)(w / h);
                r = g0 + (int)(w % h);
            }
            return;
        }
        u -= cnt;
        g0 += h;
    }
}

// Split mode: linear tile index -> (ab pair block, cd pair block).  Super-rows of S ab-blocks; inside a super-row,
// super-columns of S cd-blocks; inside a super-tile cd-major ((ab) fastest).  I = index arithmetic type (32-bit when n_tiles fits:
// 64-bit divisions are ~150-instruction subroutines, and every warp decodes every tile).
template <typename I>
__host__ __device__ __forceinline__ void decode_tile2_t(const FusedParams &p, I T, long long &ab, long long &cd)
{
    const I S = (I)p.supertile, n_ab = (I)p.n_ab_blk, n_cd = (I)p.n_cd_blk;
    const I per_sr = S * n_cd;
    const I sr = T / per_sr;
    const I rem = T - sr * per_sr;
    const I rows = (n_ab - sr * S) < S ? (n_ab - sr * S) : S;
    const I sc = rem / (rows * S);
    const I rem2 = rem - sc * rows * S;
    const I cdl = rem2 / rows;                    // (ab) fastest: see decode_tile4_t
    ab = (long long)(sr * S + (rem2 - cdl * rows));
    cd = (long long)(sc * S + cdl);
}

__host__ __device__ __forceinline__ void decode_tile2(const FusedParams &p, long long T, long long &ab, long long &cd)
{
    if (p.idx32)
        decode_tile2_t<unsigned>(p, (unsigned)T, ab, cd);
    else
        decode_tile2_t<long long>(p, T, ab, cd);
}

// Full mode: linear tile index -> block quadruple (A, B, C, D).  The block space is cut into super-tiles of
// SA x SB x SC x SD blocks (ragged at the edges, no holes), enumerated (A, B) outer / (C, D) inner; the ~148 tiles in
// flight then share SA*SC + SB*SD slabs of L, SA*SB blocks of R and SC*SD blocks of t, all of which stay L2-resident.
template <typename I>
__host__ __device__ __forceinline__ void decode_tile4_t(const FusedParams &p, I T, int &A, int &B, int &Cb, int &D)
{
    auto mn = [](I a, I b) { return a < b ? a : b; };
    const I nA = (I)p.nA, nB = (I)p.nB, nC = (I)p.nC, nD = (I)p.nD;
    const I SA = (I)p.SA, SB = (I)p.SB, SC = (I)p.SC, SD = (I)p.SD;
    I per = SA * nB * nC * nD;
    const I sa = T / per;
    T -= sa * per;
    const I na = mn(SA, nA - sa * SA);
    per = na * SB * nC * nD;
    const I sb = T / per;
    T -= sb * per;
    const I nb = mn(SB, nB - sb * SB);
    per = na * nb * SC * nD;
    const I sc = T / per;
    T -= sc * per;
    const I nc = mn(SC, nC - sc * SC);
    per = na * nb * nc * SD;
    const I sd = T / per;
    T -= sd * per;
    const I nd = mn(SD, nD - sd * SD);
    // inside the super-tile: (c, d, a, b) with b fastest.  The grid (148 CTAs) and the super-tile (144 tiles) are
    // not multiples of each other, so the tiles in flight straddle two super-tiles; with (a,b) fastest the straddle
    // adds one or two (c,d) blocks (t blocks, L slabs) to the live set instead of a whole second super-tile's.
    const I q1 = T / nb, bl = T - q1 * nb;
    const I q2 = q1 / na, al = q1 - q2 * na;
    const I cl = q2 / nd, dl = q2 - cl * nd;
    A = (int)(sa * SA + al);
    B = (int)(sb * SB + bl);
    Cb = (int)(sc * SC + cl);
    D = (int)(sd * SD + dl);
}

__host__ __device__ __forceinline__ void decode_tile4(const FusedParams &p, long long T, int &A, int &B, int &Cb, int &D)
{
    if (p.idx32)
        decode_tile4_t<unsigned>(p, (unsigned)T, A, B, Cb, D);
    else
        decode_tile4_t<long long>(p, T, A, B, Cb, D);
}

template <int TA_, int TB_, int TC_, int TD_, int KS_, int NW_ = 8, int G1S_ = 4>
struct WsCfg {
    static constexpr int TA = TA_, TB = TB_, TC = TC_, TD = TD_;
    static constexpr int M1 = TA * TC;          // GEMM-1 tile rows  (a,c)
    static constexpr int N1 = TB * TD;          // GEMM-1 tile cols  (b,d)
    static constexpr int NAB = TA * TB;         // (a,b) pairs per tile = GEMM-2 N
    static constexpr int NCD = TC * TD;         // (c,d) pairs per tile = GEMM-2 K
    static constexpr int NW = NW_;              // DMMA (consumer) warps: 8 (2 per SM sub-partition) or 16 (4)
    static constexpr int CONSUMERS = 32 * NW;
    // consumer warp grids (M x N).  GEMM-1: warp = wm1 * WN1 + wn1; GEMM-2: warp = wn2 * WM2 + wm2.
    static constexpr int WM1 = NW / 4, WN1 = 4;
    static constexpr int WM2 = NW / 4, WN2 = 4;
    // registers per thread after setmaxnreg: the CTA's pool is THREADS x (registers at launch)
    static constexpr int REGS_CONSUMER = (NW == 8) ? 232 : 104;
    static constexpr int REGS_PRODUCER = 40;
    static constexpr int THREADS = CONSUMERS + 128;  // + 1 producer warpgroup: warps X-lower, Y, t, X-upper (also the tile scheduler)
    static constexpr int KC = 16;               // Cholesky vectors per GEMM-1 stage
    static constexpr int PX = M1 + 4;           // pitch of a staged L row (== 4 mod 16 doubles: conflict-free LDS.64)
    static constexpr int PY = N1 + 4;
    static constexpr int G1_STAGE = KC * (PX + PY);
    static constexpr int G1_STAGES = G1S_;     // depth of the GEMM-1 stage ring (plus the head slot)
    // park a finished chunk's sums in a second register set and drain them under the next chunk (else: reduce at once)
    static constexpr bool PARK = (TA_ * TB_ <= 96);
    static constexpr int PV = NCD + ((NCD % 8 == 0) ? 4 : 0);   // pitch of Vs[(a,b)][(c,d)]: 4 or 12 mod 16
    static constexpr int V_DOUBLES = NAB * PV;
    static constexpr int MC = 64;               // ij rows per GEMM-2 chunk
    static constexpr int KS = KS_;              // (c,d) pairs per staged t slab
    static constexpr int NKS = NCD / KS;
    static constexpr int PT = KS + ((KS % 8 == 0) ? 4 : 0);
    static constexpr int T_STAGE = MC * PT;
    static constexpr int REGION0 = (V_DOUBLES > G1_STAGES * G1_STAGE) ? V_DOUBLES : G1_STAGES * G1_STAGE;
    // The first GEMM-1 stage of a tile has a slot of its own ("head", slot index G1_STAGES) outside REGION0, so the
    // producers can fetch it while the previous tile's GEMM-2 still reads Vs.
    static constexpr bool fits(int ts) { return (REGION0 + ts * T_STAGE + G1_STAGE) * 8 + 512 <= 232448; }
    static constexpr int T_STAGES = fits(4) ? 4 : (fits(3) ? 3 : 2);   // depth of the t slab ring: what shared memory leaves
    static constexpr int QD = 4;                // depth of the tile-index queue of the dynamic scheduler
    // [g1_full | g1_empty | t_full | t_empty | r0_free | x_free | x_landed | q_full x QD | q_empty x QD | q entries x QD]
    static constexpr int NBARS = 2 * (G1_STAGES + 1) + 2 * T_STAGES + 3 + 3 * QD;
    static constexpr int SMEM_BYTES = (REGION0 + T_STAGES * T_STAGE + G1_STAGE) * 8 + NBARS * 8;
    // consumer warp tiling.  GEMM-1: 2 (M) x 4 (N), wm = warp>>2; GEMM-2: 2 (M) x 4 (N), wn = warp>>1.
    static constexpr int MI1 = M1 / WM1 / 8, NI1 = N1 / WN1 / 8;
    static constexpr int MI2 = MC / WM2 / 8, NI2 = NAB / WN2 / 8;
    static_assert(NW == 8 || NW == 16, "consumer warps");
    static_assert(M1 % (8 * WM1) == 0 && N1 % (8 * WN1) == 0 && MC % (8 * WM2) == 0 && NAB % (8 * WN2) == 0,
                  "warp tiles are whole 8 x 8 fragments");
    static_assert(M1 % 16 == 0 && N1 % 32 == 0, "GEMM-1 warp grid 2 x 4 of 8 x 8 fragments");
    static_assert(MI1 * NI1 <= 32, "GEMM-1 accumulators: at most 64 doubles per lane");
    static_assert(NAB % 32 == 0, "GEMM-2 warp grid 2 x 4");
    static_assert(TC % 2 == 0 && TD % 2 == 0, "16-byte copies and regroup stores need even c and d block widths");
    static_assert(NCD % KS == 0 && KS % 4 == 0, "t slabs");
    static_assert(PV % 16 == 4 || PV % 16 == 12, "Vs pitch must be conflict-free");
    static_assert(PT % 16 == 4 || PT % 16 == 12, "t slab pitch must be conflict-free");
    static_assert(SMEM_BYTES <= 232448, "shared memory");
};

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}

template <int NTHREADS>
__device__ __forceinline__ void consumer_sync()   // named barrier 1: the consumer warps only
{
    asm volatile("bar.sync 1, %0;\n" ::"n"(NTHREADS) : "memory");
}

// cluster-scope handshakes of split mode (CTA pairs)
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr)
{
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];\n" ::"r"(cluster_addr) : "memory");
}

__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "CCL_MBARC_WAIT:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
        "@p bra CCL_MBARC_DONE;\n"
        "bra CCL_MBARC_WAIT;\n"
        "CCL_MBARC_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// ---------------------------------------------------------------------------------------------------- tile source
// Where a warp's next tile index comes from.  Static: blockIdx.x + k * gridDim.x.  Dynamic (full mode): the CTA's
// scheduler warp draws indices from a global counter and publishes them through a QD-deep queue in shared memory
// ("full" barrier: one arrival by the scheduler; "empty": one arrival by each of the 4 producer and NW consumer warps).
// With static round-robin the CTAs that share a t block or an L slab (neighbouring indices) drift apart in time over
// the thousands of tiles each of them runs, until the 126 MB L2 no longer holds a line from one sharer's read to the
// next and every tile fetches its 9-12 MB from HBM (profiles/round2_ncu.md: 68 TB per evaluation at configs[4]).  Handing
// out tiles in index order keeps the tiles in flight the ~148 most recent indices, started a few microseconds apart.
struct TileSource {
    long long next, step, n_tiles;      // static
    uint32_t q_full, q_empty, q_data;   // dynamic: shared-memory addresses
    uint32_t qn;                        // entries consumed so far
    bool dynamic;
};

template <class C>
__device__ __forceinline__ TileSource make_tile_source(const FusedParams &p, long long first, long long step, uint32_t bars_u32)
{
    TileSource ts;
    ts.next = first;
    ts.step = step;
    ts.n_tiles = p.n_tiles;
    ts.q_full = bars_u32 + 8u * (2 * (C::G1_STAGES + 1) + 2 * C::T_STAGES + 3);
    ts.q_empty = ts.q_full + 8u * C::QD;
    ts.q_data = ts.q_empty + 8u * C::QD;
    ts.qn = 0;
    ts.dynamic = p.tile_counter != nullptr;
    return ts;
}

template <class C>
__device__ __forceinline__ bool next_tile(TileSource &ts, int lane, long long &T)
{
    if (!ts.dynamic) {
        T = ts.next;
        ts.next += ts.step;
        return T < ts.n_tiles;
    }
    const uint32_t slot = ts.qn % C::QD, ph = (ts.qn / C::QD) & 1u;
    mbar_wait(ts.q_full + 8u * slot, ph);
    asm volatile("ld.shared.s64 %0, [%1];\n" : "=l"(T) : "r"(ts.q_data + 8u * slot) : "memory");
    __syncwarp();
    if (T >= ts.n_tiles) return false;          // the sentinel: the scheduler has stopped, nothing to release
    if (lane == 0) mbar_arrive(ts.q_empty + 8u * slot);
    ++ts.qn;
    return true;
}

// The scheduler of a CTA: a duty of the producer warpgroup's fourth warp (which also copies half of the X slabs).  It keeps
// the queue ahead of its readers: entry n may be written once every reader has consumed entry n - QD.
struct TileScheduler {
    uint32_t written;      // entries published so far
    bool on, done;         // dynamic scheduling in use; the sentinel has been published
};

template <class C>
__device__ __forceinline__ void sched_publish(const FusedParams &p, const TileSource &ts, TileScheduler &sc, int lane)
{
    const uint32_t slot = sc.written % C::QD;
    long long T = 0;
    if (lane == 0) {
        T = (long long)atomicAdd(p.tile_counter, 1ULL);
        asm volatile("st.shared.s64 [%0], %1;\n" ::"r"(ts.q_data + 8u * slot), "l"(T) : "memory");
        mbar_arrive(ts.q_full + 8u * slot);
    }
    T = __shfl_sync(0xffffffffu, T, 0);
    ++sc.written;
    if (T >= p.n_tiles) sc.done = true;
}

// Called by the scheduler warp before it reads its own next entry (index ts.qn): publish whatever the queue has room for
// (non-blocking), and at least the entry this warp is about to read (its slot is free: this warp is the last reader of
// entry qn - QD that can be behind, all others only ever wait for this warp's copies of tiles it has already finished).
template <class C>
__device__ __forceinline__ void sched_pump(const FusedParams &p, const TileSource &ts, TileScheduler &sc, int lane)
{
    if (!sc.on) return;
    while (!sc.done) {
        const uint32_t slot = sc.written % C::QD, ph = (sc.written / C::QD) & 1u;
        if (sc.written > ts.qn) {
            if (!__shfl_sync(0xffffffffu, (int)mbar_test(ts.q_empty + 8u * slot, ph ^ 1u), 0)) break;
        } else {
            mbar_wait(ts.q_empty + 8u * slot, ph ^ 1u);
        }
        sched_publish<C>(p, ts, sc, lane);
    }
}

// ---------------------------------------------------------------------------------------------------- producers
// Four warps, one in each SM sub-partition (roles 0 and 3: the lower / upper half of the Cholesky vectors of every
// X = L[P, A, C] stage, role 1: Y = L[P, B, D] stages, role 2: t slabs; role 3 is also the CTA's tile scheduler).
// Each walks the same tile list as the consumers and keeps its ring full: per tile nk GEMM-1 stages of KC Cholesky
// vectors, and the t slabs of GEMM-2.  A slot is refilled when all 8 consumer warps have released it ("empty" barrier);
// every lane's copies report to the slot's "full" barrier when they land (cp.async.mbarrier.arrive.noinc).
// Out-of-range elements are zero-filled.  A lane owns fixed positions inside a staged row, so that per copy only one
// pointer addition and one predicate remain.

// One operand slab of GEMM-1: rows (r_l, w_l) of a [TR x TW] block pair, TR*TW = ROWLEN doubles per Cholesky vector,
// shared-memory pitch PITCH.  r0 / w0: first orbital index of the block along the slow / fast axis of L[P][r][w].
// PL0, PL1: the staged rows (Cholesky vectors of a stage) this warp copies -- the X slab is split between two warps.
// FAST8: the full-stage path also with 8-byte copies (full mode; in split mode, where a stage of the square partition is
// twice as many copies per warp, issuing them back to back measured 1.2 % slower than the general path's loop).
template <class C, bool ALIGN2, bool FAST8, int TW, int ROWLEN, int PITCH, int PL0, int PL1>
__device__ __forceinline__ void ws_produce_l(const FusedParams &p, const double *const Lb, const size_t ps,
                                             const int rstride, const int nrows, int lane, int r0, int w0, int nk,
                                             uint32_t &g1_it, uint32_t tiles_done, uint32_t ring_u32, uint32_t head_u32,
                                             uint32_t g1_full, uint32_t g1_empty, uint32_t r0_free)
{
    constexpr int CPR = ROWLEN / 2;              // 16-byte chunks per staged row
    constexpr int NPOS = (CPR + 31) / 32;        // chunk positions per lane
    int off[NPOS];          // (r0 + r_l) * rstride + w0 + w_l of the chunk's first element; -1: row outside the operand, or no chunk
    bool ok1[NPOS];         // second element inside (8-byte copies only)
    uint32_t dst[NPOS];
#pragma unroll
    for (int k = 0; k < NPOS; ++k) {
        const int mc = lane + 32 * k, m = 2 * mc;
        const int r = r0 + m / TW, w = w0 + m % TW;
        const bool ok = (mc < CPR) && (r < nrows) && (w < p.v);
        off[k] = ok ? r * rstride + w : -1;
        ok1[k] = ok && (w + 1 < p.v);
        dst[k] = (uint32_t)(m * 8);
    }
    const size_t psb = ps * sizeof(double);
    // running source pointers of the lane's chunks (they advance by one Cholesky vector per staged row, across the
    // stages of the tile): a chunk outside the operand reads nothing (zero fill), from the start of the vector
    const char *cur[NPOS];
    const char *cur1[NPOS];         // 8-byte copies only: the chunk's second element (the first again where it does not exist)
#pragma unroll
    for (int k = 0; k < NPOS; ++k) {
        cur[k] = reinterpret_cast<const char *>(Lb + (off[k] >= 0 ? off[k] : 0)) + PL0 * psb;
        cur1[k] = cur[k] + (ok1[k] ? 8 : 0);
    }
    for (int kc = 0; kc < nk; ++kc) {
        // stage 0 of a tile goes to the head slot (free as soon as the previous tile's first stage was consumed);
        // the others go round the ring, which shares its shared memory with Vs: before the first of them the
        // previous tile's GEMM-2 must be over in every consumer warp (r0_free).  g1_it counts ring stages.
        uint32_t slot, ph, sb;
        if (kc == 0) {
            slot = C::G1_STAGES;
            ph = tiles_done & 1u;
            sb = head_u32;
        } else {
            if (kc == 1 && tiles_done > 0) mbar_wait(r0_free, (tiles_done - 1u) & 1u);
            slot = g1_it % C::G1_STAGES;
            ph = (g1_it / C::G1_STAGES) & 1u;
            sb = ring_u32 + slot * (uint32_t)(C::G1_STAGE * 8);
            ++g1_it;
        }
        mbar_wait(g1_empty + 8u * slot, ph ^ 1u);
        const int P0 = kc * C::KC;
        const int prow = p.x - P0;               // Cholesky vectors left: rows pl >= prow are zero-filled
        const double *Lk = Lb + (size_t)P0 * ps;
        if ((ALIGN2 || FAST8) && prow >= C::KC) {
            // Full stage (all but a tile's last): a copy costs one 64-bit pointer increment -- the producer shares its SM
            // sub-partition's issue slots with two DMMA warps, and every instruction it does not issue is a cycle the DMMA
            // stream is not held up (the consumers next to the X producer ran 5 % behind the others, profiles/round2_ncu.md)
            uint32_t sd[NPOS];
#pragma unroll
            for (int k = 0; k < NPOS; ++k) sd[k] = sb + dst[k];
#pragma unroll
            for (int pl = PL0; pl < PL1; ++pl) {
#pragma unroll
                for (int k = 0; k < NPOS; ++k)
                    if (NPOS * 32 == CPR || lane + 32 * k < CPR) {
                        const size_t step = (pl + 1 == PL1) ? (C::KC - (PL1 - PL0) + 1) * psb : psb;   // last row: on to this
                        if (ALIGN2) {                                                                  // warp's rows of the next stage
                            cp_async_16(sd[k] + (uint32_t)(pl * PITCH * 8), cur[k], off[k] >= 0);
                        } else {
                            cp_async_8(sd[k] + (uint32_t)(pl * PITCH * 8), cur[k], off[k] >= 0);
                            cp_async_8(sd[k] + (uint32_t)(pl * PITCH * 8 + 8), cur1[k], ok1[k]);
                            cur1[k] += step;
                            asm volatile("" : "+l"(cur1[k]));
                        }
                        cur[k] += step;
                        asm volatile("" : "+l"(cur[k]));      // keep the increment an increment (ptxas would rebuild base + pl * psb)
                    }
            }
        } else {
#pragma unroll 4
            for (int pl = PL0; pl < PL1; ++pl) {
#pragma unroll
                for (int k = 0; k < NPOS; ++k) {
                    if (NPOS * 32 == CPR || lane + 32 * k < CPR) {
                        const bool ok = (off[k] >= 0) && (pl < prow);
                        const double *src = ok ? Lk + (size_t)pl * ps + off[k] : Lb;
                        const uint32_t d = sb + (uint32_t)(pl * PITCH * 8) + dst[k];
                        if (ALIGN2) {
                            cp_async_16(d, src, ok);
                        } else {
                            cp_async_8(d, src, ok);
                            cp_async_8(d + 8, (ok && ok1[k]) ? src + 1 : Lb, ok && ok1[k]);
                        }
                    }
                }
            }
        }
        cp_async_mbar_arrive(g1_full + 8u * slot);
    }
}

// 8-fold-symmetry mode (SYMM): of a tile (A,B,C,D) and its mirror (C,D,A,B) only the one with (A,B) <= (C,D)
// (lexicographic) is processed; its integral tile then serves both R[:, (a,b)] and R[:, (c,d)].
__device__ __forceinline__ bool symm_canonical(int A, int B, int Cb, int D) { return A < Cb || (A == Cb && B <= D); }

template <class C, bool ALIGN2, bool SPLIT, bool IAJB, bool SYMM>
__device__ __forceinline__ void ws_producer(const FusedParams &p, const int role, uint32_t rank, long long tile_first,
                                            long long tile_step, uint32_t region0_u32, uint32_t tbuf_u32,
                                            uint32_t bars_u32)
{
    const int lane = threadIdx.x & 31;
    const size_t v = (size_t)p.v, vv = v * v;
    const int nk = (p.x + C::KC - 1) / C::KC;
    const long long nchunks = (p.oo + C::MC - 1) / C::MC;
    const double *const t_in = (SPLIT && rank) ? p.tm : p.t;
    const uint32_t g1_full = bars_u32, g1_empty = bars_u32 + 8u * (C::G1_STAGES + 1);
    const uint32_t t_full = bars_u32 + 16u * (C::G1_STAGES + 1), t_empty = t_full + 8u * C::T_STAGES;
    const uint32_t r0_free = t_empty + 8u * C::T_STAGES;
    const uint32_t head_u32 = tbuf_u32 + (uint32_t)(C::T_STAGES * C::T_STAGE * 8);
    uint32_t g1_it = 0;                // GEMM-1 ring stages issued so far (all tiles): slot = it % STAGES, phase = it / STAGES
    uint32_t t_slot = 0, t_ph = 0;     // t ring: slot and phase parity of the next slab to fill
    uint32_t tiles_done = 0;
    // t slab copy role: RPI rows per pass, lane -> (row in pass, chunk column)
    constexpr int CPT = C::KS / 2;                       // 16-byte chunks per slab row
    constexpr int RPI = (32 / CPT) > 0 ? (32 / CPT) : 1; // rows per pass of the warp
    constexpr int CPL = (CPT + 31) / 32;                 // chunk columns per lane (1 unless KS > 64)
    static_assert(CPL == 1, "t slab rows of at most 32 chunks");
    const int t_rl = lane / CPT, t_kl = 2 * (lane % CPT);
    const bool t_lane = lane < RPI * CPT;

    TileSource tiles = make_tile_source<C>(p, tile_first, tile_step, bars_u32);
    TileScheduler sched = {0u, role == 3 && tiles.dynamic, false};
    for (long long T;;) {
        sched_pump<C>(p, tiles, sched, lane);
        if (!next_tile<C>(tiles, lane, T)) break;
        int A, B, Cb, D;
        if (SPLIT) {
            long long ab_blk, cd_blk;
            decode_tile2(p, T, ab_blk, cd_blk);
            decode_banded(ab_blk, p.nA, p.SA, A, B);
            decode_banded(cd_blk, p.nC, p.SC, Cb, D);
        } else {
            decode_tile4(p, T, A, B, Cb, D);
        }
        if (SYMM && !symm_canonical(A, B, Cb, D)) continue;
        const int a0 = A * C::TA, b0 = B * C::TB, c0 = Cb * C::TC, d0 = D * C::TD;
        // rows of the GEMM-1 tile are (ra, c), columns (rb, d): (a, b) from (X, Y), or (b, a) from (Y, X) on rank 1 of a
        // split pair / in the exchange variant
        const int ra0 = rank ? b0 : a0, rb0 = rank ? a0 : b0;

        if (role != 2) {
            // roles 0 and 3 copy the lower / upper half of the rows (Cholesky vectors) of every X stage, role 1 the Y stage:
            // three warps in three SM sub-partitions with about the same number of copies each
            const bool from_x = (role != 1) != (rank != 0);      // which operand array feeds this role
            const double *const Lb = from_x ? p.X : p.Y;
            const size_t ps = (size_t)(from_x ? p.xps : p.yps);
            const int rstride = (int)(from_x ? p.xrs : p.yrs), nrows = from_x ? p.nr : p.ns;
            constexpr int HK = C::KC / 2;
            if (role == 0)
                ws_produce_l<C, ALIGN2, !SPLIT, C::TC, C::M1, C::PX, 0, HK>(p, Lb, ps, rstride, nrows, lane, ra0, c0, nk, g1_it,
                                                                    tiles_done, region0_u32, head_u32, g1_full, g1_empty,
                                                                    r0_free);
            else if (role == 3)
                ws_produce_l<C, ALIGN2, !SPLIT, C::TC, C::M1, C::PX, HK, C::KC>(p, Lb, ps, rstride, nrows, lane, ra0, c0, nk, g1_it,
                                                                        tiles_done, region0_u32, head_u32, g1_full,
                                                                        g1_empty, r0_free);
            else
                ws_produce_l<C, ALIGN2, !SPLIT, C::TD, C::N1, C::PY, 0, C::KC>(p, Lb, ps, rstride, nrows, lane, rb0, d0, nk, g1_it,
                                                                       tiles_done, region0_u32 + (uint32_t)(C::KC * C::PX * 8),
                                                                       head_u32 + (uint32_t)(C::KC * C::PX * 8), g1_full,
                                                                       g1_empty, r0_free);
            ++tiles_done;
            continue;
        }

        // ------------------------------------------------------------------ t slabs: slab (chunk, ksi) holds rows
        // [chunk*MC, +MC) and the (c,d) pairs k in [ksi*KS, +KS), k = c_l*TD + d_l.  SYMM: a second sweep over the
        // (a,b) pairs of the tile (same partition: TA = TC, TB = TD) feeds the contraction with the transposed tile.
        for (int sweep = 0; sweep < ((SYMM && !(A == Cb && B == D)) ? 2 : 1); ++sweep) {
        const int c0 = sweep ? a0 : Cb * C::TC, d0 = sweep ? b0 : D * C::TD;
        for (long long chunk = 0; chunk < nchunks; ++chunk) {
            const long long rows_left = p.oo - chunk * C::MC;        // rows rl >= rows_left are zero-filled
            // first row of this lane in the chunk; IAJB: rows are (i,j) pairs at i*(v*o*v) + j*v, walked incrementally
            const unsigned row_first = (unsigned)(chunk * C::MC + t_rl);
            const unsigned i_first = IAJB ? row_first / (unsigned)p.o : 0u, j_first = IAJB ? row_first - i_first * (unsigned)p.o : 0u;
            // split mode: rows of the packed triangle T+ (rank 0) / T- (rank 1)
            const size_t trow = SPLIT ? (size_t)p.tri_nt : vv;
            const double *t_chunk = t_in + (IAJB ? (size_t)i_first * (size_t)p.ovv + (size_t)j_first * v : (size_t)row_first * trow);
            const size_t cstride = IAJB ? (size_t)p.o * v : v;       // stride of c in t
            const size_t row_step = IAJB ? (size_t)RPI * v : (size_t)RPI * trow;
            const size_t wrap_step = IAJB ? (size_t)p.ovv - (size_t)p.o * v : 0;   // extra offset when j wraps into i+1
            for (int ksi = 0; ksi < C::NKS; ++ksi) {
                const uint32_t slot = t_slot, ph = t_ph;
                if (++t_slot == C::T_STAGES) { t_slot = 0; t_ph ^= 1u; }
                mbar_wait(t_empty + 8u * slot, ph ^ 1u);
                const int k = ksi * C::KS + t_kl;
                const int c = c0 + k / C::TD, d = d0 + k % C::TD;
                // validity of the chunk's two elements (d, d+1).  Split mode reads the packed upper triangle: row c owns
                // the slot d in [4*floor(c/4), v4) at tri_base(c) + d (16-byte aligned for even d); its entries left of
                // the diagonal and in the padding are zeros, and what lies left of the slot is zero-filled here: the
                // lower halves of the diagonal block pairs (which hold every pair a second time) contribute nothing.
                bool ok0, ok1;
                long long eoff;
                if (SPLIT) {
                    ok0 = ok1 = t_lane && (c < p.v) && (d >= (c & ~3)) && (d < (int)p.tri_v4);
                    eoff = tri_base(c, p.tri_v4) + d;
                } else {
                    ok0 = t_lane && (c < p.v) && (d < p.v);
                    ok1 = ok0 && (d + 1 < p.v);
                    eoff = (long long)((size_t)c * cstride + d);
                }
                const double *src = t_chunk + ((ok0 || ok1) ? eoff : 0);
                uint32_t dst = tbuf_u32 + slot * (uint32_t)(C::T_STAGE * 8) + (uint32_t)((t_rl * C::PT + t_kl) * 8);
                unsigned j = j_first;
                if (!IAJB && rows_left >= C::MC) {
                    // full chunk: one 64-bit pointer increment per copy (see ws_produce_l)
                    if (t_lane) {
                        const char *s8 = reinterpret_cast<const char *>(src);
                        const char *s8b = s8 + (ok1 ? 8 : 0);       // 8-byte copies only: the chunk's second element
                        const size_t step8 = row_step * sizeof(double);
#pragma unroll
                        for (int it = 0; it < (C::MC + RPI - 1) / RPI; ++it) {
                            if (C::MC % RPI == 0 || t_rl + it * RPI < C::MC) {
                                if (ALIGN2 || SPLIT) {
                                    cp_async_16(dst + (uint32_t)(it * RPI * C::PT * 8), s8, ok0);
                                } else {
                                    cp_async_8(dst + (uint32_t)(it * RPI * C::PT * 8), s8, ok0);
                                    cp_async_8(dst + (uint32_t)(it * RPI * C::PT * 8 + 8), s8b, ok1);
                                }
                            }
                            s8 += step8;
                            asm volatile("" : "+l"(s8));
                            if (!(ALIGN2 || SPLIT)) {
                                s8b += step8;
                                asm volatile("" : "+l"(s8b));
                            }
                        }
                    }
                } else if (t_lane) {
#pragma unroll 4
                    for (int rl = t_rl; rl < C::MC; rl += RPI) {
                        const bool row_ok = rl < rows_left;
                        if (ALIGN2 || SPLIT) {
                            cp_async_16(dst, (ok0 && row_ok) ? src : t_in, ok0 && row_ok);
                        } else {
                            cp_async_8(dst, (ok0 && row_ok) ? src : t_in, ok0 && row_ok);
                            cp_async_8(dst + 8, (ok1 && row_ok) ? src + 1 : t_in, ok1 && row_ok);
                        }
                        src += row_step;
                        if (IAJB) {
                            j += RPI;
                            while (j >= (unsigned)p.o) {
                                j -= (unsigned)p.o;
                                src += wrap_step;
                            }
                        }
                        dst += (uint32_t)(RPI * C::PT * 8);
                    }
                }
                cp_async_mbar_arrive(t_full + 8u * slot);
            }
        }
        }
        ++tiles_done;
    }
    cp_async_wait<0>();   // nothing of this warp is in flight when it leaves
}

// ---------------------------------------------------------------------------------------------------- consumers
template <class C, bool SPLIT, bool IAJB, bool SYMM>
__device__ __forceinline__ void ws_consumer(const FusedParams &p, uint32_t rank, long long tile_first,
                                            long long tile_step, double *region0, double *tbuf, uint32_t region0_u32,
                                            uint32_t bars_u32)
{
    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, q = lane & 3;
    const int wm1 = warp / C::WN1, wn1 = warp % C::WN1;     // GEMM-1 warp grid (a sub-partition holds every wm1 once)
    const int wm2 = warp % C::WM2, wn2 = warp / C::WM2;     // GEMM-2 warp grid
    const size_t rs = (size_t)p.rs;               // row stride of R ([i][j][r][s] storage; split mode: of W+ / W-)
    const int nk = (p.x + C::KC - 1) / C::KC;
    const long long nchunks = (p.oo + C::MC - 1) / C::MC;
    double *const r_out = (SPLIT && rank) ? p.Rm : p.R;
    const uint32_t g1_full = bars_u32, g1_empty = bars_u32 + 8u * (C::G1_STAGES + 1);
    const uint32_t t_full = bars_u32 + 16u * (C::G1_STAGES + 1), t_empty = t_full + 8u * C::T_STAGES;
    const uint32_t r0_free = t_empty + 8u * C::T_STAGES;                          // "Vs is dead" (per tile)
    const double *const head = tbuf + C::T_STAGES * C::T_STAGE;                    // first GEMM-1 stage of a tile
    uint32_t tiles_done = 0;
    const uint32_t x_free = r0_free + 8u, x_landed = x_free + 8u;                 // split mode pair handshakes
    // per-lane fragment offsets inside a GEMM-1 stage / a t slab (plain values: making them opaque to stop ptxas from
    // rematerialising them at every stage boundary cost registers and 0.8 % of speed)
    const int xoff = wm1 * (C::M1 / C::WM1) + g + q * C::PX;
    const int yoff = C::KC * C::PX + wn1 * (C::N1 / C::WN1) + g + q * C::PY;
    const int toff = (wm2 * (C::MC / C::WM2) + g) * C::PT + q;
    uint32_t g1_it = 0, x_ph = 0;
    uint32_t tslot = 0, tph = 0;       // t ring: slot and phase parity of the next slab to consume (kept incrementally:
                                       // T_STAGES may be 3, and a division per slab is not free)

    // GEMM-2 column permutation: column n of an 8-wide output fragment is the (a,b) pair n0 + pi(n),
    // pi = [0,6,1,7,2,4,3,5]: the lane's first accumulator then sits at pair n0 + q and the second at n0 + [6,7,4,5][q],
    // so every red instruction of a warp covers 8 rows x one full 32-byte sector (when 4 | nvirt and 4 | TB), while
    // the B-fragment rows n0 + pi(g) stay bank-conflict-free.
    const int pig = (g & 1) ? (4 + (((g >> 1) + 2) & 3)) : (g >> 1);
    const int sq = (q < 2) ? (6 + q) : (2 + q);

    TileSource tiles = make_tile_source<C>(p, tile_first, tile_step, bars_u32);
    for (long long T; next_tile<C>(tiles, lane, T);) {
        int A, B, Cb, D;
        if (SPLIT) {
            long long ab_blk, cd_blk;
            decode_tile2(p, T, ab_blk, cd_blk);
            decode_banded(ab_blk, p.nA, p.SA, A, B);
            decode_banded(cd_blk, p.nC, p.SC, Cb, D);
        } else {
            decode_tile4(p, T, A, B, Cb, D);
        }
        if (SYMM && !symm_canonical(A, B, Cb, D)) continue;
        const int a0 = A * C::TA, b0 = B * C::TB;

        // ------------------------------------------------------------------ GEMM-1: (ac|bd) tile, K = nchol
        // Register-lean software pipeline: the A fragments (MI1 of them) are reloaded row by row for the next k-step
        // right after the DMMAs that used them ("rolling"), the few B fragments are double-buffered.  The next
        // stage's "full" barrier is probed one k-step early (non-blocking), and the last k-step of a stage already
        // rolls in the next stage's first fragments, so neither shared-memory latency nor the barrier round trip is
        // exposed.
        double acc1[C::MI1][C::NI1][2];
#pragma unroll
        for (int i = 0; i < C::MI1; ++i)
#pragma unroll
            for (int j = 0; j < C::NI1; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
        {
            double af[C::MI1], bfA[C::NI1], bfB[C::NI1];
            auto lda = [&](const double *Xs, int kk) {
#pragma unroll
                for (int i = 0; i < C::MI1; ++i) af[i] = Xs[kk * 4 * C::PX + i * 8];
            };
            auto ldb = [&](double(&bf)[C::NI1], const double *Ys, int kk) {
#pragma unroll
                for (int j = 0; j < C::NI1; ++j) bf[j] = Ys[kk * 4 * C::PY + j * 8];
            };
            // DMMAs of one k-step; with ROLL each A fragment is reloaded from (Xnext, kk_next) as soon as its row is done
            // (the reload of a row's fragment is issued one row of DMMAs late: an LDS into a register that a DMMA issued
            // just before still has to read waits on the scoreboard and holds up the DMMAs behind it)
            auto mm = [&](const double(&bf)[C::NI1], auto roll_tag, const double *Xnext, int kk_next) {
                constexpr bool ROLL = decltype(roll_tag)::value;
#pragma unroll
                for (int i = 0; i < C::MI1; ++i) {
#pragma unroll
                    for (int j = 0; j < C::NI1; ++j) dmma_8x8x4(acc1[i][j][0], acc1[i][j][1], af[i], bf[j]);
                    if (ROLL && i >= 1) af[i - 1] = Xnext[kk_next * 4 * C::PX + (i - 1) * 8];
                }
            };
            auto roll_last = [&](const double *Xnext, int kk_next) {      // the last row's reload, after the caller's ldb
                af[C::MI1 - 1] = Xnext[kk_next * 4 * C::PX + (C::MI1 - 1) * 8];
            };
            using std::false_type;
            using std::true_type;
            static_assert(C::KC == 16, "four k-steps per stage: the B buffers alternate A, B, A, B");
            // stage 0 sits in the head slot (index G1_STAGES, phase = tile parity), the others go round the ring
            uint32_t slot = C::G1_STAGES;
            mbar_wait(g1_full + 8u * slot, tiles_done & 1u);
            const double *Xs = head + xoff;      // lane's element of k-row 0: (row q, column wm1 * M1/WM1 + g)
            const double *Ys = head + yoff;
            lda(Xs, 0);
            ldb(bfA, Ys, 0);
            for (int kc = 0; kc < nk; ++kc) {
                const bool has_next = kc + 1 < nk;
                const uint32_t nslot = g1_it % C::G1_STAGES, nph = (g1_it / C::G1_STAGES) & 1u;
                if (has_next) ++g1_it;
                const double *Xn = region0 + nslot * C::G1_STAGE + xoff;
                const double *Yn = region0 + nslot * C::G1_STAGE + yoff;
                const int ksteps = (p.x - kc * C::KC + 3) >> 2;     // k-steps holding real Cholesky vectors
                if (ksteps >= C::KC / 4) {
                    ldb(bfB, Ys, 1);
                    mm(bfA, true_type{}, Xs, 1);
                    ldb(bfA, Ys, 2);
                    roll_last(Xs, 1);
                    mm(bfB, true_type{}, Xs, 2);
                    ldb(bfB, Ys, 3);
                    roll_last(Xs, 2);
                    const bool ready = has_next && mbar_test(g1_full + 8u * nslot, nph);
                    mm(bfA, true_type{}, Xs, 3);
                    if (has_next) {
                        if (!ready) mbar_wait(g1_full + 8u * nslot, nph);
                        ldb(bfA, Yn, 0);
                        roll_last(Xs, 3);
                        mm(bfB, true_type{}, Xn, 0);
                        roll_last(Xn, 0);
                    } else {
                        roll_last(Xs, 3);
                        mm(bfB, false_type{}, Xs, 0);
                    }
                } else {                                              // tail stage (always the last one)
#pragma unroll 1
                    for (int kk = 0; kk < ksteps; ++kk) {
                        mm(bfA, false_type{}, Xs, 0);
                        if (kk + 1 < ksteps) {
                            lda(Xs, kk + 1);
                            ldb(bfA, Ys, kk + 1);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(g1_empty + 8u * slot);
                slot = nslot;
                Xs = Xn;
                Ys = Yn;
            }
        }

        // ------------------------------------------------------------------ regroup (ac)(bd) -> Vs[(ab)][(cd)]
        // A lane's accumulator pair sits at tile row m = (ra_l, c_l) and columns n, n+1 = (rb_l, d_l), (rb_l, d_l+1):
        // two adjacent (c,d) pairs of one (a,b) pair, i.e. one 16-byte store into Vs[(a_l,b_l)][(c_l,d_l)].
        auto vs_pos = [&](int i, int j) {
            const int m = wm1 * (C::M1 / C::WM1) + i * 8 + g;
            const int n = wn1 * (C::N1 / C::WN1) + j * 8 + 2 * q;
            const int ral = m / C::TC, cl = m % C::TC, rbl = n / C::TD, dl = n % C::TD;
            const int al = rank ? rbl : ral, bl = rank ? ral : rbl;
            return (al * C::TB + bl) * C::PV + cl * C::TD + dl;
        };
        if (!SPLIT) {
            consumer_sync<C::CONSUMERS>();   // every warp is done with the stage ring: region0 may become Vs
#pragma unroll
            for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                for (int j = 0; j < C::NI1; ++j)
                    *reinterpret_cast<double2 *>(region0 + vs_pos(i, j)) = make_double2(acc1[i][j][0], acc1[i][j][1]);
        } else {
            // V+ = w/2 [(ac|bd) + (ad|bc)] on rank 0, V- = w/2 [(ac|bd) - (ad|bc)] on rank 1, w = 1/2 on diagonal (C == D)
            // block pairs (they hold every (c,d) pair twice), else 1  (reading 10).
            // Each CTA writes its tile into the partner's Vs, then folds the partner's tile into its own registers.
            const uint32_t peer = rank ^ 1u;
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(map_to_cta(x_free, peer));   // this warp no longer reads our ring
            mbar_wait_cluster(x_free, x_ph);                                // all partner warps left theirs
            const uint32_t peer_r0 = map_to_cta(region0_u32, peer);
#pragma unroll
            for (int i = 0; i < C::MI1; ++i)
#pragma unroll
                for (int j = 0; j < C::NI1; ++j)
                    st_cluster_f64x2(peer_r0 + (uint32_t)(vs_pos(i, j) * 8), acc1[i][j][0], acc1[i][j][1]);
            __syncwarp();
            if (lane == 0) mbar_arrive_remote(map_to_cta(x_landed, peer));  // release.cluster: our stores are visible
            mbar_wait_cluster(x_landed, x_ph);                               // the partner's whole tile has landed
            x_ph ^= 1u;
            const double sc = 0.5;                  // V+- = 1/2 [(ac|bd) +- (ad|bc)], diagonal block pairs included
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
        consumer_sync<C::CONSUMERS>();   // Vs complete

        // ------------------------------------------------------------------ GEMM-2: R[(ij),(ab)] += t . Vs^T
        // The 64-row chunks of t stream through the ring; the partial sums of a finished chunk are parked in a second
        // register set (pend) and leave as red.global.add.f64 a few at a time from inside the next chunk's first K
        // slab, so the reductions (fire-and-forget, done by the L2 atomic units) overlap the DMMA stream.
        // Fragments are double-buffered across k-steps and slabs exactly as in GEMM-1.
        // TRANS (SYMM mode, second sweep): R[(ij),(cd)] += t[(ij),(ab)] . Vs -- the same tile read transposed: output
        // columns are the (c,d) pairs of block (n_a0, n_b0) = (c0, d0), K runs over the (a,b) pairs = the rows of Vs.
        auto gemm2 = [&](auto trans_tag, const int a0, const int b0) {
        constexpr bool TRANS = decltype(trans_tag)::value;
        constexpr int VJ = TRANS ? 8 : 8 * C::PV;               // Vs step between the 8-wide column fragments
        constexpr int VK = TRANS ? 4 * C::PV : 4;               // ... between k-steps
        constexpr int VSLAB = TRANS ? C::KS * C::PV : C::KS;    // ... between K slabs
        const int astride = IAJB ? p.o * p.ns : p.ns;   // stride of r in R ([i][j][r][s], or the paper's [i][r][j][s])
        int off0[C::NI2], off1[C::NI2];     // r*astride + s of the lane's two columns per fragment, -1 = outside R
                                            // (r*astride + s < 2^31 is checked on the host)
#pragma unroll
        for (int j = 0; j < C::NI2; ++j) {
            const int n = wn2 * (C::NAB / C::WN2) + j * 8;
            const int aq = a0 + (n + q) / C::TB, bq = b0 + (n + q) % C::TB;
            const int as = a0 + (n + sq) / C::TB, bs = b0 + (n + sq) % C::TB;
            if (SPLIT) {
                // packed triangles W+-: row a owns the slot b in [4*floor(a/4), v4) at tri_base(a) + b (what a diagonal
                // block pair computes a second time, a > b, lands in the slot's unused entries or, like the padding
                // rows, in the row's sink), so every tile takes the unpredicated path with full 32-byte sectors
                const bool v0 = aq < p.v && bq >= (aq & ~3) && bq < (int)p.tri_v4;
                const bool v1 = as < p.v && bs >= (as & ~3) && bs < (int)p.tri_v4;
                off0[j] = (int)(v0 ? tri_base(aq, p.tri_v4) + bq : p.tri_nt + (bq & 7));
                off1[j] = (int)(v1 ? tri_base(as, p.tri_v4) + bs : p.tri_nt + (bs & 7));
            } else {
                off0[j] = (aq < p.nr && bq < p.ns) ? aq * astride + bq : -1;
                off1[j] = (as < p.nr && bs < p.ns) ? as * astride + bs : -1;
            }
        }
        const bool interior = C::PARK && (SPLIT || ((a0 + C::TA <= p.nr) && (b0 + C::TB <= p.ns)));
        double *r_row = r_out + (size_t)(wm2 * (C::MC / C::WM2) + g) * rs;    // row of fragment i = 0 in the current chunk
        const size_t vv8 = 8 * rs;
        // IAJB: rows 8 apart are not equally spaced in memory, so the row pointers of the current and of the parked
        // chunk are kept per fragment row (dead code and dead registers otherwise)
        double *rrow[C::MI2], *prw[C::MI2];

        double acc2[C::MI2][C::NI2][2], pend[C::MI2][C::NI2][2];
#pragma unroll
        for (int i = 0; i < C::MI2; ++i)
#pragma unroll
            for (int j = 0; j < C::NI2; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;

        constexpr int NK4 = C::KS / 4;                                  // k-steps per slab
        constexpr int NPAIR = C::MI2 * C::NI2;                          // accumulator pairs per lane
        constexpr int ROWS = NK4 * C::MI2;                              // rows of DMMAs (MI2 per k-step) per slab
        // The parked sums (RPSLAB = 2 * NPAIR reductions per lane and chunk) drain from inside the next chunk's first slab,
        // one after every RSTRIDE-th row of DMMAs (RPR per row if there are more reductions than rows).
        constexpr int RPSLAB = 2 * NPAIR;
        constexpr int RPR = (RPSLAB + ROWS - 1) / ROWS;
        constexpr int RSTRIDE = (RPR > 1) ? 1 : (ROWS / RPSLAB);
        static_assert(NK4 % 2 == 0, "the fragment buffers alternate A, B over an even number of k-steps per slab");

        double tfA[C::MI2], vfA[C::NI2], tfB[C::MI2], vfB[C::NI2];
        auto ldf2 = [&](double(&af)[C::MI2], double(&bf)[C::NI2], const double *Ts, const double *Vs, int k4) {
#pragma unroll
            for (int i = 0; i < C::MI2; ++i) af[i] = Ts[i * 8 * C::PT + k4 * 4];
#pragma unroll
            for (int j = 0; j < C::NI2; ++j) bf[j] = Vs[j * VJ + k4 * VK];
        };
        const double *const Ts0 = tbuf + toff;      // (row wm2 * MC/WM2 + g, column q)            + slot * T_STAGE
        const double *const Vs0 = TRANS ? region0 + q * C::PV + wn2 * (C::NAB / C::WN2) + pig   // + ksi * KS * PV
                                        : region0 + (wn2 * (C::NAB / C::WN2) + pig) * C::PV + q;  // + ksi * KS
        mbar_wait(t_full + 8u * tslot, tph);
        ldf2(tfA, vfA, Ts0 + tslot * C::T_STAGE, Vs0, 0);

        // One K slab.  FULL: all MI2 row fragments of this warp hold real rows (else only the first mi_lim);
        // PSEL >= 0: also drain part PSEL of the previous chunk's parked sums (its rows are prow, always a full chunk).
        // Sums are only parked in interior tiles (every (a,b) column inside R), so the drain needs no predicates -- ptxas
        // turns a predicated RED into a branch, which would cut the DMMA stream into three-instruction blocks.
        // On entry buffer A holds the fragments of k-step 0; on exit those of the next slab (if there is one).
        auto slab = [&](auto full_tag, auto psel_tag, int ksi, int mi_lim, double *prow, bool has_next) {
            constexpr bool FULL = decltype(full_tag)::value;
            constexpr int PSEL = decltype(psel_tag)::value;
            const double *Ts = Ts0 + tslot * C::T_STAGE;
            const double *Vs = Vs0 + ksi * VSLAB;
            const uint32_t nslot = (tslot + 1 == C::T_STAGES) ? 0u : tslot + 1u, nph = tph ^ (nslot == 0u ? 1u : 0u);
            const double *Tn = Ts0 + nslot * C::T_STAGE;
            const double *Vn = Vs0 + (ksi + 1 == C::NKS ? 0 : ksi + 1) * VSLAB;
            bool ready = false;
            double *pp = nullptr;       // row pointer of the parked reductions in flight (PSEL >= 0)
            // k-step k4: MI2 x NI2 DMMAs on (af, bf).  LD: the other buffer pair (naf, nbf) is refilled from (Tl, Vl, kl)
            // from inside this k-step, one row of DMMAs after the k-step that last read it has been issued (an LDS
            // into a register a just-issued DMMA still has to read would wait on the scoreboard and stall the DMMAs
            // behind it).  The parked reductions of this slab go out after every RSTRIDE-th row.
            auto mm2 = [&](const double(&af)[C::MI2], const double(&bf)[C::NI2], int k4, auto ld_tag, double(&naf)[C::MI2],
                           double(&nbf)[C::NI2], const double *Tl, const double *Vl, int kl) {
                constexpr bool LD = decltype(ld_tag)::value;
#pragma unroll
                for (int i = 0; i < C::MI2; ++i) {
                    if (FULL || i < mi_lim) {
#pragma unroll
                        for (int j = 0; j < C::NI2; ++j) dmma_8x8x4(acc2[i][j][0], acc2[i][j][1], af[i], bf[j]);
                    }
                    if (LD && i == 0) {
#pragma unroll
                        for (int ii = 0; ii < C::MI2; ++ii) naf[ii] = Tl[ii * 8 * C::PT + kl * 4];
                    }
                    if (LD && i == (C::MI2 > 1 ? 1 : 0)) {
#pragma unroll
                        for (int j = 0; j < C::NI2; ++j) nbf[j] = Vl[j * VJ + kl * VK];
                    }
                    if (PSEL >= 0) {
                        const int row = k4 * C::MI2 + i;                 // 0 .. ROWS-1
                        if (row % RSTRIDE == 0) {
#pragma unroll
                            for (int u = 0; u < RPR; ++u) {
                                const int w = (row / RSTRIDE) * RPR + u;  // reduction index within this slab's share
                                const int e = PSEL * RPSLAB + w;
                                if (w < RPSLAB && e < 2 * NPAIR) {
                                    const int pi = (e >> 1) / C::NI2, pj = (e >> 1) % C::NI2;
                                    // one running row pointer (the reductions go out row fragment by row fragment), so that a
                                    // reduction costs one multiply-add for its address instead of the 64-bit sums ptxas
                                    // otherwise builds per (row, column) pair
                                    if (e % (2 * C::NI2) == 0) {
                                        if (IAJB) pp = prw[pi];
                                        else if (e == PSEL * RPSLAB) pp = prow + (size_t)pi * vv8;
                                        else pp += vv8;
                                        asm volatile("" : "+l"(pp));
                                    }
                                    if (e & 1) red_add_f64(pp + off1[pj], pend[pi][pj][1]);     // interior tile: no check
                                    else red_add_f64(pp + off0[pj], pend[pi][pj][0]);
                                }
                            }
                        }
                    }
                }
            };
            using std::false_type;
            using std::true_type;
#pragma unroll
            for (int k4 = 0; k4 < NK4; k4 += 2) {
                mm2(tfA, vfA, k4, true_type{}, tfB, vfB, Ts, Vs, k4 + 1);
                if (k4 + 2 < NK4) {
                    if (k4 + 4 >= NK4) ready = has_next && mbar_test(t_full + 8u * nslot, nph);
                    mm2(tfB, vfB, k4 + 1, true_type{}, tfA, vfA, Ts, Vs, k4 + 2);
                } else if (has_next) {
                    if (!ready) mbar_wait(t_full + 8u * nslot, nph);
                    mm2(tfB, vfB, k4 + 1, true_type{}, tfA, vfA, Tn, Vn, 0);
                } else {
                    mm2(tfB, vfB, k4 + 1, false_type{}, tfA, vfA, Ts, Vs, 0);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(t_empty + 8u * tslot);
            tslot = nslot;
            tph = nph;
        };
        using std::false_type;
        using std::true_type;
        using no_pend = std::integral_constant<int, -1>;
        // all K slabs of one chunk
        // all K slabs of one chunk: the parked sums drain from inside the first slab.  (Draining in different slabs in the
        // two warps of an SM sub-partition, or spread over all slabs, measured no faster: the cost is the ~46 clk the
        // load/store unit takes per RED, during which the other warp's fragment loads queue up behind it.)
        auto chunk_slabs = [&](auto full_tag, bool drain, int mi_lim, double *prow, bool more_chunks) {
            if constexpr (C::PARK) {
                if (drain) slab(full_tag, std::integral_constant<int, 0>{}, 0, mi_lim, prow, more_chunks || C::NKS > 1);
                else slab(full_tag, no_pend{}, 0, mi_lim, prow, more_chunks || C::NKS > 1);
            } else {
                slab(full_tag, no_pend{}, 0, mi_lim, prow, more_chunks || C::NKS > 1);
            }
#pragma unroll 1
            for (int ksi = 1; ksi < C::NKS; ++ksi)
                slab(full_tag, no_pend{}, ksi, mi_lim, prow, more_chunks || ksi + 1 < C::NKS);
        };

        for (long long chunk = 0; chunk < nchunks; ++chunk) {
            // row fragments of this warp that hold real rows (only the last chunk is ragged)
            const long long rows_left = p.oo - (chunk * C::MC + wm2 * (C::MC / C::WM2));
            const bool full_rows = rows_left >= C::MC / C::WM2;
            const int mi_lim = full_rows ? C::MI2 : (rows_left <= 0 ? 0 : (int)((rows_left + 7) >> 3));
            double *prow = r_row - (size_t)C::MC * rs;      // the parked chunk's rows
            if (IAJB) {
#pragma unroll
                for (int i = 0; i < C::MI2; ++i)
                    rrow[i] = r_out + row_offset<true>(p, chunk * C::MC + wm2 * (C::MC / C::WM2) + i * 8 + g, rs);
            }
            const bool more_chunks = chunk + 1 < nchunks;
            if (full_rows) chunk_slabs(true_type{}, chunk > 0 && interior, mi_lim, prow, more_chunks);
            else chunk_slabs(false_type{}, chunk > 0 && interior, mi_lim, prow, more_chunks);
            if (more_chunks && interior) {      // park the sums; they drain during the next chunk
#pragma unroll
                for (int i = 0; i < C::MI2; ++i)
#pragma unroll
                    for (int j = 0; j < C::NI2; ++j) {
                        pend[i][j][0] = acc2[i][j][0];
                        pend[i][j][1] = acc2[i][j][1];
                        acc2[i][j][0] = acc2[i][j][1] = 0.0;
                    }
                if (IAJB) {
#pragma unroll
                    for (int i = 0; i < C::MI2; ++i) prw[i] = rrow[i];
                }
            } else {                        // last chunk of the tile, or a tile on the edge of R: reduce at once, checked
#pragma unroll
                for (int i = 0; i < C::MI2; ++i) {
                    if (i < mi_lim) {
                        double *dst = IAJB ? rrow[i] : r_row + (size_t)i * vv8;
                        const bool rok = full_rows || (i * 8 + g) < rows_left;
#pragma unroll
                        for (int j = 0; j < C::NI2; ++j) {
                            red_add_f64_if(dst + off0[j], acc2[i][j][0], rok && off0[j] >= 0);
                            red_add_f64_if(dst + off1[j], acc2[i][j][1], rok && off1[j] >= 0);
                        }
                    }
#pragma unroll
                    for (int j = 0; j < C::NI2; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
                }
            }
            r_row += (size_t)C::MC * rs;
        }
        };      // gemm2

        gemm2(std::false_type{}, a0, b0);
        if constexpr (SYMM) {
            if (!(A == Cb && B == D)) gemm2(std::true_type{}, Cb * C::TC, D * C::TD);
        }

        // Vs is dead for this warp: the producers may start the next tile's stage ring in the same shared memory
        __syncwarp();
        if (lane == 0) mbar_arrive(r0_free);
        ++tiles_done;
    }
}

// ---------------------------------------------------------------------------------------------------- kernel
template <class C, bool ALIGN2, bool SPLIT, bool IAJB, bool SYMM = false>
__global__ void __launch_bounds__(C::THREADS, 1) ladder_ws_kernel(const FusedParams p)
{
    static_assert(!(SPLIT && IAJB), "the paper's [i,a,j,b] storage is a full-mode option");
    static_assert(!SYMM || (!SPLIT && !IAJB && C::TA == C::TC && C::TB == C::TD),
                  "the 8-fold-symmetry mode needs the same block partition for (a,b) and (c,d)");
    static_assert(!SPLIT || (C::TA == C::TB && C::TC == C::TD), "split mode needs square block partitions");
    // "rank 1" = GEMM-1 with a and b swapped, i.e. the exchange integrals (bc|ad) = (ad|bc) land in Vs[(a,b)][(c,d)].
    // Split mode: rank 0 of a CTA pair builds (ac|bd), rank 1 (ad|bc).  Exchange option (Eq. 7): every CTA is "rank 1".
    const uint32_t rank = SPLIT ? cluster_ctarank() : ((C::TA == C::TB && C::TC == C::TD && p.exchange) ? 1u : 0u);
    const long long tile_first = SPLIT ? (long long)(blockIdx.x >> 1) : (long long)blockIdx.x;
    const long long tile_step = SPLIT ? (long long)(gridDim.x >> 1) : (long long)gridDim.x;
    extern __shared__ __align__(16) double smem[];
    double *region0 = smem;                    // GEMM-1 stage ring, then the Vs tile
    double *tbuf = smem + C::REGION0;          // t slab ring
    const uint32_t region0_u32 = smem_u32(region0);
    const uint32_t tbuf_u32 = smem_u32(tbuf);
    const uint32_t bars_u32 = tbuf_u32 + (uint32_t)((C::T_STAGES * C::T_STAGE + C::G1_STAGE) * 8);
    if (threadIdx.x == 0) {
        // [g1_full x (G1_STAGES+1) | g1_empty x (G1_STAGES+1) | t_full x T_STAGES | t_empty x T_STAGES | r0_free |
        //  x_free | x_landed]
        constexpr int NG = C::G1_STAGES + 1;
        for (int i = 0; i < NG; ++i) {
            mbar_init(bars_u32 + 8u * i, 96);                              // the lanes of the three L producer warps
            mbar_init(bars_u32 + 8u * (NG + i), C::NW);                    // the consumer warps
        }
        for (int i = 0; i < C::T_STAGES; ++i) {
            mbar_init(bars_u32 + 8u * (2 * NG + i), 32);
            mbar_init(bars_u32 + 8u * (2 * NG + C::T_STAGES + i), C::NW);
        }
        mbar_init(bars_u32 + 8u * (2 * NG + 2 * C::T_STAGES), C::NW);       // r0_free: the consumer warps
        mbar_init(bars_u32 + 8u * (2 * NG + 2 * C::T_STAGES + 1), C::NW);   // x_free: the partner's consumer warps
        mbar_init(bars_u32 + 8u * (2 * NG + 2 * C::T_STAGES + 2), C::NW);   // x_landed
        for (int i = 0; i < C::QD; ++i) {
            mbar_init(bars_u32 + 8u * (2 * NG + 2 * C::T_STAGES + 3 + i), 1);                   // q_full: the scheduler
            mbar_init(bars_u32 + 8u * (2 * NG + 2 * C::T_STAGES + 3 + C::QD + i), 4 + C::NW);   // q_empty: every reader warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    if (SPLIT) cluster_sync_all();    // the partner's barriers exist before anything arrives on them

    // 16384 registers per SM sub-partition = 2 consumer warps x 32 x 232 + 1 producer warp x 32 x 40 (+ slack)
    if (threadIdx.x >= C::CONSUMERS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(C::REGS_PRODUCER));
        const int role = (int)(threadIdx.x - C::CONSUMERS) >> 5;
        ws_producer<C, ALIGN2, SPLIT, IAJB, SYMM>(p, role, rank, tile_first, tile_step, region0_u32, tbuf_u32, bars_u32);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(C::REGS_CONSUMER));
        ws_consumer<C, SPLIT, IAJB, SYMM>(p, rank, tile_first, tile_step, region0, tbuf, region0_u32, bars_u32);
    }

    if (SPLIT) cluster_sync_all();    // no CTA of a pair exits while its partner may still write to it
}

}  // namespace ccl
