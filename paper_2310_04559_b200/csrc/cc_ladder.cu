// C ABI of the B200-native Cholesky vvvv ladder (include/cc_ladder.h): plan / options / scheduler set-up / launches.
// Host logic only; the arithmetic lives in ladder_ws.cuh (the fused DMMA kernel), ladder_split.cuh (t+/t- pack / unpack)
// and ladder_simple.cuh (on-GPU cross-check).
#include "../../include/cc_ladder.h"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "ladder_ws.cuh"
#include "ladder_simple.cuh"
#include "ladder_split.cuh"
#include "fp64_peak.cuh"

using namespace ccl;


namespace {

// tile shapes <TA,TB,TC,TD,KS>: block edges along a (r), b (s), c, d and the (c,d) pairs per staged t slab
using CfgP2 = WsCfg<8, 12, 16, 8, 32>;        //  96 (ab) x 128 (cd): generic nvirt
using CfgP12 = WsCfg<12, 8, 12, 12, 24>;      //  96 (ab) x 144 (cd): every edge but b's divides 300 and 420
using CfgP20 = WsCfg<8, 12, 20, 8, 32>;       //  96 (ab) x 160 (cd): the auto choice for nvirt = 120, 300, 420
using CfgSplit = WsCfg<8, 8, 16, 16, 32>;     // split mode / exchange: square partitions, 64 (ab) x 256 (cd)
using CfgSplit12 = WsCfg<8, 8, 12, 12, 48>;   // split mode, CC_LADDER_OPT_TILE = 4: 12-wide (c,d) blocks (no padding when 12 | nvirt)
// 8-fold-symmetry mode: the same partition for (a,b) and (c,d), 128 x 128 pairs; 3-deep GEMM-1 ring and 2-deep t ring
// (what shared memory leaves next to the 135 KB tile), sums reduced at once instead of parked (no registers left for that)
using CfgSymm = WsCfg<16, 8, 16, 8, 32, 8, 3>;

constexpr size_t kSimpleChunkBytes = size_t(256) << 20;

}  // namespace

struct cc_ladder_plan_s {
    int o, v, x;
    int device, num_sms;
    long long l2_bytes;
    long long opt_split, opt_algo, opt_num_ctas, opt_supertile, opt_tile, opt_exchange, opt_layout;
    long long opt_schedule;       // CC_LADDER_SCHEDULE_DYNAMIC (default) / _STATIC
    unsigned long long *counters; // device: tile counters of the dynamic scheduler (two: cc_ladder_host alternates streams)
    long long opt_symm;           // 1 = L is symmetric in its orbital indices: build only (A,B) <= (C,D) integral tiles
    long long opt_index_bits;     // 0 = auto, 64 = decode tile indices in 64-bit arithmetic even when 32 bits would do
    long long opt_nr, opt_ns;     // rows of the X / Y operand blocks the info keys and the tile choice refer to (0 = nvirt)
    long long opt_host_budget;    // cc_ladder_host: device bytes it may allocate (0 = what cudaMemGetInfo reports as free)
    long long opt_host_block_rows; // cc_ladder_host: rows of a per streamed R block when everything fits (0 auto, -1 off)
    long long host_chunks;        // R column blocks the last cc_ladder_host call streamed (1 = everything resident)
    void *ws;
    size_t ws_bytes;
    char cuda_err[256];
};

namespace {

int fail_cuda(cc_ladder_plan_t p, cudaError_t e, const char *where)
{
    if (p) snprintf(p->cuda_err, sizeof(p->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return CC_LADDER_ECUDA;
}

struct TileGeom {
    int id, TA, TB, TC, TD, smem;
};

template <class C>
TileGeom geom(int id)
{
    return {id, C::TA, C::TB, C::TC, C::TD, C::SMEM_BYTES};
}

// One evaluation's operands: the ladder itself is X = Y = L, nr = ns = nvirt (Eq. 6); cc_ladder_xy passes
// rectangular blocks of Cholesky vectors (Eqs. 8-9).
struct Operands {
    const double *X, *Y;
    long long xps, xrs, yps, yrs;
    int nr, ns;
    const double *t;
    double *out;
    int counter_slot;      // which of the plan's two tile counters this launch uses (launches that may overlap differ)
};

// the 8-fold-symmetry mode applies to the plain ladder only (full mode, default storage, no exchange)
bool symm_on(const cc_ladder_plan_s *p) { return p->opt_symm && !p->opt_split && !p->opt_exchange; }

int rows_x(const cc_ladder_plan_s *p) { return p->opt_nr > 0 ? (int)p->opt_nr : p->v; }
int rows_y(const cc_ladder_plan_s *p) { return p->opt_ns > 0 ? (int)p->opt_ns : p->v; }

// padded tile-space volume of a shape: prod_dim ceil(n / T) * T
double padded_volume(int nr, int ns, int v, const TileGeom &g)
{
    auto pad = [](int n, int T) { return (double)ceil_div(n, T) * T; };
    return pad(nr, g.TA) * pad(ns, g.TB) * pad(v, g.TC) * pad(v, g.TD);
}

// step a1, plan time: the tile shape.  Auto picks the compiled shape with the least estimated time = padded volume
// (each dimension of the (r,s,c,d) space is padded to a multiple of its block edge) / relative efficiency measured on
// the B200 (profiles/): <12,8,12,12> runs ~3 % slower per flop than the other two (shorter K slabs and GEMM-1 stages
// per tile: more stage boundaries per flop).  The generic shape wins ties.  (A former penalty for shapes whose
// super-tile footprint exceeds L2 is gone: at nvirt = 520 it chose <8,12,16,8>, which moves ~15 % more bytes per flop
// than <8,12,20,8>, drew 1 kW instead of 913 W and ran 4.6 % slower under the power cap.)
TileGeom geom_of(const cc_ladder_plan_s *p, int nr, int ns)
{
    if (p->opt_split) {
        // square partitions: <8,8,16,16> unless the 12-wide (c,d) blocks of <8,8,12,12> execute at least 10 % fewer flops.
        // They execute fewer wherever 12 | nvirt (nvirt = 420: 5.5 % fewer, 300: 2.6 %) but more bytes and reductions per
        // flop (K = 144 instead of 256 per tile): measured on the final kernel, 0.4 % faster at nvirt = 300, 1.1 % slower
        // at 420, 10 % faster at nvirt = 120 (13.8 % fewer flops).  CC_LADDER_OPT_TILE = 4 / 5 force one or the other.
        if (p->opt_tile == 4) return geom<CfgSplit12>(6);
        if (p->opt_tile == 5) return geom<CfgSplit>(0);
        auto pad2 = [&](int T) { const double n = (double)ceil_div(p->v, T) * T; return n * n; };
        return (pad2(12) <= 0.90 * pad2(16)) ? geom<CfgSplit12>(6) : geom<CfgSplit>(0);
    }
    if (p->opt_exchange) return geom<CfgSplit>(4);      // the a <-> b swap needs square block partitions
    if (p->opt_symm) return geom<CfgSymm>(5);
    const TileGeom cand[3] = {geom<CfgP2>(1), geom<CfgP12>(2), geom<CfgP20>(3)};
    if (p->opt_tile >= 1 && p->opt_tile <= 3) return cand[p->opt_tile - 1];
    const double base_eff[3] = {1.0, 0.97, 1.0};
    double cost[3];
    for (int k = 0; k < 3; ++k) cost[k] = padded_volume(nr, ns, p->v, cand[k]) / base_eff[k];
    int best = 0;
    for (int k = 1; k < 3; ++k)
        if (cost[k] < 0.998 * cost[best]) best = k;
    return cand[best];
}

void fill_params(const cc_ladder_plan_s *p, const TileGeom &g, int nr, int ns, FusedParams &fp)
{
    fp.o = p->o;
    fp.v = p->v;
    fp.x = p->x;
    fp.nr = nr;
    fp.ns = ns;
    fp.oo = (long long)p->o * p->o;
    fp.rs = (long long)nr * ns;
    fp.nA = ceil_div(nr, g.TA);
    fp.nB = ceil_div(ns, g.TB);
    fp.nC = ceil_div(p->v, g.TC);
    fp.nD = ceil_div(p->v, g.TD);
    if (p->opt_split) {   // block pairs A <= B and C <= D of the square partitions
        fp.n_ab_blk = (long long)fp.nA * (fp.nA + 1) / 2;
        fp.n_cd_blk = (long long)fp.nC * (fp.nC + 1) / 2;
    } else {
        fp.n_ab_blk = (long long)fp.nA * fp.nB;
        fp.n_cd_blk = (long long)fp.nC * fp.nD;
    }
    fp.n_tiles = fp.n_ab_blk * fp.n_cd_blk;
    fp.tm = nullptr;
    fp.Rm = nullptr;
    fp.tile_counter = nullptr;
    fp.tri_nt = tri_size(p->v);
    fp.tri_v4 = tri_v4(p->v);
    if (p->opt_split) fp.rs = fp.tri_nt + 8;
    fp.exchange = p->opt_exchange ? 1 : 0;
    fp.ovv = (long long)p->v * p->o * p->v;
    fp.ovv_out = (long long)nr * p->o * ns;
    // L2 super-tile: S (ab)-blocks x S (cd)-blocks in flight, each an SA x SB (SC x SD) rectangle of blocks
    const int S = p->opt_supertile > 0 ? (int)p->opt_supertile : 12;
    fp.supertile = S;
    int sa = 1;
    while ((sa + 1) * (sa + 1) <= S) ++sa;
    fp.SA = fp.SC = sa;
    fp.SB = fp.SD = ceil_div(S, sa);
    // the device decodes tile indices in 32-bit arithmetic when its largest intermediate products fit
    // (CC_LADDER_OPT_INDEX_BITS = 64 forces the 64-bit decode; the schedule is the same either way)
    const double big = (double)fp.n_tiles * (double)(p->opt_split ? (long long)S * S : (long long)fp.SB * fp.SB);
    fp.idx32 = (big < 2.0e9 && p->opt_index_bits != 64) ? 1 : 0;
}

size_t simple_pairs_per_chunk(const cc_ladder_plan_s *p)
{
    const size_t vv = (size_t)p->v * p->v;
    size_t n = kSimpleChunkBytes / (vv * sizeof(double));
    if (n < 1) n = 1;
    if (n > vv) n = vv;
    return n;
}

template <class C, bool ALIGN2, bool SPLIT, bool IAJB, bool SYMM = false>
int launch_fused_one(cc_ladder_plan_t p, const FusedParams &fp, int grid, cudaStream_t s)
{
    auto kern = ladder_ws_kernel<C, ALIGN2, SPLIT, IAJB, SYMM>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaFuncSetAttribute");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = C::SMEM_BYTES;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    if (SPLIT) {   // CTA pairs exchanging tiles through distributed shared memory
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
    }
    if (SPLIT) {   // a persistent grid of pairs: no more clusters than can be co-resident (a GPC with an odd SM count hosts one fewer)
        int max_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&max_clusters, kern, &cfg) == cudaSuccess && max_clusters > 0 &&
            2 * max_clusters < grid)
            cfg.gridDim = dim3((unsigned)(2 * max_clusters));
        (void)cudaGetLastError();
    }
    e = cudaLaunchKernelEx(&cfg, kern, fp);
    if (e != cudaSuccess) return fail_cuda(p, e, "ladder_ws_kernel launch");
    return CC_LADDER_OK;
}

// 16-byte cp.async needs every staged row to start on a 16-byte boundary: even nvirt (rows of t), even strides of the
// X / Y blocks, 16-byte aligned bases.  Otherwise the producers fall back to 8-byte copies (the consumers are unaware).
bool aligned2(const cc_ladder_plan_s *p, const FusedParams &fp)
{
    if (p->v % 2) return false;
    if ((fp.xps | fp.xrs | fp.yps | fp.yrs) & 1) return false;
    if (((uintptr_t)fp.X | (uintptr_t)fp.Y) & 15u) return false;
    if (!p->opt_split && ((uintptr_t)fp.t & 15u)) return false;      // split mode reads its own (aligned) packed T+-
    return true;
}

template <class C, bool SPLIT>
int launch_fused(cc_ladder_plan_t p, const FusedParams &fp, int grid, cudaStream_t s)
{
    const bool a2 = aligned2(p, fp);
    if (!SPLIT && p->opt_layout == CC_LADDER_LAYOUT_IAJB) {
        if (a2) return launch_fused_one<C, true, false, true>(p, fp, grid, s);
        return launch_fused_one<C, false, false, true>(p, fp, grid, s);
    }
    if (a2) return launch_fused_one<C, true, SPLIT, false>(p, fp, grid, s);
    return launch_fused_one<C, false, SPLIT, false>(p, fp, grid, s);
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = (const char *)a, *pb = (const char *)b;
    return pa < pb + nb && pb < pa + na;
}

// bytes spanned by an operand block X[P][r][c] with strides (ps, rs)
size_t span_bytes(int x, long long ps, int nrows, long long rs, int v)
{
    return ((size_t)(x - 1) * (size_t)ps + (size_t)(nrows - 1) * (size_t)rs + (size_t)v) * sizeof(double);
}

int check_device(cc_ladder_plan_t p)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaGetDevice");
    return dev == p->device ? CC_LADDER_OK : CC_LADDER_EINVAL;      // a plan belongs to the device it was made on
}

// Enqueue one evaluation out[i,j,r,s] += sum_cd (sum_P X[P,r,c] Y[P,s,d]) t[i,j,c,d] (full mode; options exchange / layout).
int run_fused(cc_ladder_plan_t p, const Operands &op, cudaStream_t s)
{
    const TileGeom g = geom_of(p, op.nr, op.ns);
    FusedParams fp;
    fill_params(p, g, op.nr, op.ns, fp);
    fp.X = op.X;
    fp.Y = op.Y;
    fp.xps = op.xps;
    fp.xrs = op.xrs;
    fp.yps = op.yps;
    fp.yrs = op.yrs;
    fp.t = op.t;
    fp.R = op.out;
    long long grid = p->opt_num_ctas > 0 ? p->opt_num_ctas : p->num_sms;
    if (grid > fp.n_tiles) grid = fp.n_tiles;
    if (p->opt_schedule == CC_LADDER_SCHEDULE_DYNAMIC && p->counters) {     // tiles handed out in index order at run time
        fp.tile_counter = p->counters + 16 * (op.counter_slot & 1);
        cudaError_t e = cudaMemsetAsync(fp.tile_counter, 0, sizeof(unsigned long long), s);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemsetAsync(tile counter)");
    }
    if (g.id == 5) {
        if (aligned2(p, fp)) return launch_fused_one<CfgSymm, true, false, false, true>(p, fp, (int)grid, s);
        return launch_fused_one<CfgSymm, false, false, false, true>(p, fp, (int)grid, s);
    }
    if (g.id == 4) return launch_fused<CfgSplit, false>(p, fp, (int)grid, s);
    if (g.id == 2) return launch_fused<CfgP12, false>(p, fp, (int)grid, s);
    if (g.id == 3) return launch_fused<CfgP20, false>(p, fp, (int)grid, s);
    return launch_fused<CfgP2, false>(p, fp, (int)grid, s);
}

// the kernels address R with 32-bit offsets inside one (i,j) row group: r * stride_r + s must stay below 2^31
bool offsets_fit(const cc_ladder_plan_s *p, int nr, int ns)
{
    const long long lim = (1LL << 31) - 1;
    if ((long long)nr * ns > lim) return false;
    if (p->opt_layout == CC_LADDER_LAYOUT_IAJB && (long long)nr * p->o * ns > lim) return false;
    return true;
}

}  // namespace

extern "C" {

int cc_ladder_version(void) { return 200; }

const char *cc_ladder_status_string(int status)
{
    switch (status) {
        case CC_LADDER_OK: return "ok";
        case CC_LADDER_EINVAL: return "invalid argument (size <= 0, null/misaligned/overlapping pointer, bad option, wrong device)";
        case CC_LADDER_EARCH: return "current device is not a compute-capability 10.x (sm_100) GPU";
        case CC_LADDER_EWORKSPACE: return "workspace missing or too small";
        case CC_LADDER_ECUDA: return "CUDA runtime error (see cc_ladder_last_cuda_error)";
        case CC_LADDER_ENOMEM: return "out of memory";
        case CC_LADDER_ESCRATCH:
            return "problem needs more scratch than the library's static device array holds "
                   "(cc_ladder_split_static_bytes > cc_ladder_static_scratch_bytes); use cc_ladder with a workspace";
        default: return "unknown status";
    }
}

const char *cc_ladder_last_cuda_error(cc_ladder_plan_t plan) { return plan ? plan->cuda_err : ""; }

int cc_ladder_plan(cc_ladder_plan_t *plan, int nocc, int nvirt, int nchol)
{
    if (!plan) return CC_LADDER_EINVAL;
    *plan = nullptr;
    if (nocc <= 0 || nvirt <= 0 || nchol <= 0) return CC_LADDER_EINVAL;
    // nocc^2 * nvirt^2 must be addressable; nvirt^2 and nocc^2 must fit the int block arithmetic
    if (nvirt > 30000 || nocc > 30000) return CC_LADDER_EINVAL;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return CC_LADDER_ECUDA; }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return CC_LADDER_ECUDA; }
    if (prop.major != 10) return CC_LADDER_EARCH;
    cc_ladder_plan_s *p = new (std::nothrow) cc_ladder_plan_s();
    if (!p) return CC_LADDER_ENOMEM;
    memset(p, 0, sizeof(*p));
    p->o = nocc;
    p->v = nvirt;
    p->x = nchol;
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;
    p->l2_bytes = prop.l2CacheSize;
    p->opt_algo = CC_LADDER_ALGO_FUSED;
    p->host_chunks = 0;
    if (cudaMalloc(&p->counters, 256) != cudaSuccess) {      // 2 x 8 bytes used, 128 bytes apart
        (void)cudaGetLastError();
        delete p;
        return CC_LADDER_ENOMEM;
    }
    *plan = p;
    return CC_LADDER_OK;
}

int cc_ladder_set_option(cc_ladder_plan_t p, int key, long long value)
{
    if (!p) return CC_LADDER_EINVAL;
    switch (key) {
        case CC_LADDER_OPT_SPLIT:
            if (value != 0 && value != 1) return CC_LADDER_EINVAL;
            p->opt_split = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_ALGO:
            if (value != CC_LADDER_ALGO_FUSED && value != CC_LADDER_ALGO_SIMPLE) return CC_LADDER_EINVAL;
            p->opt_algo = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_NUM_CTAS:
            if (value < 0 || value > 65535) return CC_LADDER_EINVAL;
            p->opt_num_ctas = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_SUPERTILE:
            if (value < 0 || value > 4096) return CC_LADDER_EINVAL;
            p->opt_supertile = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_TILE:
            if (value < 0 || value > 5) return CC_LADDER_EINVAL;
            p->opt_tile = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_EXCHANGE:
            if (value != 0 && value != 1) return CC_LADDER_EINVAL;
            p->opt_exchange = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_LAYOUT:
            if (value != CC_LADDER_LAYOUT_IJAB && value != CC_LADDER_LAYOUT_IAJB) return CC_LADDER_EINVAL;
            p->opt_layout = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_XY_ROWS_X:
            if (value < 0 || value > 30000) return CC_LADDER_EINVAL;
            p->opt_nr = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_XY_ROWS_Y:
            if (value < 0 || value > 30000) return CC_LADDER_EINVAL;
            p->opt_ns = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_HOST_BUDGET:
            if (value < 0) return CC_LADDER_EINVAL;
            p->opt_host_budget = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_INDEX_BITS:
            if (value != 0 && value != 64) return CC_LADDER_EINVAL;
            p->opt_index_bits = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_SYMM_L:
            if (value != 0 && value != 1) return CC_LADDER_EINVAL;
            p->opt_symm = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_SCHEDULE:
            if (value != CC_LADDER_SCHEDULE_DYNAMIC && value != CC_LADDER_SCHEDULE_STATIC) return CC_LADDER_EINVAL;
            p->opt_schedule = value;
            return CC_LADDER_OK;
        case CC_LADDER_OPT_HOST_BLOCK_ROWS:
            if (value < -1 || value > 30000) return CC_LADDER_EINVAL;
            p->opt_host_block_rows = value;
            return CC_LADDER_OK;
        default: return CC_LADDER_EINVAL;
    }
}

int cc_ladder_get_option(cc_ladder_plan_t p, int key, long long *value)
{
    if (!p || !value) return CC_LADDER_EINVAL;
    switch (key) {
        case CC_LADDER_OPT_SPLIT: *value = p->opt_split; return CC_LADDER_OK;
        case CC_LADDER_OPT_ALGO: *value = p->opt_algo; return CC_LADDER_OK;
        case CC_LADDER_OPT_NUM_CTAS: *value = p->opt_num_ctas; return CC_LADDER_OK;
        case CC_LADDER_OPT_SUPERTILE: *value = p->opt_supertile; return CC_LADDER_OK;
        case CC_LADDER_OPT_TILE: *value = p->opt_tile; return CC_LADDER_OK;
        case CC_LADDER_OPT_EXCHANGE: *value = p->opt_exchange; return CC_LADDER_OK;
        case CC_LADDER_OPT_LAYOUT: *value = p->opt_layout; return CC_LADDER_OK;
        case CC_LADDER_OPT_XY_ROWS_X: *value = p->opt_nr; return CC_LADDER_OK;
        case CC_LADDER_OPT_XY_ROWS_Y: *value = p->opt_ns; return CC_LADDER_OK;
        case CC_LADDER_OPT_HOST_BUDGET: *value = p->opt_host_budget; return CC_LADDER_OK;
        case CC_LADDER_OPT_INDEX_BITS: *value = p->opt_index_bits; return CC_LADDER_OK;
        case CC_LADDER_OPT_SYMM_L: *value = p->opt_symm; return CC_LADDER_OK;
        case CC_LADDER_OPT_SCHEDULE: *value = p->opt_schedule; return CC_LADDER_OK;
        case CC_LADDER_OPT_HOST_BLOCK_ROWS: *value = p->opt_host_block_rows; return CC_LADDER_OK;
        default: return CC_LADDER_EINVAL;
    }
}

int cc_ladder_get_info(cc_ladder_plan_t p, int key, long long *value)
{
    if (!p || !value) return CC_LADDER_EINVAL;
    const int nr = rows_x(p), ns = rows_y(p);
    const TileGeom g = geom_of(p, nr, ns);
    FusedParams fp;
    fill_params(p, g, nr, ns, fp);
    const long long vv = (long long)p->v * p->v;
    switch (key) {
        case CC_LADDER_INFO_NUM_TILES:
            if (p->opt_algo == CC_LADDER_ALGO_SIMPLE)
                *value = (long long)((vv + (long long)simple_pairs_per_chunk(p) - 1) / (long long)simple_pairs_per_chunk(p));
            else if (symm_on(p))      // tiles with (A,B) <= (C,D): the others are skipped by every CTA
                *value = fp.n_ab_blk * (fp.n_ab_blk + 1) / 2;
            else
                *value = fp.n_tiles;
            return CC_LADDER_OK;
        case CC_LADDER_INFO_KERNEL_LAUNCHES:
            if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) {
                const long long n = (long long)simple_pairs_per_chunk(p);
                *value = 2 * ((vv + n - 1) / n);
            } else {
                *value = p->opt_split ? 3 : 1;   // split: pack, fused (CTA pairs), unpack
            }
            return CC_LADDER_OK;
        case CC_LADDER_INFO_FLOPS_EXECUTED: {
            if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) {
                *value = 2 * vv * vv * ((long long)p->x + (long long)p->o * p->o);
            } else {
                // per tile: GEMM-1 2*M1*N1*ceil4(x), GEMM-2 2*ceil8(o^2)*NAB*NCD  (M1*N1 == NAB*NCD)
                const long long nab = (long long)g.TA * g.TB, ncd = (long long)g.TC * g.TD;
                const long long xk = (long long)ceil_div(p->x, 4) * 4;
                const long long mr = ((fp.oo + 7) / 8) * 8;
                if (symm_on(p))     // GEMM-1 once per canonical tile, GEMM-2 twice off the diagonal
                    *value = fp.n_ab_blk * (fp.n_ab_blk + 1) / 2 * (2 * nab * ncd * xk) + fp.n_tiles * (2 * mr * nab * ncd);
                else
                    *value = fp.n_tiles * (2 * nab * ncd * xk + 2 * mr * nab * ncd) * (p->opt_split ? 2 : 1);
            }
            return CC_LADDER_OK;
        }
        case CC_LADDER_INFO_FLOPS_FULL:     // 2 nr ns v^2 (x + o^2); the ladder: nr = ns = v
            *value = 2 * (long long)nr * ns * vv * ((long long)p->x + (long long)p->o * p->o);
            return CC_LADDER_OK;
        case CC_LADDER_INFO_NUM_SMS: *value = p->num_sms; return CC_LADDER_OK;
        case CC_LADDER_INFO_SMEM_BYTES: *value = (p->opt_algo == CC_LADDER_ALGO_SIMPLE) ? 0 : g.smem; return CC_LADDER_OK;
        case CC_LADDER_INFO_TILE_SHAPE:
            *value = ((long long)g.TA << 24) | ((long long)g.TB << 16) | ((long long)g.TC << 8) | (long long)g.TD;
            return CC_LADDER_OK;
        case CC_LADDER_INFO_SUPERTILE_SHAPE:
            *value = ((long long)fp.SA << 24) | ((long long)fp.SB << 16) | ((long long)fp.SC << 8) | (long long)fp.SD;
            return CC_LADDER_OK;
        case CC_LADDER_INFO_INDEX_BITS: *value = fp.idx32 ? 32 : 64; return CC_LADDER_OK;
        case CC_LADDER_INFO_HOST_CHUNKS: *value = p->host_chunks; return CC_LADDER_OK;
        default: return CC_LADDER_EINVAL;
    }
}

size_t cc_ladder_workspace_bytes(cc_ladder_plan_t p)
{
    if (!p) return 0;
    if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) return simple_pairs_per_chunk(p) * (size_t)p->v * p->v * sizeof(double);
    if (p->opt_split) {     // packed triangles T+, T- (nt doubles per (i,j)) and W+, W- (nt + 8): ~2 v^2 doubles per (i,j)
        const size_t nt = (size_t)tri_size(p->v);
        return (size_t)p->o * p->o * (4 * nt + 16) * sizeof(double);
    }
    return 0;
}

int cc_ladder_set_workspace(cc_ladder_plan_t p, void *dev_ptr, size_t bytes)
{
    if (!p) return CC_LADDER_EINVAL;
    if (dev_ptr && ((uintptr_t)dev_ptr & 255u)) return CC_LADDER_EINVAL;
    p->ws = dev_ptr;
    p->ws_bytes = dev_ptr ? bytes : 0;
    return CC_LADDER_OK;
}

int cc_ladder(cc_ladder_plan_t p, const double *L, const double *t, double *R, void *stream)
{
    if (!p || !L || !t || !R) return CC_LADDER_EINVAL;
    if (((uintptr_t)L | (uintptr_t)t | (uintptr_t)R) & 15u) return CC_LADDER_EINVAL;
    const size_t vv = (size_t)p->v * p->v;
    const size_t nL = (size_t)p->x * vv * sizeof(double);
    const size_t nT = (size_t)p->o * p->o * vv * sizeof(double);
    if (overlaps(R, nT, L, nL) || overlaps(R, nT, t, nT)) return CC_LADDER_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    // the simple path is a cross-check of the plain ladder only; split combines with exchange and the paper's storage
    // through its pack / unpack kernels (the fused kernel works on the packed workspace either way)
    if (p->opt_algo == CC_LADDER_ALGO_SIMPLE && (p->opt_split || p->opt_exchange || p->opt_layout)) return CC_LADDER_EINVAL;
    if (p->opt_symm && (p->opt_split || p->opt_exchange || p->opt_layout || p->opt_algo == CC_LADDER_ALGO_SIMPLE))
        return CC_LADDER_EINVAL;
    if (!offsets_fit(p, p->v, p->v)) return CC_LADDER_EINVAL;
    int rc = check_device(p);
    if (rc != CC_LADDER_OK) return rc;
    const size_t need = cc_ladder_workspace_bytes(p);
    if (need) {
        if (!p->ws || p->ws_bytes < need) return CC_LADDER_EWORKSPACE;
        if (overlaps(p->ws, need, L, nL) || overlaps(p->ws, need, t, nT) || overlaps(p->ws, need, R, nT))
            return CC_LADDER_EINVAL;
    }

    if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) {
        const long long npc = (long long)simple_pairs_per_chunk(p);
        double *Vc = (double *)p->ws;
        const long long oo = (long long)p->o * p->o;
        for (long long pair0 = 0; pair0 < (long long)vv; pair0 += npc) {
            const int np = (int)(((long long)vv - pair0) < npc ? ((long long)vv - pair0) : npc);
            simple_eri_chunk<<<p->num_sms * 8, 256, 0, s>>>(L, Vc, p->v, p->x, pair0, np);
            simple_contract_chunk<<<p->num_sms * 8, 256, 0, s>>>(t, Vc, R, oo, p->v, pair0, np);
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(p, e, "simple path launch");
        return CC_LADDER_OK;
    }

    if (p->opt_split) {
        // a0 pack (+ zero W+-) -> fused kernel on CTA pairs -> a5 unpack; workspace = packed triangles
        // [T+ : o^2 nt | T- : o^2 nt | W+ : o^2 (nt + 8) | W- : o^2 (nt + 8)], nt = tri_size(v) (a multiple of 4)
        const TileGeom g = geom_of(p, p->v, p->v);
        FusedParams fp;
        fill_params(p, g, p->v, p->v, fp);
        const long long oo = (long long)p->o * p->o;
        double *Tp = (double *)p->ws, *Tm = Tp + (size_t)oo * fp.tri_nt, *Wp = Tm + (size_t)oo * fp.tri_nt,
               *Wm = Wp + (size_t)oo * (fp.tri_nt + 8);
        const int nt = ceil_div(p->v, kTT);
        const dim3 tgrid((unsigned)nt, (unsigned)nt, (unsigned)(oo < 32768 ? oo : 32768));
        const int iajb = p->opt_layout == CC_LADDER_LAYOUT_IAJB ? 1 : 0;
        split_pack_kernel<<<tgrid, 256, 0, s>>>(t, Tp, Tm, Wp, Wm, oo, p->v, p->o, iajb);
        fp.X = fp.Y = L;
        fp.xps = fp.yps = (long long)vv;
        fp.xrs = fp.yrs = p->v;
        fp.t = Tp;
        fp.tm = Tm;
        fp.R = Wp;
        fp.Rm = Wm;
        long long pairs = (p->opt_num_ctas > 0 ? p->opt_num_ctas : p->num_sms) / 2;
        if (pairs < 1) pairs = 1;
        if (pairs > fp.n_tiles) pairs = fp.n_tiles;
        rc = (g.id == 6) ? launch_fused<CfgSplit12, true>(p, fp, (int)(2 * pairs), s)
                         : launch_fused<CfgSplit, true>(p, fp, (int)(2 * pairs), s);
        if (rc != CC_LADDER_OK) return rc;
        // exchange (Eq. 7) = the ladder of t with c and d swapped: same T+, negated T-, hence W+ -+ W-
        split_unpack_kernel<<<tgrid, 256, 0, s>>>(Wp, Wm, R, oo, p->v, p->o, iajb, p->opt_exchange ? -1.0 : 1.0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(p, e, "split pack/unpack launch");
        return CC_LADDER_OK;
    }
    const Operands op = {L, L, (long long)vv, (long long)p->v, (long long)vv, (long long)p->v, p->v, p->v, t, R, 0};
    return run_fused(p, op, s);
}

int cc_ladder_xy(cc_ladder_plan_t p, const double *X, long long x_pstride, long long x_rstride, int nr, const double *Y,
                 long long y_pstride, long long y_rstride, int ns, const double *t, double *out, void *stream)
{
    if (!p || !X || !Y || !t || !out) return CC_LADDER_EINVAL;
    if (nr <= 0 || ns <= 0 || nr > 30000 || ns > 30000) return CC_LADDER_EINVAL;
    if (x_rstride < p->v || y_rstride < p->v) return CC_LADDER_EINVAL;
    if (x_pstride < (long long)(nr - 1) * x_rstride + p->v || y_pstride < (long long)(ns - 1) * y_rstride + p->v)
        return CC_LADDER_EINVAL;
    if (x_rstride > (1LL << 31) / nr || y_rstride > (1LL << 31) / ns) return CC_LADDER_EINVAL;   // 32-bit row offsets
    if (((uintptr_t)X | (uintptr_t)Y) & 7u) return CC_LADDER_EINVAL;
    if (((uintptr_t)t | (uintptr_t)out) & 15u) return CC_LADDER_EINVAL;
    if (p->opt_split || p->opt_symm || p->opt_algo == CC_LADDER_ALGO_SIMPLE) return CC_LADDER_EINVAL;   // full mode only
    if (!offsets_fit(p, nr, ns)) return CC_LADDER_EINVAL;
    const size_t nX = span_bytes(p->x, x_pstride, nr, x_rstride, p->v), nY = span_bytes(p->x, y_pstride, ns, y_rstride, p->v);
    const size_t nT = (size_t)p->o * p->o * (size_t)p->v * p->v * sizeof(double);
    const size_t nO = (size_t)p->o * p->o * (size_t)nr * ns * sizeof(double);
    if (overlaps(out, nO, X, nX) || overlaps(out, nO, Y, nY) || overlaps(out, nO, t, nT)) return CC_LADDER_EINVAL;
    int rc = check_device(p);
    if (rc != CC_LADDER_OK) return rc;
    p->opt_nr = nr;
    p->opt_ns = ns;
    const Operands op = {X, Y, x_pstride, x_rstride, y_pstride, y_rstride, nr, ns, t, out, 0};
    return run_fused(p, op, (cudaStream_t)stream);
}

namespace {

bool is_pinned(const void *ptr)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeHost;
}

// Host-resident streaming (the paper's batch loop over chunks of `a`, here with L and t resident and
// the copies overlapped with the kernels).  R is cut into column blocks a in [a0, a0 + na): block k lives in device
// buffer k % 2 as a dense out[i][j][r][s] (or out[i][r][j][s]) array with nr = na rows, i.e. exactly what
// cc_ladder_xy writes for X = L[:, a0:a0+na, :], Y = L.  Two streams alternate: H2D of block k+1 and D2H of block k-1
// run while block k computes.  Pageable host memory goes through two pinned staging buffers per direction.
int host_streamed(cc_ladder_plan_t p, const double *L_host, const double *t_host, double *R_host, size_t budget,
                  long long na_req = 0)
{
    const int o = p->o, v = p->v;
    const size_t vv = (size_t)v * v, oo = (size_t)o * o;
    const size_t nL = (size_t)p->x * vv * sizeof(double), nT = oo * vv * sizeof(double);
    if (p->opt_split || p->opt_symm || p->opt_algo == CC_LADDER_ALGO_SIMPLE) return CC_LADDER_ENOMEM;   // resident-only modes
    if (budget <= nL + nT) return CC_LADDER_ENOMEM;
    // rows of `a` per block: a multiple of 24 (every compiled block edge TA divides it), as many as fit twice
    const size_t per_a = oo * (size_t)v * sizeof(double);
    long long na = (long long)((budget - nL - nT) / 2 / per_a);
    if (na_req > 0 && na_req < na) na = na_req;       // the caller's block size (overlap of copies and kernels), if it fits
    if (na >= v) na = v;
    else na = (na / 24) * 24;
    if (na < 1) return CC_LADDER_ENOMEM;
    const int nblk = ceil_div(v, (int)na);
    const size_t nC = (size_t)na * per_a;
    const bool iajb = p->opt_layout == CC_LADDER_LAYOUT_IAJB;
    // one 2-D copy per block: IJAB rows = (i,j), width na*v; IAJB rows = i, width na*o*v
    const size_t rows = iajb ? (size_t)o : oo;
    const size_t host_pitch = (iajb ? (size_t)v * o * v : vv) * sizeof(double);
    auto width_of = [&](int nab) { return (iajb ? (size_t)nab * o * v : (size_t)nab * v) * sizeof(double); };
    auto host_off = [&](int a0) { return (iajb ? (size_t)a0 * o * v : (size_t)a0 * v); };

    double *dL = nullptr, *dT = nullptr, *dC[2] = {nullptr, nullptr}, *stage_in[2] = {nullptr, nullptr},
           *stage_out[2] = {nullptr, nullptr};
    cudaStream_t st[2] = {nullptr, nullptr};
    cudaEvent_t in_free[2] = {nullptr, nullptr}, out_done[2] = {nullptr, nullptr}, lt_ready = nullptr;
    const bool pinned = is_pinned(R_host);
    const long long saved_nr = p->opt_nr, saved_ns = p->opt_ns;
    int rc = CC_LADDER_OK;
    cudaError_t e = cudaSuccess;
    auto ck = [&](cudaError_t err, const char *where) {
        if (err != cudaSuccess && rc == CC_LADDER_OK)
            rc = (err == cudaErrorMemoryAllocation) ? CC_LADDER_ENOMEM : fail_cuda(p, err, where);
        return err == cudaSuccess;
    };
    // scatter a finished block from its pinned staging buffer into R_host (pageable path)
    auto drain = [&](int k) {
        const int a0 = k * (int)na, nab = (v - a0) < (int)na ? (v - a0) : (int)na;
        if (!ck(cudaEventSynchronize(out_done[k & 1]), "cudaEventSynchronize")) return;
        const size_t w = width_of(nab);
        for (size_t r = 0; r < rows; ++r)
            memcpy((char *)(R_host + host_off(a0)) + r * host_pitch, (const char *)stage_out[k & 1] + r * w, w);
    };

    for (int k = 0; k < 2 && rc == CC_LADDER_OK; ++k) {
        ck(cudaStreamCreateWithFlags(&st[k], cudaStreamNonBlocking), "cudaStreamCreate");
        ck(cudaEventCreateWithFlags(&in_free[k], cudaEventDisableTiming), "cudaEventCreate");
        ck(cudaEventCreateWithFlags(&out_done[k], cudaEventDisableTiming), "cudaEventCreate");
        ck(cudaMalloc(&dC[k], nC), "cudaMalloc");
        if (!pinned) {
            ck(cudaMallocHost(&stage_in[k], nC), "cudaMallocHost");
            ck(cudaMallocHost(&stage_out[k], nC), "cudaMallocHost");
        }
    }
    if (rc == CC_LADDER_OK) ck(cudaEventCreateWithFlags(&lt_ready, cudaEventDisableTiming), "cudaEventCreate");
    if (rc == CC_LADDER_OK) ck(cudaMalloc(&dL, nL), "cudaMalloc");
    if (rc == CC_LADDER_OK) ck(cudaMalloc(&dT, nT), "cudaMalloc");
    if (rc != CC_LADDER_OK) goto done;
    if (!ck(cudaMemcpyAsync(dL, L_host, nL, cudaMemcpyHostToDevice, st[0]), "cudaMemcpy H2D") ||
        !ck(cudaMemcpyAsync(dT, t_host, nT, cudaMemcpyHostToDevice, st[0]), "cudaMemcpy H2D") ||
        !ck(cudaEventRecord(lt_ready, st[0]), "cudaEventRecord") ||
        !ck(cudaStreamWaitEvent(st[1], lt_ready, 0), "cudaStreamWaitEvent"))
        goto done;

    for (int k = 0; k < nblk && rc == CC_LADDER_OK; ++k) {
        const int b = k & 1;
        const int a0 = k * (int)na, nab = (v - a0) < (int)na ? (v - a0) : (int)na;
        const size_t w = width_of(nab);
        if (pinned) {
            e = cudaMemcpy2DAsync(dC[b], w, R_host + host_off(a0), host_pitch, w, rows, cudaMemcpyHostToDevice, st[b]);
        } else {
            if (k >= 2 && !ck(cudaEventSynchronize(in_free[b]), "cudaEventSynchronize")) break;   // staging buffer reusable
            for (size_t r = 0; r < rows; ++r)
                memcpy((char *)stage_in[b] + r * w, (const char *)(R_host + host_off(a0)) + r * host_pitch, w);
            e = cudaMemcpyAsync(dC[b], stage_in[b], rows * w, cudaMemcpyHostToDevice, st[b]);
            if (e == cudaSuccess) e = cudaEventRecord(in_free[b], st[b]);
        }
        if (!ck(e, "cudaMemcpy H2D (R block)")) break;
        {   // out[i,j,r,s] += sum_cd (sum_P L[P,a0+r,c] L[P,s,d]) t[i,j,c,d]  on the block's stream
            const Operands op = {dL + (size_t)a0 * v, dL, (long long)vv, (long long)v, (long long)vv, (long long)v,
                                 nab, v, dT, dC[b], b};
            if (!offsets_fit(p, nab, v)) { rc = CC_LADDER_EINVAL; break; }
            rc = run_fused(p, op, st[b]);
            if (rc != CC_LADDER_OK) break;
        }
        if (pinned) {
            e = cudaMemcpy2DAsync(R_host + host_off(a0), host_pitch, dC[b], w, w, rows, cudaMemcpyDeviceToHost, st[b]);
        } else {
            e = cudaMemcpyAsync(stage_out[b], dC[b], rows * w, cudaMemcpyDeviceToHost, st[b]);
            if (e == cudaSuccess) e = cudaEventRecord(out_done[b], st[b]);
        }
        if (!ck(e, "cudaMemcpy D2H (R block)")) break;
        if (!pinned && k >= 1) drain(k - 1);          // overlaps the kernel of block k
    }
    if (rc == CC_LADDER_OK && !pinned) drain(nblk - 1);
    for (int k = 0; k < 2; ++k)
        if (st[k]) ck(cudaStreamSynchronize(st[k]), "cudaStreamSynchronize");
    if (rc == CC_LADDER_OK) p->host_chunks = nblk;
done:
    for (int k = 0; k < 2; ++k) {
        if (st[k]) { (void)cudaStreamSynchronize(st[k]); (void)cudaStreamDestroy(st[k]); }
        if (in_free[k]) cudaEventDestroy(in_free[k]);
        if (out_done[k]) cudaEventDestroy(out_done[k]);
        if (dC[k]) cudaFree(dC[k]);
        if (stage_in[k]) cudaFreeHost(stage_in[k]);
        if (stage_out[k]) cudaFreeHost(stage_out[k]);
    }
    if (lt_ready) cudaEventDestroy(lt_ready);
    if (dL) cudaFree(dL);
    if (dT) cudaFree(dT);
    p->opt_nr = saved_nr;
    p->opt_ns = saved_ns;
    (void)cudaGetLastError();
    return rc;
}

}  // namespace

int cc_ladder_host(cc_ladder_plan_t p, const double *L_host, const double *t_host, double *R_host)
{
    if (!p || !L_host || !t_host || !R_host) return CC_LADDER_EINVAL;
    const size_t vv = (size_t)p->v * p->v;
    const size_t nL = (size_t)p->x * vv * sizeof(double);
    const size_t nT = (size_t)p->o * p->o * vv * sizeof(double);
    if (overlaps(R_host, nT, L_host, nL) || overlaps(R_host, nT, t_host, nT)) return CC_LADDER_EINVAL;
    int rc = check_device(p);
    if (rc != CC_LADDER_OK) return rc;
    const size_t need = cc_ladder_workspace_bytes(p);
    // device bytes this call may use: the option, else what the device reports as free (minus a margin)
    size_t budget = (size_t)p->opt_host_budget;
    if (budget == 0) {
        size_t fr = 0, tot = 0;
        if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { (void)cudaGetLastError(); return CC_LADDER_ECUDA; }
        budget = fr - fr / 32;
    }
    if (nL + 2 * nT + need > budget) return host_streamed(p, L_host, t_host, R_host, budget, p->opt_host_block_rows);
    // Everything fits.  With pinned host memory R is still streamed in column blocks (full mode only): the H2D / D2H
    // copies of R then overlap the kernels, and only the upload of L and t and one block's copies stay exposed
    // (configs[2]: 1384 -> 1331 ms end to end; the kernel alone takes 1303 ms).  CC_LADDER_OPT_HOST_BLOCK_ROWS: 0 = auto
    // (about six blocks, a multiple of 24 rows of a; problems under 256 MB of R stay resident), -1 = off, n = rows.
    if (p->opt_host_block_rows >= 0 && !p->opt_split && !p->opt_symm &&
        p->opt_algo == CC_LADDER_ALGO_FUSED && is_pinned(R_host)) {
        long long na = p->opt_host_block_rows;
        if (na == 0 && nT >= (size_t(256) << 20)) na = (ceil_div(ceil_div(p->v, 6), 24)) * 24;
        if (na > 0 && na < p->v) return host_streamed(p, L_host, t_host, R_host, budget, ((na + 23) / 24) * 24);
    }

    double *dL = nullptr, *dT = nullptr, *dR = nullptr;
    void *dW = nullptr;
    void *saved_ws = p->ws;
    size_t saved_ws_bytes = p->ws_bytes;
    cudaError_t e;
    cudaStream_t s = nullptr;
    if ((e = cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking)) != cudaSuccess) return fail_cuda(p, e, "cudaStreamCreate");
    if ((e = cudaMalloc(&dL, nL)) != cudaSuccess || (e = cudaMalloc(&dT, nT)) != cudaSuccess ||
        (e = cudaMalloc(&dR, nT)) != cudaSuccess || (need && (e = cudaMalloc(&dW, need)) != cudaSuccess)) {
        rc = (e == cudaErrorMemoryAllocation) ? CC_LADDER_ENOMEM : fail_cuda(p, e, "cudaMalloc");
        (void)cudaGetLastError();
        goto done;
    }
    if (need) { p->ws = dW; p->ws_bytes = need; }
    if ((e = cudaMemcpyAsync(dL, L_host, nL, cudaMemcpyHostToDevice, s)) != cudaSuccess ||
        (e = cudaMemcpyAsync(dT, t_host, nT, cudaMemcpyHostToDevice, s)) != cudaSuccess ||
        (e = cudaMemcpyAsync(dR, R_host, nT, cudaMemcpyHostToDevice, s)) != cudaSuccess) {
        rc = fail_cuda(p, e, "cudaMemcpy H2D");
        goto done;
    }
    rc = cc_ladder(p, dL, dT, dR, s);
    if (rc != CC_LADDER_OK) goto done;
    if ((e = cudaMemcpyAsync(R_host, dR, nT, cudaMemcpyDeviceToHost, s)) != cudaSuccess ||
        (e = cudaStreamSynchronize(s)) != cudaSuccess) {
        rc = fail_cuda(p, e, "cudaMemcpy D2H");
        goto done;
    }
    p->host_chunks = 1;
done:
    if (s) { (void)cudaStreamSynchronize(s); (void)cudaStreamDestroy(s); }
    p->ws = saved_ws;
    p->ws_bytes = saved_ws_bytes;
    if (dL) cudaFree(dL);
    if (dT) cudaFree(dT);
    if (dR) cudaFree(dR);
    if (dW) cudaFree(dW);
    return rc;
}

int cc_ladder_check_symmetric(cc_ladder_plan_t p, const double *L, long long *n_mismatch, void *stream)
{
    if (!p || !L || !n_mismatch) return CC_LADDER_EINVAL;
    int rc = check_device(p);
    if (rc != CC_LADDER_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned long long *cnt = nullptr, h = 0;
    cudaError_t e = cudaMalloc(&cnt, sizeof(*cnt));
    if (e != cudaSuccess) return fail_cuda(p, e, "cudaMalloc");
    if ((e = cudaMemsetAsync(cnt, 0, sizeof(*cnt), s)) == cudaSuccess) {
        const int nt = ceil_div(p->v, kTT);
        const dim3 grid((unsigned)nt, (unsigned)nt, (unsigned)(p->x < 32768 ? p->x : 32768));
        symm_check_kernel<<<grid, 256, 0, s>>>(L, p->x, p->v, cnt);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, cnt, sizeof(h), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(cnt);
    if (e != cudaSuccess) return fail_cuda(p, e, "cc_ladder_check_symmetric");
    *n_mismatch = (long long)h;
    return CC_LADDER_OK;
}

int cc_ladder_fp64_peak(double *tflops, double *flop_per_clk_per_sm, void *stream)
{
    if (!tflops && !flop_per_clk_per_sm) return CC_LADDER_EINVAL;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return CC_LADDER_ECUDA;
    }
    if (prop.major != 10) return CC_LADDER_EARCH;
    cudaStream_t s = (cudaStream_t)stream;
    const int nsm = prop.multiProcessorCount, iters = 200000;      // 8 warps x 8 DMMA x 200000 per SM: ~0.2 s
    double *sink = nullptr;
    long long *cyc = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = CC_LADDER_ECUDA;
    float ms = 0.f;
    long long *hc = (long long *)malloc(sizeof(long long) * (size_t)nsm);
    if (!hc) return CC_LADDER_ENOMEM;
    if (cudaMalloc(&sink, 8) != cudaSuccess || cudaMalloc(&cyc, sizeof(long long) * (size_t)nsm) != cudaSuccess) goto out;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) goto out;
    fp64_peak_kernel<<<nsm, 256, 0, s>>>(sink, 2000, cyc);      // warm-up
    if (cudaEventRecord(e0, s) != cudaSuccess) goto out;
    fp64_peak_kernel<<<nsm, 256, 0, s>>>(sink, iters, cyc);
    if (cudaEventRecord(e1, s) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) goto out;
    if (cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) goto out;
    if (cudaMemcpy(hc, cyc, sizeof(long long) * (size_t)nsm, cudaMemcpyDeviceToHost) != cudaSuccess) goto out;
    {
        const double flop_sm = 512.0 * 8.0 * 8.0 * (double)iters;      // one DMMA.8x8x4 = 8*8*4*2 flop
        long long cmax = 1;
        for (int i = 0; i < nsm; ++i) cmax = hc[i] > cmax ? hc[i] : cmax;
        if (tflops) *tflops = flop_sm * nsm / ((double)ms * 1e-3) / 1e12;
        if (flop_per_clk_per_sm) *flop_per_clk_per_sm = flop_sm / (double)cmax;
        rc = CC_LADDER_OK;
    }
out:
    (void)cudaGetLastError();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (sink) cudaFree(sink);
    if (cyc) cudaFree(cyc);
    free(hc);
    return rc;
}

int cc_ladder_destroy(cc_ladder_plan_t p)
{
    if (p && p->counters) (void)cudaFree(p->counters);
    delete p;
    return CC_LADDER_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// cc_ladder_split_static: the allocation-free entry point (include/cc_ladder.h).  The split-mode workspace (packed
// triangles T+, T-, W+, W-) is this file-scope array instead of caller memory; split_pack_kernel, the fused kernel on CTA
// pairs and split_unpack_kernel get its DEVICE address, which host code has to ask the runtime for: the name
// `g_static_scratch` in host code is a host-side stand-in, not a device pointer.
static __device__ __align__(256) unsigned char g_static_scratch[CC_LADDER_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;

struct StaticDevice {       // set-up of one device, done once with that device current
    bool ready;
    void *scratch;          // device address of g_static_scratch on this device
    int num_sms, cc_major;
};

StaticDevice g_static_dev[kMaxDevices];
std::mutex g_static_mutex;
char g_static_err[256];

int static_fail(cudaError_t e, const char *where)
{
    snprintf(g_static_err, sizeof(g_static_err), "%s: %s", where, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return CC_LADDER_ECUDA;
}

// the current device's entry of g_static_dev, set up on first use (no allocation: attribute queries and the symbol look-up)
int static_device(int *dev_out, StaticDevice *out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return CC_LADDER_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice &d = g_static_dev[dev];
    if (!d.ready) {
        if ((e = cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess)
            return static_fail(e, "cudaDeviceGetAttribute(compute capability)");
        if (d.cc_major != 10) return CC_LADDER_EARCH;
        if ((e = cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
            return static_fail(e, "cudaDeviceGetAttribute(SM count)");
        void *ptr = nullptr;
        if ((e = cudaGetSymbolAddress(&ptr, g_static_scratch)) != cudaSuccess)
            return static_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!ptr || ((uintptr_t)ptr & 255u)) {
            snprintf(g_static_err, sizeof(g_static_err), "cudaGetSymbolAddress returned an unusable address %p", ptr);
            return CC_LADDER_ECUDA;
        }
        d.scratch = ptr;
        d.ready = true;
    }
    *dev_out = dev;
    *out = d;
    return CC_LADDER_OK;
}

}  // namespace

extern "C" {

size_t cc_ladder_static_scratch_bytes(void) { return sizeof(g_static_scratch); }

size_t cc_ladder_split_static_bytes(int nocc, int nvirt)
{
    if (nocc <= 0 || nvirt <= 0) return 0;
    return (size_t)nocc * nocc * (4 * (size_t)tri_size(nvirt) + 16) * sizeof(double);
}

const char *cc_ladder_split_static_error(void) { return g_static_err; }

int cc_ladder_split_static(int nocc, int nvirt, int nchol, const double *L, const double *t, double *R, void *stream)
{
    if (nocc <= 0 || nvirt <= 0 || nchol <= 0 || nvirt > 30000 || nocc > 30000) return CC_LADDER_EINVAL;
    if (!L || !t || !R) return CC_LADDER_EINVAL;
    if (cc_ladder_split_static_bytes(nocc, nvirt) > sizeof(g_static_scratch)) return CC_LADDER_ESCRATCH;
    int dev = -1;
    StaticDevice d;
    int rc = static_device(&dev, &d);
    if (rc != CC_LADDER_OK) return rc;
    // a plan on the stack (nothing to allocate in split mode: no tile counter), default options, workspace = the array
    cc_ladder_plan_s plan;
    memset(&plan, 0, sizeof(plan));
    plan.o = nocc;
    plan.v = nvirt;
    plan.x = nchol;
    plan.device = dev;
    plan.num_sms = d.num_sms;
    plan.opt_algo = CC_LADDER_ALGO_FUSED;
    plan.opt_split = 1;
    plan.ws = d.scratch;
    plan.ws_bytes = sizeof(g_static_scratch);
    rc = cc_ladder(&plan, L, t, R, stream);
    if (rc == CC_LADDER_ECUDA) snprintf(g_static_err, sizeof(g_static_err), "%s", plan.cuda_err);
    return rc;
}

}  // extern "C"
