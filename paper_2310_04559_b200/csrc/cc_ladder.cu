// C ABI of the B200-native Cholesky vvvv ladder (include/cc_ladder.h): plan / options / scheduler set-up / launches.
// Host logic only; the arithmetic lives in ladder_fused.cuh (default) and ladder_simple.cuh (on-GPU cross-check).
#include "../../include/cc_ladder.h"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "ladder_ws.cuh"
#include "ladder_simple.cuh"
#include "ladder_split.cuh"

using namespace ccl;

namespace {

// tile shapes <TA,TB,TC,TD,KS>: block edges along a, b, c, d and the (c,d) pairs per staged t slab
using CfgP2 = WsCfg<8, 12, 16, 8, 32>;        //  96 (ab) x 128 (cd): generic nvirt
using CfgP12 = WsCfg<12, 8, 12, 12, 24>;      //  96 (ab) x 144 (cd): nvirt = 300, 420, 120 (12 | nvirt, b padded to 8)
using CfgP20 = WsCfg<8, 12, 20, 8, 32>;       //  96 (ab) x 160 (cd): nvirt = 520 (b padded to 12)
using CfgSplit = WsCfg<8, 8, 16, 16, 32>;     // split mode: square partitions, 64 (a<=b block pair) x 256 (c<=d)

constexpr size_t kSimpleChunkBytes = size_t(256) << 20;

}  // namespace

struct cc_ladder_plan_s {
    int o, v, x;
    int device, num_sms;
    long long l2_bytes;
    long long opt_split, opt_algo, opt_num_ctas, opt_supertile, opt_tile, opt_exchange, opt_layout;
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

// padded tile-space volume of a shape: prod_dim ceil(v / T) * T
double padded_volume(int v, const TileGeom &g)
{
    auto pad = [v](int T) { return (double)ceil_div(v, T) * T; };
    return pad(g.TA) * pad(g.TB) * pad(g.TC) * pad(g.TD);
}

// Bytes the ~148 tiles in flight touch with the default 3 x 4 x 3 x 4 super-tile: 9 X slabs, 16 Y slabs of L,
// 12 blocks of R and 12 blocks of t.
double supertile_footprint(const cc_ladder_plan_s *p, const TileGeom &g)
{
    const double oo = (double)p->o * p->o, x = (double)p->x;
    return 8.0 * (9.0 * x * g.TA * g.TC + 16.0 * x * g.TB * g.TD + 12.0 * oo * g.TA * g.TB + 12.0 * oo * g.TC * g.TD);
}

// step a1, plan time: the tile shape.  Auto picks the compiled shape with the least estimated time = padded volume
// (each dimension of the (a,b,c,d) space is padded to a multiple of its block edge) / relative efficiency measured on
// the B200 (profiles/): <12,8,12,12> runs ~3 % slower per flop than the other two, and a shape whose super-tile
// footprint overflows L2 pays ~3 % (DRAM traffic pushes the chip into its 1 kW power cap).  The generic shape wins ties.
TileGeom geom_of(const cc_ladder_plan_s *p)
{
    if (p->opt_split) return geom<CfgSplit>(0);
    if (p->opt_exchange) return geom<CfgSplit>(4);      // the a <-> b swap needs square block partitions
    const TileGeom cand[3] = {geom<CfgP2>(1), geom<CfgP12>(2), geom<CfgP20>(3)};
    if (p->opt_tile >= 1 && p->opt_tile <= 3) return cand[p->opt_tile - 1];
    const double base_eff[3] = {1.0, 0.97, 1.0};
    double cost[3];
    for (int k = 0; k < 3; ++k) {
        const double eff = base_eff[k] * (supertile_footprint(p, cand[k]) > (double)p->l2_bytes ? 0.97 : 1.0);
        cost[k] = padded_volume(p->v, cand[k]) / eff;
    }
    int best = 0;
    for (int k = 1; k < 3; ++k)
        if (cost[k] < 0.998 * cost[best]) best = k;
    return cand[best];
}

void fill_params(const cc_ladder_plan_s *p, const TileGeom &g, FusedParams &fp)
{
    fp.o = p->o;
    fp.v = p->v;
    fp.x = p->x;
    fp.oo = (long long)p->o * p->o;
    fp.nA = ceil_div(p->v, g.TA);
    fp.nB = ceil_div(p->v, g.TB);
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
    fp.exchange = p->opt_exchange ? 1 : 0;
    fp.ovv = (long long)p->v * p->o * p->v;
    // L2 super-tile: S (ab)-blocks x S (cd)-blocks in flight, each an SA x SB (SC x SD) rectangle of blocks
    const int S = p->opt_supertile > 0 ? (int)p->opt_supertile : 12;
    fp.supertile = S;
    int sa = 1;
    while ((sa + 1) * (sa + 1) <= S) ++sa;
    fp.SA = fp.SC = sa;
    fp.SB = fp.SD = ceil_div(S, sa);
    // the device decodes tile indices in 32-bit arithmetic when its largest intermediate products fit
    const double big = (double)fp.n_tiles * (double)(p->opt_split ? (long long)S * S : (long long)fp.SB * fp.SB);
    fp.idx32 = big < 2.0e9 ? 1 : 0;
}

size_t simple_pairs_per_chunk(const cc_ladder_plan_s *p)
{
    const size_t vv = (size_t)p->v * p->v;
    size_t n = kSimpleChunkBytes / (vv * sizeof(double));
    if (n < 1) n = 1;
    if (n > vv) n = vv;
    return n;
}

template <class C, bool ALIGN2, bool SPLIT, bool IAJB>
int launch_fused_one(cc_ladder_plan_t p, const FusedParams &fp, int grid, cudaStream_t s)
{
    auto kern = ladder_ws_kernel<C, ALIGN2, SPLIT, IAJB>;
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
    e = cudaLaunchKernelEx(&cfg, kern, fp);
    if (e != cudaSuccess) return fail_cuda(p, e, "ladder_ws_kernel launch");
    return CC_LADDER_OK;
}

template <class C, bool SPLIT>
int launch_fused(cc_ladder_plan_t p, const FusedParams &fp, int grid, cudaStream_t s)
{
    if (!SPLIT && p->opt_layout == CC_LADDER_LAYOUT_IAJB) {
        if (p->v % 2 == 0) return launch_fused_one<C, true, false, true>(p, fp, grid, s);
        return launch_fused_one<C, false, false, true>(p, fp, grid, s);
    }
    if (p->v % 2 == 0) return launch_fused_one<C, true, SPLIT, false>(p, fp, grid, s);
    return launch_fused_one<C, false, SPLIT, false>(p, fp, grid, s);
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = (const char *)a, *pb = (const char *)b;
    return pa < pb + nb && pb < pa + na;
}

}  // namespace

extern "C" {

int cc_ladder_version(void) { return 100; }

const char *cc_ladder_status_string(int status)
{
    switch (status) {
        case CC_LADDER_OK: return "ok";
        case CC_LADDER_EINVAL: return "invalid argument (size <= 0, null/misaligned/overlapping pointer, bad option)";
        case CC_LADDER_EARCH: return "current device is not a compute-capability 10.x (sm_100) GPU";
        case CC_LADDER_EWORKSPACE: return "workspace missing or too small";
        case CC_LADDER_ECUDA: return "CUDA runtime error (see cc_ladder_last_cuda_error)";
        case CC_LADDER_ENOMEM: return "out of memory";
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
    p->o = nocc;
    p->v = nvirt;
    p->x = nchol;
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;
    p->l2_bytes = prop.l2CacheSize;
    p->opt_split = 0;
    p->opt_algo = CC_LADDER_ALGO_FUSED;
    p->opt_num_ctas = 0;
    p->opt_supertile = 0;
    p->opt_tile = 0;
    p->opt_exchange = 0;
    p->opt_layout = 0;
    p->ws = nullptr;
    p->ws_bytes = 0;
    p->cuda_err[0] = 0;
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
            if (value < 0 || value > 3) return CC_LADDER_EINVAL;
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
        default: return CC_LADDER_EINVAL;
    }
}

int cc_ladder_get_info(cc_ladder_plan_t p, int key, long long *value)
{
    if (!p || !value) return CC_LADDER_EINVAL;
    const TileGeom g = geom_of(p);
    FusedParams fp;
    fill_params(p, g, fp);
    const long long vv = (long long)p->v * p->v;
    switch (key) {
        case CC_LADDER_INFO_NUM_TILES:
            *value = (p->opt_algo == CC_LADDER_ALGO_SIMPLE)
                         ? (long long)((vv + (long long)simple_pairs_per_chunk(p) - 1) / (long long)simple_pairs_per_chunk(p))
                         : fp.n_tiles;
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
                *value = fp.n_tiles * (2 * nab * ncd * xk + 2 * mr * nab * ncd) * (p->opt_split ? 2 : 1);
            }
            return CC_LADDER_OK;
        }
        case CC_LADDER_INFO_FLOPS_FULL:
            *value = 2 * vv * vv * ((long long)p->x + (long long)p->o * p->o);
            return CC_LADDER_OK;
        case CC_LADDER_INFO_NUM_SMS: *value = p->num_sms; return CC_LADDER_OK;
        case CC_LADDER_INFO_SMEM_BYTES: *value = (p->opt_algo == CC_LADDER_ALGO_SIMPLE) ? 0 : g.smem; return CC_LADDER_OK;
        case CC_LADDER_INFO_TILE_SHAPE:
            *value = ((long long)g.TA << 24) | ((long long)g.TB << 16) | ((long long)g.TC << 8) | (long long)g.TD;
            return CC_LADDER_OK;
        default: return CC_LADDER_EINVAL;
    }
}

size_t cc_ladder_workspace_bytes(cc_ladder_plan_t p)
{
    if (!p) return 0;
    if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) return simple_pairs_per_chunk(p) * (size_t)p->v * p->v * sizeof(double);
    if (p->opt_split) return 4 * (size_t)p->o * p->o * (size_t)p->v * p->v * sizeof(double);   // T+, T-, W+, W-
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
    if (p->opt_split && p->opt_algo == CC_LADDER_ALGO_SIMPLE) return CC_LADDER_EINVAL;
    if (p->opt_exchange && (p->opt_split || p->opt_algo == CC_LADDER_ALGO_SIMPLE)) return CC_LADDER_EINVAL;
    if (p->opt_layout && (p->opt_split || p->opt_algo == CC_LADDER_ALGO_SIMPLE)) return CC_LADDER_EINVAL;

    if (p->opt_algo == CC_LADDER_ALGO_SIMPLE) {
        const size_t need = cc_ladder_workspace_bytes(p);
        if (!p->ws || p->ws_bytes < need) return CC_LADDER_EWORKSPACE;
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

    const TileGeom g = geom_of(p);
    FusedParams fp;
    fill_params(p, g, fp);
    fp.L = L;
    fp.t = t;
    fp.R = R;
    long long grid = p->opt_num_ctas > 0 ? p->opt_num_ctas : p->num_sms;
    if (p->opt_split) {
        // a0 pack -> fused kernel on CTA pairs -> a5 unpack; workspace = [T+ | T- | W+ | W-], each o^2 v^2 doubles
        const size_t need = cc_ladder_workspace_bytes(p);
        if (!p->ws || p->ws_bytes < need) return CC_LADDER_EWORKSPACE;
        const size_t n = (size_t)p->o * p->o * vv;
        double *Tp = (double *)p->ws, *Tm = Tp + n, *Wp = Tm + n, *Wm = Wp + n;
        const long long oo = (long long)p->o * p->o;
        const int nt = ceil_div(p->v, kTT);
        const dim3 tgrid((unsigned)nt, (unsigned)nt, (unsigned)(oo < 32768 ? oo : 32768));
        cudaError_t e = cudaMemsetAsync(Wp, 0, 2 * n * sizeof(double), s);
        if (e != cudaSuccess) return fail_cuda(p, e, "cudaMemsetAsync");
        split_pack_kernel<<<tgrid, 256, 0, s>>>(t, Tp, Tm, oo, p->v);
        fp.t = Tp;
        fp.tm = Tm;
        fp.R = Wp;
        fp.Rm = Wm;
        long long pairs = grid / 2;
        if (pairs < 1) pairs = 1;
        if (pairs > fp.n_tiles) pairs = fp.n_tiles;
        const int rc = launch_fused<CfgSplit, true>(p, fp, (int)(2 * pairs), s);
        if (rc != CC_LADDER_OK) return rc;
        split_unpack_kernel<<<tgrid, 256, 0, s>>>(Wp, Wm, R, oo, p->v, CfgSplit::TA);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(p, e, "split pack/unpack launch");
        return CC_LADDER_OK;
    }
    if (grid > fp.n_tiles) grid = fp.n_tiles;
    if (g.id == 4) return launch_fused<CfgSplit, false>(p, fp, (int)grid, s);
    if (g.id == 2) return launch_fused<CfgP12, false>(p, fp, (int)grid, s);
    if (g.id == 3) return launch_fused<CfgP20, false>(p, fp, (int)grid, s);
    return launch_fused<CfgP2, false>(p, fp, (int)grid, s);
}

int cc_ladder_host(cc_ladder_plan_t p, const double *L_host, const double *t_host, double *R_host)
{
    if (!p || !L_host || !t_host || !R_host) return CC_LADDER_EINVAL;
    const size_t vv = (size_t)p->v * p->v;
    const size_t nL = (size_t)p->x * vv * sizeof(double);
    const size_t nT = (size_t)p->o * p->o * vv * sizeof(double);
    if (overlaps(R_host, nT, L_host, nL) || overlaps(R_host, nT, t_host, nT)) return CC_LADDER_EINVAL;
    double *dL = nullptr, *dT = nullptr, *dR = nullptr;
    void *dW = nullptr;
    void *saved_ws = p->ws;
    size_t saved_ws_bytes = p->ws_bytes;
    int rc = CC_LADDER_OK;
    cudaError_t e;
    const size_t need = cc_ladder_workspace_bytes(p);
    if ((e = cudaMalloc(&dL, nL)) != cudaSuccess || (e = cudaMalloc(&dT, nT)) != cudaSuccess ||
        (e = cudaMalloc(&dR, nT)) != cudaSuccess || (need && (e = cudaMalloc(&dW, need)) != cudaSuccess)) {
        rc = (e == cudaErrorMemoryAllocation) ? CC_LADDER_ENOMEM : fail_cuda(p, e, "cudaMalloc");
        (void)cudaGetLastError();
        goto done;
    }
    if (need) { p->ws = dW; p->ws_bytes = need; }
    if ((e = cudaMemcpyAsync(dL, L_host, nL, cudaMemcpyHostToDevice, 0)) != cudaSuccess ||
        (e = cudaMemcpyAsync(dT, t_host, nT, cudaMemcpyHostToDevice, 0)) != cudaSuccess ||
        (e = cudaMemcpyAsync(dR, R_host, nT, cudaMemcpyHostToDevice, 0)) != cudaSuccess) {
        rc = fail_cuda(p, e, "cudaMemcpy H2D");
        goto done;
    }
    rc = cc_ladder(p, dL, dT, dR, nullptr);
    if (rc != CC_LADDER_OK) goto done;
    if ((e = cudaMemcpyAsync(R_host, dR, nT, cudaMemcpyDeviceToHost, 0)) != cudaSuccess ||
        (e = cudaStreamSynchronize(0)) != cudaSuccess) {
        rc = fail_cuda(p, e, "cudaMemcpy D2H");
        goto done;
    }
done:
    p->ws = saved_ws;
    p->ws_bytes = saved_ws_bytes;
    if (dL) cudaFree(dL);
    if (dT) cudaFree(dT);
    if (dR) cudaFree(dR);
    if (dW) cudaFree(dW);
    return rc;
}

int cc_ladder_destroy(cc_ladder_plan_t p)
{
    delete p;
    return CC_LADDER_OK;
}

}  // extern "C"
