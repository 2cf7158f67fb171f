// FP64 microbenchmarks behind the roofline denominator and the kernel design (DESIGN.md sections 4 and 6):
// DMMA.8x8x4 issue rate / latency, DFMA rate, DMMA+DFMA mixing, shared-memory-fed DMMA warp tiles, sustained
// clocks, and red.global.add.f64 throughput in the accumulate step's access pattern.
// Stand-alone program (no library code):  python -m paper_2310_04559_b200.build --microbench
//                                         ./paper_2310_04559_b200/microbench_fp64.bin sustained
// Results of this pool's B200: profiles/r01_microbench.md.
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int ILP>
__global__ void k_dmma(double *out, int iters, long long *cyc) {
    double acc[ILP][2];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { acc[i][0] = threadIdx.x; acc[i][1] = i; }
    double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) dmma(acc[i][0], acc[i][1], a, b);
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += acc[i][0] + acc[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

template <int ILP>
__global__ void k_dfma(double *out, int iters, long long *cyc) {
    double acc[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) acc[i] = threadIdx.x + i;
    double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9 * threadIdx.x;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) acc[i] = fma(acc[i], a, b);
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

// mixed: per iteration NM dmma + NF dfma (independent)
template <int NM, int NF>
__global__ void k_mix(double *out, int iters, long long *cyc) {
    double acc[NM][2];
    double f[NF > 0 ? NF : 1];
#pragma unroll
    for (int i = 0; i < NM; ++i) { acc[i][0] = threadIdx.x; acc[i][1] = i; }
#pragma unroll
    for (int i = 0; i < NF; ++i) f[i] = threadIdx.x + i;
    double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < (NM > NF ? NM : NF); ++i) {
            if (i < NM) dmma(acc[i][0], acc[i][1], a, b);
            if (i < NF) f[i] = fma(f[i], a, b);
        }
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < NM; ++i) s += acc[i][0] + acc[i][1];
#pragma unroll
    for (int i = 0; i < NF; ++i) s += f[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

// DMMA fed from shared memory like a GEMM inner loop: warp tile (8*MI) x (8*NI), k-step 4.
template <int MI, int NI>
__global__ void k_dmma_smem(double *out, int iters, long long *cyc) {
    extern __shared__ double sm[];
    const int PITCH = 132;
    for (int i = threadIdx.x; i < 2 * 16 * PITCH; i += blockDim.x) sm[i] = 1.0 + i * 1e-9;
    __syncthreads();
    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) { acc[i][j][0] = 0; acc[i][j][1] = 0; }
    int lane = threadIdx.x & 31, g = lane >> 2, q = lane & 3;
    int warp = threadIdx.x >> 5;
    const double *A = sm + (warp & 1) * 8 * MI;
    const double *B = sm + 16 * PITCH + (warp >> 1) * 8 * NI % 64;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            double af[MI], bf[NI];
#pragma unroll
            for (int i = 0; i < MI; ++i) af[i] = A[(kk * 4 + q) * PITCH + i * 8 + g];
#pragma unroll
            for (int j = 0; j < NI; ++j) bf[j] = B[(kk * 4 + q) * PITCH + j * 8 + g];
#pragma unroll
            for (int i = 0; i < MI; ++i)
#pragma unroll
                for (int j = 0; j < NI; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) s += acc[i][j][0] + acc[i][j][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

// RED.f64 in the epilogue pattern: each warp-instruction covers 8 rows x 64 B; rows are `rowstride` doubles apart.
__global__ void k_red(double *buf, size_t nrows, size_t rowstride, int segs_per_row, int iters) {
    int lane = threadIdx.x & 31, g = lane >> 2, q = lane & 3;
    size_t warp = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    size_t nwarps = (size_t)gridDim.x * (blockDim.x >> 5);
    // each warp walks over (row-block of 8, segment) space
    size_t nblk = (nrows / 8) * (size_t)segs_per_row;
    size_t idx = warp % nblk;
    for (int it = 0; it < iters; ++it) {
        size_t rb = idx / segs_per_row, seg = idx % segs_per_row;
        double *p = buf + (rb * 8 + g) * rowstride + seg * 8 + 2 * q;
        asm volatile("red.global.add.f64 [%0], %1;" :: "l"(p), "d"(1.0) : "memory");
        asm volatile("red.global.add.f64 [%0], %1;" :: "l"(p + 1), "d"(1.0) : "memory");
        idx += nwarps; if (idx >= nblk) idx -= nblk * (idx / nblk);
    }
}

template <typename F>
float time_ms(F f, int reps = 3) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    f(); CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0); f(); cudaEventRecord(e1); CK(cudaEventSynchronize(e1));
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    return best;
}

int main(int argc, char **argv) {
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    printf("device %s cc %d.%d SMs %d clock %d kHz smem/block optin %zu L2 %d MB regs/SM %d\n", p.name, p.major, p.minor,
           p.multiProcessorCount, p.clockRate, p.sharedMemPerBlockOptin, p.l2CacheSize >> 20, p.regsPerMultiprocessor);
    int nsm = p.multiProcessorCount;
    double *out; CK(cudaMalloc(&out, sizeof(double) * nsm * 1024 * 4));
    long long *cyc; CK(cudaMallocManaged(&cyc, 8));
    const int iters = 20000;

#define RUN_DMMA(ILP, WARPS) { \
        float ms = time_ms([&] { k_dmma<ILP><<<nsm, 32 * WARPS>>>(out, iters, cyc); }); \
        CK(cudaDeviceSynchronize()); \
        double fl = (double)nsm * WARPS * iters * ILP * 512.0; \
        printf("DMMA ilp %d warps/SM %2d: %.3f ms %.2f TF/s  cyc/dmma/warp %.2f  flop/clk/SM %.1f\n", ILP, WARPS, ms, fl / ms * 1e-9, \
               (double)*cyc / (iters * ILP), (double)WARPS * iters * ILP * 512.0 / (double)*cyc); }
    RUN_DMMA(1, 1) RUN_DMMA(2, 1) RUN_DMMA(4, 1) RUN_DMMA(8, 1) RUN_DMMA(16, 1)
    RUN_DMMA(1, 4) RUN_DMMA(2, 4) RUN_DMMA(4, 4) RUN_DMMA(8, 4) RUN_DMMA(16, 4)
    RUN_DMMA(4, 8) RUN_DMMA(8, 8) RUN_DMMA(16, 8)
    RUN_DMMA(4, 16) RUN_DMMA(8, 16)
    RUN_DMMA(8, 32)

#define RUN_DFMA(ILP, WARPS) { \
        float ms = time_ms([&] { k_dfma<ILP><<<nsm, 32 * WARPS>>>(out, iters, cyc); }); \
        CK(cudaDeviceSynchronize()); \
        double fl = (double)nsm * WARPS * iters * ILP * 64.0; \
        printf("DFMA ilp %d warps/SM %2d: %.3f ms %.2f TF/s  cyc/dfma/warp %.2f  flop/clk/SM %.1f\n", ILP, WARPS, ms, fl / ms * 1e-9, \
               (double)*cyc / (iters * ILP), (double)WARPS * iters * ILP * 64.0 / (double)*cyc); }
    RUN_DFMA(1, 1) RUN_DFMA(8, 1) RUN_DFMA(8, 4) RUN_DFMA(8, 8) RUN_DFMA(8, 16) RUN_DFMA(8, 32)

#define RUN_MIX(NM, NF, WARPS) { \
        float ms = time_ms([&] { k_mix<NM, NF><<<nsm, 32 * WARPS>>>(out, iters, cyc); }); \
        CK(cudaDeviceSynchronize()); \
        double fl = (double)nsm * WARPS * iters * (NM * 512.0 + NF * 64.0); \
        printf("MIX dmma %d dfma %d warps/SM %2d: %.3f ms %.2f TF/s flop/clk/SM %.1f\n", NM, NF, WARPS, ms, fl / ms * 1e-9, \
               (double)WARPS * iters * (NM * 512.0 + NF * 64.0) / (double)*cyc); }
    RUN_MIX(8, 0, 8) RUN_MIX(8, 8, 8) RUN_MIX(8, 16, 8) RUN_MIX(4, 16, 8) RUN_MIX(8, 32, 8)

#define RUN_SM(MI, NI, WARPS) { \
        CK(cudaFuncSetAttribute(k_dmma_smem<MI, NI>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024)); \
        float ms = time_ms([&] { k_dmma_smem<MI, NI><<<nsm, 32 * WARPS, 2 * 16 * 132 * 8>>>(out, iters / 4, cyc); }); \
        CK(cudaDeviceSynchronize()); \
        double fl = (double)nsm * WARPS * (iters / 4) * 4.0 * MI * NI * 512.0; \
        printf("DMMA+LDS tile %dx%d warps/SM %2d: %.3f ms %.2f TF/s flop/clk/SM %.1f\n", MI * 8, NI * 8, WARPS, ms, fl / ms * 1e-9, \
               (double)WARPS * (iters / 4) * 4.0 * MI * NI * 512.0 / (double)*cyc); }
    RUN_SM(4, 4, 8) RUN_SM(8, 4, 8) RUN_SM(4, 8, 8) RUN_SM(4, 4, 16) RUN_SM(4, 2, 16) RUN_SM(2, 4, 16) RUN_SM(2, 2, 16) RUN_SM(8, 4, 4)

    // long sustained DMMA run for clocks (about 4 s)
    if (argc > 1) {
        float ms = time_ms([&] { k_dmma<8><<<nsm, 32 * 8>>>(out, 4000000, cyc); }, 1);
        double fl = (double)nsm * 8 * 4000000.0 * 8 * 512.0;
        printf("SUSTAINED DMMA: %.1f ms %.2f TF/s flop/clk/SM %.1f\n", ms, fl / ms * 1e-9, 8.0 * 4000000.0 * 8 * 512.0 / (double)*cyc);
        ms = time_ms([&] { k_dfma<8><<<nsm, 32 * 32>>>(out, 8000000, cyc); }, 1);
        fl = (double)nsm * 32 * 8000000.0 * 8 * 64.0;
        printf("SUSTAINED DFMA: %.1f ms %.2f TF/s flop/clk/SM %.1f\n", ms, fl / ms * 1e-9, 32.0 * 8000000.0 * 8 * 64.0 / (double)*cyc);
    }

    // RED throughput
    {
        size_t big = (size_t)6 << 30;
        double *buf; CK(cudaMalloc(&buf, big)); CK(cudaMemset(buf, 0, big));
        struct { size_t nrows, rowstride; int segs; const char *name; } cases[] = {
            {1600, 90000, 16, "cfg2-like R block, 148 CTA same block? rows 1600 x 128 doubles (1.6MB)"},
            {4096, 270400, 16, "cfg4-like R block rows 4096 x 128 doubles (4MB)"},
            {4096, 2048, 256, "dense 64 MB region"},
            {4096 * 32, 2048, 256, "dense 2 GB region"},
        };
        for (auto &c : cases) {
            if ((c.nrows - 1) * c.rowstride * 8 + c.segs * 64 > big) { printf("skip %s\n", c.name); continue; }
            for (int warps : {2, 8}) {
                int it = 2000;
                float ms = time_ms([&] { k_red<<<nsm, 32 * warps>>>(buf, c.nrows, c.rowstride, c.segs, it); });
                double n = (double)nsm * warps * it * 64.0;
                printf("RED %-70s warps/SM %d: %.3f ms  %.3e doubles/s  (%.1f GB/s payload)\n", c.name, warps, ms, n / ms * 1e3, n * 8 / ms * 1e-6);
            }
        }
        CK(cudaFree(buf));
    }
    return 0;
}
