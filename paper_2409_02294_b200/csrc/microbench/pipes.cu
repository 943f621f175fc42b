// pipes.cu -- microbenchmarks behind the pipe model of DESIGN.md section 7 (what bounds the FFT kernels on sm_100a).
// Not part of the library; built and run by `python bench.py --pipes` on the GPU box.  Three questions:
//   1. How fast does the FP64 pipe issue, by operand pattern and by warps per SM sub-partition?
//      (a DFMA with three distinct register-pair sources needs several warps to reach the pipe's rate)
//   2. Do FP64 arithmetic and shared-memory traffic of different warps of one SM overlap?
//   3. What does a warp-wide 16-byte store / load cost when it is scattered over runs of R elements
//      (the transposed accesses of the row kernels: runs of 4 rows = 64 bytes)?
// Output: one line per measurement, "name value unit".
#include <cstdio>
#include <cuda_runtime.h>

// ---------------------------------------------------------------- 1. FP64 issue rate
template <int MODE>
__global__ void fp64_rate(double *out, int iters, double a, double b)
{
    double x[8], y[8], z[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 1e-3 + i; y[i] = a + i * 1e-9; z[i] = b + i * 1e-9; }
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE == 0) x[i] = fma(x[i], y[i], b);             // two register pairs + a uniform operand
                else if (MODE == 1) x[i] = fma(x[i], y[i], z[i]);     // three distinct register pairs
                else if (MODE == 2) x[i] = x[i] + y[i];               // DADD
                else x[i] = x[i] * y[i];                              // DMUL
            }
        }
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = (double)(t1 - t0);
}
template <int MODE>
static void run_rate(const char *name, int warps, double *d)
{
    const int iters = 2000;
    fp64_rate<MODE><<<148, warps * 32>>>(d, 10, 1.0000001, 1e-9);
    fp64_rate<MODE><<<148, warps * 32>>>(d, iters, 1.0000001, 1e-9);
    cudaDeviceSynchronize();
    double clk; cudaMemcpy(&clk, d, 8, cudaMemcpyDeviceToHost);
    printf("fp64_issue[%s,warps_per_smsp=%d] %.2f clk_per_warp_instruction_per_smsp\n", name, warps / 4, clk / ((double)iters * 32 * warps / 4));
}

// ---------------------------------------------------------------- 2. FP64 || shared memory
__global__ void __launch_bounds__(512, 1) overlap(double *out, int itF, int itL, long long *clk)
{
    extern __shared__ __align__(16) double2 sm[];
    const int w = threadIdx.x / 32;
    long long t0 = clock64();
    double acc = 0;
    if (w < 8) {                       // warps 0..7: FP64 only
        double x[16], y[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) { x[i] = threadIdx.x * 1e-3 + i; y[i] = 1.0 + i * 1e-9; }
        for (int it = 0; it < itF; ++it) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = x[i] + y[i];
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) acc += x[i];
    } else {                           // warps 8..15: 16 STS.128 + 16 LDS.128 per round, conflict-free
        double2 v[16];
        double2 *p = sm + (threadIdx.x - 256) + ((threadIdx.x - 256) / 8);
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = make_double2(threadIdx.x + i, i);
        for (int it = 0; it < itL; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i) p[i * 300] = v[i];
            __syncwarp();
#pragma unroll
            for (int i = 0; i < 16; ++i) { double2 t = p[((i + 1) & 15) * 300]; v[i].x += t.x; v[i].y = t.y; }
            __syncwarp();
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) acc += v[i].x + v[i].y;
    }
    long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x % 256 == 0 && blockIdx.x == 0) clk[threadIdx.x / 256] = t1 - t0;
}
static void run_overlap(const char *name, int itF, int itL, double *d, long long *c)
{
    cudaFuncSetAttribute(overlap, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    overlap<<<148, 512, 100 * 1024>>>(d, itF, itL, c);
    overlap<<<148, 512, 100 * 1024>>>(d, itF, itL, c);
    cudaDeviceSynchronize();
    long long h[2]; cudaMemcpy(h, c, 16, cudaMemcpyDeviceToHost);
    if (itF) printf("overlap[%s].fp64 %.2f clk_per_warp_instruction_per_smsp\n", name, (double)h[0] / (itF * 64.0 * 2));
    if (itL) printf("overlap[%s].lsu %.2f clk_per_16B_warp_access_per_sm\n", name, (double)h[1] / (itL * 32.0 * 8));
}

// ---------------------------------------------------------------- 3. scattered 16-byte accesses
template <int RUN, bool LOAD>
__global__ void __launch_bounds__(256, 1) scatter(double2 *w, long col_stride, int iters, long long *clk)
{
    const int lane = threadIdx.x % 32, warp = threadIdx.x / 32;
    double2 *p = w + (long)blockIdx.x * 4096 * col_stride / 148 + (long)(warp * (32 / RUN) + lane / RUN) * col_stride + (lane % RUN);
    double2 v = make_double2(lane, warp), acc = make_double2(0, 0);
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            double2 *q = p + (long)j * 256 * col_stride / 64 + (it & 7) * RUN;
            if (LOAD) { double2 t = *q; acc.x += t.x; acc.y += t.y; }
            else *q = v;
        }
    }
    long long t1 = clock64();
    if (LOAD && acc.x == 123.456) w[0] = acc;
    if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
}
template <int RUN, bool LOAD>
static void run_scatter(double2 *w, long long *c)
{
    const int iters = 200;
    scatter<RUN, LOAD><<<148, 256>>>(w, 2048, iters, c);
    scatter<RUN, LOAD><<<148, 256>>>(w, 2048, iters, c);
    cudaDeviceSynchronize();
    long long h; cudaMemcpy(&h, c, 8, cudaMemcpyDeviceToHost);
    printf("scatter[%s,run_bytes=%d] %.1f clk_per_warp_instruction_per_sm\n", LOAD ? "ldg128" : "stg128", RUN * 16, (double)h / (iters * 16.0 * 8));
}

int main()
{
    double *d; long long *c; double2 *w;
    cudaMalloc(&d, 148 * 1024 * 8); cudaMalloc(&c, 16); cudaMalloc(&w, (size_t)1100 * 2048 * 16 * 4);
    for (int warps : {4, 8, 16}) {
        run_rate<0>("dfma_2reg_1uniform", warps, d);
        run_rate<1>("dfma_3reg", warps, d);
        run_rate<2>("dadd", warps, d);
        run_rate<3>("dmul", warps, d);
    }
    run_overlap("fp64_alone", 2000, 0, d, c);
    run_overlap("lsu_alone", 0, 500, d, c);
    run_overlap("together", 2000, 500, d, c);
    run_scatter<2, false>(w, c); run_scatter<4, false>(w, c); run_scatter<8, false>(w, c); run_scatter<16, false>(w, c);
    run_scatter<2, true>(w, c); run_scatter<4, true>(w, c); run_scatter<8, true>(w, c); run_scatter<16, true>(w, c);
    cudaError_t e = cudaDeviceSynchronize();
    printf("status %s\n", cudaGetErrorString(e));
    return e == cudaSuccess ? 0 : 1;
}
