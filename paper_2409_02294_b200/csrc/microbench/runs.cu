// runs.cu -- microbenchmarks behind two design decisions of DESIGN.md section 7.  Not part of the library; built and run
// by `python bench.py --pipes` on the GPU box next to pipes.cu.  Output: one line per measurement, "name value unit".
//   1. What does the memory system deliver for the TRANSPOSED accesses of the row kernels -- W[m][i] touched in runs of
//      ROWS x 16 bytes -- by run length and by path (STG / LDG from registers, or a 4-D TMA tile store / load whose inner
//      box is one run)?  33.6 MB per pass at n_r = 2048: 32-byte runs cap at 4.0 TB/s on every path, 64-byte runs reach
//      5.3 (STG) .. 7.7 TB/s (LDG); the TMA store stays at 4.0.  (-> 4 rows per CTA, plain stores.)
//   2. Does a 16 x 16 complex128 transpose among 16 lanes cost less by warp shuffles than through shared memory (the
//      pass B <-> C exchange of the column transform, which north_star's "warp-shuffle butterflies" would apply to)?
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1); } } while (0)

typedef double2 cplx;
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

template <int ROWS, int RA>
__global__ void __launch_bounds__(128) tma_store_kernel(const __grid_constant__ CUtensorMap tm, int n_items, int sts)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *tile = reinterpret_cast<cplx *>(smem_raw);
    constexpr int TILE = RA * 64 * ROWS;     // complex slots
    const int tid = threadIdx.x;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        if (sts) {
#pragma unroll
            for (int j = 0; j < TILE / 128; ++j) tile[tid + 128 * j] = make_double2(item + j, tid);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(&tm),
                         "r"(2 * ROWS * item), "r"(0), "r"(0), "r"(0), "r"(smem_addr(tile))
                         : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        __syncthreads();
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

template <int ROWS, int RA>
__global__ void __launch_bounds__(128) tma_load_kernel(const __grid_constant__ CUtensorMap tm, int n_items, double *out)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *tile = reinterpret_cast<cplx *>(smem_raw);
    constexpr int TILE = RA * 64 * ROWS;
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x;
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_addr(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned phase = 0;
    double acc = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        if (tid == 0) {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(&bar)), "r"(TILE * 16) : "memory");
            asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(smem_addr(tile)),
                         "l"(&tm), "r"(2 * ROWS * item), "r"(0), "r"(0), "r"(0), "r"(smem_addr(&bar))
                         : "memory");
        }
        unsigned done;
        do {
            asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}" : "=r"(done) : "r"(smem_addr(&bar)), "r"(phase) : "memory");
        } while (!done);
        phase ^= 1;
#pragma unroll
        for (int j = 0; j < TILE / 128; ++j) acc += tile[tid + 128 * j].x;
        __syncthreads();
    }
    if (acc == 1.2345) out[0] = acc;
}

// scattered reference: thread (t, rp) stores 16 modes k = 128 C + 16 a + b  (as the row kernel does)
template <int ROWS>
__global__ void __launch_bounds__(128) stg_kernel(cplx *W, int n_rows, int n_items, int L)
{
    const int tid = threadIdx.x;
    const int rp = tid % ROWS, t = tid / ROWS;
    const int T = 128 / ROWS;
    const int NB = L / 8;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        cplx *Wf = W + item * ROWS + rp;
        const int b1 = (8 + t) % NB;
        const int RA = L / 64;
        const int q1 = b1 / 8 + RA * (b1 % 8);
#pragma unroll
        for (int C = 0; C < 8; ++C) {
            const int k = q1 + NB * C;
            Wf[(long)k * n_rows] = make_double2(item, C);
            Wf[(long)(L - k) * n_rows] = make_double2(item, -C);
        }
    }
    (void)T;
}
template <int ROWS>
__global__ void __launch_bounds__(128) ldg_kernel(const cplx *W, int n_rows, int n_items, int L, double *out)
{
    const int tid = threadIdx.x;
    const int rp = tid % ROWS, t = tid / ROWS;
    const int NB = L / 8;
    double acc = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const cplx *Wf = W + item * ROWS + rp;
        const int b1 = (8 + t) % NB;
        const int RA = L / 64;
        const int q1 = b1 / 8 + RA * (b1 % 8);
#pragma unroll
        for (int C = 0; C < 8; ++C) {
            const int k = q1 + NB * C;
            acc += Wf[(long)k * n_rows].x + Wf[(long)(L - k) * n_rows].x;
        }
    }
    if (acc == 1.2345) out[0] = acc;
}

static PFN_cuTensorMapEncodeTiled get_encode()
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    CK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !fn) { printf("no cuTensorMapEncodeTiled\n"); exit(1); }
    return (PFN_cuTensorMapEncodeTiled)fn;
}

template <int ROWS, int RA>
static void run(int n_rows, bool a_before_c)
{
    const int L = 64 * RA;
    const size_t wn = (size_t)(L + 1) * n_rows;
    cplx *W; double *out;
    CK(cudaMalloc(&W, wn * sizeof(cplx)));
    CK(cudaMalloc(&out, 64));
    CK(cudaMemset(W, 0, wn * sizeof(cplx)));
    auto enc = get_encode();
    CUtensorMap tm;
    cuuint64_t dims[4], strides[3];
    cuuint32_t box[4], es[4] = {1, 1, 1, 1};
    dims[0] = 2 * (cuuint64_t)n_rows; box[0] = 2 * ROWS;
    if (a_before_c) {
        dims[1] = 64; strides[0] = (cuuint64_t)RA * n_rows * 16; box[1] = 64;
        dims[2] = RA; strides[1] = (cuuint64_t)n_rows * 16;      box[2] = RA;
    } else {
        dims[1] = RA; strides[0] = (cuuint64_t)n_rows * 16;      box[1] = RA;
        dims[2] = 64; strides[1] = (cuuint64_t)RA * n_rows * 16; box[2] = 64;
    }
    dims[3] = 1; strides[2] = (cuuint64_t)wn * 16; box[3] = 1;
    CUresult r = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, W, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { printf("status tensor map rejected (%d)\n", (int)r); cudaFree(W); cudaFree(out); return; }
    char tag[64];
    snprintf(tag, sizeof tag, "run_bytes=%d,n_rows=%d", 16 * ROWS, n_rows);
    const int n_items = n_rows / ROWS;
    const size_t smem = (size_t)RA * 64 * ROWS * 16;
    CK(cudaFuncSetAttribute(tma_store_kernel<ROWS, RA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaFuncSetAttribute(tma_load_kernel<ROWS, RA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const double mb = (double)L * n_rows * 16 / 1e6;
    for (int ctas = 2; ctas <= 4; ctas += 2) {
        const int grid = 148 * ctas;
        float ms;
        const int reps = 20;
        for (int sts = 0; sts < 2; ++sts) {
            tma_store_kernel<ROWS, RA><<<grid, 128, smem>>>(tm, n_items, sts);
            CK(cudaDeviceSynchronize());
            cudaEventRecord(e0);
            for (int k = 0; k < reps; ++k) tma_store_kernel<ROWS, RA><<<grid, 128, smem>>>(tm, n_items, sts);
            cudaEventRecord(e1); CK(cudaDeviceSynchronize());
            cudaEventElapsedTime(&ms, e0, e1);
            if (sts) printf("tma_store[%s,ctas_per_sm=%d] %.0f GB/s\n", tag, ctas, mb / (ms / reps));
        }
        tma_load_kernel<ROWS, RA><<<grid, 128, smem>>>(tm, n_items, out);
        CK(cudaDeviceSynchronize());
        cudaEventRecord(e0);
        for (int k = 0; k < reps; ++k) tma_load_kernel<ROWS, RA><<<grid, 128, smem>>>(tm, n_items, out);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
        cudaEventElapsedTime(&ms, e0, e1);
        printf("tma_load[%s,ctas_per_sm=%d] %.0f GB/s\n", tag, ctas, mb / (ms / reps));
        stg_kernel<ROWS><<<grid, 128>>>(W, n_rows, n_items, L);
        CK(cudaDeviceSynchronize());
        cudaEventRecord(e0);
        for (int k = 0; k < reps; ++k) stg_kernel<ROWS><<<grid, 128>>>(W, n_rows, n_items, L);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
        cudaEventElapsedTime(&ms, e0, e1);
        printf("stg[%s,ctas_per_sm=%d] %.0f GB/s\n", tag, ctas, mb / (ms / reps));
        ldg_kernel<ROWS><<<grid, 128>>>(W, n_rows, n_items, L, out);
        CK(cudaDeviceSynchronize());
        cudaEventRecord(e0);
        for (int k = 0; k < reps; ++k) ldg_kernel<ROWS><<<grid, 128>>>(W, n_rows, n_items, L, out);
        cudaEventRecord(e1); CK(cudaDeviceSynchronize());
        cudaEventElapsedTime(&ms, e0, e1);
        printf("ldg[%s,ctas_per_sm=%d] %.0f GB/s\n", tag, ctas, mb / (ms / reps));
    }
    // correctness of the tile mapping: store once with sts, read back, check a few entries
    tma_store_kernel<ROWS, RA><<<148, 128, smem>>>(tm, n_items, 1);
    CK(cudaDeviceSynchronize());
    cplx *h = (cplx *)malloc(wn * sizeof(cplx));
    CK(cudaMemcpy(h, W, wn * sizeof(cplx), cudaMemcpyDeviceToHost));
    // tile slot s = tid + 128 j holds (item + j, tid); slot order = [outer box dim][middle][rows]
    int bad = 0;
    for (int item = 0; item < n_items; item += 97) {
        for (int s = 0; s < RA * 64 * ROWS; s += 13) {
            const int rp = s % ROWS;
            const int mid = (s / ROWS) % (a_before_c ? 64 : RA);
            const int outer = s / ROWS / (a_before_c ? 64 : RA);
            const int a = a_before_c ? mid : outer, c = a_before_c ? outer : mid;
            const int m = RA * a + c;
            const cplx got = h[(size_t)m * n_rows + item * ROWS + rp];
            if (got.x != item + s / 128 || got.y != s % 128) ++bad;
        }
    }
    printf("tma_tile_mapping_errors[%s] %d count\n", tag, bad);
    free(h);
    cudaFree(W); cudaFree(out);
}


// ---------------------------------------------------------------- 2. 16 x 16 complex128 transpose among 16 lanes
// out[j] of lane l = in[l] of lane j.  SHARED: 16 STS.128 into a padded [16][17] tile per 16-lane group, __syncwarp,
// 16 LDS.128 (what cols_kernel does between passes B and C).  SHUFFLE: four butterfly stages, each exchanging half
// of the registers with the lane at distance 1, 2, 4, 8 (8 complex = 32 SHFL.32 per stage, plus the selects that
// static register indexing needs).
template <int MODE>
__global__ void __launch_bounds__(256) transpose16(double *out, int iters, long long *clk)
{
    extern __shared__ __align__(16) unsigned char tile_raw[];
    cplx (*tile)[16 * 17] = reinterpret_cast<cplx (*)[16 * 17]>(tile_raw);
    cplx v[16];
    const int lane = threadIdx.x & 15, grp = threadIdx.x >> 4;
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = make_double2(threadIdx.x + 0.001 * j, j);
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if (MODE == 0) {
#pragma unroll
            for (int j = 0; j < 16; ++j) tile[grp][17 * lane + j] = v[j];
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = tile[grp][17 * j + lane];
            __syncwarp();
        } else {
#pragma unroll
            for (int b = 1; b < 16; b <<= 1) {
                const bool up = (lane & b) != 0;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    if (j & b) continue;
                    const cplx send = up ? v[j] : v[j | b];
                    cplx recv;
                    recv.x = __shfl_xor_sync(0xffffffffu, send.x, b);
                    recv.y = __shfl_xor_sync(0xffffffffu, send.y, b);
                    if (up) v[j] = recv; else v[j | b] = recv;
                }
            }
        }
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) s += v[j].x + v[j].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) clk[0] = t1 - t0;
}
static void run_transpose()
{
    double *out; long long *clk;
    CK(cudaMalloc(&out, 148 * 256 * sizeof(double)));
    CK(cudaMalloc(&clk, 8));
    const int iters = 2000;
    long long c[2];
    const size_t sm = 16 * 16 * 17 * sizeof(cplx);
    CK(cudaFuncSetAttribute(transpose16<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    CK(cudaFuncSetAttribute(transpose16<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    transpose16<0><<<148, 256, sm>>>(out, 10, clk);
    transpose16<0><<<148, 256, sm>>>(out, iters, clk);
    CK(cudaDeviceSynchronize()); CK(cudaMemcpy(&c[0], clk, 8, cudaMemcpyDeviceToHost));
    transpose16<1><<<148, 256, sm>>>(out, 10, clk);
    transpose16<1><<<148, 256, sm>>>(out, iters, clk);
    CK(cudaDeviceSynchronize()); CK(cudaMemcpy(&c[1], clk, 8, cudaMemcpyDeviceToHost));
    // 8 warps per SM, each exchange moves 16 complex per lane
    printf("transpose16x16[shared_memory,8_warps_per_sm] %.1f clk_per_exchange_per_warp\n", (double)c[0] / iters / 8.0);
    printf("transpose16x16[warp_shuffle,8_warps_per_sm] %.1f clk_per_exchange_per_warp\n", (double)c[1] / iters / 8.0);
    cudaFree(out); cudaFree(clk);
}

int main()
{
    run<2, 16>(2048, true);
    run<4, 16>(2048, true);
    run_transpose();
    printf("status ok\n");
    return 0;
}
