// cartesian.cuh -- kernels of row NEXT-2: the paper's own per-GPU workload, the convolution
// method on ONE uniform 3-D Cartesian mesh level of N^3 cells, isolated boundary by zero
// padding to (2N)^3 (readings C1-C4 of DESIGN.md section 3; the method's ref. [13] is not available).
//
//   Phi = -G h^2 * crop( IFFT3( Ghat . FFT3( pad(rho) ) ) ),   G(d) = 1/|d| on the lag grid, G(0) = S (cube integral)
//
// The volume is treated as N "fields" (z slices) of N rows (y) of M = 2N reals (x, zero padded), so that the x pass is
// rows_fwd_kernel<M, HALF> / rows_inv_kernel<M, HALF> of kernels.cuh (packed real transform, Hermitian half
// kx = 0..N, transposed store W1[z][kx][y]; HALF: the zero half of a row is neither read nor written, rho and Phi are
// accessed in place), and the z pass is cols_kernel<N> unchanged (zero-padded 2N-point transform x Ghat x
// inverse with crop, fused) over the (N+1) x 2N columns Yt[kx][ey][z].  New here: the y pass in between, which is
// the forward half of cols_kernel (N values in, all 2N bins out, in the plan's bin order ey) and its inverse half,
// with the transposition [z][kx][y] <-> [kx][ey][z] folded into their global accesses, and the one-time spectrum of
// the Green's function.  None of the padded arrays is ever formed.
#pragma once
#include "kernels.cuh"

namespace pgk {

// Green's function on the padded lag grid [2n][2n][2n]: lag = l (l < n), l - 2n (l > n); slots l = n unused (0)
__global__ void green3_fill_kernel(double *__restrict__ G, const int n, const double self, const long total)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int m = 2 * n;
    const int lx = (int)(idx % m), ly = (int)((idx / m) % m), lz = (int)(idx / ((long)m * m));
    double val = 0.0;
    if (lx != n && ly != n && lz != n) {
        const double dx = lx < n ? lx : lx - m, dy = ly < n ? ly : ly - m, dz = lz < n ? lz : lz - m;
        const double d2 = dx * dx + dy * dy + dz * dz;
        val = d2 > 0.0 ? rsqrt(d2) : self;
    }
    G[idx] = val;
}

// Shape of the y pass: YM columns per CTA (consecutive z of one kx).  Passes A / B run with thread = (column, u), u
// fastest (a column is read / written as 16-byte elements contiguous in y); pass C runs with thread = (u, column),
// the COLUMN fastest, so that the bins leave / arrive as runs of YM consecutive z (YM x 16 bytes) of one (kx, ey):
// the transposition [z][kx][y] <-> [kx][ey][z] costs no extra shared-memory round trip.  The line stride is odd in
// 16-byte units so that the column-fastest accesses spread over the bank groups.
template <int N>
struct YShape {
    static constexpr int L = 2 * N;
    typedef Plan<L, COL> P;
    static constexpr int T = P::T;
    static constexpr int YM = (256 / T < 8) ? 256 / T : 8;
    static constexpr int THREADS = YM * T;
    static constexpr int STRIDE = P::LINE | 1;
    static constexpr size_t SMEM = (size_t)YM * STRIDE * sizeof(cplx);
    static_assert(N % YM == 0, "a CTA's columns share one kx");
};

// y pass forward: column (kx, z) of W1[z][kx][y], y < N, zero padded to 2N -> all 2N bins, Yt[(kx M + ey) N + z]
template <int N>
__global__ void __launch_bounds__(YShape<N>::THREADS)
ycols_fwd_kernel(const cplx *__restrict__ W1, cplx *__restrict__ Yt, const cplx *__restrict__ tw)
{
    typedef YShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N, YM = S::YM;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int c0 = blockIdx.x * YM;                 // columns c = kx N + z, z fastest
    const int kx = c0 / N, z0 = c0 % N;
    Bases<L, COL> bases;
    {
        const int u = tid % T, ml = tid / T;
        cplx *line = smem + ml * S::STRIDE;
        const cplx *col = W1 + (long)(z0 + ml) * (N + 1) * N + (long)kx * N;
        cplx v[16];
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) v[jj] = col[u + T * jj];
        bases.load(tw, u, false);
        fwd_a_compute_zero_upper<L, COL>(v, bases, u);
        fwd_a_store<L, COL>(v, line, u);
        __syncthreads();
        if constexpr (P::NPASS == 3) {
            fwd_b<L, COL>(line, bases, u);
            __syncthreads();
        }
    }
    {
        const int ml = tid % YM, u = tid / YM;
        cplx v[16];
        fwd_c_col<L>(v, smem + ml * S::STRIDE, u);
        cplx *dst = Yt + ((long)kx * M + u) * N + z0 + ml;
#pragma unroll
        for (int k = 0; k < 16; ++k) dst[(long)(T * k) * N] = v[k];
    }
}
// y pass inverse: Yt[(kx M + ey) N + z] -> W1[z][kx][y], y < N (crop)
template <int N>
__global__ void __launch_bounds__(YShape<N>::THREADS)
ycols_inv_kernel(const cplx *__restrict__ Yt, cplx *__restrict__ W1, const cplx *__restrict__ tw)
{
    typedef YShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N, YM = S::YM;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int c0 = blockIdx.x * YM;
    const int kx = c0 / N, z0 = c0 % N;
    {
        const int ml = tid % YM, u = tid / YM;
        const cplx *src = Yt + ((long)kx * M + u) * N + z0 + ml;
        cplx v[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = src[(long)(T * k) * N];
        inv_c_col<L>(v, smem + ml * S::STRIDE, u);
    }
    __syncthreads();
    {
        const int u = tid % T, ml = tid / T;
        cplx *line = smem + ml * S::STRIDE;
        Bases<L, COL> bases;
        bases.load(tw, u, false);
        if constexpr (P::NPASS == 3) {
            inv_b<L, COL>(line, bases, u);
            __syncthreads();
        }
        cplx v[16];
        inv_a_load<L, COL>(v, line, u);
        inv_a_compute_lower_half<L, COL>(v, bases, u);
        cplx *col = W1 + (long)(z0 + ml) * (N + 1) * N + (long)kx * N;
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) col[u + T * jj] = v[jj];
    }
}

// One-time spectrum of the Green's function: full (unpruned) 2N-point forward transforms along y' then z'.
//   MODE 0 (y'): column (z', kx) of GW[z'][kx][y'], y' < 2N  ->  GY[(kx M + ey) M + z']                 (complex)
//   MODE 1 (z'): column (kx, ey) of GY[(kx M + ey) M + z']   ->  Ghat[(kx M + ey)][.] = scale Re X      (real: G is even;
//                stored as its symmetric half in ez, ColShape<N>::KH doubles per column)
template <int N, int MODE>
__global__ void __launch_bounds__(ColShape<N>::THREADS)
gcols_kernel(const cplx *__restrict__ src, cplx *__restrict__ dstc, double *__restrict__ dstr, const cplx *__restrict__ tw,
             const int n_cols, const double scale)
{
    typedef ColShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int u = tid % T, ml = tid / T;
    const int c_raw = blockIdx.x * S::MODES + ml;
    const bool live = c_raw < n_cols;
    const int c = live ? c_raw : n_cols - 1;
    cplx *line = smem + ml * S::STRIDE;
    const cplx *col = src + (long)c * M;        // MODE 0: c = z' (N+1) + kx;  MODE 1: c = kx M + ey
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) v[jj] = col[u + T * jj];
    Bases<L, COL> bases;
    bases.load(tw, u, false);
    fwd_a<L, COL>(v, line, bases, u);
    __syncthreads();
    if constexpr (P::NPASS == 3) {
        fwd_b<L, COL>(line, bases, u);
        __syncthreads();
    }
    fwd_c_col<L>(v, line, u);
    if (live) {
        if constexpr (MODE == 0) {
            const int zp = c / (N + 1), kx = c % (N + 1);
#pragma unroll
            for (int k = 0; k < 16; ++k) dstc[((long)kx * M + (u + T * k)) * M + zp] = v[k];
        } else {
            double *kh = dstr + (long)c * (L / 2 + 2);     // symmetric half in ez, the layout cols_kernel reads
#pragma unroll
            for (int k = 0; k < 8; ++k) kh[u + T * k] = scale * v[k].x;
            if (u == 0) { kh[8 * T] = scale * v[8].x; kh[8 * T + 1] = 0.0; }
        }
    }
}

}  // namespace pgk
