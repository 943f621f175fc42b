// cartesian.cuh -- kernels of row NEXT-2: the paper's own per-GPU workload, the convolution
// method on ONE uniform 3-D Cartesian mesh level of N^3 cells, isolated boundary by zero
// padding to (2N)^3 (readings C1-C4 of DESIGN.md section 3; the method's ref. [13] is not available).
//
//   Phi = -G h^2 * crop( IFFT3( Ghat . FFT3( pad(rho) ) ) ),   G(d) = 1/|d| on the lag grid, G(0) = S (cube integral)
//
// The volume is treated as N "fields" (z slices) of N rows (y) of M = 2N reals (x, zero padded), so that the x pass is
// rows_fwd_kernel<M> / rows_inv_kernel<M> of kernels.cuh unchanged (packed real transform, Hermitian half kx = 0..N,
// transposed store W1[z][kx][y]), and the z pass is cols_kernel<N> unchanged (zero-padded 2N-point transform x Ghat x
// inverse with crop, fused) over the (N+1) x 2N columns Yt[kx][ey][z].  New here: the y pass in between, which is
// the forward half of cols_kernel (N values in, all 2N bins out, in the plan's bin order ey) and its inverse half,
// with the transposition [z][kx][y] <-> [kx][ey][z] folded into their global accesses; the padding / cropping of x;
// and the one-time spectrum of the Green's function.  None of the padded arrays in y or z is ever formed.
#pragma once
#include "kernels.cuh"

namespace pgk {

// P[row][x] = rho[row][x] for x < n, 0 for n <= x < 2n   (row = z n + y)
__global__ void pad3_kernel(const double *__restrict__ rho, double *__restrict__ P, const int n, const long total)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int x = (int)(idx % (2 * n));
    const long row = idx / (2 * n);
    P[idx] = x < n ? rho[row * n + x] : 0.0;
}
__global__ void crop3_kernel(const double *__restrict__ P, double *__restrict__ phi, const int n, const long total)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int x = (int)(idx % n);
    const long row = idx / n;
    phi[idx] = P[row * 2 * n + x];
}

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

// y pass forward: column (z, kx) of W1[z][kx][y], y < N, zero padded to 2N -> all 2N bins, Yt[(kx M + ey) N + z]
template <int N>
__global__ void __launch_bounds__(ColShape<N>::THREADS)
ycols_fwd_kernel(const cplx *__restrict__ W1, cplx *__restrict__ Yt, const cplx *__restrict__ tw, const int n_cols)
{
    typedef ColShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int u = tid % T, ml = tid / T;
    const int c_raw = blockIdx.x * S::MODES + ml;
    const bool live = c_raw < n_cols;
    const int c = live ? c_raw : n_cols - 1;
    const int z = c / (N + 1), kx = c % (N + 1);
    cplx *line = smem + ml * S::STRIDE;
    const cplx *col = W1 + (long)z * (N + 1) * N + (long)kx * N;
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) v[jj] = col[u + T * jj];
    Bases<L, COL> bases;
    bases.load(tw, u, false);
    fwd_a_compute_zero_upper<L, COL>(v, bases, u);
    fwd_a_store<L, COL>(v, line, u);
    __syncthreads();
    if constexpr (P::NPASS == 3) {
        fwd_b<L, COL>(line, bases, u);
        __syncthreads();
    }
    fwd_c_col<L>(v, line, u);
    if (live) {
#pragma unroll
        for (int k = 0; k < 16; ++k) Yt[((long)kx * M + (u + T * k)) * N + z] = v[k];
    }
}
// y pass inverse: Yt[(kx M + ey) N + z] -> W1[z][kx][y], y < N (crop)
template <int N>
__global__ void __launch_bounds__(ColShape<N>::THREADS)
ycols_inv_kernel(const cplx *__restrict__ Yt, cplx *__restrict__ W1, const cplx *__restrict__ tw, const int n_cols)
{
    typedef ColShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int u = tid % T, ml = tid / T;
    const int c_raw = blockIdx.x * S::MODES + ml;
    const bool live = c_raw < n_cols;
    const int c = live ? c_raw : n_cols - 1;
    const int z = c / (N + 1), kx = c % (N + 1);
    cplx *line = smem + ml * S::STRIDE;
    cplx *col = W1 + (long)z * (N + 1) * N + (long)kx * N;
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = Yt[((long)kx * M + (u + T * k)) * N + z];
    Bases<L, COL> bases;
    bases.load(tw, u, false);
    inv_c_col<L>(v, line, u);
    if constexpr (P::NPASS == 3) {
        __syncthreads();
        inv_b<L, COL>(line, bases, u);
    }
    __syncthreads();
    inv_a_load<L, COL>(v, line, u);
    inv_a_compute_lower_half<L, COL>(v, bases, u);
    if (live) {
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) col[u + T * jj] = v[jj];
    }
}

// One-time spectrum of the Green's function: full (unpruned) 2N-point forward transforms along y' then z'.
//   MODE 0 (y'): column (z', kx) of GW[z'][kx][y'], y' < 2N  ->  GY[(kx M + ey) M + z']                 (complex)
//   MODE 1 (z'): column (kx, ey) of GY[(kx M + ey) M + z']   ->  Ghat[(kx M + ey) M + ez] = scale Re X  (real: G is even)
template <int N, int MODE>
__global__ void __launch_bounds__(ColShape<N>::THREADS)
gcols_kernel(const cplx *__restrict__ src, cplx *__restrict__ dstc, double *__restrict__ dstr, const cplx *__restrict__ tw,
             const int n_cols, const double scale)
{
    typedef ColShape<N> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T, M = 2 * N;
    extern __shared__ __align__(16) unsigned char smem_raw[];
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
#pragma unroll
            for (int k = 0; k < 16; ++k) dstr[(long)c * M + (u + T * k)] = scale * v[k].x;
        }
    }
}

}  // namespace pgk
