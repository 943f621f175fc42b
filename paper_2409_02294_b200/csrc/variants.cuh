// variants.cuh -- kernels of the NEXT-4 variants of the path (readings
// N1 and N2): softening length of the field or of the source cell (the pair kernel is then not even in the radial
// lag and its spectrum is complex), and the softened pair acceleration (-grad Phi for source softening) as two
// more convolutions that share the forward transform of the density with the potential.
//
//   D(k,l)      = 4 sinh^2(k du/2) + 4 sin^2(l dphi/2) + eta^2 g(k),   g = 1 | e^{+k du} (field) | e^{-k du} (source),
//                 k = i - i' (field ring minus source ring), l = j - j'
//   K_Phi       = D^(-1/2)                                   Phi   = -c r_i^(-1/2) sum (Sigma r'^(3/2)) K_Phi
//   K_r         = (e^{k du} - cos(l dphi)) D^(-3/2)          a_r   = -c r_i^(-3/2) sum (Sigma r'^(3/2)) K_r
//   K_phi       = sin(l dphi) D^(-3/2)                       a_phi = -c r_i^(-3/2) sum (Sigma r'^(3/2)) K_phi
//   c = G sinh(du) dphi, eta^2 = eps^2 sinh(du) dphi.
//
// The solve kernels of kernels.cuh are untouched: these paths reuse rows_fwd_kernel / rows_inv_kernel and replace
// the column kernel by cols_cplx_kernel (complex spectrum read straight from global memory, separate source and
// destination so that one forward spectrum W serves several outputs).
#pragma once
#include "kernels.cuh"

namespace pgk {

// Kpad[k][l] for the padded lag grid (see green_fill_kernel); kind 0 = K_Phi, 1 = K_r, 2 = K_phi
__global__ void green_fill_var_kernel(double *__restrict__ Kpad, const int n_r, const int n_phi, const double du,
                                      const double eta2, const int soft, const int kind)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long total = 2L * n_r * n_phi;
    if (idx >= total) return;
    const int k = (int)(idx / n_phi), l = (int)(idx % n_phi);
    double val = 0.0;
    if (k != n_r) {
        const int lag = k < n_r ? k : k - 2 * n_r;
        const double x = du * (double)lag;
        const double sh = sinh(0.5 * x);
        const double sn = sinpi((double)l / (double)n_phi);
        const double g = soft == 1 ? exp(x) : (soft == 2 ? exp(-x) : 1.0);
        const double D = 4.0 * sh * sh + 4.0 * sn * sn + eta2 * g;
        const double inv = rsqrt(D);
        if (kind == 0) val = inv;
        else if (kind == 1) val = (expm1(x) + 2.0 * sn * sn) * inv / D;       // e^x - cos(l dphi), cancellation-free
        else val = sinpi(2.0 * (double)l / (double)n_phi) * inv / D;
    }
    Kpad[idx] = val;
}

// Column pass of a kernel spectrum, complex result kept: KhatC[m][c T + u] = scale X[bin0(u) + T c]
template <int NR>
__global__ void __launch_bounds__(NR / 8)
khat_cols_cplx_kernel(const cplx *__restrict__ WK, cplx *__restrict__ KhatC, const cplx *__restrict__ tw, const double scale)
{
    constexpr int L = 2 * NR;
    typedef Plan<L, COL> P;
    constexpr int T = P::T;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *line = reinterpret_cast<cplx *>(smem_raw);
    const int u = threadIdx.x;
    const int m = blockIdx.x;
    const cplx *col = WK + (long)m * L;
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) v[jj] = col[u + T * jj];
    Bases<L, COL> bases;
    bases.load(tw, u, false);
    fwd_a<L, COL>(v, line, bases, u);
    if constexpr (P::NPASS == 3) {
        __syncthreads();
        fwd_b<L, COL>(line, bases, u);
    }
    __syncthreads();
    fwd_c_col<L>(v, line, u);
    cplx *kh = KhatC + (long)m * L;
#pragma unroll
    for (int k = 0; k < 16; ++k) kh[u + T * k] = make_double2(scale * v[k].x, scale * v[k].y);
}

// a3 + a4 (r part) with a complex spectrum: dst column = crop(IFFT(KhatC . FFT(pad(src column)))).
template <int NR>
__global__ void __launch_bounds__(ColShape<NR>::THREADS, ColShape<NR>::MIN_CTAS)
cols_cplx_kernel(const cplx *__restrict__ Wsrc, cplx *__restrict__ Wdst, const cplx *__restrict__ KhatC,
                 const cplx *__restrict__ tw, const int n_modes, const long w_field_stride)
{
    typedef ColShape<NR> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    const int tid = threadIdx.x;
    const int u = tid % T, ml = tid / T;
    const int m_raw = blockIdx.x * S::MODES + ml;
    const bool live = m_raw < n_modes;
    const int mode = live ? m_raw : n_modes - 1;
    cplx *line = smem + ml * S::STRIDE;
    const cplx *src = Wsrc + blockIdx.y * w_field_stride + (long)mode * NR;
    cplx *dst = Wdst + blockIdx.y * w_field_stride + (long)mode * NR;
    const cplx *kh = KhatC + (long)mode * L;
    pdl_wait();
    pdl_launch_dependents();
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) v[jj] = src[u + T * jj];
    Bases<L, COL> bases;
    bases.load(tw, u, false);
    const Sync<T, S::THREADS> sync(ml + 1);
    fwd_a_compute_zero_upper<L, COL>(v, bases, u);
    fwd_a_store<L, COL>(v, line, u);
    sync();
    if constexpr (P::NPASS == 3) {
        fwd_b<L, COL>(line, bases, u);
        sync();
    }
    fwd_c_col<L>(v, line, u);
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = cmul(v[k], __ldg(&kh[u + T * k]));
    inv_c_col<L>(v, line, u);
    if constexpr (P::NPASS == 3) {
        sync();
        inv_b<L, COL>(line, bases, u);
    }
    sync();
    inv_a_load<L, COL>(v, line, u);
    inv_a_compute_lower_half<L, COL>(v, bases, u);
    if (live) {
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) dst[u + T * jj] = v[jj];
    }
}

}  // namespace pgk
