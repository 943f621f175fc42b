// kernels.cuh -- the sm_100a kernels of the FFT-convolution path (rows a1-a5 of DESIGN.md).
//
// Data layout in HBM (all fp64 / complex128):
//   Sigma, Phi : [B][n_r][n_phi]           phi fastest (user arrays)
//   W          : [B][Mc][n_r]  complex     TRANSPOSED half-spectrum: column m (azimuthal mode,
//                                          m = 0..n_phi/2, padded to Mc) is contiguous in r
//   Khat       : [Mc][2][n_r]  real        spectrum of the Green's kernel for mode m, split into
//                                          the even (2k) and odd (2k+1) bins of the 2 n_r-point
//                                          padded radial transform
#pragma once
#include "fft.cuh"

namespace pgk {

// ---------------------------------------------------------------- shapes
// rows per CTA in the phi passes: W is written/read in runs of ROWS*16 bytes
__host__ __device__ constexpr int rows_per_cta(int nphi)
{
    const int T = nphi / 32;
    const int r = 256 / (T > 0 ? T : 1);
    return r < 4 ? 4 : (r > 16 ? 16 : r);
}
// azimuthal modes (columns) per CTA in the r pass
__host__ __device__ constexpr int cols_per_cta(int nr)
{
    const int T = nr / 16;
    const int c = 128 / T;
    return c < 1 ? 1 : (c > 8 ? 8 : c);
}
// shared-memory slots between the lines of two rows of a CTA: offset them so that the
// (row, mode) quarter-warps of the transposed store hit distinct 16-byte bank groups
template <int NPHI>
struct RowShape {
    static constexpr int L = NPHI / 2;
    static constexpr int T = L / 16;
    static constexpr int ROWS = rows_per_cta(NPHI);
    static constexpr int SKEW = (ROWS >= 8) ? 1 : (8 / ROWS);
    static constexpr int STRIDE = ((pad_idx(L) + 1 + 7) / 8) * 8 + SKEW;   // slots per row line
    static constexpr int THREADS = ROWS * T;
    static constexpr size_t SMEM = (size_t)ROWS * STRIDE * sizeof(cplx);
};
template <int NR>
struct ColShape {
    static constexpr int L = NR;
    static constexpr int T = L / 16;
    static constexpr int C = cols_per_cta(NR);
    static constexpr int GROUPS = 2 * C;                    // (column, branch) transforms per CTA
    static constexpr int STRIDE = Plan<L>::LINE;
    static constexpr int THREADS = GROUPS * T;
    static constexpr size_t SMEM = (size_t)GROUPS * STRIDE * sizeof(cplx);
    static constexpr int MIN_CTAS = (THREADS <= 256) ? 2 : 1;   // cap registers at 128/thread
};

__device__ __forceinline__ void prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// ---------------------------------------------------------------- a2: rows forward
// One CTA transforms ROWS consecutive rows.  Row i: s = Sigma_i * scale_i (scale = r_i^{3/2}, or 1
// when rscale == nullptr), packed as z[n] = s[2n] + i s[2n+1], complex FFT of length L = n_phi/2,
// then the real-FFT split X[k] = (Z[k] + conj Z[L-k])/2 - (i/2) w^k (Z[k] - conj Z[L-k]),
// w = exp(-2 pi i / n_phi), written TRANSPOSED: W[k][i] for k = 0..L (k = L is the Nyquist mode).
//   rtw[k] = -(i/2) w^k.
template <int NPHI>
__global__ void __launch_bounds__(RowShape<NPHI>::THREADS)
rows_fwd_kernel(const double *__restrict__ sigma, cplx *__restrict__ W, const cplx *__restrict__ tw,
                const cplx *__restrict__ rtw, const double *__restrict__ rscale, const int n_rows,
                const long sigma_field_stride, const long w_field_stride)
{
    typedef RowShape<NPHI> S;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int i0 = blockIdx.x * ROWS;
    const int i = i0 + rho;
    cplx *line = smem + rho * S::STRIDE;

    const cplx *x = reinterpret_cast<const cplx *>(sigma + blockIdx.y * sigma_field_stride + (long)i * NPHI);
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) v[jj] = x[u + T * jj];
    if (rscale != nullptr) {
        const double sc = __ldg(&rscale[i]);
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) { v[jj].x *= sc; v[jj].y *= sc; }
    }
    fft_fwd<L>(v, line, tw, u);
#pragma unroll
    for (int k = 0; k < 16; ++k) line[pad_idx(u + T * k)] = v[k];
    __syncthreads();

    cplx *Wf = W + blockIdx.y * w_field_stride;
#pragma unroll 4
    for (int w = tid; w < L * ROWS; w += S::THREADS) {
        const int k = w / ROWS, r2 = w % ROWS;
        const cplx *ln = smem + r2 * S::STRIDE;
        const cplx zk = ln[pad_idx(k)];
        const cplx zm = ln[pad_idx((L - k) & (L - 1))];
        const cplx a = make_double2(zk.x + zm.x, zk.y - zm.y);   // Z[k] + conj Z[L-k]
        const cplx b = make_double2(zk.x - zm.x, zk.y + zm.y);   // Z[k] - conj Z[L-k]
        const cplx t = __ldg(&rtw[k]);
        cplx X;
        X.x = fma(0.5, a.x, fma(-b.y, t.y, b.x * t.x));
        X.y = fma(0.5, a.y, fma(b.y, t.x, b.x * t.y));
        Wf[(long)k * n_rows + i0 + r2] = X;
        if (k == 0) Wf[(long)L * n_rows + i0 + r2] = make_double2(zk.x - zk.y, 0.0);
    }
}

// ---------------------------------------------------------------- a4 (phi part): rows inverse
// Reads W[k][i] (k = 0..L), rebuilds Z'[k] = (X[k] + conj X[L-k]) + i w^{-k} (X[k] - conj X[L-k])
// (= 2 Z[k]; the 1/2 and the FFT normalisation live in Khat), inverse complex FFT, multiplies row i
// by oscale_i (= r_i^{-1/2}) and stores Phi_i.   itw[k] = i w^{-k}.
template <int NPHI>
__global__ void __launch_bounds__(RowShape<NPHI>::THREADS)
rows_inv_kernel(const cplx *__restrict__ W, double *__restrict__ phi, const cplx *__restrict__ tw,
                const cplx *__restrict__ itw, const double *__restrict__ oscale, const int n_rows,
                const long w_field_stride, const long phi_field_stride)
{
    typedef RowShape<NPHI> S;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int i0 = blockIdx.x * ROWS;
    const int i = i0 + rho;
    cplx *line = smem + rho * S::STRIDE;

    const cplx *Wf = W + blockIdx.y * w_field_stride;
#pragma unroll 4
    for (int w = tid; w < (L + 1) * ROWS; w += S::THREADS) {
        const int k = w / ROWS, r2 = w % ROWS;
        smem[r2 * S::STRIDE + pad_idx(k)] = Wf[(long)k * n_rows + i0 + r2];
    }
    __syncthreads();

    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int k = u + T * jj;
        const cplx xk = line[pad_idx(k)];
        const cplx xm = line[pad_idx(L - k)];
        const cplx a = make_double2(xk.x + xm.x, xk.y - xm.y);
        const cplx b = make_double2(xk.x - xm.x, xk.y + xm.y);
        const cplx t = __ldg(&itw[k]);
        v[jj].x = a.x + fma(-b.y, t.y, b.x * t.x);
        v[jj].y = a.y + fma(b.y, t.x, b.x * t.y);
    }
    __syncthreads();
    fft_inv<L>(v, line, tw, u);

    const double sc = __ldg(&oscale[i]);
    cplx *y = reinterpret_cast<cplx *>(phi + blockIdx.y * phi_field_stride + (long)i * NPHI);
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) y[u + T * jj] = make_double2(v[jj].x * sc, v[jj].y * sc);
}

// ---------------------------------------------------------------- a3 + a4 (r part): columns
// One CTA owns C azimuthal modes.  For mode m the column x[0..n_r) = W[m][:] is convolved with the
// Green's kernel over the radial lags, zero-padded to 2 n_r, and cropped back to n_r, IN PLACE:
//   y[n] = (1/2N) sum_{k'<2N} Khat[k'] Xpad[k'] e^{+2 pi i k' n / 2N},   n < N = n_r.
// The padded 2N-point transform with a zero upper half and a cropped output is exactly two N-point
// problems (decimation in frequency forward / in time backward):
//   even bins: FFT_N(x)             * Khat[2k]    -> IFFT_N -> e[n]
//   odd  bins: FFT_N(x[n] mod[n])   * Khat[2k+1]  -> IFFT_N -> o[n],   mod[n] = exp(-i pi n / N)
//   y[n] = e[n] + conj(mod[n]) o[n]                (1/2N folded into Khat)
// so the padded array and the discarded half are never formed (a3: multiply fused into the last
// forward pass; a4: inverse with fused crop).  The two branches run on separate thread groups.
template <int NR>
__global__ void __launch_bounds__(ColShape<NR>::THREADS, ColShape<NR>::MIN_CTAS)
cols_kernel(cplx *__restrict__ W, const double *__restrict__ Khat, const cplx *__restrict__ tw,
            const cplx *__restrict__ mod, const long w_field_stride)
{
    typedef ColShape<NR> S;
    constexpr int L = S::L, T = S::T, C = S::C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, g = tid / T;
    const int br = g & 1, c = g >> 1;
    const int m = blockIdx.x * C + c;
    cplx *line = smem + g * S::STRIDE;
    cplx *col = W + blockIdx.y * w_field_stride + (long)m * L;
    const double *kh = Khat + ((long)m * 2 + br) * L;

    // pull this thread group's slice of Khat towards the SM while the forward transform runs
    // (T threads cover the 8*L bytes of one (mode, branch) line in 128-byte steps)
    for (int off = u * 16; off < L; off += T * 16) prefetch_l2(kh + off);

    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) v[jj] = col[u + T * jj];
    if (br) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) v[jj] = cmul(v[jj], __ldg(&mod[u + T * jj]));
    }
    fft_fwd<L>(v, line, tw, u);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const double kv = __ldg(&kh[u + T * k]);
        v[k].x *= kv;
        v[k].y *= kv;
    }
    fft_inv<L>(v, line, tw, u);
    if (br) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj)
            line[pad_idx(u + T * jj)] = cmulc(v[jj], __ldg(&mod[u + T * jj]));
    }
    __syncthreads();
    if (!br) {
        const cplx *other = line + S::STRIDE;
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) col[u + T * jj] = cadd(v[jj], other[pad_idx(u + T * jj)]);
    }
}

// ---------------------------------------------------------------- a1: Green's kernel
// Kpad[k][l], k in [0, 2 n_r), l in [0, n_phi):  lag = k (k < n_r), k - 2 n_r (k > n_r), slot n_r = 0.
//   K(lag, l) = [4 sinh^2(lag du / 2) + 4 sin^2(pi l / n_phi) + eta2]^(-1/2)
__global__ void green_fill_kernel(double *__restrict__ Kpad, const int n_r, const int n_phi, const double du,
                                  const double eta2)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long total = 2L * n_r * n_phi;
    if (idx >= total) return;
    const int k = (int)(idx / n_phi), l = (int)(idx % n_phi);
    double val = 0.0;
    if (k != n_r) {
        const int lag = k < n_r ? k : k - 2 * n_r;
        const double sh = sinh(0.5 * du * (double)lag);
        const double sn = sinpi((double)l / (double)n_phi);
        val = rsqrt(4.0 * sh * sh + 4.0 * sn * sn + eta2);
    }
    Kpad[idx] = val;
}

// Column pass of the kernel spectrum: the full 2N-point forward transform of column m of the
// row-transformed Kpad (Wk[m][0..2N)), split into even / odd bins exactly as cols_kernel consumes
// them, real part scaled and stored:  Khat[m][0][k] = scale Re X[2k],  Khat[m][1][k] = scale Re X[2k+1].
// (K is even in both lags, so X is real up to rounding.)
template <int NR>
__global__ void __launch_bounds__(ColShape<NR>::THREADS)
khat_cols_kernel(const cplx *__restrict__ Wk, double *__restrict__ Khat, const cplx *__restrict__ tw,
                 const cplx *__restrict__ mod, const double scale, const int n_cols)
{
    typedef ColShape<NR> S;
    constexpr int L = S::L, T = S::T, C = S::C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, g = tid / T;
    const int br = g & 1, c = g >> 1;
    const int m = blockIdx.x * C + c;
    const bool live = m < n_cols;
    cplx *line = smem + g * S::STRIDE;
    const cplx *col = Wk + (long)(live ? m : 0) * (2 * L);

    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int n = u + T * jj;
        const cplx a = col[n], b = col[n + L];
        v[jj] = br ? cmul(csub(a, b), __ldg(&mod[n])) : cadd(a, b);
    }
    fft_fwd<L>(v, line, tw, u);
    double *kh = Khat + ((long)m * 2 + br) * L;
#pragma unroll
    for (int k = 0; k < 16; ++k) kh[u + T * k] = live ? scale * v[k].x : 0.0;
}

// ---------------------------------------------------------------- a5: direct summation
// Tiled all-pairs sum from the coordinates, one CTA per target ring i (grid.x) and field (grid.y):
//   Phi_ij = - sum_{i'} dA_{i'} sum_{j'} Sigma_{i'j'} / sqrt((r_i - r_i')^2 + 4 r_i r_i' s2[(j-j') mod n_phi]
//                                                          + eps^2 h_i h_i'),   s2[l] = sin^2(pi l / n_phi)
// Source ring i' is staged in shared memory together with the n_phi pair-kernel values of the ring
// pair; each thread accumulates TPT targets in two levels (within the ring, then over rings).
template <int TPT>
__global__ void __launch_bounds__(256)
direct_kernel(const double *__restrict__ sigma, double *__restrict__ phi, const double *__restrict__ r,
              const double *__restrict__ dA, const double *__restrict__ s2, const int n_r, const int n_phi,
              const double eps2, const int ring0, const long sigma_field_stride, const long phi_field_stride)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *w = reinterpret_cast<double *>(smem_raw);   // [n_phi] Sigma of the source ring
    double *g = w + n_phi;                              // [n_phi] pair kernel by azimuthal lag
    const int i = ring0 + blockIdx.x;
    const double ri = r[i], hi = sqrt(dA[i]);
    const double *sg = sigma + blockIdx.y * sigma_field_stride;
    const int mask = n_phi - 1;
    const int nt = blockDim.x;

    double acc[TPT];
#pragma unroll
    for (int q = 0; q < TPT; ++q) acc[q] = 0.0;

    for (int ip = 0; ip < n_r; ++ip) {
        const double rp = r[ip], ap = dA[ip];
        const double dr = ri - rp;
        const double base = fma(dr, dr, eps2 * hi * sqrt(ap));
        const double rr4 = 4.0 * ri * rp;
        __syncthreads();
        for (int l = threadIdx.x; l < n_phi; l += nt) {
            w[l] = sg[(long)ip * n_phi + l];
            g[l] = rsqrt(fma(rr4, s2[l], base));
        }
        __syncthreads();
        double ring[TPT];
#pragma unroll
        for (int q = 0; q < TPT; ++q) ring[q] = 0.0;
        for (int jp = 0; jp < n_phi; ++jp) {
            const double wv = w[jp];
#pragma unroll
            for (int q = 0; q < TPT; ++q) {
                const int j = threadIdx.x + q * nt;
                ring[q] = fma(wv, g[(j - jp) & mask], ring[q]);
            }
        }
#pragma unroll
        for (int q = 0; q < TPT; ++q) acc[q] = fma(ap, ring[q], acc[q]);
    }
    double *out = phi + blockIdx.y * phi_field_stride + (long)blockIdx.x * n_phi;
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
        const int j = threadIdx.x + q * nt;
        if (j < n_phi) out[j] = -acc[q];
    }
}

}  // namespace pgk
