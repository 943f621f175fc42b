// kernels.cuh -- the sm_100a kernels of the FFT-convolution path (rows a1-a5 of DESIGN.md).
//
// Data layout in HBM (all fp64 / complex128), H = n_phi/2:
//   Sigma, Phi : [B][n_r][n_phi]          phi fastest (user arrays)
//   Z          : [B][H][n_r]   complex    TRANSPOSED packed spectrum.  Row i of Sigma (times r_i^{3/2})
//                                         is packed as z[n] = s[2n] + i s[2n+1] and transformed with a
//                                         complex FFT of length H; Z[k][i] is bin k of row i, so that
//                                         column k is contiguous in r.  The Hermitian half-spectrum of
//                                         the real row (modes 0..H) is an elementwise function of the
//                                         column pair (k, H-k); it is formed inside the column kernel.
//   Khat       : [H+1][2][n_r] real       spectrum of the Green's kernel for azimuthal mode m, split into
//                                         the even (2k) and odd (2k+1) bins of the 2 n_r-point padded
//                                         radial transform; all normalisations folded in
//   root_row   : [H]      exp(-2 pi i b / H)            root_col : [2 n_r]  exp(-2 pi i b / (2 n_r))
//   cphi       : [H+1]    i exp(-2 pi i m / n_phi)      (long double on the host)
#pragma once
#include "fft.cuh"

namespace pgk {

// ---------------------------------------------------------------- shapes
// rows per CTA in the phi passes: Z is written/read in runs of ROWS*16 bytes
__host__ __device__ constexpr int rows_per_cta(int nphi)
{
    const int T = nphi / 32;
    const int r = 256 / (T > 0 ? T : 1);
    return r < 4 ? 4 : (r > 16 ? 16 : r);
}
// column pairs (k, H-k) per CTA in the r pass
__host__ __device__ constexpr int pairs_per_cta(int nr)
{
    const int T = nr / 16;
    const int c = 64 / T;
    return c < 1 ? 1 : (c > 8 ? 8 : c);
}
// Shared-memory slots between the lines of two rows of a CTA.  In the row-fastest pass a
// quarter-warp touches (8 rows) or (4 rows x 2 neighbouring 17-slot blocks): STRIDE = 1 (mod 8)
// resp. 2 (mod 8) spreads them over the eight 16-byte bank groups.
template <int NPHI>
struct RowShape {
    static constexpr int L = NPHI / 2;
    static constexpr int T = L / 16;
    static constexpr int ROWS = rows_per_cta(NPHI);
    static constexpr int SKEW = (ROWS >= 8) ? 1 : (8 / ROWS);
    static constexpr int STRIDE = ((pad_idx(L) + 1 + 7) / 8) * 8 + SKEW;   // slots per row line
    static constexpr int THREADS = ROWS * T;
    static constexpr size_t SMEM = (size_t)ROWS * STRIDE * sizeof(cplx);
    static constexpr int MIN_CTAS = (THREADS <= 256) ? 2 : 1;
};
template <int NR>
struct ColShape {
    static constexpr int L = NR;
    static constexpr int T = L / 16;
    static constexpr int PAIRS = pairs_per_cta(NR);
    static constexpr int GROUPS = 4 * PAIRS;                // (pair, column of the pair, branch)
    static constexpr int STRIDE = Plan<L>::LINE;
    static constexpr int THREADS = GROUPS * T;
    static constexpr size_t SMEM = (size_t)GROUPS * STRIDE * sizeof(cplx);
    static constexpr int MIN_CTAS = (THREADS <= 256) ? 2 : 1;   // cap registers at 128/thread
};

__device__ __forceinline__ void prefetch_l1(const void *p)
{
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
}
// Coherent loads: unlike ld.global.nc they cannot be hoisted across a barrier by ptxas, which
// keeps them (and the registers they occupy) where they are written.
__device__ __forceinline__ double ld_f64(const double *p)
{
    double r;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ cplx ld_c128(const cplx *p)
{
    cplx r;
    asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

// ---------------------------------------------------------------- a2: rows forward
// One CTA transforms ROWS consecutive rows.  Row i: s = Sigma_i * scale_i (scale = r_i^{3/2}, or 1
// when rscale == nullptr), packed as z[n] = s[2n] + i s[2n+1], complex FFT of length H = n_phi/2.
// All passes but the last run with thread = (row, u) and u fastest (coalesced row loads); the last
// radix-16 pass runs with thread = (u', row) and the ROW fastest, so that its outputs Z[u' + T k][i]
// leave as runs of ROWS consecutive rows of one column: the transposed store costs no extra
// shared-memory round trip.
template <int NPHI>
__global__ void __launch_bounds__(RowShape<NPHI>::THREADS, RowShape<NPHI>::MIN_CTAS)
rows_fwd_kernel(const double *__restrict__ sigma, cplx *__restrict__ Z, const cplx *__restrict__ root,
                const double *__restrict__ rscale, const int n_rows, const long sigma_field_stride,
                const long z_field_stride)
{
    typedef RowShape<NPHI> S;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int i0 = blockIdx.x * ROWS;
    const int i = i0 + rho;

    Twid<L> tw;
    tw.load(root, 1, u);
    const cplx *x = reinterpret_cast<const cplx *>(sigma + blockIdx.y * sigma_field_stride + (long)i * NPHI);
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) v[jj] = x[u + T * jj];
    if (rscale != nullptr) {
        const double sc = __ldg(&rscale[i]);
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) { v[jj].x *= sc; v[jj].y *= sc; }
    }
    const Sync<T, S::THREADS> sync(rho);
    fwd_head<L>(v, smem + rho * S::STRIDE, tw, u, sync);
    __syncthreads();

    const int rp = tid % ROWS, up = tid / ROWS;
    fwd_last<L>(v, smem + rp * S::STRIDE, up);
    cplx *Zf = Z + blockIdx.y * z_field_stride + i0 + rp;
#pragma unroll
    for (int k = 0; k < 16; ++k) Zf[(long)(up + T * k) * n_rows] = v[k];
}

// ---------------------------------------------------------------- a4 (phi part): rows inverse
// Reads Z'[k][i] (already rebuilt by the column kernel so that the packed inverse transform gives
// the real row), first radix-16 pass in the row-fastest mapping (coalesced transposed load), the
// remaining passes with u fastest, multiplies row i by oscale_i (= r_i^{-1/2}) and stores Phi_i.
template <int NPHI>
__global__ void __launch_bounds__(RowShape<NPHI>::THREADS, RowShape<NPHI>::MIN_CTAS)
rows_inv_kernel(const cplx *__restrict__ Z, double *__restrict__ phi, const cplx *__restrict__ root,
                const double *__restrict__ oscale, const int n_rows, const long z_field_stride,
                const long phi_field_stride)
{
    typedef RowShape<NPHI> S;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int i0 = blockIdx.x * ROWS;
    const int i = i0 + rho;
    const int rp = tid % ROWS, up = tid / ROWS;

    const cplx *Zf = Z + blockIdx.y * z_field_stride + i0 + rp;
    cplx v[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = Zf[(long)(up + T * k) * n_rows];
    Twid<L> tw;
    tw.load(root, 1, u);
    inv_first<L>(v, smem + rp * S::STRIDE, up);
    __syncthreads();

    const Sync<T, S::THREADS> sync(rho);
    inv_tail<L>(v, smem + rho * S::STRIDE, tw, u, sync, false);
    const double sc = __ldg(&oscale[i]);
    cplx *y = reinterpret_cast<cplx *>(phi + blockIdx.y * phi_field_stride + (long)i * NPHI);
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) y[u + T * jj] = make_double2(v[jj].x * sc, v[jj].y * sc);
}

// ---------------------------------------------------------------- a3 + a4 (r part): columns
// One CTA owns PAIRS column pairs (k, H-k), k = 0..H/2.  For a pair, with A = Z[k][n], B = Z[H-k][n]
// and c = i exp(-2 pi i k / n_phi), the two azimuthal modes of the real row transform are
//     2 X_k     = (1 - c) A + (1 + c) conj(B)            mode k      ("a" column)
//     2 X_{H-k} = conj( (1 + c) A + (1 - c) conj(B) )    mode H - k  ("b" column)
// (k = 0 pairs column 0 with itself and yields modes 0 and H, the Nyquist mode; k = H/2 yields the
// same mode twice and the "b" result is dropped).  Each mode column x[0..n_r) is convolved with the
// Green's kernel over the radial lags, zero-padded to 2 n_r, and cropped back to n_r:
//   y[n] = (1/2N) sum_{k'<2N} Khat[k'] Xpad[k'] e^{+2 pi i k' n / 2N},   n < N = n_r.
// The padded 2N-point transform with a zero upper half and a cropped output is exactly two N-point
// problems (decimation in frequency forward / in time backward):
//   even bins: FFT_N(x)             * Khat[2k]    -> IFFT_N -> e[n]
//   odd  bins: FFT_N(x[n] mod[n])   * Khat[2k+1]  -> IFFT_N -> o[n],   mod[n] = exp(-i pi n / N)
//   y[n] = e[n] + conj(mod[n]) o[n]                (1/2N folded into Khat)
// so the padded array and the discarded half are never formed (a3: multiply fused into the last
// forward pass; a4: inverse with fused crop).  The four (column, branch) transforms of a pair run on
// four thread groups with their own named barriers; they meet once, at the end, where the packed
// spectrum of the inverse row transform is rebuilt IN PLACE:
//     Z'[k]   = conj(1 - c) Y_k     + conj(1 + c) conj(Y_{H-k})
//     Z'[H-k] =     (1 - c) Y_{H-k} +     (1 + c) conj(Y_k)
template <int Q, int L, int T, int STRIDE>
__device__ __forceinline__ void cols_combine(const cplx (&v)[16], const cplx *__restrict__ pair_lines, const int u,
                                             const cplx alpha, const cplx beta, cplx *__restrict__ za,
                                             cplx *__restrict__ zb, const bool store_a, const bool store_b)
{
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        constexpr int dummy = 0;
        (void)dummy;
        const int jj = 4 * Q + d;
        const int n = u + T * jj;
        cplx c[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) c[q] = (q == Q) ? v[4 * Q + d] : pair_lines[q * STRIDE + n];
        const cplx ya = cadd(c[0], c[1]);   // column a: branch 0 + branch 1
        const cplx yb = cadd(c[2], c[3]);   // column b
        if (store_a) {
            cplx r = cmulc(ya, alpha);                       // conj(alpha) Y_a
            r = cfmac(beta, cconj(yb), r);                   // + conj(beta) conj(Y_b)
            za[n] = r;
        }
        if (store_b) {
            cplx r = cmul(yb, alpha);                        // alpha Y_b
            r = cfmac(ya, beta, r);                          // + beta conj(Y_a)
            zb[n] = r;
        }
    }
}

template <int NR>
__global__ void __launch_bounds__(ColShape<NR>::THREADS, ColShape<NR>::MIN_CTAS)
cols_kernel(cplx *__restrict__ Z, const double *__restrict__ Khat, const cplx *__restrict__ root2,
            const cplx *__restrict__ cphi, const int half, const long z_field_stride)
{
    typedef ColShape<NR> S;
    constexpr int L = S::L, T = S::T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, g = tid / T;
    const int q = g & 3, br = g & 1, cb = (g >> 1) & 1, pl = g >> 2;
    const int p_raw = blockIdx.x * S::PAIRS + pl;
    const bool live = p_raw <= half / 2;
    const int p = live ? p_raw : half / 2;
    const int ka = p, kb = (half - p) % half;        // Z columns of the pair
    const int mode = cb ? half - p : p;              // azimuthal mode of this group's column
    cplx *line = smem + g * S::STRIDE;
    cplx *zf = Z + blockIdx.y * z_field_stride;
    const double *kh = Khat + ((long)mode * 2 + br) * L;

    // pull this group's slice of Khat into L1 while the forward transform runs
#pragma unroll
    for (int k = 0; k < 16; ++k) prefetch_l1(kh + u + T * k);

    Twid<L> tw;
    tw.load(root2, 2, u);
    const cplx c = __ldg(&cphi[p]);
    const cplx alpha0 = make_double2(1.0 - c.x, -c.y), beta0 = make_double2(1.0 + c.x, c.y);
    // this group's column: X = al P + be conj(Q)
    const cplx al = cb ? cconj(alpha0) : alpha0, be = cb ? cconj(beta0) : beta0;
    const cplx *P = zf + (long)(cb ? kb : ka) * L, *Qc = zf + (long)(cb ? ka : kb) * L;

    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const cplx a = P[u + T * jj], b = Qc[u + T * jj];
        v[jj] = cfmac(b, be, cmul(a, al));
    }
    if (br) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) v[jj] = cmul(v[jj], __ldg(&root2[u + T * jj]));
    }
    const Sync<T, S::THREADS> sync(g);
    fwd_head<L>(v, line, tw, u, sync);
    if constexpr (Plan<L>::HAS_EXCHANGE) sync();
    double kv[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) kv[k] = ld_f64(kh + u + T * k);
    fwd_last<L>(v, line, u);
#pragma unroll
    for (int k = 0; k < 16; ++k) { v[k].x *= kv[k]; v[k].y *= kv[k]; }
    // inv_first writes exactly the 16 slots this thread has just read: no barrier in between
    inv_first<L>(v, line, u);
    if constexpr (Plan<L>::HAS_EXCHANGE) sync();
    inv_tail<L>(v, line, tw, u, sync, true);
    if (br) {
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) v[jj] = cmulc(v[jj], __ldg(&root2[u + T * jj]));
    }
    // hand the twelve results other groups will finish to them (slot n = u + T jj of this group's line)
#pragma unroll
    for (int jj = 0; jj < 16; ++jj)
        if ((jj >> 2) != q) line[u + T * jj] = v[jj];
    __syncthreads();

    const cplx *pair_lines = smem + (pl * 4) * S::STRIDE;
    cplx *za = zf + (long)ka * L, *zb = zf + (long)kb * L;
    const bool store_a = live, store_b = live && (ka != kb);
    switch (q) {
        case 0: cols_combine<0, L, T, S::STRIDE>(v, pair_lines, u, alpha0, beta0, za, zb, store_a, store_b); break;
        case 1: cols_combine<1, L, T, S::STRIDE>(v, pair_lines, u, alpha0, beta0, za, zb, store_a, store_b); break;
        case 2: cols_combine<2, L, T, S::STRIDE>(v, pair_lines, u, alpha0, beta0, za, zb, store_a, store_b); break;
        default: cols_combine<3, L, T, S::STRIDE>(v, pair_lines, u, alpha0, beta0, za, zb, store_a, store_b); break;
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

// Column pass of the kernel spectrum (one-time, a1).  ZK[k][0..2N) is the packed row transform of the
// padded kernel Kpad (2N rows).  For azimuthal mode m = 0..H the mode column is rebuilt from the
// column pair (m mod H, (H - m) mod H) exactly as in cols_kernel, then its full 2N-point forward
// transform is taken, split into even / odd bins exactly as cols_kernel consumes them; the real
// part is scaled and stored:  Khat[m][0][k] = scale Re X[2k],  Khat[m][1][k] = scale Re X[2k+1].
// (K is even in both lags, so X is real up to rounding.)
template <int NR>
__global__ void __launch_bounds__(2 * (NR / 16))
khat_cols_kernel(const cplx *__restrict__ ZK, double *__restrict__ Khat, const cplx *__restrict__ root2,
                 const cplx *__restrict__ cphi, const double scale, const int half)
{
    constexpr int L = NR, T = L / 16, STRIDE = Plan<L>::LINE;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, br = tid / T;
    const int m = blockIdx.x;                         // mode 0..H
    const int ka = m % half, kb = (half - m) % half;
    const cplx c = __ldg(&cphi[m]);
    const cplx al = make_double2(1.0 - c.x, -c.y), be = make_double2(1.0 + c.x, c.y);
    const cplx *P = ZK + (long)ka * (2 * L), *Q = ZK + (long)kb * (2 * L);

    Twid<L> tw;
    tw.load(root2, 2, u);
    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 16; ++jj) {
        const int n = u + T * jj;
        const cplx x1 = cfmac(Q[n], be, cmul(P[n], al));
        const cplx x2 = cfmac(Q[n + L], be, cmul(P[n + L], al));
        v[jj] = br ? cmul(csub(x1, x2), __ldg(&root2[n])) : cadd(x1, x2);
    }
    const Sync<T, 2 * T> sync(br);
    fft_fwd<L>(v, smem + br * STRIDE, tw, u, sync, false);
    double *kh = Khat + ((long)m * 2 + br) * L;
#pragma unroll
    for (int k = 0; k < 16; ++k) kh[u + T * k] = scale * v[k].x;
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
