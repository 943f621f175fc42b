// fft.cuh -- in-register / shared-memory complex128 FFT building block for sm_100a.
//
// A length-L transform (L = R1 * 16^n16, R1 in {1,2,4,8}, n16 in {1,2}) is carried by T = L/16
// threads holding 16 elements each.  Every pass is a radix-R DFT done entirely in registers;
// between passes the T threads exchange data through a padded shared-memory line
// (pad_idx: one spare slot every 16 keeps the stride-16 reads of the last pass conflict-free
// for 16-byte accesses, which the hardware serves a quarter-warp at a time).
//
// Element distribution: thread u holds indices u + T*jj (jj = 0..15) on input AND on output,
// for both directions, so global loads/stores are coalesced and the forward spectrum can be
// consumed by the inverse transform without any reordering (PAPER.md:19 names "FFT
// operations" as the GPU-resident work; the decomposition is ours).
//
// Twiddle tables are read-only global arrays built on the host in long double:
//   tw0[k1*(L/R1) + b]  = exp(-2 pi i b k1 / L),        k1 in [0,R1), b in [0,L/R1)   (if R1 > 1)
//   tw1[k*T3 + t]       = exp(-2 pi i t k / (L/R1)),    k in [0,16),  t in [0,T3=L/(16 R1)) (if n16 == 2)
// laid out as [tw0 | tw1].
#pragma once
#include <cuda_runtime.h>

namespace pgk {

typedef double2 cplx;

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
// a * w
__device__ __forceinline__ cplx cmul(cplx a, cplx w)
{
    return make_double2(fma(-a.y, w.y, a.x * w.x), fma(a.y, w.x, a.x * w.y));
}
// a * conj(w)
__device__ __forceinline__ cplx cmulc(cplx a, cplx w)
{
    return make_double2(fma(a.y, w.y, a.x * w.x), fma(a.y, w.x, -(a.x * w.y)));
}

// Table load.  Deliberately a plain (coherent) ld.global, not ld.global.nc / __ldg: ptxas hoists
// non-coherent loads across bar.sync all the way to the kernel entry, which put every twiddle of
// every pass in flight at once and spilled them (measured: 300-680 bytes of spills at 128
// registers).  A coherent load cannot cross a barrier, so each pass loads its own twiddles while
// the previous butterfly computes.  The tables stay L1/L2 resident either way.
__device__ __forceinline__ cplx ld_table(const cplx *p)
{
    cplx r;
    asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

__host__ __device__ constexpr int pad_idx(int a) { return a + (a >> 4); }

// ------------------------------------------------------------------ compile-time twiddles
// cos / sin of 2 pi n / 16, n = 0..7
__host__ __device__ constexpr double cos16(int n)
{
    return n == 0 ? 1.0
         : n == 1 ? 0.92387953251128673848
         : n == 2 ? 0.70710678118654752440
         : n == 3 ? 0.38268343236508977173
         : n == 4 ? 0.0
         : n == 5 ? -0.38268343236508977173
         : n == 6 ? -0.70710678118654752440
         :          -0.92387953251128673848;
}
__host__ __device__ constexpr double sin16(int n)
{
    return n == 0 ? 0.0
         : n == 1 ? 0.38268343236508977173
         : n == 2 ? 0.70710678118654752440
         : n == 3 ? 0.92387953251128673848
         : n == 4 ? 1.0
         : n == 5 ? 0.92387953251128673848
         : n == 6 ? 0.70710678118654752440
         :          0.38268343236508977173;
}

// z * exp(-/+ 2 pi i J / N)   (- forward, + inverse), 0 <= J < N/2, N in {2,4,8,16}
template <int J, int N, bool INV>
__device__ __forceinline__ cplx mulw(cplx z)
{
    constexpr int n16 = J * (16 / N);
    if constexpr (n16 == 0) {
        return z;
    } else if constexpr (n16 == 4) {
        return INV ? make_double2(-z.y, z.x) : make_double2(z.y, -z.x);
    } else {
        constexpr double c = cos16(n16);
        constexpr double s = INV ? sin16(n16) : -sin16(n16);   // w = c + i s
        return make_double2(fma(-z.y, s, z.x * c), fma(z.y, c, z.x * s));
    }
}

// ------------------------------------------------------------------ radix-N DFT in registers
// In-place decimation-in-frequency on x[0..N): output X[k] lands at slot bitrev(k).
template <int N, bool INV, int J = 0>
struct DifStage {
    static __device__ __forceinline__ void run(cplx *x)
    {
        if constexpr (J < N / 2) {
            const cplx a = x[J], b = x[J + N / 2];
            x[J] = cadd(a, b);
            x[J + N / 2] = mulw<J, N, INV>(csub(a, b));
            DifStage<N, INV, J + 1>::run(x);
        }
    }
};

template <int N, bool INV>
struct Dif {
    static __device__ __forceinline__ void run(cplx *x)
    {
        if constexpr (N >= 2) {
            DifStage<N, INV>::run(x);
            Dif<N / 2, INV>::run(x);
            Dif<N / 2, INV>::run(x + N / 2);
        }
    }
};

template <int N>
__host__ __device__ constexpr int bitrev(int k)
{
    int r = 0;
    for (int b = 1; b < N; b <<= 1) { r = (r << 1) | (k & 1); k >>= 1; }
    return r;
}

// natural order in -> natural order out
template <int N, bool INV>
__device__ __forceinline__ void dft(cplx (&x)[N])
{
    Dif<N, INV>::run(x);
    cplx y[N];
#pragma unroll
    for (int k = 0; k < N; ++k) y[k] = x[bitrev<N>(k)];
#pragma unroll
    for (int k = 0; k < N; ++k) x[k] = y[k];
}

// ------------------------------------------------------------------ plan
template <int L>
struct Plan {
    static_assert(L == 16 || L == 32 || L == 64 || L == 128 || L == 256 || L == 512 || L == 1024 ||
                      L == 2048,
                  "unsupported FFT length");
    static constexpr int T = L / 16;                         // threads per transform
    static constexpr int N16 = (L >= 256) ? 2 : 1;           // number of radix-16 passes
    static constexpr int R1 = L / (N16 == 2 ? 256 : 16);     // leading small radix (1 = absent)
    static constexpr int T2 = L / R1;                        // sub-length after the leading pass
    static constexpr int T3 = T2 / 16;                       // sub-length after the first radix-16 pass
    static constexpr int TW0 = (R1 > 1) ? L : 0;             // entries in tw0
    static constexpr int TW1 = (N16 == 2) ? T2 : 0;          // entries in tw1
    static constexpr int TW = TW0 + TW1;
    static constexpr int LINE = pad_idx(L) + 8;              // smem slots per transform (>= pad_idx(L)+1)
};

// CTA-wide barrier used between exchange phases.  All threads of the CTA must call the
// transforms together.
__device__ __forceinline__ void cta_sync() { __syncthreads(); }

// ------------------------------------------------------------------ shared-memory addressing
// Every exchange address is written as (per-thread base) + (compile-time constant), so that the
// forward and the inverse transform of one kernel share three base registers instead of keeping
// dozens of computed addresses alive (which spilled at 128 registers per thread).
//   pad_idx(a + c) = pad_idx(a) + c + c/16            when c is a multiple of 16
//   pad_idx(16 a + j) = 17 a + j                      for 0 <= j < 16
template <int L>
struct Lines {
    typedef Plan<L> P;
    cplx *lin;   // sm + pad_idx(u)            consecutive-lane side of the radix-16 exchanges
    cplx *blk;   // sm + 17 u                  16 consecutive slots of the last radix-16 pass
    cplx *mid;   // sm + pad_idx(q T2 + t)     strided side of the leading-pass exchange
    __device__ __forceinline__ Lines(cplx *sm, int u)
    {
        lin = sm + (P::N16 == 2 ? pad_idx(u) : u);
        blk = sm + 17 * u;
        mid = (P::N16 == 2) ? sm + (u / P::T3) * pad_idx(P::T2) + (u % P::T3) : blk;
    }
    // leading pass, element (k, b = u + T m):  pad_idx(k T2 + b)
    static __host__ __device__ constexpr int lead(int k, int m)
    {
        return (P::N16 == 2) ? k * pad_idx(P::T2) + pad_idx(P::T * m) : 17 * k + P::T * m;
    }
    // first radix-16 pass after a leading pass reads  pad_idx(q T2 + t + T3 j)
    static __host__ __device__ constexpr int midj(int j) { return (P::N16 == 2) ? 17 * j : j; }
    // exchange between the two radix-16 passes writes  pad_idx(u + T k)
    static __host__ __device__ constexpr int link(int k) { return pad_idx(P::T * k); }
};

// ------------------------------------------------------------------ forward transform
// v[jj] = x[u + T*jj]  ->  v[k] = X[u + T*k],  X[k] = sum_n x[n] exp(-2 pi i n k / L)
template <int L>
__device__ __forceinline__ void fft_fwd(cplx (&v)[16], cplx *__restrict__ sm, const cplx *__restrict__ tw,
                                        const int u)
{
    typedef Plan<L> P;
    typedef Lines<L> A;
    constexpr int T = P::T, R1 = P::R1, T2 = P::T2, T3 = P::T3;
    const A a(sm, u);
    if constexpr (R1 > 1) {
        constexpr int M = 16 / R1;   // butterflies per thread in the leading pass
#pragma unroll
        for (int m = 0; m < M; ++m) {
            cplx x[R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = v[m + M * j];
            dft<R1, false>(x);
            const cplx *twb = tw + u + T * m;
#pragma unroll
            for (int k = 1; k < R1; ++k) x[k] = cmul(x[k], ld_table(&twb[k * T2]));
#pragma unroll
            for (int k = 0; k < R1; ++k) a.lin[A::lead(k, m)] = x[k];
        }
        cta_sync();
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = a.mid[A::midj(j)];
        cta_sync();
    }
    dft<16, false>(v);
    if constexpr (P::N16 == 2) {
        const cplx *tw1 = tw + P::TW0 + (u % T3);
#pragma unroll
        for (int k = 1; k < 16; ++k) v[k] = cmul(v[k], ld_table(&tw1[k * T3]));
#pragma unroll
        for (int k = 0; k < 16; ++k) a.lin[A::link(k)] = v[k];
        cta_sync();
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = a.blk[j];
        cta_sync();
        dft<16, false>(v);
    }
}

// ------------------------------------------------------------------ inverse transform (unnormalised)
// v[k] = X[u + T*k]  ->  v[jj] = sum_k X[k] exp(+2 pi i n k / L),  n = u + T*jj
// Exact transpose of fft_fwd's flow graph, with conjugated twiddles.
template <int L>
__device__ __forceinline__ void fft_inv(cplx (&v)[16], cplx *__restrict__ sm, const cplx *__restrict__ tw,
                                        const int u)
{
    typedef Plan<L> P;
    typedef Lines<L> A;
    constexpr int T = P::T, R1 = P::R1, T2 = P::T2, T3 = P::T3;
    const A a(sm, u);
    if constexpr (P::N16 == 2) {
        dft<16, true>(v);
#pragma unroll
        for (int j = 0; j < 16; ++j) a.blk[j] = v[j];
        cta_sync();
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = a.lin[A::link(k)];
        cta_sync();
        const cplx *tw1 = tw + P::TW0 + (u % T3);
#pragma unroll
        for (int k = 1; k < 16; ++k) v[k] = cmulc(v[k], ld_table(&tw1[k * T3]));
    }
    dft<16, true>(v);
    if constexpr (R1 > 1) {
        constexpr int M = 16 / R1;
#pragma unroll
        for (int j = 0; j < 16; ++j) a.mid[A::midj(j)] = v[j];
        cta_sync();
#pragma unroll
        for (int m = 0; m < M; ++m) {
            cplx x[R1];
#pragma unroll
            for (int k = 0; k < R1; ++k) x[k] = a.lin[A::lead(k, m)];
            const cplx *twb = tw + u + T * m;
#pragma unroll
            for (int k = 1; k < R1; ++k) x[k] = cmulc(x[k], ld_table(&twb[k * T2]));
            dft<R1, true>(x);
#pragma unroll
            for (int j = 0; j < R1; ++j) v[m + M * j] = x[j];
        }
        cta_sync();
    }
}

}  // namespace pgk
