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
// Twiddles.  The first version of this file read every inter-pass twiddle from a global table
// (29 16-byte loads per thread and transform at L = 2048).  ncu showed the L1TEX data pipe as the
// busiest unit of all three kernels with ~40 % of its wavefronts spent on those table reads, and
// their L1/L2 latency exposed once per pass (profiles/r1_01_baseline.md).  Now a thread loads only
// its BASE roots once (Twid<L>: w_L^(u + T m) for the leading pass, w_T2^t for the radix-16 link)
// from one unit-root table  root[b * rs] = exp(-2 pi i b / L)  built on the host in long double,
// and forms the powers it needs by two interleaved multiplication chains (step p^2), which costs
// ~16 % more FP64 instructions but no table traffic.  Chains are at most 7 products deep: the
// twiddle error stays below ~10 ulp, far inside the 1e-10 parity bar.
//
// The transform is split into a HEAD (everything up to the stores of the last exchange) and a
// LAST pass (16 consecutive slots -> radix-16), so that a kernel may hand the last pass to a
// different thread than the one that ran the head (rows kernels: row-fastest mapping for a
// coalesced transposed store without an extra shared-memory transposition).
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
// w * w
__device__ __forceinline__ cplx csq(cplx w)
{
    const double t = w.x * w.y;
    return make_double2(fma(w.x, w.x, -(w.y * w.y)), t + t);
}
// acc + a * w
__device__ __forceinline__ cplx cfma(cplx a, cplx w, cplx acc)
{
    return make_double2(fma(-a.y, w.y, fma(a.x, w.x, acc.x)), fma(a.y, w.x, fma(a.x, w.y, acc.y)));
}
// acc + conj(a) * w
__device__ __forceinline__ cplx cfmac(cplx a, cplx w, cplx acc)
{
    return make_double2(fma(a.y, w.y, fma(a.x, w.x, acc.x)), fma(-a.y, w.x, fma(a.x, w.y, acc.y)));
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }

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
    static constexpr int M = 16 / R1;                        // butterflies per thread in the leading pass
    static constexpr int T2 = L / R1;                        // sub-length after the leading pass
    static constexpr int T3 = T2 / 16;                       // sub-length after the first radix-16 pass
    static constexpr int NLEAD = (R1 > 1) ? M : 1;           // base roots held for the leading pass
    static constexpr int LINE = pad_idx(L) + 8;              // smem slots per transform (>= pad_idx(L)+1)
    static constexpr bool HAS_EXCHANGE = (L > 16);           // false: the whole transform is one radix-16
};

// ------------------------------------------------------------------ barriers
// Sync<T, CTA>: barrier among the T threads of one transform.  When a transform is made of whole
// warps (T >= 32) and the CTA holds several transforms, each gets its own named barrier
// (bar.sync id, T), so that the transforms of a CTA drift apart instead of marching in lockstep;
// otherwise the CTA-wide barrier is used (every thread of the CTA then runs the same sequence).
template <int T, int CTA_THREADS>
struct Sync {
    static constexpr bool NAMED = (T >= 32) && (T < CTA_THREADS) && (CTA_THREADS / T <= 15);
    int id;
    __device__ __forceinline__ explicit Sync(int group) : id(group + 1) {}
    __device__ __forceinline__ void operator()() const
    {
        if constexpr (NAMED) asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(T) : "memory");
        else __syncthreads();
    }
};

// ------------------------------------------------------------------ shared-memory addressing
// Every exchange address is written as (per-thread base) + (compile-time constant), so that the
// forward and the inverse transform of one kernel share three base registers instead of keeping
// dozens of computed addresses alive.
//   pad_idx(a + c) = pad_idx(a) + c + c/16            when c is a multiple of 16
//   pad_idx(16 a + j) = 17 a + j                      for 0 <= j < 16
template <int L>
struct Lines {
    typedef Plan<L> P;
    cplx *lin;   // sm + pad_idx(u)            consecutive-lane side of the radix-16 exchanges
    cplx *mid;   // sm + pad_idx(q T2 + t)     strided side of the leading-pass exchange
    __device__ __forceinline__ Lines(cplx *sm, int u)
    {
        lin = sm + (P::N16 == 2 ? pad_idx(u) : u);
        mid = (P::N16 == 2) ? sm + (u / P::T3) * pad_idx(P::T2) + (u % P::T3) : sm + 17 * u;
    }
    // 16 consecutive slots of the last radix-16 pass of thread u
    static __device__ __forceinline__ cplx *blk(cplx *sm, int u) { return sm + 17 * u; }
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

// ------------------------------------------------------------------ twiddle bases and powers
// root[b * rs] = exp(-2 pi i b / L) for 0 <= b < L  (rs = table length / L)
template <int L>
struct Twid {
    typedef Plan<L> P;
    cplx lead[P::NLEAD];   // w_L^(u + T m), m < M            (R1 > 1)
    cplx link;             // w_T2^t = w_L^(R1 t), t = u % T3  (N16 == 2)
    __device__ __forceinline__ void load(const cplx *__restrict__ root, const int rs, const int u)
    {
        if constexpr (P::R1 > 1) {
#pragma unroll
            for (int m = 0; m < P::M; ++m) lead[m] = __ldg(&root[(u + P::T * m) * rs]);
        }
        if constexpr (P::N16 == 2) link = __ldg(&root[(u % P::T3) * P::R1 * rs]);
    }
};

// x[k] *= p^k (CONJ: conj(p)^k) for k = 1..K-1.  Two interleaved chains a = p^(odd), b = p^(even),
// both advanced by p^2: depth K/2, three live roots.
template <int K, bool CONJ>
__device__ __forceinline__ void apply_powers(cplx *x, const cplx p)
{
    if constexpr (K >= 2) {
        x[1] = CONJ ? cmulc(x[1], p) : cmul(x[1], p);
        if constexpr (K > 2) {
            const cplx p2 = csq(p);
            cplx a = p, b = p2;
            x[2] = CONJ ? cmulc(x[2], b) : cmul(x[2], b);
#pragma unroll
            for (int k = 3; k < K; k += 2) {
                a = cmul(a, p2);
                x[k] = CONJ ? cmulc(x[k], a) : cmul(x[k], a);
                if (k + 1 < K) {
                    b = cmul(b, p2);
                    x[k + 1] = CONJ ? cmulc(x[k + 1], b) : cmul(x[k + 1], b);
                }
            }
        }
    }
}

// ------------------------------------------------------------------ forward transform
// v[jj] = x[u + T*jj]  ->  v[k] = X[u + T*k],  X[k] = sum_n x[n] exp(-2 pi i n k / L)
//
// fwd_head: all passes but the last, ending with the STORES of the last exchange (no barrier).
// fwd_last: after a barrier that covers those stores, thread u' of the transform whose line is
//           `sm` reads its 16 slots and runs the last radix-16: v[k] = X[u' + T*k].
// For L == 16 the head is empty and fwd_last transforms the registers it is given.
template <int L, class SyncT>
__device__ __forceinline__ void fwd_head(cplx (&v)[16], cplx *__restrict__ sm, const Twid<L> &tw, const int u,
                                         const SyncT &sync)
{
    typedef Plan<L> P;
    typedef Lines<L> A;
    constexpr int T = P::T, R1 = P::R1, M = P::M;
    (void)T;
    const A a(sm, u);
    if constexpr (R1 > 1) {
#pragma unroll
        for (int m = 0; m < M; ++m) {
            cplx x[R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = v[m + M * j];
            dft<R1, false>(x);
            apply_powers<R1, false>(x, tw.lead[m]);
#pragma unroll
            for (int k = 0; k < R1; ++k) a.lin[A::lead(k, m)] = x[k];
        }
    }
    if constexpr (P::N16 == 2) {
        if constexpr (R1 > 1) {
            sync();
#pragma unroll
            for (int j = 0; j < 16; ++j) v[j] = a.mid[A::midj(j)];
            sync();
        }
        dft<16, false>(v);
        apply_powers<16, false>(v, tw.link);
#pragma unroll
        for (int k = 0; k < 16; ++k) a.lin[A::link(k)] = v[k];
    }
}

template <int L>
__device__ __forceinline__ void fwd_last(cplx (&v)[16], const cplx *__restrict__ sm, const int u)
{
    if constexpr (Plan<L>::HAS_EXCHANGE) {
        const cplx *b = sm + 17 * u;
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = b[j];
    }
    dft<16, false>(v);
}

// ------------------------------------------------------------------ inverse transform (unnormalised)
// v[k] = X[u + T*k]  ->  v[jj] = sum_k X[k] exp(+2 pi i n k / L),  n = u + T*jj
// Exact transpose of the forward flow graph, with conjugated twiddles.
//
// inv_first: radix-16 on X[u' + T*k] and the stores of the first exchange (no barrier).
// inv_tail : after a barrier, thread u finishes the transform.
template <int L>
__device__ __forceinline__ void inv_first(cplx (&v)[16], cplx *__restrict__ sm, const int u)
{
    dft<16, true>(v);
    if constexpr (Plan<L>::HAS_EXCHANGE) {
        cplx *b = sm + 17 * u;
#pragma unroll
        for (int j = 0; j < 16; ++j) b[j] = v[j];
    }
}

// `trailing`: issue a barrier after the last shared-memory read (needed when the line is reused).
template <int L, class SyncT>
__device__ __forceinline__ void inv_tail(cplx (&v)[16], cplx *__restrict__ sm, const Twid<L> &tw, const int u,
                                         const SyncT &sync, const bool trailing)
{
    typedef Plan<L> P;
    typedef Lines<L> A;
    constexpr int R1 = P::R1, M = P::M;
    const A a(sm, u);
    if constexpr (P::N16 == 2) {
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = a.lin[A::link(k)];
        apply_powers<16, true>(v, tw.link);
        dft<16, true>(v);
        if constexpr (R1 > 1) {
            sync();
#pragma unroll
            for (int j = 0; j < 16; ++j) a.mid[A::midj(j)] = v[j];
            sync();
        }
    }
    if constexpr (R1 > 1) {
#pragma unroll
        for (int m = 0; m < M; ++m) {
            cplx x[R1];
#pragma unroll
            for (int k = 0; k < R1; ++k) x[k] = a.lin[A::lead(k, m)];
            apply_powers<R1, true>(x, tw.lead[m]);
            dft<R1, true>(x);
#pragma unroll
            for (int j = 0; j < R1; ++j) v[m + M * j] = x[j];
        }
    }
    if (P::HAS_EXCHANGE && trailing) sync();
}

// ------------------------------------------------------------------ whole transforms, one thread mapping
template <int L, class SyncT>
__device__ __forceinline__ void fft_fwd(cplx (&v)[16], cplx *__restrict__ sm, const Twid<L> &tw, const int u,
                                        const SyncT &sync, const bool trailing)
{
    fwd_head<L>(v, sm, tw, u, sync);
    if constexpr (Plan<L>::HAS_EXCHANGE) sync();
    fwd_last<L>(v, sm, u);
    if (Plan<L>::HAS_EXCHANGE && trailing) sync();
}

template <int L, class SyncT>
__device__ __forceinline__ void fft_inv(cplx (&v)[16], cplx *__restrict__ sm, const Twid<L> &tw, const int u,
                                        const SyncT &sync, const bool trailing)
{
    inv_first<L>(v, sm, u);
    if constexpr (Plan<L>::HAS_EXCHANGE) sync();
    inv_tail<L>(v, sm, tw, u, sync, trailing);
}

}  // namespace pgk
