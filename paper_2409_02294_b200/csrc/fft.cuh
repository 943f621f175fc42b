// fft.cuh -- in-register / shared-memory complex128 FFT building block for sm_100a.
//
// A length-L transform is carried by T = L/16 threads holding 16 elements each.  It is split into up
// to three passes  L = RA * RB * RC  (decimation in frequency forward, the exact transpose backward);
// every pass is a set of radix-R DFTs done entirely in registers, and between passes the T threads
// exchange data through ONE padded shared-memory line.  (PAPER.md:19 names "FFT operations" as the
// GPU-resident work; the decomposition is ours.)
//
//   pass A  radix RA, GA = 16/RA DFTs per thread, over the elements  n = MA a + b   (MA = L/RA)
//           thread u holds n = u + T jj  (jj = a GA + g, b = u + T g): coalesced global access;
//           y[d][b] = DFT_RA(x[.][b])[d] * w_L^(b d)                   -> slot  d MA + b
//   pass B  radix RB (three-pass plans only), IN PLACE: thread v owns the slots
//           { da MA + a' RC + b' : a' < RB },  b' = v mod RC,  da = v / RC (+ T/RC per extra DFT);
//           z[da][db][b'] = DFT_RB(y[da][. RC + b'])[db] * w_MA^(b' db)  -> slot  da MA + db RC + b'
//   pass C  radix RC on RC consecutive slots ("block" q' = da RB + db):
//           X[q + (L/RC) c] = DFT_RC(z[da][db][.])[c],   q = da + RA db
// Because pass B is in place, a barrier is needed only between passes (two per transform), and the
// spectrum comes out in a fixed, plan-defined order: block q' holds the bins  q(q') + (L/RC) c.
//
// Two plan kinds:
//   COL  RC = 16, one block per thread in pass C.  The consumer (spectral multiply by a table that
//        is stored in the same order) never needs the natural order.
//   ROW  RC = 8, two blocks per thread in pass C, chosen as the pair (q, L/8 - q): a thread then
//        holds bin k together with bin L - k, which is what the real-data split ("untangle") of a
//        packed real transform needs, so that split costs no extra exchange.
//
// Zero-padded transforms (COL plans): the input's upper half is zero and only the lower half of the
// inverse is wanted, so pass A starts from a pruned radix-RA DFT (dft_zero_upper) and the last inverse
// pass ends in one (idft_lower_half): a thread then moves 8 elements to and from global memory while
// it holds 16 spectrum bins in between.
//
// Twiddles: a thread loads only BASE roots (one per DFT of pass A, one for pass B) from small
// compact tables built on the host in long double, and forms the powers it needs by two interleaved
// multiplication chains.  Chains are at most 8 products deep: the twiddle error stays below ~10 ulp,
// far inside the 1e-10 parity bar.
//
// Shared-memory padding: slot p lives at p + p/RC, i.e. one spare slot per block, so that the block
// stride is odd (conflict-free 16-byte accesses in pass C, which the hardware serves a quarter-warp
// at a time) while runs of RC consecutive slots stay contiguous (passes A and B).
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
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }

// ------------------------------------------------------------------ compile-time roots of unity
// cos / sin of 2 pi n / 32 for any integer n
__host__ __device__ constexpr double cos32q(int n)   // 0 <= n <= 8
{
    return n == 0 ? 1.0
         : n == 1 ? 0.9807852804032304491262
         : n == 2 ? 0.9238795325112867561282
         : n == 3 ? 0.8314696123025452370788
         : n == 4 ? 0.7071067811865475244008
         : n == 5 ? 0.5555702330196022247428
         : n == 6 ? 0.3826834323650897717285
         : n == 7 ? 0.1950903220161282678483
         :          0.0;
}
__host__ __device__ constexpr double cos32(int n)
{
    n = ((n % 32) + 32) % 32;
    return n <= 8 ? cos32q(n) : n <= 16 ? -cos32q(16 - n) : n <= 24 ? -cos32q(n - 16) : cos32q(32 - n);
}
__host__ __device__ constexpr double sin32(int n) { return cos32(n - 8); }

// z * exp(-/+ 2 pi i NUM / 32)   (- forward, + inverse)
template <int NUM, bool INV>
__device__ __forceinline__ cplx mulroot(cplx z)
{
    constexpr int n = ((NUM % 32) + 32) % 32;
    if constexpr (n == 0) {
        return z;
    } else if constexpr (n == 8) {
        return INV ? make_double2(-z.y, z.x) : make_double2(z.y, -z.x);
    } else if constexpr (n == 16) {
        return make_double2(-z.x, -z.y);
    } else if constexpr (n == 24) {
        return INV ? make_double2(z.y, -z.x) : make_double2(-z.y, z.x);
    } else {
        constexpr double c = cos32(n);
        constexpr double s = INV ? sin32(n) : -sin32(n);   // w = c + i s
        return make_double2(fma(-z.y, s, z.x * c), fma(z.y, c, z.x * s));
    }
}

// ------------------------------------------------------------------ radix-N DFT in registers
// Decimation in time on bit-reversed inputs.  A butterfly (a, b) -> (a + w b, a - w b) with a non-trivial
// constant root w = c (1 + i t) costs 6 FMAs instead of a 4-instruction product and 4 additions:
//   u = b.x - t b.y,  v = b.y + t b.x,   a +- c (u, v).
// A radix-16 DFT is then 148 FP64 instructions instead of 168 (all of them occupy the same pipe).
template <int N>
__host__ __device__ constexpr int bitrev(int k)
{
    int r = 0;
    for (int b = 1; b < N; b <<= 1) { r = (r << 1) | (k & 1); k >>= 1; }
    return r;
}

// (a, b) <- (a + w b, a - w b),  w = exp(-/+ 2 pi i NUM / 32)   (- forward, + inverse),  0 <= NUM < 16
template <int NUM, bool INV>
__device__ __forceinline__ void butterfly(cplx &a, cplx &b)
{
    static_assert(NUM >= 0 && NUM < 16, "root");
    if constexpr (NUM == 0) {
        const cplx s = cadd(a, b), d = csub(a, b);
        a = s; b = d;
    } else if constexpr (NUM == 8) {        // w = -i (forward), +i (inverse)
        const cplx wb = INV ? make_double2(-b.y, b.x) : make_double2(b.y, -b.x);
        const cplx s = cadd(a, wb), d = csub(a, wb);
        a = s; b = d;
    } else {
        constexpr double c = cos32(NUM);
        constexpr double t = (INV ? sin32(NUM) : -sin32(NUM)) / cos32(NUM);
        const double u = fma(-t, b.y, b.x);
        const double v = fma(t, b.x, b.y);
        const cplx s = make_double2(fma(c, u, a.x), fma(c, v, a.y));
        const cplx d = make_double2(fma(-c, u, a.x), fma(-c, v, a.y));
        a = s; b = d;
    }
}
// the butterflies of the stage that merges blocks of LEN/2 into blocks of LEN
template <int N, int LEN, bool INV, int B = 0, int J = 0>
__device__ __forceinline__ void dit_stage(cplx *y)
{
    if constexpr (B < N) {
        if constexpr (J < LEN / 2) {
            butterfly<J * (32 / LEN), INV>(y[B + J], y[B + J + LEN / 2]);
            dit_stage<N, LEN, INV, B, J + 1>(y);
        } else {
            dit_stage<N, LEN, INV, B + LEN, 0>(y);
        }
    }
}
template <int N, int LEN, bool INV>
__device__ __forceinline__ void dit_stages(cplx *y)
{
    if constexpr (LEN <= N) {
        dit_stage<N, LEN, INV>(y);
        dit_stages<N, 2 * LEN, INV>(y);
    }
}

// the stages LEN, 2 LEN, ..., LAST only
template <int N, int LEN, int LAST, bool INV>
__device__ __forceinline__ void dit_stages_upto(cplx *y)
{
    if constexpr (LEN <= LAST) {
        dit_stage<N, LEN, INV>(y);
        dit_stages_upto<N, 2 * LEN, LAST, INV>(y);
    }
}

// natural order in -> natural order out (x is any array of at least N elements)
template <int N, bool INV>
__device__ __forceinline__ void dft(cplx *x)
{
    static_assert(N <= 32, "radix");
    if constexpr (N >= 2) {
        cplx y[N];
#pragma unroll
        for (int k = 0; k < N; ++k) y[k] = x[bitrev<N>(k)];
        dit_stages<N, 2, INV>(y);
#pragma unroll
        for (int k = 0; k < N; ++k) x[k] = y[k];
    }
}

// ------------------------------------------------------------------ pruned radix-N DFTs (zero-padded transforms)
// Forward DFT of N points whose upper half is zero: x[0..N/2) in, X[0..N) out (natural order).  In the
// bit-reversed input order of the decimation-in-time flow the zeros are the odd positions, so the first stage
// degenerates to copies.
template <int N>
__device__ __forceinline__ void dft_zero_upper(cplx *x)
{
    static_assert(N >= 2 && N <= 32, "radix");
    cplx y[N];
#pragma unroll
    for (int j = 0; j < N / 2; ++j) y[2 * j] = y[2 * j + 1] = x[bitrev<N>(2 * j)];
    dit_stages<N, 4, false>(y);
#pragma unroll
    for (int k = 0; k < N; ++k) x[k] = y[k];
}
// a <- a + w b,  w = exp(-/+ 2 pi i NUM / 32): the half of a butterfly whose other output is not wanted
template <int NUM, bool INV>
__device__ __forceinline__ void half_butterfly(cplx &a, const cplx b)
{
    static_assert(NUM >= 0 && NUM < 16, "root");
    if constexpr (NUM == 0) {
        a = cadd(a, b);
    } else if constexpr (NUM == 8) {
        a = INV ? make_double2(a.x - b.y, a.y + b.x) : make_double2(a.x + b.y, a.y - b.x);
    } else {
        constexpr double c = cos32(NUM);
        constexpr double t = (INV ? sin32(NUM) : -sin32(NUM)) / cos32(NUM);
        const double u = fma(-t, b.y, b.x);
        const double v = fma(t, b.x, b.y);
        a = make_double2(fma(c, u, a.x), fma(c, v, a.y));
    }
}
template <int N, int J = 0>
__device__ __forceinline__ void lower_half_stage(cplx *y)
{
    if constexpr (J < N / 2) {
        half_butterfly<J * (32 / N), true>(y[J], y[J + N / 2]);
        lower_half_stage<N, J + 1>(y);
    }
}
// Inverse DFT of N points of which only the lower half of the outputs is wanted:
// y[n] = sum_d X[d] exp(+2 pi i n d / N), n < N/2, left in x[0..N/2): the last decimation-in-time stage is halved
template <int N>
__device__ __forceinline__ void idft_lower_half(cplx *x)
{
    static_assert(N >= 2 && N <= 32, "radix");
    cplx y[N];
#pragma unroll
    for (int k = 0; k < N; ++k) y[k] = x[bitrev<N>(k)];
    if constexpr (N >= 4) dit_stages_upto<N, 2, N / 2, true>(y);
    lower_half_stage<N>(y);
#pragma unroll
    for (int k = 0; k < N / 2; ++k) x[k] = y[k];
}

// ------------------------------------------------------------------ plan
enum { COL = 0, ROW = 1 };

template <int L, int KIND>
struct Plan {
    static constexpr int RC = (KIND == ROW) ? 8 : 16;
    static_assert(L >= 16 && L <= 4096 && (L & (L - 1)) == 0, "unsupported FFT length");
    static constexpr int REST = L / RC;                                  // RA * RB
    static constexpr int NPASS = REST == 1 ? 1 : (REST <= 16 ? 2 : 3);
    static constexpr int RB = NPASS == 3 ? RC : 1;
    static constexpr int RA = REST / RB;
    static constexpr int T = L / 16;                 // threads per transform
    static constexpr int GA = 16 / RA;               // DFTs per thread in pass A
    static constexpr int GB = 16 / RB;               // DFTs per thread in pass B (three-pass plans)
    static constexpr int GC = 16 / RC;               // blocks per thread in pass C
    static constexpr int MA = L / RA;                // sub-length after pass A
    static constexpr int NB = L / RC;                // number of blocks = stride of the bins of a block
    static constexpr int LINE = L + L / RC;          // padded slots per transform
    // compact twiddle table of a transform (host: polargrav.cu fills it in this order)
    static constexpr int TW_A = 0;                   // [MA]  exp(-2 pi i b / L)
    static constexpr int TW_B = MA;                  // [RC]  exp(-2 pi i b' / MA)
    static constexpr int TW_UN = TW_B + RC;          // [NB]  i exp(-2 pi i q / 2L)         (ROW only)
    static constexpr int TW_LEN = TW_UN + ((KIND == ROW) ? NB : 0);
    static_assert(NPASS < 3 || T % RC == 0, "pass B mapping needs T to be a multiple of RC");
    // first bin of block q'
    static __host__ __device__ constexpr int bin0(int qp) { return NPASS == 3 ? (qp / RB) + RA * (qp % RB) : qp; }
};

template <int RC>
__host__ __device__ constexpr int pad(int p) { return p + p / RC; }

// ------------------------------------------------------------------ barriers
// Barrier among ALL threads that run a kernel body.  CtaBarrier: the whole CTA (the stand-alone kernels).
// PartBarrier<N>: the first N threads of a larger CTA, on named barrier 15 (the fused small-grid kernel, kernels.cuh,
// whose phases use different thread counts; N is a multiple of 32).
struct CtaBarrier {
    static __device__ __forceinline__ void sync() { __syncthreads(); }
};
template <int N>
struct PartBarrier {
    static_assert(N % 32 == 0, "whole warps");
    static __device__ __forceinline__ void sync() { asm volatile("bar.sync 15, %0;" ::"n"(N) : "memory"); }
};

// Sync<T, CTA, CB>: barrier among the T threads of one transform.  When a transform is made of whole
// warps (T >= 32) and the CTA holds several transforms, each gets its own named barrier
// (bar.sync id, T; ids 1 .. 8), so that the transforms of a CTA drift apart instead of marching in lockstep;
// otherwise the barrier CB of all the body's threads is used (every thread then runs the same sequence).
template <int T, int CTA_THREADS, class CB = CtaBarrier>
struct Sync {
    static constexpr bool NAMED = (T >= 32) && (T < CTA_THREADS);
    int id;
    __device__ __forceinline__ explicit Sync(int barrier_id) : id(barrier_id) {}
    __device__ __forceinline__ void operator()() const
    {
        if constexpr (NAMED) asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(T) : "memory");
        else CB::sync();
    }
};

// ------------------------------------------------------------------ twiddle powers
// x[d] *= s^d  (CONJ: conj(s)^d),  d = 0..K-1.  Two interleaved chains advanced by the same step
// (s^2) keep the dependency depth at K/2.
template <int K, bool CONJ>
__device__ __forceinline__ void apply_powers(cplx *x, const cplx s)
{
    if constexpr (K >= 2) {
        const cplx s2 = csq(s);
        cplx a = s2;               // s^2, s^4, ...   (even d >= 2)
        cplx b = s;                // s^1, s^3, ...   (odd d)
        x[1] = CONJ ? cmulc(x[1], b) : cmul(x[1], b);
#pragma unroll
        for (int d = 2; d < K; ++d) {
            if (d & 1) {
                b = cmul(b, s2);
                x[d] = CONJ ? cmulc(x[d], b) : cmul(x[d], b);
            } else {
                if (d > 2) a = cmul(a, s2);
                x[d] = CONJ ? cmulc(x[d], a) : cmul(x[d], a);
            }
        }
    }
}

// ------------------------------------------------------------------ twiddle bases of one thread
// Only the table addresses are kept; a base root is loaded where it is used (holding the roots in
// registers across the transform costs 8-12 registers and pushes the 128-register kernels into
// local-memory spills: measured 76 -> 97 us per solve at 2048^2).
template <int L, int KIND>
struct Bases {
    typedef Plan<L, KIND> P;
    const cplx *tw;
    __device__ __forceinline__ void load(const cplx *__restrict__ table, const int, const bool) { tw = table; }
    __device__ __forceinline__ cplx a(const int u, const int g) const { return __ldg(tw + P::TW_A + u + P::T * g); }
    __device__ __forceinline__ cplx b(const int u) const { return __ldg(tw + P::TW_B + u % P::RC); }
};

// ------------------------------------------------------------------ forward passes
// Every pass comes in three parts -- load (shared memory -> v), compute (v in place, registers only),
// store (v -> shared memory) -- so that a kernel can put its own synchronisation between them
// (cols_kernel alternates the compute parts of two transforms, kernels.cuh).  The fused forms
// fwd_a / fwd_b / ... below keep the older call sites short.
//
// pass A: v[jj] = x[u + T jj] on entry.  DFT g of the thread works on v[a GA + g], a < RA, in place:
// output d of DFT g is left in v[d GA + g].  One-pass plans do nothing here.
template <int L, int KIND>
__device__ __forceinline__ void fwd_a_compute(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA;
    if constexpr (P::NPASS > 1) {
#pragma unroll
        for (int g = 0; g < GA; ++g) {
            cplx x[RA];
#pragma unroll
            for (int a = 0; a < RA; ++a) x[a] = v[a * GA + g];
            const cplx s = tw.a(u, g);
            dft<RA, false>(x);
            apply_powers<RA, false>(x, s);
#pragma unroll
            for (int d = 0; d < RA; ++d) v[d * GA + g] = x[d];
        }
    }
}
template <int L, int KIND>
__device__ __forceinline__ void fwd_a_store(const cplx (&v)[16], cplx *__restrict__ line, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA, T = P::T, MA = P::MA, RC = P::RC;
    if constexpr (P::NPASS > 1) {
        cplx *base = line + pad<RC>(u);
#pragma unroll
        for (int g = 0; g < GA; ++g) {
#pragma unroll
            for (int d = 0; d < RA; ++d) {
                if ((T * g) % RC == 0) base[pad<RC>(d * MA + T * g)] = v[d * GA + g];
                else line[pad<RC>(d * MA + u + T * g)] = v[d * GA + g];
            }
        }
    }
}
template <int L, int KIND>
__device__ __forceinline__ void fwd_a(cplx (&v)[16], cplx *__restrict__ line, const Bases<L, KIND> &tw, const int u)
{
    fwd_a_compute<L, KIND>(v, tw, u);
    fwd_a_store<L, KIND>(v, line, u);
}

// Pass A of a transform whose input is zero in its upper half (the zero-padded radial transform):
// only v[0..8) is read (element n = u + T jj < L/2); all 16 outputs are produced as in fwd_a_compute.
template <int L, int KIND>
__device__ __forceinline__ void fwd_a_compute_zero_upper(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA;
    static_assert(P::NPASS > 1 && RA >= 2, "zero-padded plans have at least two passes");
    cplx y[16];
#pragma unroll
    for (int g = 0; g < GA; ++g) {
        cplx x[RA];
#pragma unroll
        for (int a = 0; a < RA / 2; ++a) x[a] = v[a * GA + g];
        const cplx s = tw.a(u, g);
        dft_zero_upper<RA>(x);
        apply_powers<RA, false>(x, s);
#pragma unroll
        for (int d = 0; d < RA; ++d) y[d * GA + g] = x[d];
    }
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = y[j];
}
// Inverse pass A keeping only the lower half of the outputs (the crop back to L/2 points):
// v[jj], jj < 8, is element n = u + T jj
template <int L, int KIND>
__device__ __forceinline__ void inv_a_compute_lower_half(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA;
    static_assert(P::NPASS > 1 && RA >= 2, "zero-padded plans have at least two passes");
    cplx y[8];
#pragma unroll
    for (int g = 0; g < GA; ++g) {
        cplx x[RA];
        const cplx s = tw.a(u, g);
#pragma unroll
        for (int d = 0; d < RA; ++d) x[d] = v[d * GA + g];
        apply_powers<RA, true>(x, s);
        idft_lower_half<RA>(x);
#pragma unroll
        for (int a = 0; a < RA / 2; ++a) y[a * GA + g] = x[a];
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = y[j];
}

// pass B in place (three-pass plans; no-op otherwise): DFT h of the thread sits in v[h RB + a]
template <int L, int KIND>
__device__ __forceinline__ cplx *pass_b_base(cplx *__restrict__ line, const int u)
{
    typedef Plan<L, KIND> P;
    return line + pad<P::RC>((u / P::RC) * P::MA) + u % P::RC;
}
template <int L, int KIND>
__device__ __forceinline__ void pass_b_load(cplx (&v)[16], const cplx *__restrict__ base)
{
    typedef Plan<L, KIND> P;
    if constexpr (P::NPASS == 3) {
        constexpr int RB = P::RB, GB = P::GB, T = P::T, MA = P::MA, RC = P::RC;
#pragma unroll
        for (int h = 0; h < GB; ++h)
#pragma unroll
            for (int a = 0; a < RB; ++a) v[h * RB + a] = base[pad<RC>((T / RC) * h * MA + a * RC)];
    }
}
template <int L, int KIND>
__device__ __forceinline__ void pass_b_store(const cplx (&v)[16], cplx *__restrict__ base)
{
    typedef Plan<L, KIND> P;
    if constexpr (P::NPASS == 3) {
        constexpr int RB = P::RB, GB = P::GB, T = P::T, MA = P::MA, RC = P::RC;
#pragma unroll
        for (int h = 0; h < GB; ++h)
#pragma unroll
            for (int a = 0; a < RB; ++a) base[pad<RC>((T / RC) * h * MA + a * RC)] = v[h * RB + a];
    }
}
template <int L, int KIND>
__device__ __forceinline__ void fwd_b_compute(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    if constexpr (P::NPASS == 3) {
        constexpr int RB = P::RB, GB = P::GB;
        const cplx s = tw.b(u);
#pragma unroll
        for (int h = 0; h < GB; ++h) {
            dft<RB, false>(&v[h * RB]);
            apply_powers<RB, false>(&v[h * RB], s);
        }
    }
}
// fwd_b: call after a barrier; no barrier inside
template <int L, int KIND>
__device__ __forceinline__ void fwd_b(cplx *__restrict__ line, const Bases<L, KIND> &tw, const int u)
{
    if constexpr (Plan<L, KIND>::NPASS == 3) {
        cplx v[16];
        cplx *base = pass_b_base<L, KIND>(line, u);
        pass_b_load<L, KIND>(v, base);
        fwd_b_compute<L, KIND>(v, tw, u);
        pass_b_store<L, KIND>(v, base);
    }
}

// pass C (COL): thread u owns block u = 16 consecutive slots
template <int L>
__device__ __forceinline__ void pass_c_col_load(cplx (&v)[16], const cplx *__restrict__ line, const int u)
{
    if constexpr (Plan<L, COL>::NPASS > 1) {
        const cplx *b = line + 17 * u;
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = b[j];
    }
}
template <int L>
__device__ __forceinline__ void pass_c_col_store(const cplx (&v)[16], cplx *__restrict__ line, const int u)
{
    if constexpr (Plan<L, COL>::NPASS > 1) {
        cplx *b = line + 17 * u;
#pragma unroll
        for (int j = 0; j < 16; ++j) b[j] = v[j];
    }
}
// fwd_c (COL): after a barrier, thread u reads block u and runs the last radix-16:
// v[c] = X[bin0(u) + T c].  One-pass plans transform the registers they are given.
template <int L>
__device__ __forceinline__ void fwd_c_col(cplx (&v)[16], const cplx *__restrict__ line, const int u)
{
    pass_c_col_load<L>(v, line, u);
    dft<16, false>(v);
}

// fwd_c (ROW): blocks b1 -> v[0..8), b2 -> v[8..16); v[c] = X[bin0(b1) + NB c], v[8+c] = X[bin0(b2) + NB c]
template <int L>
__device__ __forceinline__ void fwd_c_row(cplx (&v)[16], const cplx *__restrict__ line, const int b1, const int b2)
{
    const cplx *p1 = line + 9 * b1, *p2 = line + 9 * b2;
#pragma unroll
    for (int j = 0; j < 8; ++j) { v[j] = p1[j]; v[8 + j] = p2[j]; }
    dft<8, false>(&v[0]);
    dft<8, false>(&v[8]);
}

// ------------------------------------------------------------------ inverse passes (unnormalised)
// Exact transpose of the forward flow graph with conjugated twiddles.
template <int L>
__device__ __forceinline__ void inv_c_col(cplx (&v)[16], cplx *__restrict__ line, const int u)
{
    dft<16, true>(v);
    pass_c_col_store<L>(v, line, u);
}

template <int L>
__device__ __forceinline__ void inv_c_row(cplx (&v)[16], cplx *__restrict__ line, const int b1, const int b2)
{
    dft<8, true>(&v[0]);
    dft<8, true>(&v[8]);
    cplx *p1 = line + 9 * b1, *p2 = line + 9 * b2;
#pragma unroll
    for (int j = 0; j < 8; ++j) { p1[j] = v[j]; p2[j] = v[8 + j]; }
}

template <int L, int KIND>
__device__ __forceinline__ void inv_b_compute(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    if constexpr (P::NPASS == 3) {
        constexpr int RB = P::RB, GB = P::GB;
        const cplx s = tw.b(u);
#pragma unroll
        for (int h = 0; h < GB; ++h) {
            apply_powers<RB, true>(&v[h * RB], s);
            dft<RB, true>(&v[h * RB]);
        }
    }
}
template <int L, int KIND>
__device__ __forceinline__ void inv_b(cplx *__restrict__ line, const Bases<L, KIND> &tw, const int u)
{
    if constexpr (Plan<L, KIND>::NPASS == 3) {
        cplx v[16];
        cplx *base = pass_b_base<L, KIND>(line, u);
        pass_b_load<L, KIND>(v, base);
        inv_b_compute<L, KIND>(v, tw, u);
        pass_b_store<L, KIND>(v, base);
    }
}

// inverse pass A: load leaves input d of DFT g in v[d GA + g]; compute leaves element n = u + T jj in v[jj]:
// v[jj] = sum_k X[k] exp(+2 pi i n k / L)
template <int L, int KIND>
__device__ __forceinline__ void inv_a_load(cplx (&v)[16], const cplx *__restrict__ line, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA, T = P::T, MA = P::MA, RC = P::RC;
    if constexpr (P::NPASS > 1) {
        const cplx *base = line + pad<RC>(u);
#pragma unroll
        for (int g = 0; g < GA; ++g) {
#pragma unroll
            for (int d = 0; d < RA; ++d) {
                if ((T * g) % RC == 0) v[d * GA + g] = base[pad<RC>(d * MA + T * g)];
                else v[d * GA + g] = line[pad<RC>(d * MA + u + T * g)];
            }
        }
    }
}
template <int L, int KIND>
__device__ __forceinline__ void inv_a_compute(cplx (&v)[16], const Bases<L, KIND> &tw, const int u)
{
    typedef Plan<L, KIND> P;
    constexpr int RA = P::RA, GA = P::GA;
    if constexpr (P::NPASS > 1) {
#pragma unroll
        for (int g = 0; g < GA; ++g) {
            cplx x[RA];
            const cplx s = tw.a(u, g);
#pragma unroll
            for (int d = 0; d < RA; ++d) x[d] = v[d * GA + g];
            apply_powers<RA, true>(x, s);
            dft<RA, true>(x);
#pragma unroll
            for (int a = 0; a < RA; ++a) v[a * GA + g] = x[a];
        }
    }
}
// inv_a: after a barrier
template <int L, int KIND>
__device__ __forceinline__ void inv_a(cplx (&v)[16], const cplx *__restrict__ line, const Bases<L, KIND> &tw, const int u)
{
    inv_a_load<L, KIND>(v, line, u);
    inv_a_compute<L, KIND>(v, tw, u);
}

// slot of element n = u + T jj of the natural order (pass A's side of the line): thread u owns
// these 16 slots during pass A, forward and inverse
template <int L, int KIND>
__device__ __forceinline__ int own_slot(const int u, const int jj)
{
    return pad<Plan<L, KIND>::RC>(u + Plan<L, KIND>::T * jj);
}

// ------------------------------------------------------------------ ROW plans: pass-C block pairs
// Thread t of a transform takes the blocks (b1, b2) whose bins are mirror images:
//   bins of b1:  k = q1 + NB c,   bins of b2:  L - k = q2 + NB (7 - c),   q2 = NB - q1.
// One thread per transform is SPECIAL: it takes the two self-mirrored blocks, q = 0 (c <-> 8 - c,
// with c = 0 the DC / Nyquist pair and c = 4 its own mirror) and q = NB/2 (c <-> 7 - c).
template <int L>
__device__ __forceinline__ void row_blocks(const int t, int &b1, int &b2, bool &special)
{
    typedef Plan<L, ROW> P;
    if constexpr (P::NPASS == 3) {
        constexpr int NREG = P::T - P::RB / 2;
        if (t < NREG) { b1 = P::RB + t; b2 = P::NB - 1 - t; special = false; }
        else {
            const int s = t - NREG;
            special = (s == 0);
            b1 = s; b2 = P::RB - s;
            if (special) b2 = P::RB / 2;
        }
    } else {
        special = (t == 0);
        b1 = t; b2 = special ? P::RA / 2 : P::RA - t;
    }
}

}  // namespace pgk
