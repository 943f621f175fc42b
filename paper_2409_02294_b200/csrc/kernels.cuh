// kernels.cuh -- the sm_100a kernels of the FFT-convolution path (rows a1-a5 of DESIGN.md).
//
// Data layout in HBM (all fp64 / complex128), H = n_phi/2:
//   Sigma, Phi : [B][n_r][n_phi]          phi fastest (user arrays)
//   W          : [B][H+1][n_r] complex    TRANSPOSED Hermitian half-spectrum: W[m][i] = 2 x (azimuthal mode m
//                                         of row i of Sigma r^{3/2}), m = 0..H; column m is contiguous in r.
//                                         Row i is packed as z[n] = s[2n] + i s[2n+1], transformed with a
//                                         complex FFT of length H, and split into the modes of the real row
//                                         inside the last pass of the row kernel (fft.cuh, ROW plans).
//                                         The column kernel transforms W in place; the inverse row kernel
//                                         re-packs and transforms back.
//   Khat       : [H+1][2 n_r] real        spectrum of the Green's kernel for azimuthal mode m over the bins of
//                                         the 2 n_r-point padded radial transform, STORED IN THE ORDER THE
//                                         COLUMN KERNEL HOLDS THEM
//                                         (entry c T + u is bin  bin0(u) + T c); all normalisations folded in
//   tw_row, tw_col : compact twiddle tables (Plan<L,KIND>::TW_*), long double on the host
#pragma once
#include <cooperative_groups.h>
#include <cuda.h>          // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint)
#include "fft.cuh"

#ifndef PG_ROW_THREADS
#define PG_ROW_THREADS 128
#endif
#ifndef PG_ROW_THREADS_BIG
#define PG_ROW_THREADS_BIG 256      // n_phi >= 2048, forward row kernel: 4 rows per CTA (64-byte runs in W), two CTAs per
                                    // SM.  W is stored transposed, so a CTA of ROWS rows touches it in runs of ROWS * 16
                                    // bytes, and the L2 serves 32-byte runs at half the rate of 64-byte ones (4.0 against
                                    // 5.3 (stores) .. 7.7 TB/s (loads), measured): with 2 rows per CTA the kernel's
                                    // transposed STORES were bound by it.
#endif
#ifndef PG_ROW_THREADS_BIG_INV
#define PG_ROW_THREADS_BIG_INV 128  // n_phi >= 2048, inverse row kernel: 2 rows per CTA, FOUR CTAs per SM.  Its transposed
                                    // READS are one TMA tile per item (asynchronous, off the LSU), so the run length
                                    // matters less than the number of independent items an SM has in flight: 12.47 us
                                    // (4 rows, 2 CTAs) -> 11.57 us (2 rows, 4 CTAs) per 2048^2 field at saturation.
#endif
#ifndef PG_ROW_INLINE_FROM
#define PG_ROW_INLINE_FROM 2048     // from this n_phi on the row kernels stage their input INSIDE the rows' own lines
#endif
#ifndef PG_ROW_TILE
#define PG_ROW_TILE 1               // ... and rows_inv_kernel receives its modes as ONE 4-D TMA tile per item
#endif

namespace pgk {

// ---------------------------------------------------------------- shapes
// rows per CTA in the phi passes: W is written/read in runs of ROWS*16 bytes
__host__ __device__ constexpr int rows_per_cta(int nphi, bool inverse = false)
{
    const int T = nphi / 32;
    const int r = (nphi >= 2048 ? (inverse ? PG_ROW_THREADS_BIG_INV : PG_ROW_THREADS_BIG) : PG_ROW_THREADS) / (T > 0 ? T : 1);
    return r < 2 ? 2 : (r > 16 ? 16 : r);
}
// azimuthal modes per CTA in the r pass
__host__ __device__ constexpr int modes_per_cta(int nr)
{
    const int T = nr / 8;          // threads of one 2 n_r-point transform
    const int c = 256 / T;
    return c < 1 ? 1 : (c > 8 ? 8 : c);
}
// Shared-memory slots between the lines of two rows of a CTA.  In the row-fastest pass a
// quarter-warp touches (8 rows) or (4 rows x 2 neighbouring 9-slot blocks): STRIDE = 1 (mod 8)
// resp. 2 (mod 8) spreads them over the eight 16-byte bank groups.
// INV: the shape of the inverse row kernel (it differs from the forward kernel's only at n_phi >= 2048, see above)
template <int NPHI, bool INV = false>
struct RowShape {
    static constexpr int L = NPHI / 2;
    typedef Plan<L, ROW> P;
    static constexpr int T = P::T;
    static constexpr int ROWS = rows_per_cta(NPHI, INV);
    static constexpr int SKEW = (ROWS >= 8) ? 1 : (8 / ROWS);
    static constexpr int STRIDE = ((P::LINE + 7) / 8) * 8 + SKEW;   // slots per row line
    static constexpr int THREADS = ROWS * T;
    static constexpr int SLOTS = 17;                                // prefetch slots per thread (16 fwd, 17 inv)
    // INLINE: no staging area of its own -- the next item's input is fetched into the lines themselves once the current
    // item has left them (a shorter prefetch distance, but half the shared memory: twice the rows resident per SM)
    static constexpr bool INLINE = (NPHI >= PG_ROW_INLINE_FROM);
    // TILE (rows_inv_kernel): the modes of an item, W[m][i0 .. i0 + ROWS) for m < L, arrive as one 4-D tensor-map copy
    // (TMA) into the lines, laid out [m mod RA][m / RA][row]: the transposed gather in runs of ROWS x 16 bytes is done by
    // the copy engine instead of 17 LDGSTS per thread (a quarter of the kernel's LSU wavefronts), and a quarter-warp of
    // the row-fastest pass reads 128 contiguous bytes of the tile.  Mode L (Nyquist) comes by a plain load.
    static constexpr bool TILE = INLINE && (PG_ROW_TILE != 0);
    static constexpr unsigned TILE_BYTES = (unsigned)(L * ROWS * sizeof(cplx));
    static_assert(!TILE || (L * ROWS <= ROWS * STRIDE), "the tile must fit into the lines");
    static_assert(!INLINE || SLOTS * THREADS <= ROWS * STRIDE, "the prefetch slots must fit into the lines");
    static constexpr size_t SMEM = INLINE ? (size_t)ROWS * STRIDE * sizeof(cplx) + 64
                                          : ((size_t)ROWS * STRIDE + (size_t)SLOTS * THREADS) * sizeof(cplx);
    // resident CTAs per SM are set by shared memory (227 KB); registers are capped to match
    static constexpr int BY_SMEM = (int)((227 * 1024) / (SMEM + 1024));
    static constexpr int MIN_CTAS = BY_SMEM < 1 ? 1 : (BY_SMEM * THREADS > 512 ? (512 / THREADS > 0 ? 512 / THREADS : 1) : BY_SMEM);
};
template <int NR>
struct ColShape {
    static constexpr int L = 2 * NR;                        // the zero-padded radial transform
    typedef Plan<L, COL> P;
    static constexpr int T = P::T;                          // threads per mode = n_r / 8
    static constexpr int MODES = modes_per_cta(NR);
    static constexpr int STRIDE = P::LINE;
    static constexpr int THREADS = MODES * T;
    static constexpr size_t LINES = (size_t)MODES * STRIDE * sizeof(cplx);
    // Khat is stored as its symmetric half (Khat[k'] = Khat[2N - k'], K is even in the radial lag): KH doubles per
    // mode -- bins 0..N in the order the threads hold them: entry c T + u is bin  bin0(u) + T c  for c < 8, entry 8 T
    // is bin N, one more pads the slice to 16 bytes.  Thread u finds its bins c >= 8 in the entries of the thread that
    // holds bin0 = T - bin0(u) (col_partner), read backwards: half the HBM traffic and half the staging space.
    static constexpr int KH = L / 2 + 2;
    static constexpr size_t STAGE = (size_t)MODES * KH * sizeof(double);    // Khat slices of the CTA's modes
    static constexpr size_t SMEM = LINES + STAGE + 16;                      // + one mbarrier
    static constexpr int MIN_CTAS = (THREADS >= 512) ? 1 : (THREADS <= 128 ? 4 : 512 / THREADS);   // cap registers at 128/thread
};

__device__ __forceinline__ void prefetch_l1(const void *p)
{
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
}
__device__ __forceinline__ void named_barrier(const int id, const int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void named_barrier_arrive(const int id, const int threads)
{
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
// programmatic dependent launch: wait for the preceding kernel of the stream (no-op without the
// launch attribute) / allow the following kernel's CTAs to be scheduled as this grid drains
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
#ifndef PG_PDL_EARLY
#define PG_PDL_EARLY 1              // 0: the dependents are released when a CTA exits (tuning runs)
#endif
__device__ __forceinline__ void pdl_launch_dependents()
{
#if PG_PDL_EARLY
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}
// orders this thread's view of earlier generic-proxy shared-memory accesses before an asynchronous copy
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---------------------------------------------------------------- bulk asynchronous copy (TMA, 1-D)
// global -> shared, completion signalled on an mbarrier by transferred bytes
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, const int arrivals)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(arrivals) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_load(void *dst_smem, const void *src_global, const unsigned bytes,
                                          unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_addr(dst_smem)),
                 "l"(src_global), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, const unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done)
                     : "r"(smem_addr(bar)), "r"(parity)
                     : "memory");
    } while (!done);
}

// ---------------------------------------------------------------- real-data split of the packed transform
// (A, B) = (Z[k], Z[H-k]) of the packed transform of a real row, ck = i exp(-2 pi i k / n_phi)
// = un * w16^C with un = i exp(-2 pi i q / n_phi) the thread's base and k = q + (H/8) C:
//   2 X[k]   = S - ck D,          S = A + conj(B),  D = A - conj(B)
//   2 X[H-k] = conj(S + ck D)
template <int C>
__device__ __forceinline__ void untangle(const cplx A, const cplx B, const cplx un, cplx &Xk, cplx &Xm)
{
    const cplx S = make_double2(A.x + B.x, A.y - B.y);
    const cplx D = make_double2(A.x - B.x, A.y + B.y);
    const cplx P = cmul(mulroot<2 * C, false>(D), un);
    Xk = make_double2(S.x - P.x, S.y - P.y);
    Xm = make_double2(S.x + P.x, -(S.y + P.y));
}
// inverse: (Yk, Ym) = (Y[k], Y[H-k]) of the Hermitian half-spectrum  ->  packed (Z'[k], Z'[H-k]):
//   Z'[k] = S + Q,  Z'[H-k] = conj(S - Q),   S = Yk + conj(Ym),  Q = -conj(ck) (Yk - conj(Ym))
template <int C>
__device__ __forceinline__ void retangle(const cplx Yk, const cplx Ym, const cplx un, cplx &Zk, cplx &Zm)
{
    const cplx S = make_double2(Yk.x + Ym.x, Yk.y - Ym.y);
    const cplx D = make_double2(Yk.x - Ym.x, Yk.y + Ym.y);
    const cplx Q = mulroot<2 * C, true>(cmulc(D, un));      // conj(ck) D
    Zk = make_double2(S.x - Q.x, S.y - Q.y);
    Zm = make_double2(S.x + Q.x, -(S.y + Q.y));
}

// Pass C of the ROW plan plus the split, for the regular thread (blocks b1 | b2 mirror each other)
// and the special thread (blocks 0 and NB/2 mirror themselves).  STORE(k, value) consumes mode k.
template <int L, int C = 0, class F>
__device__ __forceinline__ void split_regular(const cplx (&v)[16], const cplx un, const int q1, F &&store)
{
    if constexpr (C < 8) {
        constexpr int NB = Plan<L, ROW>::NB;
        cplx xk, xm;
        untangle<C>(v[C], v[15 - C], un, xk, xm);
        store(q1 + NB * C, xk);
        store(L - q1 - NB * C, xm);
        split_regular<L, C + 1>(v, un, q1, store);
    }
}
template <int L, int C = 0, class F>
__device__ __forceinline__ void split_special(const cplx (&v)[16], const cplx un0, const cplx unh, F &&store)
{
    constexpr int NB = Plan<L, ROW>::NB;
    if constexpr (C < 5) {          // block 0: bins NB c, mirror NB (8 - c); c = 0 is the DC / Nyquist pair
        cplx xk, xm;
        untangle<C>(v[C], v[(8 - C) % 8], un0, xk, xm);
        store(NB * C, xk);
        if (C < 4) store(L - NB * C, xm);
        split_special<L, C + 1>(v, un0, unh, store);
    } else if constexpr (C < 9) {   // block NB/2: bins NB/2 + NB c, mirror c <-> 7 - c
        constexpr int c = C - 5;
        cplx xk, xm;
        untangle<c>(v[8 + c], v[15 - c], unh, xk, xm);
        store(NB / 2 + NB * c, xk);
        store(L - NB / 2 - NB * c, xm);
        split_special<L, C + 1>(v, un0, unh, store);
    }
}
// Inverse direction.  The modes a thread needs are enumerated twice in the same order: once to
// prefetch them (modes_*: f(slot, k)), once to consume them (merge_*: get(slot)).
//   regular: slot 2C   = mode q1 + NB C,  slot 2C+1 = its mirror
//   special: slots 0..8 = block 0 (0, L | NB, L-NB | 2NB, L-2NB | 3NB, L-3NB | L/2), slots 9..16 = block NB/2
template <int L, int C = 0, class F>
__device__ __forceinline__ void modes_regular(const int q1, F &&f)
{
    if constexpr (C < 8) {
        constexpr int NB = Plan<L, ROW>::NB;
        f(2 * C, q1 + NB * C);
        f(2 * C + 1, L - q1 - NB * C);
        modes_regular<L, C + 1>(q1, f);
    }
}
template <int L, int C = 0, class F>
__device__ __forceinline__ void modes_special(F &&f)
{
    constexpr int NB = Plan<L, ROW>::NB;
    if constexpr (C < 4) {
        f(2 * C, NB * C);
        f(2 * C + 1, L - NB * C);
        modes_special<L, C + 1>(f);
    } else if constexpr (C == 4) {
        f(8, L / 2);
        modes_special<L, C + 1>(f);
    } else if constexpr (C < 9) {
        constexpr int c = C - 5;
        f(9 + 2 * c, NB / 2 + NB * c);
        f(10 + 2 * c, L - NB / 2 - NB * c);
        modes_special<L, C + 1>(f);
    }
}
template <int L, int C = 0, class F>
__device__ __forceinline__ void merge_regular(cplx (&v)[16], const cplx un, F &&get)
{
    if constexpr (C < 8) {
        retangle<C>(get(2 * C), get(2 * C + 1), un, v[C], v[15 - C]);
        merge_regular<L, C + 1>(v, un, get);
    }
}
template <int L, int C = 0, class F>
__device__ __forceinline__ void merge_special(cplx (&v)[16], const cplx un0, const cplx unh, F &&get)
{
    if constexpr (C < 4) {
        cplx zk, zm;
        retangle<C>(get(2 * C), get(2 * C + 1), un0, zk, zm);
        v[C] = zk;
        if (C > 0) v[8 - C] = zm;
        merge_special<L, C + 1>(v, un0, unh, get);
    } else if constexpr (C == 4) {
        cplx zk, zm;
        const cplx y = get(8);
        retangle<4>(y, y, un0, zk, zm);
        v[4] = zk;
        merge_special<L, C + 1>(v, un0, unh, get);
    } else if constexpr (C < 9) {
        constexpr int c = C - 5;
        retangle<c>(get(9 + 2 * c), get(10 + 2 * c), unh, v[8 + c], v[15 - c]);
        merge_special<L, C + 1>(v, un0, unh, get);
    }
}

// ---------------------------------------------------------------- per-thread asynchronous prefetch
// cp.async (LDGSTS) global -> shared, 16 bytes, bypassing L1 and the register file.  Each thread
// prefetches exactly the elements it will consume itself, into slots only it touches
// (slot j of thread tid = stage[j * THREADS + tid]: conflict-free), so no barrier is involved:
// the thread waits for its own group, moves the slots to registers and at once reuses them for
// the next work item.
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src_global)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr(dst_smem)), "l"(src_global) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---------------------------------------------------------------- a2: rows forward
// PERSISTENT: a CTA walks over work items (ROWS consecutive rows of one field), item = blockIdx.x +
// k gridDim.x, prefetching the next item's rows with cp.async while it transforms the current one.
// Row i: s = Sigma_i * scale_i (scale = r_i^{3/2}, or 1 when rscale == nullptr), packed as
// z[n] = s[2n] + i s[2n+1], complex FFT of length H = n_phi/2.
// Passes A and B run with thread = (row, u) and u fastest (coalesced row loads); pass C and the
// real-data split run with thread = (t, row) and the ROW fastest, so that the modes W[m][i] leave as
// runs of ROWS consecutive rows of one column: the transposed store costs no extra shared-memory
// round trip.
// HALF (the x pass of the 3-D mesh path, cartesian.cuh): the rows in memory hold only the first n_phi/2 reals, the
// second half of the transform's input is zero padding that is never read.
// The body runs as CTA `block` of `nblocks` (block / nblocks in the stand-alone kernel; the fused small-grid kernel
// passes its own) on the shared memory it is given; CB is the barrier among the body's threads.
template <int NPHI, bool HALF, class CB>
__device__ __forceinline__ void rows_fwd_body(const double *__restrict__ sigma, cplx *__restrict__ W, const cplx *__restrict__ tw,
                                              const double *__restrict__ rscale, const int n_rows, const int n_items,
                                              const long sigma_field_stride, const long w_field_stride, const int early_load,
                                              const int block, const int nblocks, unsigned char *smem_raw)
{
    typedef RowShape<NPHI> S;
    typedef Plan<S::L, ROW> P;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    cplx *stage = smem + ROWS * S::STRIDE + threadIdx.x;

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int rp = tid % ROWS, t = tid / ROWS;
    const int items_per_field = n_rows / ROWS;
    cplx *line = smem + rho * S::STRIDE;
    int b1, b2;
    bool special;
    row_blocks<L>(t, b1, b2, special);
    const int q1 = P::bin0(b1);
    const cplx un1 = __ldg(tw + P::TW_UN + (special ? 0 : q1));
    const cplx un2 = __ldg(tw + P::TW_UN + P::NB / 2);
    Bases<L, ROW> bases;
    bases.load(tw, u, false);

    // Rows carried by whole warps (n_phi >= 1024) are fetched by ONE 1-D bulk asynchronous copy (TMA) per row into a
    // raw staging row, completion on a per-row mbarrier: the copy engine writes shared memory itself, so the 16
    // LDGSTS per thread and their LSU issue slots go away.  The next item's row is requested by the row's first thread
    // right after the row barrier that follows pass A (by then the 64 threads of the row have taken their elements).
    // Narrower rows keep the per-thread cp.async slots.
    // INLINE (RowShape): the raw row lands in the row's own line; it is requested once pass C has read the line
    // (CTA-wide barrier), travels while the split and the transposed stores of the current item run, and a row barrier
    // between taking the elements and the stores of pass A keeps the two uses of the line apart.
    constexpr bool INLINE = S::INLINE;
    static_assert(!INLINE || ((T >= 32) && (P::NPASS == 3)), "inline staging is written for rows carried by whole warps");
    constexpr bool TMA_IN = INLINE || ((T >= 32) && (P::NPASS == 3) && (ROWS >= 2));
    constexpr unsigned ROW_BYTES = (HALF ? NPHI / 2 : NPHI) * sizeof(double);
    cplx *stage_row = INLINE ? line : smem + ROWS * S::STRIDE + rho * L;
    unsigned long long *row_bar =
        reinterpret_cast<unsigned long long *>(smem + ROWS * S::STRIDE + (INLINE ? 0 : 16 * S::THREADS)) + rho;
    auto prefetch = [&](const int item) {
        const int f = item / items_per_field, i = (item % items_per_field) * ROWS + rho;
        const double *row = sigma + f * sigma_field_stride + (long)i * (HALF ? NPHI / 2 : NPHI);
        if constexpr (TMA_IN) {
            if (u == 0) {
                if constexpr (INLINE) fence_proxy_async();     // the line was last touched through the generic proxy
                bulk_load(stage_row, row, ROW_BYTES, row_bar);
            }
        } else {
            const cplx *x = reinterpret_cast<const cplx *>(row) + u;
#pragma unroll
            for (int jj = 0; jj < (HALF ? 8 : 16); ++jj) cp_async16(stage + jj * S::THREADS, x + T * jj);
            cp_async_commit();
        }
    };
    if constexpr (TMA_IN) {
        if (u == 0) mbar_init(row_bar, 1);
        CB::sync();
    }
    unsigned row_phase = 0;

    // Dependence on the preceding kernel of the stream (polargrav.cu decides, `early_load`):
    //   0  Sigma may be its output, and it may still read W: wait before anything else.
    //   1  Sigma is known to be complete, W is the buffer the preceding kernel reads: the first item is
    //      fetched ahead of the wait, nothing is stored before it.
    //   2  Sigma is complete AND W is a buffer no kernel in flight touches (the solver alternates between
    //      two): this kernel depends on nothing that runs before it.  It does all its work at once --
    //      filling the SMs the preceding kernel leaves idle in its last, uneven round -- and waits at its
    //      END, so that its own completion still implies that of everything before it.
    int item = block;
    if (early_load && item < n_items) prefetch(item);
    if (early_load < 2) pdl_wait();
    pdl_launch_dependents();
    if (!early_load && item < n_items) prefetch(item);
    auto row_scale = [&](const int it) {
        return (rscale != nullptr && it < n_items) ? __ldg(&rscale[(it % items_per_field) * ROWS + rho]) : 1.0;
    };
    double sc_next = row_scale(item);
    for (; item < n_items; item += nblocks) {
        const int f = item / items_per_field, i0 = (item % items_per_field) * ROWS;
        cplx v[16];
        const double sc = sc_next;
        sc_next = row_scale(item + nblocks);
        const Sync<T, S::THREADS, CB> sync(rho + 1);
        if constexpr (TMA_IN) {
            mbar_wait(row_bar, row_phase);
            row_phase ^= 1;
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) v[jj] = (HALF && jj >= 8) ? make_double2(0.0, 0.0) : stage_row[u + T * jj];
            if constexpr (INLINE) sync();      // the row's threads have taken their elements: pass A may rewrite the line
        } else {
            cp_async_wait_all();
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) v[jj] = (HALF && jj >= 8) ? make_double2(0.0, 0.0) : stage[jj * S::THREADS];
            if (item + nblocks < n_items) prefetch(item + nblocks);
        }
        if (rscale != nullptr) {
#pragma unroll
            for (int jj = 0; jj < 16; ++jj) { v[jj].x *= sc; v[jj].y *= sc; }
        }
        fwd_a<L, ROW>(v, line, bases, u);
        if constexpr (P::NPASS == 3) {
            sync();
            if constexpr (TMA_IN && !INLINE) {
                if (item + nblocks < n_items) prefetch(item + nblocks);   // the row's staging is free
            }
            fwd_b<L, ROW>(line, bases, u);
        }
        CB::sync();

        fwd_c_row<L>(v, smem + rp * S::STRIDE, b1, b2);
        if constexpr (INLINE) {
            CB::sync();       // every line has been read: the next item's rows may land in them
            if (item + nblocks < n_items) prefetch(item + nblocks);
        }
        cplx *Wf = W + f * w_field_stride + i0 + rp;
        auto store = [&](const int k, const cplx val) { Wf[(long)k * n_rows] = val; };
        if (!special) split_regular<L>(v, un1, q1, store);
        else split_special<L>(v, un1, un2, store);
        if constexpr (!INLINE) CB::sync();   // the lines are rewritten by the next item's pass A
    }
    if (early_load == 2) pdl_wait();
}
template <int NPHI, bool HALF = false>
__global__ void __launch_bounds__(RowShape<NPHI>::THREADS, RowShape<NPHI>::MIN_CTAS)
rows_fwd_kernel(const double *__restrict__ sigma, cplx *__restrict__ W, const cplx *__restrict__ tw,
                const double *__restrict__ rscale, const int n_rows, const int n_items, const long sigma_field_stride,
                const long w_field_stride, const int early_load)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    rows_fwd_body<NPHI, HALF, CtaBarrier>(sigma, W, tw, rscale, n_rows, n_items, sigma_field_stride, w_field_stride, early_load,
                                          blockIdx.x, gridDim.x, smem_raw);
}

// ---------------------------------------------------------------- a4 (phi part): rows inverse
// PERSISTENT like rows_fwd_kernel.  Prefetches the modes W[m][i] it needs in the row-fastest
// mapping (transposed access in runs of ROWS rows), re-packs them into the spectrum of the packed
// row, inverse pass C; the remaining passes with u fastest; multiplies row i by oscale_i
// (= r_i^{-1/2}) and stores Phi_i.
// HALF: only the first n_phi/2 reals of every output row are stored, in rows of that length (the crop of the x pass).
// modes a thread of the inverse row kernel needs, by prefetch slot (the order of modes_regular / modes_special)
template <int L>
__device__ __forceinline__ int mode_of_slot_regular(const int slot, const int q1)
{
    constexpr int NB = Plan<L, ROW>::NB;
    return (slot & 1) ? L - q1 - NB * (slot >> 1) : q1 + NB * (slot >> 1);
}
template <int L>
__device__ __forceinline__ int mode_of_slot_special(const int slot)
{
    constexpr int NB = Plan<L, ROW>::NB;
    if (slot < 8) return (slot & 1) ? L - NB * (slot >> 1) : NB * (slot >> 1);
    if (slot == 8) return L / 2;
    const int c = (slot - 9) >> 1;
    return ((slot - 9) & 1) ? L - NB / 2 - NB * c : NB / 2 + NB * c;
}

template <int NPHI, bool HALF, class CB>
__device__ __forceinline__ void rows_inv_body(const cplx *__restrict__ W, double *__restrict__ phi, const cplx *__restrict__ tw,
                                              const double *__restrict__ oscale, const int n_rows, const int n_items,
                                              const long w_field_stride, const long phi_field_stride, const int block,
                                              const int nblocks, unsigned char *smem_raw, const CUtensorMap *tmap)
{
    typedef RowShape<NPHI, true> S;
    typedef Plan<S::L, ROW> P;
    constexpr int L = S::L, T = S::T, ROWS = S::ROWS;
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);
    // INLINE (RowShape): the prefetched modes lie inside the lines; the next item's modes are requested once pass A has
    // taken the current item out of them and travel while pass A computes and the rows are stored
    constexpr bool INLINE = S::INLINE;
    constexpr bool TILE = S::TILE && !HALF;
    cplx *stage = smem + (INLINE ? 0 : ROWS * S::STRIDE) + threadIdx.x;

    const int tid = threadIdx.x;
    const int u = tid % T, rho = tid / T;
    const int rp = tid % ROWS, t = tid / ROWS;
    const int items_per_field = n_rows / ROWS;
    cplx *line = smem + rho * S::STRIDE;
    int b1, b2;
    bool special;
    row_blocks<L>(t, b1, b2, special);
    const int q1 = P::bin0(b1);
    const cplx un1 = __ldg(tw + P::TW_UN + (special ? 0 : q1));
    const cplx un2 = __ldg(tw + P::TW_UN + P::NB / 2);
    Bases<L, ROW> bases;
    bases.load(tw, u, false);

    auto prefetch = [&](const int item) {
        const int f = item / items_per_field, i0 = (item % items_per_field) * ROWS;
        const cplx *Wf = W + f * w_field_stride + i0 + rp;
        auto fetch = [&](const int slot, const int k) { cp_async16(stage + slot * S::THREADS, Wf + (long)k * n_rows); };
        if (!special) modes_regular<L>(q1, fetch);
        else modes_special<L>(fetch);
        cp_async_commit();
    };
    auto get = [&](const int slot) { return stage[slot * S::THREADS]; };

    // TILE: one tensor-map copy per item, completion on an mbarrier in the spare bytes behind the lines
    unsigned long long *tile_bar = reinterpret_cast<unsigned long long *>(smem + ROWS * S::STRIDE);
    cplx nyq = make_double2(0.0, 0.0);                 // mode L of row rp (special thread)
    unsigned phase = 0;
    auto request = [&](const int item) {               // thread 0
        const int f = item / items_per_field, i0 = (item % items_per_field) * ROWS;
        fence_proxy_async();                           // the lines were last touched through the generic proxy
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(tile_bar)), "r"(S::TILE_BYTES) : "memory");
        asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
                         smem_addr(smem)),
                     "l"(tmap), "r"(2 * i0), "r"(0), "r"(0), "r"(f), "r"(smem_addr(tile_bar))
                     : "memory");
    };
    auto load_nyq = [&](const int item) {
        const int f = item / items_per_field, i0 = (item % items_per_field) * ROWS;
        return W[f * w_field_stride + (long)L * n_rows + i0 + rp];
    };
    auto tile_at = [&](const int k) {                  // k < L:  [k mod RA][k / RA][row]
        return smem[((k % P::RA) * (L / P::RA) + k / P::RA) * ROWS + rp];
    };
    auto get_regular = [&](const int slot) { return tile_at(mode_of_slot_regular<L>(slot, q1)); };
    auto get_special = [&](const int slot) { return slot == 1 ? nyq : tile_at(mode_of_slot_special<L>(slot)); };
    if constexpr (TILE) {
        if (tid == 0) mbar_init(tile_bar, 1);
        CB::sync();
    }

    pdl_wait();                    // W is written by the preceding kernel of the stream
    pdl_launch_dependents();
    int item = block;
    if (item < n_items) {
        if constexpr (TILE) {
            if (tid == 0) request(item);
            if (special) nyq = load_nyq(item);
        } else {
            prefetch(item);
        }
    }
    for (; item < n_items; item += nblocks) {
        const int f = item / items_per_field, i0 = (item % items_per_field) * ROWS;
        cplx v[16];
        const double sc = __ldg(&oscale[i0 + rho]);
        if constexpr (TILE) {
            mbar_wait(tile_bar, phase);
            phase ^= 1;
            if (!special) merge_regular<L>(v, un1, get_regular);
            else merge_special<L>(v, un1, un2, get_special);
        } else {
            cp_async_wait_all();
            if (!special) merge_regular<L>(v, un1, get);
            else merge_special<L>(v, un1, un2, get);
        }
        if constexpr (INLINE) CB::sync();     // the modes live in the lines: all of them read before pass C writes
        else if (item + nblocks < n_items) prefetch(item + nblocks);
        inv_c_row<L>(v, smem + rp * S::STRIDE, b1, b2);
        CB::sync();

        if constexpr (P::NPASS == 3) {
            const Sync<T, S::THREADS, CB> sync(rho + 1);
            inv_b<L, ROW>(line, bases, u);
            sync();
        }
        inv_a_load<L, ROW>(v, line, u);
        if constexpr (INLINE) {
            CB::sync();       // the lines are free: the next item's modes may land in them
            if (item + nblocks < n_items) {
                if constexpr (TILE) {
                    if (tid == 0) request(item + nblocks);
                    if (special) nyq = load_nyq(item + nblocks);
                } else {
                    prefetch(item + nblocks);
                }
            }
        }
        inv_a_compute<L, ROW>(v, bases, u);
        cplx *y = reinterpret_cast<cplx *>(phi + f * phi_field_stride + (long)(i0 + rho) * (HALF ? NPHI / 2 : NPHI));
#pragma unroll
        for (int jj = 0; jj < (HALF ? 8 : 16); ++jj) y[u + T * jj] = make_double2(v[jj].x * sc, v[jj].y * sc);
        if constexpr (!INLINE) CB::sync();   // the lines are rewritten by the next item's pass C
    }
}
template <int NPHI, bool HALF = false>
__global__ void __launch_bounds__(RowShape<NPHI, true>::THREADS, RowShape<NPHI, true>::MIN_CTAS)
rows_inv_kernel(const cplx *__restrict__ W, double *__restrict__ phi, const cplx *__restrict__ tw,
                const double *__restrict__ oscale, const int n_rows, const int n_items, const long w_field_stride,
                const long phi_field_stride, const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    rows_inv_body<NPHI, HALF, CtaBarrier>(W, phi, tw, oscale, n_rows, n_items, w_field_stride, phi_field_stride, blockIdx.x,
                                          gridDim.x, smem_raw, &tmap);
}

// thread of a column transform that holds the mirror bins of thread u: bin0(partner) = T - bin0(u)  (u != 0)
template <int L>
__device__ __forceinline__ int col_partner(const int u)
{
    typedef Plan<L, COL> P;
    if constexpr (P::NPASS == 3) {
        const int q = P::T - ((u / P::RB) + P::RA * (u % P::RB));
        return (q % P::RA) * P::RB + q / P::RA;
    } else {
        return P::T - u;
    }
}

// ---------------------------------------------------------------- a3 + a4 (r part): columns
// One CTA owns MODES azimuthal modes; mode m is the column x[0..n_r) = W[m][.].  It is convolved
// with the Green's kernel over the radial lags, zero-padded to 2 n_r, and cropped back to n_r:
//   y[n] = (1/2N) sum_{k'<2N} Khat[k'] Xpad[k'] e^{+2 pi i k' n / 2N},   n < N = n_r.
// The 2N-point transform is carried by T = N/8 threads with 16 spectrum bins each, but a thread reads
// only 8 column elements (the upper half of the padded input is zero: pass A starts from a pruned
// radix-RA DFT, fft.cuh dft_zero_upper) and writes only 8 (the crop: the last inverse pass keeps the
// lower half of its outputs, idft_lower_half).  The padded array and the discarded half are never
// formed in memory (a3: multiply fused into the last forward pass; a4: inverse with fused crop).
// The body transforms mode group `group` of field `field` (group / field in the stand-alone kernel).
template <int NR, class CB>
__device__ __forceinline__ void cols_body(cplx *__restrict__ W, const double *__restrict__ Khat, const cplx *__restrict__ tw,
                                          const int n_modes, const long w_field_stride, const int group, const int field,
                                          unsigned char *smem_raw)
{
    typedef ColShape<NR> S;
    typedef Plan<S::L, COL> P;
    constexpr int L = S::L, T = S::T;
    cplx *smem = reinterpret_cast<cplx *>(smem_raw);

    const int tid = threadIdx.x;
    const int u = tid % T, ml = tid / T;
    const int m_raw = group * S::MODES + ml;
    const bool live = m_raw < n_modes;
    const int mode = live ? m_raw : n_modes - 1;
    cplx *line = smem + ml * S::STRIDE;
    cplx *col = W + field * w_field_stride + (long)mode * NR;

    // the Khat slices of this CTA's modes are contiguous: one bulk asynchronous copy into shared
    // memory, issued now and waited for after the forward transform
    double *kstage = reinterpret_cast<double *>(smem_raw + S::LINES);
    unsigned long long *kbar = reinterpret_cast<unsigned long long *>(smem_raw + S::LINES + S::STAGE);
    if (tid == 0) mbar_init(kbar, 1);
    CB::sync();
    if (tid == 0) {
        const int m0 = group * S::MODES;
        const int nm = (n_modes - m0 < S::MODES) ? n_modes - m0 : S::MODES;
        bulk_load(kstage, Khat + (long)m0 * S::KH, (unsigned)(nm * S::KH * sizeof(double)), kbar);
    }
    const double *kh = kstage + ml * S::KH;
    const int kq = (u == 0) ? T : col_partner<L>(u);      // bins c >= 8: entry (15 - c) T + kq
    pdl_wait();                    // W is written by the preceding kernel of the stream
    pdl_launch_dependents();

    cplx v[16];
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) v[jj] = col[u + T * jj];
    Bases<L, COL> bases;
    bases.load(tw, u, false);

    const Sync<T, S::THREADS, CB> sync(ml + 1);
    fwd_a_compute_zero_upper<L, COL>(v, bases, u);
    fwd_a_store<L, COL>(v, line, u);
    // Three-pass plans: pass B (in place) and pass C of a thread touch only slots of the 16 blocks
    // 16 (u/16) .. 16 (u/16) + 15, i.e. the B <-> C exchanges stay inside aligned groups of 16 threads, and a
    // warp-level barrier is enough for them.  Between the two CTA-wide barriers that are left the warps
    // of a transform run free (pass B, pass C, multiply, inverse C, inverse B), so that the FP64 phases
    // of some overlap the shared-memory phases of others.
    static_assert(P::NPASS < 3 || (P::GB == 1 && P::MA == 16 * P::RC), "B <-> C exchange must stay inside 16-thread groups");
    if constexpr (P::NPASS == 3) {
        sync();
        fwd_b<L, COL>(line, bases, u);
        __syncwarp();
    } else {
        sync();
    }
    fwd_c_col<L>(v, line, u);
    mbar_wait(kbar, 0);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const double kv = k < 8 ? kh[u + T * k] : kh[kq + T * (15 - k)];
        v[k].x *= kv;
        v[k].y *= kv;
    }
    // inv_c writes exactly the 16 slots this thread has just read: no barrier in between
    inv_c_col<L>(v, line, u);
    if constexpr (P::NPASS == 3) {
        __syncwarp();
        inv_b<L, COL>(line, bases, u);
    }
    sync();
    inv_a_load<L, COL>(v, line, u);
    inv_a_compute_lower_half<L, COL>(v, bases, u);
    if (live) {
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) col[u + T * jj] = v[jj];
    }
}
template <int NR>
__global__ void __launch_bounds__(ColShape<NR>::THREADS, ColShape<NR>::MIN_CTAS)
cols_kernel(cplx *__restrict__ W, const double *__restrict__ Khat, const cplx *__restrict__ tw, const int n_modes,
            const long w_field_stride)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cols_body<NR, CtaBarrier>(W, Khat, tw, n_modes, w_field_stride, blockIdx.x, blockIdx.y, smem_raw);
}

// ---------------------------------------------------------------- small grids: the whole solve in ONE launch
// For grids of up to 512 x 512 the three kernels above take 1-3 us each and a solve is bound by the host's launch rate
// (three launches, 7-14 us).  fused_solve_kernel runs the three bodies in one COOPERATIVE launch, separated by
// grid-wide barriers; W stays in the L2 in between.  Phase a2 / a4phi: CTA b takes the row items b, b + gridDim.x, ...
// with its first RowShape::THREADS threads; phase a3+a4r: CTA b takes mode group b (field b / groups) with its first
// ColShape::THREADS threads.  The host sizes the grid to max(items, groups * batch) and uses this kernel only when that
// many CTAs are resident at once (polargrav.cu, solve_fields).
template <int NR, int NPHI>
struct FusedShape {
    typedef RowShape<NPHI> RS;
    typedef ColShape<NR> CS;
    static_assert(RowShape<NPHI, true>::ROWS == RS::ROWS && RowShape<NPHI, true>::SMEM == RS::SMEM, "one row shape below 2048");
    static_assert(!RS::INLINE && NPHI >= 64 && NPHI <= 512 && NR >= 64 && NR <= 512, "fused path: 64 .. 512 per axis");
    static constexpr int THREADS = RS::THREADS > CS::THREADS ? RS::THREADS : CS::THREADS;
    static constexpr size_t SMEM = RS::SMEM > CS::SMEM ? RS::SMEM : CS::SMEM;
};
template <int NR, int NPHI>
__global__ void __launch_bounds__(FusedShape<NR, NPHI>::THREADS)
fused_solve_kernel(const double *__restrict__ sigma, double *__restrict__ phi, cplx *__restrict__ W,
                   const double *__restrict__ Khat, const cplx *__restrict__ tw_row, const cplx *__restrict__ tw_col,
                   const double *__restrict__ rscale, const double *__restrict__ oscale, const int batch,
                   const long field_stride, const long w_field_stride)
{
    typedef FusedShape<NR, NPHI> F;
    typedef typename F::RS RS;
    typedef typename F::CS CS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const int n_items = (NR / RS::ROWS) * batch;
    constexpr int n_modes = NPHI / 2 + 1;
    constexpr int groups = (n_modes + CS::MODES - 1) / CS::MODES;

    if (threadIdx.x < RS::THREADS)
        rows_fwd_body<NPHI, false, PartBarrier<RS::THREADS>>(sigma, W, tw_row, rscale, NR, n_items, field_stride,
                                                            w_field_stride, 0, blockIdx.x, gridDim.x, smem_raw);
    grid.sync();
    fence_proxy_async();           // the Khat slices arrive by bulk copy in shared memory the row phase has used
    if ((int)blockIdx.x < groups * batch && threadIdx.x < CS::THREADS)
        cols_body<NR, PartBarrier<CS::THREADS>>(W, Khat, tw_col, n_modes, w_field_stride, blockIdx.x % groups,
                                                blockIdx.x / groups, smem_raw);
    grid.sync();
    if (threadIdx.x < RS::THREADS)
        rows_inv_body<NPHI, false, PartBarrier<RS::THREADS>>(W, phi, tw_row, oscale, NR, n_items, w_field_stride,
                                                            field_stride, blockIdx.x, gridDim.x, smem_raw, nullptr);
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

// Column pass of the kernel spectrum (one-time, a1).  WK[m][0..2N) is azimuthal mode m of the padded
// kernel Kpad (2N rows, from rows_fwd_kernel).  Its 2N-point forward transform is taken with the plan
// cols_kernel uses (no pruning here: all 2N lags are populated), and the real part is scaled and stored
// in the order cols_kernel holds the bins:   Khat[m][c T + u] = scale Re X[bin0(u) + T c].
// (K is even in both lags, so X is real up to rounding.)
template <int NR>
__global__ void __launch_bounds__(NR / 8)
khat_cols_kernel(const cplx *__restrict__ WK, double *__restrict__ Khat, const cplx *__restrict__ tw, const double scale)
{
    constexpr int L = 2 * NR;
    typedef Plan<L, COL> P;
    constexpr int T = P::T;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx *line = reinterpret_cast<cplx *>(smem_raw);

    const int u = threadIdx.x;
    const int m = blockIdx.x;                         // mode 0..H
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
    double *kh = Khat + (long)m * (L / 2 + 2);          // symmetric half, ColShape<NR>::KH doubles per mode
#pragma unroll
    for (int k = 0; k < 8; ++k) kh[u + T * k] = scale * v[k].x;
    if (u == 0) { kh[8 * T] = scale * v[8].x; kh[8 * T + 1] = 0.0; }
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
    extern __shared__ __align__(128) unsigned char smem_raw[];
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

// Register-tiled variant for n_phi >= 256.  For one ring pair the sum over j' is a cyclic correlation of the
// source ring w[j'] with the pair kernel g[(j - j') mod n_phi]: a thread that owns R CONSECUTIVE targets
// j0 .. j0+R-1 and walks over the sources in blocks of 8 needs, per block, 8 values of w and the R + 7 kernel
// values of the lags j0 - j'0 - 7 .. j0 - j'0 + R - 1 -- a window that slides down by 8 from block to block, so
// that only 8 new values are loaded per block: 8 R FMAs for 8 + 8 shared-memory doubles, against two loads per
// FMA in direct_kernel.  The kernel is stored twice over (lags 0 .. 2 n_phi - 1) so that a window never wraps,
// in groups of R padded to R + 2 doubles (lane stride an odd number of 16-byte units: conflict-free loads).  Same arithmetic per
// pair and the same two-level accumulation as direct_kernel; the summation order within a ring differs.
template <int R>
__global__ void __launch_bounds__(128)
direct_tiled_kernel(const double *__restrict__ sigma, double *__restrict__ phi, const double *__restrict__ r,
                    const double *__restrict__ dA, const double *__restrict__ s2, const int n_r, const int n_phi,
                    const double eps2, const int ring0, const long sigma_field_stride, const long phi_field_stride)
{
    static_assert(R % 8 == 0 && R >= 8 && R <= 16, "targets per thread");
    constexpr int NG = R / 8 + 1;                       // groups of 8 lags in the window
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *w = reinterpret_cast<double *>(smem_raw);   // [n_phi] Sigma of the source ring
    double *g = w + n_phi;                              // [2 n_phi / R][R + 2] pair kernel by lag, twice over
    auto slot = [](const int lag) { return (lag / R) * (R + 2) + lag % R; };
    const int i = ring0 + blockIdx.x;
    const double ri = r[i], hi = sqrt(dA[i]);
    const double *sg = sigma + blockIdx.y * sigma_field_stride;
    const int nt = blockDim.x;
    const int j0 = R * threadIdx.x;

    double acc[R];
#pragma unroll
    for (int q = 0; q < R; ++q) acc[q] = 0.0;

    for (int ip = 0; ip < n_r; ++ip) {
        const double rp = r[ip], ap = dA[ip];
        const double dr = ri - rp;
        const double base = fma(dr, dr, eps2 * hi * sqrt(ap));
        const double rr4 = 4.0 * ri * rp;
        __syncthreads();
        for (int l = threadIdx.x; l < n_phi; l += nt) {
            w[l] = sg[(long)ip * n_phi + l];
            const double gv = rsqrt(fma(rr4, s2[l], base));
            g[slot(l)] = gv;
            g[slot(l + n_phi)] = gv;
        }
        __syncthreads();
        double ring[R];
#pragma unroll
        for (int q = 0; q < R; ++q) ring[q] = 0.0;
        // window gw[k] = g_ext[n_phi + j0 - jp0 - 8 + k], k < 8 NG; target j0 + q, source jp0 + t: lag index q - t + 8
        double gw[8 * NG];
        const int lag0 = n_phi + j0 - 8;                     // first lag of the window for jp0 = 0
#pragma unroll
        for (int k = 1; k < NG; ++k) {                       // groups above the lowest one, for jp0 = 0
            const double2 *gp = reinterpret_cast<const double2 *>(g + slot(lag0 + 8 * k));
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const double2 t2 = gp[h];
                gw[8 * k + 2 * h] = t2.x;
                gw[8 * k + 2 * h + 1] = t2.y;
            }
        }
        for (int jp0 = 0; jp0 < n_phi; jp0 += 8) {
            const double2 *gp = reinterpret_cast<const double2 *>(g + slot(lag0 - jp0));
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const double2 t2 = gp[h];
                gw[2 * h] = t2.x;
                gw[2 * h + 1] = t2.y;
            }
            const double2 *wp = reinterpret_cast<const double2 *>(w + jp0);
            double wv[8];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const double2 t2 = wp[h];
                wv[2 * h] = t2.x;
                wv[2 * h + 1] = t2.y;
            }
#pragma unroll
            for (int t = 0; t < 8; ++t)
#pragma unroll
                for (int q = 0; q < R; ++q) ring[q] = fma(wv[t], gw[q - t + 8], ring[q]);
            // slide the window: the groups move up by one
#pragma unroll
            for (int k = 8 * NG - 1; k >= 8; --k) gw[k] = gw[k - 8];
        }
#pragma unroll
        for (int q = 0; q < R; ++q) acc[q] = fma(ap, ring[q], acc[q]);
    }
    double *out = phi + blockIdx.y * phi_field_stride + (long)blockIdx.x * n_phi + j0;
#pragma unroll
    for (int q = 0; q < R; ++q) out[q] = -acc[q];
}

}  // namespace pgk
