/*
 * polargrav.h -- C ABI of libpolargrav.so (B200 / sm_100a only).
 *
 * Gravitational potential of a razor-thin disk on a log-polar grid,
 *
 *     Phi_ij = -G * sum_{i'j'} Sigma_{i'j'} dA_{i'} / sqrt(d2(i,j;i',j')),      G = 1,
 *     d2     = (r_i - r_i')^2 + 4 r_i r_i' sin^2((phi_j - phi_j')/2) + eps^2 h_i h_i',
 *
 * evaluated as a zero-padded FFT convolution on the GPU ("the convolution method for
 * solving potential fields"; "FFT operations" are the GPU-resident work,
 * PAPER.md:19).  PAPER.md prints no formula; the sum is BASELINE.json north_star's and
 * every convention is a reading listed in DESIGN.md section 3 (A1..A8):
 *
 *     edges   re_i = r_in (r_out/r_in)^(i/n_r);  centres r_i = sqrt(re_i re_{i+1}) = r_in exp((i+1/2) du)
 *     phi_j   = (j+1/2) dphi,  dphi = 2 pi / n_phi,  du = ln(r_out/r_in)/n_r
 *     dA_i    = (re_{i+1}^2 - re_i^2) dphi / 2 = r_i^2 sinh(du) dphi;   h_i = sqrt(dA_i)
 *     the self term (i'=i, j'=j) is included: it contributes -Sigma_ij h_i / eps.
 *
 * The seam is a C ABI on purpose: the paper's own conclusion is that a C binding is the
 * robust boundary between tool-chains, with addresses handed across once and no hidden
 * copies (App. A :397-400), and that the CUDA side should own the pinned
 * host memory (Fig. 4 :202).
 *
 * Conventions for every call
 *   - Arrays are C order [batch][n_r][n_phi], phi fastest, contiguous, IEEE fp64.  PG_MEM_DEVICE arrays must
 *     be 16-byte aligned (the kernels move them as 16-byte vectors); a misaligned device pointer is rejected
 *     with PG_ERR_INVALID_ARG.  Host arrays need 8-byte alignment only.
 *   - A call leaves the caller's current CUDA device as it found it.
 *   - No C++ types, no exceptions, never abort(): every call returns a pg_status;
 *     pg_last_error() gives the text of the last failure on that solver.
 *   - There is NO CPU fallback and no alternative backend: without a CUDA device of
 *     compute capability 10.x pg_create* fails with PG_ERR_UNSUPPORTED / PG_ERR_CUDA.
 *   - One solver per host thread at a time; distinct solvers are independent.
 */
#ifndef POLARGRAV_H
#define POLARGRAV_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pg_solver pg_solver; /* opaque */

typedef enum {
    PG_OK = 0,
    PG_ERR_INVALID_ARG = -1, /* null pointer, r_in<=0, r_out<=r_in, eps<=0, batch out of range */
    PG_ERR_UNSUPPORTED = -2, /* n_r/n_phi not a power of two in [PG_MIN_N, PG_MAX_N], device not sm_100 */
    PG_ERR_CUDA = -3,        /* a CUDA call failed; text in pg_last_error */
    PG_ERR_NOMEM = -4,       /* host or device allocation failed */
    PG_ERR_STATE = -5        /* pg_potential* before any pg_set_density */
} pg_status;

/* Where a caller-owned buffer lives. */
typedef enum {
    PG_MEM_HOST = 0,        /* pageable host memory: staged through the solver's pinned buffer */
    PG_MEM_HOST_PINNED = 1, /* page-locked host memory (e.g. from pg_host_alloc): async copy, no staging */
    PG_MEM_DEVICE = 2       /* device memory on the solver's device */
} pg_memspace;

#define PG_MIN_N 32
#define PG_MAX_N 2048
#define PG_MAX_LANES 4 /* PG_OPT_LANES: independent resident solves in flight */

/*
 * pg_create / pg_create_ex -- build a solver for one grid (north_star: pg_create(grid: N_r, N_phi,
 * r_in, r_out, eps)).  One-time work (row a1 of DESIGN.md): Green's kernel
 *     K(k,l) = [4 sinh^2(k du/2) + 4 sin^2(l dphi/2) + eta^2]^(-1/2),  eta^2 = eps^2 sinh(du) dphi,
 * on the lags k in (-n_r, n_r), l in [0, n_phi), its 2-D FFT on the 2 n_r x n_phi padded lag grid
 * (real, because K is even in both lags), with -G sinh(du) dphi and the FFT normalisation folded in.
 *
 *   out        receives the solver; *out is set to NULL on failure.
 *   n_r,n_phi  powers of two in [PG_MIN_N, PG_MAX_N].
 *   r_in,r_out inner / outer EDGE of the grid, 0 < r_in < r_out.
 *   eps        dimensionless softening in units of the local cell size h = sqrt(dA), > 0.
 *   max_batch  largest `batch` later calls may pass (>= 1); workspace scales with it.
 *   device     CUDA device ordinal, or -1 for the current device.
 *   cuda_stream a cudaStream_t (borrowed, may be NULL = the legacy default stream).  All work
 *              of this solver is enqueued on it.
 * Ownership: the solver owns the spectrum, tables, workspace and pinned staging buffers.
 */
pg_status pg_create(pg_solver **out, int n_r, int n_phi, double r_in, double r_out, double eps);
pg_status pg_create_ex(pg_solver **out, int n_r, int n_phi, double r_in, double r_out, double eps,
                       int max_batch, int device, void *cuda_stream);

/*
 * pg_set_density -- hand the surface density Sigma[batch][n_r][n_phi] to the solver.
 *   PG_MEM_DEVICE      : BORROWED, no copy, 16-byte aligned.  Must stay valid and unmodified until the work of
 *                        the following pg_potential* call has completed on the stream.
 *   PG_MEM_HOST_PINNED : cudaMemcpyAsync to an owned device buffer; returns after enqueue; the
 *                        caller must not modify `sigma` until the stream has passed the copy.
 *   PG_MEM_HOST        : memcpy into the owned pinned staging buffer, then cudaMemcpyAsync; returns
 *                        once `sigma` may be reused (row a6; pinned staging per PAPER.md:97-101,:119).
 * 1 <= batch <= max_batch.  NaN/Inf/negative values are not checked and propagate (linearity).
 */
pg_status pg_set_density(pg_solver *s, const double *sigma, int batch, pg_memspace where);

/*
 * pg_potential -- FFT-convolution solve (rows a2-a4): writes Phi[batch][n_r][n_phi] for the density
 * last set; `batch` must equal that call's batch.
 *   PG_MEM_DEVICE / PG_MEM_HOST_PINNED : returns after enqueue (use pg_synchronize or sync the stream).
 *   PG_MEM_HOST                        : blocks until `phi` is filled.
 * For host memspaces with batch > 1 the copies of one field overlap the solves of its neighbours
 * (separate copy stream + events).  `phi` may not overlap the density: a PG_MEM_DEVICE `phi` that overlaps a
 * PG_MEM_DEVICE density is rejected with PG_ERR_INVALID_ARG (no in-place solves).
 */
pg_status pg_potential(pg_solver *s, double *phi, int batch, pg_memspace where);

/*
 * pg_potential_direct -- tiled all-pairs direct summation on the GPU (row a5), evaluated from the
 * coordinates, used as an on-device cross-check of pg_potential.  O((n_r n_phi)^2): seconds at
 * 512^2, not meant for production.  Same argument rules as pg_potential.  NOT a fallback: nothing
 * in the library calls it.
 * pg_potential_direct_rings -- the same for target rings [ring0, ring0+n_rings) of field 0 only;
 * `phi` receives [n_rings][n_phi].
 */
pg_status pg_potential_direct(pg_solver *s, double *phi, int batch, pg_memspace where);
pg_status pg_potential_direct_rings(pg_solver *s, double *phi, int ring0, int n_rings, pg_memspace where);

/* ---------------------------------------------------------------- variants of the path
 * Not in the paper (PAPER.md:267 only names the convolution method); readings N1 and N2 of DESIGN.md section 3.
 *
 * pg_set_softening -- which cell lends its size to the softening length of a pair (field ring i, source ring i'):
 *     PG_SOFT_SYMMETRIC  eps^2 h_i h_i'   (default; the pair kernel is even in the radial lag, its spectrum real)
 *     PG_SOFT_FIELD      eps^2 h_i^2      (softening length of the field cell)
 *     PG_SOFT_SOURCE     eps^2 h_i'^2     (softening length of the source cell)
 * All three depend on index differences only (eps is dimensionless), so the FFT convolution stays exact; for the
 * last two the kernel spectrum is complex and the column pass multiplies complex by complex.  Blocking: it
 * synchronises the stream and rebuilds the spectrum.  Affects pg_potential and pg_acceleration; the direct kernel
 * (pg_potential_direct*) always uses the symmetric form.
 *
 * pg_acceleration -- the softened pair acceleration of the density last set, in the polar basis of the field cell,
 *     a_r   = - sum Sigma' dA' (r - r' cos(phi - phi')) / d2^(3/2),
 *     a_phi = - sum Sigma' dA'  r' sin(phi - phi')      / d2^(3/2),      d2 as in the header of this file,
 * with the softening length of each pair held fixed (the force law hydro codes apply; equal to -grad Phi for
 * PG_SOFT_SOURCE).  Two more convolutions that share the forward transform of the density with each other.
 * a_r, a_phi: [batch][n_r][n_phi] each, same memspace; they may overlap neither each other nor the density.
 * PG_MEM_DEVICE returns after enqueue; host memspaces block until both arrays are filled.  The two kernel
 * spectra are built on the first call (and again after pg_set_softening). */
typedef enum { PG_SOFT_SYMMETRIC = 0, PG_SOFT_FIELD = 1, PG_SOFT_SOURCE = 2 } pg_softening;
pg_status pg_set_softening(pg_solver *s, pg_softening mode);
pg_status pg_acceleration(pg_solver *s, double *a_r, double *a_phi, int batch, pg_memspace where);

/*
 * pg_potential_series -- `count` single-field solves enqueued by ONE host call (time series
 * and ensembles on small grids are bound by the host's per-call cost, not by the GPU):
 *     Phi_k = potential of Sigma_k,   Sigma_k = sigma + k * stride,  Phi_k = phi + k * stride,   k = 0 .. count-1,
 * exactly as `count` pairs  pg_set_density(s, Sigma_k, 1, PG_MEM_DEVICE); pg_potential(s, Phi_k, 1, PG_MEM_DEVICE)
 * would, in that order, with the same kernels (bit-identical results) and the same ordering rules: on the solver's
 * stream, or -- with PG_OPT_LANES >= 2 and PG_OPT_DENSITY_STABLE -- dealt out to the lanes and complete after
 * pg_flush / pg_synchronize.  The fields are independent of each other (Sigma_k is not read from Phi_(k-1)).
 *   sigma, phi  device memory of the solver's device, 16-byte aligned; the two ranges of count * stride doubles may
 *               not overlap.   stride  in doubles, even, >= n_r * n_phi.   count >= 1 (not limited by max_batch).
 * Returns after enqueue; afterwards the density last set is Sigma_(count-1) with batch 1.
 */
pg_status pg_potential_series(pg_solver *s, const double *sigma, double *phi, int count, size_t stride);

/* pg_destroy -- frees everything the solver owns. pg_destroy(NULL) is a no-op returning PG_OK. */
pg_status pg_destroy(pg_solver *s);

/* ---------------------------------------------------------------- the one call that never allocates
 * pg_potential_direct_static -- the direct summation of pg_potential_direct (row a5; same kernels, same grid
 * conventions, symmetric softening, G = 1) for ONE field, with no solver object and no allocation of any kind.
 *
 * Who it is for.  Everything else in this header starts from pg_create*, which takes device memory (tables, the
 * spectrum, workspaces -- and pg_potential may add more on first use: a second workspace under
 * PG_OPT_DENSITY_STABLE, one pair per lane, staging buffers for host memspaces).  Some programs cannot give it any:
 *   - a simulation that sized its own arena (or a framework's caching allocator) to take all free HBM at start-up:
 *     a cudaMalloc issued later simply fails;
 *   - a job held to a fixed device-memory budget (a MIG slice or an MPS limit sized to the application);
 *   - a plug-in or callback that is handed device pointers by its host program and has no licence to create
 *     device buffers of its own.
 * Such a caller can still cross-check a potential it holds, or solve a small grid outright (the sum costs
 * (n_r n_phi)^2 pair terms: microseconds at 64^2, about a second at 2048^2), by passing its own two arrays.
 *
 * How.  Beyond Sigma and Phi the kernel reads three grid tables (r_i, dA_i, sin^2(pi l / n_phi)).  For this call
 * they live in a fixed array inside the library image: 3 * PG_STATIC_MAX_N doubles = 48 KiB, present on every GPU
 * that loads the library until the process exits, whether or not the call is ever made.  The tables are computed
 * on the host exactly as pg_create* computes them and sent to that array on `cuda_stream` ahead of the kernel, so
 * the result equals pg_potential_direct's for the same grid.  The call uses no cudaMalloc, cudaFree,
 * cudaHostAlloc or other allocating routine, and creates no stream or event.
 *
 *   sigma, phi   device pointers on `device`, [n_r][n_phi], 16-byte aligned, not overlapping; borrowed for the
 *                duration of the enqueued work.
 *   n_r, n_phi   powers of two in [PG_MIN_N, PG_STATIC_MAX_N]; anything larger does not fit the fixed array and is
 *                refused with PG_ERR_UNSUPPORTED (the text names the limit).  r_in, r_out, eps as in pg_create.
 *   device       CUDA device ordinal, or -1 for the current device.  cuda_stream: borrowed, NULL = default stream.
 * Returns after enqueue; the tables leave from ordinary (pageable) host memory, so the host may first wait for
 * work already on the stream.  Errors: the status, with the text in pg_last_error(NULL).
 *
 * One-time set-up.  The first call on each device asks the runtime for the device address of the fixed array
 * (cudaGetSymbolAddress, with that device current) and checks the device is sm_100.  Make that first call before
 * any stream capture is begun.
 *
 * Sharing.  There is ONE array per GPU, used by every call from every thread and stream, and it keeps whatever the
 * last call wrote.  Nothing in it has to start at zero: each call rewrites every entry its kernel will read.
 * Calls on the same stream are ordered and safe.  Calls whose GPU work may overlap -- different streams with no
 * event between them, different host threads -- race on the tables: one call's upload can land under the other's
 * running kernel.  Order them (one stream, or an event from each call to the next). */
#define PG_STATIC_MAX_N 2048
pg_status pg_potential_direct_static(const double *sigma, double *phi, int n_r, int n_phi, double r_in,
                                     double r_out, double eps, int device, void *cuda_stream);

/* ---------------------------------------------------------------- helpers */

/* Grid tables (host pointers, any may be NULL): r[n_r] cell-centre radii, phi[n_phi] cell-centre
 * azimuths, cell_area[n_r] exact sector areas.  Callers never need to recompute conventions. */
pg_status pg_grid(const pg_solver *s, double *r, double *phi, double *cell_area);

/* Replace the (borrowed) stream; synchronises the old one first. */
pg_status pg_set_stream(pg_solver *s, void *cuda_stream);

/* Options (off by default).
 *   PG_OPT_DENSITY_STABLE  The caller promises that a PG_MEM_DEVICE density is complete in memory by the
 *       time pg_potential is called: it is not being written by work still in flight on the stream (it was
 *       produced before a synchronisation, or on another stream that has been joined).  The first forward
 *       kernel may then fetch it while the previous kernel of the stream is still draining (programmatic
 *       dependent launch; the library itself checks that it does not alias the potential that the
 *       previous solve ON THE SAME STREAM -- of this or of any other solver of the process -- is still writing; the
 *       record is kept per stream, so solves on other streams in between do not erase it), and, working alternately in two copies of its intermediate spectrum
 *       (a second workspace of max_batch * (n_phi/2 + 1) * n_r * 16 bytes is allocated on first use), runs
 *       entirely alongside the tail of the previous solve's last kernel.  Time series and batches with
 *       densities resident in HBM (the case bench.py times) qualify; a density written by the caller's
 *       kernel enqueued just before does not.
 *   PG_OPT_LANES  (1 .. PG_MAX_LANES, default 1)  Throughput mode for INDEPENDENT resident solves (a batch dealt out one field at a
 *       time, a time series whose steps do not feed each other).  With n >= 2, and PG_OPT_DENSITY_STABLE set, consecutive
 *       PG_MEM_DEVICE pg_potential calls go in turn to n internal streams, so that n solves are in flight and
 *       the tail and hand-over bubbles of one solve's kernels are filled by the other's.  This CHANGES THE ORDERING
 *       CONTRACT of those calls: their work is not on the solver's stream any more; it is complete after pg_synchronize,
 *       or, stream-ordered, after pg_flush (which makes the solver's stream wait for all lanes).  The caller promises,
 *       for every such call, that the density is complete in memory and that neither the density nor `phi` is read or
 *       written by anything else in flight -- work of the caller or the solve of the call before -- until then.
 *       Host memspaces, pg_profile passes, pg_acceleration and non-symmetric softening keep using the solver's stream.
 *       Setting the option synchronises.  Costs one more pair of W buffers per lane.
 *   PG_OPT_FUSED  (0 or 1, default 1)  Grids of 64 .. 512 cells per axis are solved by ONE cooperative kernel launch
 *       (the three steps a2, a3+a4r, a4phi separated by grid-wide barriers, the spectrum staying in the L2) instead of
 *       three launches, as long as the batch is small enough for all its CTAs to be resident at once: such solves are
 *       bound by the host's launch rate, not by the GPU.  Same arithmetic, bit-identical results.  0 forces the
 *       three-kernel path (which pg_profile passes, pg_acceleration and non-symmetric softening always take).
 *       Trade-off: the fused launch is what makes several small solves in flight (PG_OPT_LANES, host-staged pipelines)
 *       cheap -- one launch each -- but ONE solve takes longer in it (two grid-wide barriers: 9.6 / 13.9 / 16.3 us at
 *       64^2 / 256^2 / 512^2) than in three kernels chained by programmatic dependent launch once the launch queue is
 *       full (8.5 / 8.7 / 10.2 us); a long time series of DEPENDENT small solves on one stream may prefer 0.
 * Returns PG_ERR_INVALID_ARG for an unknown option or value. */
typedef enum { PG_OPT_DENSITY_STABLE = 1, PG_OPT_LANES = 2, PG_OPT_FUSED = 3 } pg_option;
pg_status pg_set_option(pg_solver *s, pg_option option, int value);
/* Stream-ordered join of the lanes of PG_OPT_LANES: work enqueued on the solver's stream after this call runs after
 * every solve enqueued before it.  No-op with one lane.  Returns after enqueue. */
pg_status pg_flush(pg_solver *s);
/* Block until all work enqueued by this solver has completed. */
pg_status pg_synchronize(pg_solver *s);

/* Page-locked host memory owned by the CUDA side (Fig. 4).  Needs a CUDA device. */
pg_status pg_host_alloc(void **p, size_t bytes);
pg_status pg_host_free(void *p);

/* Per-kernel device timing.  When enabled, CUDA events are recorded around each kernel of
 * pg_potential on the solver's stream; pg_kernel_times returns the accumulated milliseconds and
 * launch counts since the last pg_profile(s, 1) call (it synchronises the stream).
 *   index 0: a2 row forward (pre-weight + phi R2C)   1: a3+a4r column pass (FFT, x K^, IFFT, crop)
 *   index 2: a4 row inverse (phi C2R + post-scale)                                              */
#define PG_NUM_KERNELS 3
pg_status pg_profile(pg_solver *s, int enable);
pg_status pg_kernel_times(pg_solver *s, double ms[PG_NUM_KERNELS], long launches[PG_NUM_KERNELS]);

/* Number of kernels this library has launched on behalf of `s` since creation. */
long pg_launch_count(const pg_solver *s);

/* Algorithmic HBM bytes of one pg_potential call of `batch` fields, and of
 * kernel `index` alone (same indices as pg_kernel_times). */
double pg_algorithmic_bytes(const pg_solver *s, int batch);
double pg_kernel_algorithmic_bytes(const pg_solver *s, int index, int batch);

const char *pg_status_string(pg_status st);
const char *pg_last_error(const pg_solver *s); /* s may be NULL: last error of a failed pg_create* */
const char *pg_version(void);

/* ---------------------------------------------------------------- one 3-D Cartesian mesh level
 * The paper's own per-GPU workload: "the convolution method for solving potential fields on nested grids in three
 * dimensions" on ONE uniform mesh level of n^3 cells, n = 64 or 128 in the paper's runs.
 * The method's reference ([13]) is not available and PAPER.md prints no formula; readings C1-C4 of
 * DESIGN.md section 3:
 *     Phi_c = -G h^3 sum_{c'} rho_{c'} g(c - c'),  g(d) = 1/(h |d|) (cells as point masses), g(0) = S / h with
 *     S = integral of 1/|x| over the unit cube = 3 ln(2 + sqrt 3) - pi/2,  G = 1,  h = box / n,
 * over the n^3 cells of the mesh only (isolated boundary: zero padding to (2n)^3, none of which is ever stored in
 * y or z).  Arrays are [z][y][x], x fastest, contiguous fp64; PG_MEM_DEVICE arrays 16-byte aligned.
 *   pg3_create        n in {32, 64, 128, 256}; box > 0 is the edge length of the mesh; device -1 = current; the stream
 *                     is borrowed.  One-time work: the real spectrum of g on the (2n)^3 lag grid.
 *   pg3_set_density   PG_MEM_DEVICE: borrowed until the following pg3_potential has completed; host memspaces are
 *                     copied to an owned device buffer (PG_MEM_HOST blocks until `rho` may be reused).
 *   pg3_potential     PG_MEM_DEVICE / PG_MEM_HOST_PINNED return after enqueue; PG_MEM_HOST blocks until filled.
 *                     `phi` may not overlap a device density.  PG_ERR_STATE before any pg3_set_density.
 * Nested levels and their exchange across GPUs (Fig. 8) are the pg3n_* calls below. */
typedef struct pg3_solver pg3_solver; /* opaque */
pg_status pg3_create(pg3_solver **out, int n, double box, int device, void *cuda_stream);
pg_status pg3_set_density(pg3_solver *s, const double *rho, pg_memspace where);
pg_status pg3_potential(pg3_solver *s, double *phi, pg_memspace where);
pg_status pg3_synchronize(pg3_solver *s);
pg_status pg3_destroy(pg3_solver *s); /* pg3_destroy(NULL) is a no-op returning PG_OK */
long pg3_launch_count(const pg3_solver *s);
double pg3_algorithmic_bytes(const pg3_solver *s);
const char *pg3_last_error(const pg3_solver *s); /* s may be NULL: last error of a failed pg3_create */

/* ---------------------------------------------------------------- nested 3-D mesh levels
 * The paper's distributed scheme: depth D nested meshes of n^3 cells with a common centre, each half the edge of the
 * one before, "each nested mesh ... allocated one GPU" (Fig. 8 :306).  PAPER.md prints no coupling
 * scheme (it is in ref. [13], :376, not available); readings M1-M6 of DESIGN.md section 3:
 *   M1  box_l = box0 / 2^l; level l+1 covers the central (n/2)^3 cells [n/4, 3n/4)^3 of level l, 2 cells per parent cell.
 *   M2  restriction, finest first: the central (n/2)^3 cells of rho_l are replaced by the means of their 8 children.
 *   M3  own_l = Phi[rho_l] and, for l < D-1, out_l = Phi[rho_l with the central cells zeroed], each the isolated
 *       single-level convolution pg3_potential computes (readings C1-C4).
 *   M4  E_0 = 0, E_(l+1) = P[out_l + E_l]: the potential of everything outside box_(l+1).
 *   M5  P: trilinear interpolation between the parent's cell centres onto the child's (weights 3/4, 1/4); the parent
 *       cells [n/4 - 1, 3n/4]^3 -- (n/2 + 2)^3 values -- cross the level boundary.
 *   M6  Phi_l = own_l + E_l.
 * One pg3n_level per level; all calls enqueue on the level's (borrowed) stream and return, except PG_MEM_HOST
 * copies, which block.  The two messages between neighbouring levels are plain device arrays the CALLER moves: by
 * pointer when both levels live on one GPU, by NCCL send / recv (NVLink) when each level has its own GPU
 * (paper_2409_02294_b200/nested.py does either).  Call order for one solve:
 *   pg3n_set_density on every level                          (copied: M2 rewrites the centre)
 *   l = D-1 .. 1:  pg3n_restrict(l, msg) ; pg3n_absorb(l-1, msg)              msg: (n/2)^3 doubles, device
 *   every level:   pg3n_solve                                                  (independent across levels)
 *   l = 0 .. D-1:  pg3n_add_exterior(l, l ? halo : NULL) ; if l < D-1: pg3n_pack_exterior(l, halo)
 *                                                                              halo: (n/2 + 2)^3 doubles, device
 *   pg3n_potential on every level.
 * n in {32, 64, 128, 256}; device pointers 16-byte aligned.  PG_ERR_STATE for calls out of order or on the wrong end
 * of the hierarchy (restrict on level 0, absorb / pack on the finest level).
 *
 * One-sided exchange.  The paper's images move level-boundary data by one-sided transfers: "one image is allowed to
 * access the data from another without any action from the target image" (section 2.5).  The same here:
 * every level owns two INBOXES (device arrays of the two message sizes); a neighbour opens them -- by CUDA IPC handle
 * from another process / GPU (peer access over NVLink is enabled on open), or by plain pointer inside one process --
 * and the kernels of pg3n_restrict / pg3n_pack_exterior then write their message STRAIGHT INTO the neighbour's inbox:
 * the transfer is the kernel's own stores, no copy kernel, no staging.  Pass NULL where the calls above take a message
 * pointer:  pg3n_restrict(l, NULL) puts into the parent's MEAN inbox, pg3n_absorb(l, NULL) reads this level's MEAN
 * inbox, pg3n_pack_exterior(l, NULL) puts into the child's HALO inbox, pg3n_add_exterior(l > 0, NULL) reads this
 * level's HALO inbox.  The library does not signal: the sender's stream must have completed the putting kernel before
 * the receiver is told to go on (nested.py: event synchronise, then a one-byte message), and the receiver must have
 * consumed an inbox before the next put into it (guaranteed by the order of the two chains within a solve).
 *   pg3n_inbox_export  allocates the inbox on first use; returns its IPC handle (64 bytes; may be NULL) and its
 *                      device address (may be NULL).  PG_ERR_STATE if the level receives no such message.
 *   pg3n_peer_open     opens the NEIGHBOUR's inbox from its handle: MEAN = the parent's (target of pg3n_restrict),
 *                      HALO = the child's (target of pg3n_pack_exterior).  pg3n_peer_set: same, by device pointer.
 */
#define PG_IPC_HANDLE_BYTES 64
typedef enum { PG3N_INBOX_MEAN = 0, PG3N_INBOX_HALO = 1 } pg3n_inbox;
typedef struct pg3n_level pg3n_level; /* opaque */
pg_status pg3n_create(pg3n_level **out, int n, double box0, int level, int depth, int device, void *cuda_stream);
pg_status pg3n_set_density(pg3n_level *s, const double *rho, pg_memspace where);
pg_status pg3n_restrict(pg3n_level *s, double *child_mean_out);
pg_status pg3n_absorb(pg3n_level *s, const double *child_mean);
pg_status pg3n_solve(pg3n_level *s);
pg_status pg3n_add_exterior(pg3n_level *s, const double *parent_halo);
pg_status pg3n_pack_exterior(pg3n_level *s, double *halo_out);
pg_status pg3n_potential(pg3n_level *s, double *phi, pg_memspace where);
pg_status pg3n_inbox_export(pg3n_level *s, pg3n_inbox which, unsigned char handle[PG_IPC_HANDLE_BYTES], double **local_ptr);
pg_status pg3n_peer_open(pg3n_level *s, pg3n_inbox which, const unsigned char handle[PG_IPC_HANDLE_BYTES]);
pg_status pg3n_peer_set(pg3n_level *s, pg3n_inbox which, double *neighbour_inbox);
pg_status pg3n_synchronize(pg3n_level *s);
pg_status pg3n_destroy(pg3n_level *s); /* pg3n_destroy(NULL) is a no-op returning PG_OK */
long pg3n_launch_count(const pg3n_level *s);
const char *pg3n_last_error(const pg3n_level *s); /* s may be NULL: last error of a failed pg3n_create */

#ifdef __cplusplus
}
#endif
#endif /* POLARGRAV_H */
