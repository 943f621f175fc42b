// polargrav.cu -- C ABI (include/polargrav.h) and host-side runtime of libpolargrav.so.
//
// Host logic only: argument checks, table construction (long double), buffer ownership,
// stream/event plumbing for the pinned staging pipeline (row a6), kernel dispatch by grid size.
// Every step of the numerical path runs in the kernels of kernels.cuh.  There is no CPU
// fallback: without an sm_100 device pg_create* fails.
#include "../../include/polargrav.h"
#include "kernels.cuh"
#include "variants.cuh"
#include "cartesian.cuh"
#include "nested.cuh"

#include <cmath>
#include <cudaTypedefs.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using pgk::cplx;

namespace {

constexpr int kMaxProfiledCalls = 2048;

#ifndef PG_TMAP_L2
#define PG_TMAP_L2 CU_TENSOR_MAP_L2_PROMOTION_NONE   // L2 promotion of the tile loads (128B / 256B tried: no difference)
#endif

thread_local char g_create_error[512] = "";

struct Events4 { cudaEvent_t e[4]; };

}  // namespace

struct pg_solver {
    int n_r = 0, n_phi = 0, max_batch = 1, device = 0;
    double r_in = 0, r_out = 0, eps = 0, du = 0, dphi = 0;
    int sm_count = 0, row_ctas = 0, row_ctas_inv = 0;   // persistent grids of the forward / inverse row kernel
    // small grids (64 .. 512 per axis): the whole solve in one cooperative launch (kernels.cuh, fused_solve_kernel)
    // tensor maps of the W buffers rows_inv_kernel reads as 4-D TMA tiles (n_phi >= PG_ROW_INLINE_FROM), by buffer
    struct RowTmap { const void *base; int n_rows, fields; long stride; CUtensorMap map; };
    std::vector<RowTmap> row_tmaps;
    int fused = 1;                    // PG_OPT_FUSED
    int fused_cap = 0;                // CTAs of the fused kernel resident at once (0: the grid has no fused kernel)
    int fused_items = 0, fused_groups = 0;   // row items and mode groups per field
    int half = 0;      // H = n_phi/2: azimuthal modes are 0..H (H + 1 columns of W)
    size_t field = 0;  // n_r * n_phi

    cudaStream_t stream = nullptr;             // borrowed
    cudaStream_t h2d = nullptr, d2h = nullptr; // owned copy streams
    std::vector<cudaEvent_t> ev_in, ev_solved, ev_out;
    cudaEvent_t ev_main = nullptr;
    std::vector<char> in_pending;

    // device memory (owned)
    cplx *d_W = nullptr;          // W: [max_batch][half+1][n_r]
    cplx *d_W_alt = nullptr;      // second W (lazily allocated): resident solves alternate, see solve_fields
    const cplx *last_w = nullptr; // the W buffer the most recent solve of this solver works in
    // PG_OPT_LANES: consecutive resident solves alternate between two internal streams (each with its own pair of W
    // buffers), so that the tail and the hand-over bubbles of one solve's kernels are filled by the other's
    int lanes = 1, lane_next = 0;
    cudaStream_t lane_stream[PG_MAX_LANES] = {};
    cudaEvent_t lane_done[PG_MAX_LANES] = {};
    cplx *lane_W[PG_MAX_LANES][2] = {};
    int lane_w_next[PG_MAX_LANES] = {};
    bool lane_used[PG_MAX_LANES] = {};
    double *d_khat = nullptr;     // [half+1][2][n_r]
    cplx *d_tw_row = nullptr;     // Plan<n_phi/2, ROW> twiddle table
    cplx *d_tw_col = nullptr;     // Plan<2 n_r, COL> twiddle table
    double *d_rs_in = nullptr, *d_rs_out = nullptr;
    // NEXT-4 variants (variants.cuh): softening mode, complex kernel spectra [Phi, a_r, a_phi] for it, the post-scale
    // r^(-3/2) of the acceleration, and a second spectrum workspace (the column pass is out of place there)
    int soft = PG_SOFT_SYMMETRIC;
    cplx *d_khat_c[3] = {nullptr, nullptr, nullptr};
    bool khat_c_valid[3] = {false, false, false};
    double *d_rs_out32 = nullptr;
    cplx *d_W_var = nullptr;
    double *d_r = nullptr, *d_dA = nullptr, *d_s2 = nullptr;
    // [max_batch][n_r][n_phi] each, lazily allocated, TWO slots per direction: the upload of the next
    // density does not wait for the solve that still reads the previous one, and a solve does not wait for
    // the download of the previous potential
    double *d_sigma_own[2] = {nullptr, nullptr}, *d_phi_own[2] = {nullptr, nullptr};
    int in_slot = 0, out_slot = 0;
    cudaEvent_t ev_in_free[2] = {nullptr, nullptr};    // main stream: the solves reading sigma slot k are done
    cudaEvent_t ev_out_done[2] = {nullptr, nullptr};   // d2h stream: the downloads from phi slot k are done
    // pinned host staging (owned, lazily allocated)
    double *h_in = nullptr, *h_out = nullptr;

    // current density
    const double *d_sigma = nullptr;
    int cur_batch = 0;
    bool sigma_from_host = false;
    bool density_stable = false;   // PG_OPT_DENSITY_STABLE

    // host tables
    std::vector<double> r, phi, dA;

    // profiling
    bool profile = false;
    std::vector<Events4> prof_pool;
    int prof_used = 0;
    double prof_ms[PG_NUM_KERNELS] = {0, 0, 0};
    long prof_n[PG_NUM_KERNELS] = {0, 0, 0};
    long launches = 0;

    char err[512] = "";
};

namespace {

void set_err(pg_solver *s, const char *fmt, ...)
{
    char *dst = s ? s->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
}

#define PG_CUDA(s, call)                                                                       \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            set_err((s), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__,     \
                    __LINE__);                                                                 \
            return e_ == cudaErrorMemoryAllocation ? PG_ERR_NOMEM : PG_ERR_CUDA;               \
        }                                                                                      \
    } while (0)

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// ------------------------------------------------------------------ tables
const long double kPiL = 3.141592653589793238462643383279502884L;

cplx unit(long double turns)   // exp(-2 pi i turns)
{
    const long double a = 2.0L * kPiL * turns;
    return make_double2((double)cosl(a), (double)(-sinl(a)));
}


// compact twiddle table of Plan<L, KIND> (fft.cuh): base roots only, long double on the host
template <int L, int KIND>
void fill_twiddles(std::vector<cplx> &tw)
{
    typedef pgk::Plan<L, KIND> P;
    tw.assign(P::TW_LEN, make_double2(0.0, 0.0));
    for (int b = 0; b < P::MA; ++b) {
        tw[P::TW_A + b] = unit((long double)b / L);
    }
    for (int b = 0; b < P::RC; ++b) tw[P::TW_B + b] = unit((long double)b / P::MA);
    if (KIND == pgk::ROW) {
        for (int q = 0; q < P::NB; ++q) {       // i exp(-2 pi i q / 2L)
            const long double a = 2.0L * kPiL * q / (2.0L * L);
            tw[P::TW_UN + q] = make_double2((double)sinl(a), (double)cosl(a));
        }
    }
}

template <int KIND>
bool twiddles_for(int len, std::vector<cplx> &tw)
{
    switch (len) {
        case 16: fill_twiddles<16, KIND>(tw); return true;
        case 32: fill_twiddles<32, KIND>(tw); return true;
        case 64: fill_twiddles<64, KIND>(tw); return true;
        case 128: fill_twiddles<128, KIND>(tw); return true;
        case 256: fill_twiddles<256, KIND>(tw); return true;
        case 512: fill_twiddles<512, KIND>(tw); return true;
        case 1024: fill_twiddles<1024, KIND>(tw); return true;
        case 2048: fill_twiddles<2048, KIND>(tw); return true;
        case 4096: if (KIND == pgk::COL) { fill_twiddles<4096, pgk::COL>(tw); return true; } return false;
        default: return false;
    }
}

template <class T>
pg_status upload(pg_solver *s, T **dst, const std::vector<T> &src)
{
    PG_CUDA(s, cudaMalloc((void **)dst, src.size() * sizeof(T)));
    PG_CUDA(s, cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return PG_OK;
}

// ------------------------------------------------------------------ kernel dispatch
// Launch with programmatic stream serialization: the kernel's CTAs may be scheduled while the
// preceding kernel of the stream drains; every kernel calls griddepcontrol.wait before it touches
// data that kernel may read or write (kernels.cuh, pdl_wait).
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// Output range of the last kernel of this library that releases its dependents before it has
// finished writing (rows_inv_kernel), PER STREAM: a rows_fwd_kernel launched right behind it on the same
// stream may read its input ahead of griddepcontrol.wait only if that input does not overlap this range.
// The programmatic dependency exists only between consecutive kernels of one stream, so the record is keyed
// by (device, stream): solves of other solvers on other streams in between do not erase it, and two solvers
// that share a stream see each other's outputs.  (Any other producer of Sigma on the stream -- a copy, a
// kernel of the caller -- does not release dependents early, so the launch itself is ordered behind its
// completion; a producer on ANOTHER stream is the caller's promise, PG_OPT_DENSITY_STABLE.)
struct OutRange { int device; cudaStream_t stream; const char *begin, *end; };
std::mutex g_out_mutex;
std::vector<OutRange> g_out_ranges;

void note_early_release_output(int device, cudaStream_t st, const void *p, size_t bytes)
{
    std::lock_guard<std::mutex> lock(g_out_mutex);
    for (auto &r : g_out_ranges)
        if (r.device == device && r.stream == st) { r.begin = (const char *)p; r.end = r.begin + bytes; return; }
    g_out_ranges.push_back(OutRange{device, st, (const char *)p, (const char *)p + bytes});
}
bool overlaps_early_release_output(int device, cudaStream_t st, const void *p, size_t bytes)
{
    std::lock_guard<std::mutex> lock(g_out_mutex);
    const char *b = (const char *)p, *e = b + bytes;
    for (const auto &r : g_out_ranges)
        if (r.device == device && r.stream == st) return b < r.end && r.begin < e;
    return false;
}
// a stream that has been synchronised (or is being abandoned) has nothing in flight
void forget_early_release_output(int device, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_out_mutex);
    for (size_t k = 0; k < g_out_ranges.size(); ++k)
        if (g_out_ranges[k].device == device && g_out_ranges[k].stream == st) {
            g_out_ranges[k] = g_out_ranges.back();
            g_out_ranges.pop_back();
            return;
        }
}

// restores the caller's current device when an ABI call returns
struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int device)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) changed = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

bool ranges_overlap(const void *a, size_t na, const void *b, size_t nb)
{
    const char *a0 = (const char *)a, *b0 = (const char *)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

template <int NPHI>
pg_status launch_rows_fwd(pg_solver *s, const double *sigma, cplx *Z, const double *rscale, int n_rows,
                          int batch, long sigma_stride, long z_stride, cudaStream_t st, int early_mode)
{
    typedef pgk::RowShape<NPHI> S;
    const int n_items = (n_rows / S::ROWS) * batch;      // persistent CTAs walk over the items
    const int grid = n_items < s->row_ctas ? n_items : s->row_ctas;
    PG_CUDA(s, launch_pdl(pgk::rows_fwd_kernel<NPHI>, dim3(grid), dim3(S::THREADS), S::SMEM, st, sigma, Z, s->d_tw_row,
                          rscale, n_rows, n_items, sigma_stride, z_stride,
                          early_mode));
    s->launches++;
    return PG_OK;
}

// Tensor map of a W buffer for the tile loads of rows_inv_kernel (kernels.cuh, RowShape::TILE): as doubles,
//   dim 0  2 n_rows (one column of W, contiguous)           box 2 ROWS   (one run of ROWS rows)
//   dim 1  a = m / RA, L / RA values, stride RA columns      box L / RA
//   dim 2  c = m mod RA, RA values, stride one column        box RA       -> tile [c][a][row] in shared memory
//   dim 3  field                                             box 1
// Mode L (the 1025th column at n_phi = 2048) is outside the map and fetched by a plain load.
template <int NPHI>
pg_status row_tmap(pg_solver *s, const cplx *Z, int n_rows, int fields, long z_stride, CUtensorMap *out)
{
    typedef pgk::RowShape<NPHI, true> S;
    typedef pgk::Plan<S::L, pgk::ROW> P;
    memset(out, 0, sizeof *out);
    if constexpr (!S::TILE) {
        (void)s; (void)Z; (void)n_rows; (void)fields; (void)z_stride;
        return PG_OK;
    } else {
        for (const auto &e : s->row_tmaps)
            if (e.base == Z && e.n_rows == n_rows && e.fields == fields && e.stride == z_stride) { *out = e.map; return PG_OK; }
        static PFN_cuTensorMapEncodeTiled encode = nullptr;
        if (!encode) {
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult q;
            if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
                q != cudaDriverEntryPointSuccess || !fn) {
                set_err(s, "cuTensorMapEncodeTiled is not available from this driver");
                return PG_ERR_CUDA;
            }
            encode = (PFN_cuTensorMapEncodeTiled)fn;
        }
        const cuuint64_t dims[4] = {2ull * (cuuint64_t)n_rows, (cuuint64_t)(S::L / P::RA), (cuuint64_t)P::RA, (cuuint64_t)fields};
        const cuuint64_t strides[3] = {(cuuint64_t)P::RA * n_rows * sizeof(cplx), (cuuint64_t)n_rows * sizeof(cplx),
                                       (cuuint64_t)z_stride * sizeof(cplx)};
        const cuuint32_t box[4] = {2u * S::ROWS, (cuuint32_t)(S::L / P::RA), (cuuint32_t)P::RA, 1u};
        const cuuint32_t es[4] = {1, 1, 1, 1};
        pg_solver::RowTmap e{Z, n_rows, fields, z_stride, {}};
        const CUresult r = encode(&e.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<cplx *>(Z), dims, strides, box, es,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, PG_TMAP_L2,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { set_err(s, "cuTensorMapEncodeTiled failed (%d)", (int)r); return PG_ERR_CUDA; }
        if (s->row_tmaps.size() >= 64) s->row_tmaps.clear();
        s->row_tmaps.push_back(e);
        *out = e.map;
        return PG_OK;
    }
}

template <int NPHI>
pg_status launch_rows_inv(pg_solver *s, const cplx *Z, double *phi, int batch, long z_stride, long phi_stride,
                          cudaStream_t st, const double *oscale)
{
    typedef pgk::RowShape<NPHI, true> S;
    const int n_items = (s->n_r / S::ROWS) * batch;
    const int grid = n_items < s->row_ctas_inv ? n_items : s->row_ctas_inv;
    CUtensorMap tmap;
    pg_status rc = row_tmap<NPHI>(s, Z, s->n_r, batch, z_stride, &tmap);
    if (rc != PG_OK) return rc;
    PG_CUDA(s, launch_pdl(pgk::rows_inv_kernel<NPHI>, dim3(grid), dim3(S::THREADS), S::SMEM, st, Z, phi, s->d_tw_row,
                          oscale, s->n_r, n_items, z_stride, phi_stride, tmap));
    note_early_release_output(s->device, st, phi, (size_t)s->n_r * NPHI * sizeof(double) * batch);
    s->launches++;
    return PG_OK;
}

template <int NR>
pg_status launch_cols(pg_solver *s, cplx *Z, int batch, long z_stride, cudaStream_t st)
{
    typedef pgk::ColShape<NR> S;
    const int modes = s->half + 1;
    dim3 grid((modes + S::MODES - 1) / S::MODES, batch);
    PG_CUDA(s, launch_pdl(pgk::cols_kernel<NR>, grid, dim3(S::THREADS), S::SMEM, st, Z, (const double *)s->d_khat,
                          (const cplx *)s->d_tw_col, modes, z_stride));
    s->launches++;
    return PG_OK;
}

// ---- small grids: one cooperative launch per solve
template <int NR, int NPHI>
pg_status prepare_fused(pg_solver *s)
{
    typedef pgk::FusedShape<NR, NPHI> F;
    PG_CUDA(s, cudaFuncSetAttribute(pgk::fused_solve_kernel<NR, NPHI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F::SMEM));
    int occ = 0;
    PG_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pgk::fused_solve_kernel<NR, NPHI>, F::THREADS, F::SMEM));
    s->fused_cap = occ * s->sm_count;
    s->fused_items = NR / F::RS::ROWS;
    s->fused_groups = (NPHI / 2 + 1 + F::CS::MODES - 1) / F::CS::MODES;
    return PG_OK;
}
template <int NR, int NPHI>
pg_status launch_fused(pg_solver *s, const double *sigma, double *phi, cplx *W, int batch, cudaStream_t st)
{
    typedef pgk::FusedShape<NR, NPHI> F;
    const int items = s->fused_items * batch, cols = s->fused_groups * batch;
    const int grid = items > cols ? items : cols;
    long fs = (long)s->field, ws = (long)(s->half + 1) * s->n_r;
    const double *khat = s->d_khat, *rs_in = s->d_rs_in, *rs_out = s->d_rs_out;
    const cplx *tw_row = s->d_tw_row, *tw_col = s->d_tw_col;
    void *args[] = {(void *)&sigma, (void *)&phi, (void *)&W, (void *)&khat, (void *)&tw_row, (void *)&tw_col,
                    (void *)&rs_in, (void *)&rs_out, (void *)&batch, (void *)&fs, (void *)&ws};
    PG_CUDA(s, cudaLaunchCooperativeKernel((const void *)pgk::fused_solve_kernel<NR, NPHI>, dim3(grid), dim3(F::THREADS), args,
                                           F::SMEM, st));
    s->launches++;
    // an ordinary (non-PDL-releasing) kernel: everything before it on the stream, including the output range an earlier
    // rows_inv_kernel recorded, is complete before any kernel behind it starts
    forget_early_release_output(s->device, st);
    return PG_OK;
}
#define PG_FUSED_DISPATCH_PHI(NR, CALL)                         \
    switch (s->n_phi) {                                         \
        case 64: return CALL(NR, 64);                           \
        case 128: return CALL(NR, 128);                         \
        case 256: return CALL(NR, 256);                         \
        case 512: return CALL(NR, 512);                         \
        default: return PG_ERR_UNSUPPORTED;                     \
    }
#define PG_FUSED_DISPATCH(CALL)                                 \
    switch (s->n_r) {                                           \
        case 64: PG_FUSED_DISPATCH_PHI(64, CALL)                \
        case 128: PG_FUSED_DISPATCH_PHI(128, CALL)              \
        case 256: PG_FUSED_DISPATCH_PHI(256, CALL)              \
        case 512: PG_FUSED_DISPATCH_PHI(512, CALL)              \
        default: return PG_ERR_UNSUPPORTED;                     \
    }
bool fused_size(const pg_solver *s)
{
    return s->n_r >= 64 && s->n_r <= 512 && s->n_phi >= 64 && s->n_phi <= 512;
}
pg_status prepare_kernels_fused(pg_solver *s)
{
    if (!fused_size(s)) return PG_OK;
#define CALL(NR, NPHI) prepare_fused<NR, NPHI>(s)
    PG_FUSED_DISPATCH(CALL)
#undef CALL
}
pg_status fused_solve(pg_solver *s, const double *sigma, double *phi, cplx *W, int batch, cudaStream_t st)
{
#define CALL(NR, NPHI) launch_fused<NR, NPHI>(s, sigma, phi, W, batch, st)
    PG_FUSED_DISPATCH(CALL)
#undef CALL
}
// the fused kernel serves this solve: enabled, symmetric softening, no per-kernel profiling, all its CTAs resident at once
bool fused_ok(const pg_solver *s, int batch, bool profiled)
{
    if (!s->fused || s->fused_cap <= 0 || profiled) return false;
    const int items = s->fused_items * batch, cols = s->fused_groups * batch;
    return (items > cols ? items : cols) <= s->fused_cap;
}

template <int NR>
pg_status launch_khat_cols(pg_solver *s, const cplx *ZK, double scale, cudaStream_t st)
{
    const int threads = NR / 8;
    const size_t smem = (size_t)pgk::Plan<2 * NR, pgk::COL>::LINE * sizeof(cplx);
    pgk::khat_cols_kernel<NR><<<s->half + 1, threads, smem, st>>>(ZK, s->d_khat, s->d_tw_col, scale);
    PG_CUDA(s, cudaGetLastError());
    s->launches++;
    return PG_OK;
}

template <int NR>
pg_status launch_khat_cols_cplx(pg_solver *s, const cplx *ZK, cplx *out, double scale, cudaStream_t st)
{
    const int threads = NR / 8;
    const size_t smem = (size_t)pgk::Plan<2 * NR, pgk::COL>::LINE * sizeof(cplx);
    PG_CUDA(s, cudaFuncSetAttribute(pgk::khat_cols_cplx_kernel<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    pgk::khat_cols_cplx_kernel<NR><<<s->half + 1, threads, smem, st>>>(ZK, out, s->d_tw_col, scale);
    PG_CUDA(s, cudaGetLastError());
    s->launches++;
    return PG_OK;
}
template <int NR>
pg_status launch_cols_cplx(pg_solver *s, const cplx *src, cplx *dst, const cplx *khat_c, int batch, long z_stride, cudaStream_t st)
{
    typedef pgk::ColShape<NR> S;
    const int modes = s->half + 1;
    PG_CUDA(s, cudaFuncSetAttribute(pgk::cols_cplx_kernel<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::LINES));
    dim3 grid((modes + S::MODES - 1) / S::MODES, batch);
    PG_CUDA(s, launch_pdl(pgk::cols_cplx_kernel<NR>, grid, dim3(S::THREADS), S::LINES, st, src, dst, khat_c,
                          (const cplx *)s->d_tw_col, modes, z_stride));
    s->launches++;
    return PG_OK;
}

// opt in to > 48 KiB of dynamic shared memory, once per solver (the attribute is per device)
template <int NPHI>
pg_status prepare_rows(pg_solver *s)
{
    typedef pgk::RowShape<NPHI> S;
    typedef pgk::RowShape<NPHI, true> SI;
    PG_CUDA(s, cudaFuncSetAttribute(pgk::rows_fwd_kernel<NPHI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)S::SMEM));
    PG_CUDA(s, cudaFuncSetAttribute(pgk::rows_inv_kernel<NPHI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)SI::SMEM));
    // persistent grids: as many CTAs as are resident at once
    int occ_f = 0, occ_i = 0;
    PG_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, pgk::rows_fwd_kernel<NPHI>, S::THREADS, S::SMEM));
    PG_CUDA(s, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_i, pgk::rows_inv_kernel<NPHI>, SI::THREADS, SI::SMEM));
    s->row_ctas = (occ_f > 0 ? occ_f : 1) * s->sm_count;
    s->row_ctas_inv = (occ_i > 0 ? occ_i : 1) * s->sm_count;
    return PG_OK;
}
template <int NR>
pg_status prepare_cols(pg_solver *s)
{
    typedef pgk::ColShape<NR> S;
    PG_CUDA(s, cudaFuncSetAttribute(pgk::cols_kernel<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)S::SMEM));
    PG_CUDA(s, cudaFuncSetAttribute(pgk::khat_cols_kernel<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)(pgk::Plan<2 * NR, pgk::COL>::LINE * sizeof(cplx))));
    return PG_OK;
}

#define PG_DISPATCH(n, CALL)                                                   \
    switch (n) {                                                               \
        case 32: return CALL(32);                                              \
        case 64: return CALL(64);                                              \
        case 128: return CALL(128);                                            \
        case 256: return CALL(256);                                            \
        case 512: return CALL(512);                                            \
        case 1024: return CALL(1024);                                          \
        case 2048: return CALL(2048);                                          \
        default: set_err(s, "unsupported size %d", (n)); return PG_ERR_UNSUPPORTED; \
    }

pg_status rows_fwd(pg_solver *s, const double *sigma, cplx *W, const double *rscale, int n_rows, int batch,
                   long sigma_stride, long w_stride, cudaStream_t st, int early_mode)
{
#define CALL(N) launch_rows_fwd<N>(s, sigma, W, rscale, n_rows, batch, sigma_stride, w_stride, st, early_mode)
    PG_DISPATCH(s->n_phi, CALL)
#undef CALL
}
pg_status rows_inv(pg_solver *s, const cplx *W, double *phi, int batch, long w_stride, long phi_stride,
                   cudaStream_t st, const double *oscale = nullptr)
{
    if (!oscale) oscale = s->d_rs_out;
#define CALL(N) launch_rows_inv<N>(s, W, phi, batch, w_stride, phi_stride, st, oscale)
    PG_DISPATCH(s->n_phi, CALL)
#undef CALL
}
pg_status cols(pg_solver *s, cplx *W, int batch, long w_stride, cudaStream_t st)
{
#define CALL(N) launch_cols<N>(s, W, batch, w_stride, st)
    PG_DISPATCH(s->n_r, CALL)
#undef CALL
}
pg_status prepare_kernels_rows(pg_solver *s)
{
#define CALL(N) prepare_rows<N>(s)
    PG_DISPATCH(s->n_phi, CALL)
#undef CALL
}
pg_status prepare_kernels_cols(pg_solver *s)
{
#define CALL(N) prepare_cols<N>(s)
    PG_DISPATCH(s->n_r, CALL)
#undef CALL
}
pg_status khat_cols_cplx(pg_solver *s, const cplx *Wk, cplx *out, double scale, cudaStream_t st)
{
#define CALL(N) launch_khat_cols_cplx<N>(s, Wk, out, scale, st)
    PG_DISPATCH(s->n_r, CALL)
#undef CALL
}
pg_status cols_cplx(pg_solver *s, const cplx *src, cplx *dst, const cplx *khat_c, int batch, long w_stride, cudaStream_t st)
{
#define CALL(N) launch_cols_cplx<N>(s, src, dst, khat_c, batch, w_stride, st)
    PG_DISPATCH(s->n_r, CALL)
#undef CALL
}
pg_status khat_cols(pg_solver *s, const cplx *Wk, double scale, cudaStream_t st)
{
#define CALL(N) launch_khat_cols<N>(s, Wk, scale, st)
    PG_DISPATCH(s->n_r, CALL)
#undef CALL
}

// ------------------------------------------------------------------ one-time spectrum of the Green's kernel (a1)
pg_status build_khat(pg_solver *s)
{
    const int n_r = s->n_r, n_phi = s->n_phi;
    double *d_kpad = nullptr;
    cplx *d_wk = nullptr;
    const size_t kpad_n = (size_t)2 * n_r * n_phi;
    const size_t wk_n = (size_t)(s->half + 1) * 2 * n_r;
    PG_CUDA(s, cudaMalloc((void **)&d_kpad, kpad_n * sizeof(double)));
    cudaError_t e = cudaMalloc((void **)&d_wk, wk_n * sizeof(cplx));
    if (e != cudaSuccess) {
        cudaFree(d_kpad);
        set_err(s, "cudaMalloc(kernel workspace) failed: %s", cudaGetErrorString(e));
        return PG_ERR_NOMEM;
    }
    pg_status st = PG_OK;
    do {
        const double eta2 = s->eps * s->eps * std::sinh(s->du) * s->dphi;
        const int threads = 256;
        const long blocks = (long)((kpad_n + threads - 1) / threads);
        pgk::green_fill_kernel<<<(unsigned)blocks, threads, 0, s->stream>>>(d_kpad, n_r, n_phi, s->du, eta2);
        s->launches++;
        if (cudaGetLastError() != cudaSuccess) { st = PG_ERR_CUDA; break; }
        // packed phi transform of the 2 n_r lag rows (no radial weight), transposed into ZK[k][2 n_r]
        st = rows_fwd(s, d_kpad, d_wk, nullptr, 2 * n_r, 1, 0, 0, s->stream, 0);
        if (st != PG_OK) break;
        // -G sinh(du) dphi (cell area / r^2), and the normalisation of the unnormalised transforms:
        // 1/(2 n_r) for the padded radial pair; 1/(2 n_phi) for the azimuthal pair (cols_kernel forms
        // 2 X on the way in and 2 Z on the way out, the packed transform has length n_phi/2);
        // another 1/2 because khat_cols_kernel forms 2 X of the kernel itself.
        const double scale = -std::sinh(s->du) * s->dphi / (8.0 * (double)n_r * (double)n_phi);
        st = khat_cols(s, d_wk, scale, s->stream);
        if (st != PG_OK) break;
        if (cudaStreamSynchronize(s->stream) != cudaSuccess) { st = PG_ERR_CUDA; break; }
    } while (0);
    if (st == PG_ERR_CUDA && s->err[0] == 0) set_err(s, "Green's kernel precompute failed: %s", cudaGetErrorString(cudaGetLastError()));
    cudaFree(d_kpad);
    cudaFree(d_wk);
    return st;
}

// Complex spectrum of one of the variant kernels (variants.cuh: kind 0 = K_Phi, 1 = K_r, 2 = K_phi) for the
// solver's softening mode; same pipeline and normalisation as build_khat, the column pass keeps the complex value.
pg_status build_khat_variant(pg_solver *s, int kind)
{
    if (s->khat_c_valid[kind]) return PG_OK;
    const int n_r = s->n_r, n_phi = s->n_phi;
    const size_t kpad_n = (size_t)2 * n_r * n_phi;
    const size_t wk_n = (size_t)(s->half + 1) * 2 * n_r;
    if (!s->d_khat_c[kind]) PG_CUDA(s, cudaMalloc((void **)&s->d_khat_c[kind], wk_n * sizeof(cplx)));
    if (!s->d_rs_out32) {
        std::vector<double> w(n_r);
        for (int i = 0; i < n_r; ++i) w[i] = (double)(1.0L / ((long double)s->r[i] * sqrtl((long double)s->r[i])));
        pg_status up = upload(s, &s->d_rs_out32, w);
        if (up != PG_OK) return up;
    }
    double *d_kpad = nullptr;
    cplx *d_wk = nullptr;
    PG_CUDA(s, cudaMalloc((void **)&d_kpad, kpad_n * sizeof(double)));
    if (cudaMalloc((void **)&d_wk, wk_n * sizeof(cplx)) != cudaSuccess) {
        cudaFree(d_kpad);
        set_err(s, "cudaMalloc(kernel workspace) failed");
        return PG_ERR_NOMEM;
    }
    pg_status st = PG_OK;
    do {
        const double eta2 = s->eps * s->eps * std::sinh(s->du) * s->dphi;
        const int threads = 256;
        const long blocks = (long)((kpad_n + threads - 1) / threads);
        pgk::green_fill_var_kernel<<<(unsigned)blocks, threads, 0, s->stream>>>(d_kpad, n_r, n_phi, s->du, eta2, s->soft, kind);
        s->launches++;
        if (cudaGetLastError() != cudaSuccess) { st = PG_ERR_CUDA; break; }
        st = rows_fwd(s, d_kpad, d_wk, nullptr, 2 * n_r, 1, 0, 0, s->stream, 0);
        if (st != PG_OK) break;
        const double scale = -std::sinh(s->du) * s->dphi / (8.0 * (double)n_r * (double)n_phi);
        st = khat_cols_cplx(s, d_wk, s->d_khat_c[kind], scale, s->stream);
        if (st != PG_OK) break;
        if (cudaStreamSynchronize(s->stream) != cudaSuccess) { st = PG_ERR_CUDA; break; }
    } while (0);
    if (st == PG_ERR_CUDA && s->err[0] == 0) set_err(s, "variant kernel precompute failed: %s", cudaGetErrorString(cudaGetLastError()));
    cudaFree(d_kpad);
    cudaFree(d_wk);
    if (st == PG_OK) s->khat_c_valid[kind] = true;
    return st;
}

pg_status ensure_var_workspace(pg_solver *s)
{
    if (!s->d_W_var) {
        const size_t w_bytes = (size_t)s->max_batch * (s->half + 1) * s->n_r * sizeof(cplx);
        PG_CUDA(s, cudaMalloc((void **)&s->d_W_var, w_bytes));
    }
    return PG_OK;
}

// rows_fwd once, then one (complex column pass, inverse row pass) per requested output
pg_status solve_variant(pg_solver *s, const double *d_sigma, cplx *d_W, int batch, int n_out, const int *kinds,
                        double *const *outs)
{
    const long fs = (long)s->field, ws = (long)(s->half + 1) * s->n_r;
    pg_status st = ensure_var_workspace(s);
    if (st != PG_OK) return st;
    for (int q = 0; q < n_out; ++q)
        if ((st = build_khat_variant(s, kinds[q])) != PG_OK) return st;
    if ((st = rows_fwd(s, d_sigma, d_W, s->d_rs_in, s->n_r, batch, fs, ws, s->stream, 0)) != PG_OK) return st;
    s->last_w = d_W;
    for (int q = 0; q < n_out; ++q) {
        if ((st = cols_cplx(s, d_W, s->d_W_var, s->d_khat_c[kinds[q]], batch, ws, s->stream)) != PG_OK) return st;
        if ((st = rows_inv(s, s->d_W_var, outs[q], batch, ws, fs, s->stream, kinds[q] == 0 ? s->d_rs_out : s->d_rs_out32)) != PG_OK) return st;
    }
    return PG_OK;
}

pg_status ensure_staging(pg_solver *s, bool need_in, bool need_out)
{
    const size_t bytes = s->field * (size_t)s->max_batch * sizeof(double);
    for (int k = 0; k < 2; ++k) {
        if (need_in && !s->d_sigma_own[k]) PG_CUDA(s, cudaMalloc((void **)&s->d_sigma_own[k], bytes));
        if (need_out && !s->d_phi_own[k]) PG_CUDA(s, cudaMalloc((void **)&s->d_phi_own[k], bytes));
    }
    return PG_OK;
}
pg_status ensure_pinned(pg_solver *s, bool in, bool out)
{
    const size_t bytes = s->field * (size_t)s->max_batch * sizeof(double);
    if (in && !s->h_in) PG_CUDA(s, cudaHostAlloc((void **)&s->h_in, bytes, cudaHostAllocDefault));
    if (out && !s->h_out) PG_CUDA(s, cudaHostAlloc((void **)&s->h_out, bytes, cudaHostAllocDefault));
    return PG_OK;
}

pg_status drain_profile(pg_solver *s)
{
    if (s->prof_used == 0) return PG_OK;
    const int used = s->prof_used;
    s->prof_used = 0;          // whatever happens below, the slots are free again: one failure must not fail every later call
    PG_CUDA(s, cudaStreamSynchronize(s->stream));
    for (int c = 0; c < used; ++c) {
        for (int k = 0; k < PG_NUM_KERNELS; ++k) {
            float ms = 0.f;
            PG_CUDA(s, cudaEventElapsedTime(&ms, s->prof_pool[c].e[k], s->prof_pool[c].e[k + 1]));
            s->prof_ms[k] += ms;
            s->prof_n[k] += 1;
        }
    }
    return PG_OK;
}

// the three kernels of one solve of `batch` fields starting at the given pointers.  allow_lanes: the solve may go to
// a lane stream (PG_OPT_LANES) -- only the all-resident call site of potential_common says so; the staged host
// pipeline orders its copies against the solver's stream and must stay on it (polargrav.h: host memspaces keep
// using the solver's stream)
pg_status solve_fields(pg_solver *s, const double *d_sigma, double *d_phi, cplx *d_W, int batch, bool allow_lanes)
{
    const long fs = (long)s->field, ws = (long)(s->half + 1) * s->n_r;
    if (s->soft != PG_SOFT_SYMMETRIC) {
        // field / source softening: complex spectrum, variants.cuh.  No per-kernel profiling on this path, so no
        // profiling slot is taken for it (a slot with unrecorded events would poison drain_profile).
        const int kind = 0;
        double *out = d_phi;
        return solve_variant(s, d_sigma, d_W, batch, 1, &kind, &out);
    }
    Events4 *ev = nullptr;
    if (s->profile) {
        if (s->prof_used == kMaxProfiledCalls) {
            pg_status st = drain_profile(s);
            if (st != PG_OK) return st;
        }
        if ((int)s->prof_pool.size() <= s->prof_used) {
            Events4 q;
            for (int k = 0; k < 4; ++k) PG_CUDA(s, cudaEventCreate(&q.e[k]));
            s->prof_pool.push_back(q);
        }
        ev = &s->prof_pool[s->prof_used++];
        PG_CUDA(s, cudaEventRecord(ev->e[0], s->stream));
    }
    if (allow_lanes && s->lanes >= 2 && s->density_stable && !s->sigma_from_host && !ev && d_W == s->d_W) {
        // two solves in flight: this one goes to the lane the previous one did not take.  The caller has promised
        // (polargrav.h, PG_OPT_LANES) that density and potential are touched by nothing else in flight.
        const int L = s->lane_next;
        s->lane_next = (L + 1) % s->lanes;
        cudaStream_t lst = s->lane_stream[L];
        cplx *W = s->lane_W[L][s->lane_w_next[L]];
        s->lane_w_next[L] ^= 1;
        pg_status st = PG_OK;
        if (fused_ok(s, batch, false)) {
            if ((st = fused_solve(s, d_sigma, d_phi, W, batch, lst)) != PG_OK) return st;
            s->lane_used[L] = true;        // joined by pg_flush / pg_synchronize
            return PG_OK;
        }
        const int early = overlaps_early_release_output(s->device, lst, d_sigma, (size_t)batch * s->field * sizeof(double)) ? 0 : 2;
        if ((st = rows_fwd(s, d_sigma, W, s->d_rs_in, s->n_r, batch, fs, ws, lst, early)) != PG_OK) return st;
        if ((st = cols(s, W, batch, ws, lst)) != PG_OK) return st;
        if ((st = rows_inv(s, W, d_phi, batch, ws, fs, lst)) != PG_OK) return st;
        s->lane_used[L] = true;            // joined by pg_flush / pg_synchronize
        return PG_OK;
    }
    if (fused_ok(s, batch, ev != nullptr)) {
        s->last_w = d_W;
        return fused_solve(s, d_sigma, d_phi, d_W, batch, s->stream);
    }
    // How much rows_fwd depends on the kernel before it (kernels.cuh): with a stable density that does not
    // alias the potential still being written, the first item is fetched early (1); if the solve also
    // works in the W buffer the previous solve did not use, it depends on nothing in flight (2).
    int early = 0;
    if (s->density_stable && !s->sigma_from_host &&
        !overlaps_early_release_output(s->device, s->stream, d_sigma, (size_t)batch * s->field * sizeof(double))) {
        early = 1;
        if (d_W == s->d_W && !ev) {
            if (!s->d_W_alt) {
                const size_t w_bytes = (size_t)s->max_batch * (s->half + 1) * s->n_r * sizeof(cplx);
                if (cudaMalloc((void **)&s->d_W_alt, w_bytes) != cudaSuccess) { s->d_W_alt = nullptr; (void)cudaGetLastError(); }
            }
            if (s->d_W_alt) {
                d_W = (s->last_w == s->d_W) ? s->d_W_alt : s->d_W;     // the one the previous solve does not use
                early = 2;
            }
        }
    }
    s->last_w = (d_W == s->d_W_alt) ? s->d_W_alt : s->d_W;
    pg_status st = rows_fwd(s, d_sigma, d_W, s->d_rs_in, s->n_r, batch, fs, ws, s->stream, early);
    if (st != PG_OK) return st;
    if (ev) PG_CUDA(s, cudaEventRecord(ev->e[1], s->stream));
    st = cols(s, d_W, batch, ws, s->stream);
    if (st != PG_OK) return st;
    if (ev) PG_CUDA(s, cudaEventRecord(ev->e[2], s->stream));
    st = rows_inv(s, d_W, d_phi, batch, ws, fs, s->stream);
    if (st != PG_OK) return st;
    if (ev) PG_CUDA(s, cudaEventRecord(ev->e[3], s->stream));
    return PG_OK;
}

pg_status launch_direct(pg_solver *s, const double *d_sigma, double *d_phi, int ring0, int n_rings, int batch)
{
    if (s->n_phi >= 256) {
        // register-tiled kernel: 16 consecutive targets per thread (8 below 1024), Sigma ring + doubled, padded kernel
        const int R = s->n_phi >= 1024 ? 16 : 8;
        const size_t smem = ((size_t)s->n_phi + (size_t)(2 * s->n_phi / R) * (R + 2)) * sizeof(double);
        const double eps2 = s->eps * s->eps;
        dim3 grid(n_rings, batch);
        const long fs = (long)s->field;
        if (s->n_phi >= 1024) {
            PG_CUDA(s, cudaFuncSetAttribute(pgk::direct_tiled_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            pgk::direct_tiled_kernel<16><<<grid, s->n_phi / 16, smem, s->stream>>>(d_sigma, d_phi, s->d_r, s->d_dA, s->d_s2, s->n_r,
                                                                                   s->n_phi, eps2, ring0, fs, fs);
        } else {
            pgk::direct_tiled_kernel<8><<<grid, s->n_phi / 8, smem, s->stream>>>(d_sigma, d_phi, s->d_r, s->d_dA, s->d_s2, s->n_r,
                                                                                 s->n_phi, eps2, ring0, fs, fs);
        }
        PG_CUDA(s, cudaGetLastError());
        s->launches++;
        return PG_OK;
    }
    const int threads = s->n_phi < 256 ? s->n_phi : 256;
    const int tpt = s->n_phi / threads;
    const size_t smem = 2 * (size_t)s->n_phi * sizeof(double);
    const double eps2 = s->eps * s->eps;
    dim3 grid(n_rings, batch);
    const long fs = (long)s->field;
#define DIRECT(TPT)                                                                                          \
    pgk::direct_kernel<TPT><<<grid, threads, smem, s->stream>>>(d_sigma, d_phi, s->d_r, s->d_dA, s->d_s2, s->n_r, \
                                                                 s->n_phi, eps2, ring0, fs, fs)
    switch (tpt) {
        case 1: DIRECT(1); break;
        case 2: DIRECT(2); break;
        case 4: DIRECT(4); break;
        case 8: DIRECT(8); break;
        default: set_err(s, "direct: unsupported n_phi"); return PG_ERR_UNSUPPORTED;
    }
#undef DIRECT
    PG_CUDA(s, cudaGetLastError());
    s->launches++;
    return PG_OK;
}

pg_status lanes_enable(pg_solver *s, int n_lanes)
{
    const size_t w_bytes = (size_t)s->max_batch * (s->half + 1) * s->n_r * sizeof(cplx);
    for (int L = 0; L < n_lanes; ++L) {
        if (!s->lane_stream[L]) PG_CUDA(s, cudaStreamCreateWithFlags(&s->lane_stream[L], cudaStreamNonBlocking));
        if (!s->lane_done[L]) PG_CUDA(s, cudaEventCreateWithFlags(&s->lane_done[L], cudaEventDisableTiming));
        for (int k = 0; k < 2; ++k)
            if (!s->lane_W[L][k]) PG_CUDA(s, cudaMalloc((void **)&s->lane_W[L][k], w_bytes));
    }
    return PG_OK;
}
// everything the lanes have in flight is complete when this returns
pg_status lanes_drain(pg_solver *s)
{
    for (int L = 0; L < PG_MAX_LANES; ++L)
        if (s->lane_stream[L]) {
            PG_CUDA(s, cudaStreamSynchronize(s->lane_stream[L]));
            forget_early_release_output(s->device, s->lane_stream[L]);
            s->lane_used[L] = false;
        }
    return PG_OK;
}

void free_all(pg_solver *s)
{
    if (!s) return;
    for (int L = 0; L < PG_MAX_LANES; ++L) {
        if (s->lane_stream[L]) { cudaStreamSynchronize(s->lane_stream[L]); forget_early_release_output(s->device, s->lane_stream[L]); cudaStreamDestroy(s->lane_stream[L]); }
        if (s->lane_done[L]) cudaEventDestroy(s->lane_done[L]);
        for (int k = 0; k < 2; ++k) cudaFree(s->lane_W[L][k]);
    }
    cudaFree(s->d_W); cudaFree(s->d_W_alt); cudaFree(s->d_khat); cudaFree(s->d_tw_row); cudaFree(s->d_tw_col);
    cudaFree(s->d_rs_in); cudaFree(s->d_rs_out); cudaFree(s->d_rs_out32); cudaFree(s->d_W_var);
    for (int k = 0; k < 3; ++k) cudaFree(s->d_khat_c[k]);
    cudaFree(s->d_r); cudaFree(s->d_dA); cudaFree(s->d_s2); 
    for (int k = 0; k < 2; ++k) {
        cudaFree(s->d_sigma_own[k]); cudaFree(s->d_phi_own[k]);
        if (s->ev_in_free[k]) cudaEventDestroy(s->ev_in_free[k]);
        if (s->ev_out_done[k]) cudaEventDestroy(s->ev_out_done[k]);
    }
    if (s->h_in) cudaFreeHost(s->h_in);
    if (s->h_out) cudaFreeHost(s->h_out);
    for (auto e : s->ev_in) if (e) cudaEventDestroy(e);
    for (auto e : s->ev_solved) if (e) cudaEventDestroy(e);
    for (auto e : s->ev_out) if (e) cudaEventDestroy(e);
    if (s->ev_main) cudaEventDestroy(s->ev_main);
    for (auto &q : s->prof_pool) for (int k = 0; k < 4; ++k) cudaEventDestroy(q.e[k]);
    if (s->h2d) cudaStreamDestroy(s->h2d);
    if (s->d2h) cudaStreamDestroy(s->d2h);
    delete s;
}

pg_status create_impl(pg_solver *s)
{
    const int n_r = s->n_r, n_phi = s->n_phi;
    int ndev = 0;
    PG_CUDA(s, cudaGetDeviceCount(&ndev));
    if (s->device < 0) PG_CUDA(s, cudaGetDevice(&s->device));
    if (s->device >= ndev) { set_err(s, "device %d out of range (%d devices)", s->device, ndev); return PG_ERR_INVALID_ARG; }
    DeviceGuard guard(s->device);      // the caller's current device is restored on return
    cudaDeviceProp prop;
    PG_CUDA(s, cudaGetDeviceProperties(&prop, s->device));
    s->sm_count = prop.multiProcessorCount;
    if (prop.major != 10) {
        set_err(s, "device %d is sm_%d%d; this library is built for sm_100a (B200) only and has no fallback",
                s->device, prop.major, prop.minor);
        return PG_ERR_UNSUPPORTED;
    }

    s->du = std::log(s->r_out / s->r_in) / n_r;
    s->dphi = 2.0 * M_PI / n_phi;
    s->half = n_phi / 2;
    s->field = (size_t)n_r * n_phi;

    // grid tables (A1, A2): geometric centres, exact sector areas in their sinh form
    s->r.resize(n_r); s->dA.resize(n_r); s->phi.resize(n_phi);
    std::vector<double> rs_in(n_r), rs_out(n_r), s2(n_phi);
    {
        const long double du = logl((long double)s->r_out / (long double)s->r_in) / n_r;
        const long double dphi = 2.0L * kPiL / n_phi;
        for (int i = 0; i < n_r; ++i) {
            const long double ri = (long double)s->r_in * expl(((long double)i + 0.5L) * du);
            s->r[i] = (double)ri;
            s->dA[i] = (double)(ri * ri * sinhl(du) * dphi);
            rs_in[i] = (double)(ri * sqrtl(ri));
            rs_out[i] = (double)(1.0L / sqrtl(ri));
        }
        for (int j = 0; j < n_phi; ++j) {
            s->phi[j] = (double)(((long double)j + 0.5L) * dphi);
            const long double sn = sinl(kPiL * j / n_phi);
            s2[j] = (double)(sn * sn);
        }
    }
    // FFT tables: base roots of the packed row transform (length n_phi/2) and of the zero-padded 2 n_r-point
    // column transform, in the layout Plan<L,KIND>::TW_* expects
    std::vector<cplx> tw_row, tw_col;
    if (!twiddles_for<pgk::ROW>(s->half, tw_row) || !twiddles_for<pgk::COL>(2 * n_r, tw_col)) {
        set_err(s, "unsupported transform length");
        return PG_ERR_UNSUPPORTED;
    }

    pg_status st;
    if ((st = upload(s, &s->d_tw_row, tw_row)) != PG_OK) return st;
    if ((st = upload(s, &s->d_tw_col, tw_col)) != PG_OK) return st;
    if ((st = upload(s, &s->d_rs_in, rs_in)) != PG_OK) return st;
    if ((st = upload(s, &s->d_rs_out, rs_out)) != PG_OK) return st;
    if ((st = upload(s, &s->d_r, s->r)) != PG_OK) return st;
    if ((st = upload(s, &s->d_dA, s->dA)) != PG_OK) return st;
    if ((st = upload(s, &s->d_s2, s2)) != PG_OK) return st;

    const size_t w_n = (size_t)s->max_batch * (s->half + 1) * n_r;
    PG_CUDA(s, cudaMalloc((void **)&s->d_W, w_n * sizeof(cplx)));
    PG_CUDA(s, cudaMalloc((void **)&s->d_khat, (size_t)(s->half + 1) * 2 * n_r * sizeof(double)));

    PG_CUDA(s, cudaStreamCreateWithFlags(&s->h2d, cudaStreamNonBlocking));
    PG_CUDA(s, cudaStreamCreateWithFlags(&s->d2h, cudaStreamNonBlocking));
    s->ev_in.assign(s->max_batch, nullptr);
    s->ev_solved.assign(s->max_batch, nullptr);
    s->ev_out.assign(s->max_batch, nullptr);
    s->in_pending.assign(s->max_batch, 0);
    for (int b = 0; b < s->max_batch; ++b) {
        PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_in[b], cudaEventDisableTiming));
        PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_solved[b], cudaEventDisableTiming));
        PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_out[b], cudaEventDisableTiming));
    }
    PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_main, cudaEventDisableTiming));
    for (int k = 0; k < 2; ++k) {
        PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_in_free[k], cudaEventDisableTiming));
        PG_CUDA(s, cudaEventCreateWithFlags(&s->ev_out_done[k], cudaEventDisableTiming));
    }

    if ((st = prepare_kernels_rows(s)) != PG_OK) return st;
    if ((st = prepare_kernels_cols(s)) != PG_OK) return st;
    if ((st = prepare_kernels_fused(s)) != PG_OK) return st;
    return build_khat(s);
}

}  // namespace

// =================================================================== C ABI
extern "C" {

pg_status pg_create_ex(pg_solver **out, int n_r, int n_phi, double r_in, double r_out, double eps, int max_batch,
                       int device, void *cuda_stream)
{
    g_create_error[0] = 0;
    if (!out) { set_err(nullptr, "out is NULL"); return PG_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!(r_in > 0.0) || !(r_out > r_in) || !(eps > 0.0) || !std::isfinite(r_out) || !std::isfinite(eps) ||
        max_batch < 1) {
        set_err(nullptr, "invalid argument: need 0 < r_in < r_out, eps > 0, max_batch >= 1");
        return PG_ERR_INVALID_ARG;
    }
    if (!is_pow2(n_r) || !is_pow2(n_phi) || n_r < PG_MIN_N || n_phi < PG_MIN_N || n_r > PG_MAX_N ||
        n_phi > PG_MAX_N) {
        set_err(nullptr, "unsupported grid %dx%d: n_r and n_phi must be powers of two in [%d, %d]", n_r, n_phi,
                PG_MIN_N, PG_MAX_N);
        return PG_ERR_UNSUPPORTED;
    }
    pg_solver *s = new (std::nothrow) pg_solver;
    if (!s) { set_err(nullptr, "out of host memory"); return PG_ERR_NOMEM; }
    s->n_r = n_r; s->n_phi = n_phi; s->r_in = r_in; s->r_out = r_out; s->eps = eps;
    s->max_batch = max_batch; s->device = device; s->stream = (cudaStream_t)cuda_stream;
    pg_status st = create_impl(s);
    if (st != PG_OK) {
        snprintf(g_create_error, sizeof g_create_error, "%s", s->err);
        free_all(s);
        return st;
    }
    *out = s;
    return PG_OK;
}

pg_status pg_create(pg_solver **out, int n_r, int n_phi, double r_in, double r_out, double eps)
{
    return pg_create_ex(out, n_r, n_phi, r_in, r_out, eps, 1, -1, nullptr);
}

pg_status pg_destroy(pg_solver *s)
{
    if (!s) return PG_OK;
    DeviceGuard guard(s->device);
    cudaStreamSynchronize(s->stream);
    forget_early_release_output(s->device, s->stream);
    if (s->h2d) cudaStreamSynchronize(s->h2d);
    if (s->d2h) cudaStreamSynchronize(s->d2h);
    free_all(s);
    return PG_OK;
}

pg_status pg_set_density(pg_solver *s, const double *sigma, int batch, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!sigma || batch < 1 || batch > s->max_batch) {
        set_err(s, "pg_set_density: sigma is NULL or batch %d outside [1, %d]", batch, s->max_batch);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    const size_t fbytes = s->field * sizeof(double);
    if (where == PG_MEM_DEVICE) {
        // the kernels move device arrays as 16-byte vectors (cp.async / double2): a misaligned pointer would
        // raise a sticky "misaligned address" fault that takes the whole CUDA context down
        if (((uintptr_t)sigma & 15u) != 0) {
            set_err(s, "pg_set_density: a PG_MEM_DEVICE density must be 16-byte aligned (got %p)", (const void *)sigma);
            return PG_ERR_INVALID_ARG;
        }
        s->d_sigma = sigma;
        s->sigma_from_host = false;
    } else if (where == PG_MEM_HOST || where == PG_MEM_HOST_PINNED) {
        pg_status st = ensure_staging(s, true, false);
        if (st != PG_OK) return st;
        if (where == PG_MEM_HOST && (st = ensure_pinned(s, true, false)) != PG_OK) return st;
        // the other staging slot: only the solves that read THAT one (two densities ago) must be done
        s->in_slot ^= 1;
        double *d_own = s->d_sigma_own[s->in_slot];
        PG_CUDA(s, cudaStreamWaitEvent(s->h2d, s->ev_in_free[s->in_slot], 0));
        for (int b = 0; b < batch; ++b) {
            const double *src = sigma + (size_t)b * s->field;
            if (where == PG_MEM_HOST) {
                double *stage = s->h_in + (size_t)b * s->field;
                if (s->in_pending[b]) PG_CUDA(s, cudaEventSynchronize(s->ev_in[b]));   // slot still in flight
                memcpy(stage, src, fbytes);
                src = stage;
            }
            PG_CUDA(s, cudaMemcpyAsync(d_own + (size_t)b * s->field, src, fbytes, cudaMemcpyHostToDevice, s->h2d));
            PG_CUDA(s, cudaEventRecord(s->ev_in[b], s->h2d));
            s->in_pending[b] = 1;
        }
        s->d_sigma = d_own;
        s->sigma_from_host = true;
    } else {
        set_err(s, "pg_set_density: unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    s->cur_batch = batch;
    return PG_OK;
}

static pg_status potential_common(pg_solver *s, double *phi, int batch, pg_memspace where, bool direct, int ring0,
                                  int n_rings)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!phi) { set_err(s, "phi is NULL"); return PG_ERR_INVALID_ARG; }
    if (s->cur_batch == 0 || !s->d_sigma) { set_err(s, "no density set: call pg_set_density first"); return PG_ERR_STATE; }
    if (batch != s->cur_batch) {
        set_err(s, "batch %d does not match the density's batch %d", batch, s->cur_batch);
        return PG_ERR_INVALID_ARG;
    }
    if (where != PG_MEM_DEVICE && where != PG_MEM_HOST && where != PG_MEM_HOST_PINNED) {
        set_err(s, "unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    const bool rings = n_rings >= 0;
    if (rings && (ring0 < 0 || n_rings < 1 || ring0 + n_rings > s->n_r)) {
        set_err(s, "ring range [%d, %d) outside [0, %d)", ring0, ring0 + n_rings, s->n_r);
        return PG_ERR_INVALID_ARG;
    }
    const size_t out_field = rings ? (size_t)n_rings * s->n_phi : s->field;
    const size_t obytes = out_field * sizeof(double);
    const bool host_out = where != PG_MEM_DEVICE;
    if (!host_out) {
        if (((uintptr_t)phi & 15u) != 0) {
            set_err(s, "a PG_MEM_DEVICE potential must be 16-byte aligned (got %p)", (void *)phi);
            return PG_ERR_INVALID_ARG;
        }
        // `phi` may not alias the density it is computed from (polargrav.h): the last kernel writes Phi rows
        // while other CTAs of the chain may still be reading Sigma rows of a later field or solve
        if (!s->sigma_from_host &&
            ranges_overlap(phi, (size_t)batch * out_field * sizeof(double), s->d_sigma, (size_t)batch * s->field * sizeof(double))) {
            set_err(s, "phi overlaps the density (in-place solves are not supported)");
            return PG_ERR_INVALID_ARG;
        }
    }
    pg_status st;
    if (host_out) {
        if ((st = ensure_staging(s, false, true)) != PG_OK) return st;
        if (where == PG_MEM_HOST && (st = ensure_pinned(s, false, true)) != PG_OK) return st;
    }

    if (!host_out && !s->sigma_from_host) {
        // everything resident: one batched launch per kernel
        if (direct) return launch_direct(s, s->d_sigma, phi, rings ? ring0 : 0, rings ? n_rings : s->n_r, batch);
        return solve_fields(s, s->d_sigma, phi, s->d_W, batch, true);
    }

    // staged pipeline: field b is solved as soon as its H2D copy has landed, and copied back
    // while field b+1 is being solved (copy streams h2d / d2h, compute on the caller's stream)
    double *d_out = nullptr;
    if (host_out) {
        // the other staging slot: only the downloads from THAT one (two potentials ago) must be done
        s->out_slot ^= 1;
        d_out = s->d_phi_own[s->out_slot];
        PG_CUDA(s, cudaStreamWaitEvent(s->stream, s->ev_out_done[s->out_slot], 0));
    }
    for (int b = 0; b < batch; ++b) {
        if (s->sigma_from_host) PG_CUDA(s, cudaStreamWaitEvent(s->stream, s->ev_in[b], 0));
        const double *sg = s->d_sigma + (size_t)b * s->field;
        double *dst = host_out ? d_out + (size_t)b * s->field : phi + (size_t)b * out_field;
        if (direct) st = launch_direct(s, sg, dst, rings ? ring0 : 0, rings ? n_rings : s->n_r, 1);
        else st = solve_fields(s, sg, dst, s->d_W + (size_t)b * (s->half + 1) * s->n_r, 1, false);
        if (st != PG_OK) return st;
        if (host_out) {
            PG_CUDA(s, cudaEventRecord(s->ev_solved[b], s->stream));
            PG_CUDA(s, cudaStreamWaitEvent(s->d2h, s->ev_solved[b], 0));
            double *hdst = (where == PG_MEM_HOST) ? s->h_out + (size_t)b * s->field : phi + (size_t)b * out_field;
            PG_CUDA(s, cudaMemcpyAsync(hdst, dst, obytes, cudaMemcpyDeviceToHost, s->d2h));
            PG_CUDA(s, cudaEventRecord(s->ev_out[b], s->d2h));
        }
    }
    if (host_out) PG_CUDA(s, cudaEventRecord(s->ev_out_done[s->out_slot], s->d2h));
    if (s->sigma_from_host) PG_CUDA(s, cudaEventRecord(s->ev_in_free[s->in_slot], s->stream));
    if (where == PG_MEM_HOST) {
        for (int b = 0; b < batch; ++b) {
            PG_CUDA(s, cudaEventSynchronize(s->ev_out[b]));
            memcpy(phi + (size_t)b * out_field, s->h_out + (size_t)b * s->field, obytes);
        }
    }
    return PG_OK;
}

pg_status pg_potential(pg_solver *s, double *phi, int batch, pg_memspace where)
{
    return potential_common(s, phi, batch, where, false, 0, -1);
}

pg_status pg_potential_series(pg_solver *s, const double *sigma, double *phi, int count, size_t stride)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!sigma || !phi || count < 1) { set_err(s, "pg_potential_series: sigma or phi is NULL, or count %d < 1", count); return PG_ERR_INVALID_ARG; }
    if (stride < s->field || (stride & 1u)) {
        set_err(s, "pg_potential_series: stride %zu must be even and >= n_r * n_phi = %zu doubles", stride, s->field);
        return PG_ERR_INVALID_ARG;
    }
    if ((((uintptr_t)sigma | (uintptr_t)phi) & 15u) != 0) {
        set_err(s, "pg_potential_series: sigma and phi must be 16-byte aligned device pointers");
        return PG_ERR_INVALID_ARG;
    }
    const size_t span = ((size_t)(count - 1) * stride + s->field) * sizeof(double);
    if (ranges_overlap(sigma, span, phi, span)) {
        set_err(s, "pg_potential_series: the phi range overlaps the sigma range");
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    s->sigma_from_host = false;
    s->cur_batch = 1;
    for (int k = 0; k < count; ++k) {
        s->d_sigma = sigma + (size_t)k * stride;
        pg_status st = solve_fields(s, s->d_sigma, phi + (size_t)k * stride, s->d_W, 1, true);
        if (st != PG_OK) return st;
    }
    return PG_OK;
}

pg_status pg_potential_direct(pg_solver *s, double *phi, int batch, pg_memspace where)
{
    return potential_common(s, phi, batch, where, true, 0, -1);
}

pg_status pg_potential_direct_rings(pg_solver *s, double *phi, int ring0, int n_rings, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (n_rings < 1) { set_err(s, "n_rings must be >= 1"); return PG_ERR_INVALID_ARG; }
    const int saved = s->cur_batch;
    if (saved == 0) { set_err(s, "no density set: call pg_set_density first"); return PG_ERR_STATE; }
    s->cur_batch = 1;   // field 0 only
    pg_status st = potential_common(s, phi, 1, where, true, ring0, n_rings);
    s->cur_batch = saved;
    return st;
}

pg_status pg_set_softening(pg_solver *s, pg_softening mode)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (mode != PG_SOFT_SYMMETRIC && mode != PG_SOFT_FIELD && mode != PG_SOFT_SOURCE) {
        set_err(s, "pg_set_softening: unknown mode %d", (int)mode);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    PG_CUDA(s, cudaStreamSynchronize(s->stream));
    if ((int)mode != s->soft) {
        s->soft = (int)mode;
        for (int k = 0; k < 3; ++k) s->khat_c_valid[k] = false;
    }
    return mode == PG_SOFT_SYMMETRIC ? PG_OK : build_khat_variant(s, 0);
}

pg_status pg_acceleration(pg_solver *s, double *a_r, double *a_phi, int batch, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!a_r || !a_phi) { set_err(s, "pg_acceleration: a_r or a_phi is NULL"); return PG_ERR_INVALID_ARG; }
    if (s->cur_batch == 0 || !s->d_sigma) { set_err(s, "no density set: call pg_set_density first"); return PG_ERR_STATE; }
    if (batch != s->cur_batch) {
        set_err(s, "batch %d does not match the density's batch %d", batch, s->cur_batch);
        return PG_ERR_INVALID_ARG;
    }
    if (where != PG_MEM_DEVICE && where != PG_MEM_HOST && where != PG_MEM_HOST_PINNED) {
        set_err(s, "unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    const size_t bytes = (size_t)batch * s->field * sizeof(double);
    double *outs[2] = {a_r, a_phi};
    if (where == PG_MEM_DEVICE) {
        if ((((uintptr_t)a_r | (uintptr_t)a_phi) & 15u) != 0) {
            set_err(s, "PG_MEM_DEVICE outputs must be 16-byte aligned");
            return PG_ERR_INVALID_ARG;
        }
        if (ranges_overlap(a_r, bytes, a_phi, bytes) ||
            (!s->sigma_from_host && (ranges_overlap(a_r, bytes, s->d_sigma, bytes) || ranges_overlap(a_phi, bytes, s->d_sigma, bytes)))) {
            set_err(s, "a_r, a_phi and the density may not overlap");
            return PG_ERR_INVALID_ARG;
        }
    } else {
        // host outputs: through the owned device staging slots (two potentials' worth), blocking
        pg_status st = ensure_staging(s, false, true);
        if (st != PG_OK) return st;
        PG_CUDA(s, cudaStreamSynchronize(s->d2h));
        outs[0] = s->d_phi_own[0];
        outs[1] = s->d_phi_own[1];
    }
    if (s->sigma_from_host)
        for (int b = 0; b < batch; ++b) PG_CUDA(s, cudaStreamWaitEvent(s->stream, s->ev_in[b], 0));
    const int kinds[2] = {1, 2};
    pg_status st = solve_variant(s, s->d_sigma, s->d_W, batch, 2, kinds, outs);
    if (st != PG_OK) return st;
    if (s->sigma_from_host) PG_CUDA(s, cudaEventRecord(s->ev_in_free[s->in_slot], s->stream));
    if (where != PG_MEM_DEVICE) {
        PG_CUDA(s, cudaMemcpyAsync(a_r, outs[0], bytes, cudaMemcpyDeviceToHost, s->stream));
        PG_CUDA(s, cudaMemcpyAsync(a_phi, outs[1], bytes, cudaMemcpyDeviceToHost, s->stream));
        PG_CUDA(s, cudaStreamSynchronize(s->stream));
    }
    return PG_OK;
}

pg_status pg_grid(const pg_solver *s, double *r, double *phi, double *cell_area)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (r) memcpy(r, s->r.data(), s->r.size() * sizeof(double));
    if (phi) memcpy(phi, s->phi.data(), s->phi.size() * sizeof(double));
    if (cell_area) memcpy(cell_area, s->dA.data(), s->dA.size() * sizeof(double));
    return PG_OK;
}

pg_status pg_set_stream(pg_solver *s, void *cuda_stream)
{
    if (!s) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    pg_status st = drain_profile(s);
    if (st != PG_OK) return st;
    PG_CUDA(s, cudaStreamSynchronize(s->stream));
    forget_early_release_output(s->device, s->stream);
    if ((st = lanes_drain(s)) != PG_OK) return st;
    s->stream = (cudaStream_t)cuda_stream;
    return PG_OK;
}

pg_status pg_set_option(pg_solver *s, pg_option option, int value)
{
    if (!s) return PG_ERR_INVALID_ARG;
    switch (option) {
        case PG_OPT_DENSITY_STABLE: s->density_stable = value != 0; return PG_OK;
        case PG_OPT_FUSED: s->fused = value != 0; return PG_OK;
        case PG_OPT_LANES: {
            if (value < 1 || value > PG_MAX_LANES) { set_err(s, "PG_OPT_LANES: 1 .. %d", PG_MAX_LANES); return PG_ERR_INVALID_ARG; }
            DeviceGuard guard(s->device);
            PG_CUDA(s, cudaStreamSynchronize(s->stream));      // what is in flight on the solver's stream comes first
            pg_status st = lanes_drain(s);
            if (st != PG_OK) return st;
            if (value >= 2 && (st = lanes_enable(s, value)) != PG_OK) return st;
            s->lanes = value;
            s->lane_next = 0;
            return PG_OK;
        }
    }
    set_err(s, "pg_set_option: unknown option %d", (int)option);
    return PG_ERR_INVALID_ARG;
}

pg_status pg_flush(pg_solver *s)
{
    if (!s) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    for (int L = 0; L < PG_MAX_LANES; ++L)
        if (s->lane_used[L]) {
            PG_CUDA(s, cudaEventRecord(s->lane_done[L], s->lane_stream[L]));
            PG_CUDA(s, cudaStreamWaitEvent(s->stream, s->lane_done[L], 0));
        }
    return PG_OK;
}

pg_status pg_synchronize(pg_solver *s)
{
    if (!s) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    PG_CUDA(s, cudaStreamSynchronize(s->h2d));
    PG_CUDA(s, cudaStreamSynchronize(s->stream));
    PG_CUDA(s, cudaStreamSynchronize(s->d2h));
    forget_early_release_output(s->device, s->stream);
    return lanes_drain(s);
}

pg_status pg_host_alloc(void **p, size_t bytes)
{
    if (!p || bytes == 0) return PG_ERR_INVALID_ARG;
    *p = nullptr;
    cudaError_t e = cudaHostAlloc(p, bytes, cudaHostAllocDefault);
    if (e != cudaSuccess) {
        set_err(nullptr, "cudaHostAlloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
        return e == cudaErrorMemoryAllocation ? PG_ERR_NOMEM : PG_ERR_CUDA;
    }
    return PG_OK;
}

pg_status pg_host_free(void *p)
{
    if (!p) return PG_OK;
    cudaError_t e = cudaFreeHost(p);
    if (e != cudaSuccess) { set_err(nullptr, "cudaFreeHost failed: %s", cudaGetErrorString(e)); return PG_ERR_CUDA; }
    return PG_OK;
}

pg_status pg_profile(pg_solver *s, int enable)
{
    if (!s) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    pg_status st = drain_profile(s);
    if (st != PG_OK) return st;
    s->profile = enable != 0;
    if (enable) for (int k = 0; k < PG_NUM_KERNELS; ++k) { s->prof_ms[k] = 0.0; s->prof_n[k] = 0; }
    return PG_OK;
}

pg_status pg_kernel_times(pg_solver *s, double ms[PG_NUM_KERNELS], long launches[PG_NUM_KERNELS])
{
    if (!s || !ms || !launches) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    pg_status st = drain_profile(s);
    if (st != PG_OK) return st;
    for (int k = 0; k < PG_NUM_KERNELS; ++k) { ms[k] = s->prof_ms[k]; launches[k] = s->prof_n[k]; }
    return PG_OK;
}

long pg_launch_count(const pg_solver *s) { return s ? s->launches : 0; }

double pg_kernel_algorithmic_bytes(const pg_solver *s, int index, int batch)
{
    if (!s || batch < 1) return 0.0;
    const double cells = (double)s->n_r * s->n_phi;
    // Hermitian half-spectrum of M_h = n_phi/2 + 1 modes (the columns of W)
    const double m_h = s->half + 1;
    const double spec = 16.0 * s->n_r * m_h;          // one half-spectrum, complex128
    const double khat = 8.0 * 2.0 * s->n_r * m_h;     // real spectrum of the padded kernel
    switch (index) {
        case 0: return batch * (8.0 * cells + spec);              // read Sigma, write W
        case 1: return batch * (2.0 * spec) + khat;               // read W, write W, read Khat once
        case 2: return batch * (spec + 8.0 * cells);              // read W, write Phi
        default: return 0.0;
    }
}

double pg_algorithmic_bytes(const pg_solver *s, int batch)
{
    return pg_kernel_algorithmic_bytes(s, 0, batch) + pg_kernel_algorithmic_bytes(s, 1, batch) +
           pg_kernel_algorithmic_bytes(s, 2, batch);
}

const char *pg_status_string(pg_status st)
{
    switch (st) {
        case PG_OK: return "PG_OK";
        case PG_ERR_INVALID_ARG: return "PG_ERR_INVALID_ARG";
        case PG_ERR_UNSUPPORTED: return "PG_ERR_UNSUPPORTED";
        case PG_ERR_CUDA: return "PG_ERR_CUDA";
        case PG_ERR_NOMEM: return "PG_ERR_NOMEM";
        case PG_ERR_STATE: return "PG_ERR_STATE";
    }
    return "PG_ERR_UNKNOWN";
}

const char *pg_last_error(const pg_solver *s) { return s ? s->err : g_create_error; }

const char *pg_version(void) { return "polargrav 0.1 (sm_100a)"; }

}  // extern "C"

// =================================================================== NEXT-2: one 3-D Cartesian mesh level
struct pg3_solver {
    int n = 0, device = 0;
    double box = 0, h = 0;
    pg_solver *inner = nullptr;      // tables, stream and launch helpers of a polar solver with n_r = n, n_phi = 2 n
    cplx *d_Yt = nullptr;            // [n+1][2n][n]: spectrum after the x and y passes, z contiguous
    double *d_ghat = nullptr;        // [n+1][2n][2n] real spectrum of the Green's function (all normalisations folded in)
    double *d_ones = nullptr;        // post-scale of the inverse x pass (none)
    double *d_rho = nullptr, *d_phi = nullptr;   // staging for host memspaces (lazily allocated)
    const double *cur_rho = nullptr;
    bool rho_from_host = false;
    char err[512] = "";
};

namespace {

void set_err3(pg3_solver *s, const char *fmt, ...)
{
    char *dst = s ? s->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
}
#define PG3_CUDA(s, call)                                                                      \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            set_err3((s), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return e_ == cudaErrorMemoryAllocation ? PG_ERR_NOMEM : PG_ERR_CUDA;               \
        }                                                                                      \
    } while (0)

template <int N>
pg_status cart_build_ghat(pg3_solver *s)
{
    typedef pgk::ColShape<N> S;
    constexpr int M = 2 * N;
    pg_solver *in = s->inner;
    cudaStream_t st = in->stream;
    const long g_n = (long)M * M * M, gw_n = (long)M * (N + 1) * M;
    double *d_g = nullptr;
    cplx *d_gw = nullptr, *d_gy = nullptr;
    PG3_CUDA(s, cudaMalloc((void **)&d_g, g_n * sizeof(double)));
    if (cudaMalloc((void **)&d_gw, gw_n * sizeof(cplx)) != cudaSuccess || cudaMalloc((void **)&d_gy, gw_n * sizeof(cplx)) != cudaSuccess) {
        cudaFree(d_g); cudaFree(d_gw); cudaFree(d_gy);
        set_err3(s, "out of device memory for the Green's function workspace");
        return PG_ERR_NOMEM;
    }
    pg_status rc = PG_OK;
    do {
        const double self = 3.0 * std::log(2.0 + std::sqrt(3.0)) - 2.0 * std::atan(1.0);      // reading C3
        pgk::green3_fill_kernel<<<(unsigned)((g_n + 255) / 256), 256, 0, st>>>(d_g, N, self, g_n);
        // x' pass: the 2N x 2N rows as 2N fields of 2N rows -> GW[z'][kx][y']
        rc = rows_fwd(in, d_g, d_gw, nullptr, M, M, (long)M * M, (long)(N + 1) * M, st, 0);
        if (rc != PG_OK) { snprintf(s->err, sizeof s->err, "%s", in->err); break; }
        const size_t smem = S::LINES;
        cudaFuncSetAttribute(pgk::gcols_kernel<N, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        cudaFuncSetAttribute(pgk::gcols_kernel<N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        const int n_cols = M * (N + 1);
        const unsigned grid = (unsigned)((n_cols + S::MODES - 1) / S::MODES);
        // -G h^2 (cells as point masses: h^3 / h), and the normalisation of the unnormalised transforms: x pair 1/(2M)
        // (packed real transform: 2 X on the way in, 2 Z on the way out) and another 1/2 because the kernel's own x'
        // pass forms 2 X; y and z pairs 1/M each.
        const double scale = -s->h * s->h / (4.0 * (double)M * (double)M * (double)M);
        pgk::gcols_kernel<N, 0><<<grid, S::THREADS, smem, st>>>(d_gw, d_gy, nullptr, in->d_tw_col, n_cols, 0.0);
        pgk::gcols_kernel<N, 1><<<grid, S::THREADS, smem, st>>>(d_gy, nullptr, s->d_ghat, in->d_tw_col, n_cols, scale);
        in->launches += 3;
        if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) {
            set_err3(s, "Green's function precompute failed: %s", cudaGetErrorString(cudaGetLastError()));
            rc = PG_ERR_CUDA;
        }
    } while (0);
    cudaFree(d_g); cudaFree(d_gw); cudaFree(d_gy);
    return rc;
}

template <int N>
pg_status cart_solve(pg3_solver *s, const double *d_rho, double *d_phi)
{
    typedef pgk::ColShape<N> S;
    constexpr int M = 2 * N;
    pg_solver *in = s->inner;
    cudaStream_t st = in->stream;
    const long ws = (long)(N + 1) * N;
    typedef pgk::RowShape<M> RS;
    const int n_items = (N / RS::ROWS) * N;
    const int rgrid = n_items < in->row_ctas ? n_items : in->row_ctas;
    PG3_CUDA(s, cudaFuncSetAttribute(pgk::rows_fwd_kernel<M, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RS::SMEM));
    PG3_CUDA(s, cudaFuncSetAttribute(pgk::rows_inv_kernel<M, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RS::SMEM));
    // x pass: N fields (z) of N rows (y) of N reals, zero padded to M inside the kernel -> W1[z][kx][y]
    PG3_CUDA(s, launch_pdl(pgk::rows_fwd_kernel<M, true>, dim3(rgrid), dim3(RS::THREADS), RS::SMEM, st, d_rho, in->d_W,
                           (const cplx *)in->d_tw_row, (const double *)nullptr, N, n_items, (long)N * N, ws, 0));
    in->launches++;
    typedef pgk::YShape<N> Y;
    const unsigned ygrid = (unsigned)((N + 1) * N / Y::YM);
    PG3_CUDA(s, cudaFuncSetAttribute(pgk::ycols_fwd_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Y::SMEM));
    PG3_CUDA(s, cudaFuncSetAttribute(pgk::ycols_inv_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Y::SMEM));
    pgk::ycols_fwd_kernel<N><<<ygrid, Y::THREADS, Y::SMEM, st>>>(in->d_W, s->d_Yt, in->d_tw_col);
    in->launches++;
    // z pass: cols_kernel unchanged -- zero-padded 2N-point transform x Ghat, inverse, crop -- over the (N+1) 2N columns
    const int n_modes = (N + 1) * M;
    dim3 zgrid((n_modes + S::MODES - 1) / S::MODES, 1);
    PG3_CUDA(s, launch_pdl(pgk::cols_kernel<N>, zgrid, dim3(S::THREADS), S::SMEM, st, s->d_Yt, (const double *)s->d_ghat,
                           (const cplx *)in->d_tw_col, n_modes, 0L));
    in->launches++;
    pgk::ycols_inv_kernel<N><<<ygrid, Y::THREADS, Y::SMEM, st>>>(s->d_Yt, in->d_W, in->d_tw_col);
    in->launches++;
    // inverse x pass, cropped to the first N reals of every row: Phi[z][y][x]
    typedef pgk::RowShape<M, true> RSI;
    static_assert(RSI::ROWS == RS::ROWS && RSI::SMEM == RS::SMEM, "one row shape below 2048");
    const int rgrid_inv = n_items < in->row_ctas_inv ? n_items : in->row_ctas_inv;
    PG3_CUDA(s, launch_pdl(pgk::rows_inv_kernel<M, true>, dim3(rgrid_inv), dim3(RSI::THREADS), RSI::SMEM, st, (const cplx *)in->d_W,
                           d_phi, (const cplx *)in->d_tw_row, (const double *)s->d_ones, N, n_items, ws, (long)N * N, CUtensorMap{}));
    in->launches++;
    // rows_inv_kernel releases its dependents before it has finished writing: a polar solver on this stream that is
    // fed Phi as its density must not fetch it early (same per-stream record as launch_rows_inv keeps)
    note_early_release_output(s->device, st, d_phi, (size_t)N * N * N * sizeof(double));
    PG3_CUDA(s, cudaGetLastError());
    return PG_OK;
}

#define PG3_DISPATCH(n, CALL)                          \
    switch (n) {                                        \
        case 32: return CALL(32);                       \
        case 64: return CALL(64);                       \
        case 128: return CALL(128);                     \
        case 256: return CALL(256);                     \
        default: return PG_ERR_UNSUPPORTED;             \
    }
pg_status cart_build(pg3_solver *s)
{
#define CALL(N) cart_build_ghat<N>(s)
    PG3_DISPATCH(s->n, CALL)
#undef CALL
}
pg_status cart_run(pg3_solver *s, const double *d_rho, double *d_phi)
{
#define CALL(N) cart_solve<N>(s, d_rho, d_phi)
    PG3_DISPATCH(s->n, CALL)
#undef CALL
}

void cart_free(pg3_solver *s)
{
    if (!s) return;
    cudaFree(s->d_Yt); cudaFree(s->d_ghat); cudaFree(s->d_ones); cudaFree(s->d_rho); cudaFree(s->d_phi);
    if (s->inner) pg_destroy(s->inner);
    delete s;
}

}  // namespace

extern "C" {

pg_status pg3_create(pg3_solver **out, int n, double box, int device, void *cuda_stream)
{
    g_create_error[0] = 0;
    if (!out) { set_err3(nullptr, "out is NULL"); return PG_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!(box > 0.0) || !std::isfinite(box)) { set_err3(nullptr, "invalid argument: need box > 0"); return PG_ERR_INVALID_ARG; }
    if (n != 32 && n != 64 && n != 128 && n != 256) {
        set_err3(nullptr, "unsupported mesh %d^3: n must be 32, 64, 128 or 256", n);
        return PG_ERR_UNSUPPORTED;
    }
    pg3_solver *s = new (std::nothrow) pg3_solver;
    if (!s) { set_err3(nullptr, "out of host memory"); return PG_ERR_NOMEM; }
    s->n = n; s->box = box; s->h = box / n;
    // tables (twiddles of the 2n-point transforms), stream and workspace W1 = [n][n+1][n] come with a polar solver of
    // n_r = n, n_phi = 2n, max_batch = n; its own Green's kernel is not used
    pg_status rc = pg_create_ex(&s->inner, n, 2 * n, 1.0, 2.0, 1.0, n, device, cuda_stream);
    if (rc != PG_OK) { delete s; return rc; }
    s->device = s->inner->device;
    DeviceGuard guard(s->device);
    const size_t m = 2 * (size_t)n;
    std::vector<double> ones(n, 1.0);
    cudaError_t e = cudaMalloc((void **)&s->d_Yt, (size_t)(n + 1) * m * n * sizeof(cplx));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_ghat, (size_t)(n + 1) * m * m * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void **)&s->d_ones, n * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(s->d_ones, ones.data(), n * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        const bool nomem = e == cudaErrorMemoryAllocation;
        set_err3(nullptr, nomem ? "device allocation failed: %s" : "pg3_create: CUDA error while setting up the mesh: %s", cudaGetErrorString(e));
        (void)cudaGetLastError();
        cart_free(s);
        return nomem ? PG_ERR_NOMEM : PG_ERR_CUDA;
    }
    rc = cart_build(s);
    if (rc != PG_OK) {
        snprintf(g_create_error, sizeof g_create_error, "%s", s->err);
        cart_free(s);
        return rc;
    }
    *out = s;
    return PG_OK;
}

pg_status pg3_set_density(pg3_solver *s, const double *rho, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!rho) { set_err3(s, "pg3_set_density: rho is NULL"); return PG_ERR_INVALID_ARG; }
    DeviceGuard guard(s->device);
    const size_t bytes = (size_t)s->n * s->n * s->n * sizeof(double);
    if (where == PG_MEM_DEVICE) {
        if (((uintptr_t)rho & 15u) != 0) { set_err3(s, "a PG_MEM_DEVICE density must be 16-byte aligned"); return PG_ERR_INVALID_ARG; }
        s->cur_rho = rho;
        s->rho_from_host = false;
    } else if (where == PG_MEM_HOST || where == PG_MEM_HOST_PINNED) {
        if (!s->d_rho) PG3_CUDA(s, cudaMalloc((void **)&s->d_rho, bytes));
        PG3_CUDA(s, cudaMemcpyAsync(s->d_rho, rho, bytes, cudaMemcpyHostToDevice, s->inner->stream));
        if (where == PG_MEM_HOST) PG3_CUDA(s, cudaStreamSynchronize(s->inner->stream));
        s->cur_rho = s->d_rho;
        s->rho_from_host = true;
    } else {
        set_err3(s, "pg3_set_density: unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    return PG_OK;
}

pg_status pg3_potential(pg3_solver *s, double *phi, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!phi) { set_err3(s, "pg3_potential: phi is NULL"); return PG_ERR_INVALID_ARG; }
    if (!s->cur_rho) { set_err3(s, "no density set: call pg3_set_density first"); return PG_ERR_STATE; }
    DeviceGuard guard(s->device);
    const size_t bytes = (size_t)s->n * s->n * s->n * sizeof(double);
    if (where == PG_MEM_DEVICE) {
        if (((uintptr_t)phi & 15u) != 0) { set_err3(s, "a PG_MEM_DEVICE potential must be 16-byte aligned"); return PG_ERR_INVALID_ARG; }
        if (!s->rho_from_host && ranges_overlap(phi, bytes, s->cur_rho, bytes)) {
            set_err3(s, "phi overlaps the density");
            return PG_ERR_INVALID_ARG;
        }
        return cart_run(s, s->cur_rho, phi);
    }
    if (where != PG_MEM_HOST && where != PG_MEM_HOST_PINNED) { set_err3(s, "unknown memspace %d", (int)where); return PG_ERR_INVALID_ARG; }
    if (!s->d_phi) PG3_CUDA(s, cudaMalloc((void **)&s->d_phi, bytes));
    pg_status rc = cart_run(s, s->cur_rho, s->d_phi);
    if (rc != PG_OK) return rc;
    PG3_CUDA(s, cudaMemcpyAsync(phi, s->d_phi, bytes, cudaMemcpyDeviceToHost, s->inner->stream));
    if (where == PG_MEM_HOST) PG3_CUDA(s, cudaStreamSynchronize(s->inner->stream));
    return PG_OK;
}

pg_status pg3_synchronize(pg3_solver *s)
{
    if (!s) return PG_ERR_INVALID_ARG;
    return pg_synchronize(s->inner);
}

pg_status pg3_destroy(pg3_solver *s)
{
    if (!s) return PG_OK;
    DeviceGuard guard(s->device);
    cudaStreamSynchronize(s->inner->stream);
    cart_free(s);
    return PG_OK;
}

long pg3_launch_count(const pg3_solver *s) { return s ? s->inner->launches : 0; }

const char *pg3_last_error(const pg3_solver *s) { return s ? s->err : g_create_error; }

/* Algorithmic HBM bytes of one pg3_potential call: rho in, Phi out, and each intermediate
 * spectrum written and read once at its pruned size -- x pass out / y pass in (n+1) n^2, y pass out / z pass in-out /
 * y pass in (n+1) 2n n, complex128 -- plus the real Green's spectrum (n+1)(2n)^2 once. */
double pg3_algorithmic_bytes(const pg3_solver *s)
{
    if (!s) return 0.0;
    const double n = s->n, cells = n * n * n;
    const double w1 = 16.0 * (n + 1) * n * n, yt = 16.0 * (n + 1) * 2.0 * n * n, gh = 8.0 * (n + 1) * 4.0 * n * n;
    return 2.0 * 8.0 * cells + 2.0 * w1 + 2.0 * w1 + 4.0 * yt + gh;
}

}  // extern "C"

// =================================================================== NEXT-3: nested 3-D mesh levels
// One object per level ("each nested mesh was allocated one GPU"): the level's own single-level solver
// (box_0 / 2^level) plus the buffers of the coupling steps of nested.cuh.  Every call enqueues on the level's stream
// and returns; the caller (paper_2409_02294_b200/nested.py) moves the two small boundary messages between levels --
// (n/2)^3 restricted densities upwards, (n/2 + 2)^3 exterior potentials downwards -- by pointer on one GPU or by
// NCCL send / recv between GPUs.
struct pg3n_level {
    int n = 0, level = 0, depth = 1, device = 0;
    pg3_solver *mesh = nullptr;
    double *d_rho = nullptr, *d_mask = nullptr, *d_own = nullptr, *d_out = nullptr, *d_ext = nullptr, *d_phi = nullptr;
    bool have_rho = false, solved = false, have_phi = false;
    // one-sided exchange: this level's two inboxes (owned, cudaMalloc'ed so that they can be exported to
    // another process) and the neighbours' inboxes it puts into ([0] the parent's MEAN inbox, [1] the child's HALO inbox)
    double *inbox[2] = {nullptr, nullptr};
    double *peer[2] = {nullptr, nullptr};
    bool peer_ipc[2] = {false, false};
    long launches = 0;
    char err[512] = "";
};

namespace {

void set_err3n(pg3n_level *s, const char *fmt, ...)
{
    char *dst = s ? s->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
}
#define PG3N_CUDA(s, call)                                                                     \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            set_err3n((s), "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return e_ == cudaErrorMemoryAllocation ? PG_ERR_NOMEM : PG_ERR_CUDA;               \
        }                                                                                      \
    } while (0)

unsigned blocks_for(long count) { return (unsigned)((count + 255) / 256); }

bool dev_ptr_ok(pg3n_level *s, const void *p, const char *what)
{
    if (!p) { set_err3n(s, "%s is NULL", what); return false; }
    if (((uintptr_t)p & 15u) != 0) { set_err3n(s, "%s must be a 16-byte aligned device pointer", what); return false; }
    return true;
}

void nest_free(pg3n_level *s)
{
    if (!s) return;
    cudaFree(s->d_rho); cudaFree(s->d_mask); cudaFree(s->d_own); cudaFree(s->d_out); cudaFree(s->d_ext); cudaFree(s->d_phi);
    for (int k = 0; k < 2; ++k) {
        if (s->peer[k] && s->peer_ipc[k]) cudaIpcCloseMemHandle(s->peer[k]);
        cudaFree(s->inbox[k]);
    }
    if (s->mesh) pg3_destroy(s->mesh);
    delete s;
}

}  // namespace

extern "C" {

pg_status pg3n_create(pg3n_level **out, int n, double box0, int level, int depth, int device, void *cuda_stream)
{
    g_create_error[0] = 0;
    if (!out) { set_err3n(nullptr, "out is NULL"); return PG_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!(box0 > 0.0) || !std::isfinite(box0) || depth < 1 || depth > 32 || level < 0 || level >= depth) {
        set_err3n(nullptr, "invalid argument: need box0 > 0, 1 <= depth <= 32, 0 <= level < depth");
        return PG_ERR_INVALID_ARG;
    }
    pg3n_level *s = new (std::nothrow) pg3n_level;
    if (!s) { set_err3n(nullptr, "out of host memory"); return PG_ERR_NOMEM; }
    s->n = n; s->level = level; s->depth = depth;
    pg_status rc = pg3_create(&s->mesh, n, std::ldexp(box0, -level), device, cuda_stream);   // M1: box_l = box_0 / 2^l
    if (rc != PG_OK) { delete s; return rc; }
    s->device = s->mesh->device;
    DeviceGuard guard(s->device);
    const size_t bytes = (size_t)n * n * n * sizeof(double);
    double **bufs[] = {&s->d_rho, &s->d_mask, &s->d_own, &s->d_out, &s->d_ext, &s->d_phi};
    for (double **b : bufs) {
        if (b == &s->d_mask || b == &s->d_out) { if (level == depth - 1) continue; }          // the finest level has no child
        if (cudaMalloc((void **)b, bytes) != cudaSuccess) {
            set_err3n(nullptr, "out of device memory for the level's buffers");
            nest_free(s);
            return PG_ERR_NOMEM;
        }
    }
    *out = s;
    return PG_OK;
}

pg_status pg3n_set_density(pg3n_level *s, const double *rho, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!rho) { set_err3n(s, "pg3n_set_density: rho is NULL"); return PG_ERR_INVALID_ARG; }
    if (where != PG_MEM_DEVICE && where != PG_MEM_HOST && where != PG_MEM_HOST_PINNED) {
        set_err3n(s, "pg3n_set_density: unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    cudaStream_t st = s->mesh->inner->stream;
    const size_t bytes = (size_t)s->n * s->n * s->n * sizeof(double);
    // always copied: M2 rewrites the central cells of every level that has a child
    PG3N_CUDA(s, cudaMemcpyAsync(s->d_rho, rho, bytes, where == PG_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    if (where == PG_MEM_HOST) PG3N_CUDA(s, cudaStreamSynchronize(st));
    s->have_rho = true; s->solved = false; s->have_phi = false;
    return PG_OK;
}

pg_status pg3n_restrict(pg3n_level *s, double *child_mean_out)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!s->have_rho) { set_err3n(s, "no density set"); return PG_ERR_STATE; }
    if (s->level == 0) { set_err3n(s, "level 0 has no parent to restrict to"); return PG_ERR_STATE; }
    if (!child_mean_out) {                     // one-sided: straight into the parent's inbox (peer memory)
        if (!s->peer[PG3N_INBOX_MEAN]) { set_err3n(s, "pg3n_restrict(NULL): the parent's inbox has not been opened (pg3n_peer_open / pg3n_peer_set)"); return PG_ERR_STATE; }
        child_mean_out = s->peer[PG3N_INBOX_MEAN];
    }
    if (!dev_ptr_ok(s, child_mean_out, "child_mean_out")) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    const long q = s->n / 2;
    pgk::nest_restrict_kernel<<<blocks_for(q * q * q), 256, 0, s->mesh->inner->stream>>>(s->d_rho, child_mean_out, s->n);
    PG3N_CUDA(s, cudaGetLastError());
    s->launches++;
    return PG_OK;
}

pg_status pg3n_absorb(pg3n_level *s, const double *child_mean)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!s->have_rho) { set_err3n(s, "no density set"); return PG_ERR_STATE; }
    if (s->level == s->depth - 1) { set_err3n(s, "the finest level has no child to absorb"); return PG_ERR_STATE; }
    if (!child_mean) {                         // one-sided: what the child has put into this level's inbox
        if (!s->inbox[PG3N_INBOX_MEAN]) { set_err3n(s, "pg3n_absorb(NULL): this level has no MEAN inbox (pg3n_inbox_export)"); return PG_ERR_STATE; }
        child_mean = s->inbox[PG3N_INBOX_MEAN];
    }
    if (!dev_ptr_ok(s, child_mean, "child_mean")) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    const long q = s->n / 2;
    pgk::nest_absorb_kernel<<<blocks_for(q * q * q), 256, 0, s->mesh->inner->stream>>>(s->d_rho, child_mean, s->n);
    PG3N_CUDA(s, cudaGetLastError());
    s->launches++;
    s->solved = false;
    return PG_OK;
}

pg_status pg3n_solve(pg3n_level *s)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!s->have_rho) { set_err3n(s, "no density set"); return PG_ERR_STATE; }
    DeviceGuard guard(s->device);
    const long before = s->mesh->inner->launches;
    pg_status rc = cart_run(s->mesh, s->d_rho, s->d_own);                                  // M3: own_l
    if (rc == PG_OK && s->level < s->depth - 1) {
        const long cells = (long)s->n * s->n * s->n;
        pgk::nest_mask_kernel<<<blocks_for(cells), 256, 0, s->mesh->inner->stream>>>(s->d_rho, s->d_mask, s->n);
        s->launches++;
        rc = cart_run(s->mesh, s->d_mask, s->d_out);                                       // M3: out_l
    }
    if (rc != PG_OK) { snprintf(s->err, sizeof s->err, "%s", s->mesh->err); return rc; }
    PG3N_CUDA(s, cudaGetLastError());
    s->launches += s->mesh->inner->launches - before;
    s->solved = true; s->have_phi = false;
    return PG_OK;
}

pg_status pg3n_add_exterior(pg3n_level *s, const double *parent_halo)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!s->solved) { set_err3n(s, "pg3n_add_exterior before pg3n_solve"); return PG_ERR_STATE; }
    if (s->level == 0 && parent_halo) { set_err3n(s, "level 0 is isolated: parent_halo must be NULL"); return PG_ERR_INVALID_ARG; }
    if (s->level > 0 && !parent_halo) {        // one-sided: what the parent has put into this level's inbox
        if (!s->inbox[PG3N_INBOX_HALO]) { set_err3n(s, "parent_halo is NULL and this level has no HALO inbox (pg3n_inbox_export)"); return PG_ERR_STATE; }
        parent_halo = s->inbox[PG3N_INBOX_HALO];
    }
    if (s->level > 0 && !dev_ptr_ok(s, parent_halo, "parent_halo")) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    const long cells = (long)s->n * s->n * s->n;
    pgk::nest_prolong_kernel<<<blocks_for(cells), 256, 0, s->mesh->inner->stream>>>(parent_halo, s->d_own, s->d_ext, s->d_phi, s->n);
    PG3N_CUDA(s, cudaGetLastError());
    s->launches++;
    s->have_phi = true;
    return PG_OK;
}

pg_status pg3n_pack_exterior(pg3n_level *s, double *halo_out)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!s->have_phi) { set_err3n(s, "pg3n_pack_exterior before pg3n_add_exterior"); return PG_ERR_STATE; }
    if (s->level == s->depth - 1) { set_err3n(s, "the finest level has no child"); return PG_ERR_STATE; }
    if (!halo_out) {                           // one-sided: straight into the child's inbox (peer memory)
        if (!s->peer[PG3N_INBOX_HALO]) { set_err3n(s, "pg3n_pack_exterior(NULL): the child's inbox has not been opened (pg3n_peer_open / pg3n_peer_set)"); return PG_ERR_STATE; }
        halo_out = s->peer[PG3N_INBOX_HALO];
    }
    if (!dev_ptr_ok(s, halo_out, "halo_out")) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    const long m = s->n / 2 + 2;
    pgk::nest_pack_kernel<<<blocks_for(m * m * m), 256, 0, s->mesh->inner->stream>>>(s->d_out, s->d_ext, halo_out, s->n);
    PG3N_CUDA(s, cudaGetLastError());
    s->launches++;
    return PG_OK;
}

pg_status pg3n_potential(pg3n_level *s, double *phi, pg_memspace where)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!phi) { set_err3n(s, "pg3n_potential: phi is NULL"); return PG_ERR_INVALID_ARG; }
    if (!s->have_phi) { set_err3n(s, "pg3n_potential before pg3n_add_exterior"); return PG_ERR_STATE; }
    if (where != PG_MEM_DEVICE && where != PG_MEM_HOST && where != PG_MEM_HOST_PINNED) {
        set_err3n(s, "unknown memspace %d", (int)where);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(s->device);
    cudaStream_t st = s->mesh->inner->stream;
    const size_t bytes = (size_t)s->n * s->n * s->n * sizeof(double);
    PG3N_CUDA(s, cudaMemcpyAsync(phi, s->d_phi, bytes, where == PG_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    if (where == PG_MEM_HOST) PG3N_CUDA(s, cudaStreamSynchronize(st));
    return PG_OK;
}

pg_status pg3n_inbox_export(pg3n_level *s, pg3n_inbox which, unsigned char handle[PG_IPC_HANDLE_BYTES], double **local_ptr)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (which != PG3N_INBOX_MEAN && which != PG3N_INBOX_HALO) { set_err3n(s, "unknown inbox %d", (int)which); return PG_ERR_INVALID_ARG; }
    if ((which == PG3N_INBOX_MEAN && s->level == s->depth - 1) || (which == PG3N_INBOX_HALO && s->level == 0)) {
        set_err3n(s, "level %d of %d receives no such message", s->level, s->depth);
        return PG_ERR_STATE;
    }
    static_assert(sizeof(cudaIpcMemHandle_t) == PG_IPC_HANDLE_BYTES, "IPC handle size");
    DeviceGuard guard(s->device);
    if (!s->inbox[which]) {
        const long m = which == PG3N_INBOX_MEAN ? s->n / 2 : s->n / 2 + 2;
        PG3N_CUDA(s, cudaMalloc((void **)&s->inbox[which], (size_t)(m * m * m) * sizeof(double)));
    }
    if (handle) {
        cudaIpcMemHandle_t hnd;
        PG3N_CUDA(s, cudaIpcGetMemHandle(&hnd, s->inbox[which]));
        memcpy(handle, &hnd, sizeof hnd);
    }
    if (local_ptr) *local_ptr = s->inbox[which];
    return PG_OK;
}

static pg_status peer_replace(pg3n_level *s, pg3n_inbox which, double *ptr, bool ipc)
{
    if (s->peer[which] && s->peer_ipc[which]) PG3N_CUDA(s, cudaIpcCloseMemHandle(s->peer[which]));
    s->peer[which] = ptr;
    s->peer_ipc[which] = ipc;
    return PG_OK;
}

pg_status pg3n_peer_open(pg3n_level *s, pg3n_inbox which, const unsigned char handle[PG_IPC_HANDLE_BYTES])
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (!handle || (which != PG3N_INBOX_MEAN && which != PG3N_INBOX_HALO)) { set_err3n(s, "pg3n_peer_open: bad argument"); return PG_ERR_INVALID_ARG; }
    if ((which == PG3N_INBOX_MEAN && s->level == 0) || (which == PG3N_INBOX_HALO && s->level == s->depth - 1)) {
        set_err3n(s, "level %d of %d sends no such message", s->level, s->depth);
        return PG_ERR_STATE;
    }
    DeviceGuard guard(s->device);
    cudaIpcMemHandle_t hnd;
    memcpy(&hnd, handle, sizeof hnd);
    void *p = nullptr;
    PG3N_CUDA(s, cudaIpcOpenMemHandle(&p, hnd, cudaIpcMemLazyEnablePeerAccess));
    return peer_replace(s, which, (double *)p, true);
}

pg_status pg3n_peer_set(pg3n_level *s, pg3n_inbox which, double *neighbour_inbox)
{
    if (!s) return PG_ERR_INVALID_ARG;
    if (which != PG3N_INBOX_MEAN && which != PG3N_INBOX_HALO) { set_err3n(s, "unknown inbox %d", (int)which); return PG_ERR_INVALID_ARG; }
    if (neighbour_inbox && !dev_ptr_ok(s, neighbour_inbox, "neighbour_inbox")) return PG_ERR_INVALID_ARG;
    DeviceGuard guard(s->device);
    return peer_replace(s, which, neighbour_inbox, false);
}

pg_status pg3n_synchronize(pg3n_level *s)
{
    if (!s) return PG_ERR_INVALID_ARG;
    return pg3_synchronize(s->mesh);
}

pg_status pg3n_destroy(pg3n_level *s)
{
    if (!s) return PG_OK;
    DeviceGuard guard(s->device);
    cudaStreamSynchronize(s->mesh->inner->stream);
    nest_free(s);
    return PG_OK;
}

long pg3n_launch_count(const pg3n_level *s) { return s ? s->launches : 0; }

const char *pg3n_last_error(const pg3n_level *s) { return s ? s->err : g_create_error; }

}  // extern "C"

// =================================================================== the one call that never allocates
// pg_potential_direct_static (polargrav.h): direct summation for callers that cannot obtain device memory -- their
// program gave all of it to its own arena at start-up, runs inside a fixed memory budget, or only lends them pointers.
// The three grid tables the direct kernels read (r, dA, s2: the only global memory they touch besides Sigma and Phi,
// cudaMalloc'ed by create_impl on the ordinary path) sit here in a fixed array of the library image instead:
// 3 * PG_STATIC_MAX_N doubles = 48 KiB per GPU that loads the library, held until the process exits.
//
// The name below is only a stand-in on the host side: host code may not pass it to a kernel or a copy as if it were a
// device address.  static_tables_address() obtains the real address once per device, with that device current, and
// everything on the host goes through that pointer.
static __device__ __align__(256) double g_static_tables[3 * PG_STATIC_MAX_N];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
double *g_static_tables_on[kStaticMaxDevices] = {};   // device address of g_static_tables, by device ordinal

// One-time set-up per device.  `device` must be the current device (the caller holds a DeviceGuard).
pg_status static_tables_address(int device, double **out)
{
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_tables_on[device]) {
        int major = 0;
        PG_CUDA(nullptr, cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major != 10) {
            set_err(nullptr, "device %d is not sm_100; this library is built for sm_100a (B200) only and has no fallback", device);
            return PG_ERR_UNSUPPORTED;
        }
        double *p = nullptr;
        PG_CUDA(nullptr, cudaGetSymbolAddress((void **)&p, g_static_tables));
        if (!p) { set_err(nullptr, "cudaGetSymbolAddress returned a null address for the static tables"); return PG_ERR_CUDA; }
        g_static_tables_on[device] = p;
    }
    *out = g_static_tables_on[device];
    return PG_OK;
}

}  // namespace

extern "C" pg_status pg_potential_direct_static(const double *sigma, double *phi, int n_r, int n_phi, double r_in,
                                                double r_out, double eps, int device, void *cuda_stream)
{
    g_create_error[0] = 0;
    // host-side checks first: none of them needs a device
    if (!sigma || !phi) { set_err(nullptr, "pg_potential_direct_static: sigma or phi is NULL"); return PG_ERR_INVALID_ARG; }
    if (!(r_in > 0.0) || !(r_out > r_in) || !(eps > 0.0) || !std::isfinite(r_out) || !std::isfinite(eps)) {
        set_err(nullptr, "pg_potential_direct_static: need 0 < r_in < r_out and eps > 0");
        return PG_ERR_INVALID_ARG;
    }
    if (n_r > PG_STATIC_MAX_N || n_phi > PG_STATIC_MAX_N) {
        set_err(nullptr, "pg_potential_direct_static: grid %dx%d does not fit the fixed table array (at most %d cells per "
                         "axis); this call cannot allocate a larger one -- use pg_create + pg_potential_direct",
                n_r, n_phi, PG_STATIC_MAX_N);
        return PG_ERR_UNSUPPORTED;
    }
    if (!is_pow2(n_r) || !is_pow2(n_phi) || n_r < PG_MIN_N || n_phi < PG_MIN_N) {
        set_err(nullptr, "pg_potential_direct_static: unsupported grid %dx%d: n_r and n_phi must be powers of two in [%d, %d]",
                n_r, n_phi, PG_MIN_N, PG_STATIC_MAX_N);
        return PG_ERR_UNSUPPORTED;
    }
    const size_t fbytes = (size_t)n_r * n_phi * sizeof(double);
    if ((((uintptr_t)sigma | (uintptr_t)phi) & 15u) != 0) {
        set_err(nullptr, "pg_potential_direct_static: sigma and phi must be 16-byte aligned device pointers");
        return PG_ERR_INVALID_ARG;
    }
    if (ranges_overlap(sigma, fbytes, phi, fbytes)) {
        set_err(nullptr, "pg_potential_direct_static: phi overlaps sigma");
        return PG_ERR_INVALID_ARG;
    }
    int ndev = 0;
    PG_CUDA(nullptr, cudaGetDeviceCount(&ndev));
    if (device < 0) PG_CUDA(nullptr, cudaGetDevice(&device));
    if (device >= ndev || device >= kStaticMaxDevices) {
        set_err(nullptr, "pg_potential_direct_static: device %d out of range (%d devices)", device, ndev);
        return PG_ERR_INVALID_ARG;
    }
    DeviceGuard guard(device);          // current for the set-up, the copy and the launch; restored on return
    double *tables = nullptr;
    pg_status st = static_tables_address(device, &tables);
    if (st != PG_OK) return st;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    // the tables of create_impl (readings A1, A2), packed [r | dA | s2]; every entry the kernel reads is rewritten
    double host[3 * PG_STATIC_MAX_N];
    double *h_r = host, *h_dA = host + n_r, *h_s2 = host + 2 * n_r;
    {
        const long double du = logl((long double)r_out / (long double)r_in) / n_r;
        const long double dphi = 2.0L * kPiL / n_phi;
        for (int i = 0; i < n_r; ++i) {
            const long double ri = (long double)r_in * expl(((long double)i + 0.5L) * du);
            h_r[i] = (double)ri;
            h_dA[i] = (double)(ri * ri * sinhl(du) * dphi);
        }
        for (int j = 0; j < n_phi; ++j) {
            const long double sn = sinl(kPiL * j / n_phi);
            h_s2[j] = (double)(sn * sn);
        }
    }
    // pageable source: the runtime has taken its copy of `host` when this returns
    PG_CUDA(nullptr, cudaMemcpyAsync(tables, host, (size_t)(2 * n_r + n_phi) * sizeof(double), cudaMemcpyHostToDevice, stream));
    const double *d_r = tables, *d_dA = tables + n_r, *d_s2 = tables + 2 * n_r;

    // same shapes as launch_direct
    const double eps2 = eps * eps;
    const long fs = (long)n_r * n_phi;
    const dim3 grid(n_r, 1);
    if (n_phi >= 256) {
        const int R = n_phi >= 1024 ? 16 : 8;
        const size_t smem = ((size_t)n_phi + (size_t)(2 * n_phi / R) * (R + 2)) * sizeof(double);
        if (R == 16) {
            PG_CUDA(nullptr, cudaFuncSetAttribute(pgk::direct_tiled_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            pgk::direct_tiled_kernel<16><<<grid, n_phi / 16, smem, stream>>>(sigma, phi, d_r, d_dA, d_s2, n_r, n_phi, eps2, 0, fs, fs);
        } else {
            pgk::direct_tiled_kernel<8><<<grid, n_phi / 8, smem, stream>>>(sigma, phi, d_r, d_dA, d_s2, n_r, n_phi, eps2, 0, fs, fs);
        }
    } else {
        const size_t smem = 2 * (size_t)n_phi * sizeof(double);
        pgk::direct_kernel<1><<<grid, n_phi, smem, stream>>>(sigma, phi, d_r, d_dA, d_s2, n_r, n_phi, eps2, 0, fs, fs);
    }
    PG_CUDA(nullptr, cudaGetLastError());
    return PG_OK;
}
