// api.cu -- the C ABI of include/vjp_b200.h: argument validation, workspace accounting and
// dispatch.  No arithmetic of the method lives here.
#include <cstdint>
#include <cstring>

#include "internal.h"

using namespace vjp;

namespace {

bool op_ok(const vjp_op_t *op) {
    return op && op->code >= VJP_OP_ADD && op->code <= VJP_OP_MATMUL3 &&
           (op->dtype == VJP_F32 || op->dtype == VJP_F64);
}
// every data pointer must be 16-byte aligned (128-bit accesses); NULL passes (checked separately)
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
template <class... P>
bool all_aligned(P... p) { return (aligned16(p) && ...); }
size_t dtype_bytes(int dtype) { return dtype == VJP_F64 ? 8 : 4; }

bool scan_supported(const vjp_op_t *op) {
    switch (op->code) {
    case VJP_OP_ADD:
    case VJP_OP_MUL: return true;
    case VJP_OP_MIN:
    case VJP_OP_MAX:
    case VJP_OP_LINREC:
    case VJP_OP_MATMUL2:
    case VJP_OP_MATMUL3:
    case VJP_OP_MATMUL5: return op->dtype == VJP_F32;
    default: return false;
    }
}
// Which reduce-by-index route an operator takes: 0 none, 1 '+', 2 min/max, 3 '*', 4 general.
int rbi_route(const vjp_op_t *op) {
    const bool f32 = op->dtype == VJP_F32;
    switch (op->code) {
    case VJP_OP_ADD: return op->force_general ? (f32 ? 4 : 0) : 1;
    case VJP_OP_MIN:
    case VJP_OP_MAX: return f32 ? (op->force_general ? 4 : 2) : 0;
    case VJP_OP_MUL: return f32 ? (op->force_general ? 4 : 3) : 0;
    case VJP_OP_SATADD: return f32 ? 4 : 0;
    default: return 0;  // LINREC / MATMUL are not commutative
    }
}
const int64_t RBI_MAX_N = 0xfffffffell;  // packed 32-bit positions

cudaStream_t as_stream(void *s) { return static_cast<cudaStream_t>(s); }

}  // namespace

// ------------------------------------------------------------------ instrumentation ------
namespace vjp {
namespace {
const char *const KERNEL_NAMES[K_COUNT] = {
    "scan_lookback_kernel<MODE_SCAN>", "scan_lookback_kernel<MODE_TILEAGG>",
    "tile_exscan_kernel", "scan_vjp_reverse_kernel",
    "rbi_fill_kernel", "rbi_forward_kernel", "rbi_vjp_add_kernel",
    "rbi_minmax_lifted_kernel", "rbi_minmax_finish_kernel", "rbi_cached_small_kernel", "rbi_cached_big_kernel",
    "rbi_cached_fold_kernel", "rbi_mul_finish_kernel", "rbi_mul_sweep_kernel",
    "sort_hist_kernel", "u32_exclusive_scan_kernel", "sort_scatter_kernel", "seg_forward_kernel",
    "seg_reverse_vjp_kernel", "sort_export_kernel",
    "reduce_partial_kernel", "reduce_finish_kernel", "reduce_sweep_kernel", "reduce_pack_kernel",
    "sop_forward_kernel", "sop_finish_kernel", "sop_inv_sweep_kernel", "rows_to_cols / cols_to_rows",
    "ms_forward_kernel", "ms_seg_agg / ms_carry_kernel", "ms_backward_kernel", "ms_hist_kernel", "shift_words_kernel", "tile_agg_tma_kernel"};
constexpr int PROF_MAX = 8192;
struct ProfRec { int kid; cudaEvent_t a, b; };
long long g_launches[K_COUNT];
bool g_prof_on = false;
ProfRec g_rec[PROF_MAX];
int g_nrec = 0, g_nalloc = 0;
}  // namespace

void prof_begin(int kid, cudaStream_t s) {
    __atomic_add_fetch(&g_launches[kid], 1, __ATOMIC_RELAXED);
    if (!g_prof_on || g_nrec >= PROF_MAX) return;
    if (g_nrec >= g_nalloc) {
        if (cudaEventCreate(&g_rec[g_nalloc].a) != cudaSuccess) return;
        if (cudaEventCreate(&g_rec[g_nalloc].b) != cudaSuccess) return;
        g_nalloc++;
    }
    g_rec[g_nrec].kid = kid;
    cudaEventRecord(g_rec[g_nrec].a, s);
}
void prof_end(int kid, cudaStream_t s) {
    if (!g_prof_on || g_nrec >= g_nalloc || g_nrec >= PROF_MAX || g_rec[g_nrec].kid != kid) return;
    cudaEventRecord(g_rec[g_nrec].b, s);
    g_nrec++;
}
}  // namespace vjp

extern "C" {

int vjp_kernel_count(void) { return K_COUNT; }
const char *vjp_kernel_name(int kid) { return (kid >= 0 && kid < K_COUNT) ? KERNEL_NAMES[kid] : nullptr; }
int64_t vjp_launch_count(int kid) {
    if (kid >= 0 && kid < K_COUNT) return g_launches[kid];
    long long t = 0;
    for (int i = 0; i < K_COUNT; i++) t += g_launches[i];
    return t;
}
void vjp_profile_enable(int on) {
    g_prof_on = on != 0;
    g_nrec = 0;
}
int vjp_profile_read(int kid, double *total_ms, int64_t *launches) {
    if (kid < 0 || kid >= K_COUNT || !total_ms || !launches) return VJP_ERR_INVALID_ARG;
    double t = 0.0;
    int64_t c = 0;
    for (int i = 0; i < g_nrec; i++) {
        if (g_rec[i].kid != kid) continue;
        if (cudaEventSynchronize(g_rec[i].b) != cudaSuccess) return VJP_ERR_CUDA;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, g_rec[i].a, g_rec[i].b) != cudaSuccess) return VJP_ERR_CUDA;
        t += ms;
        c++;
    }
    *total_ms = t;
    *launches = c;
    return VJP_OK;
}

int vjp_scan_arity(const vjp_op_t *op) {
    if (!op) return -1;
    switch (op->code) {
    case VJP_OP_ADD:
    case VJP_OP_MIN:
    case VJP_OP_MAX:
    case VJP_OP_MUL: return 1;
    case VJP_OP_LINREC: return 2;
    case VJP_OP_MATMUL2: return 4;
    case VJP_OP_MATMUL3: return 9;
    case VJP_OP_MATMUL5: return 25;
    default: return -1;
    }
}

const char *vjp_version(void) { return "vjp_b200 0.1 (sm_100a, CUDA " VJP_STR(CUDART_VERSION) ")"; }

// ------------------------------------------------------------------------------ scan -----

size_t vjp_scan_workspace_bytes(const vjp_op_t *op, int64_t n) {
    if (!op_ok(op) || !scan_supported(op) || n < 0) return 0;
    return scan_workspace_bytes(op->code, op->dtype, n);
}

int scan_forward(const vjp_op_t *op, int64_t n, const void *xs, void *ys, void *ws,
                 size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (!scan_supported(op)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!xs || !ys || !ws || !all_aligned(xs, ys, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < scan_workspace_bytes(op->code, op->dtype, n)) return VJP_ERR_WORKSPACE;
    return launch_scan_forward(op->code, op->dtype, n, xs, ys, ws, as_stream(stream));
}

int vjp_scan(const vjp_op_t *op, int64_t n, const void *xs, const void *ys_bar, void *xs_bar,
             void *ws, size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (!scan_supported(op)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!ys_bar || !xs_bar || !ws || (!xs && op->code != VJP_OP_ADD)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(xs, ys_bar, xs_bar, ws)) return VJP_ERR_INVALID_ARG;
    if (xs_bar == ys_bar && (op->code != VJP_OP_ADD || op->accumulate)) return VJP_ERR_INVALID_ARG;  // in place: '+' only
    if (ws_bytes < scan_workspace_bytes(op->code, op->dtype, n)) return VJP_ERR_WORKSPACE;
    return launch_scan_vjp(op->code, op->dtype, n, xs, ys_bar, xs_bar, ws, op->accumulate, as_stream(stream));
}

// ------------------------------------------------------------------ exclusive scan -------
// Words of the neutral element of a scan operator (EW = arity * dtype words); returns EW.
static int neutral_words(const vjp_op_t *op, ShiftFill &f) {
    const int arity = vjp_scan_arity(op);
    const bool f64 = op->dtype == VJP_F64;
    for (int i = 0; i < 32; i++) f.w[i] = 0u;
    switch (op->code) {
    case VJP_OP_ADD: break;
    case VJP_OP_MUL: if (f64) f.w[1] = 0x3ff00000u; else f.w[0] = 0x3f800000u; break;
    case VJP_OP_MIN: f.w[0] = 0x7f800000u; break;   // +inf
    case VJP_OP_MAX: f.w[0] = 0xff800000u; break;   // -inf
    case VJP_OP_LINREC: f.w[0] = 0x3f800000u; break;  // (a, b) = (1, 0)
    default: {
        const int q = arity == 4 ? 2 : arity == 9 ? 3 : 5;
        for (int i = 0; i < q; i++) f.w[i * q + i] = 0x3f800000u;
    }
    }
    return arity * (f64 ? 2 : 1);
}
static size_t exc_tmp_bytes(const vjp_op_t *op, int64_t n) {
    return align_up((size_t)n * vjp_scan_arity(op) * dtype_bytes(op->dtype), 256);
}

size_t vjp_scan_exclusive_workspace_bytes(const vjp_op_t *op, int64_t n) {
    if (!op_ok(op) || !scan_supported(op) || n < 0) return 0;
    return exc_tmp_bytes(op, n) + scan_workspace_bytes(op->code, op->dtype, n);
}

int scan_exclusive_forward(const vjp_op_t *op, int64_t n, const void *xs, void *ys, void *ws, size_t ws_bytes,
                           void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (!scan_supported(op)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!xs || !ys || !ws || !all_aligned(xs, ys, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < vjp_scan_exclusive_workspace_bytes(op, n)) return VJP_ERR_WORKSPACE;
    ShiftFill fill;
    const int ew = neutral_words(op, fill);
    char *tmp = static_cast<char *>(ws), *inner = tmp + exc_tmp_bytes(op, n);
    const int rc = launch_scan_forward(op->code, op->dtype, n, xs, tmp, inner, as_stream(stream));
    if (rc != VJP_OK) return rc;
    return launch_shift_words(n * ew, ew, tmp, ys, fill, as_stream(stream));   // ys_0 = e, ys_i = inclusive_{i-1}
}

int vjp_scan_exclusive(const vjp_op_t *op, int64_t n, const void *xs, const void *ys_bar, void *xs_bar, void *ws,
                       size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (!scan_supported(op)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!ys_bar || !xs_bar || !ws || (!xs && op->code != VJP_OP_ADD)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(xs, ys_bar, xs_bar, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < vjp_scan_exclusive_workspace_bytes(op, n)) return VJP_ERR_WORKSPACE;
    ShiftFill fill;
    const int ew = neutral_words(op, fill);
    char *tmp = static_cast<char *>(ws), *inner = tmp + exc_tmp_bytes(op, n);
    // S^T ys_bar: the adjoint of output i + 1 belongs to inclusive output i; nothing flows into the last one
    const int rc = launch_shift_words(n * ew, -ew, ys_bar, tmp, fill, as_stream(stream));
    if (rc != VJP_OK) return rc;
    return launch_scan_vjp(op->code, op->dtype, n, xs, tmp, xs_bar, inner, op->accumulate, as_stream(stream));
}

int64_t vjp_scan_add_f32_noalloc_max_n(void) { return scan_noalloc_max_n(); }

int vjp_scan_add_f32_noalloc(int64_t n, const float *ys_bar, float *xs_bar, int accumulate, void *stream) {
    if (n < 0) return VJP_ERR_INVALID_ARG;
    if (n > scan_noalloc_max_n()) return VJP_ERR_UNSUPPORTED;  // beyond the static scratch: use vjp_scan
    if (n == 0) return VJP_OK;
    if (!ys_bar || !xs_bar || !all_aligned(ys_bar, xs_bar)) return VJP_ERR_INVALID_ARG;
    if (xs_bar == ys_bar && accumulate) return VJP_ERR_INVALID_ARG;
    return launch_scan_add_f32_noalloc(n, ys_bar, xs_bar, accumulate != 0, as_stream(stream));
}

size_t vjp_scan_host_scratch_bytes(const vjp_op_t *op, int64_t n) {
    if (!op_ok(op) || !scan_supported(op) || n < 0) return 0;
    const size_t arr = align_up((size_t)n * vjp_scan_arity(op) * dtype_bytes(op->dtype), 256);
    return 3 * arr + scan_workspace_bytes(op->code, op->dtype, n);
}

int vjp_scan_host(const vjp_op_t *op, int64_t n, const void *xs_host, const void *ys_bar_host,
                  void *xs_bar_host, void *dev_scratch, size_t dev_scratch_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (!scan_supported(op)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!ys_bar_host || !xs_bar_host || !dev_scratch || (!xs_host && op->code != VJP_OP_ADD))
        return VJP_ERR_INVALID_ARG;
    if (!aligned16(dev_scratch)) return VJP_ERR_INVALID_ARG;
    if (dev_scratch_bytes < vjp_scan_host_scratch_bytes(op, n)) return VJP_ERR_WORKSPACE;
    cudaStream_t s = as_stream(stream);
    const size_t bytes = (size_t)n * vjp_scan_arity(op) * dtype_bytes(op->dtype);
    const size_t arr = align_up(bytes, 256);
    char *d = static_cast<char *>(dev_scratch);
    char *dx = d, *dy = d + arr, *dout = d + 2 * arr, *ws = d + 3 * arr;
    if (xs_host && op->code != VJP_OP_ADD &&
        cudaMemcpyAsync(dx, xs_host, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    if (cudaMemcpyAsync(dy, ys_bar_host, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    if (op->accumulate &&
        cudaMemcpyAsync(dout, xs_bar_host, bytes, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    int rc = launch_scan_vjp(op->code, op->dtype, n, dx, dy, dout, ws, op->accumulate, s);
    if (rc != VJP_OK) return rc;
    if (cudaMemcpyAsync(xs_bar_host, dout, bytes, cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    return cuda_status(cudaStreamSynchronize(s));
}

// ------------------------------------------------------------------- reduce-by-index -----

size_t vjp_reduce_by_index_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t num_bins) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return 0;
    size_t need;
    switch (rbi_route(op)) {
    case 1:
    case 2:
    case 3: need = rbi_special_workspace_bytes(op->code, op->dtype, n, num_bins); break;
    case 4: need = rbi_general_workspace_bytes(n, num_bins); break;
    default: return 0;
    }
    const size_t fwd = rbi_forward_workspace_bytes(op->code, n, num_bins);  // one query serves both calls
    return need > fwd ? need : fwd;
}

int reduce_by_index_forward(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                            const void *vs, void *hist, void *ws, size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (rbi_route(op) == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if ((num_bins > 0 && !hist) || (n > 0 && (!is || !vs))) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(is, vs, hist, ws)) return VJP_ERR_INVALID_ARG;
    if (num_bins > 0 && op->code != VJP_OP_ADD &&
        (!ws || ws_bytes < rbi_forward_workspace_bytes(op->code, n, num_bins)))
        return VJP_ERR_WORKSPACE;
    return launch_rbi_forward(op->code, op->dtype, op->param, n, num_bins, is, vs, hist, ws,
                              as_stream(stream));
}

int vjp_reduce_by_index(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                        const void *vs, const void *hist_bar, void *vs_bar, void *ws,
                        size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    const int route = rbi_route(op);
    if (route == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!is || !vs_bar || (num_bins > 0 && !hist_bar) || (!vs && route != 1)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(is, vs, hist_bar, vs_bar, ws)) return VJP_ERR_INVALID_ARG;
    if (!ws || ws_bytes < vjp_reduce_by_index_workspace_bytes(op, n, num_bins)) return VJP_ERR_WORKSPACE;
    cudaStream_t s = as_stream(stream);
    const int acc = op->accumulate != 0;
    switch (route) {
    case 1: return launch_rbi_vjp_add(op->dtype, n, num_bins, is, hist_bar, vs_bar, acc, s);
    case 2:
        return launch_rbi_minmax(op->code, n, num_bins, is, static_cast<const float *>(vs),
                                 static_cast<const float *>(hist_bar), static_cast<float *>(vs_bar),
                                 nullptr, nullptr, ws, acc, s);
    case 3:
        return launch_rbi_mul(n, num_bins, is, static_cast<const float *>(vs),
                              static_cast<const float *>(hist_bar), static_cast<float *>(vs_bar),
                              nullptr, nullptr, ws, acc, s);
    default:
        return launch_rbi_general_vjp(op->code, op->param, n, num_bins, is,
                                      static_cast<const float *>(vs),
                                      static_cast<const float *>(hist_bar),
                                      static_cast<float *>(vs_bar), ws, acc, op->force_general == 2, s);
    }
}

size_t vjp_reduce_by_index_host_scratch_bytes(const vjp_op_t *op, int64_t n, int64_t num_bins) {
    if (!op_ok(op) || n < 0 || num_bins < 0 || rbi_route(op) == 0) return 0;
    const size_t e = dtype_bytes(op->dtype);
    return align_up((size_t)n * 8, 256) + 2 * align_up((size_t)n * e, 256) +
           align_up((size_t)num_bins * e, 256) + vjp_reduce_by_index_workspace_bytes(op, n, num_bins);
}

int vjp_reduce_by_index_host_async(const vjp_op_t *op, int64_t n, int64_t num_bins,
                                   const int64_t *is_host, const void *vs_host,
                                   const void *hist_bar_host, void *vs_bar_host, void *dev_scratch,
                                   size_t dev_scratch_bytes, void *stream) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    const int route = rbi_route(op);
    if (route == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;  // before anything is enqueued
    if (route == 3 && !rbi_cached_supported(num_bins)) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!aligned16(dev_scratch)) return VJP_ERR_INVALID_ARG;
    if (!is_host || !vs_bar_host || !dev_scratch || (num_bins > 0 && !hist_bar_host) ||
        (!vs_host && route != 1))
        return VJP_ERR_INVALID_ARG;
    if (dev_scratch_bytes < vjp_reduce_by_index_host_scratch_bytes(op, n, num_bins))
        return VJP_ERR_WORKSPACE;
    cudaStream_t s = as_stream(stream);
    const size_t e = dtype_bytes(op->dtype);
    char *d = static_cast<char *>(dev_scratch);
    char *dis = d;
    char *dvs = dis + align_up((size_t)n * 8, 256);
    char *dout = dvs + align_up((size_t)n * e, 256);
    char *dhb = dout + align_up((size_t)n * e, 256);
    char *ws = dhb + align_up((size_t)num_bins * e, 256);
    const size_t ws_bytes = vjp_reduce_by_index_workspace_bytes(op, n, num_bins);
    if (cudaMemcpyAsync(dis, is_host, (size_t)n * 8, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    if (route != 1 &&
        cudaMemcpyAsync(dvs, vs_host, (size_t)n * e, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    if (num_bins > 0 &&
        cudaMemcpyAsync(dhb, hist_bar_host, (size_t)num_bins * e, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    if (op->accumulate &&
        cudaMemcpyAsync(dout, vs_bar_host, (size_t)n * e, cudaMemcpyHostToDevice, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    int rc = vjp_reduce_by_index(op, n, num_bins, reinterpret_cast<const int64_t *>(dis), dvs, dhb,
                                 dout, ws, ws_bytes, stream);
    if (rc != VJP_OK) return rc;
    if (cudaMemcpyAsync(vs_bar_host, dout, (size_t)n * e, cudaMemcpyDeviceToHost, s) != cudaSuccess)
        return VJP_ERR_CUDA;
    return VJP_OK;
}

int vjp_reduce_by_index_host(const vjp_op_t *op, int64_t n, int64_t num_bins,
                             const int64_t *is_host, const void *vs_host,
                             const void *hist_bar_host, void *vs_bar_host, void *dev_scratch,
                             size_t dev_scratch_bytes, void *stream) {
    const int rc = vjp_reduce_by_index_host_async(op, n, num_bins, is_host, vs_host, hist_bar_host,
                                                  vs_bar_host, dev_scratch, dev_scratch_bytes, stream);
    if (rc != VJP_OK || n == 0) return rc;
    return cuda_status(cudaStreamSynchronize(as_stream(stream)));
}

int rbi_argext(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is, const void *vs,
               int64_t *arg, void *ext, void *ws, size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if ((op->code != VJP_OP_MIN && op->code != VJP_OP_MAX) || op->dtype != VJP_F32)
        return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (num_bins == 0) return VJP_OK;
    if (!arg || !ext || (n > 0 && (!is || !vs))) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(is, vs, arg, ext, ws)) return VJP_ERR_INVALID_ARG;
    if (!ws || ws_bytes < rbi_special_workspace_bytes(op->code, op->dtype, n, num_bins))
        return VJP_ERR_WORKSPACE;
    return launch_rbi_minmax(op->code, n, num_bins, is, static_cast<const float *>(vs), nullptr,
                             nullptr, arg, static_cast<float *>(ext), ws, 0, as_stream(stream));
}

int rbi_zero_prod(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                  const void *vs, int64_t *zeros, void *prod_nz, void *ws, size_t ws_bytes,
                  void *stream) {
    if (!op_ok(op) || n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (op->code != VJP_OP_MUL || op->dtype != VJP_F32) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (num_bins == 0) return VJP_OK;
    if (!zeros || !prod_nz || (n > 0 && (!is || !vs))) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(is, vs, zeros, prod_nz, ws)) return VJP_ERR_INVALID_ARG;
    if (!ws || ws_bytes < rbi_special_workspace_bytes(op->code, op->dtype, n, num_bins))
        return VJP_ERR_WORKSPACE;
    return launch_rbi_mul(n, num_bins, is, static_cast<const float *>(vs), nullptr, nullptr, zeros,
                          static_cast<float *>(prod_nz), ws, 0, as_stream(stream));
}

// ----------------------------------------------------------------- vectorised operators ----

namespace {
struct VecWs {
    float *cols, *outs, *hbs;
    char *inner;
    int64_t ncol, wcol;
    size_t total;
};
// columns are padded to a multiple of 4 floats so that every column start is 16-byte aligned
VecWs vec_carve(void *ws, int64_t n, int64_t d, int64_t w, size_t inner_bytes, int64_t a = 1) {
    VecWs v;
    v.ncol = (n + 3) / 4 * 4;
    v.wcol = (w + 3) / 4 * 4;
    char *p = static_cast<char *>(ws);
    auto take = [&](size_t bytes) { char *r = p; p += align_up(bytes < 16 ? 16 : bytes, 256); return r; };
    v.cols = reinterpret_cast<float *>(take((size_t)v.ncol * d * a * 4));
    v.outs = reinterpret_cast<float *>(take((size_t)v.ncol * d * a * 4));
    v.hbs = reinterpret_cast<float *>(take((size_t)v.wcol * d * a * 4));
    v.inner = take(inner_bytes);
    v.total = (size_t)(p - static_cast<char *>(ws));
    return v;
}
bool vec_op_ok(const vjp_op_t *op) { return op_ok(op) && op->dtype == VJP_F32; }
// `map2 (*)` on rows of d = 2^ld scalars: d histograms = ONE histogram over (bin, column) pairs, run as
// a scalar '*' problem on the flat arrays with virtual keys -- no transposes, keys read once per row.  Returns ld, or
// 0 if this form does not apply (then: transpose + the scalar rule per column).
int vec_mul_fused_ld(const vjp_op_t *op, int64_t n, int64_t d, int64_t num_bins) {
    if (op->code != VJP_OP_MUL || op->force_general || d < 2 || (d & (d - 1)) != 0) return 0;
    int ld = 0;
    while (((int64_t)1 << ld) < d) ld++;
    return rbi_mul_vec_fused(n, num_bins, ld) ? ld : 0;
}
}  // namespace

size_t vjp_reduce_by_index_vec_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t d, int64_t num_bins) {
    if (!vec_op_ok(op) || n < 0 || d < 1 || num_bins < 0) return 0;
    const size_t inner = vjp_reduce_by_index_workspace_bytes(op, n, num_bins);
    if (!inner) return 0;
    size_t need = vec_carve(nullptr, n, d, num_bins, inner).total;
    if (const int ld = vec_mul_fused_ld(op, n, d, num_bins)) {
        const size_t fused = rbi_special_workspace_bytes(VJP_OP_MUL, VJP_F32, n << ld, num_bins << ld);
        if (fused > need) need = fused;
    }
    return need;
}

int vjp_reduce_by_index_vec(const vjp_op_t *op, int64_t n, int64_t d, int64_t num_bins, const int64_t *is,
                            const void *vss, const void *hist_bar, void *vss_bar, void *ws, size_t ws_bytes,
                            void *stream) {
    if (!op_ok(op) || n < 0 || d < 1 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (!vec_op_ok(op) || rbi_route(op) == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N || d > 4096) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    const bool needs_vs = rbi_route(op) != 1;
    if (!is || !vss_bar || !ws || (num_bins > 0 && !hist_bar) || (needs_vs && !vss)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(is, vss, hist_bar, vss_bar, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < vjp_reduce_by_index_vec_workspace_bytes(op, n, d, num_bins)) return VJP_ERR_WORKSPACE;
    if (const int ld = vec_mul_fused_ld(op, n, d, num_bins))
        return launch_rbi_mul(n << ld, num_bins << ld, is, static_cast<const float *>(vss), static_cast<const float *>(hist_bar),
                              static_cast<float *>(vss_bar), nullptr, nullptr, ws, op->accumulate != 0, as_stream(stream), ld);
    const size_t inner = vjp_reduce_by_index_workspace_bytes(op, n, num_bins);
    const VecWs v = vec_carve(ws, n, d, num_bins, inner);
    cudaStream_t s = as_stream(stream);
    int rc;
    if (needs_vs && (rc = launch_rows_to_cols(n, d, v.ncol, static_cast<const float *>(vss), v.cols, s)) != VJP_OK) return rc;
    if ((rc = launch_rows_to_cols(num_bins, d, v.wcol, static_cast<const float *>(hist_bar), v.hbs, s)) != VJP_OK) return rc;
    vjp_op_t col = *op;
    col.accumulate = 0;  // the "+=" is fused into the transpose back
    for (int64_t c = 0; c < d; c++) {  // the scalar rule on every column (eq. 3: map (reduce ...) (transpose ...))
        rc = vjp_reduce_by_index(&col, n, num_bins, is, needs_vs ? v.cols + c * v.ncol : nullptr, v.hbs + c * v.wcol,
                                 v.outs + c * v.ncol, v.inner, inner, stream);
        if (rc != VJP_OK) return rc;
    }
    return launch_cols_to_rows(n, d, v.ncol, v.outs, static_cast<float *>(vss_bar), op->accumulate != 0, s);
}

size_t vjp_scan_vec_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t d) {
    if (!vec_op_ok(op) || n < 0 || d < 1 || vjp_scan_arity(op) < 1) return 0;
    const size_t inner = vjp_scan_workspace_bytes(op, n);
    return inner ? vec_carve(nullptr, n, d, n, inner, vjp_scan_arity(op)).total : 0;  // hbs holds the transposed output adjoints
}

// Rows of d entries of a = arity(op) floats.  a = 1: scan with map2 (.) (ISWIM).  a > 1 (LINREC, MATMUL*):
// the operator applies (.) to each of the d blocks of a row, its Jacobian is block-diagonal with d DIFFERENT blocks
// (non-redundant BDS), and "the computation of rs_bar is performed with k different scans, each of them
// using a scaled-down operator": the block columns are gathered, the small operator's rule runs on each, and the
// result is put back.
int vjp_scan_vec(const vjp_op_t *op, int64_t n, int64_t d, const void *xss, const void *yss_bar, void *xss_bar,
                 void *ws, size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0 || d < 1) return VJP_ERR_INVALID_ARG;
    if (!vec_op_ok(op) || !scan_supported(op) || vjp_scan_arity(op) < 1 || d > 4096) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    const int a = vjp_scan_arity(op);
    const bool needs_xs = op->code != VJP_OP_ADD;
    if (!yss_bar || !xss_bar || !ws || (needs_xs && !xss)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(xss, yss_bar, xss_bar, ws)) return VJP_ERR_INVALID_ARG;
    const size_t inner = vjp_scan_workspace_bytes(op, n);
    const VecWs v = vec_carve(ws, n, d, n, inner, a);  // hbs holds the transposed output adjoints
    if (ws_bytes < v.total) return VJP_ERR_WORKSPACE;
    cudaStream_t s = as_stream(stream);
    int rc;
    if (needs_xs && (rc = launch_rows_to_cols(n, d, v.ncol, static_cast<const float *>(xss), v.cols, s, a)) != VJP_OK) return rc;
    if ((rc = launch_rows_to_cols(n, d, v.wcol, static_cast<const float *>(yss_bar), v.hbs, s, a)) != VJP_OK) return rc;
    vjp_op_t col = *op;
    col.accumulate = 0;
    for (int64_t c = 0; c < d; c++) {  // ISWIM: scan (map2 (.)) = map (scan (.)) on the transpose
        rc = vjp_scan(&col, n, needs_xs ? v.cols + c * v.ncol * a : nullptr, v.hbs + c * v.wcol * a, v.outs + c * v.ncol * a,
                      v.inner, inner, stream);
        if (rc != VJP_OK) return rc;
    }
    return launch_cols_to_rows(n, d, v.ncol, v.outs, static_cast<float *>(xss_bar), op->accumulate != 0, s, a);
}

// --------------------------------------------------------------------------- sumOfProd ----

size_t rbi_sumofprod_workspace_bytes(int64_t n, int64_t num_bins, int use_general) {
    if (n < 0 || num_bins < 0) return 0;
    return use_general ? rbi_general_workspace_bytes(n, num_bins) : rbi_sop_workspace_bytes(num_bins);
}

int rbi_sumofprod_forward(int64_t n, int64_t num_bins, const int64_t *is, const float *vs, float *hist,
                          void *ws, size_t ws_bytes, void *stream) {
    if (n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if ((num_bins > 0 && (!hist || !ws)) || (n > 0 && (!is || !vs)) || !all_aligned(is, vs, hist, ws))
        return VJP_ERR_INVALID_ARG;
    if (ws_bytes < rbi_sop_workspace_bytes(num_bins)) return VJP_ERR_WORKSPACE;
    return launch_rbi_sop_forward(n, num_bins, is, vs, hist, ws, as_stream(stream));
}

int vjp_rbi_sumofprod(int64_t n, int64_t num_bins, const int64_t *is, const float *vs, const float *hist_bar,
                      float *vs_bar, int use_general, int accumulate, void *ws, size_t ws_bytes, void *stream) {
    if (n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!is || !vs || !vs_bar || !ws || (num_bins > 0 && !hist_bar) || !all_aligned(is, vs, hist_bar, vs_bar, ws))
        return VJP_ERR_INVALID_ARG;
    if (ws_bytes < rbi_sumofprod_workspace_bytes(n, num_bins, use_general)) return VJP_ERR_WORKSPACE;
    if (use_general)
        return launch_rbi_sop_general_vjp(n, num_bins, is, vs, hist_bar, vs_bar, ws, accumulate != 0, use_general == 2, as_stream(stream));
    return launch_rbi_sop_vjp_inv(n, num_bins, is, vs, hist_bar, vs_bar, ws, accumulate != 0, as_stream(stream));
}

// ------------------------------------------------------------------------------ reduce ----

namespace {
// Which route a reduce operator takes: 0 none, 1 specialised, 2 general (two exclusive scans).
int reduce_route(const vjp_op_t *op) {
    const bool f32 = op->dtype == VJP_F32;
    switch (op->code) {
    case VJP_OP_ADD: return op->force_general ? (f32 ? 2 : 0) : 1;
    case VJP_OP_MIN:
    case VJP_OP_MAX:
    case VJP_OP_MUL: return f32 ? (op->force_general ? 2 : 1) : 0;
    case VJP_OP_SATADD: return f32 ? 2 : 0;
    default: return 0;
    }
}
}  // namespace

size_t vjp_reduce_workspace_bytes(const vjp_op_t *op, int64_t n) {
    if (!op_ok(op) || n < 0) return 0;
    switch (reduce_route(op)) {
    case 1: return reduce_special_workspace_bytes();
    case 2: {
        const size_t a = rbi_general_workspace_bytes(n, 1), b = reduce_special_workspace_bytes();
        return a > b ? a : b;
    }
    default: return 0;
    }
}

int reduce_forward(const vjp_op_t *op, int64_t n, const void *xs, void *y, void *ws, size_t ws_bytes,
                   void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if (reduce_route(op) == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (!y || !ws || (n > 0 && !xs) || !all_aligned(xs, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < reduce_special_workspace_bytes()) return VJP_ERR_WORKSPACE;
    // n == 0 runs too (an empty grid-stride loop): y = the neutral element
    return launch_reduce_forward(op->code, op->dtype, op->param, n, xs, y, nullptr, nullptr, 0, ws, as_stream(stream));
}

int reduce_lifted(const vjp_op_t *op, int64_t n, const void *xs, int64_t *aux_i, void *aux_v, void *ws,
                  size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    if ((op->code != VJP_OP_MIN && op->code != VJP_OP_MAX && op->code != VJP_OP_MUL) || op->dtype != VJP_F32)
        return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (!aux_i || !aux_v || !ws || (n > 0 && !xs) || !all_aligned(xs, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < reduce_special_workspace_bytes()) return VJP_ERR_WORKSPACE;
    return launch_reduce_forward(op->code, op->dtype, op->param, n, xs, nullptr, aux_i, aux_v, 1, ws, as_stream(stream));
}

int vjp_reduce(const vjp_op_t *op, int64_t n, const void *xs, const void *y_bar, void *xs_bar, void *ws,
               size_t ws_bytes, void *stream) {
    if (!op_ok(op) || n < 0) return VJP_ERR_INVALID_ARG;
    const int route = reduce_route(op);
    if (route == 0) return VJP_ERR_UNSUPPORTED;
    if (n >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    const bool needs_xs = route == 2 || op->code != VJP_OP_ADD;
    if (!y_bar || !xs_bar || !ws || (needs_xs && !xs)) return VJP_ERR_INVALID_ARG;
    if (!all_aligned(xs, xs_bar, ws)) return VJP_ERR_INVALID_ARG;
    if (ws_bytes < vjp_reduce_workspace_bytes(op, n)) return VJP_ERR_WORKSPACE;
    if (route == 1)
        return launch_reduce_vjp(op->code, op->dtype, n, xs, y_bar, xs_bar, ws, op->accumulate != 0, as_stream(stream));
    return launch_reduce_general_vjp(op->code, op->param, n, static_cast<const float *>(xs),
                                     static_cast<const float *>(y_bar), static_cast<float *>(xs_bar), ws,
                                     op->accumulate != 0, as_stream(stream));
}

int rbi_sort_perm(int64_t n, int64_t num_bins, const int64_t *is, int64_t *sorted_keys,
                  int64_t *perm, void *ws, size_t ws_bytes, void *stream) {
    if (n < 0 || num_bins < 0) return VJP_ERR_INVALID_ARG;
    if (n >= RBI_MAX_N || num_bins >= RBI_MAX_N) return VJP_ERR_UNSUPPORTED;
    if (n == 0) return VJP_OK;
    if (!is || !sorted_keys || !perm || !all_aligned(is, sorted_keys, perm, ws)) return VJP_ERR_INVALID_ARG;
    if (!ws || ws_bytes < rbi_general_workspace_bytes(n, num_bins)) return VJP_ERR_WORKSPACE;
    return launch_rbi_sort_perm(n, num_bins, is, sorted_keys, perm, ws, as_stream(stream));
}

}  // extern "C"
