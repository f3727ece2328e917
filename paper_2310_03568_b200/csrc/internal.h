// internal.h -- host-side declarations shared by the translation units of libvjp_b200.so.
// Each launch_* function validates nothing: api.cu has already checked the arguments and the
// workspace size.  All pointers are device pointers; every function only enqueues on `stream`
// and returns a vjp_status_t.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/vjp_b200.h"

#define VJP_STR2(x) #x
#define VJP_STR(x) VJP_STR2(x)

namespace vjp {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? VJP_OK : VJP_ERR_CUDA; }
inline int last_launch_status() { return cuda_status(cudaGetLastError()); }

// ------------------------------------------------------------------ instrumentation ------
// Every kernel launch of the library goes through a LaunchScope: it counts the launch and, while
// profiling is enabled (vjp_profile_enable), brackets it with CUDA events on the launching stream.
enum KernelId : int {
    K_SCAN_LOOKBACK = 0, K_SCAN_TILEAGG, K_SCAN_TILEPRE /* tile_exscan_kernel */, K_SCAN_VJP_REVERSE,
    K_RBI_FILL, K_RBI_FORWARD, K_RBI_GATHER,
    K_MINMAX_LIFTED, K_MINMAX_FINISH, K_CACHED_SMALL, K_CACHED_BIG, K_CACHED_FOLD, K_MUL_FINISH, K_MUL_SWEEP,
    K_SORT_HIST, K_U32_SCAN, K_SORT_SCATTER, K_SEG_FORWARD, K_SEG_REVERSE, K_SORT_EXPORT,
    K_REDUCE_PARTIAL, K_REDUCE_FINISH, K_REDUCE_SWEEP, K_REDUCE_PACK,
    K_SOP_FORWARD, K_SOP_FINISH, K_SOP_SWEEP, K_VEC_TRANSPOSE,
    K_MS_FORWARD, K_MS_CARRY, K_MS_BACKWARD, K_MS_HIST, K_SHIFT_WORDS, K_SCAN_TILEAGG_TMA,
    K_COUNT
};
void prof_begin(int kid, cudaStream_t s);
void prof_end(int kid, cudaStream_t s);
struct LaunchScope {
    int k;
    cudaStream_t s;
    LaunchScope(int kid, cudaStream_t st) : k(kid), s(st) { prof_begin(k, s); }
    ~LaunchScope() { prof_end(k, s); }
};
// else-safe: "if (c) VJP_LAUNCH(..) a<<<>>>(); else VJP_LAUNCH(..) b<<<>>>();" pairs up as written
#define VJP_LAUNCH(kid, stream) if (::vjp::LaunchScope vjp_ls_{kid, stream}; false) {} else

// ------------------------------------------------------------------------------ scans ---
size_t scan_workspace_bytes(int code, int dtype, int64_t n);
int launch_scan_forward(int code, int dtype, int64_t n, const void *xs, void *ys, void *ws,
                        cudaStream_t stream);
int launch_scan_vjp(int code, int dtype, int64_t n, const void *xs, const void *ys_bar,
                    void *xs_bar, void *ws, int accumulate, cudaStream_t stream);
// '+' f32 scan VJP with its scratch in a static device array (no workspace, no allocation); n <= scan_noalloc_max_n()
int64_t scan_noalloc_max_n();
int launch_scan_add_f32_noalloc(int64_t n, const float *ys_bar, float *xs_bar, int accumulate, cudaStream_t stream);

// -------------------------------------------------------------- reduce-by-index (special) -
size_t rbi_special_workspace_bytes(int code, int dtype, int64_t n, int64_t w);
size_t rbi_forward_workspace_bytes(int code, int64_t n, int64_t w);
bool rbi_cached_supported(int64_t w);  // '*' / satadd tables: w <= 2^20
int launch_rbi_forward(int code, int dtype, double param, int64_t n, int64_t w, const int64_t *is,
                       const void *vs, void *hist, void *ws, cudaStream_t stream);
int launch_rbi_vjp_add(int dtype, int64_t n, int64_t w, const int64_t *is, const void *hist_bar,
                       void *vs_bar, int accumulate, cudaStream_t stream);
// MIN / MAX: lifted primal into ws, then (arg, ext) and / or the return sweep.
int launch_rbi_minmax(int code, int64_t n, int64_t w, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar, int64_t *arg, float *ext, void *ws,
                      int accumulate, cudaStream_t stream);
// MUL: lifted primal into ws, then (zeros, prod_nz) and / or the return sweep.
int launch_rbi_mul(int64_t n, int64_t w, const int64_t *is, const float *vs,
                   const float *hist_bar, float *vs_bar, int64_t *zeros, float *prod_nz, void *ws,
                   int accumulate, cudaStream_t stream, int ld = 0);
// `map2 (*)` on rows of 2^ld scalars as ONE scalar '*' problem on the flat arrays with virtual keys (bin, column):
// can launch_rbi_mul take (n << ld, w << ld, ..., ld)?
bool rbi_mul_vec_fused(int64_t n, int64_t w, int ld);

// -------------------------------------------------------------- reduce-by-index (general) -
size_t rbi_general_workspace_bytes(int64_t n, int64_t w);
int launch_rbi_general_vjp(int code, double param, int64_t n, int64_t w, const int64_t *is,
                           const float *vs, const float *hist_bar, float *vs_bar, void *ws,
                           int accumulate, int sorted, cudaStream_t stream);
// the sort-free route (rbi_multiscan.cu); gcode = G_ADD ... G_SOP of gen_ops.cuh
bool rbi_multiscan_fits(int64_t w);
size_t rbi_multiscan_workspace_bytes(int64_t n, int64_t w);
// the same walk as a plain histogram for '*' / satadd (rbi_kernels.cu uses it for 1024 < w <= 12288)
int rbi_ms_hist_tables(int64_t n, int64_t w);
int launch_ms_hist(int mul, int count_zeros, float S, int64_t n, int64_t w, const int64_t *is, const float *vs,
                   float *part, unsigned *zeros, int ld, cudaStream_t stream);
int launch_rbi_multiscan_vjp(int gcode, double param, int64_t n, int64_t w, const int64_t *is, const float *vs,
                             const float *hist_bar, float *vs_bar, void *ws, int accumulate, cudaStream_t stream);
int launch_rbi_sort_perm(int64_t n, int64_t w, const int64_t *is, int64_t *sorted_keys,
                         int64_t *perm, void *ws, cudaStream_t stream);

// ---------------------------------------------------------------- vectorised operators ---
// a = floats per entry (1: scalars; > 1: the blocks of a block-diagonal operator); cstride in entries
int launch_rows_to_cols(int64_t n, int64_t d, int64_t cstride, const float *in, float *out, cudaStream_t stream, int a = 1);
int launch_cols_to_rows(int64_t n, int64_t d, int64_t cstride, const float *in, float *out, int accumulate,
                        cudaStream_t stream, int a = 1);

// exclusive scan: move an array by `sh` 32-bit words (vec_rules.cu); fill = the words of the neutral element
struct ShiftFill { uint32_t w[32]; };
int launch_shift_words(int64_t nwords, int sh, const void *in, void *out, const ShiftFill &fill, cudaStream_t stream);

// -------------------------------------------------------------------------- sumOfProd ---
size_t rbi_sop_workspace_bytes(int64_t w);
int launch_rbi_sop_forward(int64_t n, int64_t w, const int64_t *is, const float *vs, float *hist, void *ws,
                           cudaStream_t stream);
int launch_rbi_sop_vjp_inv(int64_t n, int64_t w, const int64_t *is, const float *vs, const float *hist_bar,
                           float *vs_bar, void *ws, int accumulate, cudaStream_t stream);
int launch_rbi_sop_general_vjp(int64_t n, int64_t w, const int64_t *is, const float *vs, const float *hist_bar,
                               float *vs_bar, void *ws, int accumulate, int sorted, cudaStream_t stream);

// ----------------------------------------------------------------------------- reduce ---
size_t reduce_special_workspace_bytes();
// primal (lift = 0: y) or lifted primal (lift = 1: aux_i / aux_v of min, max, '*'); n >= 1
int launch_reduce_forward(int code, int dtype, double param, int64_t n, const void *xs, void *y,
                          int64_t *aux_i, void *aux_v, int lift, void *ws, cudaStream_t stream);
int launch_reduce_vjp(int code, int dtype, int64_t n, const void *xs, const void *y_bar, void *xs_bar,
                      void *ws, int accumulate, cudaStream_t stream);
int launch_reduce_general_vjp(int code, double param, int64_t n, const float *xs, const float *y_bar,
                              float *xs_bar, void *ws, int accumulate, cudaStream_t stream);

}  // namespace vjp
