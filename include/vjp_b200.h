/*
 * vjp_b200.h -- C ABI of the B200-native library for the reverse-mode vector-Jacobian
 * products (VJPs) of inclusive scan and reduce-by-index (generalised histogram).
 *
 * Method: arxiv/paper_2310_03568, "Reverse-Mode AD of Reduce-by-Index and Scan in Futhark".
 * "P:Lnnn" below is a line of the paper text; Qn is a reading listed in DESIGN.md.
 *
 * Conventions common to every entry point
 *   - Pointers named xs, ys, ys_bar, xs_bar, is, vs, hist, hist_bar, vs_bar, arg, ext, zeros,
 *     prod_nz, sorted_keys, perm and ws are DEVICE pointers owned by the caller, 16-byte
 *     aligned (a torch allocation is; a view such as x[1:] is not).  The library never allocates, frees or synchronises:
 *     a call validates its arguments on the host, enqueues kernels / memsets on `stream`
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream) and returns.
 *     The *_host entry points are the exception: their data pointers are HOST pointers, they
 *     copy host->device, run the same kernels, copy the result back and synchronise `stream`.
 *     Because a device-pointer call only enqueues, it may be issued on a stream that is being
 *     CAPTURED into a CUDA graph (after one call of the same kind outside the capture: kernel
 *     attributes are set on first use); replaying the graph repeats the call on the same buffers
 *     (tests/test_gpu_boundary.py, bench.py).  The scan VJP passes a TMA tensor map by value.
 *   - Scan elements are [n][d] contiguous row-major, d = vjp_scan_arity(op): 1 ('+', '*'),
 *     2 (linear recurrence (a,b)), 4 (2x2 row-major matrix), 9 (3x3), 25 (5x5 row-major matrix).
 *   - Bin indices `is` are int64.  An index outside [0, num_bins) -- negative
 *     included -- is ignored by the primal and receives adjoint exactly 0 (P:L335-336,
 *     P:L361-362; Q3).
 *   - With op.accumulate == 0 outputs are overwritten with the adjoint CONTRIBUTION (the paper's
 *     "+=" target taken as zero, Q1); with op.accumulate != 0 the VJP calls ADD the contribution
 *     to what xs_bar / vs_bar hold (the paper writes every return sweep as "+=": P:L83-88, P:L367,
 *     P:L450), fused into the kernel's final store.  The primal calls ignore the field.
 *     Outputs must not alias inputs, with one exception: vjp_scan with VJP_OP_ADD and
 *     accumulate == 0 may run in place (xs_bar == ys_bar).
 *   - Every data pointer must be 16-byte aligned (the kernels use 128-bit accesses); a misaligned
 *     pointer is VJP_ERR_INVALID_ARG.
 *   - `ws` is scratch of at least *_workspace_bytes(...) bytes; its contents need not be
 *     initialised and are garbage afterwards.  Two calls that may overlap in time need two
 *     workspaces.
 *   - Return value: VJP_OK (0) or a negative vjp_status_t; on error nothing was enqueued
 *     (VJP_ERR_CUDA excepted: a launch failed part-way).  n == 0 is VJP_OK and a no-op
 *     (reduce_by_index_forward still neutral-initialises hist).  NaN inputs are unsupported.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with
 *     VJP_ERR_CUDA.
 */
#ifndef VJP_B200_H
#define VJP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    VJP_OK = 0,
    VJP_ERR_INVALID_ARG = -1, /* NULL or misaligned pointer, negative size, unknown op / dtype */
    VJP_ERR_UNSUPPORTED = -2, /* op not defined for this combinator / dtype, n too large     */
    VJP_ERR_WORKSPACE = -3,   /* ws_bytes smaller than the *_workspace_bytes query          */
    VJP_ERR_CUDA = -4         /* a CUDA runtime call or launch failed                        */
} vjp_status_t;

typedef enum {
    VJP_OP_ADD = 0,     /* a + b, neutral 0.                       scan + reduce-by-index   */
    VJP_OP_MIN = 1,     /* min, neutral +inf, lowest index on ties.  rbi, reduce, and scan
                           (f32; the left operand keeps ties: round 2, NEXT row f4)   */
    VJP_OP_MAX = 2,     /* max, neutral -inf, lowest index on ties (Q4).      as MIN            */
    VJP_OP_MUL = 3,     /* a * b, neutral 1, exact with zeros.     scan + reduce-by-index   */
    VJP_OP_LINREC = 4,  /* (A,B)(+)(a,b) = (a*A, a*B+b), neutral (1,0) (BASELINE
                           config 3).  scan only (not commutative)                   */
    VJP_OP_MATMUL2 = 5, /* 2x2 row-major matrix product R x X, neutral I.  scan only */
    VJP_OP_MATMUL5 = 6, /* 5x5 row-major matrix product.                            scan only */
    VJP_OP_SATADD = 7,  /* min(a+b, S) on non-negative reals, neutral 0 (Q16).
                           reduce-by-index / reduce only; always the general rule (Fig. 4)   */
    VJP_OP_MATMUL3 = 8  /* 3x3 row-major matrix product (the paper's worst
                           measured overhead).  scan only (round 2, NEXT row f4)              */
} vjp_opcode_t;

typedef enum { VJP_F32 = 0, VJP_F64 = 1 } vjp_dtype_t;

/* Operator descriptor. */
typedef struct {
    int32_t code;          /* vjp_opcode_t                                                    */
    int32_t dtype;         /* vjp_dtype_t of xs / vs and of every real-valued output          */
    double param;          /* S for VJP_OP_SATADD, ignored otherwise                          */
    int32_t force_general; /* reduce-by-index only: != 0 routes '+', '*', min, max through the
                              general rule (eq. 5) instead of their specialisation
                              (P:L412-416).  1: the library picks how l_i and r_i are computed
                              (see vjp_reduce_by_index); 2: Fig. 4 as written: sort
                              + segmented scans.  SATADD always takes the general rule; for it
                              0 and 1 mean the same                                           */
    int32_t accumulate;    /* VJP calls only: != 0 adds the contribution to the output instead of
                              overwriting it               */
} vjp_op_t;

/* Scalars per scan element for op, or -1 if op is not a scan operator. */
int vjp_scan_arity(const vjp_op_t *op);

/* Library build information ("sm_100a ..." string, static storage). */
const char *vjp_version(void);

/* ------------------------------------------------------------------------------ scan ----- */

size_t vjp_scan_workspace_bytes(const vjp_op_t *op, int64_t n);

/* Primal inclusive scan ys[i] = xs[0] (.) ... (.) xs[i].  Single-pass
 * decoupled-look-back kernel.  Exists for the AD-overhead denominator.
 * Supported: ADD (f32, f64), MUL (f32, f64), MIN / MAX (f32), LINREC (f32), MATMUL2 / MATMUL3 / MATMUL5 (f32). */
int scan_forward(const vjp_op_t *op, int64_t n, const void *xs, void *ys,
                 void *ws, size_t ws_bytes, void *stream);

/* Input adjoints of the inclusive scan: xs_bar = J^T ys_bar (Fig. 7; return sweep
 * P:L553-558).
 *   ADD:   xs_bar = reverse inclusive sum of ys_bar; xs may be NULL.
 *   MIN/MAX: as `other`, but the 1-by-1 Jacobian [x_{i+1} does not win] depends on the running prefix:
 *          the reverse kernel rebuilds the forward prefixes of its tile first.
 *   other: forward tile prefixes r_{i-1} are recomputed from xs (no tape), then ONE
 *          fused reverse kernel forms the Jacobians on the fly (never stored), runs
 *          the reverse linear-recurrence scan rbar_i = ys_bar_i + J_i^T rbar_{i+1} with lin_o
 *           in its redundant-block-diagonal form, and applies the
 *          final map xs_bar_i = (d(r_{i-1} (.) x_i)/d x_i)^T rbar_i. */
int vjp_scan(const vjp_op_t *op, int64_t n, const void *xs, const void *ys_bar, void *xs_bar,
             void *ws, size_t ws_bytes, void *stream);

/* Exclusive scan, the scan^exc of the paper's Fig. 2: ys_0 = e (the operator's neutral element),
 * ys_i = x_0 (.) ... (.) x_{i-1}, and its input adjoints.  Output i is output i - 1 of the inclusive scan, so
 * xs_bar = (the inclusive rule above) applied to ys_bar moved down by one element with a zero in the last place;
 * x_{n-1} enters no output and gets adjoint 0.  Same operators, layouts, alignment and error behaviour as scan_forward
 * / vjp_scan (xs may be NULL for ADD; op.accumulate adds to xs_bar); outputs must not alias inputs.  The workspace
 * holds one array of n elements in addition to the inclusive calls' (vjp_scan_exclusive_workspace_bytes). */
size_t vjp_scan_exclusive_workspace_bytes(const vjp_op_t *op, int64_t n);
int scan_exclusive_forward(const vjp_op_t *op, int64_t n, const void *xs, void *ys,
                           void *ws, size_t ws_bytes, void *stream);
int vjp_scan_exclusive(const vjp_op_t *op, int64_t n, const void *xs, const void *ys_bar, void *xs_bar,
                       void *ws, size_t ws_bytes, void *stream);

/* The '+' rule of vjp_scan (f32: xs_bar = reverse inclusive sum of ys_bar) for callers that cannot
 * allocate and cannot pass a workspace (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc).  Same kernel as vjp_scan(VJP_OP_ADD, VJP_F32); its scratch (ticket + look-back slots, 131 328 bytes)
 * is a static __device__ array inside the library, held by every GPU that loads the library until the process
 * exits.  The call performs no cudaMalloc / cudaFree and calls no allocating routine: it clears the status words it
 * needs with a memset on `stream` and launches.
 *   n        at most vjp_scan_add_f32_noalloc_max_n() = 2^24 elements; larger n returns VJP_ERR_UNSUPPORTED
 *            (nothing is enqueued): use vjp_scan with a caller-owned workspace.  n == 0: VJP_OK, no-op.
 *   ys_bar   DEVICE, [n] f32, 16-byte aligned;  xs_bar: DEVICE, [n] f32, 16-byte aligned, may equal ys_bar
 *            (in place) unless accumulate != 0, which adds the result to xs_bar.
 *   NULL / misaligned pointer or n < 0: VJP_ERR_INVALID_ARG.  The scratch address could not be resolved on the
 *   current device, or the launch failed: VJP_ERR_CUDA.
 * ALL calls on a device share the one scratch array, and it keeps the last call's contents (each call re-clears
 * what it needs): calls that may overlap on the GPU -- different streams, or graph branches that run
 * concurrently -- race on it and give wrong results.  Calls on one stream are safe. */
int64_t vjp_scan_add_f32_noalloc_max_n(void);
int vjp_scan_add_f32_noalloc(int64_t n, const float *ys_bar, float *xs_bar, int accumulate, void *stream);

/* Same, with HOST pointers for xs, ys_bar, xs_bar.  dev_scratch is a DEVICE buffer of at least
 * vjp_scan_host_scratch_bytes() bytes (holds the three arrays and the workspace). */
size_t vjp_scan_host_scratch_bytes(const vjp_op_t *op, int64_t n);
int vjp_scan_host(const vjp_op_t *op, int64_t n, const void *xs_host, const void *ys_bar_host,
                  void *xs_bar_host, void *dev_scratch, size_t dev_scratch_bytes, void *stream);

/* ------------------------------------------------------------------- reduce-by-index ----- */

/* Workspace of vjp_reduce_by_index; the same size also covers reduce_by_index_forward, rbi_argext and
 * rbi_zero_prod of the same operator (rbi_sort_perm: query with op.code = VJP_OP_SATADD). */
size_t vjp_reduce_by_index_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t num_bins);

/* Primal reduce_by_index over a neutral-initialised histogram (P:L332-336 after the rewrite of
 * there is no hist_0 argument).  hist[num_bins] is fully written.
 * Supported: ADD (f32, f64), MIN, MAX, MUL, SATADD (f32).  ADD needs no workspace (ws may be NULL);
 * the others return VJP_ERR_WORKSPACE if ws is too small.  MUL and SATADD keep shared-memory tables of
 * 32768 bins per CTA, split over groups of up to 32 CTAs: num_bins > 2^20 returns VJP_ERR_UNSUPPORTED. */
int reduce_by_index_forward(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                            const void *vs, void *hist, void *ws, size_t ws_bytes, void *stream);

/* Input adjoints vs_bar[n] of reduce_by_index w.r.t. vs, given hist_bar[num_bins].
 *   ADD:      gather vs_bar[i] = hist_bar[is[i]]; vs may be NULL.  Bit-exact copy.
 *   MIN/MAX:  lifted primal (index, value) per bin, lowest index on ties (Fig. 5),
 *             then vs_bar = 0 and vs_bar[arg[k]] = hist_bar[k].  Bit-exact copy.
 *   MUL:      lifted primal (zero count, product of non-zeros) (Fig. 3),
 *             then the three-way map of P:L208-219 / P:L243-246.  num_bins <= 2^20, else
 *             VJP_ERR_UNSUPPORTED (force_general handles any num_bins).
 *   SATADD or force_general: the general rule, eq. 5:
 *             vs_bar_i = d(l_i (.) x (.) r_i)/dx at vs_i * hist_bar[is_i], l_i / r_i = the fold of the
 *             same-bin values before / after i.  Two routes to l and r, same results:
 *             - num_bins <= 12288 and force_general != 2: no sort.  Two in-order walks over the input,
 *               each warp with a running per-bin table in shared memory (forward: l, backward: r),
 *               per-chunk carries scanned in between; every array is read and written in its
 *               original order (36 bytes per element).
 *             - otherwise (or force_general == 2): Fig. 4 as written: stable radix sort
 *               by clamped bin, forward and reverse segmented exclusive scans, derivative, un-permute.
 *             min / max give the adjoint of tied extrema to the lowest index on both routes.
 * n must be < 2^32 - 1 (packed 32-bit positions). */
int vjp_reduce_by_index(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                        const void *vs, const void *hist_bar, void *vs_bar,
                        void *ws, size_t ws_bytes, void *stream);

/* Same, with HOST pointers for is, vs, hist_bar, vs_bar. */
size_t vjp_reduce_by_index_host_scratch_bytes(const vjp_op_t *op, int64_t n, int64_t num_bins);
int vjp_reduce_by_index_host(const vjp_op_t *op, int64_t n, int64_t num_bins,
                             const int64_t *is_host, const void *vs_host,
                             const void *hist_bar_host, void *vs_bar_host,
                             void *dev_scratch, size_t dev_scratch_bytes, void *stream);
/* The same without the final synchronisation: copies in, kernels and the copy out are only enqueued
 * on `stream` (host buffers should be pinned for the copies to be asynchronous).  The caller
 * synchronises `stream` before it reads vs_bar_host or reuses dev_scratch / the host inputs; calls on
 * different streams with different dev_scratch buffers overlap their copies with each other's kernels. */
int vjp_reduce_by_index_host_async(const vjp_op_t *op, int64_t n, int64_t num_bins,
                                   const int64_t *is_host, const void *vs_host,
                                   const void *hist_bar_host, void *vs_bar_host,
                                   void *dev_scratch, size_t dev_scratch_bytes, void *stream);

/* Inspection entry points: the integer-valued intermediates, for bit-exact comparison. */

/* MIN / MAX lifted primal (Fig. 5): arg[k] = lowest index attaining the extremum of bin k, or n
 * for an empty bin; ext[k] = the extremum (+-inf for an empty bin), dtype f32. */
int rbi_argext(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is, const void *vs,
               int64_t *arg, void *ext, void *ws, size_t ws_bytes, void *stream);

/* MUL lifted primal: zeros[k] = #{i : is[i]=k, vs[i]==0} (IEEE equality, Q7),
 * prod_nz[k] = product of the non-zero members (1 if none), dtype f32. */
int rbi_zero_prod(const vjp_op_t *op, int64_t n, int64_t num_bins, const int64_t *is,
                  const void *vs, int64_t *zeros, void *prod_nz, void *ws, size_t ws_bytes,
                  void *stream);

/* Stable sort of (key', iota) by key' = is[i] if in range else num_bins (Fig. 4 P:L350-351;
 * Q18).  sorted_keys[n], perm[n] are int64.  Workspace: that of the general rule
 * (query with op.code = VJP_OP_SATADD). */
int rbi_sort_perm(int64_t n, int64_t num_bins, const int64_t *is, int64_t *sorted_keys,
                  int64_t *perm, void *ws, size_t ws_bytes, void *stream);

/* ---------------------------------------------------------------- vectorised operators ----- */

/* reduce_by_index and scan with the vectorised operator `map2 (.)` on rows of d f32 scalars
 * (sections 3.2.4 / 4.2.5): vss, vss_bar are [n][d], hist_bar is [num_bins][d]; xss, yss_bar, xss_bar are [n][d].
 * The rule is the INTERCHANGE of the combinator with the inner map (IRWIM eq. 3 P:L252-263 and its
 * reduce-by-index form P:L464-466; ISWIM P:L655-657): the arrays are transposed, the scalar rule runs on each of
 * the d columns (any scalar operator the scalar entry point accepts in f32: ADD, MIN, MAX, MUL, SATADD for
 * reduce_by_index; ADD, MUL, MIN, MAX for scan), and the result is transposed back (op.accumulate fused there).
 * reduce_by_index with MUL, d a power of two and 1024 < num_bins * d <= 12288 skips the transposes: the d histograms
 * are one histogram over (bin, column) pairs, computed on the flat arrays with virtual keys is[j / d] * d + j % d.
 * vjp_scan_vec also takes the operators of arity a > 1 (LINREC, MATMUL2 / 3 / 5): rows are d blocks of a scalars, the
 * operator applies (.) to every block -- a block-diagonal Jacobian of d DIFFERENT blocks (non-redundant BDS,
 * rs_bar by d scans with the scaled-down operator); xss, yss_bar, xss_bar are [n][d * a].
 * d <= 4096. */
size_t vjp_reduce_by_index_vec_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t d, int64_t num_bins);
int vjp_reduce_by_index_vec(const vjp_op_t *op, int64_t n, int64_t d, int64_t num_bins, const int64_t *is,
                            const void *vss, const void *hist_bar, void *vss_bar,
                            void *ws, size_t ws_bytes, void *stream);
size_t vjp_scan_vec_workspace_bytes(const vjp_op_t *op, int64_t n, int64_t d);
int vjp_scan_vec(const vjp_op_t *op, int64_t n, int64_t d, const void *xss, const void *yss_bar,
                 void *xss_bar, void *ws, size_t ws_bytes, void *stream);

/* -------------------------------------------------------------------------- sumOfProd ----- */

/* reduce_by_index with the invertible operator sumOfProd (sections 3.3 and 4.2.4 of the paper):
 *   (p1,s1) sumOfProd (p2,s2) = (p1 + p2 + s1*s2, s1 + s2), neutral (0,0)
 * Elements are f32 pairs: vs [n][2] = (p, s), hist / hist_bar [num_bins][2], vs_bar [n][2].
 * Primal: the fold of a bin has the closed form P = sum p + ((sum s)^2 - sum s^2) / 2 = sum (p - s^2 / 2) + S^2 / 2,
 * S = sum s, so the histogram is two float atomicAdd histograms and a finish pass. */
size_t rbi_sumofprod_workspace_bytes(int64_t n, int64_t num_bins, int use_general);
int rbi_sumofprod_forward(int64_t n, int64_t num_bins, const int64_t *is, const float *vs, float *hist,
                          void *ws, size_t ws_bytes, void *stream);

/* Input adjoints vs_bar of the above.
 *   use_general == 0: the invertible-operator rule of Fig. 6: xs = the primal histogram,
 *                     b_i = xs[k_i] sumOfProd_inv v_i, vs_bar_i = (d(b_i (.) x)/dx)^T hist_bar[k_i]
 *                     -- a histogram and a map.
 *   use_general != 0: the general rule (eq. 5) for the same operator -- the paper's 8 - 92x against
 *                     1.1 - 2.1x contrast.  1: route picked as in vjp_reduce_by_index (no sort
 *                     for num_bins <= 12288); 2: Fig. 4 as written (sort by bin + segmented scans).
 * accumulate != 0 adds to vs_bar.  Keys outside [0, num_bins) get (0, 0). */
int vjp_rbi_sumofprod(int64_t n, int64_t num_bins, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar, int use_general, int accumulate,
                      void *ws, size_t ws_bytes, void *stream);

/* ----------------------------------------------------------------------------- reduce ----- */

/* reduce (section 3 of the paper): y = a_0 (.) a_1 (.) ... (.) a_{n-1}, one scalar.
 * y, y_bar point to ONE scalar of op.dtype in DEVICE memory (naturally aligned is enough).
 * Operators: ADD (f32, f64), MIN, MAX, MUL, SATADD (f32).  n < 2^32 - 1. */
size_t vjp_reduce_workspace_bytes(const vjp_op_t *op, int64_t n);

/* Primal y = reduce (.) e xs; n == 0 gives the neutral element.  Two-level tree
 * reduction (one partial per CTA, folded in a fixed order: deterministic). */
int reduce_forward(const vjp_op_t *op, int64_t n, const void *xs, void *y, void *ws, size_t ws_bytes,
                   void *stream);

/* Input adjoints xs_bar[n] of reduce, given y_bar.
 *   ADD:     xs_bar = replicate n y_bar; xs may be NULL.
 *   MIN/MAX: lifted primal (k, y) with the smallest index on ties, then xs_bar = 0 and
 *            xs_bar[k] = y_bar.  Bit-exact copy.
 *   MUL:     lifted primal (number of zeros, product of the non-zeros), then the three-way map of
 *            Fig. 3.
 *   SATADD or force_general: the general rule, eq. 2 -- forward and reverse exclusive
 *            scans l_i, r_i (Fig. 2), xs_bar_i = d(l_i (.) x_i (.) r_i)/dx_i * y_bar;
 *            runs the segmented-scan kernels of the reduce-by-index general rule with one segment.
 * op.accumulate adds to xs_bar ("as_bar +="). */
int vjp_reduce(const vjp_op_t *op, int64_t n, const void *xs, const void *y_bar, void *xs_bar,
               void *ws, size_t ws_bytes, void *stream);

/* Inspection: the lifted primal's integer and value (device scalars), for bit-exact comparison.
 *   MIN/MAX: *aux_i = k (n for an empty array), *aux_v = the extremum (f32).
 *   MUL:     *aux_i = number of zeros (IEEE equality, Q7), *aux_v = product of the non-zeros. */
int reduce_lifted(const vjp_op_t *op, int64_t n, const void *xs, int64_t *aux_i, void *aux_v,
                  void *ws, size_t ws_bytes, void *stream);

/* ------------------------------------------------------------------ instrumentation ----- */

/* The library's kernels are numbered 0 .. vjp_kernel_count()-1; vjp_kernel_name gives the kernel's
 * name (static storage; NULL if out of range).  vjp_launch_count(kid) is the number of launches of
 * kernel kid since the library was loaded, kid < 0 the total over all kernels (cudaMemsetAsync
 * calls are not kernels of this library and are not counted). */
int vjp_kernel_count(void);
const char *vjp_kernel_name(int kid);
int64_t vjp_launch_count(int kid);

/* While enabled, every kernel launch is bracketed by CUDA events on its stream (at most 8192
 * launches are recorded; enabling clears the record).  vjp_profile_read synchronises on the
 * recorded events and returns the summed duration and the number of recorded launches of kernel
 * kid.  Not thread-safe; meant for bench.py's per-kernel roofline, off by default. */
void vjp_profile_enable(int on);
int vjp_profile_read(int kid, double *total_ms, int64_t *launches);

#ifdef __cplusplus
}
#endif
#endif /* VJP_B200_H */
