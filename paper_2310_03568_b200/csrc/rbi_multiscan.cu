// rbi_multiscan.cu -- the general-case rule for reduce-by-index (eq. 5) WITHOUT the sort:
//
//   vs_bar_i = d(l_i (.) x (.) r_i)/dx at x = vs_i  *  hist_bar[is_i],
//   l_i = fold of the same-bin values BEFORE i,   r_i = fold of the same-bin values AFTER i
//
// Fig. 4 gets l and r by sorting (key, iota) and running two segmented scans over the sorted values:
// six passes over n-sized arrays, two of them scatters, and a random un-permute at the end (rbi_general.cu; the paper
// itself reports that the sort dominates).  The sort is only a means: what eq. 5 needs is, per element,
// the per-bin exclusive folds in index order.  When a bin table fits a warp's share of shared memory (w = 4096 f32
// states = 16 KB, 13 warps per SM: the C5 workload; accepted up to w = 12 288 = 3 warps per SM, where the walks still take
// half the time of the sort-based route: 0.41 against 0.81 ms at n = 2^24) they come from two in-order walks with a RUNNING per-bin table, with no data movement
// at all -- every array is read and written in its original order, fully coalesced:
//
//   forward   each warp owns a contiguous chunk of the input and a private table tab[w] (neutral-initialised).  Per row
//             of 32 consecutive elements: lanes holding the same bin are found with match.any; an exclusive fold along
//             each such group in lane (= index) order by pointer jumping; l_local_i = tab[bin] (.) that fold; the last
//             lane of the group stores the group's inclusive fold back.  l_local -> global (4 B / element); at the end of
//             the chunk the table IS the chunk's per-bin aggregate -> agg[chunk][w].
//   carry     per bin, exclusive prefix L[chunk][bin] and exclusive suffix R[chunk][bin] of agg over the chunks, in two
//             levels: among the chunks of one CTA in the forward kernel's epilogue (the tables are still in shared
//             memory), among the CTAs by two small kernels over the 148 CTA aggregates.
//   backward  the same walk from the end of the chunk towards its start, table initialised with R[chunk][.]: gives
//             r_i directly; l_i = L[chunk][bin] (.) l_local_i; then the derivative and the store of vs_bar_i in place
//             (original order: no scatter).  Out-of-range keys take no part and get 0.
//             The operator is commutative, so d(l (.) x (.) r)/dx depends on l and r only through l (.) r:
//             for every operator but min / max the table starts as L[chunk][.] (.) R[chunk][.] and l_local stands
//             for l -- no per-element gather of L (16 M random L2 reads cost 158 us at w = 4096, more than the rest
//             of the kernel).  min / max break ties by index ("v < l" strict, "r < v" not), so they keep the gather.
//             hist_bar sits in shared memory next to the tables (its gather from L1 / L2 cost another 48 us).
//
// Index order matters beyond associativity only for min / max, whose ties give the adjoint to the lowest index
// (P:L425-428): rows are 32 CONSECUTIVE elements and chunks are contiguous, so "before" is always the true index order.
// Traffic: forward 12 B read + 4 B written per element, backward 16 B read + 4 B written: 36 B / element against
// ~90 B for the sort-based route.
#include "gen_ops.cuh"
#include "internal.h"
#include "ms_walk.cuh"

namespace vjp {

constexpr size_t MS_SMEM_BUDGET = 224 * 1024;  // warp tables of one CTA
constexpr int MS_W_MAX = 12288;                // bins (one f32 state each) a warp-private table may hold
constexpr int MS_SEG = 32;                     // chunks per carry segment (held in registers)
constexpr int MS_MIN_ROWS = 8;                 // do not split the input finer than this many rows per warp

bool rbi_multiscan_fits(int64_t w) { return w >= 1 && w <= MS_W_MAX; }

// shared memory of a CTA: hist_bar (hw words per bin: 2 for the pairs of sumOfProd) + one table of w floats per warp
static int ms_warps_per_cta(int64_t w, int hw) {
    const int fit = (int)((MS_SMEM_BUDGET - (size_t)w * 4 * hw) / ((size_t)w * 4));
    return fit > 32 ? 32 : fit;
}

struct MsShape {
    int wpc, grid;
    int64_t G, R, segs;  // chunks (warps), rows per chunk, carry segments (of MS_SEG CTAs)
};
static MsShape ms_shape(int64_t n, int64_t w, int hw) {
    MsShape s;
    s.wpc = ms_warps_per_cta(w, hw);
    const int64_t rows = (n + 31) / 32;
    int64_t want = (rows + MS_MIN_ROWS - 1) / MS_MIN_ROWS;
    const int64_t cap = (int64_t)NUM_SMS_B200 * s.wpc;
    if (want > cap) want = cap;
    if (want < 1) want = 1;
    s.grid = (int)((want + s.wpc - 1) / s.wpc);
    s.G = (int64_t)s.grid * s.wpc;
    s.R = (rows + s.G - 1) / s.G;
    if (s.R < 1) s.R = 1;
    s.segs = (s.grid + MS_SEG - 1) / MS_SEG;  // the carry kernels scan the CTA aggregates
    return s;
}

// One row of the backward walk.  Returns r (later same-bin lanes (.) table) and updates the table.
template <int CODE>
VJP_DEVINL float ms_row_backward(const GenOp<CODE> &op, float *tab, int64_t k, float x, int64_t w, int lane) {
    const bool inr = (uint64_t)k < (uint64_t)w;
    const uint32_t key = inr ? (uint32_t)k : (0x80000000u | (uint32_t)lane);
    uint32_t *tabu = reinterpret_cast<uint32_t *>(tab);
    const float t = inr ? tab[key] : op.neutral();
    __syncwarp();
    if (inr) tabu[key] = MS_CLAIM | (uint32_t)lane;
    __syncwarp();
    const bool lost = inr && tabu[key] != (MS_CLAIM | (uint32_t)lane);
    if (!__any_sync(FULL_MASK, lost)) {
        if (inr) tab[key] = op.apply(x, t);
        __syncwarp();
        return t;
    }
    const uint32_t m = __match_any_sync(FULL_MASK, key);
    const uint32_t higher = m & (0xfffffffeu << lane);
    const int next0 = higher ? __ffs(higher) - 1 : -1;
    float suf = x;  // fold over [lane, nj) along the group's list
    int nj = next0;
    while (__any_sync(FULL_MASK, nj >= 0)) {
        const int src = nj < 0 ? lane : nj;
        const float sv = __shfl_sync(FULL_MASK, suf, src);
        const int nn = __shfl_sync(FULL_MASK, nj, src);
        if (nj >= 0) {
            suf = op.apply(suf, sv);
            nj = nn;
        }
    }
    const float exv = __shfl_sync(FULL_MASK, suf, next0 < 0 ? lane : next0);
    const float r = next0 < 0 ? t : op.apply(exv, t);
    const bool first = (m & ((1u << lane) - 1u)) == 0u;
    if (inr & first) tab[key] = op.apply(suf, t);
    __syncwarp();
    return r;
}

// WMAX = warps per CTA the kernel is compiled for (register budget), D = rows of loads in flight per warp.
template <int CODE, int WMAX, int D>
__global__ void __launch_bounds__(WMAX * 32, 1)
ms_forward_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const float *__restrict__ vs, int vstride,
                  float *__restrict__ ls, float *__restrict__ intraA, float *__restrict__ intraB,
                  float *__restrict__ ctaagg, int64_t R, GenOp<CODE> op) {
    extern __shared__ float ms_smem[];
    constexpr bool SYM = CODE != G_MIN && CODE != G_MAX;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    float *tab = ms_smem + (size_t)warp * (size_t)w;
    for (int i = lane; i < (int)w; i += 32) tab[i] = op.neutral();
    __syncwarp();
    const int64_t g = (int64_t)blockIdx.x * wpc + warp;
    const int64_t rows = (n + 31) >> 5;
    const int64_t r0 = min(g * R, rows), r1 = min(r0 + R, rows);
    const int64_t rfull = min(r1, n >> 5);  // rows below rfull have all 32 elements
    const int64_t vs32 = 32 * (int64_t)vstride;
    int64_t kn[D];
    float vn[D];
    // a block of D whole rows inside the chunk: plain loads at constant offsets (the common case, ~20 instructions
    // per row fewer than the predicated form: the walk is issue-bound at 13 warps per SM)
    auto fetch = [&](int64_t rb) {
        if (rb + D <= rfull) {
            const int64_t *kp = is + rb * 32 + lane;
            const float *vp = vs + (rb * 32 + lane) * vstride;
#pragma unroll
            for (int d = 0; d < D; d++) {
                kn[d] = __ldg(kp + d * 32);
                vn[d] = __ldg(vp + d * vs32);
            }
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) {
                const int64_t idx = (rb + d) * 32 + lane;
                const bool ok = (rb + d < r1) & (idx < n);
                kn[d] = ok ? __ldg(is + idx) : (int64_t)-1;
                vn[d] = ok ? __ldg(vs + idx * vstride) : 0.f;
            }
        }
    };
    fetch(r0);
    for (int64_t rb = r0; rb < r1; rb += D) {
        int64_t k[D];
        float v[D];
#pragma unroll
        for (int d = 0; d < D; d++) {
            k[d] = kn[d];
            v[d] = vn[d];
        }
        fetch(rb + D);  // the next block's loads fly while this one is walked
        if (rb + D <= rfull) {
            float *lp = ls + rb * 32 + lane;
#pragma unroll
            for (int d = 0; d < D; d++) lp[d * 32] = ms_row_forward<CODE>(op, tab, k[d], v[d], w, lane);
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) {
                if (rb + d < r1) {  // warp-uniform
                    const float l = ms_row_forward<CODE>(op, tab, k[d], v[d], w, lane);
                    const int64_t idx = (rb + d) * 32 + lane;
                    if (idx < n) ls[idx] = l;
                }
            }
        }
    }
    // Epilogue: the tables of the CTA's warps are the aggregates of wpc CONSECUTIVE chunks.  Per bin, what the other
    // chunks of this CTA contribute to chunk j -- the fold of the warps before it (P_j) and after it (S_j) -- is formed
    // here, from shared memory; only the CTA totals go through the carry kernels (148 rows instead of ~1900).
    //   SYM operators:  intraA[g][b] = P_j (.) S_j          (L and R are only ever used as L (.) R, see the header)
    //   min / max:      intraA[g][b] = P_j,  intraB[g][b] = S_j
    __syncthreads();
    const int64_t g0 = (int64_t)blockIdx.x * wpc;
    for (int b = threadIdx.x; b < (int)w; b += blockDim.x) {
        float sfx[WMAX];
        float suf = op.neutral();
#pragma unroll
        for (int j = WMAX - 1; j >= 0; j--) {
            sfx[j] = suf;
            if (j < wpc) suf = op.apply(ms_smem[(size_t)j * w + b], suf);
        }
        float pre = op.neutral();
#pragma unroll
        for (int j = 0; j < WMAX; j++) {
            if (j < wpc) {
                if constexpr (SYM) {
                    intraA[(g0 + j) * w + b] = op.apply(pre, sfx[j]);
                } else {
                    intraA[(g0 + j) * w + b] = pre;
                    intraB[(g0 + j) * w + b] = sfx[j];
                }
                pre = op.apply(pre, ms_smem[(size_t)j * w + b]);
            }
        }
        ctaagg[(int64_t)blockIdx.x * w + b] = pre;
    }
}

template <int CODE, int WMAX, int D>
__global__ void __launch_bounds__(WMAX * 32, 1)
ms_backward_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const float *__restrict__ vs, int vstride,
                   const float *__restrict__ ls, float *intraA, const float *__restrict__ intraB,
                   const float *__restrict__ ctaL, const float *__restrict__ ctaR,
                   const float *__restrict__ hist_bar, float *__restrict__ vs_bar, int64_t R, GenOp<CODE> op,
                   int accumulate) {
    extern __shared__ float ms_smem[];
    constexpr bool SYM = CODE != G_MIN && CODE != G_MAX;  // see the header: L folded into the table
    constexpr int HW = CODE == G_SOP ? 2 : 1;             // words of hist_bar per bin
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    float *hs = ms_smem;                                  // [w][HW]
    float *tab = ms_smem + (size_t)w * HW + (size_t)warp * (size_t)w;
    const int64_t g = (int64_t)blockIdx.x * wpc + warp;
    for (int i = threadIdx.x; i < (int)w * HW; i += blockDim.x) hs[i] = hist_bar[i];
    // what lies outside the chunk: the other chunks of this CTA (forward kernel's epilogue) and the other CTAs (carry
    // kernels).  SYM: all of it on the r side.  min / max: the right part in the table, the left part L[g][.] written
    // back over intraA for the per-element gather.
    float *Lg = intraA + g * w;
    const float *cl = ctaL + (int64_t)blockIdx.x * w, *cr = ctaR + (int64_t)blockIdx.x * w;
    for (int i = lane; i < (int)w; i += 32) {
        if constexpr (SYM) {
            tab[i] = op.apply(op.apply(cl[i], Lg[i]), cr[i]);
        } else {
            tab[i] = op.apply(intraB[g * w + i], cr[i]);
            Lg[i] = op.apply(cl[i], Lg[i]);
        }
    }
    __syncthreads();
    const int64_t rows = (n + 31) >> 5;
    const int64_t r0 = min(g * R, rows), r1 = min(r0 + R, rows);
    // rows are walked from r1 - 1 down to r0, D at a time: block b covers rows r1 - 1 - b*D - d
    int64_t kn[D];
    float vn[D], ln[D];
    const int64_t nfull = n >> 5;  // rows below nfull have all 32 elements
    const int64_t vs32 = 32 * (int64_t)vstride;
    auto fetch = [&](int64_t top) {  // top = highest row of the block
        if (top - (D - 1) >= r0 && top < nfull) {  // D whole rows inside the chunk
            const int64_t *kp = is + top * 32 + lane;
            const float *vp = vs + (top * 32 + lane) * vstride;
            const float *lp = ls + top * 32 + lane;
#pragma unroll
            for (int d = 0; d < D; d++) {
                kn[d] = __ldg(kp - d * 32);
                vn[d] = __ldg(vp - d * vs32);
                ln[d] = __ldg(lp - d * 32);
            }
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) {
                const int64_t row = top - d;
                const int64_t idx = row * 32 + lane;
                const bool ok = (row >= r0) & (idx < n);
                kn[d] = ok ? __ldg(is + idx) : (int64_t)-1;
                vn[d] = ok ? __ldg(vs + idx * vstride) : 0.f;
                ln[d] = ok ? __ldg(ls + idx) : 0.f;
            }
        }
    };
    fetch(r1 - 1);
    for (int64_t top = r1 - 1; top >= r0; top -= D) {
        int64_t k[D];
        float v[D], ll[D], lc[SYM ? 1 : D];
#pragma unroll
        for (int d = 0; d < D; d++) {
            k[d] = kn[d];
            v[d] = vn[d];
            ll[d] = ln[d];
        }
        fetch(top - D);
        if constexpr (!SYM) {
#pragma unroll
            for (int d = 0; d < D; d++)  // the gathers of the whole block are issued before the walk
                lc[d] = (uint64_t)k[d] < (uint64_t)w ? Lg[k[d]] : op.neutral();  // written above by this warp: no __ldg
        }
        // the table walk of the whole block first (shared-memory latencies only), then the outputs: by then the
        // gathers have arrived, and a wait on them no longer sits between two rows of the (in-order) walk
        const bool fullb = (top - (D - 1) >= r0) & (top < nfull);  // D whole rows inside the chunk (warp-uniform)
        // one element's output; `o1` points at vs_bar[idx] (pairs for sumOfProd)
        auto emit = [&](int d, float r, float *o1) {
            const bool inr = (uint64_t)k[d] < (uint64_t)w;
            float l = ll[d];
            if constexpr (!SYM) l = op.apply(lc[d], l);
            const float h0 = inr ? hs[(uint32_t)k[d] * HW] : 0.f;
            const float gq = inr ? op.dfdx(l, v[d], r) * h0 : 0.f;  // 0 out of range
            if constexpr (CODE == G_SOP) {  // vs_bar_i = (Pbar, Pbar * (ls + rs) + Sbar)
                float2 *dst = reinterpret_cast<float2 *>(o1);
                float2 o = make_float2(h0, gq + (inr ? hs[(uint32_t)k[d] * 2 + 1] : 0.f));
                if (accumulate) {
                    const float2 pr = *dst;
                    o.x += pr.x;
                    o.y += pr.y;
                }
                *dst = o;
            } else {
                *o1 = accumulate ? *o1 + gq : gq;
            }
        };
        float rr[D];
        if (fullb) {
#pragma unroll
            for (int d = 0; d < D; d++) rr[d] = ms_row_backward<CODE>(op, tab, k[d], v[d], w, lane);
            float *op1 = vs_bar + (top * 32 + lane) * HW;
#pragma unroll
            for (int d = 0; d < D; d++) emit(d, rr[d], op1 - d * 32 * HW);
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) {
                rr[d] = op.neutral();
                if (top - d >= r0) rr[d] = ms_row_backward<CODE>(op, tab, k[d], v[d], w, lane);  // warp-uniform
            }
#pragma unroll
            for (int d = 0; d < D; d++) {
                const int64_t row = top - d;
                const int64_t idx = row * 32 + lane;
                if (row >= r0 && idx < n) emit(d, rr[d], vs_bar + idx * HW);
            }
        }
    }
}

// The same walk as a plain HISTOGRAM for the operators with no hardware atomic ('*', satadd; H0 / H4 for
// 1024 < w <= MS_W_MAX, where rbi_cached_big_kernel needs CTA-wide claim rounds between barriers): no l is stored, the
// epilogue folds the CTA's warp tables in warp order into ONE partial table per CTA (deterministic), which the fold
// kernels of rbi_kernels.cu combine.  COUNT_ZEROS (the lifted '*' of P:L460): an exact zero is counted in zeros[bin]
// and takes no part in the product.
// VEC (the vectorised operator `map2 (.)` on rows of d = 2^ld scalars, eq. 3 P:L252-263 / P:L464-466): reduce_by_index
// with map2 (.) is d independent histograms = ONE histogram over (bin, column) pairs.  The [n][d] values are walked as
// a flat array of n * d scalars whose element j has the virtual key is[j >> ld] * d + (j & (d - 1)), with w * d
// virtual bins: the keys are read once per row, nothing is transposed.  Here n and w are the FLAT sizes.
template <int CODE, int WMAX, int D, bool COUNT_ZEROS, bool VEC>
__global__ void __launch_bounds__(WMAX * 32, 1)
ms_hist_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const float *__restrict__ vs,
               float *__restrict__ part, unsigned *zeros, int64_t R, GenOp<CODE> op, int ld) {
    extern __shared__ float ms_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    float *tab = ms_smem + (size_t)warp * (size_t)w;
    for (int i = lane; i < (int)w; i += 32) tab[i] = op.neutral();
    __syncwarp();
    const int64_t g = (int64_t)blockIdx.x * wpc + warp;
    const int64_t rows = (n + 31) >> 5;
    const int64_t r0 = min(g * R, rows), r1 = min(r0 + R, rows);
    const int64_t rfull = min(r1, n >> 5);
    int64_t kn[D];
    float vn[D];
    auto fetch = [&](int64_t rb) {
        if (rb + D <= rfull) {
            const float *vp = vs + rb * 32 + lane;
#pragma unroll
            for (int d = 0; d < D; d++) {
                kn[d] = __ldg(is + (VEC ? (rb * 32 + lane + d * 32) >> ld : rb * 32 + lane + d * 32));
                vn[d] = __ldg(vp + d * 32);
            }
        } else {
#pragma unroll
            for (int d = 0; d < D; d++) {
                const int64_t idx = (rb + d) * 32 + lane;
                const bool ok = (rb + d < r1) & (idx < n);
                kn[d] = ok ? __ldg(is + (VEC ? idx >> ld : idx)) : (int64_t)-1;
                vn[d] = ok ? __ldg(vs + idx) : 1.f;
            }
        }
    };
    fetch(r0);
    for (int64_t rb = r0; rb < r1; rb += D) {
        int64_t k[D];
        float v[D];
#pragma unroll
        for (int d = 0; d < D; d++) {
            k[d] = kn[d];
            v[d] = vn[d];
            if constexpr (VEC) {  // virtual key (bin, column); a key outside [0, w >> ld) stays out of range
                const int64_t col = ((rb + d) * 32 + lane) & (((int64_t)1 << ld) - 1);
                k[d] = (uint64_t)k[d] < (uint64_t)(w >> ld) ? (k[d] << ld) | col : (int64_t)-1;
            }
        }
        fetch(rb + D);
#pragma unroll
        for (int d = 0; d < D; d++) {
            if (rb + d < r1) {  // warp-uniform
                if (COUNT_ZEROS) {
                    if ((uint64_t)k[d] < (uint64_t)w && v[d] == 0.f) {  // IEEE equality: +-0 only (Q7)
                        atomicAdd(zeros + k[d], 1u);
                        k[d] = -1;
                    }
                }
                ms_row_forward<CODE>(op, tab, k[d], v[d], w, lane);
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < (int)w; b += blockDim.x) {
        float acc = ms_smem[b];
        for (int j = 1; j < wpc; j++) acc = op.apply(acc, ms_smem[(size_t)j * w + b]);
        part[(int64_t)blockIdx.x * w + b] = acc;
    }
}

// Carry, level 1: segagg[seg][b] = fold of agg[g][b] over the chunks g of segment seg (in order).
template <int CODE>
__global__ void ms_seg_agg_kernel(int64_t w, int64_t G, const float *__restrict__ agg, float *__restrict__ segagg,
                                  GenOp<CODE> op) {
    const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t seg = blockIdx.y;
    if (b >= w) return;
    const int64_t g0 = seg * MS_SEG, g1 = min(g0 + MS_SEG, G);
    float a[MS_SEG];
#pragma unroll
    for (int j = 0; j < MS_SEG; j++) a[j] = g0 + j < g1 ? __ldg(agg + (g0 + j) * w + b) : op.neutral();
    float acc = op.neutral();
#pragma unroll
    for (int j = 0; j < MS_SEG; j++) acc = op.apply(acc, a[j]);
    segagg[seg * w + b] = acc;
}

// Carry, level 2: L[g][b] (in place of agg) and R[g][b] for the chunks of one segment.
template <int CODE>
__global__ void ms_carry_kernel(int64_t w, int64_t G, int64_t segs, float *__restrict__ aggL, float *__restrict__ Rc,
                                const float *__restrict__ segagg, GenOp<CODE> op) {
    const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t seg = blockIdx.y;
    if (b >= w) return;
    const int64_t g0 = seg * MS_SEG, g1 = min(g0 + MS_SEG, G);
    float a[MS_SEG];
#pragma unroll
    for (int j = 0; j < MS_SEG; j++) a[j] = g0 + j < g1 ? aggL[(g0 + j) * w + b] : op.neutral();
    // the segments before / after this one: loads in batches of 16 (independent), folds in order
    float pre = op.neutral(), suf = op.neutral();
    for (int64_t s0 = 0; s0 < seg; s0 += 16) {
        float q[16];
#pragma unroll
        for (int j = 0; j < 16; j++) q[j] = s0 + j < seg ? __ldg(segagg + (s0 + j) * w + b) : op.neutral();
#pragma unroll
        for (int j = 0; j < 16; j++) pre = op.apply(pre, q[j]);
    }
    for (int64_t s0 = segs - 1; s0 > seg; s0 -= 16) {
        float q[16];
#pragma unroll
        for (int j = 0; j < 16; j++) q[j] = s0 - j > seg ? __ldg(segagg + (s0 - j) * w + b) : op.neutral();
#pragma unroll
        for (int j = 0; j < 16; j++) suf = op.apply(q[j], suf);
    }
#pragma unroll
    for (int j = 0; j < MS_SEG; j++) {
        if (g0 + j < g1) aggL[(g0 + j) * w + b] = pre;
        pre = op.apply(pre, a[j]);
    }
#pragma unroll
    for (int j = MS_SEG - 1; j >= 0; j--) {
        if (g0 + j < g1) Rc[(g0 + j) * w + b] = suf;
        suf = op.apply(a[j], suf);
    }
}

// ------------------------------------------------------------------ host side -------------

struct MsWs {
    float *ls, *intraA, *intraB, *ctaL, *ctaR, *segagg;
    size_t total;
};
static MsWs ms_carve(void *ws, int64_t n, int64_t w) {
    // the workspace query does not know the operator: rows for whichever of the two table shapes (hist_bar of 1 or 2
    // words per bin) has more chunks / more CTAs at this (n, w)
    const MsShape s1 = ms_shape(n < 1 ? 1 : n, w < 1 ? 1 : w, 1), s2 = ms_shape(n < 1 ? 1 : n, w < 1 ? 1 : w, 2);
    const size_t G = (size_t)(s1.G > s2.G ? s1.G : s2.G), grid = (size_t)(s1.grid > s2.grid ? s1.grid : s2.grid);
    const size_t segs = (size_t)(s1.segs > s2.segs ? s1.segs : s2.segs);
    MsWs m;
    char *p = static_cast<char *>(ws);
    auto take = [&](size_t bytes) { char *r = p; p += align_up(bytes, 256); return r; };
    m.ls = reinterpret_cast<float *>(take((size_t)(n < 1 ? 1 : n) * 4));
    m.intraA = reinterpret_cast<float *>(take(G * (size_t)w * 4));
    m.intraB = reinterpret_cast<float *>(take(G * (size_t)w * 4));  // min / max only
    m.ctaL = reinterpret_cast<float *>(take(grid * (size_t)w * 4));   // CTA aggregates, then their prefixes
    m.ctaR = reinterpret_cast<float *>(take(grid * (size_t)w * 4));
    m.segagg = reinterpret_cast<float *>(take(segs * (size_t)w * 4));
    m.total = (size_t)(p - static_cast<char *>(ws));
    return m;
}

size_t rbi_multiscan_workspace_bytes(int64_t n, int64_t w) {
    if (!rbi_multiscan_fits(w)) return 0;
    return ms_carve(nullptr, n, w).total;
}

template <int CODE, int WMAX, int D>
static int ms_run(float S, int64_t n, int64_t w, const int64_t *is, const float *vs, int vstride,
                  const float *hist_bar, float *vs_bar, const MsWs &m, const MsShape &s, int accumulate,
                  cudaStream_t stream) {
    const GenOp<CODE> op{S};
    const size_t smem = (size_t)w * 4 * (CODE == G_SOP ? 2 : 1) + (size_t)s.wpc * (size_t)w * 4;
    auto kf = ms_forward_kernel<CODE, WMAX, D>;
    auto kb = ms_backward_kernel<CODE, WMAX, D>;
    if (cudaFuncSetAttribute(kf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MS_SMEM_BUDGET) != cudaSuccess ||
        cudaFuncSetAttribute(kb, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MS_SMEM_BUDGET) != cudaSuccess)
        return VJP_ERR_CUDA;
    VJP_LAUNCH(K_MS_FORWARD, stream) kf<<<s.grid, s.wpc * 32, smem, stream>>>(n, w, is, vs, vstride, m.ls, m.intraA, m.intraB,
                                                                              m.ctaL, s.R, op);
    // exclusive prefix (in place) and suffix of the CTA aggregates over the CTAs
    const dim3 cg((unsigned)((w + 127) / 128), (unsigned)s.segs);
    VJP_LAUNCH(K_MS_CARRY, stream) ms_seg_agg_kernel<CODE><<<cg, 128, 0, stream>>>(w, s.grid, m.ctaL, m.segagg, op);
    VJP_LAUNCH(K_MS_CARRY, stream) ms_carry_kernel<CODE><<<cg, 128, 0, stream>>>(w, s.grid, s.segs, m.ctaL, m.ctaR, m.segagg, op);
    VJP_LAUNCH(K_MS_BACKWARD, stream) kb<<<s.grid, s.wpc * 32, smem, stream>>>(
        n, w, is, vs, vstride, m.ls, m.intraA, m.intraB, m.ctaL, m.ctaR, hist_bar, vs_bar, s.R, op, accumulate);
    return last_launch_status();
}

template <int CODE>
static int ms_dispatch(float S, int64_t n, int64_t w, const int64_t *is, const float *vs, int vstride,
                       const float *hist_bar, float *vs_bar, void *ws, int accumulate, cudaStream_t stream) {
    const MsShape s = ms_shape(n, w, CODE == G_SOP ? 2 : 1);
    const MsWs m = ms_carve(ws, n, w);
    if (s.wpc <= 16) return ms_run<CODE, 16, 8>(S, n, w, is, vs, vstride, hist_bar, vs_bar, m, s, accumulate, stream);
    return ms_run<CODE, 32, 2>(S, n, w, is, vs, vstride, hist_bar, vs_bar, m, s, accumulate, stream);
}

// gcode: G_ADD ... G_SOP (gen_ops.cuh).  vs: values (G_SOP: the pairs, the s component is read with stride 2).
int launch_rbi_multiscan_vjp(int gcode, double param, int64_t n, int64_t w, const int64_t *is, const float *vs,
                             const float *hist_bar, float *vs_bar, void *ws, int accumulate, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    if (!rbi_multiscan_fits(w)) return VJP_ERR_UNSUPPORTED;
    const float S = (float)param;
    switch (gcode) {
    case G_ADD: return ms_dispatch<G_ADD>(S, n, w, is, vs, 1, hist_bar, vs_bar, ws, accumulate, stream);
    case G_MIN: return ms_dispatch<G_MIN>(S, n, w, is, vs, 1, hist_bar, vs_bar, ws, accumulate, stream);
    case G_MAX: return ms_dispatch<G_MAX>(S, n, w, is, vs, 1, hist_bar, vs_bar, ws, accumulate, stream);
    case G_MUL: return ms_dispatch<G_MUL>(S, n, w, is, vs, 1, hist_bar, vs_bar, ws, accumulate, stream);
    case G_SATADD: return ms_dispatch<G_SATADD>(S, n, w, is, vs, 1, hist_bar, vs_bar, ws, accumulate, stream);
    case G_SOP: return ms_dispatch<G_SOP>(0.f, n, w, is, vs + 1, 2, hist_bar, vs_bar, ws, accumulate, stream);
    default: return VJP_ERR_UNSUPPORTED;
    }
}

// ------------------------------------------------------------------ histogram (primal) by the same walk

static MsShape ms_hist_shape(int64_t n, int64_t w) { return ms_shape(n < 1 ? 1 : n, w < 1 ? 1 : w, 0); }

// number of partial tables launch_ms_hist writes (= its grid)
int rbi_ms_hist_tables(int64_t n, int64_t w) { return ms_hist_shape(n, w).grid; }

template <int CODE, bool COUNT_ZEROS, bool VEC>
static int ms_hist_run(float S, int64_t n, int64_t w, const int64_t *is, const float *vs, float *part, unsigned *zeros,
                       int ld, cudaStream_t stream) {
    const MsShape s = ms_hist_shape(n, w);
    const GenOp<CODE> op{S};
    const size_t smem = (size_t)s.wpc * (size_t)w * 4;
    if (s.wpc <= 16) {
        auto k = ms_hist_kernel<CODE, 16, 8, COUNT_ZEROS, VEC>;
        if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MS_SMEM_BUDGET) != cudaSuccess) return VJP_ERR_CUDA;
        VJP_LAUNCH(K_MS_HIST, stream) k<<<s.grid, s.wpc * 32, smem, stream>>>(n, w, is, vs, part, zeros, s.R, op, ld);
    } else {
        auto k = ms_hist_kernel<CODE, 32, 2, COUNT_ZEROS, VEC>;
        if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MS_SMEM_BUDGET) != cudaSuccess) return VJP_ERR_CUDA;
        VJP_LAUNCH(K_MS_HIST, stream) k<<<s.grid, s.wpc * 32, smem, stream>>>(n, w, is, vs, part, zeros, s.R, op, ld);
    }
    return last_launch_status();
}

// part[rbi_ms_hist_tables(n, w)][w] partial histograms of '*' (mul != 0; count_zeros: the lifted form) or satadd.
// ld > 0 ('*' with zero counts only): the vectorised form, n and w flat (see ms_hist_kernel).
int launch_ms_hist(int mul, int count_zeros, float S, int64_t n, int64_t w, const int64_t *is, const float *vs,
                   float *part, unsigned *zeros, int ld, cudaStream_t stream) {
    if (ld > 0) {
        if (!mul || !count_zeros) return VJP_ERR_UNSUPPORTED;
        return ms_hist_run<G_MUL, true, true>(S, n, w, is, vs, part, zeros, ld, stream);
    }
    if (mul) {
        return count_zeros ? ms_hist_run<G_MUL, true, false>(S, n, w, is, vs, part, zeros, 0, stream)
                           : ms_hist_run<G_MUL, false, false>(S, n, w, is, vs, part, zeros, 0, stream);
    }
    return ms_hist_run<G_SATADD, false, false>(S, n, w, is, vs, part, zeros, 0, stream);
}

}  // namespace vjp
