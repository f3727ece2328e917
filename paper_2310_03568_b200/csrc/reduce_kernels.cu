// reduce_kernels.cu -- reduce (section 3 of the paper): the primal and the specialised VJP rules.
//
//   y = reduce (.) e as = a_0 (.) ... (.) a_{n-1}
//   '+'  as_bar = replicate n y_bar: one streaming fill, no primal needed.
//   min/max  lifted primal (k, y): the extremum and the SMALLEST index
//           attaining it, as a packed 64-bit key under min; return sweep as_bar = 0, as_bar[k] = y_bar.
//   '*'     (Fig. 3)  lifted primal (n^{=0}, y^{>0}); return sweep: the three-way map.
// The general rule (eq. 2, Fig. 2: two exclusive scans) lives in rbi_general.cu: it
// is the segmented-scan pair of the reduce-by-index rule with ONE segment and no sort.
//
// Every reduction is two-level: a grid of persistent CTAs leaves one partial per CTA in the workspace,
// and the CONSUMER kernel (the return sweep, or a one-CTA finish for the primal) folds the G partials
// itself in a fixed order -- deterministic, and one launch fewer than a separate final pass.
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace vjp {

constexpr int RD_NT = 512, RD_CTAS_PER_SM = 4;
constexpr int RD_MAX_PARTS = NUM_SMS_B200 * RD_CTAS_PER_SM;

enum : int { RD_ADD = 0, RD_MIN = 1, RD_MAX = 2, RD_MUL = 3, RD_SATADD = 4 };

// One partial: the running value, the zero count ('*' lifted) and the packed (value, index) key (min / max).
// The value is accumulated in f64: an n-term f32 product (or sum) drifts by about n * 3e-10 from the exact one
// in ANY association order (6e-4 at n = 2^21), which a single "bin" of 2^24 elements cannot afford against the
// 1e-4 bar; the f64 pipe is idle here and one DMUL per element costs nothing next to the HBM stream.
struct __align__(16) RedPart {
    unsigned long long key;
    double v;
    uint32_t z;
    uint32_t pad;
};

VJP_DEVINL uint32_t red_ordered(float f) {  // order-preserving image of an f32, -0 == +0 (Q6)
    const uint32_t b = __float_as_uint(f + 0.0f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
VJP_DEVINL float red_unordered(uint32_t o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}

// LIFT: the lifted primal of the VJP ('*': zeros counted and kept out of the product); else the plain primal.
template <int ACC, bool LIFT>
struct Red {
    static VJP_DEVINL RedPart neutral() {
        RedPart p;
        p.key = ~0ull;
        p.v = ACC == RD_MUL ? 1.0 : 0.0;
        p.z = 0;
        p.pad = 0;
        return p;
    }
    static VJP_DEVINL void fold(RedPart &p, float x, uint32_t idx, float S) {
        if (ACC == RD_ADD) p.v += (double)x;
        else if (ACC == RD_SATADD) p.v = fmin(p.v + (double)x, (double)S);
        else if (ACC == RD_MUL) {
            if (LIFT) {
                const bool z = x == 0.f;  // IEEE equality: +-0 only (Q7)
                p.z += z;
                p.v *= z ? 1.0 : (double)x;
            } else {
                p.v *= (double)x;
            }
        } else {
            const uint32_t o = red_ordered(x);
            const unsigned long long k = ((unsigned long long)(ACC == RD_MAX ? ~o : o) << 32) | idx;
            p.key = k < p.key ? k : p.key;
        }
    }
    static VJP_DEVINL RedPart comb(const RedPart &a, const RedPart &b, float S) {
        RedPart p;
        p.key = a.key < b.key ? a.key : b.key;
        p.z = a.z + b.z;
        p.pad = 0;
        p.v = ACC == RD_MUL ? a.v * b.v : ACC == RD_SATADD ? fmin(a.v + b.v, (double)S) : a.v + b.v;
        return p;
    }
};

template <int ACC, bool LIFT>
VJP_DEVINL RedPart red_warp(RedPart p, float S) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        RedPart o;
        o.key = __shfl_xor_sync(FULL_MASK, p.key, off);
        o.v = __shfl_xor_sync(FULL_MASK, p.v, off);
        o.z = __shfl_xor_sync(FULL_MASK, p.z, off);
        p = Red<ACC, LIFT>::comb(p, o, S);
    }
    return p;
}

// Fold of the G partials by the calling CTA (all threads call; the result is returned to every thread).
template <int ACC, bool LIFT>
VJP_DEVINL RedPart red_fold_parts(const RedPart *__restrict__ part, int G, float S) {
    __shared__ RedPart s_tot;
    if (threadIdx.x < 32) {
        RedPart p = Red<ACC, LIFT>::neutral();
        for (int g = threadIdx.x; g < G; g += 32) p = Red<ACC, LIFT>::comb(p, part[g], S);
        p = red_warp<ACC, LIFT>(p, S);
        if (threadIdx.x == 0) s_tot = p;
    }
    __syncthreads();
    return s_tot;
}

// Level 1: one partial per CTA.  zfill: xs_bar is zero-filled on the way (min / max return sweep).
template <int ACC, bool LIFT>
__global__ void __launch_bounds__(RD_NT)
reduce_partial_kernel(int64_t n, const float *__restrict__ xs, RedPart *__restrict__ part, float S,
                      float *__restrict__ zfill) {
    __shared__ RedPart s_w[RD_NT / 32];
    RedPart p = Red<ACC, LIFT>::neutral();
    const int64_t stride = (int64_t)gridDim.x * RD_NT;
    for (int64_t q = blockIdx.x * (int64_t)RD_NT + threadIdx.x; q * 4 < n; q += stride) {
        float x[4];
        const int cnt = (int)min((int64_t)4, n - q * 4);
        if (cnt == 4) {
            const uint4 a = ldg_stream(reinterpret_cast<const uint4 *>(xs) + q);
            x[0] = __uint_as_float(a.x); x[1] = __uint_as_float(a.y);
            x[2] = __uint_as_float(a.z); x[3] = __uint_as_float(a.w);
            if (zfill) stg_stream(reinterpret_cast<uint4 *>(zfill) + q, make_uint4(0u, 0u, 0u, 0u));
        } else {
#pragma unroll
            for (int j = 0; j < 4; j++) {
                x[j] = j < cnt ? xs[q * 4 + j] : 0.f;
                if (zfill && j < cnt) zfill[q * 4 + j] = 0.f;
            }
        }
#pragma unroll
        for (int j = 0; j < 4; j++)
            if (j < cnt) Red<ACC, LIFT>::fold(p, x[j], (uint32_t)(q * 4 + j), S);
    }
    p = red_warp<ACC, LIFT>(p, S);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = p;
    __syncthreads();
    if (threadIdx.x < 32) {
        p = threadIdx.x < RD_NT / 32 ? s_w[threadIdx.x] : Red<ACC, LIFT>::neutral();
        p = red_warp<ACC, LIFT>(p, S);
        if (threadIdx.x == 0) part[blockIdx.x] = p;
    }
}

template <class T>
__global__ void __launch_bounds__(RD_NT)
reduce_partial_add_f64_kernel(int64_t n, const T *__restrict__ xs, T *__restrict__ part) {
    __shared__ T s_w[RD_NT / 32];
    T acc = T(0);
    for (int64_t i = blockIdx.x * (int64_t)RD_NT + threadIdx.x; i < n; i += (int64_t)gridDim.x * RD_NT) acc += xs[i];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(FULL_MASK, acc, off);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        T t = T(0);
        for (int i = 0; i < RD_NT / 32; i++) t += s_w[i];
        part[blockIdx.x] = t;
    }
}
template <class T>
__global__ void reduce_finish_add_f64_kernel(int G, const T *__restrict__ part, T *__restrict__ y) {
    if (threadIdx.x == 0) {
        T t = T(0);
        for (int g = 0; g < G; g++) t += part[g];
        *y = t;
    }
}

// Finish kernels (one CTA): the primal's result, or the lifted primal's pair, or the min / max scatter.
template <int ACC, bool LIFT>
__global__ void __launch_bounds__(64)
reduce_finish_kernel(int64_t n, int G, const RedPart *__restrict__ part, float S, float *y,
                     int64_t *aux_i, float *aux_v, const float *__restrict__ y_bar, float *xs_bar,
                     int accumulate) {
    const RedPart t = red_fold_parts<ACC, LIFT>(part, G, S);
    if (threadIdx.x != 0) return;
    const bool minmax = ACC == RD_MIN || ACC == RD_MAX;
    const bool empty = t.key == ~0ull;
    const uint32_t o = (uint32_t)(t.key >> 32);
    const float ext = empty ? (ACC == RD_MAX ? -CUDART_INF_F : CUDART_INF_F) : red_unordered(ACC == RD_MAX ? ~o : o);
    if (y) *y = minmax ? ext : (ACC == RD_MUL && LIFT) ? (t.z ? 0.f : (float)t.v) : (float)t.v;
    if (aux_i) *aux_i = minmax ? (empty ? n : (int64_t)(uint32_t)t.key) : (int64_t)t.z;
    if (aux_v) *aux_v = minmax ? ext : (float)t.v;
    if (minmax && xs_bar && !empty) {  // as_bar[k] += y_bar
        const uint32_t k = (uint32_t)t.key;
        xs_bar[k] = accumulate ? xs_bar[k] + *y_bar : *y_bar;
    }
}

// '+': as_bar (+)= y_bar.
template <class T>
__global__ void __launch_bounds__(RD_NT)
reduce_fill_kernel(int64_t n, const T *__restrict__ y_bar, T *__restrict__ xs_bar, int accumulate) {
    const T g = *y_bar;
    constexpr int V = 16 / sizeof(T);
    const int64_t stride = (int64_t)gridDim.x * RD_NT;
    for (int64_t q = blockIdx.x * (int64_t)RD_NT + threadIdx.x; q * V < n; q += stride) {
        if (q * V + V <= n) {
            alignas(16) T o[V];
#pragma unroll
            for (int j = 0; j < V; j++) o[j] = g;
            uint4 *dst = reinterpret_cast<uint4 *>(xs_bar) + q;
            if (accumulate) {
                const uint4 pr = *dst;
                const T *pp = reinterpret_cast<const T *>(&pr);
#pragma unroll
                for (int j = 0; j < V; j++) o[j] += pp[j];
            }
            stg_stream(dst, *reinterpret_cast<const uint4 *>(o));
        } else {
            for (int64_t i = q * V; i < n; i++) xs_bar[i] = accumulate ? xs_bar[i] + g : g;
        }
    }
}

// '*' return sweep (Fig. 3): no zero -> (y / a) * y_bar; exactly one zero and a is
// that zero -> y^{>0} * y_bar; otherwise 0.
__global__ void __launch_bounds__(RD_NT)
reduce_mul_sweep_kernel(int64_t n, int G, const RedPart *__restrict__ part, const float *__restrict__ xs,
                        const float *__restrict__ y_bar, float *__restrict__ xs_bar, int accumulate) {
    const RedPart t = red_fold_parts<RD_MUL, true>(part, G, 0.f);
    const float c = (float)(t.v * (double)*y_bar);
    const uint32_t z = t.z;
    const int64_t stride = (int64_t)gridDim.x * RD_NT;
    for (int64_t q = blockIdx.x * (int64_t)RD_NT + threadIdx.x; q * 4 < n; q += stride) {
        const int cnt = (int)min((int64_t)4, n - q * 4);
        float x[4], o[4];
        if (cnt == 4) {
            const uint4 a = ldg_stream(reinterpret_cast<const uint4 *>(xs) + q);
            x[0] = __uint_as_float(a.x); x[1] = __uint_as_float(a.y);
            x[2] = __uint_as_float(a.z); x[3] = __uint_as_float(a.w);
        } else {
#pragma unroll
            for (int j = 0; j < 4; j++) x[j] = j < cnt ? xs[q * 4 + j] : 1.f;
        }
#pragma unroll
        for (int j = 0; j < 4; j++) o[j] = z == 0 ? c / x[j] : (z == 1 && x[j] == 0.f) ? c : 0.f;
        if (cnt == 4) {
            uint4 *dst = reinterpret_cast<uint4 *>(xs_bar) + q;
            if (accumulate) {
                const uint4 pr = *dst;
                o[0] += __uint_as_float(pr.x); o[1] += __uint_as_float(pr.y);
                o[2] += __uint_as_float(pr.z); o[3] += __uint_as_float(pr.w);
            }
            stg_stream(dst, make_uint4(__float_as_uint(o[0]), __float_as_uint(o[1]), __float_as_uint(o[2]),
                                       __float_as_uint(o[3])));
        } else {
            for (int j = 0; j < cnt; j++) xs_bar[q * 4 + j] = accumulate ? xs_bar[q * 4 + j] + o[j] : o[j];
        }
    }
}

// ------------------------------------------------------------------ host side ------------

static int red_grid(int64_t n, int per_thread) {
    const int64_t need = (n + (int64_t)RD_NT * per_thread - 1) / ((int64_t)RD_NT * per_thread);
    return (int)(need < 1 ? 1 : (need < RD_MAX_PARTS ? need : RD_MAX_PARTS));
}

size_t reduce_special_workspace_bytes() { return align_up((size_t)RD_MAX_PARTS * sizeof(RedPart), 256); }

template <int ACC, bool LIFT>
static int run_partial(int64_t n, const float *xs, RedPart *part, float S, float *zfill, int *G,
                       cudaStream_t stream) {
    *G = red_grid(n, 4);
    VJP_LAUNCH(K_REDUCE_PARTIAL, stream) reduce_partial_kernel<ACC, LIFT><<<*G, RD_NT, 0, stream>>>(n, xs, part, S, zfill);
    return last_launch_status();
}

template <int ACC, bool LIFT>
static int run_finish(int64_t n, int G, const RedPart *part, float S, float *y, int64_t *aux_i, float *aux_v,
                      const float *y_bar, float *xs_bar, int accumulate, cudaStream_t stream) {
    VJP_LAUNCH(K_REDUCE_FINISH, stream) reduce_finish_kernel<ACC, LIFT><<<1, 64, 0, stream>>>(
        n, G, part, S, y, aux_i, aux_v, y_bar, xs_bar, accumulate);
    return last_launch_status();
}

// Primal (lift = 0) or lifted primal (lift = 1: aux_i / aux_v of min, max, '*').  n >= 1.
int launch_reduce_forward(int code, int dtype, double param, int64_t n, const void *xs, void *y,
                          int64_t *aux_i, void *aux_v, int lift, void *ws, cudaStream_t stream) {
    const float S = (float)param;
    if (dtype == VJP_F64) {
        if (code != VJP_OP_ADD) return VJP_ERR_UNSUPPORTED;
        double *part = static_cast<double *>(ws);
        const int G = red_grid(n, 4);
        VJP_LAUNCH(K_REDUCE_PARTIAL, stream) reduce_partial_add_f64_kernel<double><<<G, RD_NT, 0, stream>>>(
            n, static_cast<const double *>(xs), part);
        VJP_LAUNCH(K_REDUCE_FINISH, stream) reduce_finish_add_f64_kernel<double><<<1, 32, 0, stream>>>(
            G, part, static_cast<double *>(y));
        return last_launch_status();
    }
    RedPart *part = static_cast<RedPart *>(ws);
    const float *x = static_cast<const float *>(xs);
    float *yy = static_cast<float *>(y), *av = static_cast<float *>(aux_v);
    int G = 0, rc;
#define RUN(ACC, LIFT)                                                                  \
    rc = run_partial<ACC, LIFT>(n, x, part, S, nullptr, &G, stream);                    \
    if (rc != VJP_OK) return rc;                                                        \
    return run_finish<ACC, LIFT>(n, G, part, S, yy, aux_i, av, nullptr, nullptr, 0, stream);
    switch (code) {
    case VJP_OP_ADD: RUN(RD_ADD, false)
    case VJP_OP_MIN: RUN(RD_MIN, false)
    case VJP_OP_MAX: RUN(RD_MAX, false)
    case VJP_OP_MUL: if (lift) { RUN(RD_MUL, true) } else { RUN(RD_MUL, false) }
    case VJP_OP_SATADD: RUN(RD_SATADD, false)
    default: return VJP_ERR_UNSUPPORTED;
    }
#undef RUN
}

// Specialised return sweeps.  n >= 1.
int launch_reduce_vjp(int code, int dtype, int64_t n, const void *xs, const void *y_bar, void *xs_bar,
                      void *ws, int accumulate, cudaStream_t stream) {
    if (code == VJP_OP_ADD) {
        const int grid = red_grid(n, 16);
        if (dtype == VJP_F32)
            VJP_LAUNCH(K_REDUCE_SWEEP, stream) reduce_fill_kernel<float><<<grid, RD_NT, 0, stream>>>(
                n, static_cast<const float *>(y_bar), static_cast<float *>(xs_bar), accumulate);
        else
            VJP_LAUNCH(K_REDUCE_SWEEP, stream) reduce_fill_kernel<double><<<grid, RD_NT, 0, stream>>>(
                n, static_cast<const double *>(y_bar), static_cast<double *>(xs_bar), accumulate);
        return last_launch_status();
    }
    if (dtype != VJP_F32) return VJP_ERR_UNSUPPORTED;
    RedPart *part = static_cast<RedPart *>(ws);
    const float *x = static_cast<const float *>(xs), *yb = static_cast<const float *>(y_bar);
    float *out = static_cast<float *>(xs_bar);
    int G = 0, rc;
    switch (code) {
    case VJP_OP_MIN:
        rc = run_partial<RD_MIN, true>(n, x, part, 0.f, accumulate ? nullptr : out, &G, stream);
        if (rc != VJP_OK) return rc;
        return run_finish<RD_MIN, true>(n, G, part, 0.f, nullptr, nullptr, nullptr, yb, out, accumulate, stream);
    case VJP_OP_MAX:
        rc = run_partial<RD_MAX, true>(n, x, part, 0.f, accumulate ? nullptr : out, &G, stream);
        if (rc != VJP_OK) return rc;
        return run_finish<RD_MAX, true>(n, G, part, 0.f, nullptr, nullptr, nullptr, yb, out, accumulate, stream);
    case VJP_OP_MUL:
        rc = run_partial<RD_MUL, true>(n, x, part, 0.f, nullptr, &G, stream);
        if (rc != VJP_OK) return rc;
        VJP_LAUNCH(K_REDUCE_SWEEP, stream) reduce_mul_sweep_kernel<<<red_grid(n, 4), RD_NT, 0, stream>>>(
            n, G, part, x, yb, out, accumulate);
        return last_launch_status();
    default: return VJP_ERR_UNSUPPORTED;
    }
}

}  // namespace vjp
