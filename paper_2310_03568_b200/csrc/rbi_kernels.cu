// rbi_kernels.cu -- reduce-by-index (generalised histogram): the primal, and the specialised
// VJP rules for '+', min/max and '*'.
//
//   primal              hist[k] = (.)_{i : is[i] = k} vs[i] over a neutral-initialised histogram;
//                       keys outside [0,w) are skipped (P:L332-336 after the rewrite of P:L338-382).
//   '+'  vs_bar[i] = hist_bar[is[i]] -- a gather, bit-exact.
//   min / max (Fig. 5)
//                       lifted primal: per bin the extremum and the LOWEST index attaining it, as one
//                       packed 64-bit key (order-preserving image of the value << 32 | index) under
//                       atomicMin; return sweep: vs_bar = 0, vs_bar[arg[k]] = hist_bar[k].
//   '*'   (Fig. 3)
//                       lifted primal: per bin the number of zeros and the product of the non-zeros;
//                       return sweep: the three-way map of Fig. 3.
//
// Histograms are privatised per CTA in shared memory ("multi-histogram"); a histogram
// that does not fit is processed in several passes over bin partitions ('*') or lives in
// global memory / L2 with a read-before-atomic filter (min/max).
#include <math_constants.h>

#include "common.cuh"
#include "internal.h"

namespace vjp {

constexpr int RBI_NT = 512;
constexpr int RBI_CTAS_PER_SM = 4;

// ------------------------------------------------------------------ element access -------

VJP_DEVINL longlong2 ldg_stream_ll2(const longlong2 *p) {
    longlong2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.s64 {%0,%1}, [%2];" : "=l"(r.x), "=l"(r.y) : "l"(p));
    return r;
}

// Elements [4q, 4q+4) of the input; `cnt` of them exist.
template <class T>
struct Quad {
    int64_t k[4];
    T v[4];
    int cnt;
};

VJP_DEVINL int load_keys4(const int64_t *__restrict__ is, int64_t i, int64_t n, int64_t (&k)[4]) {
    if (i + 4 <= n) {
        const longlong2 a = ldg_stream_ll2(reinterpret_cast<const longlong2 *>(is + i));
        const longlong2 b = ldg_stream_ll2(reinterpret_cast<const longlong2 *>(is + i) + 1);
        k[0] = a.x; k[1] = a.y; k[2] = b.x; k[3] = b.y;
        return 4;
    }
    const int cnt = (int)(n - i);
#pragma unroll
    for (int j = 0; j < 4; j++) k[j] = (j < cnt) ? is[i + j] : -1;
    return cnt;
}
VJP_DEVINL void load_vals4(const float *__restrict__ vs, int64_t i, int cnt, float (&v)[4]) {
    if (cnt == 4) {
        const uint4 a = ldg_stream(reinterpret_cast<const uint4 *>(vs + i));
        v[0] = __uint_as_float(a.x); v[1] = __uint_as_float(a.y);
        v[2] = __uint_as_float(a.z); v[3] = __uint_as_float(a.w);
    } else {
#pragma unroll
        for (int j = 0; j < 4; j++) v[j] = (j < cnt) ? vs[i + j] : 0.f;
    }
}
VJP_DEVINL void load_vals4(const double *__restrict__ vs, int64_t i, int cnt, double (&v)[4]) {
#pragma unroll
    for (int j = 0; j < 4; j++) v[j] = (j < cnt) ? vs[i + j] : 0.0;
}
VJP_DEVINL void store_vals4(float *__restrict__ out, int64_t i, int cnt, const float (&v)[4]) {
    if (cnt == 4) {
        stg_stream(reinterpret_cast<uint4 *>(out + i),
                   make_uint4(__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]),
                              __float_as_uint(v[3])));
    } else {
        for (int j = 0; j < cnt; j++) out[i + j] = v[j];
    }
}
VJP_DEVINL void store_vals4(double *__restrict__ out, int64_t i, int cnt, const double (&v)[4]) {
    for (int j = 0; j < cnt; j++) out[i + j] = v[j];
}

VJP_DEVINL bool in_range(int64_t k, int64_t w) { return (uint64_t)k < (uint64_t)w; }

static int grid_for(int64_t n, int nt, int ctas_per_sm) {
    const int64_t quads = (n + 3) / 4;
    const int64_t need = (quads + nt - 1) / nt;
    const int64_t cap = (int64_t)NUM_SMS_B200 * ctas_per_sm;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

// ------------------------------------------------------------------ value <-> ordered key -
// Order-preserving image of an f32 in u32 (IEEE total order on non-NaN values, -0 == +0: the
// paper's "<" sees them as equal, so both map to the key of +0; Q6).
VJP_DEVINL uint32_t f32_to_ordered(float f) {
    const uint32_t b = __float_as_uint(f + 0.0f);  // -0 + +0 = +0
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
VJP_DEVINL float ordered_to_f32(uint32_t o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
// min: smaller value = smaller key.  max: larger value = smaller key.  Empty bin = all ones.
template <bool IS_MAX>
VJP_DEVINL uint32_t ext_key(float f) {
    const uint32_t o = f32_to_ordered(f);
    return IS_MAX ? ~o : o;
}
template <bool IS_MAX>
VJP_DEVINL float ext_value(uint32_t key) {
    return ordered_to_f32(IS_MAX ? ~key : key);
}

// ------------------------------------------------------------------ primal ---------------

enum : int { ACC_ADD = 0, ACC_MIN = 1, ACC_MAX = 2, ACC_MUL = 3, ACC_SATADD = 4 };

// Table cell type and the atomic update of one cell, per operator.  min/max keep ordered keys.
template <int ACC, class T>
struct Cell;
template <class T>
struct Cell<ACC_ADD, T> {
    using C = T;
    static VJP_DEVINL C neutral(float) { return T(0); }
    static VJP_DEVINL C enc(T v) { return v; }
    static VJP_DEVINL void upd(C *c, C v, float) { atomicAdd(c, v); }
    static VJP_DEVINL T dec(C c) { return c; }
};
template <>
struct Cell<ACC_MIN, float> {
    using C = uint32_t;
    static VJP_DEVINL C neutral(float) { return ext_key<false>(CUDART_INF_F); }
    static VJP_DEVINL C enc(float v) { return ext_key<false>(v); }
    static VJP_DEVINL void upd(C *c, C v, float) {
        if (v < *(volatile C *)c) atomicMin(c, v);
    }
    static VJP_DEVINL float dec(C c) { return ext_value<false>(c); }
};
template <>
struct Cell<ACC_MAX, float> {
    using C = uint32_t;
    static VJP_DEVINL C neutral(float) { return ext_key<true>(-CUDART_INF_F); }
    static VJP_DEVINL C enc(float v) { return ext_key<true>(v); }
    static VJP_DEVINL void upd(C *c, C v, float) {
        if (v < *(volatile C *)c) atomicMin(c, v);
    }
    static VJP_DEVINL float dec(C c) { return ext_value<true>(c); }
};
// No hardware atomic multiply (the paper's "atomicMul-class update"): compare-and-swap.
VJP_DEVINL void atomic_mul_f32(float *c, float v) {
    unsigned *a = reinterpret_cast<unsigned *>(c);
    unsigned old = *(volatile unsigned *)a, assumed;
    do {
        assumed = old;
        old = atomicCAS(a, assumed, __float_as_uint(__uint_as_float(assumed) * v));
    } while (old != assumed);
}
template <>
struct Cell<ACC_MUL, float> {
    using C = float;
    static VJP_DEVINL C neutral(float) { return 1.f; }
    static VJP_DEVINL C enc(float v) { return v; }
    static VJP_DEVINL void upd(C *c, C v, float) { atomic_mul_f32(c, v); }
    static VJP_DEVINL float dec(C c) { return c; }
};
template <>
struct Cell<ACC_SATADD, float> {  // min(a + b, S), Q16
    using C = float;
    static VJP_DEVINL C neutral(float) { return 0.f; }
    static VJP_DEVINL C enc(float v) { return v; }
    static VJP_DEVINL void upd(C *c, C v, float S) {
        unsigned *a = reinterpret_cast<unsigned *>(c);
        unsigned old = *(volatile unsigned *)a, assumed;
        do {
            assumed = old;
            old = atomicCAS(a, assumed, __float_as_uint(fminf(__uint_as_float(assumed) + v, S)));
        } while (old != assumed);
    }
    static VJP_DEVINL float dec(C c) { return c; }
};

template <int ACC, class T>
__global__ void rbi_fill_kernel(typename Cell<ACC, T>::C *tab, int64_t w, float S) {
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w;
         k += (int64_t)gridDim.x * blockDim.x)
        tab[k] = Cell<ACC, T>::neutral(S);
}

// SMEM: per-CTA private histogram merged into `tab` at the end; else update `tab` directly.
// `tab` is the caller's hist reinterpreted as cells (same size as T), decoded in place afterwards.
template <int ACC, class T, bool SMEM>
__global__ void __launch_bounds__(RBI_NT)
rbi_forward_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const T *__restrict__ vs,
                   typename Cell<ACC, T>::C *tab, float S) {
    using CL = Cell<ACC, T>;
    using C = typename CL::C;
    extern __shared__ uint4 smem_raw[];
    C *sh = reinterpret_cast<C *>(smem_raw);
    if (SMEM) {
        for (int k = threadIdx.x; k < (int)w; k += RBI_NT) sh[k] = CL::neutral(S);
        __syncthreads();
    }
    C *dst = SMEM ? sh : tab;
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    for (int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x; q * 4 < n; q += stride) {
        int64_t k[4];
        T v[4];
        const int cnt = load_keys4(is, q * 4, n, k);
        load_vals4(vs, q * 4, cnt, v);
#pragma unroll
        for (int j = 0; j < 4; j++)
            if (in_range(k[j], w)) CL::upd(dst + k[j], CL::enc(v[j]), S);
    }
    if (SMEM) {
        __syncthreads();
        const C neutral = CL::neutral(S);
        // stagger the start so that concurrent CTAs do not walk the bins in lock step
        const int off = (int)((blockIdx.x * 97u) % (unsigned)w);
        for (int k0 = threadIdx.x; k0 < (int)w; k0 += RBI_NT) {
            int k = k0 + off;
            if (k >= (int)w) k -= (int)w;
            const C c = sh[k];
            if (c != neutral) CL::upd(tab + k, c, S);
        }
    }
}

template <int ACC, class T>
__global__ void rbi_decode_kernel(typename Cell<ACC, T>::C *tab, int64_t w) {
    using CL = Cell<ACC, T>;
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w;
         k += (int64_t)gridDim.x * blockDim.x) {
        const T v = CL::dec(tab[k]);
        reinterpret_cast<T *>(tab)[k] = v;
    }
}

constexpr size_t RBI_SMEM_TABLE_MAX = 32 * 1024;  // private histogram up to this size per CTA

template <int ACC, class T>
static int run_forward(int64_t n, int64_t w, const int64_t *is, const void *vs, void *hist,
                       float S, cudaStream_t stream) {
    using C = typename Cell<ACC, T>::C;
    static_assert(sizeof(C) == sizeof(T), "cells are decoded in place");
    C *tab = static_cast<C *>(hist);
    if (w == 0) return VJP_OK;
    const int fb = (int)((w + 255) / 256 < 1184 ? (w + 255) / 256 : 1184);
    VJP_LAUNCH(K_RBI_FILL, stream) rbi_fill_kernel<ACC, T><<<fb, 256, 0, stream>>>(tab, w, S);
    if (n > 0) {
        const int grid = grid_for(n, RBI_NT, RBI_CTAS_PER_SM);
        if ((size_t)w * sizeof(C) <= RBI_SMEM_TABLE_MAX)
            VJP_LAUNCH(K_RBI_FORWARD, stream) rbi_forward_kernel<ACC, T, true><<<grid, RBI_NT, (size_t)w * sizeof(C), stream>>>(
                n, w, is, static_cast<const T *>(vs), tab, S);
        else
            VJP_LAUNCH(K_RBI_FORWARD, stream) rbi_forward_kernel<ACC, T, false><<<grid, RBI_NT, 0, stream>>>(
                n, w, is, static_cast<const T *>(vs), tab, S);
    }
    if (ACC == ACC_MIN || ACC == ACC_MAX) VJP_LAUNCH(K_RBI_DECODE, stream) rbi_decode_kernel<ACC, T><<<fb, 256, 0, stream>>>(tab, w);
    return last_launch_status();
}

int launch_rbi_forward(int code, int dtype, double param, int64_t n, int64_t w, const int64_t *is,
                       const void *vs, void *hist, void *, cudaStream_t stream) {
    const float S = (float)param;
    if (dtype == VJP_F64) {
        if (code == VJP_OP_ADD) return run_forward<ACC_ADD, double>(n, w, is, vs, hist, S, stream);
        return VJP_ERR_UNSUPPORTED;
    }
    switch (code) {
    case VJP_OP_ADD: return run_forward<ACC_ADD, float>(n, w, is, vs, hist, S, stream);
    case VJP_OP_MIN: return run_forward<ACC_MIN, float>(n, w, is, vs, hist, S, stream);
    case VJP_OP_MAX: return run_forward<ACC_MAX, float>(n, w, is, vs, hist, S, stream);
    case VJP_OP_MUL: return run_forward<ACC_MUL, float>(n, w, is, vs, hist, S, stream);
    case VJP_OP_SATADD: return run_forward<ACC_SATADD, float>(n, w, is, vs, hist, S, stream);
    default: return VJP_ERR_UNSUPPORTED;
    }
}

// ------------------------------------------------------------------ '+' VJP: gather -------

constexpr size_t GATHER_SMEM_MAX = 64 * 1024;

template <class T, bool SMEM>
__global__ void __launch_bounds__(RBI_NT)
rbi_vjp_add_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                   const T *__restrict__ hist_bar, T *__restrict__ vs_bar) {
    extern __shared__ uint4 smem_raw[];
    T *sh = reinterpret_cast<T *>(smem_raw);
    if (SMEM) {
        for (int k = threadIdx.x; k < (int)w; k += RBI_NT) sh[k] = hist_bar[k];
        __syncthreads();
    }
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    for (int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x; q * 4 < n; q += stride) {
        int64_t k[4];
        T o[4];
        const int cnt = load_keys4(is, q * 4, n, k);
#pragma unroll
        for (int j = 0; j < 4; j++)
            o[j] = in_range(k[j], w) ? (SMEM ? sh[k[j]] : __ldg(hist_bar + k[j])) : T(0);
        store_vals4(vs_bar, q * 4, cnt, o);
    }
}

template <class T>
static int run_vjp_add(int64_t n, int64_t w, const int64_t *is, const void *hist_bar, void *vs_bar,
                       cudaStream_t stream) {
    const int grid = grid_for(n, RBI_NT, RBI_CTAS_PER_SM);
    const size_t bytes = (size_t)w * sizeof(T);
    if (bytes <= GATHER_SMEM_MAX / 2) {
        VJP_LAUNCH(K_RBI_GATHER, stream) rbi_vjp_add_kernel<T, true><<<grid, RBI_NT, bytes, stream>>>(
            n, w, is, static_cast<const T *>(hist_bar), static_cast<T *>(vs_bar));
    } else {
        VJP_LAUNCH(K_RBI_GATHER, stream) rbi_vjp_add_kernel<T, false><<<grid, RBI_NT, 0, stream>>>(
            n, w, is, static_cast<const T *>(hist_bar), static_cast<T *>(vs_bar));
    }
    return last_launch_status();
}

int launch_rbi_vjp_add(int dtype, int64_t n, int64_t w, const int64_t *is, const void *hist_bar,
                       void *vs_bar, cudaStream_t stream) {
    return dtype == VJP_F32 ? run_vjp_add<float>(n, w, is, hist_bar, vs_bar, stream)
                            : run_vjp_add<double>(n, w, is, hist_bar, vs_bar, stream);
}

// ------------------------------------------------------------------ min / max VJP ---------

constexpr unsigned long long EMPTY_KEY = ~0ull;

// Lifted primal min^L on (index, value) (Fig. 5) as an atomicMin over packed keys.
// Almost every element loses against the bin's current key, so the key is read first and the
// atomic is issued only by a candidate (the histogram then costs one shared / L2 read per
// element instead of one atomic).
template <bool IS_MAX, bool SMEM>
__global__ void __launch_bounds__(RBI_NT)
rbi_minmax_lifted_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                         const float *__restrict__ vs, unsigned long long *tab,
                         float *__restrict__ vs_bar /* zero-filled here if not NULL */) {
    extern __shared__ uint4 smem_raw[];
    unsigned long long *sh = reinterpret_cast<unsigned long long *>(smem_raw);
    if (SMEM) {
        for (int k = threadIdx.x; k < (int)w; k += RBI_NT) sh[k] = EMPTY_KEY;
        __syncthreads();
    }
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    for (int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x; q * 4 < n; q += stride) {
        int64_t k[4];
        float v[4];
        const int cnt = load_keys4(is, q * 4, n, k);
        load_vals4(vs, q * 4, cnt, v);
        if (vs_bar) {
            const float z[4] = {0.f, 0.f, 0.f, 0.f};
            store_vals4(vs_bar, q * 4, cnt, z);
        }
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if (!in_range(k[j], w)) continue;
            const unsigned long long key =
                ((unsigned long long)ext_key<IS_MAX>(v[j]) << 32) | (unsigned)(q * 4 + j);
            if (SMEM) {
                if (key < *(volatile unsigned long long *)(sh + k[j])) atomicMin(sh + k[j], key);
            } else {
                if (key < __ldcg(tab + k[j])) atomicMin(tab + k[j], key);
            }
        }
    }
    if (SMEM) {
        __syncthreads();
        const int off = (int)((blockIdx.x * 97u) % (unsigned)w);
        for (int k0 = threadIdx.x; k0 < (int)w; k0 += RBI_NT) {
            int k = k0 + off;
            if (k >= (int)w) k -= (int)w;
            const unsigned long long key = sh[k];
            if (key != EMPTY_KEY && key < __ldcg(tab + k)) atomicMin(tab + k, key);
        }
    }
}

// arg / ext of every bin (an empty bin is (n, +-inf)) and the scatter of the return sweep
// (P:L438-441).  vs_bar has been zeroed before.
template <bool IS_MAX>
__global__ void rbi_minmax_finish_kernel(int64_t n, int64_t w, const unsigned long long *tab,
                                         const float *__restrict__ hist_bar, float *vs_bar,
                                         int64_t *arg, float *ext) {
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w;
         k += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long key = tab[k];
        const bool empty = key == EMPTY_KEY;
        const int64_t idx = empty ? n : (int64_t)(unsigned)key;
        if (arg) arg[k] = idx;
        if (ext)
            ext[k] = empty ? (IS_MAX ? -CUDART_INF_F : CUDART_INF_F)
                           : ext_value<IS_MAX>((uint32_t)(key >> 32));
        if (vs_bar && !empty) vs_bar[idx] = hist_bar[k];
    }
}

constexpr size_t MINMAX_SMEM_MAX = 64 * 1024;

template <bool IS_MAX>
static int run_minmax(int64_t n, int64_t w, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar, int64_t *arg, float *ext, void *ws,
                      cudaStream_t stream) {
    unsigned long long *tab = static_cast<unsigned long long *>(ws);
    if (w == 0) {  // no bins: every adjoint is 0
        if (vs_bar && n > 0 &&
            cudaMemsetAsync(vs_bar, 0, (size_t)n * sizeof(float), stream) != cudaSuccess)
            return VJP_ERR_CUDA;
        return VJP_OK;
    }
    if (cudaMemsetAsync(tab, 0xff, (size_t)w * 8, stream) != cudaSuccess) return VJP_ERR_CUDA;
    if (n > 0) {
        const size_t bytes = (size_t)w * 8;
        if (bytes <= MINMAX_SMEM_MAX) {
            auto kern = rbi_minmax_lifted_kernel<IS_MAX, true>;
            if (bytes > 48 * 1024 &&
                cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)MINMAX_SMEM_MAX) != cudaSuccess)
                return VJP_ERR_CUDA;
            const int per_sm = bytes <= 16 * 1024 ? RBI_CTAS_PER_SM : (bytes <= 32 * 1024 ? 3 : 2);
            VJP_LAUNCH(K_MINMAX_LIFTED, stream) kern<<<grid_for(n, RBI_NT, per_sm), RBI_NT, bytes, stream>>>(n, w, is, vs, tab, vs_bar);
        } else {
            VJP_LAUNCH(K_MINMAX_LIFTED, stream) rbi_minmax_lifted_kernel<IS_MAX, false>
                <<<grid_for(n, RBI_NT, RBI_CTAS_PER_SM), RBI_NT, 0, stream>>>(n, w, is, vs, tab, vs_bar);
        }
    }
    const int fb = (int)((w + 255) / 256 < 1184 ? (w + 255) / 256 : 1184);
    VJP_LAUNCH(K_MINMAX_FINISH, stream) rbi_minmax_finish_kernel<IS_MAX><<<fb, 256, 0, stream>>>(n, w, tab, hist_bar, vs_bar, arg, ext);
    return last_launch_status();
}

int launch_rbi_minmax(int code, int64_t n, int64_t w, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar, int64_t *arg, float *ext, void *ws,
                      cudaStream_t stream) {
    return code == VJP_OP_MAX ? run_minmax<true>(n, w, is, vs, hist_bar, vs_bar, arg, ext, ws, stream)
                              : run_minmax<false>(n, w, is, vs, hist_bar, vs_bar, arg, ext, ws, stream);
}

// ------------------------------------------------------------------ '*' VJP ---------------
//
// Lifted primal: per bin (zero count, product of the non-zeros).  Each CTA owns a private
// table of products in shared memory covering a partition of at most MUL_PART bins; a histogram
// larger than that takes several passes over the input.  CTA g writes its table to
// part[g][.]; a second kernel folds the G tables per bin in a fixed order.  Zeros are rare events
// counted with integer atomics in global memory (exact, Q8).

constexpr int MUL_NT = 1024;
constexpr int MUL_PART = 48 * 1024;  // bins per pass (192 KB of f32 products)

__global__ void __launch_bounds__(MUL_NT)
rbi_mul_lifted_kernel(int64_t n, int64_t w, int part_bins, const int64_t *__restrict__ is,
                      const float *__restrict__ vs, float *__restrict__ part, unsigned *zeros) {
    extern __shared__ uint4 smem_raw[];
    float *sh = reinterpret_cast<float *>(smem_raw);
    const int64_t stride = (int64_t)gridDim.x * MUL_NT;
    for (int64_t lo = 0; lo < w; lo += part_bins) {
        const int nb = (int)min((int64_t)part_bins, w - lo);
        for (int k = threadIdx.x; k < nb; k += MUL_NT) sh[k] = 1.f;
        __syncthreads();
        for (int64_t q = blockIdx.x * (int64_t)MUL_NT + threadIdx.x; q * 4 < n; q += stride) {
            int64_t k[4];
            float v[4];
            const int cnt = load_keys4(is, q * 4, n, k);
            load_vals4(vs, q * 4, cnt, v);
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int64_t b = k[j] - lo;
                if ((uint64_t)b >= (uint64_t)nb) continue;  // other partition, or out of range
                if (v[j] == 0.f) atomicAdd(zeros + k[j], 1u);  // IEEE equality: +-0 only (Q7)
                else atomic_mul_f32(sh + b, v[j]);
            }
        }
        __syncthreads();
        float *dst = part + (size_t)blockIdx.x * (size_t)w + lo;
        for (int k = threadIdx.x; k < nb; k += MUL_NT) dst[k] = sh[k];
        __syncthreads();
    }
}

// Per bin: fold the G partial products (fixed order: deterministic), expose (zeros, prod_nz), and
// prepare the return sweep's coefficient c_k = prod_nz_k * hist_bar_k with the zero count clamped
// to {0, 1, 2}.
__global__ void rbi_mul_finish_kernel(int64_t w, int G, const float *__restrict__ part,
                                      const unsigned *__restrict__ zeros_u,
                                      const float *__restrict__ hist_bar, int64_t *zeros,
                                      float *prod_nz, float2 *coef) {
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w;
         k += (int64_t)gridDim.x * blockDim.x) {
        float p = 1.f;
        for (int g = 0; g < G; g++) p *= part[(size_t)g * (size_t)w + k];
        const unsigned z = zeros_u[k];
        if (zeros) zeros[k] = (int64_t)z;
        if (prod_nz) prod_nz[k] = p;
        if (coef) coef[k] = make_float2(p * hist_bar[k], __int_as_float((int)(z < 2u ? z : 2u)));
    }
}

// Return sweep (Fig. 3): no zero in the bin -> (y / a) * ybar; exactly one
// zero and a is that zero -> y^{>0} * ybar; otherwise 0.  Out-of-range keys get 0.
template <bool SMEM>
__global__ void __launch_bounds__(RBI_NT)
rbi_mul_sweep_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                     const float *__restrict__ vs, const float2 *__restrict__ coef,
                     float *__restrict__ vs_bar) {
    extern __shared__ uint4 smem_raw[];
    float2 *sh = reinterpret_cast<float2 *>(smem_raw);
    if (SMEM) {
        for (int k = threadIdx.x; k < (int)w; k += RBI_NT) sh[k] = coef[k];
        __syncthreads();
    }
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    for (int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x; q * 4 < n; q += stride) {
        int64_t k[4];
        float v[4], o[4];
        const int cnt = load_keys4(is, q * 4, n, k);
        load_vals4(vs, q * 4, cnt, v);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            o[j] = 0.f;
            if (!in_range(k[j], w)) continue;
            const float2 c = SMEM ? sh[k[j]] : __ldg(coef + k[j]);
            const int z = __float_as_int(c.y);
            if (z == 0) o[j] = c.x / v[j];
            else if (z == 1 && v[j] == 0.f) o[j] = c.x;
        }
        store_vals4(vs_bar, q * 4, cnt, o);
    }
}

static int mul_grid(int64_t n, int64_t w, int *part_bins, size_t *smem) {
    *part_bins = (int)(w < MUL_PART ? (w < 1 ? 1 : w) : MUL_PART);
    *smem = (size_t)*part_bins * sizeof(float);
    int per_sm = 1;
    if (*smem <= 24 * 1024) per_sm = 2;  // 2 x 1024 threads fill an SM
    return grid_for(n, MUL_NT, per_sm);
}

struct MulWs {
    unsigned *zeros;
    float2 *coef;
    float *part;
};
static MulWs mul_carve(void *ws, int64_t w) {
    MulWs m;
    char *p = static_cast<char *>(ws);
    m.zeros = reinterpret_cast<unsigned *>(p);
    p += align_up((size_t)w * 4, 256);
    m.coef = reinterpret_cast<float2 *>(p);
    p += align_up((size_t)w * 8, 256);
    m.part = reinterpret_cast<float *>(p);
    return m;
}

int launch_rbi_mul(int64_t n, int64_t w, const int64_t *is, const float *vs,
                   const float *hist_bar, float *vs_bar, int64_t *zeros, float *prod_nz, void *ws,
                   cudaStream_t stream) {
    if (w == 0) {
        if (vs_bar && n > 0 &&
            cudaMemsetAsync(vs_bar, 0, (size_t)n * sizeof(float), stream) != cudaSuccess)
            return VJP_ERR_CUDA;
        return VJP_OK;
    }
    MulWs m = mul_carve(ws, w);
    int part_bins;
    size_t smem;
    const int G = mul_grid(n, w, &part_bins, &smem);
    if (cudaMemsetAsync(m.zeros, 0, (size_t)w * 4, stream) != cudaSuccess) return VJP_ERR_CUDA;
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(rbi_mul_lifted_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(MUL_PART * sizeof(float))) != cudaSuccess)
        return VJP_ERR_CUDA;
    VJP_LAUNCH(K_MUL_LIFTED, stream) rbi_mul_lifted_kernel<<<G, MUL_NT, smem, stream>>>(n, w, part_bins, is, vs, m.part, m.zeros);
    const int fb = (int)((w + 255) / 256 < 1184 ? (w + 255) / 256 : 1184);
    VJP_LAUNCH(K_MUL_FINISH, stream) rbi_mul_finish_kernel<<<fb, 256, 0, stream>>>(w, G, m.part, m.zeros, hist_bar, zeros, prod_nz,
                                                  vs_bar ? m.coef : nullptr);
    if (vs_bar && n > 0) {
        const int grid = grid_for(n, RBI_NT, RBI_CTAS_PER_SM);
        const size_t bytes = (size_t)w * sizeof(float2);
        if (bytes <= GATHER_SMEM_MAX / 2)
            VJP_LAUNCH(K_MUL_SWEEP, stream) rbi_mul_sweep_kernel<true><<<grid, RBI_NT, bytes, stream>>>(n, w, is, vs, m.coef, vs_bar);
        else
            VJP_LAUNCH(K_MUL_SWEEP, stream) rbi_mul_sweep_kernel<false><<<grid, RBI_NT, 0, stream>>>(n, w, is, vs, m.coef, vs_bar);
    }
    return last_launch_status();
}

size_t rbi_special_workspace_bytes(int code, int, int64_t n, int64_t w) {
    if (w < 1) w = 1;
    switch (code) {
    case VJP_OP_MIN:
    case VJP_OP_MAX: return align_up((size_t)w * 8, 256);
    case VJP_OP_MUL: {
        int part_bins;
        size_t smem;
        const int G = mul_grid(n < 1 ? 1 : n, w, &part_bins, &smem);
        return align_up((size_t)w * 4, 256) + align_up((size_t)w * 8, 256) +
               align_up((size_t)G * (size_t)w * 4, 256);
    }
    default: return 256;
    }
}

}  // namespace vjp
