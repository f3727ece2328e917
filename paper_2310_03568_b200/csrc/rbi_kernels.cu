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
#include <cooperative_groups.h>
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

// vs_bar[i..i+cnt) = (acc ? vs_bar : 0) + v: the "+=" of an accumulating call fused into the store
template <class T>
VJP_DEVINL void store_adj4(T *__restrict__ out, int64_t i, int cnt, T (&v)[4], bool acc) {
    if (acc) {
        T p[4];
        load_vals4(out, i, cnt, p);
#pragma unroll
        for (int j = 0; j < 4; j++) v[j] += p[j];
    }
    store_vals4(out, i, cnt, v);
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

constexpr size_t RBI_SMEM_TABLE_MAX = 32 * 1024;  // private histogram up to this size per CTA

template <int ACC, class T>
static int run_forward(int64_t n, int64_t w, const int64_t *is, const void *vs, void *hist,
                       float S, cudaStream_t stream) {
    using C = typename Cell<ACC, T>::C;
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
    return last_launch_status();
}

// '*' and satadd have no hardware atomic: cached accumulation (defined further down)
static int launch_cached_primal(int code, int64_t n, int64_t w, const int64_t *is, const float *vs,
                                float *hist, void *ws, float S, cudaStream_t stream);

int launch_rbi_forward(int code, int dtype, double param, int64_t n, int64_t w, const int64_t *is,
                       const void *vs, void *hist, void *ws, cudaStream_t stream) {
    const float S = (float)param;
    if (dtype == VJP_F64) {
        if (code == VJP_OP_ADD) return run_forward<ACC_ADD, double>(n, w, is, vs, hist, S, stream);
        return VJP_ERR_UNSUPPORTED;
    }
    switch (code) {
    case VJP_OP_ADD: return run_forward<ACC_ADD, float>(n, w, is, vs, hist, S, stream);
    case VJP_OP_MIN:  // the packed-key kernels of the lifted operator, value part only
    case VJP_OP_MAX:
        return launch_rbi_minmax(code, n, w, is, static_cast<const float *>(vs), nullptr, nullptr, nullptr,
                                 static_cast<float *>(hist), ws, 0, stream);
    case VJP_OP_MUL:
    case VJP_OP_SATADD:
        return launch_cached_primal(code, n, w, is, static_cast<const float *>(vs),
                                    static_cast<float *>(hist), ws, S, stream);
    default: return VJP_ERR_UNSUPPORTED;
    }
}

// ------------------------------------------------------------------ '+' VJP: gather -------

constexpr size_t GATHER_SMEM_MAX = 64 * 1024;

template <class T, bool SMEM>
__global__ void __launch_bounds__(RBI_NT)
rbi_vjp_add_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                   const T *__restrict__ hist_bar, T *__restrict__ vs_bar, int accumulate) {
    extern __shared__ uint4 smem_raw[];
    T *sh = reinterpret_cast<T *>(smem_raw);
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x;
    // the keys of the thread's first quad are in flight while the table is staged (config 1 is one quad per thread: its
    // two dependent round trips become one; prefetching every next quad too cost the n = 2^26 case 4 %)
    int64_t k[4] = {-1, -1, -1, -1};
    int cnt = 0;
    if (q * 4 < n) cnt = load_keys4(is, q * 4, n, k);
    if (SMEM) {
        for (int i = threadIdx.x; i < (int)w; i += RBI_NT) sh[i] = hist_bar[i];
        __syncthreads();
    }
    for (bool first = true; q * 4 < n; q += stride, first = false) {
        if (!first) cnt = load_keys4(is, q * 4, n, k);
        T o[4];
#pragma unroll
        for (int j = 0; j < 4; j++)
            o[j] = in_range(k[j], w) ? (SMEM ? sh[k[j]] : __ldg(hist_bar + k[j])) : T(0);
        store_adj4(vs_bar, q * 4, cnt, o, accumulate != 0);
    }
}

template <class T>
static int run_vjp_add(int64_t n, int64_t w, const int64_t *is, const void *hist_bar, void *vs_bar,
                       int accumulate, cudaStream_t stream) {
    const int grid = grid_for(n, RBI_NT, RBI_CTAS_PER_SM);
    const size_t bytes = (size_t)w * sizeof(T);
    if (bytes <= GATHER_SMEM_MAX / 2) {
        VJP_LAUNCH(K_RBI_GATHER, stream) rbi_vjp_add_kernel<T, true><<<grid, RBI_NT, bytes, stream>>>(
            n, w, is, static_cast<const T *>(hist_bar), static_cast<T *>(vs_bar), accumulate);
    } else {
        VJP_LAUNCH(K_RBI_GATHER, stream) rbi_vjp_add_kernel<T, false><<<grid, RBI_NT, 0, stream>>>(
            n, w, is, static_cast<const T *>(hist_bar), static_cast<T *>(vs_bar), accumulate);
    }
    return last_launch_status();
}

int launch_rbi_vjp_add(int dtype, int64_t n, int64_t w, const int64_t *is, const void *hist_bar,
                       void *vs_bar, int accumulate, cudaStream_t stream) {
    return dtype == VJP_F32 ? run_vjp_add<float>(n, w, is, hist_bar, vs_bar, accumulate, stream)
                            : run_vjp_add<double>(n, w, is, hist_bar, vs_bar, accumulate, stream);
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
        if (vs_bar && cnt > 0) {
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

// Histograms too large for a private shared-memory copy (w > 8192): the packed keys live in global
// memory (L2) and every CTA keeps a FILTER in shared memory: per slot the top 16 bits of the best
// (ordered) value key this CTA has seen for the slot's bin.  A bin's minimum only ever decreases, so
// any value once observed is an upper bound of the current one, and an element whose 16-bit prefix
// is strictly above the filter cannot win: it is dropped without touching L2.  Racing plain stores
// can only leave a weaker (larger) bound behind.  Without the filter every element of a hot bin
// reads the same L2 sector, which a single L2 slice serialises (profiles/r1a: 0.9 ms at Zipf keys).
// TAGGED = false: w <= 65536, slot = bin, 2-byte entries.  TAGGED = true: 32768 slots of
// (bin >> 15) << 16 | prefix; a slot that holds another bin does not filter.
constexpr int MMF_NT = 1024;
constexpr int MMF_REFRESH_AT = 3;  // iterations of a CTA before its filter is refreshed from the table (1: 0.094, 3: 0.088, 1+4: 0.091 ms)
constexpr size_t MMF_FILTER = 128 * 1024;          // the filter
constexpr int MMF_SEED = 4;                        // elements of a thread's first quad that take part (1: Zipf +4 us, uniform -2 us)
constexpr int MMF_SIDE = 4096;                     // + a side table of 32-bit slots (first-batch election)
constexpr size_t MMF_SMEM = MMF_FILTER + MMF_SIDE * 4;

template <bool IS_MAX, bool TAGGED>
__global__ void __launch_bounds__(MMF_NT, 1)
rbi_minmax_filtered_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                           const float *__restrict__ vs, unsigned long long *tab,
                           float *__restrict__ vs_bar) {
    extern __shared__ uint4 smem_raw[];
    uint16_t *f16 = reinterpret_cast<uint16_t *>(smem_raw);  // [65536]
    uint32_t *f32 = reinterpret_cast<uint32_t *>(smem_raw);  // [32768]
    const int64_t stride = (int64_t)gridDim.x * MMF_NT;
    int64_t q = blockIdx.x * (int64_t)MMF_NT + threadIdx.x;
    int64_t k[4] = {-1, -1, -1, -1};
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    int cnt = 0;
    if (q * 4 < n) {  // the first loads fly while the filter is initialised
        cnt = load_keys4(is, q * 4, n, k);
        load_vals4(vs, q * 4, cnt, v);
    }
    for (int i = threadIdx.x; i < (int)(MMF_SMEM / 16); i += MMF_NT) smem_raw[i] = make_uint4(~0u, ~0u, ~0u, ~0u);
    __syncthreads();
    if (!TAGGED) {
        // Hot bins.  With an open filter every warp's first element of a hot bin (Zipf keys: 14 % of the elements in
        // one bin) queues at the bin's one L2 sector, for its read and for its atomic: two contended round trips in
        // which 35 % of the Zipf case's stall samples sat (profiles/r2e).  The CTA's first batch therefore elects, per
        // bin, its smallest 16-bit prefix in shared memory first (one 32-bit atomicMin on a direct-mapped side table of
        // (prefix, bin tag) words; bins that share a slot: the smaller prefix keeps it, the other bin just goes
        // unseeded) and seeds the filter with it: only the holders of that prefix go to L2 at all.
        uint32_t *side = reinterpret_cast<uint32_t *>(smem_raw) + MMF_FILTER / 4;
#pragma unroll
        for (int j = 0; j < MMF_SEED; j++)
            if (in_range(k[j], w))
                atomicMin(side + (k[j] & (MMF_SIDE - 1)), ((ext_key<IS_MAX>(v[j]) >> 16) << 16) | (uint32_t)(k[j] >> 12));
        __syncthreads();
#pragma unroll
        for (int j = 0; j < MMF_SEED; j++) {
            if (!in_range(k[j], w)) continue;
            const uint32_t e = side[k[j] & (MMF_SIDE - 1)];
            if ((e & 0xffffu) == (uint32_t)(k[j] >> 12)) f16[k[j]] = (uint16_t)(e >> 16);  // every writer stores the same value
        }
        __syncwarp();  // no CTA barrier: a warp that runs ahead of another one's seeds only meets an open filter
    }
    // A CTA sees only n / (148 w) elements of a bin (1.7 at w = 2^16): on its own its filter learns a bound per bin
    // once and never profits from it.  After MMF_REFRESH_AT of its iterations (~1/9 of the input, ~28 elements per
    // bin seen by the grid as a whole) it therefore takes the bounds of ALL CTAs from the table, with coalesced
    // loads: any value the table has held is an upper bound of the bin's minimum, so the filter stays valid whatever
    // races with the per-element updates below, and from then on ~3 % of the elements reach L2 instead of ~60 %.
    const int64_t total_it = (n / 4 + stride - 1) / stride;
    int64_t it = 0;
    // The loop is WARP-uniform: a lane whose quads are used up goes on with an empty quad (keys -1: out of range,
    // nothing loaded, nothing stored) until its warp is done.
    while (__any_sync(FULL_MASK, q * 4 < n)) {
        if (!TAGGED && it == MMF_REFRESH_AT && total_it >= 2 * MMF_REFRESH_AT) {
            for (int b = threadIdx.x; b < (int)w; b += MMF_NT) {
                const uint32_t g16 = (uint32_t)(__ldcg(tab + b) >> 48);
                if (g16 < f16[b]) f16[b] = (uint16_t)g16;
            }
        }
        it++;
        // next iteration's loads fly while this one walks the table (its L2 round trips are dependent)
        int64_t kn[4] = {-1, -1, -1, -1};
        float vn[4] = {0.f, 0.f, 0.f, 0.f};
        int cntn = 0;
        const int64_t qn = q + stride;
        if (qn * 4 < n) {
            cntn = load_keys4(is, qn * 4, n, kn);
            load_vals4(vs, qn * 4, cntn, vn);
        }
        if (vs_bar && cnt > 0) {
            const float z[4] = {0.f, 0.f, 0.f, 0.f};
            store_vals4(vs_bar, q * 4, cnt, z);
        }
        if (TAGGED) {
        // Histograms wider than 2^16 bins (tagged filter): one element at a time (filter, table read, update), so that a
        // hot bin's elements meet a fresh bound -- with an open filter every element of a hot bin would otherwise send
        // its own atomic to the one L2 sector (Zipf keys: 14 % of the elements).
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if (!in_range(k[j], w)) continue;
            const uint32_t vk = ext_key<IS_MAX>(v[j]);
            const uint32_t p16 = vk >> 16;
            const uint32_t b = (uint32_t)k[j];
            const bool wide = TAGGED && (b >> 31);  // the 16-bit tag cannot name bins >= 2^31: never filtered
            if (TAGGED) {
                const uint32_t e = f32[b & 32767u];
                if (!wide && (e >> 16) == (b >> 15) && p16 > (e & 0xffffu)) continue;
            } else {
                if (p16 > f16[b]) continue;
            }
            const unsigned long long key = ((unsigned long long)vk << 32) | (unsigned)(q * 4 + j);
            unsigned long long cur = __ldcg(tab + k[j]);
            if (key < cur) {
                cur = atomicMin(tab + k[j], key);
                if (key < cur) cur = key;
            }
            const uint32_t c16 = (uint32_t)(cur >> 48);
            if (TAGGED) {
                if (!wide) f32[b & 32767u] = ((b >> 15) << 16) | c16;
            } else {
                f16[b] = (uint16_t)c16;
            }
        }
        } else if (it == 1) {
        // The CTA's first iteration: one element at a time (filter, table read, atomic with its result, filter update).
        // The hot bins were seeded above; everything else meets a fresh table, and batching the quad here -- as the
        // later iterations do -- measured 8 us slower at uniform keys.
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if (!in_range(k[j], w)) continue;
            const uint32_t vk = ext_key<IS_MAX>(v[j]);
            const uint32_t b = (uint32_t)k[j];
            if ((vk >> 16) > f16[b]) continue;
            const unsigned long long key = ((unsigned long long)vk << 32) | (unsigned)(q * 4 + j);
            unsigned long long cur = __ldcg(tab + k[j]);
            if (key < cur) {
                cur = atomicMin(tab + k[j], key);
                if (key < cur) cur = key;
            }
            f16[b] = (uint16_t)(cur >> 48);
        }
        } else {
        // Later iterations (the filter knows every bin that is hot): the quad's table reads are issued TOGETHER and its
        // atomics are not waited for one by one -- four dependent L2 round trips per quad were the kernel's whole
        // duration (28 iterations x 4 x ~1 us; 71 % of the stall samples on the two L2 waits, profiles/r2e).  A
        // thread's own duplicates of a bin are resolved in registers first (only the smallest key goes on).
        unsigned long long cur[4];
        uint32_t b[4], vk[4];
        bool pass[4];
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const bool inr = in_range(k[j], w);
            b[j] = inr ? (uint32_t)k[j] : 0u;
            vk[j] = ext_key<IS_MAX>(v[j]);
            pass[j] = inr && !((vk[j] >> 16) > f16[b[j]]);
        }
#pragma unroll
        for (int j = 1; j < 4; j++)
#pragma unroll
            for (int i = 0; i < j; i++)
                if (pass[i] && pass[j] && b[i] == b[j]) {  // i < j: on equal values the lower index stays
                    if (vk[i] <= vk[j]) pass[j] = false;
                    else pass[i] = false;
                }
#pragma unroll
        for (int j = 0; j < 4; j++) {
            if (pass[j]) f16[b[j]] = (uint16_t)(vk[j] >> 16);  // the candidate's own prefix is a valid bound at once
            cur[j] = pass[j] ? __ldcg(tab + b[j]) : 0ull;
        }
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const unsigned long long key = ((unsigned long long)vk[j] << 32) | (unsigned)(q * 4 + j);
            if (pass[j] && key < cur[j]) {
                atomicMin(tab + b[j], key);  // result unused: a fire-and-forget RED, no third round trip
                cur[j] = key;                // the table now holds key or less: a valid bound for the filter
            }
        }
#pragma unroll
        for (int j = 0; j < 4; j++)
            if (pass[j]) f16[b[j]] = (uint16_t)(cur[j] >> 48);
        }
#pragma unroll
        for (int j = 0; j < 4; j++) {
            k[j] = kn[j];
            v[j] = vn[j];
        }
        cnt = cntn;
        q = qn;
    }
}

// arg / ext of every bin (an empty bin is (n, +-inf)) and the scatter of the return sweep
// (P:L438-441).  vs_bar has been zeroed before.
template <bool IS_MAX>
__global__ void rbi_minmax_finish_kernel(int64_t n, int64_t w, const unsigned long long *tab,
                                         const float *__restrict__ hist_bar, float *vs_bar,
                                         int64_t *arg, float *ext, int accumulate) {
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w;
         k += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long key = tab[k];
        const bool empty = key == EMPTY_KEY;
        const int64_t idx = empty ? n : (int64_t)(unsigned)key;
        if (arg) arg[k] = idx;
        if (ext)
            ext[k] = empty ? (IS_MAX ? -CUDART_INF_F : CUDART_INF_F)
                           : ext_value<IS_MAX>((uint32_t)(key >> 32));
        if (vs_bar && !empty) vs_bar[idx] = accumulate ? vs_bar[idx] + hist_bar[k] : hist_bar[k];  // one bin per index
    }
}

constexpr size_t MINMAX_SMEM_MAX = 64 * 1024;
static size_t minmax_ws_bytes(int64_t w) { return align_up((size_t)w * 8, 256); }  // packed keys [w]

template <bool IS_MAX>
static int run_minmax(int64_t n, int64_t w, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar_out, int64_t *arg, float *ext, void *ws,
                      int accumulate, cudaStream_t stream) {
    unsigned long long *tab = static_cast<unsigned long long *>(ws);
    // accumulate: the lifted pass does not zero-fill vs_bar, the finish kernel adds instead of storing
    float *vs_bar = accumulate ? nullptr : vs_bar_out;
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
        } else if (w <= 65536) {
            auto kern = rbi_minmax_filtered_kernel<IS_MAX, false>;
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MMF_SMEM) != cudaSuccess)
                return VJP_ERR_CUDA;
            VJP_LAUNCH(K_MINMAX_LIFTED, stream) kern<<<grid_for(n, MMF_NT, 1), MMF_NT, MMF_SMEM, stream>>>(n, w, is, vs, tab, vs_bar);
        } else {
            auto kern = rbi_minmax_filtered_kernel<IS_MAX, true>;
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MMF_SMEM) != cudaSuccess)
                return VJP_ERR_CUDA;
            VJP_LAUNCH(K_MINMAX_LIFTED, stream) kern<<<grid_for(n, MMF_NT, 1), MMF_NT, MMF_SMEM, stream>>>(n, w, is, vs, tab, vs_bar);
        }
    }
    const int fb = (int)((w + 255) / 256 < 1184 ? (w + 255) / 256 : 1184);
    VJP_LAUNCH(K_MINMAX_FINISH, stream) rbi_minmax_finish_kernel<IS_MAX><<<fb, 256, 0, stream>>>(n, w, tab, hist_bar, vs_bar_out, arg, ext, accumulate);
    return last_launch_status();
}

int launch_rbi_minmax(int code, int64_t n, int64_t w, const int64_t *is, const float *vs,
                      const float *hist_bar, float *vs_bar, int64_t *arg, float *ext, void *ws,
                      int accumulate, cudaStream_t stream) {
    return code == VJP_OP_MAX ? run_minmax<true>(n, w, is, vs, hist_bar, vs_bar, arg, ext, ws, accumulate, stream)
                              : run_minmax<false>(n, w, is, vs, hist_bar, vs_bar, arg, ext, ws, accumulate, stream);
}



// ------------------------------------------------- cached accumulation ('*', satadd) -------
//
// Operators with no hardware atomic (the paper's "atomicMul-class update").  A shared-memory
// atomicCAS is not affordable on any common path: one ATOMS.CAS warp instruction occupies the LSU for
// ~64 cycles WHATEVER the number of active lanes (profiles/r2a: three of them per batch of 128 elements
// cost as much as everything else together), and a CAS loop on a hot bin retries without bound
// (profiles/r1a: 5 ms at Zipf keys); match.any issues about once per 30 cycles per SM (profiles/r1b).
// So tables in shared memory are updated with plain loads and stores under a CLAIM ROUND.
//
// w <= CS_SLOTS (rbi_cached_small_kernel): a table per WARP, claims NaN-boxed into the table cells:
//   A. every pending element reads its bin's cell and, unless the cell already holds a claim,
//      overwrites it with a claim word naming the element -- a NaN-boxed pattern (sign 1, exponent
//      0xff, mantissa 0x7xxxxx | id) that no value the operators produce ever has (NaN inputs are
//      unsupported; FMUL / FADD generate the canonical NaN 0x7fffffff).  No separate claim array.
//   B. after a __syncwarp the element that reads its own claim back OWNS the bin for this round and
//      stores comb(old value, its value); every claimed cell has exactly one owner (the last
//      claim written), and every claim writer has read the cell's real value (values only change
//      in B, claims only appear in A).  Uniform keys at w = 1024: 6 % of the elements lose.
//   C. losers: further claim rounds over one element per lane -- no atomics anywhere.
// Skewed keys would make C the whole kernel, so every warp keeps a small DIRECTORY of hot bins
// (DIR_S direct-mapped slots) whose accumulators are LANE-PRIVATE (hot[slot][lane]: bank = lane):
// an element of a resident bin is folded into its lane's accumulator with a plain read-modify-write
// -- no claim, no conflict, whatever the multiplicity of the bin.  The directory is trained by the
// warp itself: a bin whose elements are still pending after two retry rounds (multiplicity >= 4 in a
// batch: rare at uniform keys) and that is hotter in the current batch than the slot's resident
// replaces it (the resident's 32 accumulators are folded with shuffles and written back).
// The directory is consulted only once it holds an entry: uniform keys never pay for it.
//
// w > CS_SLOTS (rbi_cached_big_kernel): one table per CTA, CTA-wide claim rounds through a separate
// claim array, guarded warp caches and a thread-private register entry for contended bins (described
// at the kernel).  CTA g writes its result to part[g][.]; a second kernel folds the G tables per bin
// in a fixed order.

constexpr uint32_t CLAIM = 0xFFF00000u;     // claim words are >= CLAIM as unsigned integers
constexpr uint32_t BIN_NONE = 0xffffffffu;  // no pending element
constexpr uint32_t DIR_EMPTY = 0xfffffffeu;
constexpr int DIR_S = 16;                   // directory slots per warp (2 KB of accumulators)

// 16 warps x 2 CTAs per SM (8 x 4: '*' w = 2^10 VJP 0.118 / 0.127 ms; 16 x 2: 0.115 / 0.122; 32 x 1: 0.115 / 0.123)
constexpr int CS_SLOTS = 1024, CS_WARPS = 16, CS_NT = CS_WARPS * 32, CS_CTAS_PER_SM = 2;   // w <= 1024
constexpr int CB_SLOTS = 64, CB_WARPS = 32, CB_NT = CB_WARPS * 32;                        // w  > 1024
constexpr int CB_PART = 32768;  // bins per CTA: 128 KB of f32 cells
constexpr int CB_MAX_SPLIT_LOG2 = 5;  // a group of up to 32 CTAs shares one histogram (w <= 2^20)
constexpr uint32_t CB_EMPTY = 0xffffffffu;  // tag word = (bin / CB_SLOTS) << 2 | hit counter

template <int ACC>
struct CachedOp;
template <>
struct CachedOp<ACC_MUL> {
    static VJP_DEVINL float neutral() { return 1.f; }
    static VJP_DEVINL float comb(float a, float b, float) { return a * b; }
};
template <>
struct CachedOp<ACC_SATADD> {
    static VJP_DEVINL float neutral() { return 0.f; }
    static VJP_DEVINL float comb(float a, float b, float S) { return fminf(a + b, S); }
};

template <int ACC>
VJP_DEVINL void smem_combine(uint32_t *cell, float v, float S) {
    unsigned old = *(volatile unsigned *)cell, assumed;
    do {
        assumed = old;
        old = atomicCAS(cell, assumed, __float_as_uint(CachedOp<ACC>::comb(__uint_as_float(assumed), v, S)));
    } while (old != assumed);
}

// fold of one value per lane over the warp (the operators are commutative)
template <int ACC>
VJP_DEVINL float warp_fold(float x, float S) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1)
        x = CachedOp<ACC>::comb(x, __shfl_xor_sync(FULL_MASK, x, off), S);
    return x;
}

// Directory of one warp: dir[DIR_S] resident bins, hot[DIR_S][32] lane-private accumulators.
struct WarpDir {
    uint32_t *dir;
    float *hot;
};

// Lookup of NI elements; a hit is folded into the lane's accumulator and removed from b[].
// hitm: bit s set if this lane hit slot s.
template <int ACC, int NI>
VJP_DEVINL void dir_lookup(const WarpDir &d, uint32_t (&b)[NI], const float (&v)[NI], int lane, float S,
                           uint32_t &hitm) {
#pragma unroll
    for (int j = 0; j < NI; j++) {
        const uint32_t s = b[j] & (DIR_S - 1);
        if (d.dir[s] == b[j]) {  // BIN_NONE never matches: entries are bins or DIR_EMPTY
            float *h = d.hot + s * 32 + lane;
            *h = CachedOp<ACC>::comb(*h, v[j], S);
            hitm |= 1u << s;
            b[j] = BIN_NONE;
        }
    }
}

// Called by the whole warp with a contended candidate bin `cand` (warp-uniform) that `c` lanes hold
// in elements still pending.  Installs it if the slot's resident is colder in this batch (fewer lanes hit
// it than hold the candidate); then the pending elements of cand are absorbed.  Returns true on install.
// flush(bin, value): adds the evicted resident's fold to the table (called by lane 0 only).
template <int ACC, int NI, class Flush>
VJP_DEVINL bool dir_train(const WarpDir &d, uint32_t cand, int c, uint32_t hitm, uint32_t (&b)[NI],
                          const float (&v)[NI], int lane, float S, int &ndir, Flush flush) {
    const uint32_t s = cand & (DIR_S - 1);
    const int h = __popc(__ballot_sync(FULL_MASK, (hitm >> s) & 1u));
    if (c <= h) return false;
    const uint32_t old = d.dir[s];
    float *hp = d.hot + s * 32 + lane;
    if (old != DIR_EMPTY) {
        const float x = warp_fold<ACC>(*hp, S);
        if (lane == 0) flush(old, x);
    } else {
        ndir++;
    }
    float acc = CachedOp<ACC>::neutral();
#pragma unroll
    for (int j = 0; j < NI; j++)
        if (b[j] == cand) {
            acc = CachedOp<ACC>::comb(acc, v[j], S);
            b[j] = BIN_NONE;
        }
    *hp = acc;
    __syncwarp();
    if (lane == 0) d.dir[s] = cand;
    __syncwarp();
    return true;
}

// COUNT_ZEROS: the lifted '*' of the VJP: zeros are counted (integer atomics, exact) and
// kept out of the product.  Otherwise: the plain primal histogram of the operator.
//
// w <= CS_SLOTS: every warp owns a private table (a slot IS a bin) and runs the claim round over the
// 128 elements of its batch (one quad per lane) with __syncwarp as the barrier.  The hot loop is
// branch-free: an element that takes no part (key out of range, a counted zero, a directory hit) is
// pointed at its lane's DUMMY cell behind the table and goes through the same loads and stores
// (profiles/r2a: the first version spent 340 instructions per quad, most of them control flow).
constexpr int CS_TAB = CS_SLOTS + 32;  // + one dummy cell per lane
constexpr size_t CS_SMEM = (size_t)CS_WARPS * (CS_TAB * 4 + DIR_S * 32 * 4 + DIR_S * 4);

template <int ACC, bool COUNT_ZEROS>
__global__ void __launch_bounds__(CS_NT, CS_CTAS_PER_SM)
rbi_cached_small_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                        const float *__restrict__ vs, float *__restrict__ part, unsigned *zeros,
                        float S) {
    using OP = CachedOp<ACC>;
    extern __shared__ uint4 smem_raw[];
    uint32_t *tabs = reinterpret_cast<uint32_t *>(smem_raw);                  // [CS_WARPS][CS_TAB]
    float *hots = reinterpret_cast<float *>(tabs + CS_WARPS * CS_TAB);        // [CS_WARPS][DIR_S][32]
    uint32_t *dirs = reinterpret_cast<uint32_t *>(hots + CS_WARPS * DIR_S * 32);  // [CS_WARPS][DIR_S]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *tab = tabs + warp * CS_TAB;
    WarpDir d;
    d.hot = hots + warp * DIR_S * 32;
    d.dir = dirs + warp * DIR_S;
    for (int s = lane; s < CS_TAB; s += 32) tab[s] = __float_as_uint(OP::neutral());
    for (int s = lane; s < DIR_S * 32; s += 32) d.hot[s] = OP::neutral();
    if (lane < DIR_S) d.dir[lane] = DIR_EMPTY;
    __syncwarp();
    int ndir = 0;  // warp-uniform: resident directory entries
    const uint32_t myid = CLAIM | (uint32_t)(lane * 4);
    const uint32_t dummy = CS_SLOTS + lane, w32 = (uint32_t)w;
    auto flush = [&](uint32_t bin, float x) { tab[bin] = __float_as_uint(OP::comb(__uint_as_float(tab[bin]), x, S)); };

    // one batch: the quad (k, v) of every lane
    auto process = [&](const int64_t (&k)[4], const float (&v)[4]) {
        uint32_t b[4];  // table index of a pending element, `dummy` otherwise
        bool zq = false;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const uint32_t lo = (uint32_t)k[j], hi = (uint32_t)((uint64_t)k[j] >> 32);
            bool act = (hi == 0u) & (lo < w32);
            if (COUNT_ZEROS) {
                const bool z = act & (v[j] == 0.f);  // IEEE equality: +-0 only (Q7)
                zq |= z;
                act &= !z;
            }
            b[j] = act ? lo : dummy;
        }
        if (COUNT_ZEROS && zq) {  // rare
#pragma unroll
            for (int j = 0; j < 4; j++)
                if (in_range(k[j], w) && v[j] == 0.f) atomicAdd(zeros + k[j], 1u);
        }
        uint32_t hitm = 0;
        if (ndir) {
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const uint32_t s = b[j] & (DIR_S - 1);
                if (d.dir[s] == b[j]) {  // a dummy index never matches: entries are bins or DIR_EMPTY
                    float *h = d.hot + s * 32 + lane;
                    *h = OP::comb(*h, v[j], S);
                    hitm |= 1u << s;
                    b[j] = dummy;
                }
            }
        }
        // claim round over the warp's 128 elements
        uint32_t o[4], c[4];
#pragma unroll
        for (int j = 0; j < 4; j++) o[j] = tab[b[j]];
#pragma unroll
        for (int j = 0; j < 4; j++)
            if (o[j] < CLAIM) tab[b[j]] = myid + j;
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 4; j++) c[j] = tab[b[j]];
        uint32_t pm = 0;  // bit j: a real element that lost
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const bool win = c[j] == myid + j;
            if (win) tab[b[j]] = __float_as_uint(OP::comb(__uint_as_float(o[j]), v[j], S));
            pm |= (uint32_t)(!win & (b[j] < (uint32_t)CS_SLOTS)) << j;
        }
        __syncwarp();
        // The losers: claim rounds over one element per lane (a shared-memory atomicCAS instead costs the
        // LSU ~64 cycles per warp instruction whatever the number of lanes: three of them per batch made this
        // kernel no faster than the one it replaced).  Elements still pending after two such rounds sit in a
        // bin of multiplicity >= 4: skewed keys -- the directory is trained with that bin.
        for (int it = 0; __any_sync(FULL_MASK, pm != 0); it++) {
            if (it >= 2 && (it & 1) == 0) {
                const unsigned lm = __ballot_sync(FULL_MASK, pm != 0);
                const uint32_t mine = (pm & 1u) ? b[0] : (pm & 2u) ? b[1] : (pm & 4u) ? b[2] : b[3];
                const uint32_t cand = __shfl_sync(FULL_MASK, mine, __ffs(lm) - 1);
                uint32_t pb[4];
#pragma unroll
                for (int j = 0; j < 4; j++) pb[j] = (pm >> j & 1u) ? b[j] : BIN_NONE;
                const bool has = (pb[0] == cand) | (pb[1] == cand) | (pb[2] == cand) | (pb[3] == cand);
                const int cl = __popc(__ballot_sync(FULL_MASK, has));
                if (dir_train<ACC, 4>(d, cand, cl, hitm, pb, v, lane, S, ndir, flush)) {
#pragma unroll
                    for (int j = 0; j < 4; j++)
                        if (pb[j] == BIN_NONE) pm &= ~(1u << j);
                    continue;
                }
            }
            uint32_t pb = dummy;
            float pv = 0.f;
            if (pm & 1u) { pb = b[0]; pv = v[0]; }
            else if (pm & 2u) { pb = b[1]; pv = v[1]; }
            else if (pm & 4u) { pb = b[2]; pv = v[2]; }
            else if (pm & 8u) { pb = b[3]; pv = v[3]; }
            const uint32_t o1 = tab[pb];
            if (o1 < CLAIM) tab[pb] = myid;
            __syncwarp();
            const uint32_t c1 = tab[pb];
            if (c1 == myid) {
                tab[pb] = __float_as_uint(OP::comb(__uint_as_float(o1), pv, S));
                pm &= pm - 1;
            }
            __syncwarp();
        }
    };

    const uint32_t nfull = (uint32_t)(n / 4);  // quads that exist entirely
    const uint32_t stride = gridDim.x * CS_NT;
    // Whole batches: unconditional 128-bit loads, TWO batches in flight per warp (one was not enough: with
    // half the instructions of the first version the kernel waited on its loads, profiles/r2b).
    struct Quad {
        longlong2 a, b;
        uint4 v;
    };
    const uint64_t keep = l2_policy_normal();
    auto fetch = [&](uint32_t q, Quad &x) {  // warp-uniform q; only whole batches are fetched here
        if (q + 32 <= nfull) {
            const longlong2 *kp = reinterpret_cast<const longlong2 *>(is) + 2 * (size_t)(q + lane);
            x.a = ldg_hint_ll2(kp, keep);
            x.b = ldg_hint_ll2(kp + 1, keep);
            x.v = ldg_hint(reinterpret_cast<const uint4 *>(vs) + (q + lane), keep);
        }
    };
    auto run = [&](const Quad &x) {
        const int64_t k[4] = {x.a.x, x.a.y, x.b.x, x.b.y};
        const float v[4] = {__uint_as_float(x.v.x), __uint_as_float(x.v.y), __uint_as_float(x.v.z), __uint_as_float(x.v.w)};
        process(k, v);
    };
    uint32_t q0 = blockIdx.x * CS_NT + warp * 32, q1 = q0 + stride;  // warp-uniform: the warp never diverges here
    Quad A = {}, B = {};
    fetch(q0, A);
    fetch(q1, B);
    for (;;) {
        if (q0 + 32 > nfull) break;
        const Quad cur = A;
        q0 += 2 * stride;
        fetch(q0, A);
        run(cur);
        if (q1 + 32 > nfull) break;
        const Quad cur1 = B;
        q1 += 2 * stride;
        fetch(q1, B);
        run(cur1);
    }
    // the ragged end of the input (at most one batch per warp: the first one that is not whole)
    const uint32_t qw = q0 < q1 ? q0 : q1;
    if ((int64_t)qw * 4 < n) {
        int64_t k[4] = {-1, -1, -1, -1};
        float v[4] = {0.f, 0.f, 0.f, 0.f};
        if ((int64_t)(qw + lane) * 4 < n) {
            const int cnt = load_keys4(is, (int64_t)(qw + lane) * 4, n, k);
            load_vals4(vs, (int64_t)(qw + lane) * 4, cnt, v);
        }
        process(k, v);
    }
    for (int s = 0; s < DIR_S; s++) {  // write the directory back
        const uint32_t bin = d.dir[s];
        if (bin == DIR_EMPTY) continue;
        const float x = warp_fold<ACC>(d.hot[s * 32 + lane], S);
        if (lane == 0) flush(bin, x);
    }
    __syncthreads();
    for (int s = threadIdx.x; s < (int)w; s += CS_NT) {
        float acc = __uint_as_float(tabs[s]);
#pragma unroll
        for (int wp = 1; wp < CS_WARPS; wp++) acc = OP::comb(acc, __uint_as_float(tabs[wp * CS_TAB + s]), S);
        part[(size_t)blockIdx.x * (size_t)w + s] = acc;
    }
}

// w > CS_SLOTS.  Returns true if (eb, evv) must go to the CTA table.
template <int ACC>
VJP_DEVINL bool claim_update_big(bool act, uint32_t b, float x, float *vl, uint32_t *tg, uint8_t *cl,
                                 float S, int lane, uint32_t &eb, float &evv) {
    bool pend = act, ev = false;
    const uint32_t slot = b & (CB_SLOTS - 1), hi = b / CB_SLOTS;
    while (__any_sync(FULL_MASK, pend)) {
        if (pend) cl[slot] = (uint8_t)lane;
        __syncwarp();
        if (pend && cl[slot] == lane) {
            pend = false;
            const uint32_t t = tg[slot];
            if (t != CB_EMPTY && (t >> 2) == hi) {             // hit
                vl[slot] = CachedOp<ACC>::comb(vl[slot], x, S);
                if ((t & 3u) != 3u) tg[slot] = t + 1;
            } else if (t == CB_EMPTY || (t & 3u) == 0u) {       // install (evicting)
                if (t != CB_EMPTY) {
                    ev = true;
                    eb = (t >> 2) * CB_SLOTS + slot;
                    evv = vl[slot];
                }
                tg[slot] = hi << 2;
                vl[slot] = x;
            } else {                                            // guarded: bypass
                tg[slot] = t - 1;
                ev = true;
                eb = b;
                evv = x;
            }
        }
        __syncwarp();
    }
    return ev;
}

// The next batch is prefetched into registers (true) or, by cp.async.bulk.prefetch, into L2 and loaded at the top of its own
// iteration (false: 12 registers fewer, so U = 2 fits without spills).  Lifted '*' at w = 2^16, uniform / Zipf keys:
// registers U = 1 0.125 / 0.222 ms; L2 U = 1 0.125 / 0.236; L2 U = 2 (half the barriers) 0.129 / 0.237.
constexpr bool CB_REGPF = true;
constexpr int CB_U = 1;               // quads per thread per batch (2 spills at 64 registers: 0.17 -> 0.24 ms)
constexpr uint32_t CB_RW = 8, CB_RMAX = 63;  // register entry: kept by a bin with more than 1/(1+CB_RW) of the elements
constexpr size_t CB_SMEM = (size_t)CB_PART * 6 + (size_t)CB_WARPS * CB_SLOTS * 9;
constexpr int CB_PROBE = 4, CB_HOLD = 8;    // batches before the first decision / in full mode after a lean batch went bad

// w > CS_SLOTS.  A CTA of 1024 threads owns a table of up to CB_PART bins in shared memory.  A
// histogram wider than that is SPLIT over the 2^c CTAs of a group by the low c bits of the bin
// (hot neighbouring bins land on different CTAs); all CTAs of a group stream the same part of the
// input at the same time (one of them pulls it from HBM, the others hit in L2) and each keeps the
// elements of its own bins: one pass over the input for any w, no traffic between the CTAs.
//
// Per batch (U quads per thread) the table is updated WITHOUT atomics:
//   0. an element whose bin is resident in the warp's cache is "hot" and goes to step 2 directly;
//   1. one CTA-wide claim round: every pending element stores its id into the bin's claim word,
//      barrier, the element that reads its id back owns the bin for this round and does a plain
//      read-modify-write of the table cell.  Uniform keys at w = 2^16: ~6 % of the elements lose.
//      A loser gets ONE compare-and-swap on the cell (uniform keys: it succeeds);
//   2. hot elements: claim rounds inside the warp on the resident cache entry (plain LDS/STS); an
//      element that lost the round AND its compare-and-swap sits in a CONTENDED bin: the warp's
//      cache installs it unless a hotter bin guards the slot (claim_update_big above).  Hot bins
//      therefore migrate into the caches and stop taking part in step 1; evictions and bypasses
//      (cold, rare) fall back to a CAS loop on the table.
// Barriers: [claim] B1 [plain updates] B2 [CAS, caches].  Two elements never own one bin in a round
// because all claims precede B1; the plain updates (between B1 and B2) never overlap a CAS (after
// B2, before the next batch's B1).
//
// LEAN mode: the register entry and the cache look-up are a third of the instructions of a batch and absorb
// nothing when no bin is hot (uniform keys).  The CTA therefore measures what they absorb: after CB_PROBE batches
// with fewer than a quarter of the threads at >= 2 absorbed elements it skips steps 0 (and the register entry);
// every lean batch counts its losers at B2 (free: the barrier carries the count), and a batch in which more than
// 3/8 of the threads hold a loser -- uniform keys: 12 % -- puts the full machinery back for CB_HOLD batches.
// Either mode is correct on any input (a cached or register-held partial product is just one more factor, folded
// into the table at the end); the switch only moves instructions.
template <bool B>
struct BoolC { static constexpr bool value = B; };

template <int ACC, bool COUNT_ZEROS, int U>
__global__ void __launch_bounds__(CB_NT, 1)
rbi_cached_big_kernel(int64_t n, int64_t w, int cl_log2, const int64_t *__restrict__ is,
                      const float *__restrict__ vs, float *__restrict__ part, unsigned *zeros,
                      float S) {
    using OP = CachedOp<ACC>;
    extern __shared__ uint4 smem_raw[];
    float *table = reinterpret_cast<float *>(smem_raw);                          // [CB_PART]
    float *vals = table + CB_PART;                                               // [CB_WARPS][CB_SLOTS]
    uint32_t *tags = reinterpret_cast<uint32_t *>(vals + CB_WARPS * CB_SLOTS);    // [CB_WARPS][CB_SLOTS]
    uint16_t *claimA = reinterpret_cast<uint16_t *>(tags + CB_WARPS * CB_SLOTS);  // [CB_PART]
    uint8_t *claim = reinterpret_cast<uint8_t *>(claimA + CB_PART);               // [CB_WARPS][CB_SLOTS]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *vl = vals + warp * CB_SLOTS;
    uint32_t *tg = tags + warp * CB_SLOTS;
    uint8_t *cl = claim + warp * CB_SLOTS;
    const uint32_t clmask = (1u << cl_log2) - 1u;
    const uint32_t rank = blockIdx.x & clmask;
    const int64_t group = blockIdx.x >> cl_log2, groups = gridDim.x >> cl_log2;
    for (int i = threadIdx.x; i < CB_PART; i += CB_NT) table[i] = OP::neutral();
    for (int s = lane; s < CB_SLOTS; s += 32) {
        vl[s] = OP::neutral();
        tg[s] = CB_EMPTY;
    }
    __syncthreads();
    constexpr int NI = 4 * U;
    const int64_t nquads = (n + 3) / 4;
    const int64_t stride = groups * (int64_t)(CB_NT * U);
    int64_t q0 = group * (int64_t)(CB_NT * U);  // CTA-uniform: no thread leaves the barriers early
    int64_t k[NI];
    float v[NI];
    const int64_t nwhole = n >> 2;  // quads that exist in full
    const uint64_t keep = l2_policy_normal();
    auto load_batch = [&](int64_t q, int64_t (&kk)[NI], float (&vv)[NI]) {
        if (q + CB_NT * U <= nwhole) {  // CTA-uniform: the whole batch exists, no per-thread guards
#pragma unroll
            for (int u = 0; u < U; u++) {
                const int64_t qq = q + u * CB_NT + threadIdx.x;
                const longlong2 *pk = reinterpret_cast<const longlong2 *>(is) + 2 * qq;
                const longlong2 a = ldg_hint_ll2(pk, keep), c = ldg_hint_ll2(pk + 1, keep);
                const uint4 x = ldg_hint(reinterpret_cast<const uint4 *>(vs) + qq, keep);
                kk[u * 4 + 0] = a.x; kk[u * 4 + 1] = a.y; kk[u * 4 + 2] = c.x; kk[u * 4 + 3] = c.y;
                vv[u * 4 + 0] = __uint_as_float(x.x); vv[u * 4 + 1] = __uint_as_float(x.y);
                vv[u * 4 + 2] = __uint_as_float(x.z); vv[u * 4 + 3] = __uint_as_float(x.w);
            }
            return;
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            int64_t k4[4] = {-1, -1, -1, -1};
            float v4[4] = {0.f, 0.f, 0.f, 0.f};
            const int64_t qq = q + u * CB_NT + threadIdx.x;
            if (qq < nquads) {
                const int cnt = load_keys4(is, qq * 4, n, k4);
                load_vals4(vs, qq * 4, cnt, v4);
            }
#pragma unroll
            for (int j = 0; j < 4; j++) {
                kk[u * 4 + j] = k4[j];
                vv[u * 4 + j] = v4[j];
            }
        }
    };
    // A claim word names the ELEMENT (thread id * NI + j): exactly one element per bin wins a round,
    // so all claim words and table cells of a round can be read before any of them is written.
    const uint32_t id0 = threadIdx.x * NI;
    // Thread-private register entry (rb, racc, rcnt) in front of everything: a bin that holds a
    // large share of the elements (one bin = 14 % at Zipf keys) is folded into a register with no
    // shared-memory access at all.  Weighted majority vote: +CB_RW on a hit, -1 on a miss, replaced
    // at 0 -- the displaced pair takes the element's place on the normal path.
    uint32_t rb = CB_EMPTY, rcnt = 0;
    float racc = OP::neutral();
    int until = CB_PROBE;       // CTA-uniform: > 0 full-mode batches until the next decision, < 0 lean mode
    load_batch(q0, k, v);
    for (;;) {
        // after the last batch of the input: one more round of the same machinery for the register
        // entries (1024 CAS on one hot cell would serialise); q0 is CTA-uniform
        const bool drain = q0 >= nquads;
        int64_t kn[CB_REGPF ? NI : 1];
        float vn[CB_REGPF ? NI : 1];
        const int64_t qn = q0 + stride;
        if constexpr (CB_REGPF) {
            load_batch(qn, kn, vn);  // next batch's loads fly while this one is processed (none past the end)
        } else if (qn + CB_NT * U <= nwhole) {  // next batch on its way into L2: no registers held across the body
            prefetch_tile_l2<CB_WARPS>(is + 4 * qn, (int64_t)CB_NT * U * 32);
            prefetch_tile_l2<CB_WARPS>(vs + 4 * qn, (int64_t)CB_NT * U * 16);
        }
        uint32_t b[NI];  // table index of a pending element, CB_EMPTY = nothing pending
        uint32_t zm = 0;
#pragma unroll
        for (int j = 0; j < NI; j++) {
            const uint32_t klo = (uint32_t)k[j];
            bool act = in_range(k[j], w) & ((klo & clmask) == rank);
            if (COUNT_ZEROS) {
                const bool z = act & (v[j] == 0.f);  // IEEE equality: +-0 only (Q7)
                zm |= (uint32_t)z << j;
                act &= !z;
            }
            b[j] = act ? klo >> cl_log2 : CB_EMPTY;
        }
        if (COUNT_ZEROS && zm) {
#pragma unroll
            for (int j = 0; j < NI; j++)
                if (zm >> j & 1u) atomicAdd(zeros + k[j], 1u);
        }
        if (drain) {
            b[0] = rb;
            v[0] = racc;
            rcnt = 1;  // keeps the loop below from re-installing it
            rb = CB_EMPTY;
            until = 1 << 30;  // full mode: 1024 partial products of one hot bin go through the caches, not through 1024 CAS
        }
        // one straight-line body per mode (a run-time flag inside one body cost both modes 7-11 %: the branches end
        // the basic blocks the loads are scheduled across)
        auto body = [&](auto LEAN_T) {
        constexpr bool lean = decltype(LEAN_T)::value;
        if constexpr (!lean) {
#pragma unroll
        for (int j = 0; j < NI; j++) {  // register entry
            if (b[j] == CB_EMPTY) continue;
            if (b[j] == rb) {
                racc = OP::comb(racc, v[j], S);
                rcnt = min(rcnt + CB_RW, CB_RMAX);
                b[j] = CB_EMPTY;
            } else if (rcnt == 0) {
                const uint32_t ob = rb;
                const float ov = racc;
                rb = b[j];
                racc = v[j];
                b[j] = ob;  // CB_EMPTY the first time
                v[j] = ov;
            } else {
                rcnt--;
            }
        }
        }
        uint32_t coldm = 0;  // bit j: pending and not resident in the warp's cache
        uint32_t hotm = 0;   // bit j: pending and resident
        if constexpr (!lean) {
            uint32_t t[NI];
#pragma unroll
            for (int j = 0; j < NI; j++) t[j] = tg[b[j] & (CB_SLOTS - 1)];
#pragma unroll
            for (int j = 0; j < NI; j++) {
                // a valid tag never equals CB_EMPTY's, and b == CB_EMPTY matches no tag
                const bool hot = (t[j] >> 2) == b[j] / CB_SLOTS;
                const bool cold = !hot & (b[j] != CB_EMPTY);
                hotm |= (uint32_t)hot << j;
                coldm |= (uint32_t)cold << j;
                if (hot & ((t[j] & 3u) != 3u)) tg[b[j] & (CB_SLOTS - 1)] = t[j] + 1;  // racing lanes store the same word
                if (cold) claimA[b[j]] = (uint16_t)(id0 + j);
            }
        } else {
#pragma unroll
            for (int j = 0; j < NI; j++) {
                const bool cold = b[j] != CB_EMPTY;
                coldm |= (uint32_t)cold << j;
                if (cold) claimA[b[j]] = (uint16_t)(id0 + j);
            }
        }
        bool plain_b1 = true;
        if constexpr (!lean) {
            if (--until == 0) {  // B1, carrying the decision: threads with a cache hit now or a register hit lately
                const int busy = __syncthreads_count(hotm != 0 || rcnt > 1);
                until = busy < CB_NT / 4 ? -1 : CB_PROBE;
                plain_b1 = false;
            }
        }
        if (plain_b1) __syncthreads();  // B1
        {
            uint16_t c[NI];
            float o[NI];
#pragma unroll
            for (int j = 0; j < NI; j++) {
                c[j] = claimA[b[j] & (CB_PART - 1)];
                o[j] = table[b[j] & (CB_PART - 1)];
            }
#pragma unroll
            for (int j = 0; j < NI; j++) {
                const bool cold = coldm >> j & 1u;
                const bool win = cold & (c[j] == (uint16_t)(id0 + j));
                if (win) table[b[j]] = OP::comb(o[j], v[j], S);
                coldm &= ~((uint32_t)win << j);
            }
        }
        // B2: the plain updates are done before any CAS touches the table
        if constexpr (lean) {
            if (__syncthreads_count(coldm != 0) > CB_NT * 3 / 8) until = CB_HOLD;  // this batch's losers still take the path below
        } else {
            __syncthreads();
        }
        if (__any_sync(FULL_MASK, coldm != 0)) {
#pragma unroll
            for (int j = 0; j < NI; j++) {  // losers: ONE compare-and-swap; a failure means the bin is contended
                if (coldm >> j & 1u) {
                    unsigned *cell = reinterpret_cast<unsigned *>(table + b[j]);
                    const unsigned old = *(volatile unsigned *)cell;
                    const unsigned upd = __float_as_uint(OP::comb(__uint_as_float(old), v[j], S));
                    if (atomicCAS(cell, old, upd) == old) coldm &= ~(1u << j);
                }
            }
        }
        if (!lean && __any_sync(FULL_MASK, hotm != 0)) {
#pragma unroll
            for (int j = 0; j < NI; j++) {  // hits: the resident entry cannot change before the installs below
                uint8_t *c = cl + (b[j] & (CB_SLOTS - 1));
                float *a = vl + (b[j] & (CB_SLOTS - 1));
                bool pend = hotm >> j & 1u;
                while (__any_sync(FULL_MASK, pend)) {
                    if (pend) *c = (uint8_t)lane;
                    __syncwarp();
                    if (pend && *c == lane) {
                        *a = OP::comb(*a, v[j], S);
                        pend = false;
                    }
                    __syncwarp();
                }
            }
        }
        if (__any_sync(FULL_MASK, coldm != 0)) {
#pragma unroll
            for (int j = 0; j < NI; j++) {
                const bool act = coldm >> j & 1u;
                if (__any_sync(FULL_MASK, act)) {
                    uint32_t eb = 0;
                    float evv = 0.f;
                    if (claim_update_big<ACC>(act, b[j], v[j], vl, tg, cl, S, lane, eb, evv))
                        smem_combine<ACC>(reinterpret_cast<uint32_t *>(table + eb), evv, S);
                }
            }
        }
        };
        if (until < 0) body(BoolC<true>{}); else body(BoolC<false>{});
        if (drain) break;
        if constexpr (CB_REGPF) {
#pragma unroll
            for (int j = 0; j < NI; j++) {
                k[j] = kn[j];
                v[j] = vn[j];
            }
        } else {
            load_batch(qn, k, v);
        }
        q0 = qn;
    }
    __syncthreads();
    for (int s = lane; s < CB_SLOTS; s += 32) {  // write the warp's cache back
        const uint32_t t = tg[s];
        if (t != CB_EMPTY) smem_combine<ACC>(reinterpret_cast<uint32_t *>(table + (t >> 2) * CB_SLOTS + s), vl[s], S);
    }
    __syncthreads();
    float *dst = part + (size_t)group * (size_t)w;
    for (int64_t i = threadIdx.x; i < CB_PART; i += CB_NT) {
        const int64_t bin = (i << cl_log2) + rank;
        if (bin < w) dst[bin] = table[i];
    }
}

// Fold of the G per-CTA tables for 32 consecutive bins by a CTA of 256 threads: thread (x, y) folds
// part[g][k0 + x] for g = y, y + 8, ... (coalesced across x, 8 independent chains per bin), then the
// 8 chains are combined in a fixed order through shared memory (deterministic).  Returns the result
// in the threads with y == 0.  One thread per bin walking all G tables was latency-bound (10 % of
// the bench step in the launch list of profiles/r1g).
// CH chains per bin (CTA of 32 * CH threads): 8, or 32 when there are hundreds of tables to fold (narrow histograms
// written by every CTA of a full grid: 592 tables at w <= 1024), where 8 chains of 74 dependent loads were the
// kernel's whole duration; at w = 2^16 (74 tables) 32 chains are slower (+13 us, round 1).
template <int ACC, int CH>
VJP_DEVINL float fold_partials(int64_t w, int G, const float *__restrict__ part, int64_t k, float S) {
    __shared__ float sm[CH][32];
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    float p = CachedOp<ACC>::neutral();
    if (k < w) {
#pragma unroll 4
        for (int g = y; g < G; g += CH) p = CachedOp<ACC>::comb(p, __ldg(part + (size_t)g * (size_t)w + k), S);
    }
    sm[y][x] = p;
    __syncthreads();
    if (y == 0) {
#pragma unroll
        for (int i = 1; i < CH; i++) p = CachedOp<ACC>::comb(p, sm[i][x], S);
    }
    return p;
}
static int fold_chains(int G) { return G >= 256 ? 32 : 8; }
static int fold_grid(int64_t w) { return (int)((w + 31) / 32); }

// out[k] = fold over the G partial tables.
template <int ACC, int CH>
__global__ void __launch_bounds__(32 * CH)
rbi_cached_fold_kernel(int64_t w, int G, const float *__restrict__ part, float *__restrict__ out, float S) {
    const int64_t k = (int64_t)blockIdx.x * 32 + (threadIdx.x & 31);
    const float p = fold_partials<ACC, CH>(w, G, part, k, S);
    if (threadIdx.x < 32 && k < w) out[k] = p;
}

// log2 of the CTAs per group: the smallest power of two with 2^c * CB_PART >= w
static int cached_split_log2(int64_t w) {
    int c = 0;
    while (((int64_t)CB_PART << c) < w) c++;
    return c;
}
static int cached_grid(int64_t n, int64_t w) {
    if (w <= CS_SLOTS) return grid_for(n < 1 ? 1 : n, CS_NT, CS_CTAS_PER_SM);
    const int c = cached_split_log2(w);
    const int64_t quads = ((n < 1 ? 1 : n) + 3) / 4;
    int64_t groups = (quads + CB_NT * CB_U - 1) / (CB_NT * CB_U);
    const int64_t cap = NUM_SMS_B200 >> c > 0 ? NUM_SMS_B200 >> c : 1;
    if (groups > cap) groups = cap;
    return (int)(groups << c);
}
// 1024 < w <= 12288: the in-order walk of rbi_multiscan.cu as a histogram (warp-private tables, no CTA-wide rounds)
static bool cached_walk(int64_t w) { return w > CS_SLOTS && rbi_multiscan_fits(w); }
// number of partial tables the accumulation kernel writes
static int cached_tables(int64_t n, int64_t w) {
    if (cached_walk(w)) return rbi_ms_hist_tables(n, w);
    return w <= CS_SLOTS ? cached_grid(n, w) : cached_grid(n, w) >> cached_split_log2(w);
}
static size_t cached_part_bytes(int64_t n, int64_t w) {
    return align_up((size_t)cached_tables(n, w) * (size_t)(w < 1 ? 1 : w) * 4, 256);
}
bool rbi_cached_supported(int64_t w) { return w <= ((int64_t)CB_PART << CB_MAX_SPLIT_LOG2); }

// Accumulates into part[G][w]; returns G in *G_out.
template <int ACC, bool COUNT_ZEROS>
static int run_cached(int64_t n, int64_t w, const int64_t *is, const float *vs, float *part,
                      unsigned *zeros, float S, int *G_out, cudaStream_t stream, int ld = 0) {
    const int G = cached_grid(n, w);
    *G_out = cached_tables(n, w);
    if (cached_walk(w))
        return launch_ms_hist(ACC == ACC_MUL, COUNT_ZEROS, S, n, w, is, vs, part, zeros, ld, stream);
    if (ld != 0) return VJP_ERR_UNSUPPORTED;  // virtual keys: the walk only (rbi_mul_vec_fused)
    if (w <= CS_SLOTS) {
        auto kern = rbi_cached_small_kernel<ACC, COUNT_ZEROS>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CS_SMEM) != cudaSuccess)
            return VJP_ERR_CUDA;
        VJP_LAUNCH(K_CACHED_SMALL, stream) kern<<<G, CS_NT, CS_SMEM, stream>>>(n, w, is, vs, part, zeros, S);
    } else {
        auto kern = rbi_cached_big_kernel<ACC, COUNT_ZEROS, CB_U>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CB_SMEM) != cudaSuccess)
            return VJP_ERR_CUDA;
        VJP_LAUNCH(K_CACHED_BIG, stream) kern<<<G, CB_NT, CB_SMEM, stream>>>(n, w, cached_split_log2(w), is, vs, part, zeros, S);
    }
    return last_launch_status();
}

static int launch_cached_primal(int code, int64_t n, int64_t w, const int64_t *is, const float *vs,
                                float *hist, void *ws, float S, cudaStream_t stream) {
    if (w == 0) return VJP_OK;
    if (!rbi_cached_supported(w)) return VJP_ERR_UNSUPPORTED;
    float *part = static_cast<float *>(ws);
    int G = 0;
    const int rc = code == VJP_OP_MUL
                       ? run_cached<ACC_MUL, false>(n, w, is, vs, part, nullptr, S, &G, stream)
                       : run_cached<ACC_SATADD, false>(n, w, is, vs, part, nullptr, S, &G, stream);
    if (rc != VJP_OK) return rc;
    const bool wide = fold_chains(G) == 32;
    if (code == VJP_OP_MUL) {
        if (wide) VJP_LAUNCH(K_CACHED_FOLD, stream) rbi_cached_fold_kernel<ACC_MUL, 32><<<fold_grid(w), 1024, 0, stream>>>(w, G, part, hist, S);
        else VJP_LAUNCH(K_CACHED_FOLD, stream) rbi_cached_fold_kernel<ACC_MUL, 8><<<fold_grid(w), 256, 0, stream>>>(w, G, part, hist, S);
    } else {
        if (wide) VJP_LAUNCH(K_CACHED_FOLD, stream) rbi_cached_fold_kernel<ACC_SATADD, 32><<<fold_grid(w), 1024, 0, stream>>>(w, G, part, hist, S);
        else VJP_LAUNCH(K_CACHED_FOLD, stream) rbi_cached_fold_kernel<ACC_SATADD, 8><<<fold_grid(w), 256, 0, stream>>>(w, G, part, hist, S);
    }
    return last_launch_status();
}

// ------------------------------------------------------------------ '*' VJP ---------------
//
// Lifted primal: per bin (zero count, product of the non-zeros) by the cached accumulation
// above, then the return sweep.

// Per bin: fold the G partial products (fixed order: deterministic), expose (zeros, prod_nz), and
// prepare the return sweep's coefficient c_k = prod_nz_k * hist_bar_k with the zero count clamped
// to {0, 1, 2}.
template <int CH>
__global__ void __launch_bounds__(32 * CH)
rbi_mul_finish_kernel(int64_t w, int G, const float *__restrict__ part,
                      const unsigned *__restrict__ zeros_u, const float *__restrict__ hist_bar,
                      int64_t *zeros, float *prod_nz, float2 *coef, int planes) {
    const int64_t k = (int64_t)blockIdx.x * 32 + (threadIdx.x & 31);
    const float p = fold_partials<ACC_MUL, CH>(w, G, part, k, 0.f);
    if (threadIdx.x < 32 && k < w) {
        const unsigned z = zeros_u[k];
        if (zeros) zeros[k] = (int64_t)z;
        if (prod_nz) prod_nz[k] = p;
        if (coef && !planes) coef[k] = make_float2(p * hist_bar[k], __int_as_float((int)(z < 2u ? z : 2u)));
        if (coef && planes) {  // wide histograms (table gathered from L1 / L2): two planes of w floats, see the sweep
            float *pl = reinterpret_cast<float *>(coef);
            const float c = p * hist_bar[k];
            pl[k] = z == 0u ? c : 0.f;
            pl[w + k] = z == 1u ? c : 0.f;
        }
    }
}

// Return sweep (Fig. 3): no zero in the bin -> (y / a) * ybar; exactly one
// zero and a is that zero -> y^{>0} * ybar; otherwise 0.  Out-of-range keys get 0.
// VEC: flat arrays of the vectorised operator with virtual keys is[j >> ld] << ld | (j & (d - 1)) (see ms_hist_kernel).
template <bool SMEM, bool VEC = false>
__global__ void __launch_bounds__(RBI_NT)
rbi_mul_sweep_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                     const float *__restrict__ vs, const float2 *__restrict__ coef,
                     float *__restrict__ vs_bar, int accumulate, int ld = 0) {
    extern __shared__ uint4 smem_raw[];
    float2 *sh = reinterpret_cast<float2 *>(smem_raw);
    if (SMEM) {
        for (int k = threadIdx.x; k < (int)w; k += RBI_NT) sh[k] = coef[k];
        __syncthreads();
    }
    const int64_t stride = (int64_t)gridDim.x * RBI_NT;
    const uint64_t strm = l2_policy_stream();
    for (int64_t q = blockIdx.x * (int64_t)RBI_NT + threadIdx.x; q * 4 < n; q += stride) {
        int64_t k[4];
        float v[4], o[4];
        int cnt;
        if constexpr (VEC) {
            cnt = (int)min((int64_t)4, n - q * 4);
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int64_t idx = q * 4 + j;
                const int64_t kr = j < cnt ? __ldg(is + (idx >> ld)) : (int64_t)-1;
                k[j] = in_range(kr, w >> ld) ? (kr << ld) | (idx & (((int64_t)1 << ld) - 1)) : (int64_t)-1;
            }
        } else if (q * 4 + 4 <= n) {
            const longlong2 *pk = reinterpret_cast<const longlong2 *>(is) + 2 * q;
            const longlong2 a = ldg_hint_ll2(pk, strm), b = ldg_hint_ll2(pk + 1, strm);
            k[0] = a.x; k[1] = a.y; k[2] = b.x; k[3] = b.y;
            cnt = 4;
        } else {
            cnt = load_keys4(is, q * 4, n, k);
        }
        if (!VEC && cnt == 4) {
            const uint4 x = ldg_hint(reinterpret_cast<const uint4 *>(vs) + q, strm);
            v[0] = __uint_as_float(x.x); v[1] = __uint_as_float(x.y); v[2] = __uint_as_float(x.z); v[3] = __uint_as_float(x.w);
        } else {
            load_vals4(vs, q * 4, cnt, v);
        }
        // the four coefficient gathers are issued together (clamped index, unconditional load): one L2 round
        // trip per quad instead of four dependent ones (profiles/r2c: 32 long-scoreboard stall cycles per issue)
        if constexpr (SMEM) {
            float2 c[4];
#pragma unroll
            for (int j = 0; j < 4; j++) c[j] = sh[in_range(k[j], w) ? k[j] : 0];
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int z = __float_as_int(c[j].y);
                float r = 0.f;
                if (z == 0) r = c[j].x / v[j];
                else if (z == 1 && v[j] == 0.f) r = c[j].x;
                o[j] = in_range(k[j], w) ? r : 0.f;
            }
        } else {
            // Wide histograms: the table comes through L1 / L2.  Two planes of w floats instead of (c, zero class) pairs:
            // plane 0 = (z == 0 ? c : 0) is all a non-zero element needs (adjoint = plane0 / v: 0 as soon as its bin holds
            // a zero) -- a 4-byte gather from a table of 256 KB at w = 2^16 (pairs: 512 KB against ~200 KB of L1), its
            // address a function of the key alone; only an element that is 0 itself reads plane 1 = (z == 1 ? c : 0).
            const float *pl = reinterpret_cast<const float *>(coef);
            float c[4];
#pragma unroll
            for (int j = 0; j < 4; j++) c[j] = __ldg(pl + (in_range(k[j], w) ? k[j] : 0));
#pragma unroll
            for (int j = 0; j < 4; j++) {
                float r = 0.f;
                if (v[j] == 0.f) {  // IEEE equality: +-0 only (Q7); rare
                    if (in_range(k[j], w)) r = __ldg(pl + w + k[j]);
                } else if (c[j] != 0.f) {
                    r = c[j] / v[j];
                }
                o[j] = in_range(k[j], w) ? r : 0.f;
            }
        }
        if (!VEC && cnt == 4 && accumulate == 0)
            stg_hint(reinterpret_cast<uint4 *>(vs_bar) + q,
                     make_uint4(__float_as_uint(o[0]), __float_as_uint(o[1]), __float_as_uint(o[2]), __float_as_uint(o[3])), strm);
        else
            store_adj4(vs_bar, q * 4, cnt, o, accumulate != 0);
    }
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

bool rbi_mul_vec_fused(int64_t n, int64_t w, int ld) {
    return ld > 0 && ld < 12 && cached_walk(w << ld) && (n << ld) < (int64_t)0xfffffffell;
}

// ld > 0: n, w, vs, hist_bar, vs_bar are the FLAT sizes / arrays of `map2 (*)` on rows of 2^ld scalars, `is` has
// n >> ld keys (rbi_mul_vec_fused says whether this form is available).
int launch_rbi_mul(int64_t n, int64_t w, const int64_t *is, const float *vs,
                   const float *hist_bar, float *vs_bar, int64_t *zeros, float *prod_nz, void *ws,
                   int accumulate, cudaStream_t stream, int ld) {
    if (w == 0) {
        if (vs_bar && n > 0 && !accumulate &&
            cudaMemsetAsync(vs_bar, 0, (size_t)n * sizeof(float), stream) != cudaSuccess)
            return VJP_ERR_CUDA;
        return VJP_OK;
    }
    if (!rbi_cached_supported(w)) return VJP_ERR_UNSUPPORTED;
    MulWs m = mul_carve(ws, w);
    if (cudaMemsetAsync(m.zeros, 0, (size_t)w * 4, stream) != cudaSuccess) return VJP_ERR_CUDA;
    int G = 0;
    const int rc = run_cached<ACC_MUL, true>(n, w, is, vs, m.part, m.zeros, 0.f, &G, stream, ld);
    if (rc != VJP_OK) return rc;
    const int planes = ld == 0 && (size_t)w * sizeof(float2) > GATHER_SMEM_MAX / 2;  // the sweep's table form
    if (fold_chains(G) == 32)
        VJP_LAUNCH(K_MUL_FINISH, stream) rbi_mul_finish_kernel<32><<<fold_grid(w), 1024, 0, stream>>>(w, G, m.part, m.zeros, hist_bar, zeros, prod_nz,
                                                                                              vs_bar ? m.coef : nullptr, planes);
    else
        VJP_LAUNCH(K_MUL_FINISH, stream) rbi_mul_finish_kernel<8><<<fold_grid(w), 256, 0, stream>>>(w, G, m.part, m.zeros, hist_bar, zeros, prod_nz,
                                                                                            vs_bar ? m.coef : nullptr, planes);
    if (vs_bar && n > 0) {
        const int grid = grid_for(n, RBI_NT, RBI_CTAS_PER_SM);
        const size_t bytes = (size_t)w * sizeof(float2);
        if (ld > 0) {  // w <= 12288 virtual bins: 96 KB of coefficients at most
            auto kern = rbi_mul_sweep_kernel<true, true>;
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 12288 * 8) != cudaSuccess) return VJP_ERR_CUDA;
            VJP_LAUNCH(K_MUL_SWEEP, stream) kern<<<bytes > 48 * 1024 ? NUM_SMS_B200 * 2 : grid, RBI_NT, bytes, stream>>>(n, w, is, vs, m.coef, vs_bar, accumulate, ld);
        } else if (bytes <= GATHER_SMEM_MAX / 2)
            VJP_LAUNCH(K_MUL_SWEEP, stream) rbi_mul_sweep_kernel<true><<<grid, RBI_NT, bytes, stream>>>(n, w, is, vs, m.coef, vs_bar, accumulate);
        else
            VJP_LAUNCH(K_MUL_SWEEP, stream) rbi_mul_sweep_kernel<false><<<grid, RBI_NT, 0, stream>>>(n, w, is, vs, m.coef, vs_bar, accumulate);
    }
    return last_launch_status();
}

// Workspace of the specialised rules; covers reduce_by_index_forward of the same operator too.
size_t rbi_special_workspace_bytes(int code, int, int64_t n, int64_t w) {
    if (w < 1) w = 1;
    switch (code) {
    case VJP_OP_MIN:
    case VJP_OP_MAX: return minmax_ws_bytes(w);
    case VJP_OP_MUL:
        return align_up((size_t)w * 4, 256) + align_up((size_t)w * 8, 256) + cached_part_bytes(n, w);
    default: return 256;
    }
}
size_t rbi_forward_workspace_bytes(int code, int64_t n, int64_t w) {
    if (code == VJP_OP_MUL || code == VJP_OP_SATADD) return cached_part_bytes(n, w);
    if (code == VJP_OP_MIN || code == VJP_OP_MAX) return minmax_ws_bytes(w < 1 ? 1 : w);
    return 256;
}

}  // namespace vjp
