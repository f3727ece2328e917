// rbi_general.cu -- the general-case rule for reduce-by-index (Fig. 4, eq. 5):
//
//   (sks, siota) = radix sort of (clamped key, iota)            P:L350-351, P:L396   G1
//   svs          = values carried through the sort as payload   P:L396               G2
//   segment flags from adjacent sorted keys (never stored)      P:L352-355           G3
//   ls = forward segmented exclusive scan of svs                P:L356, P:L400       G4
//   rs = reverse segmented exclusive scan of svs                P:L357-358, P:L402   G5
//   sv_bar_j = d(l_j (.) x (.) r_j)/dx at svs_j  *  hist_bar[sks_j]   (0 if out of range)  G6
//   vs_bar[siota_j] = sv_bar_j                                  P:L365-367           G7
//
// G1-G2: stable LSD radix sort over the ceil(log2(w+1)) key bits only, each pass = per-tile digit
// histogram, one exclusive scan over the [digit][tile] table, and a ranking + scatter kernel
// (warp-level match ranking keeps equal digits in input order).  G4 and G5-G7 are single-pass
// decoupled-look-back segmented scans whose (status, segment flag, value) triple fits one 64-bit
// word; G5-G7 are fused into one kernel.  Keys outside [0,w) are clamped to w (Q18): they sort
// behind every bin, in input order, and receive adjoint 0.
#include <math_constants.h>

#include "common.cuh"
#include "gen_ops.cuh"
#include "internal.h"

namespace vjp {

// ------------------------------------------------------------------ packed look-back ------
// word = status (bits 62-63) | payload (bits 0-32: value bits 0-31, segment flag bit 32)

enum : uint64_t { PK_EMPTY = 0, PK_AGG = 1, PK_PREFIX = 2 };
constexpr uint64_t PK_PAYLOAD = (1ull << 33) - 1;

VJP_DEVINL uint64_t ld_relaxed_u64(const uint64_t *p) {
    uint64_t v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
VJP_DEVINL uint64_t shfl_u64(uint64_t v, int src) {
    const uint32_t lo = __shfl_sync(FULL_MASK, (uint32_t)v, src);
    const uint32_t hi = __shfl_sync(FULL_MASK, (uint32_t)(v >> 32), src);
    return ((uint64_t)hi << 32) | lo;
}

// Exclusive scan of one payload per thread in processing order (REVT: thread NT-1 first).
template <int NT, bool REVT, class F>
VJP_DEVINL uint64_t block_exclusive_u64(uint64_t local, uint64_t &total, uint64_t ident, F comb,
                                        uint64_t *scratch /* NT/32 + 1 */) {
    constexpr int NW = NT / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int plane = REVT ? 31 - lane : lane;
    const int pwarp = REVT ? NW - 1 - warp : warp;
    __syncthreads();
    uint64_t incl = local;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint64_t o = shfl_u64(incl, REVT ? lane + off : lane - off);
        if (plane >= off) incl = comb(o, incl);
    }
    uint64_t ex = shfl_u64(incl, REVT ? lane + 1 : lane - 1);
    if (plane == 0) ex = ident;
    if (plane == 31) scratch[pwarp] = incl;
    __syncthreads();
    if (warp == 0) {
        const uint64_t wt = lane < NW ? scratch[lane] : ident;
        uint64_t wi = wt;
#pragma unroll
        for (int off = 1; off < NW; off <<= 1) {
            const uint64_t o = shfl_u64(wi, lane - off);
            if (lane >= off) wi = comb(o, wi);
        }
        uint64_t wex = shfl_u64(wi, lane - 1);
        if (lane == 0) wex = ident;
        __syncwarp();
        if (lane < NW) scratch[lane] = wex;
        if (lane == NW - 1) scratch[NW] = wi;
    }
    __syncthreads();
    total = scratch[NW];
    if (pwarp > 0) ex = comb(scratch[pwarp], ex);
    return ex;
}

// Called by warp 0.  Publishes the tile aggregate, folds the predecessors, publishes the inclusive
// prefix, returns the exclusive prefix of tile p (processing order).
template <class F>
VJP_DEVINL uint64_t packed_tile_prefix(uint64_t *status, int p, uint64_t total, uint64_t ident,
                                       F comb) {
    const int lane = threadIdx.x & 31;
    if (p == 0) {
        if (lane == 0) st_relaxed_u64(status, (PK_PREFIX << 62) | total);
        return ident;
    }
    if (lane == 0) st_relaxed_u64(status + p, (PK_AGG << 62) | total);
    uint64_t acc = ident;
    int base = p - 1;
    while (true) {
        const int q = base - lane;
        uint64_t word = (PK_PREFIX << 62) | ident;
        if (q >= 0) word = ld_relaxed_u64(status + q);
        while (__any_sync(FULL_MASK, (word >> 62) == PK_EMPTY)) {
            if ((word >> 62) == PK_EMPTY) {
                __nanosleep(32);
                word = ld_relaxed_u64(status + q);
            }
        }
        const unsigned pm = __ballot_sync(FULL_MASK, (word >> 62) == PK_PREFIX);
        const int first = __ffs(pm) - 1;
        uint64_t s = (first < 0 || lane <= first) ? (word & PK_PAYLOAD) : ident;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint64_t o = shfl_u64(s, lane + off);
            if (lane + off < 32) s = comb(o, s);
        }
        s = shfl_u64(s, 0);
        acc = comb(s, acc);
        if (pm != 0) break;
        base -= 32;
    }
    if (lane == 0) st_relaxed_u64(status + p, (PK_PREFIX << 62) | comb(acc, total));
    return acc;
}

// ------------------------------------------------------------------ u32 exclusive scan ----
// of the [digit][tile] histogram table.

struct AddComb {
    VJP_DEVINL uint64_t operator()(uint64_t a, uint64_t b) const { return (uint32_t)(a + b); }
};
constexpr int US_NT = 256, US_IPT = 8;

__global__ void __launch_bounds__(US_NT)
u32_exclusive_scan_kernel(uint32_t *data, int64_t m, int *ticket, uint64_t *status) {
    __shared__ uint64_t scratch[US_NT / 32 + 2];
    __shared__ int s_p;
    if (threadIdx.x == 0) s_p = atomicAdd(ticket, 1);
    __syncthreads();
    const int p = s_p;
    const int64_t base = (int64_t)p * (US_NT * US_IPT) + threadIdx.x * US_IPT;
    uint32_t v[US_IPT];
    uint32_t sum = 0;
    if (base + US_IPT <= m) {
        const uint4 a = *reinterpret_cast<const uint4 *>(data + base);
        const uint4 b = *reinterpret_cast<const uint4 *>(data + base + 4);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    } else {
#pragma unroll
        for (int j = 0; j < US_IPT; j++) v[j] = (base + j < m) ? data[base + j] : 0u;
    }
#pragma unroll
    for (int j = 0; j < US_IPT; j++) sum += v[j];
    uint64_t total;
    uint64_t ex = block_exclusive_u64<US_NT, false>(sum, total, 0ull, AddComb(), scratch);
    if (threadIdx.x < 32) {
        const uint64_t pre = packed_tile_prefix(status, p, total, 0ull, AddComb());
        if (threadIdx.x == 0) scratch[US_NT / 32 + 1] = pre;
    }
    __syncthreads();
    uint32_t run = (uint32_t)(scratch[US_NT / 32 + 1] + ex);
#pragma unroll
    for (int j = 0; j < US_IPT; j++) {
        const uint32_t c = v[j];
        v[j] = run;
        run += c;
    }
    if (base + US_IPT <= m) {
        *reinterpret_cast<uint4 *>(data + base) = make_uint4(v[0], v[1], v[2], v[3]);
        *reinterpret_cast<uint4 *>(data + base + 4) = make_uint4(v[4], v[5], v[6], v[7]);
    } else {
#pragma unroll
        for (int j = 0; j < US_IPT; j++)
            if (base + j < m) data[base + j] = v[j];
    }
}

// ------------------------------------------------------------------ radix sort passes -----

constexpr int SORT_NT = 256;
constexpr int SORT_IPT = 8;
constexpr int SORT_TILE = SORT_NT * SORT_IPT;  // 2048 keys; warp w owns keys [256 w, 256 w + 256)
constexpr int SORT_MAX_RADIX = 256;

// key' = k if 0 <= k < w else w (Q18)
VJP_DEVINL uint32_t clamp_key(int64_t k, int64_t w) {
    return (uint64_t)k < (uint64_t)w ? (uint32_t)k : (uint32_t)w;
}

template <bool FIRST>
VJP_DEVINL uint32_t sort_load_key(const int64_t *__restrict__ is, const uint32_t *__restrict__ kin,
                                  int64_t i, int64_t w) {
    return FIRST ? clamp_key(__ldg(is + i), w) : __ldg(kin + i);
}

template <bool FIRST>
__global__ void __launch_bounds__(SORT_NT)
sort_hist_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                 const uint32_t *__restrict__ kin, int shift, int radix, int num_tiles,
                 uint32_t *__restrict__ counts) {
    __shared__ uint32_t h[SORT_MAX_RADIX];
    for (int d = threadIdx.x; d < radix; d += SORT_NT) h[d] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * SORT_TILE;
    const uint32_t mask = (uint32_t)radix - 1;
#pragma unroll 4
    for (int j = 0; j < SORT_IPT; j++) {
        const int64_t i = base + j * SORT_NT + threadIdx.x;
        if (i < n) atomicAdd(&h[(sort_load_key<FIRST>(is, kin, i, w) >> shift) & mask], 1u);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < radix; d += SORT_NT)
        counts[(size_t)d * num_tiles + blockIdx.x] = h[d];
}

// Stable ranking + scatter.  In round j, lane l of warp wp holds key number 512 wp + 32 j + l of
// the tile, so "earlier in the input" = (lower warp, lower round, lower lane): the rank of a key
// among equal digits is  offset[warp][digit] + (keys of that digit in earlier rounds of the warp)
// + (lower lanes with that digit in this round).
// The tile is first reordered in shared memory (keys of one digit become contiguous), then written
// out with consecutive threads on consecutive positions: a warp's store touches a few 128-byte
// lines instead of 32 (the direct scatter spent its time in uncoalesced 4- and 8-byte stores,
// profiles/r1f: 19 % DRAM, long-scoreboard stalls).
constexpr size_t SORT_SCATTER_SMEM = (size_t)SORT_TILE * 12;

template <bool FIRST>
__global__ void __launch_bounds__(SORT_NT)
sort_scatter_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is,
                    const float *__restrict__ vs, int vstride, const uint32_t *__restrict__ kin,
                    const uint2 *__restrict__ pin, int shift, int radix, int num_tiles,
                    const uint32_t *__restrict__ offsets, uint32_t *__restrict__ kout,
                    uint2 *__restrict__ pout) {
    constexpr int NW = SORT_NT / 32;
    __shared__ uint32_t cnt[NW][SORT_MAX_RADIX];
    __shared__ uint32_t dstart[SORT_MAX_RADIX];  // tile-local start of every digit
    __shared__ uint32_t goff[SORT_MAX_RADIX];    // global start of (digit, tile) minus dstart
    __shared__ uint32_t wsum[NW];
    extern __shared__ uint4 sort_smem[];
    uint2 *spay = reinterpret_cast<uint2 *>(sort_smem);                 // [SORT_TILE]
    uint32_t *skey = reinterpret_cast<uint32_t *>(spay + SORT_TILE);   // [SORT_TILE]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int d = threadIdx.x; d < NW * SORT_MAX_RADIX; d += SORT_NT) (&cnt[0][0])[d] = 0;
    __syncthreads();
    const int64_t tbase = (int64_t)blockIdx.x * SORT_TILE;
    const int64_t wbase = tbase + warp * (32 * SORT_IPT);
    const uint32_t mask = (uint32_t)radix - 1;
    const unsigned lt = (1u << lane) - 1;
    uint32_t key[SORT_IPT];
    uint16_t rank[SORT_IPT];
#pragma unroll
    for (int j = 0; j < SORT_IPT; j++) {
        const int64_t i = wbase + j * 32 + lane;
        const bool valid = i < n;
        key[j] = valid ? sort_load_key<FIRST>(is, kin, i, w) : 0u;
        const unsigned vm = __ballot_sync(FULL_MASK, valid);
        if (valid) {
            const uint32_t d = (key[j] >> shift) & mask;
            const unsigned peers = __match_any_sync(vm, d);
            const uint32_t before = cnt[warp][d];
            __syncwarp(vm);
            if ((peers & lt) == 0) cnt[warp][d] = before + __popc(peers);
            __syncwarp(vm);
            rank[j] = (uint16_t)(before + __popc(peers & lt));
        }
    }
    __syncthreads();
    // one thread per digit (radix <= SORT_NT): exclusive prefix over the warps, then over the digits
    {
        const int d = threadIdx.x;
        uint32_t tot = 0;
        if (d < radix) {
#pragma unroll
            for (int x = 0; x < NW; x++) {
                const uint32_t c = cnt[x][d];
                cnt[x][d] = tot;
                tot += c;
            }
        }
        uint32_t incl = tot;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t o = __shfl_up_sync(FULL_MASK, incl, off);
            if (lane >= off) incl += o;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t wpre = 0;
#pragma unroll
        for (int x = 0; x < NW; x++) wpre += x < warp ? wsum[x] : 0u;
        if (d < radix) {
            const uint32_t ex = wpre + incl - tot;
            dstart[d] = ex;
            goff[d] = offsets[(size_t)d * num_tiles + blockIdx.x] - ex;
        }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < SORT_IPT; j++) {
        const int64_t i = wbase + j * 32 + lane;
        if (i < n) {
            const uint32_t d = (key[j] >> shift) & mask;
            const uint32_t lp = dstart[d] + cnt[warp][d] + rank[j];
            skey[lp] = key[j];
            spay[lp] = FIRST ? make_uint2((uint32_t)i, vs ? __float_as_uint(__ldg(vs + i * vstride)) : 0u)
                             : __ldg(pin + i);
        }
    }
    __syncthreads();
    const int tile_valid = (int)min((int64_t)SORT_TILE, n - tbase);
    for (int lp = threadIdx.x; lp < tile_valid; lp += SORT_NT) {
        const uint32_t k = skey[lp];
        const uint32_t pos = goff[(k >> shift) & mask] + (uint32_t)lp;
        kout[pos] = k;
        pout[pos] = spay[lp];
    }
}

// ------------------------------------------------------------------ operators: gen_ops.cuh

// Segmented-scan combine on payloads (flag << 32 | value bits).  REV: "earlier" holds the HIGHER
// indices, and the fold keeps index order: value = later (.) earlier.
template <int CODE, bool REV>
struct SegComb {
    GenOp<CODE> op;
    VJP_DEVINL uint64_t operator()(uint64_t earlier, uint64_t later) const {
        const float ve = __uint_as_float((uint32_t)earlier), vl = __uint_as_float((uint32_t)later);
        const bool fl = (later >> 32) & 1;
        const float v = fl ? vl : (REV ? op.apply(vl, ve) : op.apply(ve, vl));
        return (((earlier | later) >> 32) & 1) << 32 | __float_as_uint(v);
    }
};

// ------------------------------------------------------------------ segmented scans -------

constexpr int SEG_NT = 512;
constexpr int SEG_IPT = 8;
constexpr int SEG_TILE = SEG_NT * SEG_IPT;

// A thread's row of RW consecutive 32-bit words straight from / to global memory with 128-bit accesses: the
// row is 32 or 64 contiguous bytes, i.e. whole sectors, so nothing is gained by staging the tile through
// shared memory -- and the barriers around the staging were what these kernels waited on (profiles/r2d:
// 26 - 37 barrier stall cycles per issue, issue slots 12 - 19 % busy).  `valid` = words of the row that exist.
template <int RW>
VJP_DEVINL void load_row(const uint32_t *__restrict__ g, int valid, uint32_t fill, uint32_t (&r)[RW]) {
    if (valid >= RW) {
        const uint4 *g4 = reinterpret_cast<const uint4 *>(g);
#pragma unroll
        for (int c = 0; c < RW / 4; c++) {
            const uint4 v = __ldg(g4 + c);
            r[4 * c] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int i = 0; i < RW; i++) r[i] = i < valid ? __ldg(g + i) : fill;
    }
}
template <int RW>
VJP_DEVINL void store_row(uint32_t *__restrict__ g, int valid, const uint32_t (&r)[RW]) {
    if (valid >= RW) {
        uint4 *g4 = reinterpret_cast<uint4 *>(g);
#pragma unroll
        for (int c = 0; c < RW / 4; c++) g4[c] = make_uint4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
    } else {
#pragma unroll
        for (int i = 0; i < RW; i++)
            if (i < valid) g[i] = r[i];
    }
}

// G4: ls[j] = fold of the same-key elements before j (neutral at a segment head).
template <int CODE>
__global__ void __launch_bounds__(SEG_NT)
seg_forward_kernel(int64_t n, const uint32_t *__restrict__ keys, const uint2 *__restrict__ pay,
                   float *__restrict__ ls, GenOp<CODE> op, int *ticket, uint64_t *status) {
    __shared__ uint64_t scratch[SEG_NT / 32 + 2];
    __shared__ uint32_t last_key[SEG_NT];
    __shared__ int s_p;
    if (threadIdx.x == 0) s_p = atomicAdd(ticket, 1);
    __syncthreads();
    const int p = s_p;
    const int64_t base = (int64_t)p * SEG_TILE + threadIdx.x * SEG_IPT;  // this thread's first element
    const int mine = (int)max((int64_t)0, min((int64_t)SEG_IPT, n - base));  // elements of the row that exist
    uint32_t k[SEG_IPT], pw[2 * SEG_IPT];
    // padding: a key no element has (its own segment), value bits 0
    load_row<SEG_IPT>(keys + base, mine, 0xffffffffu, k);
    load_row<2 * SEG_IPT>(reinterpret_cast<const uint32_t *>(pay + base), 2 * mine, 0u, pw);
    last_key[threadIdx.x] = k[SEG_IPT - 1];
    __syncthreads();
    uint32_t prev;
    bool first_head = false;
    if (threadIdx.x > 0) prev = last_key[threadIdx.x - 1];
    else if (base > 0) prev = __ldg(keys + base - 1);
    else { prev = 0; first_head = true; }

    const SegComb<CODE, false> comb{op};
    const uint64_t ident = __float_as_uint(op.neutral());
    bool head[SEG_IPT];
    uint64_t acc = ident;
#pragma unroll
    for (int j = 0; j < SEG_IPT; j++) {
        head[j] = (j == 0) ? (first_head || k[0] != prev) : (k[j] != k[j - 1]);
        acc = comb(acc, ((uint64_t)head[j] << 32) | pw[2 * j + 1]);
    }
    uint64_t total;
    const uint64_t ex = block_exclusive_u64<SEG_NT, false>(acc, total, ident, comb, scratch);
    if (threadIdx.x < 32) {
        const uint64_t pre = packed_tile_prefix(status, p, total, ident, comb);
        if (threadIdx.x == 0) scratch[SEG_NT / 32 + 1] = pre;
    }
    __syncthreads();
    float run = __uint_as_float((uint32_t)comb(scratch[SEG_NT / 32 + 1], ex));
    uint32_t out[SEG_IPT];
#pragma unroll
    for (int j = 0; j < SEG_IPT; j++) {
        const float v = __uint_as_float(pw[2 * j + 1]);
        const float l = head[j] ? op.neutral() : run;
        out[j] = __float_as_uint(l);
        run = op.apply(l, v);
    }
    store_row<SEG_IPT>(reinterpret_cast<uint32_t *>(ls) + base, mine, out);
}

// G5-G7 fused: reverse segmented exclusive scan, per-element derivative, un-permute.
template <int CODE>
__global__ void __launch_bounds__(SEG_NT)
seg_reverse_vjp_kernel(int64_t n, int64_t w, const uint32_t *__restrict__ keys,
                       const uint2 *__restrict__ pay, const float *__restrict__ ls,
                       const float *__restrict__ hist_bar, float *__restrict__ vs_bar,
                       GenOp<CODE> op, int num_tiles, int *ticket, uint64_t *status, int accumulate) {
    __shared__ uint64_t scratch[SEG_NT / 32 + 2];
    __shared__ uint32_t first_key[SEG_NT];
    __shared__ int s_p;
    if (threadIdx.x == 0) s_p = atomicAdd(ticket, 1);
    __syncthreads();
    const int p = s_p;
    const int t = num_tiles - 1 - p;
    const int64_t tbase = (int64_t)t * SEG_TILE;
    const int64_t base = tbase + threadIdx.x * SEG_IPT;
    const int mine = (int)max((int64_t)0, min((int64_t)SEG_IPT, n - base));  // number of real elements in this row
    uint32_t k[SEG_IPT], lw[SEG_IPT], pw[2 * SEG_IPT];
    load_row<SEG_IPT>(keys + base, mine, 0xffffffffu, k);
    load_row<SEG_IPT>(reinterpret_cast<const uint32_t *>(ls) + base, mine, 0u, lw);
    load_row<2 * SEG_IPT>(reinterpret_cast<const uint32_t *>(pay + base), 2 * mine, 0u, pw);
    // the bin adjoints of the row: issued now, consumed after the scan
    float hb[SEG_IPT], hb2[CODE == G_SOP ? SEG_IPT : 1];  // G_SOP: hist_bar is [w][2] = (Pbar, Sbar)
#pragma unroll
    for (int j = 0; j < SEG_IPT; j++) {
        if constexpr (CODE == G_SOP) {
            const float2 h = k[j] < (uint32_t)w ? __ldg(reinterpret_cast<const float2 *>(hist_bar) + k[j]) : make_float2(0.f, 0.f);
            hb[j] = h.x;
            hb2[j] = h.y;
        } else {
            hb[j] = k[j] < (uint32_t)w ? __ldg(hist_bar + k[j]) : 0.f;
        }
    }
    first_key[threadIdx.x] = k[0];
    __syncthreads();
    uint32_t next;
    bool last_tail = false;
    if (threadIdx.x < SEG_NT - 1) next = first_key[threadIdx.x + 1];
    else if (tbase + SEG_TILE < n) next = __ldg(keys + tbase + SEG_TILE);
    else { next = 0; last_tail = true; }

    const SegComb<CODE, true> comb{op};
    const uint64_t ident = __float_as_uint(op.neutral());
    bool tail[SEG_IPT];  // segment boundary seen from the right
    uint64_t acc = ident;
#pragma unroll
    for (int j = SEG_IPT - 1; j >= 0; j--) {
        tail[j] = (j == SEG_IPT - 1) ? (last_tail || k[j] != next) : (k[j] != k[j + 1]);
        acc = comb(acc, ((uint64_t)tail[j] << 32) | pw[2 * j + 1]);
    }
    uint64_t total;
    const uint64_t ex = block_exclusive_u64<SEG_NT, true>(acc, total, ident, comb, scratch);
    if (threadIdx.x < 32) {
        const uint64_t pre = packed_tile_prefix(status, p, total, ident, comb);
        if (threadIdx.x == 0) scratch[SEG_NT / 32 + 1] = pre;
    }
    __syncthreads();
    float run = __uint_as_float((uint32_t)comb(scratch[SEG_NT / 32 + 1], ex));
#pragma unroll
    for (int j = SEG_IPT - 1; j >= 0; j--) {
        const float v = __uint_as_float(pw[2 * j + 1]);
        const float r = tail[j] ? op.neutral() : run;
        run = op.apply(v, r);
        if (j < mine) {
            // out-of-range keys were clamped to w: adjoint 0 (hb is 0 there)
            const float g = k[j] < (uint32_t)w ? op.dfdx(__uint_as_float(lw[j]), v, r) * hb[j] : 0.f;
            if constexpr (CODE == G_SOP) {  // vs_bar_i = (Pbar, Pbar * (ls + rs) + Sbar)
                float2 *dst = reinterpret_cast<float2 *>(vs_bar) + pw[2 * j];
                float2 o = make_float2(hb[j], g + hb2[j]);
                if (accumulate) {
                    const float2 pr = *dst;
                    o.x += pr.x;
                    o.y += pr.y;
                }
                *dst = o;
            } else {
                vs_bar[pw[2 * j]] = accumulate ? vs_bar[pw[2 * j]] + g : g;  // the permutation names every index once
            }
        }
    }
}

__global__ void sort_export_kernel(int64_t n, const uint32_t *__restrict__ keys,
                                   const uint2 *__restrict__ pay, int64_t *sorted_keys,
                                   int64_t *perm) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
         i += (int64_t)gridDim.x * blockDim.x) {
        sorted_keys[i] = keys[i];
        perm[i] = pay[i].x;
    }
}

// ------------------------------------------------------------------ host side -------------

struct GenWs {
    uint32_t *key[2];
    uint2 *pay[2];
    float *ls;
    uint32_t *counts;
    int *ticket;       // ticket + status words: zeroed before each look-back kernel
    uint64_t *status;
    size_t zero_bytes;
    size_t total;
};

static int64_t sort_tiles(int64_t n) { return (n + SORT_TILE - 1) / SORT_TILE; }
static int64_t seg_tiles(int64_t n) { return (n + SEG_TILE - 1) / SEG_TILE; }

static GenWs gen_carve(void *ws, int64_t n) {
    GenWs g;
    const size_t nn = (size_t)(n < 1 ? 1 : n);
    char *p = static_cast<char *>(ws);
    auto take = [&](size_t bytes) { char *r = p; p += align_up(bytes, 256); return r; };
    g.key[0] = reinterpret_cast<uint32_t *>(take(nn * 4));
    g.key[1] = reinterpret_cast<uint32_t *>(take(nn * 4));
    g.pay[0] = reinterpret_cast<uint2 *>(take(nn * 8));
    g.pay[1] = reinterpret_cast<uint2 *>(take(nn * 8));
    g.ls = reinterpret_cast<float *>(take(nn * 4));
    const size_t m = (size_t)SORT_MAX_RADIX * (size_t)sort_tiles(nn);
    g.counts = reinterpret_cast<uint32_t *>(take(m * 4));
    size_t lb_tiles = (m + US_NT * US_IPT - 1) / (US_NT * US_IPT);
    if ((size_t)seg_tiles(nn) > lb_tiles) lb_tiles = (size_t)seg_tiles(nn);
    g.zero_bytes = align_up(8 + 8 * lb_tiles, 256);
    char *z = take(g.zero_bytes);
    g.ticket = reinterpret_cast<int *>(z);
    g.status = reinterpret_cast<uint64_t *>(z + 8);
    g.total = (size_t)(p - static_cast<char *>(ws));
    return g;
}

// one query serves both routes of the general rule (sort-based: here; sort-free: rbi_multiscan.cu)
size_t rbi_general_workspace_bytes(int64_t n, int64_t w) {
    const size_t a = gen_carve(nullptr, n).total, b = rbi_multiscan_workspace_bytes(n, w);
    return a > b ? a : b;
}

// Sorts (clamped key, (index, value)); returns the buffer index holding the result in *out_buf.
static int run_sort(int64_t n, int64_t w, const int64_t *is, const float *vs, const GenWs &g,
                    int *out_buf, cudaStream_t stream, int vstride = 1) {
    if (cudaFuncSetAttribute(sort_scatter_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)SORT_SCATTER_SMEM) != cudaSuccess ||
        cudaFuncSetAttribute(sort_scatter_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)SORT_SCATTER_SMEM) != cudaSuccess)
        return VJP_ERR_CUDA;
    int bits = 0;
    while (bits < 32 && ((uint64_t)w >> bits) != 0) bits++;  // keys are 0..w
    if (bits < 1) bits = 1;
    if (bits > 32) return VJP_ERR_UNSUPPORTED;
    const int passes = (bits + 7) / 8;
    const int per = (bits + passes - 1) / passes;
    const int nt = (int)sort_tiles(n);
    int shift = 0, src = -1;
    for (int ps = 0; ps < passes; ps++) {
        const int b = (bits - shift) < per ? (bits - shift) : per;
        const int radix = 1 << b;
        const int dst = ps & 1;
        const int64_t m = (int64_t)radix * nt;
        if (ps == 0)
            VJP_LAUNCH(K_SORT_HIST, stream) sort_hist_kernel<true><<<nt, SORT_NT, 0, stream>>>(n, w, is, nullptr, shift, radix, nt, g.counts);
        else
            VJP_LAUNCH(K_SORT_HIST, stream) sort_hist_kernel<false><<<nt, SORT_NT, 0, stream>>>(n, w, nullptr, g.key[src], shift, radix, nt, g.counts);
        if (cudaMemsetAsync(g.ticket, 0, g.zero_bytes, stream) != cudaSuccess) return VJP_ERR_CUDA;
        const int sb = (int)((m + US_NT * US_IPT - 1) / (US_NT * US_IPT));
        VJP_LAUNCH(K_U32_SCAN, stream) u32_exclusive_scan_kernel<<<sb, US_NT, 0, stream>>>(g.counts, m, g.ticket, g.status);
        if (ps == 0)
            VJP_LAUNCH(K_SORT_SCATTER, stream) sort_scatter_kernel<true><<<nt, SORT_NT, SORT_SCATTER_SMEM, stream>>>(n, w, is, vs, vstride, nullptr, nullptr, shift, radix,
                                                                  nt, g.counts, g.key[dst], g.pay[dst]);
        else
            VJP_LAUNCH(K_SORT_SCATTER, stream) sort_scatter_kernel<false><<<nt, SORT_NT, SORT_SCATTER_SMEM, stream>>>(n, w, nullptr, nullptr, 1, g.key[src],
                                                                   g.pay[src], shift, radix, nt, g.counts,
                                                                   g.key[dst], g.pay[dst]);
        src = dst;
        shift += b;
    }
    *out_buf = src;
    return last_launch_status();
}

// G3-G7 on sorted (key, (index, value)) arrays: forward segmented scan, fused reverse scan + derivative + scatter.
template <int CODE>
static int run_segscans(float S, int64_t n, int64_t w, const uint32_t *keys, const uint2 *pay,
                        const float *hist_bar, float *vs_bar, const GenWs &g, int accumulate, cudaStream_t stream) {
    const GenOp<CODE> op{S};
    const int nt = (int)seg_tiles(n);
    if (cudaMemsetAsync(g.ticket, 0, g.zero_bytes, stream) != cudaSuccess) return VJP_ERR_CUDA;
    VJP_LAUNCH(K_SEG_FORWARD, stream) seg_forward_kernel<CODE><<<nt, SEG_NT, 0, stream>>>(
        n, keys, pay, g.ls, op, g.ticket, g.status);
    if (cudaMemsetAsync(g.ticket, 0, g.zero_bytes, stream) != cudaSuccess) return VJP_ERR_CUDA;
    VJP_LAUNCH(K_SEG_REVERSE, stream) seg_reverse_vjp_kernel<CODE><<<nt, SEG_NT, 0, stream>>>(
        n, w, keys, pay, g.ls, hist_bar, vs_bar, op, nt, g.ticket, g.status, accumulate);
    return last_launch_status();
}

template <int CODE>
static int run_general(float S, int64_t n, int64_t w, const int64_t *is, const float *vs,
                       const float *hist_bar, float *vs_bar, const GenWs &g, int accumulate, cudaStream_t stream) {
    int buf;
    int rc = run_sort(n, w, is, vs, g, &buf, stream);
    if (rc != VJP_OK) return rc;
    return run_segscans<CODE>(S, n, w, g.key[buf], g.pay[buf], hist_bar, vs_bar, g, accumulate, stream);
}

// sumOfProd through the general rule (Fig. 4): sort by bin with the s component as payload, segmented exclusive
// '+' scans of s forwards and backwards, vs_bar_i = (Pbar, Pbar * (ls_i + rs_i) + Sbar).
int launch_rbi_sop_general_vjp(int64_t n, int64_t w, const int64_t *is, const float *vs, const float *hist_bar,
                               float *vs_bar, void *ws, int accumulate, int sorted, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    if (!sorted && rbi_multiscan_fits(w))
        return launch_rbi_multiscan_vjp(G_SOP, 0.0, n, w, is, vs, hist_bar, vs_bar, ws, accumulate, stream);
    const GenWs g = gen_carve(ws, n);
    int buf;
    const int rc = run_sort(n, w, is, vs + 1, g, &buf, stream, 2);
    if (rc != VJP_OK) return rc;
    return run_segscans<G_SOP>(0.f, n, w, g.key[buf], g.pay[buf], hist_bar, vs_bar, g, accumulate, stream);
}

// reduce, general rule (eq. 2; Fig. 2): ls = forward exclusive scan, rs = reverse exclusive
// scan, as_bar_i = d(l_i (.) a_i (.) r_i)/da_i * y_bar -- the segmented-scan pair above with ONE segment
// (every key 0, the identity permutation as payload index) and no sort; y_bar plays hist_bar[0].
__global__ void reduce_pack_kernel(int64_t n, const float *__restrict__ xs, uint32_t *__restrict__ keys,
                                   uint2 *__restrict__ pay) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        keys[i] = 0u;
        pay[i] = make_uint2((uint32_t)i, __float_as_uint(__ldg(xs + i)));
    }
}

int launch_reduce_general_vjp(int code, double param, int64_t n, const float *xs, const float *y_bar,
                              float *xs_bar, void *ws, int accumulate, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    const GenWs g = gen_carve(ws, n);
    const float S = (float)param;
    const int grid = (int)((n + 255) / 256 < 2368 ? (n + 255) / 256 : 2368);
    VJP_LAUNCH(K_REDUCE_PACK, stream) reduce_pack_kernel<<<grid, 256, 0, stream>>>(n, xs, g.key[0], g.pay[0]);
    switch (code) {
    case VJP_OP_ADD: return run_segscans<G_ADD>(S, n, 1, g.key[0], g.pay[0], y_bar, xs_bar, g, accumulate, stream);
    case VJP_OP_MIN: return run_segscans<G_MIN>(S, n, 1, g.key[0], g.pay[0], y_bar, xs_bar, g, accumulate, stream);
    case VJP_OP_MAX: return run_segscans<G_MAX>(S, n, 1, g.key[0], g.pay[0], y_bar, xs_bar, g, accumulate, stream);
    case VJP_OP_MUL: return run_segscans<G_MUL>(S, n, 1, g.key[0], g.pay[0], y_bar, xs_bar, g, accumulate, stream);
    case VJP_OP_SATADD: return run_segscans<G_SATADD>(S, n, 1, g.key[0], g.pay[0], y_bar, xs_bar, g, accumulate, stream);
    default: return VJP_ERR_UNSUPPORTED;
    }
}

// sorted != 0: Fig. 4 as written (sort + segmented scans); else the sort-free walks of rbi_multiscan.cu when a bin
// table fits a warp's share of shared memory (w <= 12 288), the sort-based route otherwise.
int launch_rbi_general_vjp(int code, double param, int64_t n, int64_t w, const int64_t *is,
                           const float *vs, const float *hist_bar, float *vs_bar, void *ws,
                           int accumulate, int sorted, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    if (!sorted && rbi_multiscan_fits(w)) {
        int gc;
        switch (code) {
        case VJP_OP_ADD: gc = G_ADD; break;
        case VJP_OP_MIN: gc = G_MIN; break;
        case VJP_OP_MAX: gc = G_MAX; break;
        case VJP_OP_MUL: gc = G_MUL; break;
        case VJP_OP_SATADD: gc = G_SATADD; break;
        default: return VJP_ERR_UNSUPPORTED;
        }
        return launch_rbi_multiscan_vjp(gc, param, n, w, is, vs, hist_bar, vs_bar, ws, accumulate, stream);
    }
    const GenWs g = gen_carve(ws, n);
    const float S = (float)param;
    switch (code) {
    case VJP_OP_ADD: return run_general<G_ADD>(S, n, w, is, vs, hist_bar, vs_bar, g, accumulate, stream);
    case VJP_OP_MIN: return run_general<G_MIN>(S, n, w, is, vs, hist_bar, vs_bar, g, accumulate, stream);
    case VJP_OP_MAX: return run_general<G_MAX>(S, n, w, is, vs, hist_bar, vs_bar, g, accumulate, stream);
    case VJP_OP_MUL: return run_general<G_MUL>(S, n, w, is, vs, hist_bar, vs_bar, g, accumulate, stream);
    case VJP_OP_SATADD: return run_general<G_SATADD>(S, n, w, is, vs, hist_bar, vs_bar, g, accumulate, stream);
    default: return VJP_ERR_UNSUPPORTED;
    }
}

int launch_rbi_sort_perm(int64_t n, int64_t w, const int64_t *is, int64_t *sorted_keys,
                         int64_t *perm, void *ws, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    const GenWs g = gen_carve(ws, n);
    int buf;
    int rc = run_sort(n, w, is, nullptr, g, &buf, stream);
    if (rc != VJP_OK) return rc;
    const int grid = (int)((n + 255) / 256 < 2368 ? (n + 255) / 256 : 2368);
    VJP_LAUNCH(K_SORT_EXPORT, stream) sort_export_kernel<<<grid, 256, 0, stream>>>(n, g.key[buf], g.pay[buf], sorted_keys, perm);
    return last_launch_status();
}

}  // namespace vjp
