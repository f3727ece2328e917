// common.cuh -- device-side building blocks shared by every kernel of the library:
// word-wise warp shuffles of arbitrary POD states, ordered block scans of a monoid,
// the decoupled look-back protocol, and row-padded shared-memory tile staging with
// 128-bit global accesses.  sm_100a only.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace vjp {

constexpr unsigned FULL_MASK = 0xffffffffu;
constexpr int NUM_SMS_B200 = 148;

#define VJP_DEVINL __device__ __forceinline__

// ------------------------------------------------------------------ memory ordering ----

// streaming 128-bit accesses (data touched once: do not keep it in L1)
VJP_DEVINL uint4 ldg_stream(const uint4 *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
VJP_DEVINL void stg_stream(uint4 *p, const uint4 &v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x),
                 "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}

// L2 eviction hints for the lifted primal of '*' and the return sweep over the same (is, vs) that follows it.  The primal's
// 128-bit streaming loads carry an explicit evict_normal policy -- plain ld.global.nc.L1::no_allocate lines do not stay in
// L2 long enough for the sweep to meet them -- and the sweep reads and writes evict_first.  '*' VJP at w = 2^10 with L2
// flushed between calls (fresh inputs): 0.120 -> 0.112 ms uniform, 0.130 -> 0.118 ms Zipf; back to back 0.115 -> 0.113,
// 0.123 -> 0.119 ms (the sweep 44.9 -> 35.3 us, the primal + 4 us: it no longer meets lines the previous call's sweep
// left).  An evict_last fraction (0.4, 0.55) on the primal added nothing.  NOT used in the scan kernels: the same hint on
// every streaming load cost the scan primals 3-8 % (5x5: 0.327 -> 0.409 ms; written lines compete with the kept ones), on
// the forward pass of a scan VJP alone it moved the VJP by +-2 %, evict_first in the reverse scan kernel cost 1-5 %; in the
// sumOfProd kernels the effect was inside the run-to-run spread (+-5 % between processes).
VJP_DEVINL uint64_t l2_policy_stream() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
VJP_DEVINL uint64_t l2_policy_normal() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
VJP_DEVINL longlong2 ldg_hint_ll2(const longlong2 *p, uint64_t pol) {
    longlong2 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.s64 {%0,%1}, [%2], %3;" : "=l"(r.x), "=l"(r.y) : "l"(p), "l"(pol));
    return r;
}
VJP_DEVINL uint4 ldg_hint(const uint4 *p, uint64_t pol) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p), "l"(pol));
    return r;
}
VJP_DEVINL void stg_hint(uint4 *p, const uint4 &v, uint64_t pol) {
    asm volatile("st.global.L1::no_allocate.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y),
                 "r"(v.z), "r"(v.w), "l"(pol)
                 : "memory");
}

// ------------------------------------------------------------------ POD word helpers ---

// Copy a POD state to / from global memory through L2 (look-back payloads: written once by one
// block, read by others after an acquire on the tile's flag).
template <class S>
VJP_DEVINL void store_state_cg(S *dst, const S &s) {
    static_assert(sizeof(S) % 4 == 0, "state must be a whole number of 32-bit words");
    constexpr int W = sizeof(S) / 4;
    const uint32_t *a = reinterpret_cast<const uint32_t *>(&s);
    uint32_t *d = reinterpret_cast<uint32_t *>(dst);
#pragma unroll
    for (int i = 0; i < W; i++) __stcg(d + i, a[i]);
}
template <class S>
VJP_DEVINL S load_state_cg(const S *src) {
    constexpr int W = sizeof(S) / 4;
    S r;
    uint32_t *b = reinterpret_cast<uint32_t *>(&r);
    const uint32_t *p = reinterpret_cast<const uint32_t *>(src);
#pragma unroll
    for (int i = 0; i < W; i++) b[i] = __ldcg(p + i);
    return r;
}
template <class S>
VJP_DEVINL S shfl_state(const S &s, int src_lane) {
    constexpr int W = sizeof(S) / 4;
    S r;
    const uint32_t *a = reinterpret_cast<const uint32_t *>(&s);
    uint32_t *b = reinterpret_cast<uint32_t *>(&r);
#pragma unroll
    for (int i = 0; i < W; i++) b[i] = __shfl_sync(FULL_MASK, a[i], src_lane);
    return r;
}
template <class S>
VJP_DEVINL void store_state_smem(uint32_t *dst, const S &s) {
    constexpr int W = sizeof(S) / 4;
    const uint32_t *a = reinterpret_cast<const uint32_t *>(&s);
#pragma unroll
    for (int i = 0; i < W; i++) dst[i] = a[i];
}
template <class S>
VJP_DEVINL S load_state_smem(const uint32_t *src) {
    constexpr int W = sizeof(S) / 4;
    S r;
    uint32_t *b = reinterpret_cast<uint32_t *>(&r);
#pragma unroll
    for (int i = 0; i < W; i++) b[i] = src[i];
    return r;
}

// ------------------------------------------------------------------ ordered block scan -
//
// A monoid M provides   typename M::State (POD, whole words),
//                       static State identity(),
//                       static State combine(const State& earlier, const State& later).
// "earlier / later" refer to PROCESSING order.  With REVT = false thread t has processing rank
// t; with REVT = true thread t has rank NT-1-t (a scan that runs from the end of the tile).

struct NoHook { VJP_DEVINL void operator()(const uint32_t *) const {} };

template <class M, int NT>
struct BlockScan {
    using S = typename M::State;
    static constexpr int NW = NT / 32;
    static constexpr int SW = sizeof(S) / 4;
    // shared scratch: NW warp totals + 1 block total, as words
    static constexpr int SMEM_WORDS = (NW + 1) * SW;

    // Exclusive scan of one state per thread.  Returns the exclusive prefix of this thread
    // (within the block) and the block total in `total` (valid in every thread).
    // ENTRY_SYNC = false: the caller knows that nobody can still be reading `scratch` (the first scan of a CTA)
    // after_total(words): called by all lanes of warp 0 as soon as the block total sits in shared memory, one barrier
    // before every thread has it (the look-back kernels publish their tile aggregate from there)
    template <bool REVT, bool ENTRY_SYNC = true, class Hook = NoHook>
    static VJP_DEVINL S exclusive(const S &local, S &total, uint32_t *scratch, Hook after_total = Hook()) {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int plane = REVT ? 31 - lane : lane;
        const int pwarp = REVT ? NW - 1 - warp : warp;
        if (ENTRY_SYNC) __syncthreads();  // scratch may still be read by a previous call
        S incl = local;
        // wide states (25- and 50-word 5x5 states): keep the loop rolled -- fully unrolled, the 5x5
        // VJP kernel was 11 400 instructions (182 KB), more than the instruction cache holds, and
        // ran at 0.17 IPC with "no instruction" stalls (profiles/r1f)
#pragma unroll(SW > 16 ? 1 : 5)
        for (int off = 1; off < 32; off <<= 1) {
            S o = shfl_state(incl, REVT ? lane + off : lane - off);
            if (plane >= off) incl = M::combine(o, incl);
        }
        // exclusive within the warp
        S ex = shfl_state(incl, REVT ? lane + 1 : lane - 1);
        if (plane == 0) ex = M::identity();
        if (plane == 31) store_state_smem(scratch + pwarp * SW, incl);
        __syncthreads();
        if (warp == 0) {
            // lane l holds the total of processing-warp l; Kogge-Stone over NW lanes
            S wt = (lane < NW) ? load_state_smem<S>(scratch + lane * SW) : M::identity();
            S wi = wt;
#pragma unroll(SW > 16 ? 1 : 5)
            for (int off = 1; off < NW; off <<= 1) {
                S o = shfl_state(wi, lane - off);
                if (lane >= off) wi = M::combine(o, wi);
            }
            S wex = shfl_state(wi, lane - 1);
            if (lane == 0) wex = M::identity();
            __syncwarp();
            if (lane < NW) store_state_smem(scratch + lane * SW, wex);
            if (lane == NW - 1) store_state_smem(scratch + NW * SW, wi);
            __syncwarp();
            after_total(scratch + NW * SW);
        }
        __syncthreads();
        total = load_state_smem<S>(scratch + NW * SW);
        if (pwarp > 0) {
            S wp = load_state_smem<S>(scratch + pwarp * SW);
            ex = M::combine(wp, ex);
        }
        return ex;
    }
};

// Two independent exclusive scans of one block in ONE pass: scan A runs from the END of the tile (thread t has
// processing rank NT-1-t, as BlockScan with REVT), scan B from its start.  They share every barrier -- three instead
// of six per tile -- and the two cross-warp scans run side by side in warps 0 and 1.  The reverse kernel of the scan
// VJP needs exactly this pair (the reverse lin_o scan and the forward prefixes); ncu showed its warps mostly waiting
// at barriers (2x2: 6.6 of 16 stall cycles per issue).
template <class MA, class MB, int NT>
struct BlockScanDual {
    using SA = typename MA::State;
    using SB = typename MB::State;
    static constexpr int NW = NT / 32, WA = sizeof(SA) / 4, WB = sizeof(SB) / 4;
    static constexpr int SMEM_WORDS = (NW + 1) * (WA + WB);
    static_assert(NW >= 2, "two warps run the cross-warp scans");

    template <class M, class S>
    static VJP_DEVINL void cross_warp(uint32_t *tot, int lane) {  // tot[w] = total of processing-warp w -> its exclusive prefix
        constexpr int SW = sizeof(S) / 4;
        S wt = (lane < NW) ? load_state_smem<S>(tot + lane * SW) : M::identity();
        S wi = wt;
#pragma unroll
        for (int off = 1; off < NW; off <<= 1) {
            S o = shfl_state(wi, lane - off);
            if (lane >= off) wi = M::combine(o, wi);
        }
        S wex = shfl_state(wi, lane - 1);
        if (lane == 0) wex = M::identity();
        __syncwarp();
        if (lane < NW) store_state_smem(tot + lane * SW, wex);
        if (lane == NW - 1) store_state_smem(tot + NW * SW, wi);
    }

    // after_total_a(words): called by all lanes of warp 0 as soon as scan A's block total sits in shared memory (one
    // barrier before every thread has it): the reverse scan kernel publishes its tile aggregate from there
    template <bool ENTRY_SYNC = true, class Hook = NoHook>
    static VJP_DEVINL void exclusive(const SA &la, SA &ta, SA &exa, const SB &lb, SB &tb, SB &exb, uint32_t *scratch,
                                     Hook after_total_a = Hook()) {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        const int pwa = NW - 1 - warp;  // processing rank of this warp in scan A
        uint32_t *sa = scratch, *sb = scratch + (NW + 1) * WA;
        if (ENTRY_SYNC) __syncthreads();  // scratch may still be read by a previous call
        SA ia = la;
        SB ib = lb;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const SA oa = shfl_state(ia, lane + off);
            if (31 - lane >= off) ia = MA::combine(oa, ia);
            const SB ob = shfl_state(ib, lane - off);
            if (lane >= off) ib = MB::combine(ob, ib);
        }
        exa = shfl_state(ia, lane + 1);
        if (lane == 31) exa = MA::identity();
        exb = shfl_state(ib, lane - 1);
        if (lane == 0) exb = MB::identity();
        if (lane == 0) store_state_smem(sa + pwa * WA, ia);
        if (lane == 31) store_state_smem(sb + warp * WB, ib);
        __syncthreads();
        if (warp == 0) {
            cross_warp<MA, SA>(sa, lane);
            __syncwarp();
            after_total_a(sa + NW * WA);
        }
        if (warp == 1) cross_warp<MB, SB>(sb, lane);
        __syncthreads();
        ta = load_state_smem<SA>(sa + NW * WA);
        tb = load_state_smem<SB>(sb + NW * WB);
        if (pwa > 0) exa = MA::combine(load_state_smem<SA>(sa + pwa * WA), exa);
        if (warp > 0) exb = MB::combine(load_state_smem<SB>(sb + warp * WB), exb);
    }
};

// ------------------------------------------------------------------ decoupled look-back -
//
// Tile status of processing-order tile p: one slot of WP 64-bit words, each word = (flag << 32) |
// one 32-bit word of the payload, flag in {0 = empty, TILE_AGG, TILE_PREFIX}.  A 64-bit store is
// single-copy atomic, so every word carries its own validity: a reader that finds the same non-zero
// flag in all words of a slot has a consistent payload -- no fence, no acquire / release, plain
// relaxed loads and stores through L2 (the first version published payload -> __threadfence ->
// st.release and polled with ld.acquire: two MEMBARs per publish and a CCTL.IVALL per poll made the
// look-back 2/3 of a tile's lifetime, profiles/r1a).  The aggregate and, later, the inclusive prefix
// of a tile go to the SAME slot; a reader that catches the overwrite half-way sees mixed flags and
// polls again.  Tiles take their processing index from an atomic ticket, so every predecessor of a
// running tile is itself running or finished (forward progress).

enum : uint32_t { TILE_EMPTY = 0, TILE_AGG = 1, TILE_PREFIX = 2 };

VJP_DEVINL void st_relaxed_u64(uint64_t *p, uint64_t v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
VJP_DEVINL void ld_relaxed_v2u64(const uint64_t *p, uint64_t &a, uint64_t &b) {
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}

template <class S>
struct TileSlots {
    static constexpr int W = sizeof(S) / 4;
    static constexpr int WP = (W + 1) & ~1;  // 64-bit words per slot (16-byte aligned slots)
    // one 128-byte line per tile at least: neighbouring tiles' slots in one line made every poll of
    // the frontier hit the same L2 sectors the writers were updating (scan + 0.190 -> 0.160 ms)
    static constexpr int STRIDE = WP < 16 ? 16 : WP;
    uint64_t *slots;                         // [num_tiles][STRIDE], zeroed before the launch

    // Called by all lanes of one warp; `words` (shared memory) holds the payload.
    VJP_DEVINL void publish(int p, const uint32_t *words, uint32_t flag) const {
        uint64_t *slot = slots + (size_t)p * STRIDE;
        for (int i = threadIdx.x & 31; i < WP; i += 32)
            st_relaxed_u64(slot + i, ((uint64_t)flag << 32) | (i < W ? words[i] : 0u));
    }
    // Returns the slot's flag (0 if empty or inconsistent) and its payload.
    VJP_DEVINL uint32_t load(int q, S &out) const {
        const uint64_t *slot = slots + (size_t)q * STRIDE;
        uint32_t *o = reinterpret_cast<uint32_t *>(&out);
        uint32_t f_and = ~0u, f_or = 0u;
#pragma unroll
        for (int i = 0; i < WP; i += 2) {
            uint64_t a, b;
            ld_relaxed_v2u64(slot + i, a, b);
            o[i] = (uint32_t)a;
            if (i + 1 < W) o[i + 1] = (uint32_t)b;
            f_and &= (uint32_t)(a >> 32) & (uint32_t)(b >> 32);
            f_or |= (uint32_t)(a >> 32) | (uint32_t)(b >> 32);
        }
        return f_and == f_or ? f_or : 0u;
    }
};

// Called by ALL 32 lanes of one warp.  Returns (in every lane) the fold of tiles 0..p-1 in
// processing order.
template <class M>
VJP_DEVINL typename M::State lookback_warp(const TileSlots<typename M::State> &ts, int p) {
    using S = typename M::State;
    const int lane = threadIdx.x & 31;
    S acc = M::identity();
    int base = p - 1;
    while (true) {
        const int q = base - lane;
        uint32_t f = TILE_PREFIX;  // tiles before the first one: an identity prefix
        S s = M::identity();
        if (q >= 0) f = ts.load(q, s);
        while (__any_sync(FULL_MASK, f == TILE_EMPTY)) {
            if (f == TILE_EMPTY) {
                __nanosleep(20);
                f = ts.load(q, s);
            }
        }
        const unsigned pm = __ballot_sync(FULL_MASK, f == TILE_PREFIX);
        const int first = __ffs(pm) - 1;  // nearest tile with a full prefix; -1 if none
        if (first >= 0 && lane > first) s = M::identity();
        // ordered fold over the window: higher lanes are earlier tiles
#pragma unroll(sizeof(S) > 64 ? 1 : 5)
        for (int off = 1; off < 32; off <<= 1) {
            S o = shfl_state(s, lane + off);
            if (lane + off < 32) s = M::combine(o, s);
        }
        s = shfl_state(s, 0);
        acc = M::combine(s, acc);
        if (pm != 0) break;
        base -= 32;
    }
    return acc;
}

// L2 prefetch of the tile that will be processed `dist` tiles later (dist = the number of co-resident CTAs, i.e. the
// tile this CTA's successor on the same SM will get from the ticket counter).  With one or two CTAs per SM a tile's load,
// scan, look-back and store phases do not overlap; the prefetch keeps HBM busy during the other phases and turns the
// next load into L2 hits.  One bulk instruction per warp (UBLKPF takes a warp-uniform address); `bytes` of the tile
// starting at `tile_ptr` (16-byte aligned) are split evenly over the NW warps.
template <int NW>
VJP_DEVINL void prefetch_tile_l2(const void *tile_ptr, int64_t bytes) {
    const int warp = threadIdx.x >> 5;
    const int64_t chunk = ((bytes + NW - 1) / NW + 15) & ~(int64_t)15;
    const int64_t off = warp * chunk;
    int64_t len = bytes - off;
    if (len > chunk) len = chunk;
    len &= ~(int64_t)15;
    if ((threadIdx.x & 31) == 0 && len > 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(static_cast<const char *>(tile_ptr) + off),
                     "r"((uint32_t)len)
                     : "memory");
}

// 16 bytes of T plus 16 bytes of T (the "+=" of an accumulating VJP call, fused into the final store)
template <class T>
VJP_DEVINL uint4 chunk_add(const uint4 &a, const uint4 &b);
template <>
VJP_DEVINL uint4 chunk_add<float>(const uint4 &a, const uint4 &b) {
    return make_uint4(__float_as_uint(__uint_as_float(a.x) + __uint_as_float(b.x)),
                      __float_as_uint(__uint_as_float(a.y) + __uint_as_float(b.y)),
                      __float_as_uint(__uint_as_float(a.z) + __uint_as_float(b.z)),
                      __float_as_uint(__uint_as_float(a.w) + __uint_as_float(b.w)));
}
template <>
VJP_DEVINL uint4 chunk_add<double>(const uint4 &a, const uint4 &b) {
    const double x = __hiloint2double((int)a.y, (int)a.x) + __hiloint2double((int)b.y, (int)b.x);
    const double y = __hiloint2double((int)a.w, (int)a.z) + __hiloint2double((int)b.w, (int)b.z);
    return make_uint4((uint32_t)__double2loint(x), (uint32_t)__double2hiint(x), (uint32_t)__double2loint(y),
                      (uint32_t)__double2hiint(y));
}
// one element of T at word offset wi of g: g = (acc ? g : 0) + the words at s
template <class T>
VJP_DEVINL void elem_store(uint32_t *g, const uint32_t *s, bool acc);
template <>
VJP_DEVINL void elem_store<float>(uint32_t *g, const uint32_t *s, bool acc) {
    const float x = __uint_as_float(s[0]);
    g[0] = __float_as_uint(acc ? __uint_as_float(g[0]) + x : x);
}
template <>
VJP_DEVINL void elem_store<double>(uint32_t *g, const uint32_t *s, bool acc) {
    double x = __hiloint2double((int)s[1], (int)s[0]);
    if (acc) x += __hiloint2double((int)g[1], (int)g[0]);
    g[0] = (uint32_t)__double2loint(x);
    g[1] = (uint32_t)__double2hiint(x);
}

// ------------------------------------------------------------------ tile staging -------
//
// A tile is NT rows (one per thread) of RW 32-bit words; in shared memory a row has a pitch
// of RW + PAD words, PAD in {0, 4} chosen so that the number of 16-byte chunks per row is odd:
// then a warp's LDS.128 / STS.128 of "chunk c of my row" is bank-conflict-free.  Global <->
// shared copies move whole 16-byte chunks, consecutive lanes on consecutive chunks (coalesced).

template <int NT, int RW>
struct TileStage {
    static_assert(RW % 4 == 0, "row must be a whole number of 16-byte chunks");
    static constexpr int CPR = RW / 4;                       // chunks per row
    // Rows of 4 chunks (64 bytes): a dense layout with the chunk index XOR-ed with bits 1-2 of the row (what the TMA
    // unit's 64B swizzle does) instead of a padded pitch.  The padded pitch of 5 chunks keeps "chunk c of my row"
    // conflict-free but puts chunks t and t + 7 of a coalesced tile copy on one bank group: 14.3 M of the linrec reverse
    // kernel's 54 M shared-memory wavefronts were bank conflicts (ncu, profiles/r2i_scan_vjp.txt); the XOR layout is
    // conflict-free on both sides.  Rows of 8 chunks are conflict-free with a pitch of 9 and keep it (row_ptr users).
    static constexpr bool SWZ = CPR == 4;
    static constexpr int PITCH_C = SWZ ? CPR : ((CPR % 2 == 0) ? CPR + 1 : CPR);  // pitch in chunks
    static constexpr int TILE_WORDS = NT * RW;
    static constexpr int TILE_CHUNKS = NT * CPR;
    static constexpr int SMEM_BYTES = NT * PITCH_C * 16;

    // global (tile-relative chunk index) -> shared chunk index
    static VJP_DEVINL int smem_chunk(int c) {
        if constexpr (SWZ) return c ^ ((c >> 3) & 3);
        else return (c / CPR) * PITCH_C + (c % CPR);
    }
    // chunk j of `row` -> shared chunk index
    static VJP_DEVINL int row_chunk(int row, int j) {
        if constexpr (SWZ) return row * CPR + (j ^ ((row >> 1) & 3));
        else return row * PITCH_C + j;
    }

    // Load `valid_words` words (<= TILE_WORDS) starting at `g` (16-byte aligned) into the staged
    // layout; the rest of the tile is filled with the word pattern fill[w % FW].
    template <int FW>
    static VJP_DEVINL void load(uint4 *smem, const uint32_t *__restrict__ g, int valid_words,
                                const uint32_t (&fill)[FW]) {
        static_assert(RW % FW == 0, "fill pattern must tile a row");
        const uint4 *g4 = reinterpret_cast<const uint4 *>(g);
        if (valid_words == TILE_WORDS) {
#pragma unroll
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) smem[smem_chunk(c)] = ldg_stream(g4 + c);
        } else {
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) {
                uint32_t w[4];
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    const int wi = c * 4 + j;
                    w[j] = (wi < valid_words) ? __ldg(g + wi) : fill[wi % FW];
                }
                smem[smem_chunk(c)] = make_uint4(w[0], w[1], w[2], w[3]);
            }
        }
    }

    // Store the first `valid_words` words of the staged tile (elements of type T) to `g`; acc: g += tile.
    template <class T>
    static VJP_DEVINL void store(const uint4 *smem, uint32_t *__restrict__ g, int valid_words, bool acc) {
        uint4 *g4 = reinterpret_cast<uint4 *>(g);
        if (valid_words == TILE_WORDS) {
#pragma unroll
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) {
                uint4 v = smem[smem_chunk(c)];
                if (acc) v = chunk_add<T>(v, g4[c]);
                stg_stream(g4 + c, v);
            }
        } else {
            constexpr int TW = sizeof(T) / 4;
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) {
                const uint4 v = smem[smem_chunk(c)];
                const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int j = 0; j < 4; j += TW) {
                    const int wi = c * 4 + j;
                    if (wi < valid_words) elem_store<T>(g + wi, w + j, acc);
                }
            }
        }
    }

    // A row is contiguous in shared memory (the padding sits between rows).
    static VJP_DEVINL uint32_t *row_ptr(uint4 *smem, int row) {
        static_assert(!SWZ, "a swizzled row is not contiguous");
        return reinterpret_cast<uint32_t *>(smem + row * PITCH_C);
    }
    // Row access for the owning thread: whole row <-> registers.
    static VJP_DEVINL void read_row(const uint4 *smem, int row, uint32_t (&r)[RW]) {
#pragma unroll
        for (int c = 0; c < CPR; c++) {
            const uint4 v = smem[row_chunk(row, c)];
            r[4 * c + 0] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w;
        }
    }
    static VJP_DEVINL void write_row(uint4 *smem, int row, const uint32_t (&r)[RW]) {
#pragma unroll
        for (int c = 0; c < CPR; c++)
            smem[row_chunk(row, c)] = make_uint4(r[4 * c + 0], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
    }
};

// Rows whose word count is not a multiple of 4 (the 25-word 5x5 matrix): the tile keeps its
// global (linear) layout in shared memory.  Whole-tile copies still move 16-byte chunks; a
// thread reads its row with 32-bit accesses, conflict-free when RW is odd.
template <int NT, int RW>
struct TileStageLinear {
    static constexpr int TILE_WORDS = NT * RW;
    static_assert(TILE_WORDS % 4 == 0, "tile must be a whole number of 16-byte chunks");
    static constexpr int TILE_CHUNKS = TILE_WORDS / 4;
    static constexpr int SMEM_BYTES = TILE_WORDS * 4;

    template <int FW>
    static VJP_DEVINL void load(uint4 *smem, const uint32_t *__restrict__ g, int valid_words,
                                const uint32_t (&fill)[FW]) {
        static_assert(RW % FW == 0, "fill pattern must tile a row");
        const uint4 *g4 = reinterpret_cast<const uint4 *>(g);
        if (valid_words == TILE_WORDS) {
#pragma unroll
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) smem[c] = ldg_stream(g4 + c);
        } else {
            uint32_t *s = reinterpret_cast<uint32_t *>(smem);
            for (int wi = threadIdx.x; wi < TILE_WORDS; wi += NT)
                s[wi] = (wi < valid_words) ? __ldg(g + wi) : fill[wi % FW];
        }
    }
    template <class T>
    static VJP_DEVINL void store(const uint4 *smem, uint32_t *__restrict__ g, int valid_words, bool acc) {
        static_assert(sizeof(T) == 4, "linear tiles hold f32 elements");
        uint4 *g4 = reinterpret_cast<uint4 *>(g);
        if (valid_words == TILE_WORDS) {
#pragma unroll
            for (int c = threadIdx.x; c < TILE_CHUNKS; c += NT) {
                uint4 v = smem[c];
                if (acc) v = chunk_add<T>(v, g4[c]);
                stg_stream(g4 + c, v);
            }
        } else {
            const uint32_t *s = reinterpret_cast<const uint32_t *>(smem);
            for (int wi = threadIdx.x; wi < valid_words; wi += NT) elem_store<T>(g + wi, s + wi, acc);
        }
    }
    static VJP_DEVINL uint32_t *row_ptr(uint4 *smem, int row) {
        return reinterpret_cast<uint32_t *>(smem) + row * RW;
    }
    static VJP_DEVINL void read_row(const uint4 *smem, int row, uint32_t (&r)[RW]) {
        const uint32_t *s = reinterpret_cast<const uint32_t *>(smem) + row * RW;
#pragma unroll
        for (int k = 0; k < RW; k++) r[k] = s[k];
    }
    static VJP_DEVINL void write_row(uint4 *smem, int row, const uint32_t (&r)[RW]) {
        uint32_t *s = reinterpret_cast<uint32_t *>(smem) + row * RW;
#pragma unroll
        for (int k = 0; k < RW; k++) s[k] = r[k];
    }
};

template <int NT, int RW, bool ALIGNED = (RW % 4 == 0)>
struct StageSelect { using type = TileStage<NT, RW>; };
template <int NT, int RW>
struct StageSelect<NT, RW, false> { using type = TileStageLinear<NT, RW>; };
template <int NT, int RW>
using Stage = typename StageSelect<NT, RW>::type;

// words <-> scalars
VJP_DEVINL float word_to(const uint32_t *w, float *) { return __uint_as_float(w[0]); }
VJP_DEVINL double word_to(const uint32_t *w, double *) {
    return __hiloint2double((int)w[1], (int)w[0]);
}
VJP_DEVINL void to_word(float v, uint32_t *w) { w[0] = __float_as_uint(v); }
VJP_DEVINL void to_word(double v, uint32_t *w) {
    w[0] = (uint32_t)__double2loint(v);
    w[1] = (uint32_t)__double2hiint(v);
}

}  // namespace vjp
