// scan_kernels.cu -- single-pass decoupled-look-back scans (forward and reverse) and the fused
// reverse kernel of the scan VJP.
//
//   scan_lookback_kernel<Op, NT, IPT, REV, MODE>
//       MODE_SCAN    : out[i] = fold of in[0..i] (REV: of in[i..n-1]) -- the primal inclusive scan
//                       and, with Op = '+' and REV, the '+' rule of the scan VJP
//                      (xs_bar = reverse inclusive sum of ys_bar).
//       MODE_TILEAGG : only the aggregate of every tile is written (no look-back: a streaming
//                      reduction); tile_exscan_kernel turns the aggregates into exclusive tile
//                      prefixes fpre[t] = fold of all elements before tile t: the forward
//                      re-execution the return sweep needs (r_{i-1} of P:L613; re-execution
//                      instead of a tape).
//   scan_vjp_reverse_kernel<Op, NT, IPT>
//       the general rule of Fig. 7 in one kernel: Jacobians formed on the fly
//       (never stored), reverse linear-recurrence scan with lin_o
//        in its redundant-block-diagonal form, final map.
//
// Tile = NT threads x IPT consecutive elements per thread, staged through shared memory with
// 128-bit coalesced global accesses.  A tile's processing index comes from an atomic ticket.
#include <cooperative_groups.h>
#include <cuda.h>  // CUtensorMap and its enums only: cuTensorMapEncodeTiled is looked up at run time (no libcuda link)

#include <atomic>

#include "internal.h"
#include "scan_ops.cuh"

// Scratch of the entry point that allocates nothing (vjp_scan_add_f32_noalloc, at the end of this file): the ticket
// word and the look-back slots of the '+' scan for up to VJP_NOALLOC_MAX_N = 2^24 elements = 1024 tiles of 16 384
// elements, one 128-byte slot each, + the 256-byte ticket region: 131 328 bytes.  Held by every GPU that loads the
// library until the process exits.  In HOST code this name is only a stand-in for the symbol, not a device address:
// host code gets the address with cudaGetSymbolAddress (noalloc_scratch_ptr below).
static __device__ __align__(256) unsigned char vjp_noalloc_scratch[256 + 1024 * 128];

namespace vjp {

enum : int { MODE_SCAN = 0, MODE_TILEAGG = 2 };

template <class S>
struct LookbackWs {
    int *ticket;
    TileSlots<S> ts;
};

constexpr size_t WS_ALIGN = 256;

// ticket word (padded to WS_ALIGN) + the slots: one contiguous region, zeroed by one memset
template <class S>
static size_t lookback_bytes(int64_t num_tiles) {
    return WS_ALIGN + align_up(sizeof(uint64_t) * TileSlots<S>::STRIDE * (size_t)num_tiles, WS_ALIGN);
}
template <class S>
static LookbackWs<S> lookback_carve(char *base, int64_t num_tiles, size_t *zero_bytes) {
    LookbackWs<S> w;
    w.ticket = reinterpret_cast<int *>(base);
    w.ts.slots = reinterpret_cast<uint64_t *>(base + WS_ALIGN);
    *zero_bytes = lookback_bytes<S>(num_tiles);
    return w;
}

// Warp 0 of the block: publish the tile aggregate, look back, publish the inclusive prefix.
// Returns (in every lane of warp 0) the fold of all tiles processed before tile p.
// `words`: sizeof(State) bytes of shared memory.
// PUBLISHED: the tile aggregate (or, for p = 0, the prefix) has been published already.
template <class M, bool PUBLISHED = false>
VJP_DEVINL typename M::State tile_prefix_warp0(const TileSlots<typename M::State> &ts, int p,
                                               const typename M::State &total, uint32_t *words) {
    using S = typename M::State;
    const int lane = threadIdx.x & 31;
    if (!PUBLISHED) {
        if (lane == 0) store_state_smem(words, total);
        __syncwarp();
        ts.publish(p, words, p == 0 ? TILE_PREFIX : TILE_AGG);
    }
    if (p == 0) return M::identity();
    const S pre = lookback_warp<M>(ts, p);
    __syncwarp();
    if (lane == 0) store_state_smem(words, M::combine(pre, total));
    __syncwarp();
    ts.publish(p, words, TILE_PREFIX);
    return pre;
}

template <class Op, int NT, int IPT, bool REV, int MODE>
__global__ void __launch_bounds__(NT)
scan_lookback_kernel(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, int64_t n,
                     int num_tiles, LookbackWs<typename Op::Fwd> ws,
                     typename Op::Fwd *__restrict__ fpre, int accumulate, int pf_dist) {
    using M = FwdMonoid<Op>;
    using S = typename Op::Fwd;
    constexpr int EW = Op::EW, RW = IPT * EW;
    using St = Stage<NT, RW>;
    using BS = BlockScan<M, NT>;
    extern __shared__ uint4 smem[];
    uint32_t *scratch = reinterpret_cast<uint32_t *>(smem + St::SMEM_BYTES / 16);
    uint32_t *bcast = scratch + BS::SMEM_WORDS;
    __shared__ int s_p;

    if (MODE != MODE_TILEAGG) {
        if (threadIdx.x == 0) s_p = atomicAdd(ws.ticket, 1);
        __syncthreads();
    }
    const int p = MODE == MODE_TILEAGG ? (int)blockIdx.x : s_p;
    const int t = REV ? num_tiles - 1 - p : p;
    const int64_t base = (int64_t)t * (NT * IPT);
    const int valid = (int)min((int64_t)(NT * IPT), n - base);
    if (pf_dist > 0 && p + pf_dist < num_tiles) {
        const int64_t b2 = (int64_t)(REV ? t - pf_dist : t + pf_dist) * (NT * IPT);
        prefetch_tile_l2<NT / 32>(in + b2 * EW, min((int64_t)(NT * IPT), n - b2) * EW * 4);
    }

    uint32_t fill[EW];
    Op::identity_words(fill);
    St::load(smem, in + base * EW, valid * EW, fill);
    __syncthreads();
    // WIDE elements (the 25-word 5x5 matrix) stay in shared memory and are read element by element;
    // narrow ones are held in registers as a whole row.
    constexpr bool WIDE = EW > 8;
    uint32_t rr[WIDE ? 1 : RW];
    uint32_t *r = rr;
    if constexpr (WIDE) r = St::row_ptr(smem, threadIdx.x);
    else St::read_row(smem, threadIdx.x, rr);

    // thread-local fold in processing order
    S acc;
    if (!REV) {
        acc = Op::from_elem(r);
#pragma unroll
        for (int j = 1; j < IPT; j++) acc = Op::combine(acc, Op::from_elem(r + j * EW));
    } else {
        acc = Op::from_elem(r + (IPT - 1) * EW);
#pragma unroll
        for (int j = IPT - 2; j >= 0; j--) acc = Op::combine(Op::from_elem(r + j * EW), acc);
    }
    S total;
    // the CTA's only scan; in MODE_SCAN warp 0 publishes the tile aggregate straight from its cross-warp phase
    S ex = BS::template exclusive<REV, false>(acc, total, scratch, [&](const uint32_t *tot) {
        if (MODE == MODE_SCAN) ws.ts.publish(p, tot, p == 0 ? TILE_PREFIX : TILE_AGG);
    });
    if (MODE == MODE_TILEAGG) {  // aggregate only: no dependency on other tiles, pure streaming
        if (threadIdx.x == 0) store_state_cg(fpre + t, total);
        return;
    }

    if (threadIdx.x < 32) {
        S pre = tile_prefix_warp0<M, true>(ws.ts, p, total, bcast);
        __syncwarp();
        if (threadIdx.x == 0) store_state_smem(bcast, pre);
    }
    __syncthreads();
    const S pre = load_state_smem<S>(bcast);

    // REV is only instantiated for commutative operators ('+'): operand order is immaterial there
    S run = Op::combine(pre, ex);
    if (!REV) {
#pragma unroll
        for (int j = 0; j < IPT; j++) {
            run = Op::combine(run, Op::from_elem(r + j * EW));
            Op::to_elem(run, r + j * EW);
        }
    } else {
#pragma unroll
        for (int j = IPT - 1; j >= 0; j--) {
            run = Op::combine(Op::from_elem(r + j * EW), run);
            Op::to_elem(run, r + j * EW);
        }
    }
    if constexpr (!WIDE) St::write_row(smem, threadIdx.x, rr);
    __syncthreads();
    St::template store<typename Op::T>(smem, out + base * EW, valid * EW, accumulate != 0);
}

// In-place exclusive scan of the per-tile aggregates (a few thousand states) by ONE thread-block
// cluster: every CTA scans its contiguous share, the CTA totals are exchanged through distributed
// shared memory, one cluster barrier.  Together with MODE_TILEAGG this replaces the look-back in the
// forward re-execution of the VJP, which writes no per-element output and so gains nothing from being
// single-pass: the aggregate kernel is a pure streaming reduction (linrec: 107 us vs 161 us for the
// look-back version), the cluster scan takes a few microseconds (a single CTA took 68 - 435 us).
constexpr int XCL = 8;  // portable cluster size
// STAGED: the CTA's contiguous share of the states goes through shared memory (coalesced global accesses).  With
// one thread reading and writing "its" states word by word straight from global memory every access was a sector
// of its own, and the whole scan ran on the load/store units of 8 SMs: lg-throttle 20 stall cycles per issue, 19 us
// for 8192 2x2 states and 41 us for 5462 5x5 states (ncu); only shares too large for shared memory still do that.
template <class Op, int NT, bool STAGED>
__global__ void __launch_bounds__(NT)
tile_exscan_kernel(int num_tiles, typename Op::Fwd *__restrict__ fpre) {
    namespace cg = cooperative_groups;
    using M = FwdMonoid<Op>;
    using S = typename Op::Fwd;
    using BS = BlockScan<M, NT>;
    constexpr int SW = sizeof(S) / 4;
    __shared__ uint32_t scratch[BS::SMEM_WORDS];
    __shared__ uint32_t tot[XCL][SW];
    extern __shared__ uint4 xsm[];
    uint32_t *sst = reinterpret_cast<uint32_t *>(xsm);  // STAGED: the CTA's states, [NT * per][SW] words
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int per = (num_tiles + XCL * NT - 1) / (XCL * NT);
    const int clo = min(rank * NT * per, num_tiles), chi = min(clo + NT * per, num_tiles);  // this CTA's share
    const int lo = min(clo + (int)threadIdx.x * per, chi), hi = min(lo + per, chi);
    uint32_t *gw = reinterpret_cast<uint32_t *>(fpre + clo);
    const int words = (chi - clo) * SW;
    if constexpr (STAGED) {
#pragma unroll 8
        for (int i = threadIdx.x; i < words; i += NT) sst[i] = __ldcg(gw + i);
        __syncthreads();
    }
    auto load = [&](int i) {
        if constexpr (STAGED) return load_state_smem<S>(sst + (size_t)(i - clo) * SW);
        else return load_state_cg(fpre + i);
    };
    S acc = Op::identity();
    for (int i = lo; i < hi; i++) acc = Op::combine(acc, load(i));
    S total;
    const S ex = BS::template exclusive<false>(acc, total, scratch);
    cluster.sync();  // every CTA of the cluster has started: its shared memory may be written remotely
    if (threadIdx.x < XCL) {  // thread r delivers this CTA's total to CTA r
        uint32_t *dst = cluster.map_shared_rank(&tot[0][0], threadIdx.x) + rank * SW;
        store_state_smem(dst, total);
    }
    cluster.sync();
    S run = Op::identity();
    for (int r = 0; r < rank; r++) run = Op::combine(run, load_state_smem<S>(&tot[r][0]));
    run = Op::combine(run, ex);
    for (int i = lo; i < hi; i++) {
        const S a = load(i);
        if constexpr (STAGED) store_state_smem(sst + (size_t)(i - clo) * SW, run);
        else store_state_cg(fpre + i, run);
        run = Op::combine(run, a);
    }
    if constexpr (STAGED) {
        __syncthreads();
#pragma unroll 8
        for (int i = threadIdx.x; i < words; i += NT) __stcg(gw + i, sst[i]);
    }
}

// ---- forward tile aggregates fed by TMA -------------------------------------------------------------------------
// The aggregate pass has no dependency between tiles, so it runs as a PERSISTENT kernel with a ring of STAGES tile
// buffers: one thread issues cp.async.bulk.tensor (UTMALDG) for the tile STAGES steps ahead, the bytes land on an
// mbarrier, and the CTA folds the current tile meanwhile -- no LDG -> register -> STS staging, no load phase that the
// whole CTA waits for.  The array is described to the TMA unit as rows of RB = 64 or 128 bytes (one row = one thread's
// IPT consecutive elements) with the hardware 64B / 128B swizzle: the 16-byte chunk index is XOR-ed with address bits
// 7.. , so that "every thread reads its own row" with LDS.128 is conflict-free in a dense layout (the LDG/STS path
// pads the row pitch instead).  The last tile, if ragged, is filled by hand with the operator's identity.
VJP_DEVINL uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
VJP_DEVINL void mbar_init(uint64_t *b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(b)), "r"(count) : "memory");
}
VJP_DEVINL void mbar_arrive_expect_tx(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(b)), "r"(bytes) : "memory");
}
VJP_DEVINL void mbar_wait(uint64_t *b, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(done)
            : "r"(smem_addr(b)), "r"(parity)
            : "memory");
    } while (!done);
}
VJP_DEVINL void tma_load_rows(void *dst, const CUtensorMap *tm, int row, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_addr(dst)),
        "l"(tm), "r"(0), "r"(row), "r"(smem_addr(bar))
        : "memory");
}

template <class Op, int IPT>
constexpr bool tile_agg_tma_ok() { return Op::EW <= 8 && (IPT * Op::EW * 4 == 64 || IPT * Op::EW * 4 == 128); }

template <class Op, int NT, int IPT>
struct TileAggTma {
    static constexpr int RW = IPT * Op::EW, RB = RW * 4, CPR = RB / 16;  // a thread's row: 64 or 128 bytes
    static constexpr int TILE_BYTES = NT * RB;
    static constexpr int TROWS = TILE_BYTES / 128;                        // the TMA unit sees rows of 128 bytes
    static constexpr int BOX_ROWS = TROWS < 256 ? TROWS : 256, NBOX = TROWS / BOX_ROWS;  // a box has at most 256 rows
    // resident CTAs x ring slots: 1 x 3 for 64 KB tiles (1024 threads), 3 x 2 for 32 KB tiles
    static constexpr int STAGES = TILE_BYTES >= 64 * 1024 ? 3 : 2;
    static constexpr int NW = NT / 32, SW = sizeof(typename Op::Fwd) / 4;
    static constexpr size_t SMEM = 1024 + (size_t)STAGES * TILE_BYTES + STAGES * 8 + 2 * NW * SW * 4;
    static_assert(TILE_BYTES % 128 == 0 && TROWS % BOX_ROWS == 0, "tile = whole boxes of 128-byte rows");
};

template <class Op, int NT, int IPT>
__global__ void __launch_bounds__(NT)
tile_agg_tma_kernel(const __grid_constant__ CUtensorMap tm, const uint32_t *__restrict__ in, int64_t n, int num_tiles,
                    typename Op::Fwd *__restrict__ fpre) {
    using C = TileAggTma<Op, NT, IPT>;
    using S = typename Op::Fwd;
    constexpr int EW = Op::EW, RW = C::RW, RB = C::RB, STAGES = C::STAGES, NW = C::NW, SW = C::SW;
    extern __shared__ uint4 smem[];
    // the swizzle is a function of the shared-memory ADDRESS: ring slots start on 1024-byte boundaries
    uint8_t *stage0 = reinterpret_cast<uint8_t *>(smem) + ((1024u - (smem_addr(smem) & 1023u)) & 1023u);
    uint64_t *full = reinterpret_cast<uint64_t *>(stage0 + (size_t)STAGES * C::TILE_BYTES);  // 8-byte aligned
    uint32_t *scratch = reinterpret_cast<uint32_t *>(full + STAGES);                         // [2][NW] warp totals
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile0 = blockIdx.x, step = gridDim.x;
    const int64_t tile_elems = (int64_t)NT * IPT;
    const int nfull = (int)(n / tile_elems);  // tiles that exist in full: the TMA unit loads only these

    auto issue = [&](int it) {  // thread 0: tile of iteration `it` into its ring slot
        const int t = tile0 + it * step;
        if (t >= nfull) return;
        const int sl = it % STAGES;
        mbar_arrive_expect_tx(full + sl, C::TILE_BYTES);
#pragma unroll
        for (int b = 0; b < C::NBOX; b++)
            tma_load_rows(stage0 + (size_t)sl * C::TILE_BYTES + (size_t)b * C::BOX_ROWS * 128, &tm,
                          t * C::TROWS + b * C::BOX_ROWS, full + sl);
    };
    if (threadIdx.x == 0) {
        for (int sidx = 0; sidx < STAGES; sidx++) mbar_init(full + sidx, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        for (int it = 0; it < STAGES; it++) issue(it);
    }
    __syncthreads();

    for (int it = 0;; it++) {
        const int t = tile0 + it * step;
        if (t >= num_tiles) break;
        const int sl = it % STAGES;
        uint8_t *buf = stage0 + (size_t)sl * C::TILE_BYTES;
        if (t < nfull) {
            mbar_wait(full + sl, (uint32_t)(it / STAGES) & 1u);
        } else {  // the ragged last tile: plain loads into the same swizzled layout, identity behind the end
            const int64_t base = (int64_t)t * tile_elems;
            const int valid_words = (int)(n - base) * EW;
            uint32_t fill[EW];
            Op::identity_words(fill);
            for (int wi = threadIdx.x; wi < NT * RW; wi += NT) {
                const uint32_t off = (uint32_t)wi * 4u;
                const uint32_t v = wi < valid_words ? __ldg(in + base * EW + wi) : fill[wi % EW];
                *reinterpret_cast<uint32_t *>(buf + (off ^ (((off >> 7) & 7u) << 4))) = v;
            }
            __syncthreads();
        }
        uint32_t r[RW];
#pragma unroll
        for (int c = 0; c < C::CPR; c++) {  // 128B swizzle: chunk index (bits 4-6) ^ 128-byte row index (bits 7-9)
            const uint32_t off = (uint32_t)threadIdx.x * RB + c * 16u;
            const uint4 v = *reinterpret_cast<const uint4 *>(buf + (off ^ (((off >> 7) & 7u) << 4)));
            r[4 * c + 0] = v.x; r[4 * c + 1] = v.y; r[4 * c + 2] = v.z; r[4 * c + 3] = v.w;
        }
        S acc = Op::from_elem(r);
#pragma unroll
        for (int j = 1; j < IPT; j++) acc = Op::combine(acc, Op::from_elem(r + j * EW));
        // ordered fold of the tile (the operator need not commute): lane l ends up with lanes l .. 31, lane 0 with the warp
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const S o = shfl_state(acc, lane + off);
            if (lane + off < 32) acc = Op::combine(acc, o);
        }
        uint32_t *wt = scratch + (it & 1) * NW * SW;  // two sets of warp totals: warp 0 may still read the last tile's
        if (lane == 0) store_state_smem(wt + warp * SW, acc);
        __syncthreads();  // the only barrier per tile; behind it every row of the slot has been read
        if (warp == 0) {
            S tot = lane < NW ? load_state_smem<S>(wt + lane * SW) : Op::identity();
#pragma unroll
            for (int off = 1; off < NW; off <<= 1) {
                const S o = shfl_state(tot, lane + off);
                if (lane + off < 32) tot = Op::combine(tot, o);
            }
            if (lane == 0) {
                store_state_cg(fpre + t, tot);
                issue(it + STAGES);
            }
        }
    }
}

// The fused reverse kernel of the scan VJP.  With u_i = rbar_i * X_i^T ("what element i hands to
// element i-1", see scan_ops.cuh) the return sweep of P:L553-558 reads
//     rbar_i = ybar_i + u_{i+1},   xbar_i = (d(r_{i-1} (.) x_i)/dx_i)^T rbar_i,   u_n = 0,
// and element i acts on the incoming u as the affine map z -> (ybar_i + z) * X_i^T.
template <class Op, int NT, int IPT>
__global__ void __launch_bounds__(NT, (Op::EW <= 4 ? (NT <= 256 ? 3 : 1024 / NT) : (Op::EW == 9 ? 2 : 1)))  // 256 threads: 3 CTAs fit the shared memory
scan_vjp_reverse_kernel(const uint32_t *__restrict__ xs, const uint32_t *__restrict__ ybar,
                        uint32_t *__restrict__ xbar, int64_t n, int num_tiles,
                        const typename Op::Fwd *__restrict__ fpre,
                        LookbackWs<typename RevMonoid<Op>::State> ws, int accumulate, int pf_dist) {
    using RM = RevMonoid<Op>;
    using RS = typename RM::State;
    using FM = FwdMonoid<Op>;
    using FS = typename Op::Fwd;
    using Adj = typename Op::Adj;
    constexpr int EW = Op::EW, RW = IPT * EW;
    using St = Stage<NT, RW>;
    using RBS = BlockScan<RM, NT>;
    using FBS = BlockScan<FM, NT>;
    using DBS = BlockScanDual<RM, FM, NT>;
    constexpr bool DUAL = sizeof(RS) + sizeof(FS) <= 96;  // narrow states: both block scans in one pass (half the barriers)
    constexpr int SCR = DBS::SMEM_WORDS;                  // >= either single scan's scratch
    extern __shared__ uint4 smem[];
    uint4 *sx = smem;
    uint4 *sy = smem + St::SMEM_BYTES / 16;
    uint32_t *scratch = reinterpret_cast<uint32_t *>(sy + St::SMEM_BYTES / 16);
    uint32_t *bcast = scratch + SCR;
    __shared__ int s_p;

    if (threadIdx.x == 0) s_p = atomicAdd(ws.ticket, 1);
    __syncthreads();
    const int p = s_p;
    const int t = num_tiles - 1 - p;
    const int64_t base = (int64_t)t * (NT * IPT);
    const int valid = (int)min((int64_t)(NT * IPT), n - base);

    if (pf_dist > 0 && p + pf_dist < num_tiles) {
        const int64_t b2 = (int64_t)(t - pf_dist) * (NT * IPT);  // a full tile: only the last one (t = num_tiles - 1) is ragged
        prefetch_tile_l2<NT / 32>(xs + b2 * EW, (int64_t)(NT * IPT) * EW * 4);
        prefetch_tile_l2<NT / 32>(ybar + b2 * EW, (int64_t)(NT * IPT) * EW * 4);
    }
    uint32_t fillx[EW];
    Op::identity_words(fillx);  // identity element: u passes through unchanged
    const uint32_t filly[1] = {0u};
    St::load(sx, xs + base * EW, valid * EW, fillx);
    St::load(sy, ybar + base * EW, valid * EW, filly);
    __syncthreads();
    constexpr bool WIDE = EW > 8 || sizeof(typename Op::Fwd) > 4 * EW;  // wide states: the elements stay in shared memory
    uint32_t rrx[WIDE ? 1 : RW], rry[WIDE ? 1 : RW];
    uint32_t *rx = rrx, *ry = rry;
    if constexpr (WIDE) {
        rx = St::row_ptr(sx, threadIdx.x);
        ry = St::row_ptr(sy, threadIdx.x);
    } else {
        St::read_row(sx, threadIdx.x, rrx);
        St::read_row(sy, threadIdx.x, rry);
    }

    if constexpr (Op::PREFIX_DEP) {
        // The Jacobian of element i depends on the running prefix r_{i-1} (min / max): forward prefixes first.
        static_assert(!WIDE, "prefix-dependent operators are scalar");
        FS facc = Op::identity();
#pragma unroll
        for (int j = 0; j < IPT; j++) facc = Op::combine(facc, Op::from_elem(rx + j * EW));
        FS ftotal;
        const FS fex = FBS::template exclusive<false, false>(facc, ftotal, scratch);
        FS rp[IPT];
        rp[0] = Op::combine(load_state_cg(fpre + t), fex);
#pragma unroll
        for (int j = 1; j < IPT; j++) rp[j] = Op::combine(rp[j - 1], Op::from_elem(rx + (j - 1) * EW));
        // thread-local reverse reduce: u -> (ybar_j + u) * c_j, c_j = d(r_{j-1} (.) x_j)/dr_{j-1}
        RS racc = RM::identity();
#pragma unroll
        for (int j = IPT - 1; j >= 0; j--) {
            const typename Op::Lin c = Op::lin_at(rp[j], Op::from_elem(rx + j * EW));
            racc.b = Op::adj_mul(Op::adj_add(Op::adj_from_elem(ry + j * EW), racc.b), c);
            racc.l = Op::lin_combine(c, racc.l);
        }
        RS rtotal;
        const RS rex = RBS::template exclusive<true, false>(racc, rtotal, scratch + FBS::SMEM_WORDS,  // own scratch: no entry barrier
                                                            [&](const uint32_t *tot) { ws.ts.publish(p, tot, p == 0 ? TILE_PREFIX : TILE_AGG); });
        if (threadIdx.x < 32) {
            RS pre = tile_prefix_warp0<RM, true>(ws.ts, p, rtotal, bcast);
            __syncwarp();
            if (threadIdx.x == 0) store_state_smem(bcast, pre.b);
        }
        __syncthreads();
        const Adj ztile = load_state_smem<Adj>(bcast);  // u entering the tile from the right
        Adj u = Op::adj_add(rex.b, Op::adj_mul(ztile, rex.l));
        const int64_t first_elem = base + (int64_t)threadIdx.x * IPT;
#pragma unroll
        for (int j = IPT - 1; j >= 0; j--) {
            const FS xj = Op::from_elem(rx + j * EW);
            const Adj rbar = Op::adj_add(Op::adj_from_elem(ry + j * EW), u);
            u = Op::adj_mul(rbar, Op::lin_at(rp[j], xj));
            Op::xbar_at(rp[j], xj, rbar, first_elem + j == 0, ry + j * EW);
        }
        St::write_row(sy, threadIdx.x, rry);
    } else {
    // thread-local reduce, walking the thread's elements from the highest index down
    Adj bacc = Op::adj_zero();
    FS facc = Op::identity();
#pragma unroll(WIDE ? 1 : IPT)
    for (int j = IPT - 1; j >= 0; j--) {
        const FS xj = Op::from_elem(rx + j * EW);
        bacc = Op::adj_mul(Op::adj_add(Op::adj_from_elem(ry + j * EW), bacc), Op::lin_of(xj));
        facc = Op::combine(xj, facc);
    }
    RS racc;
    racc.b = bacc;
    racc.l = Op::lin_of(facc);  // forward product of the thread's range: the c of lin_o, transposed
    RS rtotal, rex;
    FS ftotal, fex;
    if constexpr (DUAL) {
        // the CTA's first use of scratch; warp 0 publishes the tile aggregate one barrier early, straight from the scan
        DBS::template exclusive<false>(racc, rtotal, rex, facc, ftotal, fex, scratch, [&](const uint32_t *tot) {
            ws.ts.publish(p, tot, p == 0 ? TILE_PREFIX : TILE_AGG);
        });
    } else {
        rex = RBS::template exclusive<true, false>(racc, rtotal, scratch,
                                                   [&](const uint32_t *tot) { ws.ts.publish(p, tot, p == 0 ? TILE_PREFIX : TILE_AGG); });
        fex = FBS::template exclusive<false, false>(facc, ftotal, scratch + RBS::SMEM_WORDS);  // own scratch: no entry barrier
    }

    // The forward prefixes r_{i-1} of the thread's elements depend only on fpre[t] and fex, not on the reverse
    // look-back: they are computed BEFORE the barrier that waits for warp 0, so that warps 1 .. N-1 work (and
    // the fpre load is in flight) while warp 0 walks back.
    FS rp[WIDE ? 1 : IPT];
    rp[0] = Op::combine(load_state_cg(fpre + t), fex);
    if constexpr (!WIDE) {
#pragma unroll
        for (int j = 1; j < IPT; j++) rp[j] = Op::combine(rp[j - 1], Op::from_elem(rx + (j - 1) * EW));
    }

    if (threadIdx.x < 32) {
        RS pre = tile_prefix_warp0<RM, true>(ws.ts, p, rtotal, bcast);  // the aggregate went out from the scan
        __syncwarp();
        if (threadIdx.x == 0) store_state_smem(bcast, pre.b);
    }
    __syncthreads();
    const Adj ztile = load_state_smem<Adj>(bcast);  // u entering the tile from the right

    Adj u = Op::adj_add(rex.b, Op::adj_mul(ztile, rex.l));
    if constexpr (WIDE) {
        // descending: rbar_j replaces ybar_j in shared memory; ascending: the forward prefix runs
        // along and xbar_j replaces rbar_j (keeps one prefix in registers instead of IPT)
#pragma unroll 1
        for (int j = IPT - 1; j >= 0; j--) {
            const Adj rbar = Op::adj_add(Op::adj_from_elem(ry + j * EW), u);
            u = Op::adj_mul(rbar, Op::lin_of(Op::from_elem(rx + j * EW)));
            Op::adj_to_elem(rbar, ry + j * EW);
        }
        FS run = rp[0];
#pragma unroll 1
        for (int j = 0; j < IPT; j++) {
            const Adj rbar = Op::adj_from_elem(ry + j * EW);
            Op::xbar(run, rbar, ry + j * EW);
            if (j + 1 < IPT) run = Op::combine(run, Op::from_elem(rx + j * EW));
        }
    } else {
#pragma unroll
        for (int j = IPT - 1; j >= 0; j--) {
            const Adj rbar = Op::adj_add(Op::adj_from_elem(ry + j * EW), u);
            u = Op::adj_mul(rbar, Op::lin_of(Op::from_elem(rx + j * EW)));
            Op::xbar(rp[j], rbar, ry + j * EW);
        }
        St::write_row(sy, threadIdx.x, rry);
    }
    }  // !PREFIX_DEP
    __syncthreads();
    St::template store<typename Op::T>(sy, xbar + base * EW, valid * EW, accumulate != 0);
}

// ------------------------------------------------------------------ host side ------------

template <class Op, int NT_, int IPT_, int VNT_, int VIPT_, bool PF_ = false>
struct ScanCfg {
    using op = Op;
    static constexpr int NT = NT_, IPT = IPT_;     // plain scans
    static constexpr int VNT = VNT_, VIPT = VIPT_; // VJP: forward tile prefixes + fused reverse
    // L2 prefetch of the tile the CTA's successor will take (prefetch_tile_l2): helps where a tile spends a long time
    // away from HBM (matrix operators, min / max: -3 to -5 %), costs 2 % on the scalar operators that are closest to
    // the HBM roofline ('*' f64, linrec), is neutral for '+'
    static constexpr bool PF = PF_;
};

template <class Op, int NT, int IPT>
static size_t scan_smem_bytes() {
    using St = Stage<NT, IPT * Op::EW>;
    using BS = BlockScan<FwdMonoid<Op>, NT>;
    return St::SMEM_BYTES + (BS::SMEM_WORDS + sizeof(typename Op::Fwd) / 4) * 4;
}
template <class Op, int NT, int IPT>
static size_t vjp_smem_bytes() {
    using St = Stage<NT, IPT * Op::EW>;
    constexpr int SCR = BlockScanDual<RevMonoid<Op>, FwdMonoid<Op>, NT>::SMEM_WORDS;
    return 2 * St::SMEM_BYTES + (SCR + sizeof(typename RevMonoid<Op>::State) / 4) * 4;
}

static int64_t tiles_of(int64_t n, int tile) { return (n + tile - 1) / tile; }

// Number of CTAs of `kern` that are resident on the whole GPU = the distance (in tiles) of the L2 prefetch.
template <class K>
static int resident_ctas(K kern, int nt, size_t smem) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, nt, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
    return per_sm * NUM_SMS_B200;
}

template <class Op, int NT, int IPT, bool REV, int MODE, bool PF = false>
static int run_scan(int64_t n, const void *in, void *out, typename Op::Fwd *fpre, char *ws,
                    int accumulate, cudaStream_t stream) {
    using S = typename Op::Fwd;
    const int64_t nt = tiles_of(n, NT * IPT);
    size_t zero_bytes;
    LookbackWs<S> lw = lookback_carve<S>(ws, nt, &zero_bytes);
    if (MODE != MODE_TILEAGG && cudaMemsetAsync(ws, 0, zero_bytes, stream) != cudaSuccess) return VJP_ERR_CUDA;
    auto kern = scan_lookback_kernel<Op, NT, IPT, REV, MODE>;
    const size_t smem = scan_smem_bytes<Op, NT, IPT>();
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return VJP_ERR_CUDA;
    static const int resident = resident_ctas(kern, NT, smem);
    VJP_LAUNCH(MODE == MODE_SCAN ? K_SCAN_LOOKBACK : K_SCAN_TILEAGG, stream)
    kern<<<(unsigned)nt, NT, smem, stream>>>(static_cast<const uint32_t *>(in),
                                             static_cast<uint32_t *>(out), n, (int)nt, lw, fpre, accumulate,
                                             PF ? resident : 0);
    return last_launch_status();
}

template <class Cfg>
static size_t ws_bytes_cfg(int64_t n) {
    using Op = typename Cfg::op;
    const int64_t nt = tiles_of(n, Cfg::NT * Cfg::IPT);
    return lookback_bytes<typename Op::Fwd>(nt);
}
template <class Cfg>
static size_t ws_bytes_vjp_cfg(int64_t n) {
    using Op = typename Cfg::op;
    const int64_t nt = tiles_of(n, Cfg::VNT * Cfg::VIPT);
    return lookback_bytes<typename Op::Fwd>(nt) +
           lookback_bytes<typename RevMonoid<Op>::State>(nt) +
           align_up(sizeof(typename Op::Fwd) * (size_t)nt, WS_ALIGN);
}

// cuTensorMapEncodeTiled through the runtime's driver-entry-point query (the library does not link libcuda)
using TensorMapEncodeFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                       const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static TensorMapEncodeFn tensor_map_encoder() {
    static const TensorMapEncodeFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return reinterpret_cast<TensorMapEncodeFn>(p);
    }();
    return fn;
}

// Forward tile aggregates fpre[t] (before the exclusive scan) by the TMA-fed persistent kernel.  Returns
// VJP_ERR_UNSUPPORTED if the driver has no tensor-map encoder (the caller then takes the LDG / STS kernel).
template <class Op, int NT, int IPT>
static int run_tile_agg_tma(int64_t n, const void *xs, typename Op::Fwd *fpre, cudaStream_t stream) {
    using C = TileAggTma<Op, NT, IPT>;
    const int64_t nt = tiles_of(n, NT * IPT);
    const int64_t full_rows = n / ((int64_t)NT * IPT) * C::TROWS;  // 128-byte rows of the tiles that exist in full
    CUtensorMap tm;
    memset(&tm, 0, sizeof(tm));
    if (full_rows > 0) {
        const TensorMapEncodeFn enc = tensor_map_encoder();
        if (!enc) return VJP_ERR_UNSUPPORTED;
        const cuuint64_t gdim[2] = {32, (cuuint64_t)full_rows};  // rows of 32 words = 128 bytes
        const cuuint64_t gstride[1] = {128};
        const cuuint32_t box[2] = {32, (cuuint32_t)C::BOX_ROWS};
        const cuuint32_t estr[2] = {1, 1};
        if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void *>(xs), gdim, gstride, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return VJP_ERR_UNSUPPORTED;
    }
    auto kern = tile_agg_tma_kernel<Op, NT, IPT>;
    // per call: the attribute belongs to the current device (a process may drive several GPUs)
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return VJP_ERR_CUDA;
    static const int per_gpu = resident_ctas(kern, NT, C::SMEM);
    const unsigned grid = (unsigned)(nt < per_gpu ? nt : per_gpu);
    VJP_LAUNCH(K_SCAN_TILEAGG_TMA, stream)
    kern<<<grid, NT, C::SMEM, stream>>>(tm, static_cast<const uint32_t *>(xs), n, (int)nt, fpre);
    return last_launch_status();
}

template <class Cfg>
static int run_vjp(int64_t n, const void *xs, const void *ys_bar, void *xs_bar, char *ws,
                   int accumulate, cudaStream_t stream) {
    using Op = typename Cfg::op;
    using FS = typename Op::Fwd;
    using RS = typename RevMonoid<Op>::State;
    constexpr int NT = Cfg::VNT, IPT = Cfg::VIPT;
    constexpr bool PF = Cfg::PF;
    const int64_t nt = tiles_of(n, NT * IPT);
    char *ws_fwd = ws;
    char *ws_rev = ws_fwd + lookback_bytes<FS>(nt);
    FS *fpre = reinterpret_cast<FS *>(ws_rev + lookback_bytes<RS>(nt));
    // (A) forward tile prefixes: streaming per-tile aggregates, then their exclusive scan by one cluster
    int rc;
    rc = VJP_ERR_UNSUPPORTED;
    if constexpr (tile_agg_tma_ok<Op, IPT>()) rc = run_tile_agg_tma<Op, NT, IPT>(n, xs, fpre, stream);
    if (rc == VJP_ERR_UNSUPPORTED)  // wide rows (3x3, 5x5), or a driver without cuTensorMapEncodeTiled
        rc = run_scan<Op, NT, IPT, false, MODE_TILEAGG, Cfg::PF>(n, xs, nullptr, fpre, ws_fwd, 0, stream);
    if (rc != VJP_OK) return rc;
    constexpr int XNT = sizeof(FS) > 32 ? 128 : 512;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(XCL);
    cfg.blockDim = dim3(XNT);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = XCL;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const int64_t xper = (nt + XCL * XNT - 1) / (XCL * XNT);
    const size_t xsmem = (size_t)XNT * (size_t)xper * sizeof(FS);  // a CTA's share of the states
    VJP_LAUNCH(K_SCAN_TILEPRE, stream) {
        cudaError_t e;
        if (sizeof(FS) > 16 && xsmem <= 160 * 1024) {  // 8- and 16-byte states: the direct path is as fast (9 vs 10.6 us)
            auto xk = tile_exscan_kernel<Op, XNT, true>;
            if (xsmem > 40 * 1024 &&
                cudaFuncSetAttribute(xk, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024) != cudaSuccess)
                return VJP_ERR_CUDA;
            cfg.dynamicSmemBytes = xsmem;
            e = cudaLaunchKernelEx(&cfg, xk, (int)nt, fpre);
        } else {
            e = cudaLaunchKernelEx(&cfg, tile_exscan_kernel<Op, XNT, false>, (int)nt, fpre);
        }
        if (e != cudaSuccess) return VJP_ERR_CUDA;
    }
    // (B) fused reverse kernel
    size_t zero_bytes;
    LookbackWs<RS> lw = lookback_carve<RS>(ws_rev, nt, &zero_bytes);
    if (cudaMemsetAsync(ws_rev, 0, zero_bytes, stream) != cudaSuccess) return VJP_ERR_CUDA;
    auto kern = scan_vjp_reverse_kernel<Op, NT, IPT>;
    const size_t smem = vjp_smem_bytes<Op, NT, IPT>();
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return VJP_ERR_CUDA;
    static const int resident = resident_ctas(kern, NT, smem);
    VJP_LAUNCH(K_SCAN_VJP_REVERSE, stream)
    kern<<<(unsigned)nt, NT, smem, stream>>>(static_cast<const uint32_t *>(xs),
                                             static_cast<const uint32_t *>(ys_bar),
                                             static_cast<uint32_t *>(xs_bar), n, (int)nt, fpre, lw, accumulate, PF ? resident : 0);
    return last_launch_status();
}

// tile shapes: rows of 16 words (plain scans) / 8 words (VJP: two staged arrays + more live state)
using CfgAddF32 = ScanCfg<OpAdd<float>, 512, 32, 512, 32>;
using CfgAddF64 = ScanCfg<OpAdd<double>, 512, 16, 512, 16>;
using CfgMulF32 = ScanCfg<OpMul<float>, 512, 32, 512, 16>;
using CfgMulF64 = ScanCfg<OpMul<double>, 512, 16, 512, 8>;
using CfgLinRec = ScanCfg<OpLinRec<float>, 512, 16, 512, 8>;
using CfgMinF32 = ScanCfg<OpMinMax<float, false>, 512, 32, 512, 16, true>;
using CfgMaxF32 = ScanCfg<OpMinMax<float, true>, 512, 32, 512, 16, true>;
using CfgMat2 = ScanCfg<OpMatMul<2, float, double, float>, 512, 8, 256, 8, true>;
using CfgMat3 = ScanCfg<OpMatMul<3, float, double, float>, 256, 8, 256, 6, true>;  // f64 forward products, as 2x2 (Q27)
using CfgMat5 = ScanCfg<OpMatMul<5, float, float, float>, 128, 5, 256, 3, true>;

#define VJP_SCAN_DISPATCH(code, dtype, F, FAIL)                                              \
    switch (code) {                                                                          \
    case VJP_OP_ADD: if (dtype == VJP_F32) { F(CfgAddF32) } else { F(CfgAddF64) } break;     \
    case VJP_OP_MUL: if (dtype == VJP_F32) { F(CfgMulF32) } else { F(CfgMulF64) } break;     \
    case VJP_OP_MIN: if (dtype == VJP_F32) { F(CfgMinF32) } else { FAIL } break;             \
    case VJP_OP_MAX: if (dtype == VJP_F32) { F(CfgMaxF32) } else { FAIL } break;             \
    case VJP_OP_LINREC: if (dtype == VJP_F32) { F(CfgLinRec) } else { FAIL } break;          \
    case VJP_OP_MATMUL2: if (dtype == VJP_F32) { F(CfgMat2) } else { FAIL } break;           \
    case VJP_OP_MATMUL3: if (dtype == VJP_F32) { F(CfgMat3) } else { FAIL } break;           \
    case VJP_OP_MATMUL5: if (dtype == VJP_F32) { F(CfgMat5) } else { FAIL } break;           \
    default: FAIL                                                                            \
    }

size_t scan_workspace_bytes(int code, int dtype, int64_t n) {
    if (n <= 0) return WS_ALIGN;
    if (code == VJP_OP_ADD)
        return dtype == VJP_F32 ? ws_bytes_cfg<CfgAddF32>(n) : ws_bytes_cfg<CfgAddF64>(n);
    size_t a = 0, b = 0;
#define F(C) a = ws_bytes_cfg<C>(n); b = ws_bytes_vjp_cfg<C>(n);
    switch (code) {
    case VJP_OP_MUL: if (dtype == VJP_F32) { F(CfgMulF32) } else { F(CfgMulF64) } break;
    case VJP_OP_MIN: F(CfgMinF32) break;
    case VJP_OP_MAX: F(CfgMaxF32) break;
    case VJP_OP_LINREC: F(CfgLinRec) break;
    case VJP_OP_MATMUL2: F(CfgMat2) break;
    case VJP_OP_MATMUL3: F(CfgMat3) break;
    case VJP_OP_MATMUL5: F(CfgMat5) break;
    default: return 0;
    }
#undef F
    return a > b ? a : b;
}

int launch_scan_forward(int code, int dtype, int64_t n, const void *xs, void *ys, void *ws,
                        cudaStream_t stream) {
#define F(C) return run_scan<typename C::op, C::NT, C::IPT, false, MODE_SCAN, C::PF>(n, xs, ys, nullptr, (char *)ws, 0, stream);
    VJP_SCAN_DISPATCH(code, dtype, F, return VJP_ERR_UNSUPPORTED;)
#undef F
    return VJP_ERR_UNSUPPORTED;
}

int launch_scan_vjp(int code, int dtype, int64_t n, const void *xs, const void *ys_bar,
                    void *xs_bar, void *ws, int accumulate, cudaStream_t stream) {
    if (code == VJP_OP_ADD) {  // reverse inclusive sum of ys_bar
        if (dtype == VJP_F32)
            return run_scan<OpAdd<float>, CfgAddF32::NT, CfgAddF32::IPT, true, MODE_SCAN>(
                n, ys_bar, xs_bar, nullptr, (char *)ws, accumulate, stream);
        return run_scan<OpAdd<double>, CfgAddF64::NT, CfgAddF64::IPT, true, MODE_SCAN>(
            n, ys_bar, xs_bar, nullptr, (char *)ws, accumulate, stream);
    }
#define F(C) return run_vjp<C>(n, xs, ys_bar, xs_bar, (char *)ws, accumulate, stream);
    switch (code) {
    case VJP_OP_MUL: if (dtype == VJP_F32) { F(CfgMulF32) } else { F(CfgMulF64) } break;
    case VJP_OP_MIN: if (dtype == VJP_F32) { F(CfgMinF32) } break;
    case VJP_OP_MAX: if (dtype == VJP_F32) { F(CfgMaxF32) } break;
    case VJP_OP_LINREC: if (dtype == VJP_F32) { F(CfgLinRec) } break;
    case VJP_OP_MATMUL2: if (dtype == VJP_F32) { F(CfgMat2) } break;
    case VJP_OP_MATMUL3: if (dtype == VJP_F32) { F(CfgMat3) } break;
    case VJP_OP_MATMUL5: if (dtype == VJP_F32) { F(CfgMat5) } break;
    default: break;
    }
#undef F
    return VJP_ERR_UNSUPPORTED;
}

// ------------------------------------------------------------------ no-allocation entry point
//
// vjp_scan_add_f32_noalloc: the '+' rule of the scan VJP (xs_bar = reverse inclusive sum of ys_bar) for
// callers that can neither allocate a workspace nor let the library do it (CUDA graph capture, serving loops):
// the same kernel as vjp_scan with VJP_OP_ADD / f32, its look-back scratch in the static device array above.

constexpr int64_t NOALLOC_MAX_N = (int64_t)1 << 24;
constexpr int NOALLOC_MAX_DEVICES = 64;
static_assert(sizeof(vjp_noalloc_scratch) >= WS_ALIGN + 8 * TileSlots<float>::STRIDE *
                                                 (size_t)(NOALLOC_MAX_N / (CfgAddF32::NT * CfgAddF32::IPT)),
              "static scratch too small for NOALLOC_MAX_N");

int64_t scan_noalloc_max_n() { return NOALLOC_MAX_N; }

// Device address of the static scratch on the CURRENT device: resolved once per device, with that device current.
static char *noalloc_scratch_ptr() {
    static std::atomic<char *> cache[NOALLOC_MAX_DEVICES];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) return nullptr;
    char *p = cache[dev].load(std::memory_order_acquire);
    if (p == nullptr) {
        void *sym = nullptr;
        if (cudaGetSymbolAddress(&sym, vjp_noalloc_scratch) != cudaSuccess || sym == nullptr) {
            cudaGetLastError();
            return nullptr;
        }
        p = static_cast<char *>(sym);
        cache[dev].store(p, std::memory_order_release);
    }
    return p;
}

// n in [1, NOALLOC_MAX_N] (checked by the caller).  No cudaMalloc / cudaFree: the status words are cleared with a
// memset on `stream` (run_scan), then the kernel is launched.
int launch_scan_add_f32_noalloc(int64_t n, const float *ys_bar, float *xs_bar, int accumulate, cudaStream_t stream) {
    if (lookback_bytes<float>(tiles_of(n, CfgAddF32::NT * CfgAddF32::IPT)) > sizeof(vjp_noalloc_scratch))
        return VJP_ERR_UNSUPPORTED;
    char *ws = noalloc_scratch_ptr();
    if (ws == nullptr) return VJP_ERR_CUDA;
    return run_scan<OpAdd<float>, CfgAddF32::NT, CfgAddF32::IPT, true, MODE_SCAN>(n, ys_bar, xs_bar, nullptr, ws,
                                                                                  accumulate, stream);
}

}  // namespace vjp
