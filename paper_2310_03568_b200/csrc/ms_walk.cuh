// ms_walk.cuh -- one row (32 consecutive elements, one per lane) of the in-order walk over a WARP-PRIVATE table in shared
// memory: shared by the sort-free general rule / walk histogram (rbi_multiscan.cu) and the routed histogram
// (rbi_routed.cu).
#pragma once
#include "gen_ops.cuh"

namespace vjp {

// A cell of a warp's table doubles as its claim word while a row is in flight: NaN-boxed lane id (no operator result is
// a NaN for NaN-free input; NaN input is undefined, include/vjp_b200.h).
constexpr uint32_t MS_CLAIM = 0xfff00000u;

// One row of the forward walk.  Returns l_local (table (.) earlier same-bin lanes) and updates the table.
// match.any runs on the ADU pipe at ~75 cycles per warp instruction (profiles/r2c_multiscan.txt: that pipe 91 % busy
// when every row used it), so the row first finds out through the table itself whether any two lanes share a bin:
// every lane reads its cell, then stores its claim, then reads it back; if nobody lost, each lane is alone in its bin
// and the row is a plain read-modify-write (89 % of the rows at w = 4096 with uniform keys).  Otherwise the lanes of
// a bin are grouped with match.any and folded in lane order by pointer jumping.
template <int CODE>
VJP_DEVINL float ms_row_forward(const GenOp<CODE> &op, float *tab, int64_t k, float x, int64_t w, int lane) {
    const bool inr = (uint64_t)k < (uint64_t)w;
    const uint32_t key = inr ? (uint32_t)k : (0x80000000u | (uint32_t)lane);  // out of range: a group of its own
    uint32_t *tabu = reinterpret_cast<uint32_t *>(tab);
    const float t = inr ? tab[key] : op.neutral();
    __syncwarp();  // every lane has read its cell
    if (inr) tabu[key] = MS_CLAIM | (uint32_t)lane;
    __syncwarp();
    const bool lost = inr && tabu[key] != (MS_CLAIM | (uint32_t)lane);
    if (!__any_sync(FULL_MASK, lost)) {
        if (inr) tab[key] = op.apply(t, x);
        __syncwarp();
        return t;
    }
    const uint32_t m = __match_any_sync(FULL_MASK, key);
    const uint32_t lower = m & ((1u << lane) - 1u);
    const int prev0 = lower ? 31 - __clz(lower) : -1;
    float inc = x;  // fold over (pj, lane] along the group's list
    int pj = prev0;
    while (__any_sync(FULL_MASK, pj >= 0)) {
        const int src = pj < 0 ? lane : pj;
        const float pv = __shfl_sync(FULL_MASK, inc, src);
        const int pp = __shfl_sync(FULL_MASK, pj, src);
        if (pj >= 0) {
            inc = op.apply(pv, inc);
            pj = pp;
        }
    }
    const float exv = __shfl_sync(FULL_MASK, inc, prev0 < 0 ? lane : prev0);
    const float l = prev0 < 0 ? t : op.apply(t, exv);
    const bool last = (m & (0xfffffffeu << lane)) == 0u;
    if (inr & last) tab[key] = op.apply(t, inc);  // replaces the claim: every bin of the row has one last lane
    __syncwarp();
    return l;
}

}  // namespace vjp
