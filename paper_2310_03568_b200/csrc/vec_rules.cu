// vec_rules.cu -- vectorised operators `map2 (.)` (sections 3.2.4 and 4.2.5 of the paper).
//
// reduce / reduce_by_index / scan whose operator acts element-wise on rows of d scalars are differentiated
// by INTERCHANGE (IRWIM for reduce, eq. 3; its reduce-by-index form; ISWIM for scan,
// P:L655-657): the combinator moves inside the map, i.e. the [n][d] array is transposed and the scalar rule
// is applied to each of the d rows of the transpose.  This file holds the two transposes; the host loop over
// the columns is in api.cu and calls the scalar entry points of the library.
#include "common.cuh"
#include "internal.h"

namespace vjp {

constexpr int TR_NT = 256;

// out[c * cstride + r] = in[r * d + c]   ([n][d] -> d columns of stride cstride); flat over the input, so the
// reads are coalesced and a warp writes d runs of 32 / d consecutive floats.  An "entry" is `a` consecutive floats
// (a = 1: scalars; a > 1: the blocks of a block-diagonal operator); cstride counts entries.
__global__ void __launch_bounds__(TR_NT)
rows_to_cols_kernel(int64_t n, int64_t d, int64_t cstride, const float *__restrict__ in, float *__restrict__ out, int a) {
    const int64_t total = n * d * a, stride = (int64_t)gridDim.x * TR_NT;
    for (int64_t e = blockIdx.x * (int64_t)TR_NT + threadIdx.x; e < total; e += stride) {
        const int64_t ent = e / a, j = e - ent * a;
        const int64_t r = ent / d, c = ent - r * d;
        out[(c * cstride + r) * a + j] = __ldg(in + e);
    }
}

// out[r * d + c] (+)= in[c * cstride + r]; flat over the output: coalesced writes
__global__ void __launch_bounds__(TR_NT)
cols_to_rows_kernel(int64_t n, int64_t d, int64_t cstride, const float *__restrict__ in, float *__restrict__ out,
                    int accumulate, int a) {
    const int64_t total = n * d * a, stride = (int64_t)gridDim.x * TR_NT;
    for (int64_t e = blockIdx.x * (int64_t)TR_NT + threadIdx.x; e < total; e += stride) {
        const int64_t ent = e / a, j = e - ent * a;
        const int64_t r = ent / d, c = ent - r * d;
        const float v = __ldg(in + (c * cstride + r) * a + j);
        out[e] = accumulate ? out[e] + v : v;
    }
}

static int tr_grid(int64_t total) {
    const int64_t need = (total + TR_NT - 1) / TR_NT, cap = (int64_t)NUM_SMS_B200 * 8;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

int launch_rows_to_cols(int64_t n, int64_t d, int64_t cstride, const float *in, float *out, cudaStream_t stream, int a) {
    if (n * d == 0) return VJP_OK;
    VJP_LAUNCH(K_VEC_TRANSPOSE, stream) rows_to_cols_kernel<<<tr_grid(n * d * a), TR_NT, 0, stream>>>(n, d, cstride, in, out, a);
    return last_launch_status();
}
int launch_cols_to_rows(int64_t n, int64_t d, int64_t cstride, const float *in, float *out, int accumulate,
                        cudaStream_t stream, int a) {
    if (n * d == 0) return VJP_OK;
    VJP_LAUNCH(K_VEC_TRANSPOSE, stream) cols_to_rows_kernel<<<tr_grid(n * d * a), TR_NT, 0, stream>>>(n, d, cstride, in, out, accumulate, a);
    return last_launch_status();
}

// ------------------------------------------------------------------ exclusive scan (scan^exc) ---
//
// Output i of the exclusive scan is output i - 1 of the inclusive one (output 0 is the neutral element), so the
// exclusive variants are the inclusive kernels plus a move by one element (api.cu).  An element of 4 ... 100 bytes is
// in general not 16-byte aligned after the move, so this works on 32-bit words:
//   sh > 0:  out[i] = i < sh ? fill[i] : in[i - sh]      (towards higher indices, the neutral element in front)
//   sh < 0:  out[i] = i - sh < nwords ? in[i - sh] : 0   (towards lower indices, zeros behind)
__global__ void __launch_bounds__(TR_NT)
shift_words_kernel(int64_t nwords, int sh, const uint32_t *__restrict__ in, uint32_t *__restrict__ out, ShiftFill fill) {
    const int64_t stride = (int64_t)gridDim.x * TR_NT;
    auto word = [&](int64_t i) -> uint32_t {
        if (sh > 0) return i < sh ? fill.w[i] : __ldg(in + i - sh);
        return i - sh < nwords ? __ldg(in + i - sh) : 0u;
    };
    // four words per thread: the loads are 4-byte (the source is not 16-byte aligned after the move) but hit the same
    // lines across the warp; the store is one 128-bit access
    const int64_t nq = nwords >> 2;
    for (int64_t qd = blockIdx.x * (int64_t)TR_NT + threadIdx.x; qd < nq; qd += stride) {
        const int64_t i = qd * 4;
        reinterpret_cast<uint4 *>(out)[qd] = make_uint4(word(i), word(i + 1), word(i + 2), word(i + 3));
    }
    for (int64_t i = nq * 4 + blockIdx.x * (int64_t)TR_NT + threadIdx.x; i < nwords; i += stride) out[i] = word(i);
}

int launch_shift_words(int64_t nwords, int sh, const void *in, void *out, const ShiftFill &fill, cudaStream_t stream) {
    if (nwords == 0) return VJP_OK;
    VJP_LAUNCH(K_SHIFT_WORDS, stream) shift_words_kernel<<<tr_grid((nwords + 3) / 4), TR_NT, 0, stream>>>(
        nwords, sh, static_cast<const uint32_t *>(in), static_cast<uint32_t *>(out), fill);
    return last_launch_status();
}

}  // namespace vjp
