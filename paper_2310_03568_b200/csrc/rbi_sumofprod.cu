// rbi_sumofprod.cu -- reduce-by-index with the invertible operator sumOfProd (sections 3.3 and 4.2.4):
//
//   (p1,s1) sumOfProd (p2,s2)     = (p1 + p2 + s1*s2, s1 + s2),  neutral (0,0)      (Fig. 6)
//   (p,s)   sumOfProd_inv (p2,s2) = (p - p2 - (s - s2)*s2, s - s2)                  (Fig. 6)
//
// Elements are pairs [n][2] = (p, s), the histogram is [w][2].
//
// PRIMAL.  sumOfProd has no hardware atomic, but its fold over a bin has a closed form in sums that do:
//   S = sum s_i,   P = sum p_i + sum_{i<j} s_i s_j = sum p_i + (S^2 - sum s_i^2) / 2 = sum (p_i - s_i^2 / 2) + S^2 / 2,
// so the histogram is TWO float atomicAdd histograms, A = sum (p_i - s_i^2 / 2) and S (privatised in shared memory
// when they fit; a shared-memory atomic costs ~19 cycles per warp instruction: three sums took 105 us, two take 75),
// and a finish pass P = A + S^2 / 2 -- no claim rounds, no compare-and-swap.
//
// VJP, invertible-operator rule (Fig. 6): xs = the primal histogram; per element
//   b_i = xs[k_i] (.)_inv v_i,   vs_bar_i = (d(b_i (.) x)/dx)^T xs_bar[k_i] = (Pbar, Pbar * b_i.s + Sbar)
// -- a histogram and a map.  The general rule (sort + segmented scans, Fig. 4) for the same operator is in
// rbi_general.cu (launch_rbi_sop_general_vjp): the paper's 8 - 92x against 1.1 - 2.1x contrast.
#include "common.cuh"
#include "internal.h"

namespace vjp {

constexpr int SOP_NT = 512, SOP_CTAS_PER_SM = 4;
constexpr size_t SOP_SMEM_MAX = 48 * 1024;  // private (sum p, sum s, sum s^2) tables up to this size

VJP_DEVINL bool sop_in_range(int64_t k, int64_t w) { return (uint64_t)k < (uint64_t)w; }

static int sop_grid(int64_t n) {
    const int64_t need = (n + 2 * SOP_NT - 1) / (2 * SOP_NT);
    const int64_t cap = (int64_t)NUM_SMS_B200 * SOP_CTAS_PER_SM;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

// Two elements per thread and iteration: keys as one 128-bit load, the two pairs as one 128-bit load.
struct SopPair {
    int64_t k[2];
    float p[2], s[2];
    int cnt;
};
VJP_DEVINL SopPair sop_load(const int64_t *__restrict__ is, const float *__restrict__ vs, int64_t q, int64_t n) {
    SopPair e;
    e.cnt = (int)min((int64_t)2, n - 2 * q);
    if (e.cnt == 2) {
        longlong2 kk;
        asm volatile("ld.global.nc.L1::no_allocate.v2.s64 {%0,%1}, [%2];" : "=l"(kk.x), "=l"(kk.y) : "l"(is + 2 * q));
        const uint4 v = ldg_stream(reinterpret_cast<const uint4 *>(vs) + q);
        e.k[0] = kk.x; e.k[1] = kk.y;
        e.p[0] = __uint_as_float(v.x); e.s[0] = __uint_as_float(v.y);
        e.p[1] = __uint_as_float(v.z); e.s[1] = __uint_as_float(v.w);
    } else {
        e.k[0] = is[2 * q]; e.p[0] = vs[4 * q]; e.s[0] = vs[4 * q + 1];
        e.k[1] = -1; e.p[1] = 0.f; e.s[1] = 0.f;
    }
    return e;
}

// acc[k] = (A, S, -, -) = (sum (p - s^2 / 2), sum s), zeroed before the launch
template <bool SMEM>
__global__ void __launch_bounds__(SOP_NT)
sop_forward_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const float *__restrict__ vs,
                   float4 *acc) {
    extern __shared__ uint4 smem_raw[];
    float *sh = reinterpret_cast<float *>(smem_raw);  // [w][2]
    if (SMEM) {
        for (int i = threadIdx.x; i < 2 * (int)w; i += SOP_NT) sh[i] = 0.f;
        __syncthreads();
    }
    const int64_t stride = (int64_t)gridDim.x * SOP_NT;
    for (int64_t q = blockIdx.x * (int64_t)SOP_NT + threadIdx.x; 2 * q < n; q += stride) {
        const SopPair e = sop_load(is, vs, q, n);
#pragma unroll
        for (int j = 0; j < 2; j++) {
            if (!sop_in_range(e.k[j], w)) continue;
            const float a = fmaf(-0.5f * e.s[j], e.s[j], e.p[j]);  // p - s^2 / 2
            if (SMEM) {
                float *c = sh + 2 * e.k[j];
                atomicAdd(c, a);
                atomicAdd(c + 1, e.s[j]);
            } else {
                float *c = reinterpret_cast<float *>(acc + e.k[j]);
                atomicAdd(c, a);
                atomicAdd(c + 1, e.s[j]);
            }
        }
    }
    if (SMEM) {
        __syncthreads();
        const int off = (int)((blockIdx.x * 97u) % (unsigned)w);  // concurrent CTAs do not walk the bins in lock step
        for (int k0 = threadIdx.x; k0 < (int)w; k0 += SOP_NT) {
            int k = k0 + off;
            if (k >= (int)w) k -= (int)w;
            float *c = reinterpret_cast<float *>(acc + k);
            if (sh[2 * k] != 0.f) atomicAdd(c, sh[2 * k]);
            if (sh[2 * k + 1] != 0.f) atomicAdd(c + 1, sh[2 * k + 1]);
        }
    }
}

// hist[k] = (A + S^2 / 2, S)
__global__ void sop_finish_kernel(int64_t w, const float4 *__restrict__ acc, float2 *__restrict__ hist) {
    for (int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; k < w; k += (int64_t)gridDim.x * blockDim.x) {
        const float4 a = acc[k];
        hist[k] = make_float2(fmaf(0.5f * a.y, a.y, a.x), a.y);
    }
}

// Return sweep of Fig. 6: b = xs[k] (.)_inv v;  vs_bar = (gp, gp * b.s + gs);  keys out of range get 0.
__global__ void __launch_bounds__(SOP_NT)
sop_inv_sweep_kernel(int64_t n, int64_t w, const int64_t *__restrict__ is, const float *__restrict__ vs,
                     const float2 *__restrict__ xs, const float2 *__restrict__ xs_bar,
                     float *__restrict__ vs_bar, int accumulate) {
    const int64_t stride = (int64_t)gridDim.x * SOP_NT;
    for (int64_t q = blockIdx.x * (int64_t)SOP_NT + threadIdx.x; 2 * q < n; q += stride) {
        const SopPair e = sop_load(is, vs, q, n);
        float2 x[2], g[2];
#pragma unroll
        for (int j = 0; j < 2; j++) {  // the gathers of both elements are issued together
            const int64_t kk = sop_in_range(e.k[j], w) ? e.k[j] : 0;
            x[j] = __ldg(xs + kk);
            g[j] = __ldg(xs_bar + kk);
        }
        float o[4];
#pragma unroll
        for (int j = 0; j < 2; j++) {
            // b = (P - p - (S - s) * s, S - s); only b.s enters the derivative of b (.) x with respect to x
            const float bs = x[j].y - e.s[j];
            const bool in = sop_in_range(e.k[j], w);
            o[2 * j] = in ? g[j].x : 0.f;
            o[2 * j + 1] = in ? fmaf(g[j].x, bs, g[j].y) : 0.f;
        }
        if (e.cnt == 2) {
            uint4 *dst = reinterpret_cast<uint4 *>(vs_bar) + q;
            if (accumulate) {
                const uint4 pr = *dst;
                o[0] += __uint_as_float(pr.x); o[1] += __uint_as_float(pr.y);
                o[2] += __uint_as_float(pr.z); o[3] += __uint_as_float(pr.w);
            }
            stg_stream(dst, make_uint4(__float_as_uint(o[0]), __float_as_uint(o[1]), __float_as_uint(o[2]),
                                       __float_as_uint(o[3])));
        } else {
            float *dst = vs_bar + 4 * q;
            dst[0] = accumulate ? dst[0] + o[0] : o[0];
            dst[1] = accumulate ? dst[1] + o[1] : o[1];
        }
    }
}

// ------------------------------------------------------------------ host side ------------

// acc [w] float4 + hist [w] float2 (the VJP's own copy of the primal)
size_t rbi_sop_workspace_bytes(int64_t w) {
    if (w < 1) w = 1;
    return align_up((size_t)w * 16, 256) + align_up((size_t)w * 8, 256);
}

int launch_rbi_sop_forward(int64_t n, int64_t w, const int64_t *is, const float *vs, float *hist, void *ws,
                           cudaStream_t stream) {
    if (w == 0) return VJP_OK;
    float4 *acc = static_cast<float4 *>(ws);
    if (cudaMemsetAsync(acc, 0, (size_t)w * 16, stream) != cudaSuccess) return VJP_ERR_CUDA;
    if (n > 0) {
        const size_t bytes = (size_t)w * 8;
        if (bytes <= SOP_SMEM_MAX)
            VJP_LAUNCH(K_SOP_FORWARD, stream) sop_forward_kernel<true><<<sop_grid(n), SOP_NT, bytes, stream>>>(n, w, is, vs, acc);
        else
            VJP_LAUNCH(K_SOP_FORWARD, stream) sop_forward_kernel<false><<<sop_grid(n), SOP_NT, 0, stream>>>(n, w, is, vs, acc);
    }
    const int fb = (int)((w + 255) / 256 < 1184 ? (w + 255) / 256 : 1184);
    VJP_LAUNCH(K_SOP_FINISH, stream) sop_finish_kernel<<<fb, 256, 0, stream>>>(w, acc, reinterpret_cast<float2 *>(hist));
    return last_launch_status();
}

int launch_rbi_sop_vjp_inv(int64_t n, int64_t w, const int64_t *is, const float *vs, const float *hist_bar,
                           float *vs_bar, void *ws, int accumulate, cudaStream_t stream) {
    if (n == 0) return VJP_OK;
    if (w == 0) {
        if (!accumulate && cudaMemsetAsync(vs_bar, 0, (size_t)n * 8, stream) != cudaSuccess) return VJP_ERR_CUDA;
        return VJP_OK;
    }
    float *xs = reinterpret_cast<float *>(static_cast<char *>(ws) + align_up((size_t)w * 16, 256));
    const int rc = launch_rbi_sop_forward(n, w, is, vs, xs, ws, stream);
    if (rc != VJP_OK) return rc;
    VJP_LAUNCH(K_SOP_SWEEP, stream) sop_inv_sweep_kernel<<<sop_grid(n), SOP_NT, 0, stream>>>(
        n, w, is, vs, reinterpret_cast<const float2 *>(xs), reinterpret_cast<const float2 *>(hist_bar), vs_bar, accumulate);
    return last_launch_status();
}

}  // namespace vjp
