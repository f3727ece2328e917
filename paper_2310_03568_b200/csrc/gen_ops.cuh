// gen_ops.cuh -- the operators of the general reduce-by-index rule (eq. 5): shared by the sort-based route
// (rbi_general.cu, Fig. 4 as written) and the sort-free chunked route (rbi_multiscan.cu).
#pragma once
#include <math_constants.h>

#include "common.cuh"

namespace vjp {

// G_SOP: sumOfProd.  Of l (.) x (.) r only the s components enter the derivative with respect to x
// (d yp / d xs = ls + rs), so the segmented scans carry s alone, under '+'; the output is a pair.
enum : int { G_ADD = 0, G_MIN = 1, G_MAX = 2, G_MUL = 3, G_SATADD = 4, G_SOP = 5 };

// The operator, its neutral element, and d/dx of (l (.) x) (.) r at x = v (eq. 5).
template <int CODE>
struct GenOp {
    float S;
    VJP_DEVINL float neutral() const {
        return CODE == G_MUL ? 1.f : CODE == G_MIN ? CUDART_INF_F : CODE == G_MAX ? -CUDART_INF_F : 0.f;
    }
    VJP_DEVINL float apply(float a, float b) const {
        switch (CODE) {
        case G_ADD: return a + b;
        case G_SOP: return a + b;
        case G_MUL: return a * b;
        case G_MIN: return b < a ? b : a;
        case G_MAX: return b > a ? b : a;
        default: return fminf(a + b, S);
        }
    }
    // min / max: the accumulated (left) operand wins ties, so among equal extrema the lowest index
    // gets the adjoint, as with min^L.  satadd: slope 1 strictly below S (Q17).
    VJP_DEVINL float dfdx(float l, float v, float r) const {
        switch (CODE) {
        case G_ADD: return 1.f;
        case G_SOP: return l + r;
        case G_MUL: return l * r;
        case G_MIN: return (v < l && !(r < v)) ? 1.f : 0.f;
        case G_MAX: return (v > l && !(r > v)) ? 1.f : 0.f;
        default: {
            const float s = l + v;
            return (s < S && s + r < S) ? 1.f : 0.f;
        }
        }
    }
};

}  // namespace vjp
