// scan_ops.cuh -- the scan operators and their hand-derived partial derivatives.
//
// Paper: general scan rule, Fig. 7: with r_i = r_{i-1} (.) x_i,
//     rbar_i = ybar_i + J_i^T rbar_{i+1},  J_i = d(r_i (.) x_{i+1}) / d r_i
//     xbar_i = (d(r_{i-1} (.) x_i) / d x_i)^T rbar_i
// Every operator here is LINEAR in its left operand, so J_i depends on x_{i+1} only, and J^T
// applied to an adjoint z is "z times the block that x contributes" -- the paper's redundant
// block-diagonal form: one q-by-q block shared by all rows.  We carry
//     u_i = J_{i-1}^T rbar_i   (what tile/thread i hands to its left neighbour),
// so the reverse recurrence u_i = (ybar_i + u_{i+1}) * X_i^T uses x_i itself (no one-element
// halo), and the composition over a range is the affine map  z -> b + z * L^T  where L is the
// FORWARD product of the range: lin_o of P:L594 with c = L^T.
//
// An operator Op provides
//   T, D, EW (32-bit words per element), Fwd (running prefix), Lin (what J^T needs of a forward
//   product), Adj (adjoint vector), and the functions used by scan_kernels.cu.
#pragma once

#include "common.cuh"

namespace vjp {

template <class T> struct WordsOf { static constexpr int value = sizeof(T) / 4; };

// ------------------------------------------------------------------------------ '+' -----
// Scan VJP: xbar = reverse inclusive sum of ybar.  Only the monoid is needed.
template <class T_>
struct OpAdd {
    using T = T_;
    static constexpr int D = 1;
    static constexpr int EW = WordsOf<T>::value;
    struct Fwd { T v; };
    static VJP_DEVINL Fwd identity() { return Fwd{T(0)}; }
    static VJP_DEVINL Fwd from_elem(const uint32_t *w) { return Fwd{word_to(w, (T *)nullptr)}; }
    static VJP_DEVINL void to_elem(const Fwd &f, uint32_t *w) { to_word(f.v, w); }
    static VJP_DEVINL Fwd combine(const Fwd &l, const Fwd &r) { return Fwd{l.v + r.v}; }
    static VJP_DEVINL void identity_words(uint32_t (&w)[EW]) { to_word(T(0), w); }
};

// ------------------------------------------------------------------------------ '*' -----
// r (.) x = r*x.  d/dr = x, d/dx = r: no division anywhere, exact with zeros.
template <class T_>
struct OpMul {
    using T = T_;
    static constexpr bool PREFIX_DEP = false;
    static constexpr int D = 1;
    static constexpr int EW = WordsOf<T>::value;
    struct Fwd { T v; };
    struct Lin { T v; };
    struct Adj { T v; };
    static VJP_DEVINL Fwd identity() { return Fwd{T(1)}; }
    static VJP_DEVINL Fwd from_elem(const uint32_t *w) { return Fwd{word_to(w, (T *)nullptr)}; }
    static VJP_DEVINL void to_elem(const Fwd &f, uint32_t *w) { to_word(f.v, w); }
    static VJP_DEVINL Fwd combine(const Fwd &l, const Fwd &r) { return Fwd{l.v * r.v}; }
    static VJP_DEVINL void identity_words(uint32_t (&w)[EW]) { to_word(T(1), w); }

    static VJP_DEVINL Lin lin_of(const Fwd &f) { return Lin{f.v}; }
    static VJP_DEVINL Lin lin_identity() { return Lin{T(1)}; }
    static VJP_DEVINL Lin lin_combine(const Lin &l, const Lin &r) { return Lin{l.v * r.v}; }
    static VJP_DEVINL Adj adj_zero() { return Adj{T(0)}; }
    static VJP_DEVINL Adj adj_from_elem(const uint32_t *w) { return Adj{word_to(w, (T *)nullptr)}; }
    static VJP_DEVINL Adj adj_add(const Adj &a, const Adj &b) { return Adj{a.v + b.v}; }
    static VJP_DEVINL Adj adj_mul(const Adj &z, const Lin &l) { return Adj{z.v * l.v}; }
    // xbar = r_{i-1} * rbar_i
    static VJP_DEVINL void xbar(const Fwd &rprev, const Adj &rbar, uint32_t *w) {
        to_word(rprev.v * rbar.v, w);
    }
};

// --------------------------------------------------------------------------- min / max ---
// r (.) x = min(r, x) with the LEFT (accumulated) operand winning ties (scan with min/max through
// the general rule with d = 1).  NOT linear in r: the 1-by-1 Jacobian d(r (.) x)/dr = [x does not win] depends
// on the running prefix r_{i-1} itself (PREFIX_DEP): the reverse kernel builds the forward prefixes first and
// forms c_i = lin_at(r_{i-1}, x_i) from them; the reverse scan is then that of the scalar recurrence
// u_i = (ybar_i + u_{i+1}) * c_i, and xbar_i = [x_i wins] * rbar_i (the first element always wins: P:L558).
template <class T_, bool IS_MAX>
struct OpMinMax {
    using T = T_;
    static constexpr bool PREFIX_DEP = true;
    static constexpr int D = 1;
    static constexpr int EW = WordsOf<T>::value;
    struct Fwd { T v; };
    struct Lin { T v; };
    struct Adj { T v; };
    static VJP_DEVINL T neutral_value() { return IS_MAX ? -__int_as_float(0x7f800000) : __int_as_float(0x7f800000); }
    static VJP_DEVINL bool wins(T x, T r) { return IS_MAX ? x > r : x < r; }  // strict: the left operand keeps ties
    static VJP_DEVINL Fwd identity() { return Fwd{neutral_value()}; }
    static VJP_DEVINL Fwd from_elem(const uint32_t *w) { return Fwd{word_to(w, (T *)nullptr)}; }
    static VJP_DEVINL void to_elem(const Fwd &f, uint32_t *w) { to_word(f.v, w); }
    static VJP_DEVINL Fwd combine(const Fwd &l, const Fwd &r) { return Fwd{wins(r.v, l.v) ? r.v : l.v}; }
    static VJP_DEVINL void identity_words(uint32_t (&w)[EW]) { to_word(neutral_value(), w); }

    static VJP_DEVINL Lin lin_at(const Fwd &rprev, const Fwd &x) { return Lin{wins(x.v, rprev.v) ? T(0) : T(1)}; }
    static VJP_DEVINL Lin lin_identity() { return Lin{T(1)}; }
    static VJP_DEVINL Lin lin_combine(const Lin &l, const Lin &r) { return Lin{l.v * r.v}; }
    static VJP_DEVINL Adj adj_zero() { return Adj{T(0)}; }
    static VJP_DEVINL Adj adj_from_elem(const uint32_t *w) { return Adj{word_to(w, (T *)nullptr)}; }
    static VJP_DEVINL Adj adj_add(const Adj &a, const Adj &b) { return Adj{a.v + b.v}; }
    static VJP_DEVINL Adj adj_mul(const Adj &z, const Lin &l) { return Adj{z.v * l.v}; }
    // xbar = [x wins against r_{i-1}] * rbar_i; `first`: element 0 of the array takes rbar_0 (xb[0] = rb[0])
    static VJP_DEVINL void xbar_at(const Fwd &rprev, const Fwd &x, const Adj &rbar, bool first, uint32_t *w) {
        to_word((first || wins(x.v, rprev.v)) ? rbar.v : T(0), w);
    }
};

// ------------------------------------------------------------------- linear recurrence ---
// (A,B) (+) (a,b) = (a*A, a*B + b)   (BASELINE config 3; the paper's lin_o with c = a).
// d/d(A,B) = a * I_2 (redundant block-diagonal with a 1x1 block);
// d/da = (A, B), d/db = (0, 1)  =>  abar = A*Abar + B*Bbar,  bbar = Bbar.
template <class T_>
struct OpLinRec {
    using T = T_;
    static constexpr bool PREFIX_DEP = false;
    static constexpr int D = 2;
    static constexpr int EW = 2 * WordsOf<T>::value;
    struct Fwd { T a, b; };
    struct Lin { T a; };
    struct Adj { T a, b; };
    static VJP_DEVINL Fwd identity() { return Fwd{T(1), T(0)}; }
    static VJP_DEVINL Fwd from_elem(const uint32_t *w) {
        return Fwd{word_to(w, (T *)nullptr), word_to(w + WordsOf<T>::value, (T *)nullptr)};
    }
    static VJP_DEVINL void to_elem(const Fwd &f, uint32_t *w) {
        to_word(f.a, w);
        to_word(f.b, w + WordsOf<T>::value);
    }
    static VJP_DEVINL Fwd combine(const Fwd &l, const Fwd &r) {
        return Fwd{r.a * l.a, fma(r.a, l.b, r.b)};
    }
    static VJP_DEVINL void identity_words(uint32_t (&w)[EW]) {
        to_word(T(1), w);
        to_word(T(0), w + WordsOf<T>::value);
    }

    static VJP_DEVINL Lin lin_of(const Fwd &f) { return Lin{f.a}; }
    static VJP_DEVINL Lin lin_identity() { return Lin{T(1)}; }
    static VJP_DEVINL Lin lin_combine(const Lin &l, const Lin &r) { return Lin{l.a * r.a}; }
    static VJP_DEVINL Adj adj_zero() { return Adj{T(0), T(0)}; }
    static VJP_DEVINL Adj adj_from_elem(const uint32_t *w) {
        return Adj{word_to(w, (T *)nullptr), word_to(w + WordsOf<T>::value, (T *)nullptr)};
    }
    static VJP_DEVINL Adj adj_add(const Adj &x, const Adj &y) { return Adj{x.a + y.a, x.b + y.b}; }
    static VJP_DEVINL Adj adj_mul(const Adj &z, const Lin &l) { return Adj{z.a * l.a, z.b * l.a}; }
    static VJP_DEVINL void xbar(const Fwd &rprev, const Adj &rbar, uint32_t *w) {
        to_word(fma(rprev.a, rbar.a, rprev.b * rbar.b), w);
        to_word(rbar.b, w + WordsOf<T>::value);
    }
};

// ------------------------------------------------------------------- q-by-q matmul -------
// R (.) X = R x X, row-major (Q14).  d(R X)/dR applied transposed: Rbar = G X^T -- q
// copies of the block X (redundant block-diagonal); d(R X)/dX: Xbar = R^T G.
// AF = type the forward products are accumulated in, AA = type of the reverse accumulators.
// Orthogonal factors have unit gain, so every rounding along the n-long chain survives: the
// 2x2 scan at n = 2^24 needs f64 accumulators to stay below 1e-4 (precision).
template <int Q, class T_, class AF, class AA>
struct OpMatMul {
    using T = T_;
    static constexpr bool PREFIX_DEP = false;
    static constexpr int D = Q * Q;
    static constexpr int EW = D * WordsOf<T>::value;
    struct Fwd { AF m[D]; };
    using Lin = Fwd;
    struct Adj { AA m[D]; };
    static VJP_DEVINL Fwd identity() {
        Fwd f;
#pragma unroll
        for (int i = 0; i < D; i++) f.m[i] = (i / Q == i % Q) ? AF(1) : AF(0);
        return f;
    }
    static VJP_DEVINL Fwd from_elem(const uint32_t *w) {
        Fwd f;
#pragma unroll
        for (int i = 0; i < D; i++) f.m[i] = (AF)word_to(w + i * WordsOf<T>::value, (T *)nullptr);
        return f;
    }
    static VJP_DEVINL void to_elem(const Fwd &f, uint32_t *w) {
#pragma unroll
        for (int i = 0; i < D; i++) to_word((T)f.m[i], w + i * WordsOf<T>::value);
    }
    static VJP_DEVINL Fwd combine(const Fwd &l, const Fwd &r) {
        Fwd o;
#pragma unroll
        for (int i = 0; i < Q; i++)
#pragma unroll
            for (int j = 0; j < Q; j++) {
                AF s = l.m[i * Q] * r.m[j];
#pragma unroll
                for (int k = 1; k < Q; k++) s = fma(l.m[i * Q + k], r.m[k * Q + j], s);
                o.m[i * Q + j] = s;
            }
        return o;
    }
    static VJP_DEVINL void identity_words(uint32_t (&w)[EW]) {
#pragma unroll
        for (int i = 0; i < D; i++) to_word((i / Q == i % Q) ? T(1) : T(0), w + i * WordsOf<T>::value);
    }

    static VJP_DEVINL Lin lin_of(const Fwd &f) { return f; }
    static VJP_DEVINL Lin lin_identity() { return identity(); }
    static VJP_DEVINL Lin lin_combine(const Lin &l, const Lin &r) { return combine(l, r); }
    static VJP_DEVINL Adj adj_zero() {
        Adj a;
#pragma unroll
        for (int i = 0; i < D; i++) a.m[i] = AA(0);
        return a;
    }
    static VJP_DEVINL Adj adj_from_elem(const uint32_t *w) {
        Adj a;
#pragma unroll
        for (int i = 0; i < D; i++) a.m[i] = (AA)word_to(w + i * WordsOf<T>::value, (T *)nullptr);
        return a;
    }
    static VJP_DEVINL void adj_to_elem(const Adj &a, uint32_t *w) {
#pragma unroll
        for (int i = 0; i < D; i++) to_word((T)a.m[i], w + i * WordsOf<T>::value);
    }
    static VJP_DEVINL Adj adj_add(const Adj &x, const Adj &y) {
        Adj a;
#pragma unroll
        for (int i = 0; i < D; i++) a.m[i] = x.m[i] + y.m[i];
        return a;
    }
    // z * L^T : out[a][b] = sum_k z[a][k] * L[b][k]
    static VJP_DEVINL Adj adj_mul(const Adj &z, const Lin &l) {
        Adj o;
#pragma unroll
        for (int a = 0; a < Q; a++)
#pragma unroll
            for (int b = 0; b < Q; b++) {
                AA s = z.m[a * Q] * (AA)l.m[b * Q];
#pragma unroll
                for (int k = 1; k < Q; k++) s = fma(z.m[a * Q + k], (AA)l.m[b * Q + k], s);
                o.m[a * Q + b] = s;
            }
        return o;
    }
    // Xbar = R^T G : out[a][b] = sum_k R[k][a] * G[k][b]
    static VJP_DEVINL void xbar(const Fwd &rprev, const Adj &rbar, uint32_t *w) {
#pragma unroll
        for (int a = 0; a < Q; a++)
#pragma unroll
            for (int b = 0; b < Q; b++) {
                AA s = (AA)rprev.m[a] * rbar.m[b];
#pragma unroll
                for (int k = 1; k < Q; k++) s = fma((AA)rprev.m[k * Q + a], rbar.m[k * Q + b], s);
                to_word((T)s, w + (a * Q + b) * WordsOf<T>::value);
            }
    }
};

// ------------------------------------------------------------------- monoids -------------

template <class Op>
struct FwdMonoid {
    using State = typename Op::Fwd;
    static VJP_DEVINL State identity() { return Op::identity(); }
    static VJP_DEVINL State combine(const State &earlier, const State &later) {
        return Op::combine(earlier, later);
    }
};

// Reverse scan of affine maps z -> b + z * L^T (lin_o).  "earlier" is the range with
// the HIGHER indices (processed first).  later(earlier(z)) = later.b + (earlier.b + z E^T) L^T
//   = (later.b + earlier.b * L^T) + z * (L E)^T.
template <class Op>
struct RevMonoid {
    struct State {
        typename Op::Adj b;
        typename Op::Lin l;
    };
    static VJP_DEVINL State identity() { return State{Op::adj_zero(), Op::lin_identity()}; }
    static VJP_DEVINL State combine(const State &earlier, const State &later) {
        State o;
        o.b = Op::adj_add(later.b, Op::adj_mul(earlier.b, later.l));
        o.l = Op::lin_combine(later.l, earlier.l);
        return o;
    }
};

}  // namespace vjp
