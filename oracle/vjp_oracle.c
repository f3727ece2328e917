/*
 * vjp_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded f64 CPU oracle for the reverse-mode vector-Jacobian
 * products (VJPs) of inclusive scan and reduce-by-index, written from the definitions in
 * arxiv/paper_2310_03568 ("Reverse-Mode AD of Reduce-by-Index and Scan in Futhark").
 * "P:Lnnn" below is a line of /root/reference/PAPER.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code, header, table or helper with the CUDA path under
 * paper_2310_03568_b200/, and the product never routes through it.
 *
 * Everything is evaluated sequentially, in the paper's order and notation:
 *   - scans:            the sequential scan loop and its rolled-back return
 *                       sweep (section 5.1);
 *   - reduce-by-index:  the sequential semantics, keys outside [0,w) ignored;
 *   - specialised rules: '+' gather, min/max one-hot at the lowest index
 *                       attaining the extremum, '*' as l_i * r_i
 *                        -- the plain definition, no zero-count trick;
 *   - general rule:     eq. 5 literally, l_i / r_i by per-bin forward / backward
 *                       folds (the radix sort of Fig. 4 is only a way to find them);
 *   - reduce:           the sequential fold, eq. 2 with the two
 *                       exclusive scans of Fig. 2, and the specialised rules of section 3.2
 *                       as their plain definitions (added in round 2, before the kernels);
 *   - sumOfProd:        the invertible operator of section 3.3 -- its reduce_by_index loop,
 *                       Fig. 6 (invertible-operator rule) literally, and eq. 5 with pair folds
 *                       (added in round 2, before the kernels).
 * Parity pins: tests/test_oracle_pins.py (closed forms, finite differences, brute-force
 * dense Jacobian transposes, dot-product test, PPAD's rule of Fig. 11, hand-worked
 * fixtures under tests/golden/).  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -fPIC -shared -o liboracle.so vjp_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* operator codes of this oracle (its own numbering; the product has its own header) */
enum {
    ORC_ADD = 0,    /* a + b,                neutral 0                                  */
    ORC_MIN = 1,    /* min(a, b),            neutral +inf                               */
    ORC_MAX = 2,    /* max(a, b),            neutral -inf                               */
    ORC_MUL = 3,    /* a * b,                neutral 1                                  */
    ORC_LINREC = 4, /* (A,B) (+) (a,b) = (a*A, a*B + b), neutral (1,0); BASELINE config 3;
                       = the paper's lin_o with c = a                  */
    ORC_MATMUL = 5, /* R x X, q-by-q row-major, neutral I_q (BASELINE config 4) */
    ORC_SATADD = 6  /* min(a + b, S) on non-negative reals, neutral 0 (BASELINE
                       config 5; Fig. 8 is missing from the text, reading Q16) */
};

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)

static int scan_arity(int op, int q) {
    switch (op) {
    case ORC_ADD: case ORC_MUL: case ORC_MIN: case ORC_MAX: return 1;
    case ORC_LINREC: return 2;
    case ORC_MATMUL: return q > 0 ? q * q : -1;
    default: return -1;
    }
}

int orc_scan_arity(int op, int q) { return scan_arity(op, q); }

/* r (accumulated prefix, left operand) (.) x -> out, d scalars each. out may not alias. */
static void scan_apply(int op, int q, const double *r, const double *x, double *out) {
    switch (op) {
    case ORC_ADD: out[0] = r[0] + x[0]; break;
    case ORC_MUL: out[0] = r[0] * x[0]; break;
    case ORC_MIN: out[0] = (x[0] < r[0]) ? x[0] : r[0]; break; /* left wins ties */
    case ORC_MAX: out[0] = (x[0] > r[0]) ? x[0] : r[0]; break;
    case ORC_LINREC: out[0] = x[0] * r[0]; out[1] = x[0] * r[1] + x[1]; break;
    case ORC_MATMUL:
        for (int i = 0; i < q; i++)
            for (int j = 0; j < q; j++) {
                double s = 0.0;
                for (int k = 0; k < q; k++) s += r[i * q + k] * x[k * q + j];
                out[i * q + j] = s;
            }
        break;
    }
}

/* Inclusive scan, the sequential loop of P:L525-529:
 *   rs[0] = as[0];  for i in 1..n-1: rs[i] = rs[i-1] (.) as[i]                          */
int orc_scan_forward(int op, int q, int64_t n, const double *xs, double *ys) {
    int d = scan_arity(op, q);
    if (d < 0 || n < 0) return ORC_EINVAL;
    if (n == 0) return ORC_OK;
    memcpy(ys, xs, (size_t)d * sizeof(double));
    for (int64_t i = 1; i < n; i++)
        scan_apply(op, q, ys + (i - 1) * d, xs + i * d, ys + i * d);
    return ORC_OK;
}

/* Return sweep of scan, the rolled-back loop of P:L553-558 (section 5.1):
 *   rb = copy ys_bar
 *   for i = n-1 .. 1:
 *       rb[i-1] += (d(rs[i-1] (.) as[i]) / d rs[i-1])^T . rb[i]
 *       xb[i]    = (d(rs[i-1] (.) as[i]) / d as[i]  )^T . rb[i]
 *   xb[0] = rb[0]
 * The library returns the contribution (the paper's "+=" target starts at zero, Q1).
 * Partials, hand-derived per operator (r = rs[i-1], x = as[i], g = rb[i]):
 *   '+'     : d/dr = 1, d/dx = 1
 *   '*'     : d/dr = x, d/dx = r                       (no division anywhere)
 *   min/max : the selected operand gets 1, the other 0; left operand wins ties
 *   linrec  : (A',B') = (a*A, a*B + b):  dA += a*gA, dB += a*gB;  da = A*gA + B*gB, db = gB
 *   matmul  : Y = R X:  dR = G X^T,  dX = R^T G
 */
int orc_scan_vjp(int op, int q, int64_t n, const double *xs, const double *ys_bar,
                 double *xs_bar) {
    int d = scan_arity(op, q);
    if (d < 0 || n < 0) return ORC_EINVAL;
    if (n == 0) return ORC_OK;
    size_t tot = (size_t)n * (size_t)d;
    double *rs = (double *)malloc(tot * sizeof(double));
    double *rb = (double *)malloc(tot * sizeof(double));
    if (!rs || !rb) { free(rs); free(rb); return ORC_ENOMEM; }
    orc_scan_forward(op, q, n, xs, rs);
    memcpy(rb, ys_bar, tot * sizeof(double));
    for (int64_t i = n - 1; i >= 1; i--) {
        const double *r = rs + (i - 1) * d, *x = xs + i * d, *g = rb + i * d;
        double *gr = rb + (i - 1) * d, *gx = xs_bar + i * d;
        switch (op) {
        case ORC_ADD: gr[0] += g[0]; gx[0] = g[0]; break;
        case ORC_MUL: gr[0] += x[0] * g[0]; gx[0] = r[0] * g[0]; break;
        case ORC_MIN:
            if (x[0] < r[0]) { gx[0] = g[0]; } else { gr[0] += g[0]; gx[0] = 0.0; }
            break;
        case ORC_MAX:
            if (x[0] > r[0]) { gx[0] = g[0]; } else { gr[0] += g[0]; gx[0] = 0.0; }
            break;
        case ORC_LINREC:
            gr[0] += x[0] * g[0];
            gr[1] += x[0] * g[1];
            gx[0] = r[0] * g[0] + r[1] * g[1];
            gx[1] = g[1];
            break;
        case ORC_MATMUL:
            for (int a = 0; a < q; a++)
                for (int b = 0; b < q; b++) {
                    double s = 0.0; /* (G X^T)[a][b] = sum_k G[a][k] X[b][k] */
                    for (int k = 0; k < q; k++) s += g[a * q + k] * x[b * q + k];
                    gr[a * q + b] += s;
                }
            for (int a = 0; a < q; a++)
                for (int b = 0; b < q; b++) {
                    double s = 0.0; /* (R^T G)[a][b] = sum_k R[k][a] G[k][b] */
                    for (int k = 0; k < q; k++) s += r[k * q + a] * g[k * q + b];
                    gx[a * q + b] = s;
                }
            break;
        }
    }
    memcpy(xs_bar, rb, (size_t)d * sizeof(double)); /* xb[0] = rb[0] */
    free(rs);
    free(rb);
    return ORC_OK;
}

/* ---------------------------------------------------------------- reduce-by-index ---- */

static int in_range(int64_t k, int64_t w) { return 0 <= k && k < w; }

static double rbi_neutral(int op) {
    switch (op) {
    case ORC_ADD: case ORC_SATADD: return 0.0;
    case ORC_MUL: return 1.0;
    case ORC_MIN: return INFINITY;
    case ORC_MAX: return -INFINITY;
    }
    return NAN;
}

/* a (.) b for the commutative reduce-by-index operators; a is the accumulated side. */
static double rbi_apply(int op, double S, double a, double b) {
    switch (op) {
    case ORC_ADD: return a + b;
    case ORC_MUL: return a * b;
    case ORC_MIN: return (b < a) ? b : a;
    case ORC_MAX: return (b > a) ? b : a;
    case ORC_SATADD: { double s = a + b; return (s < S) ? s : S; }
    }
    return NAN;
}

static int rbi_op_ok(int op) {
    return op == ORC_ADD || op == ORC_MUL || op == ORC_MIN || op == ORC_MAX || op == ORC_SATADD;
}

/* reduce_by_index with a neutral-initialised histogram: the loop of P:L335 after the
 * rewrite of P:L338-382 (no hist_0 argument). */
int orc_rbi_forward(int op, double S, int64_t n, int64_t w, const int64_t *is,
                    const double *vs, double *hist) {
    if (!rbi_op_ok(op) || n < 0 || w < 0) return ORC_EINVAL;
    for (int64_t k = 0; k < w; k++) hist[k] = rbi_neutral(op);
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (in_range(key, w)) hist[key] = rbi_apply(op, S, hist[key], vs[i]);
    }
    return ORC_OK;
}

/* '+' rule:  vs_bar[i] = hist_bar[is[i]] if in range else 0
 * (the "k >= n" printed at P:L450 is read as "k out of [0,w)", reading Q3). */
int orc_rbi_vjp_add(int64_t n, int64_t w, const int64_t *is, const double *hist_bar,
                    double *vs_bar) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    for (int64_t i = 0; i < n; i++)
        vs_bar[i] = in_range(is[i], w) ? hist_bar[is[i]] : 0.0;
    return ORC_OK;
}

/* min / max: per bin the extremum and the LOWEST index attaining it (P:L182, P:L425-428,
 * P:L454); empty bin -> (n, +-inf).  One sequential pass, strict comparison so
 * the first occurrence wins.  arg, ext may be NULL. vs_bar (may be NULL) is the one-hot
 * return sweep of P:L438-441. */
int orc_rbi_vjp_minmax(int op, int64_t n, int64_t w, const int64_t *is, const double *vs,
                       const double *hist_bar, int64_t *arg, double *ext, double *vs_bar) {
    if ((op != ORC_MIN && op != ORC_MAX) || n < 0 || w < 0) return ORC_EINVAL;
    int64_t *a = (int64_t *)malloc((size_t)(w > 0 ? w : 1) * sizeof(int64_t));
    double *e = (double *)malloc((size_t)(w > 0 ? w : 1) * sizeof(double));
    if (!a || !e) { free(a); free(e); return ORC_ENOMEM; }
    for (int64_t k = 0; k < w; k++) { a[k] = n; e[k] = rbi_neutral(op); }
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (!in_range(key, w)) continue;
        int better = (op == ORC_MIN) ? (vs[i] < e[key]) : (vs[i] > e[key]);
        /* min^L((n,inf),(i,inf)) = (min n i, inf): the first element of a bin
           always takes it, even when it equals the neutral value */
        if (a[key] == n || better) { a[key] = i; e[key] = vs[i]; }
    }
    if (vs_bar) {
        for (int64_t i = 0; i < n; i++) vs_bar[i] = 0.0;
        for (int64_t k = 0; k < w; k++)
            if (a[k] < n) vs_bar[a[k]] = hist_bar[k];
    }
    if (arg) memcpy(arg, a, (size_t)w * sizeof(int64_t));
    if (ext) memcpy(ext, e, (size_t)w * sizeof(double));
    free(a);
    free(e);
    return ORC_OK;
}

/* '*': vs_bar[i] = hist_bar[k_i] * prod_{j != i, k_j = k_i} vs[j] = (l_i * r_i) * hist_bar
 * (P:L236), with l_i / r_i the products of the same-bin elements before / after i,
 * from a per-bin running product forwards and backwards.  No zero counting, no division.
 * zeros / prod_nz (may be NULL) are the lifted primal's outputs (Fig. 3)
 * computed separately for the bit-exact comparison of the counts. */
int orc_rbi_vjp_mul(int64_t n, int64_t w, const int64_t *is, const double *vs,
                    const double *hist_bar, int64_t *zeros, double *prod_nz, double *vs_bar) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    size_t wn = (size_t)(w > 0 ? w : 1), nn = (size_t)(n > 0 ? n : 1);
    double *acc = (double *)malloc(wn * sizeof(double));
    double *l = (double *)malloc(nn * sizeof(double));
    if (!acc || !l) { free(acc); free(l); return ORC_ENOMEM; }
    for (int64_t k = 0; k < w; k++) acc[k] = 1.0;
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (!in_range(key, w)) { l[i] = 0.0; continue; }
        l[i] = acc[key];
        acc[key] *= vs[i];
    }
    for (int64_t k = 0; k < w; k++) acc[k] = 1.0;
    for (int64_t i = n - 1; i >= 0; i--) {
        int64_t key = is[i];
        if (!in_range(key, w)) { if (vs_bar) vs_bar[i] = 0.0; continue; }
        if (vs_bar) vs_bar[i] = (l[i] * acc[key]) * hist_bar[key];
        acc[key] *= vs[i];
    }
    if (zeros || prod_nz) {
        for (int64_t k = 0; k < w; k++) {
            if (zeros) zeros[k] = 0;
            if (prod_nz) prod_nz[k] = 1.0;
        }
        for (int64_t i = 0; i < n; i++) {
            int64_t key = is[i];
            if (!in_range(key, w)) continue;
            if (vs[i] == 0.0) { if (zeros) zeros[key] += 1; }
            else if (prod_nz) prod_nz[key] *= vs[i];
        }
    }
    free(acc);
    free(l);
    return ORC_OK;
}

/* d/dx of (l (.) x) (.) r at x = v, hand-derived per operator (eq. 5).
 * min/max: the FIRST (accumulated, left) operand wins ties, so that among equal extrema
 * the lowest index receives the adjoint, consistent with min^L.
 * satadd: d min(a+b,S)/db = 1 iff a+b < S (0 at the kink, reading Q17). */
static double general_dfdx(int op, double S, double l, double v, double r) {
    switch (op) {
    case ORC_ADD: return 1.0;
    case ORC_MUL: return l * r;
    case ORC_MIN: { double in = (v < l) ? v : l; return ((v < l) && !(r < in)) ? 1.0 : 0.0; }
    case ORC_MAX: { double in = (v > l) ? v : l; return ((v > l) && !(r > in)) ? 1.0 : 0.0; }
    case ORC_SATADD: {
        double in = l + v;
        if (!(in < S)) return 0.0;
        return (in + r < S) ? 1.0 : 0.0;
    }
    }
    return NAN;
}

/* General-case rule, eq. 5:  vs_bar[i] = d(l_i (.) v_i (.) r_i)/d v_i * hist_bar[k_i],
 * 0 for keys outside [0,w).  l_i / r_i = fold of the same-bin elements
 * before / after i in the original order -- exactly what the sorted segmented exclusive
 * scans of Fig. 4 yield, because the sort is stable.  ls_out / rs_out may be
 * NULL. */
int orc_rbi_vjp_general(int op, double S, int64_t n, int64_t w, const int64_t *is,
                        const double *vs, const double *hist_bar, double *vs_bar,
                        double *ls_out, double *rs_out) {
    if (!rbi_op_ok(op) || n < 0 || w < 0) return ORC_EINVAL;
    size_t wn = (size_t)(w > 0 ? w : 1), nn = (size_t)(n > 0 ? n : 1);
    double *acc = (double *)malloc(wn * sizeof(double));
    double *l = (double *)malloc(nn * sizeof(double));
    if (!acc || !l) { free(acc); free(l); return ORC_ENOMEM; }
    for (int64_t k = 0; k < w; k++) acc[k] = rbi_neutral(op);
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (!in_range(key, w)) { l[i] = rbi_neutral(op); continue; }
        l[i] = acc[key];
        acc[key] = rbi_apply(op, S, acc[key], vs[i]);
    }
    for (int64_t k = 0; k < w; k++) acc[k] = rbi_neutral(op);
    for (int64_t i = n - 1; i >= 0; i--) {
        int64_t key = is[i];
        if (!in_range(key, w)) {
            vs_bar[i] = 0.0;
            if (ls_out) ls_out[i] = rbi_neutral(op);
            if (rs_out) rs_out[i] = rbi_neutral(op);
            continue;
        }
        double r = acc[key];
        vs_bar[i] = general_dfdx(op, S, l[i], vs[i], r) * hist_bar[key];
        if (ls_out) ls_out[i] = l[i];
        if (rs_out) rs_out[i] = r;
        /* r_{i'} of the previous same-bin element = v_i (.) r_i (original order) */
        acc[key] = rbi_apply(op, S, vs[i], r);
    }
    free(acc);
    free(l);
    return ORC_OK;
}

/* Stable sort of (key', iota) by key' = k if in range else w (Fig. 4 P:L350-351, P:L396;
 * DESIGN.md reading Q18): valid bins ascending, then every out-of-range element, original
 * order inside each.  A counting sort -- the permutation is unique. */
int orc_rbi_sort_perm(int64_t n, int64_t w, const int64_t *is, int64_t *sorted_keys,
                      int64_t *perm) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    int64_t *start = (int64_t *)calloc((size_t)w + 2, sizeof(int64_t));
    if (!start) return ORC_ENOMEM;
    for (int64_t i = 0; i < n; i++) {
        int64_t k = in_range(is[i], w) ? is[i] : w;
        start[k + 1] += 1;
    }
    for (int64_t k = 0; k <= w; k++) start[k + 1] += start[k];
    for (int64_t i = 0; i < n; i++) {
        int64_t k = in_range(is[i], w) ? is[i] : w;
        int64_t pos = start[k]++;
        sorted_keys[pos] = k;
        perm[pos] = i;
    }
    free(start);
    return ORC_OK;
}

/* ------------------------------------------------------------------ reduce (section 3) --
 *
 * y = reduce (.) e as = a_0 (.) a_1 (.) ... (.) a_{n-1}.  Same operator set as
 * reduce_by_index ('+', '*', min, max, satadd); a reduce is a reduce_by_index with one bin. */

/* The sequential fold of P:L122-124; the neutral element for n = 0. */
int orc_reduce_forward(int op, double S, int64_t n, const double *xs, double *y) {
    if (!rbi_op_ok(op) || n < 0) return ORC_EINVAL;
    double acc = rbi_neutral(op);
    for (int64_t i = 0; i < n; i++) acc = rbi_apply(op, S, acc, xs[i]);
    *y = acc;
    return ORC_OK;
}

/* General rule, eq. 2 with Fig. 2:
 *   ls = scan^exc (.) e as                 (forward exclusive scan)
 *   rs = reverse (scan^exc (\x y -> y (.) x) e (reverse as))
 *   as_bar[i] = d(l_i (.) a_i (.) r_i)/d a_i * y_bar
 * ls_out / rs_out may be NULL. */
int orc_reduce_vjp_general(int op, double S, int64_t n, const double *xs, double y_bar,
                           double *xs_bar, double *ls_out, double *rs_out) {
    if (!rbi_op_ok(op) || n < 0) return ORC_EINVAL;
    double *l = (double *)malloc((size_t)(n > 0 ? n : 1) * sizeof(double));
    if (!l) return ORC_ENOMEM;
    double acc = rbi_neutral(op);
    for (int64_t i = 0; i < n; i++) { l[i] = acc; acc = rbi_apply(op, S, acc, xs[i]); }
    acc = rbi_neutral(op);
    for (int64_t i = n - 1; i >= 0; i--) {
        double r = acc;
        xs_bar[i] = general_dfdx(op, S, l[i], xs[i], r) * y_bar;
        if (ls_out) ls_out[i] = l[i];
        if (rs_out) rs_out[i] = r;
        acc = rbi_apply(op, S, xs[i], r); /* y (.) x of P:L148: the element on the left */
    }
    free(l);
    return ORC_OK;
}

/* Specialised rules of section 3.2, each as its plain definition:
 *   '+'  as_bar = replicate n y_bar
 *   min/max  (k, y) = the extremum and the SMALLEST index attaining
 *           it ("in case of duplicates we choose the smallest index"); as_bar = 0 except
 *           as_bar[k] = y_bar.  n = 0: k = n, y = +-inf, nothing is written.
 *   '*'  as_bar[i] = l_i * r_i * y_bar -- no zero counting, no division;
 *           the lifted primal's (n^{=0}, y^{>0}) of Fig. 3 is computed
 *           separately for the bit-exact comparison of the count.
 * aux_i (may be NULL): k for min/max, n^{=0} for '*'.  aux_v (may be NULL): the extremum for
 * min/max, y^{>0} for '*'. */
int orc_reduce_vjp(int op, int64_t n, const double *xs, double y_bar, double *xs_bar,
                   int64_t *aux_i, double *aux_v) {
    if (n < 0) return ORC_EINVAL;
    switch (op) {
    case ORC_ADD:
        for (int64_t i = 0; i < n; i++) xs_bar[i] = y_bar;
        return ORC_OK;
    case ORC_MIN:
    case ORC_MAX: {
        int64_t k = n;
        double e = rbi_neutral(op);
        for (int64_t i = 0; i < n; i++) {
            int better = (op == ORC_MIN) ? (xs[i] < e) : (xs[i] > e);
            if (k == n || better) { k = i; e = xs[i]; } /* min^L((n,inf),(i,v)): P:L184 */
        }
        for (int64_t i = 0; i < n; i++) xs_bar[i] = 0.0;
        if (k < n) xs_bar[k] = y_bar;
        if (aux_i) *aux_i = k;
        if (aux_v) *aux_v = e;
        return ORC_OK;
    }
    case ORC_MUL: {
        double *l = (double *)malloc((size_t)(n > 0 ? n : 1) * sizeof(double));
        if (!l) return ORC_ENOMEM;
        double acc = 1.0;
        for (int64_t i = 0; i < n; i++) { l[i] = acc; acc *= xs[i]; }
        acc = 1.0;
        for (int64_t i = n - 1; i >= 0; i--) { xs_bar[i] = (l[i] * acc) * y_bar; acc *= xs[i]; }
        free(l);
        int64_t z = 0;
        double p = 1.0;
        for (int64_t i = 0; i < n; i++) { if (xs[i] == 0.0) z++; else p *= xs[i]; }
        if (aux_i) *aux_i = z;
        if (aux_v) *aux_v = p;
        return ORC_OK;
    }
    default: return ORC_EINVAL;
    }
}

/* ---------------------------------------------- invertible operators: sumOfProd (3.3, 4.2.4) --
 *
 * (p1,s1) sumOfProd (p2,s2)     = (p1 + p2 + s1*s2, s1 + s2)            neutral (0,0)   (Fig. 6)
 * (p,s)   sumOfProd_inv (p2,s2) = (p - p2 - (s - s2)*s2, s - s2)                        (Fig. 6)
 * Elements are pairs stored [n][2] = (p, s); the histogram is [w][2]. */
static void sop_apply(const double *a, const double *b, double *out) {
    double p = a[0] + b[0] + a[1] * b[1], s = a[1] + b[1];
    out[0] = p; out[1] = s;
}
static void sop_inv(const double *z, const double *b, double *out) {
    double s = z[1] - b[1];
    out[0] = z[0] - b[0] - s * b[1]; out[1] = s;
}

/* reduce_by_index with sumOfProd over a neutral-initialised histogram: the loop of P:L335. */
int orc_rbi_sop_forward(int64_t n, int64_t w, const int64_t *is, const double *vs, double *hist) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    for (int64_t k = 0; k < 2 * w; k++) hist[k] = 0.0;
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (in_range(key, w)) sop_apply(hist + 2 * key, vs + 2 * i, hist + 2 * key);
    }
    return ORC_OK;
}

/* The operator and its inverse on single pairs (for the pins of property (3)). */
int orc_sop_apply(const double *a, const double *b, double *out) { sop_apply(a, b, out); return ORC_OK; }
int orc_sop_inv(const double *z, const double *b, double *out) { sop_inv(z, b, out); return ORC_OK; }

/* (d(b (.) x)/dx)^T g  at any x, for y = b sumOfProd x = (bp + xp + bs*xs, bs + xs):
 *   dyp/dxp = 1, dyp/dxs = bs, dys/dxp = 0, dys/dxs = 1   =>   xbar = (gp, gp*bs + gs). */
static void sop_vjp_right(const double *b, const double *g, double *xbar) {
    xbar[0] = g[0];
    xbar[1] = g[0] * b[1] + g[1];
}

/* Invertible-operator rule, Fig. 6 literally: xs = the primal histogram;
 * b_i = xs[k_i] (.)_inv v_i;  vs_bar_i = (d(b_i (.) x)/dx)^T xs_bar[k_i];  0 out of range. */
int orc_rbi_sop_vjp_inv(int64_t n, int64_t w, const int64_t *is, const double *vs,
                        const double *hist_bar, double *vs_bar) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    double *xs = (double *)malloc((size_t)(w > 0 ? 2 * w : 2) * sizeof(double));
    if (!xs) return ORC_ENOMEM;
    orc_rbi_sop_forward(n, w, is, vs, xs);
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (!in_range(key, w)) { vs_bar[2 * i] = vs_bar[2 * i + 1] = 0.0; continue; }
        double b[2];
        sop_inv(xs + 2 * key, vs + 2 * i, b);
        sop_vjp_right(b, hist_bar + 2 * key, vs_bar + 2 * i);
    }
    free(xs);
    return ORC_OK;
}

/* General-case rule, eq. 5 with pairs: l_i / r_i = sumOfProd-fold of the same-bin elements before /
 * after i;  y = l (.) x (.) r = (lp + xp + ls*xs + rp + (ls + xs)*rs, ls + xs + rs):
 *   dyp/dxp = 1, dyp/dxs = ls + rs, dys/dxs = 1   =>   xbar = (gp, gp*(ls + rs) + gs). */
int orc_rbi_sop_vjp_general(int64_t n, int64_t w, const int64_t *is, const double *vs,
                            const double *hist_bar, double *vs_bar) {
    if (n < 0 || w < 0) return ORC_EINVAL;
    size_t wn = (size_t)(w > 0 ? w : 1), nn = (size_t)(n > 0 ? n : 1);
    double *acc = (double *)malloc(2 * wn * sizeof(double));
    double *l = (double *)malloc(2 * nn * sizeof(double));
    if (!acc || !l) { free(acc); free(l); return ORC_ENOMEM; }
    for (int64_t k = 0; k < 2 * w; k++) acc[k] = 0.0;
    for (int64_t i = 0; i < n; i++) {
        int64_t key = is[i];
        if (!in_range(key, w)) continue;
        l[2 * i] = acc[2 * key]; l[2 * i + 1] = acc[2 * key + 1];
        sop_apply(acc + 2 * key, vs + 2 * i, acc + 2 * key);
    }
    for (int64_t k = 0; k < 2 * w; k++) acc[k] = 0.0;
    for (int64_t i = n - 1; i >= 0; i--) {
        int64_t key = is[i];
        if (!in_range(key, w)) { vs_bar[2 * i] = vs_bar[2 * i + 1] = 0.0; continue; }
        const double *r = acc + 2 * key, *g = hist_bar + 2 * key;
        vs_bar[2 * i] = g[0];
        vs_bar[2 * i + 1] = g[0] * (l[2 * i + 1] + r[1]) + g[1];
        double t[2];
        sop_apply(vs + 2 * i, r, t); /* r of the previous same-bin element = v_i (.) r_i */
        acc[2 * key] = t[0]; acc[2 * key + 1] = t[1];
    }
    free(acc);
    free(l);
    return ORC_OK;
}
