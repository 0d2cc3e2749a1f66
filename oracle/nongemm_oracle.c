/*
 * nongemm_oracle.c -- plain CPU oracle for SURVEY.md 8(f) NEXT-4: the first non-GEMM consumers of X_embed and the
 * breadth-first stream scheduling queue.  TEST INFRASTRUCTURE ONLY (same rules as dpi_oracle.c): nothing on the
 * product path may call it; it shares no code with paper_2606_21101_b200/csrc/.
 *
 * What it follows (line numbers are /root/reference/PAPER.md):
 *   - IV-D "Fusion Mechanism for non-GEMM Operators" names the operators that sit next to the
 *     embedding output: DeepFM's factorization machine ("element-wise square and reduce-sum"), DCNv2's cross network
 *     ("element-wise addition and element-wise multiplication ... besides GEMM") and the MLP's activation
 *     (PAPER.md:186).  The paper gives no formulas; DESIGN.md 11.4 readings N1-N3 fix them as the cited models'
 *     textbook definitions:
 *       oracle_fm_pairwise     y[b] = sum_{t<u} <x[b,t,:], x[b,u,:]>          (FM second-order term; the DEFINITION,
 *                              pairwise, not the square-of-sum rearrangement the GPU kernel uses)
 *       oracle_cross_combine   out = x0 * (u + bias) + xl                     (DCNv2 layer, u = W xl from the GEMM)
 *       oracle_bias_act        out = act(u + bias), act in {identity, relu, sigmoid}
 *       oracle_lr_first_order  y[b] = bias + sum_t sum_{j in bag(b,t)} w_t[indices[j]]   (DeepFM's logistic-regression
 *                              part: "table lookup ... and reduce-sum"; N7)
 *   - Algorithm 2 "Breadth-first Stream Scheduling", step by step in the paper's order:
 *       oracle_bfs_queue
 * Arithmetic: float64 throughout, results unrounded.
 *
 * Pins (tests/test_oracle_nongemm.py, `-m "not gpu"`): FM -- T = 2 is numpy.dot, all-ones fields give C(T,2)*D,
 * mutually orthogonal fields give 0, the square-of-sum identity in exact integer arithmetic, invariance under field
 * permutation, degree-2 homogeneity, hand-worked fixture tests/golden/nongemm_examples.txt.  Cross -- W = 0, b = 0 is
 * the identity layer; x0 = 0 gives xl; the scalar recurrence x_{l+1} = x0 (w x_l + b) + x_l in exact rationals;
 * fixture.  bias_act -- relu is idempotent and equals (v + |v|)/2; sigmoid(0) = 1/2, sigmoid(-v) = 1 - sigmoid(v),
 * scipy.special.expit.  LR -- constant weights give bias + kappa * (entries of the sample), one-hot is numpy take + sum,
 * equality with the (separately pinned) oracle_lookup on width-1 tables summed over the row, hand fixture.  BFS queue -- the three hand-expanded cases of Algorithm 2 in the fixture, alternation,
 * longer-module-first, per-module order preserved, every op exactly once.
 */
#include <stdint.h>
#include <stddef.h>
#include <math.h>

enum { NG_OK = 0, NG_BAD_ARG = 1 };
enum { NG_ACT_IDENTITY = 0, NG_ACT_RELU = 1, NG_ACT_SIGMOID = 2 };
enum { NG_MODULE_EXPLICIT = 0, NG_MODULE_IMPLICIT = 1 };

/*
 * FM second-order interaction over the T field embeddings of each sample (DESIGN.md 11.4 N1).
 * x is [B, ld] row-major with field t at columns [t*D, (t+1)*D) -- the X_embed block of PAPER.md:139.
 *   v[b, c] = sum_{t<u} x[b,t,c] * x[b,u,c]      (optional, [B, D]: the term before the final reduce-sum)
 *   y[b]    = sum_c v[b, c]                       (optional, [B])
 */
int oracle_fm_pairwise(int32_t B, int32_t T, int32_t D, const double *x, int64_t ld, double *y, double *v)
{
    if (B < 0 || T <= 0 || D <= 0 || !x || ld < (int64_t)T * D || (!y && !v)) return NG_BAD_ARG;
    for (int32_t b = 0; b < B; ++b) {
        const double *xb = x + (int64_t)b * ld;
        double total = 0.0;
        for (int32_t c = 0; c < D; ++c) {
            double pc = 0.0;
            for (int32_t t = 0; t < T; ++t)
                for (int32_t u = t + 1; u < T; ++u)
                    pc += xb[(int64_t)t * D + c] * xb[(int64_t)u * D + c];
            if (v) v[(int64_t)b * D + c] = pc;
            total += pc;
        }
        if (y) y[b] = total;
    }
    return NG_OK;
}

/*
 * DCNv2 cross layer, non-GEMM part (DESIGN.md 11.4 N2): out[b,f] = x0[b,f] * (u[b,f] + bias[f]) + xl[b,f],
 * all [B, F] row-major dense; bias may be NULL (= 0).
 */
int oracle_cross_combine(int32_t B, int32_t F, const double *x0, const double *xl, const double *u,
                         const double *bias, double *out)
{
    if (B < 0 || F <= 0 || !x0 || !xl || !u || !out) return NG_BAD_ARG;
    for (int32_t b = 0; b < B; ++b)
        for (int32_t f = 0; f < F; ++f) {
            int64_t i = (int64_t)b * F + f;
            out[i] = x0[i] * (u[i] + (bias ? bias[f] : 0.0)) + xl[i];
        }
    return NG_OK;
}

/* MLP layer, non-GEMM part (DESIGN.md 11.4 N3): out[b,f] = act(u[b,f] + bias[f]). */
int oracle_bias_act(int32_t B, int32_t F, const double *u, const double *bias, int act, double *out)
{
    if (B < 0 || F <= 0 || !u || !out) return NG_BAD_ARG;
    if (act != NG_ACT_IDENTITY && act != NG_ACT_RELU && act != NG_ACT_SIGMOID) return NG_BAD_ARG;
    for (int32_t b = 0; b < B; ++b)
        for (int32_t f = 0; f < F; ++f) {
            int64_t i = (int64_t)b * F + f;
            double s = u[i] + (bias ? bias[f] : 0.0);
            if (act == NG_ACT_RELU) s = s > 0.0 ? s : 0.0;
            else if (act == NG_ACT_SIGMOID) s = 1.0 / (1.0 + exp(-s));
            out[i] = s;
        }
    return NG_OK;
}

/*
 * DeepFM logistic-regression (first-order) term (DESIGN.md 11.4 N7): one scalar weight per feature,
 *   y[b] = bias + sum_t sum_{j in [offsets[b*T+t], offsets[b*T+t+1])} w_t[indices[j]]
 * Bags are sample-major CSR exactly as in oracle_lookup; offsets == NULL means one-hot (bag g is entry g).
 */
int oracle_lr_first_order(int32_t B, int32_t T, const double *const *w, const int64_t *table_rows,
                          const int32_t *indices, const int32_t *offsets, double bias, double *y)
{
    if (B < 0 || T <= 0 || !w || !table_rows || !y) return NG_BAD_ARG;
    for (int32_t b = 0; b < B; ++b) {
        double acc = bias;
        for (int32_t t = 0; t < T; ++t) {
            int64_t g = (int64_t)b * T + t;
            int64_t lo = offsets ? offsets[g] : g, hi = offsets ? offsets[g + 1] : g + 1;
            for (int64_t j = lo; j < hi; ++j) {
                int64_t r = indices[j];
                if (r < 0 || r >= table_rows[t]) return NG_BAD_ARG;
                acc += w[t][r];
            }
        }
        y[b] = acc;
    }
    return NG_OK;
}

/*
 * Algorithm 2.  Q receives n_explicit + n_implicit entries {module, op index}; the operators of a
 * module go to that module's stream (lines 5-8), Q is the launch order (lines 9-26).
 */
int oracle_bfs_queue(int32_t n_explicit, int32_t n_implicit, int32_t *q_module, int32_t *q_op)
{
    if (n_explicit < 0 || n_implicit < 0 || !q_module || !q_op) return NG_BAD_ARG;
    int64_t n = 0;
    if (n_implicit > n_explicit) {                                      /* line 9 */
        for (int32_t i = 0; i < n_explicit; ++i) {                      /* line 10 */
            q_module[n] = NG_MODULE_IMPLICIT; q_op[n] = i; ++n;         /* line 11 */
            q_module[n] = NG_MODULE_EXPLICIT; q_op[n] = i; ++n;         /* line 12 */
        }
        for (int32_t j = n_explicit; j < n_implicit; ++j) {             /* line 14 */
            q_module[n] = NG_MODULE_IMPLICIT; q_op[n] = j; ++n;         /* line 15 */
        }
    } else {                                                            /* line 18 */
        for (int32_t i = 0; i < n_implicit; ++i) {                      /* line 19 */
            q_module[n] = NG_MODULE_EXPLICIT; q_op[n] = i; ++n;         /* line 20 */
            q_module[n] = NG_MODULE_IMPLICIT; q_op[n] = i; ++n;         /* line 21 */
        }
        for (int32_t j = n_implicit; j < n_explicit; ++j) {             /* line 23 */
            q_module[n] = NG_MODULE_EXPLICIT; q_op[n] = j; ++n;         /* line 24 */
        }
    }
    return NG_OK;                                                       /* line 27 */
}
