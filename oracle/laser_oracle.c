/*
 * laser_oracle.c — fp64 CPU ORACLE for the LASER batched early-exit confidence probe.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or constant with the CUDA path under paper_2606_31580_b200/csrc/.
 *
 * What it computes (all citations are /root/reference/PAPER.md line numbers; "DESIGN A<n>" are the
 * readings listed in DESIGN.md where the paper is silent):
 *
 *   step 1  logits l[n,v] = sum_k hidden[n,k] * W[v,k]              PAPER.md:61  (§3.1: "a confidence
 *           score C is computed from the token probabilities" => softmax of the LM-head logits;
 *           no bias, temperature 1: DESIGN A2)
 *   step 2  m = max_v l ; a = min{v : l[v] == m} ; S = sum_v exp(l[v]-m) ; pmax = 1/S
 *           (plain softmax definition; lowest-index tie-break: DESIGN A9)
 *   step 3  C[r] = mean of pmax over the request's rows (DESIGN A1; Alg.1 step 4)
 *   step 4  lambda[r] = clamp(lambda_base - beta*tanh(gamma*(Lbar[r]-L_target)/L_target),
 *                             lambda_min, lambda_max)                PAPER.md:100-103 (Eq. 5), 144
 *   step 5  exit[r] = C[r] > lambda[r]   (strict)                    PAPER.md:61, 70, 122 (Alg.1 step 6)
 *
 *   variant (NEXT-1 / DESIGN A2): probability of a given (emitted) token, laser_oracle_token_prob.
 *
 * and, off the hot path (NEXT-2 rows of SURVEY §8 f):
 *   EMA      Lbar(t) = alpha*L(t) + (1-alpha)*Lbar(t-1), Lbar(0)=0
 *   budget   B = max{B_min, floor(B_base*f_diff*f_load)}             PAPER.md:152-173 (Eq. 6-8)
 *
 * Everything is the plain definition written out: no tiling, no online rescaling, no fused passes.
 * Inputs are float32 arrays (every bf16 value is exactly a float32) widened exactly to double, so
 * the oracle sees the same numbers the GPU sees.  Floating point: IEEE double everywhere.
 *
 * Summation order of step 1 (DESIGN A17): 8 independent partial sums over k (k mod 8), combined as
 * ((a0+a1)+(a2+a3))+((a4+a5)+(a6+a7)), then the k-tail added in order.  fp64 reassociation moves a
 * logit by <~ d*2^-53*sum|h||w| ~ 1e-13, nine orders below the parity tolerances.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_tau_pins.py): P1-P14 of DESIGN.md.  Parts that the
 * paper itself does not pin ("parity unpinned" by the paper, fixed only by BASELINE.json's wording):
 * the choice of aggregate (arithmetic mean, A1) and max-prob vs emitted-token prob (A2).
 *
 * Non-finite inputs (DESIGN A12): NaN logits are skipped by the max/argmax (comparisons with NaN are
 * false) but poison S, so pmax, C are NaN and exit is 0.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double lambda_base, beta, gamma, l_target, lambda_min, lambda_max;
} oracle_tau_params;

int laser_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* step 1 for one (n, v): the dot product in the documented order.  target_clones only lets gcc use
 * wider registers on CPUs that have them (the .so is built on one box and may run on another);
 * with -ffp-contract=off every clone performs the same IEEE operations in the same order. */
__attribute__((target_clones("avx512f", "avx2", "default")))
static double dot_fp64(const double* h, const float* w, int d) {
    double a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int k = 0;
    for (; k + 8 <= d; k += 8)
        for (int j = 0; j < 8; ++j) a[j] += h[k + j] * (double)w[k + j];
    double s = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
    for (; k < d; ++k) s += h[k] * (double)w[k];
    return s;
}

/*
 * Steps 1-2 for rows [0, N).  Outputs (any may be NULL): m, a, S, pmax, gap2, each [N].
 * gap2 = m - (second largest logit counting duplicates) >= 0; +inf if V == 1.
 * logits_opt: if non-NULL, [N,V] doubles receive the logits (tests on tiny cases only).
 * Returns 0, or -1 on bad arguments / allocation failure.
 */
int laser_oracle_row_stats(const float* hidden, const float* W, int64_t N, int d, int64_t V,
                           double* out_m, int32_t* out_a, double* out_S, double* out_pmax,
                           double* out_gap2, double* logits_opt) {
    if (N < 0 || d <= 0 || V <= 0 || (N > 0 && (!hidden || !W))) return -1;
    int failed = 0;
#pragma omp parallel
    {
        double* h = (double*)malloc(sizeof(double) * (size_t)d);
        double* l = (double*)malloc(sizeof(double) * (size_t)V);
        if (!h || !l) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t n = 0; n < N; ++n) {
                for (int k = 0; k < d; ++k) h[k] = (double)hidden[n * d + k];
                /* step 1 */
                for (int64_t v = 0; v < V; ++v) l[v] = dot_fp64(h, W + v * (int64_t)d, d);
                /* step 2: max, lowest-index argmax, runner-up */
                double m = -INFINITY, second = -INFINITY;
                int64_t a = 0;
                int have = 0;
                for (int64_t v = 0; v < V; ++v) {
                    double x = l[v];
                    if (x != x) continue; /* NaN: DESIGN A12 */
                    if (!have) { m = x; a = v; have = 1; }
                    else if (x > m) { second = m; m = x; a = v; }
                    else if (x > second) { second = x; }
                }
                double S = 0.0;
                for (int64_t v = 0; v < V; ++v) S += exp(l[v] - m);
                if (out_m) out_m[n] = m;
                if (out_a) out_a[n] = (int32_t)a;
                if (out_S) out_S[n] = S;
                if (out_pmax) out_pmax[n] = 1.0 / S;
                if (out_gap2) out_gap2[n] = (V > 1) ? (m - second) : INFINITY;
                if (logits_opt) memcpy(logits_opt + n * V, l, sizeof(double) * (size_t)V);
            }
        }
        free(h);
        free(l);
    }
    return failed ? -1 : 0;
}

/* Step 3: arithmetic mean per request over rows [off[r], off[r+1]), ascending n; empty -> 0. */
int laser_oracle_aggregate(const double* pmax, const int32_t* req_offsets, int64_t R, double* out_conf) {
    if (R < 0 || (R > 0 && (!pmax || !req_offsets || !out_conf))) return -1;
    for (int64_t r = 0; r < R; ++r) {
        int64_t b = req_offsets[r], e = req_offsets[r + 1];
        if (e < b) return -1;
        double s = 0.0;
        for (int64_t n = b; n < e; ++n) s += pmax[n];
        out_conf[r] = (e > b) ? s / (double)(e - b) : 0.0;
    }
    return 0;
}

/* Step 4: Eq. 5, then the clamp ("The final value is clamped"). */
double laser_oracle_tau_scalar(double load, const oracle_tau_params* p) {
    double lam = p->lambda_base - p->beta * tanh(p->gamma * (load - p->l_target) / p->l_target);
    if (lam < p->lambda_min) lam = p->lambda_min;
    if (lam > p->lambda_max) lam = p->lambda_max;
    return lam;
}

/* Eq. 5 without the clamp (for the pins that check where the clamp binds). */
double laser_oracle_tau_unclamped(double load, const oracle_tau_params* p) {
    return p->lambda_base - p->beta * tanh(p->gamma * (load - p->l_target) / p->l_target);
}

int laser_oracle_tau(const float* load, int64_t R, const oracle_tau_params* p, double* out_tau) {
    if (R < 0 || !p || (R > 0 && (!load || !out_tau))) return -1;
    for (int64_t r = 0; r < R; ++r) out_tau[r] = laser_oracle_tau_scalar((double)load[r], p);
    return 0;
}

/* Step 5: strict '>' ; NaN > x is false. */
int laser_oracle_exit(const double* conf, const double* tau, int64_t R, uint8_t* out_exit,
                      double* out_margin) {
    if (R < 0 || (R > 0 && (!conf || !tau || !out_exit))) return -1;
    for (int64_t r = 0; r < R; ++r) {
        out_exit[r] = (conf[r] > tau[r]) ? 1 : 0;
        if (out_margin) out_margin[r] = fabs(conf[r] - tau[r]);
    }
    return 0;
}

/*
 * Steps 1-5 in order.  Rows n >= req_offsets[R] are padding: argmax -1, pmax/gap2 NaN (DESIGN A11).
 * N_alloc = number of rows in `hidden`.
 */
int laser_oracle_probe(const float* hidden, const float* W, const int32_t* req_offsets,
                       const float* load, const oracle_tau_params* p, int64_t N_alloc, int d,
                       int64_t V, int64_t R, double* out_conf, int32_t* out_argmax,
                       uint8_t* out_exit, double* out_tau, double* out_pmax, double* out_gap2,
                       double* out_margin) {
    if (R < 0 || N_alloc < 0 || !p) return -1;
    int64_t N_valid = (R > 0) ? req_offsets[R] : 0;
    if (N_valid < 0 || N_valid > N_alloc) return -1;
    double* pmax = (double*)malloc(sizeof(double) * (size_t)(N_alloc > 0 ? N_alloc : 1));
    double* conf = (double*)malloc(sizeof(double) * (size_t)(R > 0 ? R : 1));
    double* tau = (double*)malloc(sizeof(double) * (size_t)(R > 0 ? R : 1));
    if (!pmax || !conf || !tau) { free(pmax); free(conf); free(tau); return -1; }
    int rc = 0;
    if (N_valid > 0)
        rc = laser_oracle_row_stats(hidden, W, N_valid, d, V, NULL, out_argmax, NULL, pmax,
                                    out_gap2, NULL);
    for (int64_t n = N_valid; n < N_alloc; ++n) {
        pmax[n] = NAN;
        if (out_argmax) out_argmax[n] = -1;
        if (out_gap2) out_gap2[n] = NAN;
    }
    if (!rc) rc = laser_oracle_aggregate(pmax, req_offsets, R, conf);
    if (!rc) rc = laser_oracle_tau(load, R, p, tau);
    if (!rc) rc = laser_oracle_exit(conf, tau, R, out_exit, out_margin);
    if (!rc) {
        if (out_conf) memcpy(out_conf, conf, sizeof(double) * (size_t)R);
        if (out_tau) memcpy(out_tau, tau, sizeof(double) * (size_t)R);
        if (out_pmax) memcpy(out_pmax, pmax, sizeof(double) * (size_t)N_alloc);
    }
    free(pmax); free(conf); free(tau);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * The merge operator (+) of the online-softmax statistics, restated on its own so that its
 * agreement with the single-pass definition above can be property-tested (pin P4 iii).  It is NOT
 * used by laser_oracle_probe.  (m,a,S) (+) (m',a',S') with the first operand covering lower vocab
 * indices:  M = max(m,m');  A = a if m >= m' else a'  (ties keep the lower index);
 *           S_out = S*exp(m-M) + S'*exp(m'-M).
 * An empty operand is (m=-inf, a=-1, S=0).
 * ---------------------------------------------------------------------------------------------- */
void laser_oracle_merge(double m1, int32_t a1, double S1, double m2, int32_t a2, double S2,
                        double* m, int32_t* a, double* S) {
    if (S1 == 0.0 && m1 == -INFINITY) { *m = m2; *a = a2; *S = S2; return; }
    if (S2 == 0.0 && m2 == -INFINITY) { *m = m1; *a = a1; *S = S1; return; }
    double M = (m1 >= m2) ? m1 : m2;
    *a = (m1 >= m2) ? a1 : a2;
    *m = M;
    *S = S1 * exp(m1 - M) + S2 * exp(m2 - M);
}

/* Row statistics of one row restricted to vocab range [v0, v1) (definition, single pass). */
int laser_oracle_row_stats_range(const float* hidden_row, const float* W, int d, int64_t v0,
                                 int64_t v1, double* out_m, int32_t* out_a, double* out_S) {
    if (d <= 0 || v1 < v0 || !hidden_row || !W) return -1;
    double* h = (double*)malloc(sizeof(double) * (size_t)d);
    if (!h) return -1;
    for (int k = 0; k < d; ++k) h[k] = (double)hidden_row[k];
    double m = -INFINITY; int64_t a = -1;
    for (int64_t v = v0; v < v1; ++v) {
        double x = dot_fp64(h, W + v * (int64_t)d, d);
        if (x != x) continue; /* NaN: DESIGN A12 */
        if (a < 0 || x > m) { m = x; a = v; }
    }
    double S = 0.0;
    for (int64_t v = v0; v < v1; ++v) S += exp(dot_fp64(h, W + v * (int64_t)d, d) - m);
    free(h);
    *out_m = m; *out_a = (int32_t)a; *out_S = S;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-1: other aggregates of the per-token max probabilities (DESIGN A1).  mode 0 = arithmetic
 * mean (the default above), 1 = geometric mean exp(mean(log pmax)), 2 = minimum.  Empty -> 0.
 * ---------------------------------------------------------------------------------------------- */
int laser_oracle_aggregate_mode(const double* pmax, const int32_t* req_offsets, int64_t R, int mode,
                                double* out_conf) {
    if (mode == 0) return laser_oracle_aggregate(pmax, req_offsets, R, out_conf);
    if (R < 0 || (R > 0 && (!pmax || !req_offsets || !out_conf))) return -1;
    for (int64_t r = 0; r < R; ++r) {
        int64_t b = req_offsets[r], e = req_offsets[r + 1];
        if (e < b) return -1;
        if (e == b) { out_conf[r] = 0.0; continue; }
        if (mode == 1) {
            double s = 0.0;
            for (int64_t n = b; n < e; ++n) s += log(pmax[n]);
            out_conf[r] = exp(s / (double)(e - b));
        } else if (mode == 2) {
            double mn = pmax[b];
            int nan = (pmax[b] != pmax[b]);
            for (int64_t n = b + 1; n < e; ++n) {
                if (pmax[n] != pmax[n]) nan = 1;
                if (pmax[n] < mn) mn = pmax[n];
            }
            out_conf[r] = nan ? NAN : mn;
        } else return -1;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-1, second half (DESIGN A2): the probability of a GIVEN token per row instead of the row
 * maximum - "the token probabilities" of the trial answer read as the probabilities
 * of the tokens that were emitted.  Plain softmax entry:
 *     p[n] = exp(l[n, t_n]) / sum_v exp(l[n, v]),   evaluated as exp(l_t - m) / sum_v exp(l_v - m).
 * A token id outside [0, V) has probability 0 (it is not in the vocabulary).  Under greedy decoding
 * t_n is the argmax and p equals pmax of step 2.
 * ---------------------------------------------------------------------------------------------- */
int laser_oracle_token_prob(const float* hidden, const float* W, const int32_t* token_ids, int64_t N,
                            int d, int64_t V, double* out_ptok) {
    if (N < 0 || d <= 0 || V <= 0 || (N > 0 && (!hidden || !W || !token_ids || !out_ptok))) return -1;
    int failed = 0;
#pragma omp parallel
    {
        double* h = (double*)malloc(sizeof(double) * (size_t)d);
        double* l = (double*)malloc(sizeof(double) * (size_t)V);
        if (!h || !l) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
#pragma omp for schedule(dynamic, 1)
            for (int64_t n = 0; n < N; ++n) {
                for (int k = 0; k < d; ++k) h[k] = (double)hidden[n * d + k];
                for (int64_t v = 0; v < V; ++v) l[v] = dot_fp64(h, W + v * (int64_t)d, d);
                double m = -INFINITY;
                for (int64_t v = 0; v < V; ++v)
                    if (l[v] > m) m = l[v];
                double S = 0.0;
                for (int64_t v = 0; v < V; ++v) S += exp(l[v] - m);
                int64_t t = token_ids[n];
                out_ptok[n] = (t >= 0 && t < V) ? exp(l[t] - m) / S : 0.0;
            }
        }
        free(h);
        free(l);
    }
    return failed ? -1 : 0;
}

/* ------------------------------------------------------------------------------------------------
 * NEXT-2: the control-plane steps either side of the probe in Algorithm 1.
 * ---------------------------------------------------------------------------------------------- */

/* EMA: Lbar(t) = alpha*L(t) + (1-alpha)*Lbar(t-1); Lbar(0) = lbar0 (0 in Alg.1
 * line 1).  Writes the whole trajectory out_lbar[0..T). */
int laser_oracle_ema(const double* L, int64_t T, double alpha, double lbar0, double* out_lbar) {
    if (T < 0 || (T > 0 && (!L || !out_lbar))) return -1;
    double prev = lbar0;
    for (int64_t t = 0; t < T; ++t) { prev = alpha * L[t] + (1.0 - alpha) * prev; out_lbar[t] = prev; }
    return 0;
}

typedef struct {
    double b_base, b_min, f_min, f_max, p_min, p_max, l_target;
} oracle_budget_params;

/* Eq. 7 */
double laser_oracle_f_diff(double prompt_tokens, const oracle_budget_params* q) {
    double f = q->f_min + (prompt_tokens - q->p_min) / (q->p_max - q->p_min) * (q->f_max - q->f_min);
    if (f < q->f_min) f = q->f_min;
    if (f > q->f_max) f = q->f_max;
    return f;
}

/* Eq. 8 */
double laser_oracle_f_load(double L, const oracle_budget_params* q) {
    double den = (L > 1.0) ? L : 1.0;
    double f = q->l_target / den;
    return (f < 1.0) ? f : 1.0;
}

/* Eq. 6: B = max{B_min, floor(B_base * f_diff * f_load)}; raw L(t) (DESIGN A14).
 * The floor is that of the real-number product.  Evaluated in binary the product can land one ulp
 * below an integer that the exact value reaches (paper defaults, |p| = 100: f_diff = 0.6 + 50/225*0.9
 * = 0.8 exactly and B = floor(10*0.8) = 8, while 0.6 + 50.0/225.0*0.9 = 0.7999999999999999), so the
 * floor is taken of product + 1e-9 (DESIGN A19) - far above any rounding error of three
 * multiplications (~1e-15) and far below the spacing of the exact values next to an integer. */
int laser_oracle_budget(const double* prompt_tokens, const double* L, int64_t R,
                        const oracle_budget_params* q, int32_t* out_B) {
    if (R < 0 || !q || (R > 0 && (!prompt_tokens || !L || !out_B))) return -1;
    for (int64_t r = 0; r < R; ++r) {
        double b = floor(q->b_base * laser_oracle_f_diff(prompt_tokens[r], q) * laser_oracle_f_load(L[r], q) + 1e-9);
        if (b < q->b_min) b = q->b_min;
        out_B[r] = (int32_t)b;
    }
    return 0;
}
