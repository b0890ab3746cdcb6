/*
 * sanitize_driver.c — runs every entry point of the fp64 oracle (laser_oracle.c, laser_sim_oracle.c)
 * on small inputs, including the edge cases the parity tests rely on (empty batches, empty requests,
 * one-row requests, V = 1, padding rows, NaN rows, out-of-vocabulary token ids), so that the oracle
 * can be built with -fsanitize=address,undefined and checked for out-of-bounds accesses, leaks and
 * undefined behaviour.  It also re-checks a few closed forms of the paper's
 * mathematics, so that a sanitized build that silently computes something else is caught too:
 *   uniform logits give pmax = 1/V and the lowest index (P1), a scaled identity gives
 *   1/(1+(V-1)e^-M) (P2), Eq. 5 at Lbar = L_target gives lambda_base and stays inside the clamp
 *   (PAPER.md:100-103, 144), Eq. 6-8 at |p| = 100 gives 8 (DESIGN A19).
 *
 * TEST INFRASTRUCTURE (like the oracle itself).  Built and run by tests/test_oracle_sanitizers.py:
 *   gcc -std=c11 -g -O1 -fsanitize=address,undefined -fno-sanitize-recover=all -fopenmp \
 *       oracle/laser_oracle.c oracle/laser_sim_oracle.c oracle/sanitize_driver.c -lm
 * Exit status 0 = every check passed (and the sanitizers stayed silent).
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef struct { double lambda_base, beta, gamma, l_target, lambda_min, lambda_max; } oracle_tau_params;
typedef struct { double b_base, b_min, f_min, f_max, p_min, p_max, l_target; } oracle_budget_params;
typedef struct {
    double lambda_base, beta, gamma, l_target, lambda_min, lambda_max, alpha;
    double b_base, b_min, f_min, f_max, p_min, p_max, budget_l_target;
    int32_t early_exit, adaptive_budget, fixed_budget, pad_;
} sim_policy;

int laser_oracle_num_threads(void);
int laser_oracle_row_stats(const float*, const float*, int64_t, int, int64_t, double*, int32_t*, double*, double*,
                           double*, double*);
int laser_oracle_aggregate(const double*, const int32_t*, int64_t, double*);
int laser_oracle_aggregate_mode(const double*, const int32_t*, int64_t, int, double*);
double laser_oracle_tau_scalar(double, const oracle_tau_params*);
double laser_oracle_tau_unclamped(double, const oracle_tau_params*);
int laser_oracle_tau(const float*, int64_t, const oracle_tau_params*, double*);
int laser_oracle_exit(const double*, const double*, int64_t, uint8_t*, double*);
int laser_oracle_probe(const float*, const float*, const int32_t*, const float*, const oracle_tau_params*, int64_t,
                       int, int64_t, int64_t, double*, int32_t*, uint8_t*, double*, double*, double*, double*);
void laser_oracle_merge(double, int32_t, double, double, int32_t, double, double*, int32_t*, double*);
int laser_oracle_row_stats_range(const float*, const float*, int, int64_t, int64_t, double*, int32_t*, double*);
int laser_oracle_token_prob(const float*, const float*, const int32_t*, int64_t, int, int64_t, double*);
int laser_oracle_ema(const double*, int64_t, double, double, double*);
double laser_oracle_f_diff(double, const oracle_budget_params*);
double laser_oracle_f_load(double, const oracle_budget_params*);
int laser_oracle_budget(const double*, const double*, int64_t, const oracle_budget_params*, int32_t*);
int laser_sim_oracle_queue(const double*, const int32_t*, int64_t, const float*, const float*, const int32_t*,
                           const float*, const float*, int64_t, int32_t, const sim_policy*, double*, int32_t*,
                           uint8_t*, int32_t*, double*);
int laser_sim_oracle_summary(const double*, const double*, const int32_t*, int64_t, double, double*);

static int failures = 0;
#define CHECK(cond) do { if (!(cond)) { fprintf(stderr, "CHECK failed line %d: %s\n", __LINE__, #cond); ++failures; } } while (0)

static uint64_t rng_state = 0x9E3779B97F4A7C15ull;
static float frand(void) {   /* xorshift: uniform in [-1, 1) */
    rng_state ^= rng_state << 13; rng_state ^= rng_state >> 7; rng_state ^= rng_state << 17;
    return (float)((double)(rng_state >> 11) / 9007199254740992.0 * 2.0 - 1.0);
}

int main(void) {
    const oracle_tau_params tp = {0.95, 0.04, 1.0, 10.0, 0.88, 0.97};
    CHECK(laser_oracle_num_threads() >= 1);

    /* ---- P1: uniform logits, several shapes incl. V = 1 */
    for (int V = 1; V <= 33; V += 8) {
        const int d = 8, N = 3;
        float* h = calloc((size_t)N * d, sizeof *h);
        float* W = malloc((size_t)V * d * sizeof *W);
        for (int i = 0; i < V * d; ++i) W[i] = frand();
        double m[3], S[3], pm[3], gap[3]; int32_t a[3];
        CHECK(laser_oracle_row_stats(h, W, N, d, V, m, a, S, pm, gap, NULL) == 0);
        for (int n = 0; n < N; ++n) CHECK(a[n] == 0 && fabs(pm[n] - 1.0 / V) < 1e-15);
        free(h); free(W);
    }
    /* ---- P2: scaled identity */
    {
        const int V = 16, d = 16; const double M = 5.0;
        float W[16 * 16] = {0}, h[16] = {0};
        for (int i = 0; i < V; ++i) W[i * d + i] = (float)M;
        h[11] = 1.0f;
        double m, S, pm, gap, logits[16]; int32_t a;
        CHECK(laser_oracle_row_stats(h, W, 1, d, V, &m, &a, &S, &pm, &gap, logits) == 0);
        CHECK(a == 11 && fabs(pm - 1.0 / (1.0 + (V - 1) * exp(-M))) < 1e-15 && fabs(gap - M) < 1e-15);
        /* chunked merge equals the single pass; token probability at the argmax equals pmax */
        double m1, S1, m2, S2, mm, SS; int32_t a1, a2, aa;
        CHECK(laser_oracle_row_stats_range(h, W, d, 0, 7, &m1, &a1, &S1) == 0);
        CHECK(laser_oracle_row_stats_range(h, W, d, 7, 16, &m2, &a2, &S2) == 0);
        laser_oracle_merge(m1, a1, S1, m2, a2, S2, &mm, &aa, &SS);
        CHECK(aa == 11 && fabs(1.0 / SS - pm) < 1e-15);
        CHECK(laser_oracle_row_stats_range(h, W, d, 3, 3, &m1, &a1, &S1) == 0);   /* empty range */
        int32_t tok[1] = {11}; double pt;
        CHECK(laser_oracle_token_prob(h, W, tok, 1, d, V, &pt) == 0 && pt == pm);
        tok[0] = -5;
        CHECK(laser_oracle_token_prob(h, W, tok, 1, d, V, &pt) == 0 && pt == 0.0);   /* out of vocabulary */
        tok[0] = V;
        CHECK(laser_oracle_token_prob(h, W, tok, 1, d, V, &pt) == 0 && pt == 0.0);
    }
    /* ---- whole pipeline: ragged requests, an empty one, padding rows, a NaN row */
    {
        const int d = 24, V = 301, R = 5, N = 20;
        const int32_t off[6] = {0, 4, 4, 5, 12, 15};           /* request 1 empty; rows 15..19 padding */
        float* h = malloc((size_t)N * d * sizeof *h);
        float* W = malloc((size_t)V * d * sizeof *W);
        for (int i = 0; i < N * d; ++i) h[i] = frand() * 3.0f;
        for (int i = 0; i < V * d; ++i) W[i] = frand();
        h[13 * d + 2] = NAN;                                     /* poisons request 4 only */
        const float load[5] = {0.0f, 5.0f, 10.0f, 20.0f, 1e6f};
        double conf[5], tau[5], pm[20], gap[20], margin[5]; int32_t am[20]; uint8_t ex[5];
        CHECK(laser_oracle_probe(h, W, off, load, &tp, N, d, V, R, conf, am, ex, tau, pm, gap, margin) == 0);
        CHECK(conf[1] == 0.0 && ex[1] == 0);
        CHECK(isnan(conf[4]) && ex[4] == 0 && !isnan(conf[3]));
        for (int n = 15; n < 20; ++n) CHECK(am[n] == -1 && isnan(pm[n]));
        for (int r = 0; r < R; ++r) CHECK(tau[r] >= 0.88 && tau[r] <= 0.97);
        CHECK(tau[2] == 0.95 && tau[0] == 0.97);                /* Eq. 5 at L_target; upper clamp at 0 */
        double c1[5], c2[5];
        CHECK(laser_oracle_aggregate(pm, off, R, conf) == 0);
        CHECK(laser_oracle_aggregate_mode(pm, off, R, 1, c1) == 0 && laser_oracle_aggregate_mode(pm, off, R, 2, c2) == 0);
        CHECK(c2[0] <= c1[0] + 1e-15 && c1[0] <= conf[0] + 1e-15);   /* min <= geometric <= arithmetic mean */
        CHECK(conf[2] == pm[4]);                                 /* one-row request */
        CHECK(laser_oracle_probe(h, W, off, load, &tp, N, d, V, 0, conf, am, ex, tau, pm, gap, margin) == 0);   /* R = 0 */
        CHECK(laser_oracle_row_stats(h, W, 0, d, V, NULL, NULL, NULL, NULL, NULL, NULL) == 0);                   /* N = 0 */
        free(h); free(W);
    }
    /* ---- Eq. 5: monotone, clamped, strict exit */
    {
        double prev = 1.0;
        for (int i = 0; i <= 400; ++i) {
            const double t = laser_oracle_tau_scalar(0.1 * i, &tp);
            CHECK(t <= prev + 1e-15 && t >= 0.88 && t <= 0.97);
            prev = t;
        }
        CHECK(fabs(laser_oracle_tau_unclamped(20.0, &tp) - (0.95 - 0.04 * tanh(1.0))) < 1e-15);
        const double conf[3] = {0.95, nextafter(0.95, 1.0), NAN}, tau[3] = {0.95, 0.95, 0.5};
        uint8_t ex[3]; double mg[3];
        CHECK(laser_oracle_exit(conf, tau, 3, ex, mg) == 0 && ex[0] == 0 && ex[1] == 1 && ex[2] == 0);
        float ld[2] = {10.0f, 40.0f}; double tt[2];
        CHECK(laser_oracle_tau(ld, 2, &tp, tt) == 0 && tt[0] == 0.95 && laser_oracle_tau(ld, 0, &tp, tt) == 0);
    }
    /* ---- EMA, Eq. 6-8 */
    {
        const double L[4] = {7, 7, 7, 7}; double lb[4];
        CHECK(laser_oracle_ema(L, 4, 0.3, 0.0, lb) == 0 && fabs(lb[3] - 7.0 * (1.0 - pow(0.7, 4))) < 1e-14);
        const oracle_budget_params q = {10, 2, 0.6, 1.5, 50, 275, 10};
        CHECK(laser_oracle_f_diff(50, &q) == 0.6 && laser_oracle_f_diff(275, &q) == 1.5 && laser_oracle_f_load(20, &q) == 0.5);
        const double p[4] = {100, 65, 50, 275}, Lq[4] = {5, 11, 1000, 0}; int32_t B[4];
        CHECK(laser_oracle_budget(p, Lq, 4, &q, B) == 0 && B[0] == 8 && B[1] == 6 && B[2] == 2 && B[3] == 15);
    }
    /* ---- serving simulation: a small queue, then its summary */
    {
        enum { S = 3, K = 4, n = 12 };
        const float ct[S * K] = {0.3f, 0.4f, 0.2f, 0.5f, 0.1f, 0.2f, 0.3f, 0.4f, 0.5f, 0.5f, 0.5f, 0.5f};
        const float cf[S * K] = {0.5f, 0.99f, 0.99f, 0.99f, 0.2f, 0.3f, 0.4f, 0.5f, 0.93f, 0.94f, 0.96f, 0.98f};
        const int32_t pt[S] = {40, 150, 300};
        const float tpre[S] = {0.03f, 0.05f, 0.08f}, tcon[S] = {0.4f, 0.5f, 0.6f};
        double arr[n], fin[n], mg[n], out[5]; int32_t sid[n], ch[n], bud[n]; uint8_t exd[n];
        for (int i = 0; i < n; ++i) { arr[i] = 0.25 * i; sid[i] = i % S; }
        sim_policy pol = {0.95, 0.04, 1.0, 10.0, 0.88, 0.97, 0.3, 10, 2, 0.6, 1.5, 50, 275, 10, 1, 1, 10, 0};
        CHECK(laser_sim_oracle_queue(arr, sid, n, ct, cf, pt, tpre, tcon, S, K, &pol, fin, ch, exd, bud, mg) == 0);
        for (int i = 0; i < n; ++i) CHECK(ch[i] >= 1 && ch[i] <= K && fin[i] > arr[i] && (i == 0 || fin[i] >= fin[i - 1]));
        CHECK(laser_sim_oracle_summary(arr, fin, ch, n, 30.0, out) == 0 && out[0] > 0 && out[1] >= out[0] * 0.5 && out[3] <= 1.0);
        pol.early_exit = 0; pol.adaptive_budget = 0; pol.fixed_budget = 7;       /* budget capped at K */
        CHECK(laser_sim_oracle_queue(arr, sid, n, ct, cf, pt, tpre, tcon, S, K, &pol, fin, ch, exd, bud, mg) == 0);
        for (int i = 0; i < n; ++i) CHECK(ch[i] == K && exd[i] == 0);
        CHECK(laser_sim_oracle_queue(arr, sid, 0, ct, cf, pt, tpre, tcon, S, K, &pol, fin, ch, exd, bud, mg) == 0);   /* n = 0 */
    }
    if (failures) { fprintf(stderr, "%d check(s) failed\n", failures); return 1; }
    printf("oracle sanitize driver: all checks passed\n");
    return 0;
}
