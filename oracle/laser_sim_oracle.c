/*
 * laser_sim_oracle.c — fp64 CPU ORACLE of the serving simulation the paper evaluates LASER with:
 * Algorithm 1 run for every request of a single-server FIFO queue (SURVEY §8 f NEXT-4).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (see laser_oracle.c).  It shares no code with the CUDA
 * path.  Citations are /root/reference/PAPER.md line numbers; "DESIGN S<n>" are the readings listed
 * in DESIGN.md §10 where the paper is silent.
 *
 * The paper's evaluation vehicle (§5.1) is a discrete-event simulation: per-sample
 * inference times and accuracy are measured once, then Poisson arrivals are played into a
 * single-server FIFO queue with an SLO deadline d = 30 s; the metrics are average latency, P95
 * latency, throughput, SLO satisfaction.  Here the per-sample data is a POOL of S
 * samples, each with its prompt length, prefill time, conclusion time and, per reasoning chunk k, the
 * chunk's duration and the confidence measured at the ATP that ends it (Eq. 2, PAPER.md:63-68:
 * t_inf = t_prefill + sum_k t_chunk_k + t_conclusion; latency l = waiting time + t_inf).
 *
 * One replication = one queue.  For request i (in arrival order) with sample s = sample_id[i]:
 *
 *   start  = max(arrival_i, finish_{i-1})                     single server, FIFO, non-preemptive
 *   L(t)   = #{j : arrival_j <= t} - i                        requests in the system at time t: all
 *            that have arrived minus the i that have finished (request i itself counts)  DESIGN S1
 *   B_i    = AllocateBudget(|p_s|, L(start))  Eq. 6-8          PAPER.md:114 (Alg. 1 line 3), 152-173;
 *            or the fixed budget when the policy disables the allocator; capped at the pool's K
 *   t      = start + t_prefill_s ; k = 0
 *   while k < B_i:                                             PAPER.md:116-131 (Alg. 1 lines 4-12)
 *       t += t_chunk[s][k]                                     generate chunk k+1 up to the next ATP
 *       Lbar = alpha * L(t) + (1 - alpha) * Lbar               EMA; ONE Lbar per
 *                                                              queue, initialised to 0
 *       lambda = clamp(Eq. 5 (Lbar))
 *       k += 1                                                 chunks generated so far
 *       if early_exit and conf[s][k-1] > lambda: exited; break PAPER.md:122 (strict >)
 *   finish_i = t + t_conclusion_s                              conclusion after an exit or when the
 *                                                              budget is exhausted
 *
 * Everything is IEEE double, evaluated in exactly the order written (compile with
 * -ffp-contract=off); the float32 pool values are widened exactly.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>

typedef struct {
    /* Eq. 5 + clamp */
    double lambda_base, beta, gamma, l_target, lambda_min, lambda_max;
    /* EMA */
    double alpha;
    /* Eq. 6-8 */
    double b_base, b_min, f_min, f_max, p_min, p_max, budget_l_target;
    /* switches */
    int32_t early_exit;       /* 0: Vanilla - never exit on confidence                        */
    int32_t adaptive_budget;  /* 0: every request gets fixed_budget chunks (no Eq. 6)          */
    int32_t fixed_budget;
    int32_t pad_;
} sim_policy;

static double sim_tau(double lbar, const sim_policy* p) {
    double lam = p->lambda_base - p->beta * tanh(p->gamma * (lbar - p->l_target) / p->l_target);
    if (lam < p->lambda_min) lam = p->lambda_min;
    if (lam > p->lambda_max) lam = p->lambda_max;
    return lam;
}

static int32_t sim_budget(double prompt_tokens, double L, const sim_policy* p) {
    double f_diff = p->f_min + (prompt_tokens - p->p_min) / (p->p_max - p->p_min) * (p->f_max - p->f_min);
    if (f_diff < p->f_min) f_diff = p->f_min;
    if (f_diff > p->f_max) f_diff = p->f_max;
    double den = (L > 1.0) ? L : 1.0;
    double f_load = p->budget_l_target / den;
    if (f_load > 1.0) f_load = 1.0;
    double b = floor(p->b_base * f_diff * f_load + 1e-9);   /* floor of the real product, DESIGN A19 */
    if (b < p->b_min) b = p->b_min;
    return (int32_t)b;
}

/*
 * One replication.  arrival[n] ascending; sample_id[n] in [0, S).  Pool arrays: chunk_time, conf
 * [S, K] row-major float32; prompt_tokens int32 [S]; t_prefill, t_conclusion float32 [S].
 * Outputs (each [n], any may be NULL): finish, chunks (generated), exited (1 = confidence exit,
 * 0 = budget exhausted), budget (after the cap at K), margin = min over the request's ATPs of
 * |conf - lambda| (how close any of its decisions came to flipping).
 * Returns 0, or -1 on bad arguments.
 */
int laser_sim_oracle_queue(const double* arrival, const int32_t* sample_id, int64_t n,
                           const float* chunk_time, const float* conf, const int32_t* prompt_tokens,
                           const float* t_prefill, const float* t_conclusion, int64_t S, int32_t K,
                           const sim_policy* pol, double* finish, int32_t* chunks, uint8_t* exited,
                           int32_t* budget, double* margin) {
    if (n < 0 || S <= 0 || K <= 0 || !pol) return -1;
    if (n > 0 && (!arrival || !sample_id || !chunk_time || !conf || !prompt_tokens || !t_prefill ||
                  !t_conclusion))
        return -1;
    double lbar = 0.0, prev_finish = -INFINITY;
    const double one_minus_alpha = 1.0 - pol->alpha;
    int64_t arrived = 0; /* number of requests with arrival <= the last time queried */
    for (int64_t i = 0; i < n; ++i) {
        const int64_t s = sample_id[i];
        if (s < 0 || s >= S) return -1;
        if (i > 0 && arrival[i] < arrival[i - 1]) return -1;
        double t = (arrival[i] > prev_finish) ? arrival[i] : prev_finish;
        while (arrived < n && arrival[arrived] <= t) ++arrived;
        double L = (double)(arrived - i);
        int32_t B = pol->adaptive_budget ? sim_budget((double)prompt_tokens[s], L, pol) : pol->fixed_budget;
        if (B > K) B = K;
        if (B < 0) B = 0;
        t = t + (double)t_prefill[s];
        int32_t k = 0;
        uint8_t ex = 0;
        double mg = INFINITY;
        while (k < B) {
            t = t + (double)chunk_time[s * K + k];
            while (arrived < n && arrival[arrived] <= t) ++arrived;
            L = (double)(arrived - i);
            lbar = pol->alpha * L + one_minus_alpha * lbar;
            const double lam = sim_tau(lbar, pol);
            const double c = (double)conf[s * K + k];
            const double dm = fabs(c - lam);
            if (dm < mg) mg = dm;
            k += 1;
            if (pol->early_exit && c > lam) { ex = 1; break; }
        }
        t = t + (double)t_conclusion[s];
        prev_finish = t;
        if (finish) finish[i] = t;
        if (chunks) chunks[i] = k;
        if (exited) exited[i] = ex;
        if (budget) budget[i] = B;
        if (margin) margin[i] = mg;
    }
    return 0;
}

static int cmp_double(const void* a, const void* b) {
    const double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}

/*
 * The paper's system metrics for one replication: out[0] average latency
 * (sum in request order / n), out[1] P95 latency (nearest rank: the ceil(0.95 n)-th smallest),
 * out[2] throughput n / (last finish - first arrival), out[3] SLO satisfaction = share of requests
 * with latency <= deadline, out[4] average chunks generated.  latency_i = finish_i - arrival_i.
 */
int laser_sim_oracle_summary(const double* arrival, const double* finish, const int32_t* chunks,
                             int64_t n, double deadline, double* out) {
    if (n <= 0 || !arrival || !finish || !chunks || !out) return -1;
    double* lat = (double*)malloc(sizeof(double) * (size_t)n);
    if (!lat) return -1;
    double sum = 0.0, csum = 0.0;
    int64_t ok = 0;
    for (int64_t i = 0; i < n; ++i) {
        lat[i] = finish[i] - arrival[i];
        sum = sum + lat[i];
        csum = csum + (double)chunks[i];
        if (lat[i] <= deadline) ++ok;
    }
    qsort(lat, (size_t)n, sizeof(double), cmp_double);
    int64_t rank = (int64_t)ceil(0.95 * (double)n);
    if (rank < 1) rank = 1;
    out[0] = sum / (double)n;
    out[1] = lat[rank - 1];
    out[2] = (double)n / (finish[n - 1] - arrival[0]);
    out[3] = (double)ok / (double)n;
    out[4] = csum / (double)n;
    free(lat);
    return 0;
}
