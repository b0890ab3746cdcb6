/*
 * laser_sim.h — C ABI of the batched serving simulation (SURVEY §8 f NEXT-4).
 *
 * The paper evaluates LASER by discrete-event simulation: Poisson (or three-phase burst) arrivals
 * into a single-server FIFO queue, every request served by Algorithm 1 with per-sample chunk times
 * and confidences measured beforehand; metrics are average latency, P95 latency, throughput and SLO
 * satisfaction at d = 30 s.  laser_sim_run() runs MANY
 * such queues at once on the GPU - one replication (seed x arrival rate x policy) per thread, the
 * sequential dependency of a queue staying inside its thread - so that a whole table of the paper's
 * kind (policies x loads x seeds) is one launch.
 *
 * Per replication r and request i (arrival order), with sample s = sample_id[i, r]:
 *
 *   start = max(arrival, finish of request i-1)                     single server, FIFO
 *   L(t)  = #{arrivals <= t} - i                                    requests in the system (DESIGN S1)
 *   B     = max{B_min, floor(B_base * f_diff(|p_s|) * f_load(L(start)))}   Eq. 6-8, PAPER.md:152-173;
 *           or policy.fixed_budget; capped at K
 *   t     = start + t_prefill[s]
 *   for k = 0 .. B-1:   t += chunk_time[s, k]
 *                       Lbar = alpha * L(t) + (1 - alpha) * Lbar    PAPER.md:148 (one Lbar per queue, 0 at start)
 *                       lambda = clamp(Eq. 5 (Lbar))
 *                       stop if early_exit and conf[s, k] > lambda  PAPER.md:122 (strict)
 *   finish = t + t_conclusion[s]
 *
 * All times, the EMA, Eq. 5 and Eq. 6-8 are evaluated in IEEE double in exactly this order (no
 * fused multiply-add), the float32 pool values widened exactly.  Same status codes as laser_probe.h.
 */
#ifndef LASER_SIM_H_
#define LASER_SIM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One serving policy.  Defaults (laser_sim_policy_default): LASER with the paper's parameters
 * (PAPER.md:166, 195).  Fixed-High / Fixed-Low: beta = 0, lambda_base = 0.95 / 0.90,
 * adaptive_budget = 0.  Vanilla: early_exit = 0, adaptive_budget = 0, fixed_budget = K. */
typedef struct {
    double lambda_base, beta, gamma, l_target, lambda_min, lambda_max; /* Eq. 5 + clamp           */
    double alpha;                                                      /* EMA, 0.3               */
    double b_base, b_min, f_min, f_max, p_min, p_max, budget_l_target; /* Eq. 6-8                */
    int32_t early_exit;      /* 0: never exit on confidence                                      */
    int32_t adaptive_budget; /* 0: every request gets fixed_budget chunks                        */
    int32_t fixed_budget;
    int32_t pad_;
} laser_sim_policy;

typedef struct {
    int32_t n_rep;  /* replications (queues) simulated at once                                   */
    int32_t n_req;  /* requests per replication                                                  */
    int32_t S;      /* samples in the pool                                                       */
    int32_t K;      /* reasoning chunks per sample (hard cap of every budget)                    */
} laser_sim_dims;

enum { LASER_SIM_MAX_POLICIES = 16, LASER_SIM_SUMMARY_COLS = 5, LASER_SIM_MAX_P95_REQUESTS = 8192 };

int laser_sim_policy_default(laser_sim_policy* out);

/*
 * Simulate dims->n_rep queues.  Asynchronous on `stream`; two kernels (queues, then P95 selection).
 *
 *   arrival       device, double [n_req, n_rep] (replication fastest), ascending along n_req
 *   sample_id     device, int32  [n_req, n_rep], values in [0, S)
 *   policy_id     device, int32  [n_rep], values in [0, n_pol)
 *   policies      HOST, [n_pol], n_pol <= LASER_SIM_MAX_POLICIES; copied by value into the launch
 *   chunk_time    device, float  [S, K]   seconds to generate chunk k and evaluate its trial answer
 *   conf          device, float  [S, K]   confidence at the ATP that ends chunk k
 *   prompt_tokens device, int32  [S];  t_prefill, t_conclusion  device, float [S]
 *   deadline      SLO deadline in seconds (the paper: 30)
 *   out_finish    device, double [n_req, n_rep]
 *   out_chunks    device, int32  [n_req, n_rep]  chunks generated
 *   out_exited_opt device, uint8 [n_req, n_rep] or NULL: 1 = confidence exit, 0 = budget exhausted
 *   out_budget_opt device, int32 [n_req, n_rep] or NULL: the budget B (after the cap at K)
 *   out_summary   device, double [n_rep, 5]: mean latency, P95 latency (nearest rank; a shared-memory sort up to
 *                 LASER_SIM_MAX_P95_REQUESTS requests per queue, a radix select over global memory above), throughput n_req / (last finish - first
 *                 arrival), share of requests with latency <= deadline, mean chunks generated
 *
 * Out-of-range sample or policy ids are a precondition violation (ids are clamped, never read out
 * of bounds).  Returns LASER_E_NULL / LASER_E_DIMS / LASER_E_PARAMS / LASER_E_ARCH / LASER_E_CUDA.
 */
int laser_sim_run(const double* arrival, const int32_t* sample_id, const int32_t* policy_id,
                  const laser_sim_policy* policies, int32_t n_pol, const float* chunk_time,
                  const float* conf, const int32_t* prompt_tokens, const float* t_prefill,
                  const float* t_conclusion, const laser_sim_dims* dims, double deadline,
                  double* out_finish, int32_t* out_chunks, uint8_t* out_exited_opt,
                  int32_t* out_budget_opt, double* out_summary, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* LASER_SIM_H_ */
