// laser_sim.cu — batched serving simulation (include/laser_sim.h): Algorithm 1 of the LASER paper
// over many independent single-server FIFO queues, one queue per thread.
//
//  laser_sim_queue_kernel   thread r walks the requests of replication r in arrival order; all
//                           per-request arrays are laid out [n_req, n_rep] so that the threads of a
//                           warp, which advance through i in lock step, read and write coalesced.
//                           The pool (chunk times, confidences: S*K floats each, a few tens of KB)
//                           is read through the read-only path and stays in L1/L2.
//  laser_sim_p95_kernel     one block per replication: latencies -> shared memory -> bitonic sort
//                           -> nearest-rank 95th percentile.
//
// Every double operation that the oracle performs is performed here in the same order with the
// round-to-nearest intrinsics (__dadd_rn, __dmul_rn, ...), which the compiler never contracts into
// fused multiply-adds, so finish times and summaries are bit-identical to the fp64 CPU oracle as
// long as no exit decision differs (tanh may differ in the last ulp between libraries).
#include "../../include/laser_sim.h"
#include "../../include/laser_probe.h"

#include <cuda_runtime.h>
#include <math_constants.h>

#include <cmath>
#include <cstdint>

namespace {

struct SimParams {
    int lanes;       // replications per warp (see laser_sim_queue_kernel)
    const double* arrival;
    const int32_t* sample_id;
    const int32_t* policy_id;
    const float* chunk_time;
    const float* conf;
    const int32_t* prompt_tokens;
    const float* t_prefill;
    const float* t_conclusion;
    double* out_finish;
    int32_t* out_chunks;
    uint8_t* out_exited;
    int32_t* out_budget;
    double* out_summary;
    double deadline;
    int32_t n_rep, n_req, S, K, n_pol;
    laser_sim_policy pol[LASER_SIM_MAX_POLICIES];
};

// Eq. 5, then the clamp.
__device__ __forceinline__ double sim_tau(double lbar, const laser_sim_policy& p) {
    const double x = __ddiv_rn(__dmul_rn(p.gamma, __dsub_rn(lbar, p.l_target)), p.l_target);
    double lam = __dsub_rn(p.lambda_base, __dmul_rn(p.beta, tanh(x)));
    if (lam < p.lambda_min) lam = p.lambda_min;
    if (lam > p.lambda_max) lam = p.lambda_max;
    return lam;
}

// Eq. 6-8: B = max{B_min, floor(B_base * f_diff * f_load)}.
__device__ __forceinline__ int32_t sim_budget(double prompt_tokens, double L, const laser_sim_policy& p) {
    double f_diff = __dadd_rn(p.f_min, __dmul_rn(__ddiv_rn(__dsub_rn(prompt_tokens, p.p_min),
                                                           __dsub_rn(p.p_max, p.p_min)),
                                                 __dsub_rn(p.f_max, p.f_min)));
    if (f_diff < p.f_min) f_diff = p.f_min;
    if (f_diff > p.f_max) f_diff = p.f_max;
    const double den = (L > 1.0) ? L : 1.0;
    double f_load = __ddiv_rn(p.budget_l_target, den);
    if (f_load > 1.0) f_load = 1.0;
    // floor of the real-number product (include/laser_probe.h, LASER_BUDGET_FLOOR_EPS; DESIGN A19)
    double b = floor(__dadd_rn(__dmul_rn(__dmul_rn(p.b_base, f_diff), f_load), LASER_BUDGET_FLOOR_EPS));
    if (b < p.b_min) b = p.b_min;
    return static_cast<int32_t>(b);
}

constexpr int kSimThreads = 32;   // one warp per block: replications spread over all SMs

// Only the first `lanes` lanes of a warp simulate (lanes = 1, 2, 4, ... 32, chosen by the host so that
// the warps fill the machine's warp slots): the lanes of a warp walk the request index in lock step and
// wait for the lane whose request generates the most chunks, so the fewer replications share a warp
// the less of that wait there is (one per warp: none), and a latency-bound kernel loses nothing by
// running more, emptier warps.
__global__ void __launch_bounds__(kSimThreads)
laser_sim_queue_kernel(const __grid_constant__ SimParams q) {
    if (static_cast<int>(threadIdx.x) >= q.lanes) return;
    const int r = blockIdx.x * q.lanes + threadIdx.x;
    if (r >= q.n_rep) return;
    const int n = q.n_req, R = q.n_rep, K = q.K;
    int pid = __ldg(q.policy_id + r);
    pid = min(max(pid, 0), q.n_pol - 1);
    const laser_sim_policy& pol = q.pol[pid];
    const double one_minus_alpha = __dsub_rn(1.0, pol.alpha);
    const bool need_tanh = pol.beta != 0.0;
    const double lam_const = fmin(fmax(pol.lambda_base, pol.lambda_min), pol.lambda_max);

    double lbar = 0.0, prev_finish = -CUDART_INF, lat_sum = 0.0, chunk_sum = 0.0;
    double first_arrival = 0.0, last_finish = 0.0;
    long long ok = 0;

    // Arrival counter: `arrived` = requests with arrival <= the last time queried.  The next kWin
    // arrival times are kept in registers and refilled by kWin independent loads, so that advancing
    // the counter over a burst of arrivals costs one memory latency per kWin arrivals, not one each.
    constexpr int kWin = 4;
    int arrived = 0, win_base = 0;      // win[] holds arrival[win_base .. win_base + kWin)
    double win[kWin];
    auto refill = [&](int base) {
        win_base = base;
#pragma unroll
        for (int j = 0; j < kWin; ++j)
            win[j] = (base + j < n) ? __ldg(q.arrival + static_cast<size_t>(base + j) * R + r) : CUDART_INF;
    };
    auto count_arrivals = [&](double t) {
        while (true) {
            int adv = 0;
#pragma unroll
            for (int j = 0; j < kWin; ++j)           // arrivals ascend: a prefix of the window is <= t
                adv += (win_base + j >= arrived && win[j] <= t) ? 1 : 0;
            arrived += adv;
            if (arrived < win_base + kWin || arrived >= n) break;
            refill(arrived);                         // window exhausted: look at the next kWin
        }
    };
    refill(0);

    // Request i + 1's own inputs are fetched while request i is simulated.
    double a_next = (n > 0) ? __ldg(q.arrival + r) : 0.0;
    int s_next = (n > 0) ? min(max(__ldg(q.sample_id + r), 0), q.S - 1) : 0;
    for (int i = 0; i < n; ++i) {
        const size_t o = static_cast<size_t>(i) * R + r;
        const double a = a_next;
        const int s = s_next;
        const double prompt = static_cast<double>(__ldg(q.prompt_tokens + s));
        const double t_pre = static_cast<double>(__ldg(q.t_prefill + s));
        const double t_conc = static_cast<double>(__ldg(q.t_conclusion + s));
        if (i + 1 < n) {
            a_next = __ldg(q.arrival + o + R);
            s_next = min(max(__ldg(q.sample_id + o + R), 0), q.S - 1);
        }
        if (i == 0) first_arrival = a;
        double t = (a > prev_finish) ? a : prev_finish;
        count_arrivals(t);
        double L = static_cast<double>(arrived - i);
        int B = pol.adaptive_budget ? sim_budget(prompt, L, pol) : pol.fixed_budget;
        B = min(B, K);
        B = max(B, 0);
        t = __dadd_rn(t, t_pre);
        int k = 0;
        uint8_t ex = 0;
        const float* ct = q.chunk_time + static_cast<size_t>(s) * K;
        const float* cf = q.conf + static_cast<size_t>(s) * K;
        // chunk k + 1's time and confidence are in flight while chunk k is evaluated
        float ct_k = (B > 0) ? __ldg(ct) : 0.f, cf_k = (B > 0) ? __ldg(cf) : 0.f;
        while (k < B) {
            const float ct_n = (k + 1 < B) ? __ldg(ct + k + 1) : 0.f;
            const float cf_n = (k + 1 < B) ? __ldg(cf + k + 1) : 0.f;
            t = __dadd_rn(t, static_cast<double>(ct_k));
            count_arrivals(t);
            L = static_cast<double>(arrived - i);
            lbar = __dadd_rn(__dmul_rn(pol.alpha, L), __dmul_rn(one_minus_alpha, lbar));
            ++k;
            if (pol.early_exit) {
                // beta == 0 (fixed-threshold policies): beta * tanh(.) is exactly 0, the threshold is
                // the clamped constant - same value, without the tanh
                const double lam = need_tanh ? sim_tau(lbar, pol) : lam_const;
                if (static_cast<double>(cf_k) > lam) { ex = 1; break; }
            }
            ct_k = ct_n; cf_k = cf_n;
        }
        t = __dadd_rn(t, t_conc);
        prev_finish = t;
        last_finish = t;
        q.out_finish[o] = t;
        q.out_chunks[o] = k;
        if (q.out_exited) q.out_exited[o] = ex;
        if (q.out_budget) q.out_budget[o] = B;
        const double lat = __dsub_rn(t, a);
        lat_sum = __dadd_rn(lat_sum, lat);
        chunk_sum = __dadd_rn(chunk_sum, static_cast<double>(k));
        if (lat <= q.deadline) ++ok;
    }
    double* out = q.out_summary + static_cast<size_t>(r) * LASER_SIM_SUMMARY_COLS;
    const double dn = static_cast<double>(n);
    out[0] = __ddiv_rn(lat_sum, dn);
    out[1] = CUDART_NAN;   // filled by laser_sim_p95_kernel
    out[2] = __ddiv_rn(dn, __dsub_rn(last_finish, first_arrival));
    out[3] = __ddiv_rn(static_cast<double>(ok), dn);
    out[4] = __ddiv_rn(chunk_sum, dn);
}

constexpr int kP95Threads = 1024;

// One block per replication.  n_pow2 = smallest power of two >= n_req (<= 8192): latencies in shared
// memory, padded with +inf, bitonic sort ascending, nearest rank ceil(0.95 n).
__global__ void __launch_bounds__(kP95Threads)
laser_sim_p95_kernel(const double* __restrict__ arrival, const double* __restrict__ finish,
                     double* __restrict__ out_summary, int n_rep, int n_req, int n_pow2) {
    extern __shared__ double lat[];
    const int r = blockIdx.x;
    for (int i = threadIdx.x; i < n_pow2; i += kP95Threads) {
        const size_t o = static_cast<size_t>(i) * n_rep + r;
        lat[i] = (i < n_req) ? __dsub_rn(finish[o], arrival[o]) : CUDART_INF;
    }
    __syncthreads();
    for (int size = 2; size <= n_pow2; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = threadIdx.x; i < n_pow2; i += kP95Threads) {
                const int j = i ^ stride;
                if (j > i) {
                    const bool up = (i & size) == 0;
                    const double x = lat[i], y = lat[j];
                    if ((x > y) == up) { lat[i] = y; lat[j] = x; }
                }
            }
            __syncthreads();
        }
    }
    if (threadIdx.x == 0) {
        int rank = static_cast<int>(ceil(__dmul_rn(0.95, static_cast<double>(n_req))));
        if (rank < 1) rank = 1;
        out_summary[static_cast<size_t>(r) * LASER_SIM_SUMMARY_COLS + 1] = lat[rank - 1];
    }
}

// n_req > LASER_SIM_MAX_P95_REQUESTS: the same nearest-rank element by an 8-pass most-significant-byte
// radix select over the latencies recomputed from global memory (a double's bits, sign-flipped, order
// like the value).  One block per replication; each pass histograms the byte of the keys that match
// the prefix found so far.
__device__ __forceinline__ unsigned long long order_key(double x) {
    const unsigned long long b = static_cast<unsigned long long>(__double_as_longlong(x));
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__global__ void __launch_bounds__(kP95Threads)
laser_sim_p95_select_kernel(const double* __restrict__ arrival, const double* __restrict__ finish,
                            double* __restrict__ out_summary, int n_rep, int n_req) {
    __shared__ unsigned int hist[256];
    __shared__ unsigned long long s_prefix;
    __shared__ unsigned int s_rank;
    const int r = blockIdx.x;
    if (threadIdx.x == 0) {
        int rank = static_cast<int>(ceil(__dmul_rn(0.95, static_cast<double>(n_req))));
        s_rank = static_cast<unsigned int>(rank < 1 ? 1 : rank);     // 1-based rank still to find
        s_prefix = 0ull;
    }
    for (int pass = 0; pass < 8; ++pass) {
        const int shift = 56 - 8 * pass;
        for (int i = threadIdx.x; i < 256; i += kP95Threads) hist[i] = 0u;
        __syncthreads();
        const unsigned long long prefix = s_prefix;
        const unsigned long long mask = pass == 0 ? 0ull : (~0ull << (shift + 8));
        for (int i = threadIdx.x; i < n_req; i += kP95Threads) {
            const size_t o = static_cast<size_t>(i) * n_rep + r;
            const unsigned long long k = order_key(__dsub_rn(finish[o], arrival[o]));
            if ((k & mask) == prefix) atomicAdd(&hist[(k >> shift) & 0xFFull], 1u);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int left = s_rank, b = 0;
            for (; b < 255u && hist[b] < left; ++b) left -= hist[b];
            s_rank = left;
            s_prefix = prefix | (static_cast<unsigned long long>(b) << shift);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const unsigned long long k = s_prefix;
        const unsigned long long b = (k >> 63) ? (k & 0x7FFFFFFFFFFFFFFFull) : ~k;
        out_summary[static_cast<size_t>(r) * LASER_SIM_SUMMARY_COLS + 1] = __longlong_as_double(static_cast<long long>(b));
    }
}

bool policy_valid(const laser_sim_policy& p) {
    return std::isfinite(p.lambda_base) && std::isfinite(p.beta) && std::isfinite(p.gamma) &&
           std::isfinite(p.l_target) && p.l_target > 0.0 && p.lambda_min <= p.lambda_max &&
           p.alpha >= 0.0 && p.alpha <= 1.0 && p.p_max > p.p_min && p.f_max >= p.f_min &&
           p.budget_l_target > 0.0 && std::isfinite(p.b_base) && std::isfinite(p.b_min) && p.fixed_budget >= 0;
}

}  // namespace

extern "C" {

int laser_sim_policy_default(laser_sim_policy* out) {
    if (!out) return LASER_E_NULL;
    *out = laser_sim_policy{0.95, 0.04, 1.0, 10.0, 0.88, 0.97,
                            0.3,                                         // alpha
                            10.0, 2.0, 0.6, 1.5, 50.0, 275.0, 10.0,
                            1, 1, 10, 0};
    return LASER_OK;
}

int laser_sim_run(const double* arrival, const int32_t* sample_id, const int32_t* policy_id,
                  const laser_sim_policy* policies, int32_t n_pol, const float* chunk_time,
                  const float* conf, const int32_t* prompt_tokens, const float* t_prefill,
                  const float* t_conclusion, const laser_sim_dims* dims, double deadline,
                  double* out_finish, int32_t* out_chunks, uint8_t* out_exited_opt,
                  int32_t* out_budget_opt, double* out_summary, void* stream_v) {
    if (!dims || !policies) return LASER_E_NULL;
    if (dims->n_rep < 0 || dims->n_req < 0 || dims->S <= 0 || dims->K <= 0) return LASER_E_DIMS;
    if (n_pol < 1 || n_pol > LASER_SIM_MAX_POLICIES) return LASER_E_DIMS;
    for (int i = 0; i < n_pol; ++i)
        if (!policy_valid(policies[i])) return LASER_E_PARAMS;
    if (!(deadline == deadline)) return LASER_E_PARAMS;
    if (dims->n_rep == 0 || dims->n_req == 0) return LASER_OK;
    if (!arrival || !sample_id || !policy_id || !chunk_time || !conf || !prompt_tokens || !t_prefill ||
        !t_conclusion || !out_finish || !out_chunks || !out_summary)
        return LASER_E_NULL;
    int dev = -1, major = 0, minor = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return LASER_E_CUDA;
    }
    if (major != 10 || minor != 0) return LASER_E_ARCH;   // sm_100a binary only, no fallback

    SimParams q{};
    q.arrival = arrival; q.sample_id = sample_id; q.policy_id = policy_id;
    q.chunk_time = chunk_time; q.conf = conf; q.prompt_tokens = prompt_tokens;
    q.t_prefill = t_prefill; q.t_conclusion = t_conclusion;
    q.out_finish = out_finish; q.out_chunks = out_chunks; q.out_exited = out_exited_opt;
    q.out_budget = out_budget_opt; q.out_summary = out_summary;
    q.deadline = deadline;
    q.n_rep = dims->n_rep; q.n_req = dims->n_req; q.S = dims->S; q.K = dims->K; q.n_pol = n_pol;
    for (int i = 0; i < n_pol; ++i) q.pol[i] = policies[i];

    cudaStream_t stream = static_cast<cudaStream_t>(stream_v);
    // as few replications per warp as keeps the warp count within 16 warps per SM (measured: 8 and 32 are
    // slower at 3840 and 30720 replications)
    int sms = 148;
    (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int lanes = 1;
    while (lanes < kSimThreads && (dims->n_rep + lanes - 1) / lanes > 16 * sms) lanes <<= 1;
    q.lanes = lanes;
    const int blocks = (dims->n_rep + lanes - 1) / lanes;
    laser_sim_queue_kernel<<<blocks, kSimThreads, 0, stream>>>(q);
    if (cudaGetLastError() != cudaSuccess) return LASER_E_CUDA;
    if (dims->n_req > LASER_SIM_MAX_P95_REQUESTS) {
        // too many latencies for shared memory: radix select over global memory, one block per queue
        laser_sim_p95_select_kernel<<<dims->n_rep, kP95Threads, 0, stream>>>(arrival, out_finish, out_summary,
                                                                         dims->n_rep, dims->n_req);
        if (cudaGetLastError() != cudaSuccess) return LASER_E_CUDA;
    } else {
        int n_pow2 = 1;
        while (n_pow2 < dims->n_req) n_pow2 <<= 1;
        const size_t smem = static_cast<size_t>(n_pow2) * sizeof(double);
        static bool attr_set_dev[64] = {};    // the attribute is per device
        bool& attr_set = attr_set_dev[dev & 63];
        if (!attr_set) {
            if (cudaFuncSetAttribute(laser_sim_p95_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     LASER_SIM_MAX_P95_REQUESTS * static_cast<int>(sizeof(double))) != cudaSuccess) {
                (void)cudaGetLastError();
                return LASER_E_CUDA;
            }
            attr_set = true;
        }
        laser_sim_p95_kernel<<<dims->n_rep, kP95Threads, smem, stream>>>(arrival, out_finish, out_summary,
                                                                        dims->n_rep, dims->n_req, n_pow2);
        if (cudaGetLastError() != cudaSuccess) return LASER_E_CUDA;
    }
    return LASER_OK;
}

}  // extern "C"
