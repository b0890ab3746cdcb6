"""Seeded synthetic inputs for the LASER confidence probe (the recipe of DESIGN.md §4).

This module is the ONE place inputs come from: the same numpy arrays are handed to the fp64 oracle
(tests, bench cpu_baseline) and to the CUDA library.  It contains none of the method's arithmetic —
no softmax, no confidence, no threshold — only random draws, an RMS normalisation of the noise, the
planted-token shift and bf16 rounding.  It imports neither `oracle` nor the CUDA binding.

The paper measures on GSM8K / MATH-500 / AMC 2023 / GPQA with 4B-7B reasoning models
(PAPER.md:183-185); none of that exists here and none of it is reproduced.  These inputs stand in for
it: LM-head shapes of the 1.5B-8B distilled reasoning family (BASELINE.json configs) and the paper's
one distributional fact, polarised confidence with 2-6 % of scores in the intermediate range
(PAPER.md:26).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 31580 * 100  # seed = SEED_BASE + config index (+ N for the C5 sweep points)
W_SEED_OFFSET = 1_000_000  # W is drawn from its own stream: seed + W_SEED_OFFSET

# Paper defaults in the NORMALISED load unit u = Lbar / (2 * L_target), i.e.
# l_target = 0.5 (DESIGN A4): BASELINE.json draws load in [0, 1].
TAU_DEFAULTS_NORMALISED = dict(lambda_base=0.95, beta=0.04, gamma=1.0, l_target=0.5,
                               lambda_min=0.88, lambda_max=0.97)


# ------------------------------------------------------------------------------------ bf16 helpers
def bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even (as torch .to(bfloat16))."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) >> np.uint32(16)).astype(np.uint16)


def bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> the exactly equal float32."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


# ------------------------------------------------------------------------------------ container
@dataclass
class Workload:
    name: str
    W_bits: np.ndarray          # uint16 [V, d]   bf16 bit patterns
    hidden_bits: np.ndarray     # uint16 [N_alloc, d]
    req_offsets: np.ndarray     # int32 [R+1]
    load: np.ndarray            # float32 [R]  (already smoothed Lbar, unit of l_target)
    tau_params: dict = field(default_factory=lambda: dict(TAU_DEFAULTS_NORMALISED))
    planted: np.ndarray | None = None   # int64 [N_alloc] planted token per row, -1 = none
    target_pmax: np.ndarray | None = None  # float64 [N_alloc] (S1 only) predicted pmax
    meta: dict = field(default_factory=dict)

    @property
    def V(self): return int(self.W_bits.shape[0])
    @property
    def d(self): return int(self.W_bits.shape[1])
    @property
    def N_alloc(self): return int(self.hidden_bits.shape[0])
    @property
    def R(self): return int(self.req_offsets.shape[0] - 1)
    @property
    def N_valid(self): return int(self.req_offsets[-1]) if self.R > 0 else 0

    def W_f32(self): return bits_to_f32(self.W_bits)
    def hidden_f32(self): return bits_to_f32(self.hidden_bits)

    def algorithmic_bytes(self) -> int:
        """W once + hidden + argmax out + (load in, conf + exit out)."""
        return 2 * self.V * self.d + 2 * self.N_valid * self.d + 4 * self.N_alloc + 9 * self.R + 4 * (self.R + 1)

    def flops(self) -> int:
        """Algorithmic flops: the valid rows only (padding rows need no projection)."""
        return 2 * self.N_valid * self.V * self.d


# ------------------------------------------------------------------------------------ pieces
def make_W(V: int, d: int, sigma: float, seed: int, chunk_rows: int = 16384) -> np.ndarray:
    """bf16 N(0, sigma^2) [V, d] as bit patterns; generated in row chunks to bound peak memory."""
    rng = np.random.default_rng(seed)
    out = np.empty((V, d), np.uint16)
    for r0 in range(0, V, chunk_rows):
        r1 = min(V, r0 + chunk_rows)
        blk = rng.standard_normal((r1 - r0, d), dtype=np.float32)
        blk *= np.float32(sigma)
        out[r0:r1] = bf16_bits(blk)
    return out


def kappa(V: int, d: int, sigma: float, c_lo: float, G0: float) -> float:
    """Shift scale of the calibrated generator: the smallest shift c_lo*kappa*W[t] puts
    the planted logit G0 nats above the log-sum-exp of the background, ln V + d sigma^2 / 2."""
    return (math.log(V) + d * sigma * sigma / 2.0 + G0) / (c_lo * d * sigma * sigma)


def _rms_normalise(z: np.ndarray) -> np.ndarray:
    return z / np.sqrt(np.mean(z.astype(np.float64) ** 2, axis=1, keepdims=True)).astype(np.float32)


def polarised_hidden(W_bits, N, rng, *, q, c_lo, c_hi, kap, normalise=True, shifted_mask=None):
    """hidden[n] = bf16( RMSnorm(z_n) + s_n * c_n * kappa * W[t_n] ),  z ~ N(0, I),
    t ~ U{0..V-1}, s ~ Bernoulli(q) (or the given mask), c ~ U(c_lo, c_hi)."""
    V, d = W_bits.shape
    z = rng.standard_normal((N, d), dtype=np.float32)
    if normalise:
        z = _rms_normalise(z)
    t = rng.integers(0, V, size=N)
    s = (rng.random(N) < q) if shifted_mask is None else np.asarray(shifted_mask, bool)
    c = rng.uniform(c_lo, c_hi, size=N).astype(np.float32)
    coef = (s * c * np.float32(kap)).astype(np.float32)
    h = z + coef[:, None] * bits_to_f32(W_bits[t])
    planted = np.where(s, t, -1).astype(np.int64)
    return bf16_bits(h), planted


def markov_load(R, rng, light=0.2, heavy=0.9, p_stay=0.8):
    """Bursty two-state Markov chain over request index, starts light (C3)."""
    out = np.empty(R, np.float32)
    state = 0
    for r in range(R):
        out[r] = light if state == 0 else heavy
        if rng.random() >= p_stay:
            state ^= 1
    return out


def fixed_offsets(R, length):
    return (np.arange(R + 1, dtype=np.int64) * length).astype(np.int32)


# ------------------------------------------------------------------------------------ configs
def config_c1(seed: int = SEED_BASE + 1) -> Workload:
    """BASELINE.json configs[0]: d=64, V=1000, 8 requests x 4 tokens; W fp32 N(0, 0.05^2) (rounded to
    bf16 once and given to both sides, DESIGN A13); hidden N(0,1) un-normalised; even-indexed
    requests shifted by 6*kappa*W[t] (whole requests, DESIGN A16); load U[0,1]."""
    V, d, R, L = 1000, 64, 8, 4
    rng = np.random.default_rng(seed)
    W_bits = bf16_bits(rng.standard_normal((V, d), dtype=np.float32) * np.float32(0.05))
    kap = kappa(V, d, 0.05, 6.0, 6.0)
    mask = np.repeat(np.arange(R) % 2 == 0, L)
    hb, planted = polarised_hidden(W_bits, R * L, rng, q=1.0, c_lo=6.0, c_hi=6.0, kap=kap,
                                   normalise=False, shifted_mask=mask)
    load = rng.random(R).astype(np.float32)
    return Workload("C1-tiny", W_bits, hb, fixed_offsets(R, L), load, planted=planted,
                    meta=dict(kappa=kap, seed=seed))


def _qwen_like(name, V, d, sigma, R, L, q, seed, load_kind, W_bits=None, W_seed=None, N_alloc=None,
               var_len=None):
    rng = np.random.default_rng(seed)
    if W_bits is None:
        W_bits = make_W(V, d, sigma, seed + W_SEED_OFFSET if W_seed is None else W_seed)
    kap = kappa(V, d, sigma, 4.0, 2.0)
    if var_len is None:
        off = fixed_offsets(R, L)
    else:
        lens = rng.integers(var_len[0], var_len[1] + 1, size=R)
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    N_valid = int(off[-1])
    N_alloc = N_valid if N_alloc is None else N_alloc
    assert N_valid <= N_alloc
    hb = np.zeros((N_alloc, d), np.uint16)
    planted = np.full(N_alloc, -1, np.int64)
    hb[:N_valid], planted[:N_valid] = polarised_hidden(W_bits, N_valid, rng, q=q, c_lo=4.0,
                                                       c_hi=10.0, kap=kap)
    if load_kind == "ramp":
        load = (np.arange(R, dtype=np.float64) / max(R - 1, 1)).astype(np.float32)
    elif load_kind == "markov":
        load = markov_load(R, rng)
    else:
        load = rng.random(R).astype(np.float32)
    return Workload(name, W_bits, hb, off, load, planted=planted,
                    meta=dict(kappa=kap, seed=seed, sigma=sigma, q=q))


def config_c2(W_bits=None, seed: int = SEED_BASE + 2) -> Workload:
    """configs[1] Qwen-1.5B-shaped: d=1536, V=151936, W bf16 N(0,0.02^2), 16 x 8 tokens (N=128),
    95 % of rows shifted, c ~ U(4,10); load ramps 0 -> 1 across requests.  THE graded config."""
    return _qwen_like("C2-qwen1.5b", 151936, 1536, 0.02, 16, 8, 0.95, seed, "ramp", W_bits)


def config_c3(W_bits=None, seed: int = SEED_BASE + 3) -> Workload:
    """configs[2] Qwen-7B-shaped: d=3584, V=152064, sigma 0.015, 32 x 8 (N=256); Markov load."""
    return _qwen_like("C3-qwen7b", 152064, 3584, 0.015, 32, 8, 0.95, seed, "markov", W_bits)


def config_c4(W_bits=None, seed: int = SEED_BASE + 4) -> Workload:
    """configs[3] Llama-8B-shaped: d=4096, V=128256, sigma 0.015, 64 requests, len ~ U{4..16}, CSR
    packed into N_alloc = 1024 rows (trailing rows are zero padding, DESIGN A11); q = 0.94."""
    return _qwen_like("C4-llama8b", 128256, 4096, 0.015, 64, None, 0.94, seed, "uniform", W_bits,
                      N_alloc=1024, var_len=(4, 16))


C5_NS = (8, 64, 512, 4096, 16384)


def config_c5(N: int, W_bits=None) -> Workload:
    """configs[4] heavy-load sweep: C2's shape and W (same matrix, seed of C2), N rows = N/8 requests
    x 8 tokens, load U[0,1]."""
    assert N % 8 == 0
    return _qwen_like(f"C5-sweep-N{N}", 151936, 1536, 0.02, N // 8, 8, 0.95, SEED_BASE + 5 + N,
                      "uniform", W_bits, W_seed=SEED_BASE + 2 + W_SEED_OFFSET)


def scaled(name, V, d, sigma, R, L, seed, q=0.9, N_alloc=None, var_len=None, load_kind="uniform"):
    """Small same-structure workload for parity tests (several tiles + ragged tails)."""
    return _qwen_like(name, V, d, sigma, R, L, q, seed, load_kind, N_alloc=N_alloc, var_len=var_len)


def literal(V, d, sigma, R, L, seed, c=None):
    """BASELINE.json's generator taken literally (shift +c*W[t], no kappa): a flat-distribution case,
    every pmax << 0.5, top-2 gaps tiny — an argmax stress, never an exit."""
    rng = np.random.default_rng(seed)
    W_bits = make_W(V, d, sigma, seed + W_SEED_OFFSET)
    hb, planted = polarised_hidden(W_bits, R * L, rng, q=0.95, c_lo=4.0 if c is None else c,
                                   c_hi=10.0 if c is None else c, kap=1.0)
    return Workload(f"literal-V{V}-d{d}", W_bits, hb, fixed_offsets(R, L),
                    rng.random(R).astype(np.float32), planted=planted, meta=dict(seed=seed))


def tau_band_stress(W_bits, sigma, R=256, L=8, seed: int = SEED_BASE + 6) -> Workload:
    """S1 — tau-band stress set: every request's rows are planted so that the PREDICTED
    per-row pmax is p*_n = clip(c*_r + U(-0.004, 0.004), 0.5, 0.9995), c*_r ~ U(0.86, 0.995); the
    request confidences then straddle the band where tau(load) decides.  The planted coefficient a
    solves  a*|W_t|^2 + z.W_t = ln(V-1) + d sigma^2/2 + logit(p*) + a^2 |W_t|^2 sigma^2 / 2
    (last term: background variance added by the shift itself), 3 fixed-point iterations.
    `target_pmax` is an analytic prediction (law of large numbers over the V-1 background logits),
    not an implementation of the probe."""
    V, d = W_bits.shape
    rng = np.random.default_rng(seed)
    N = R * L
    cstar = rng.uniform(0.86, 0.995, size=R)
    pstar = np.clip(np.repeat(cstar, L) + rng.uniform(-0.004, 0.004, size=N), 0.5, 0.9995)
    t = rng.integers(0, V, size=N)
    z = _rms_normalise(rng.standard_normal((N, d), dtype=np.float32)).astype(np.float64)
    Wt = bits_to_f32(W_bits[t]).astype(np.float64)
    n2 = np.sum(Wt * Wt, axis=1)
    zw = np.sum(z * Wt, axis=1)
    T = math.log(V - 1) + d * sigma * sigma / 2.0 + np.log(pstar / (1.0 - pstar))
    a = (T - zw) / n2
    for _ in range(3):
        a = (T + a * a * n2 * sigma * sigma / 2.0 - zw) / n2
    hb = bf16_bits((z + a[:, None] * Wt).astype(np.float32))
    load = rng.random(R).astype(np.float32)
    return Workload(f"S1-tau-band-V{V}-d{d}", W_bits, hb, fixed_offsets(R, L), load,
                    planted=t.astype(np.int64), target_pmax=pstar, meta=dict(seed=seed, sigma=sigma))


def by_name(name: str, W_cache: dict | None = None) -> Workload:
    """'C1' | 'C2' | 'C3' | 'C4' | 'C5:<N>' | 'shape:d=<d>,V=<V>,N=<N>[,sigma=<s>]' (any LM-head shape:
    N/8 requests of 8 rows, the polarised generator); W_cache lets C2/C5 share the 467 MB matrix."""
    W_cache = {} if W_cache is None else W_cache
    if name == "C1":
        return config_c1()
    if name == "C2" or name.startswith("C5"):
        if "C2" not in W_cache:
            W_cache["C2"] = make_W(151936, 1536, 0.02, SEED_BASE + 2 + W_SEED_OFFSET)
        return config_c2(W_cache["C2"]) if name == "C2" else config_c5(int(name.split(":")[1]), W_cache["C2"])
    if name == "C3":
        return config_c3()
    if name == "C4":
        return config_c4()
    if name.startswith("shape:"):
        kv = dict(t.split("=") for t in name[len("shape:"):].split(","))
        d, V, N = int(kv["d"]), int(kv["V"]), int(kv["N"])
        sigma = float(kv.get("sigma", 0.02))
        key = f"shape-W-{d}-{V}-{sigma}"
        if key not in W_cache:
            W_cache[key] = make_W(V, d, sigma, SEED_BASE + 9 + W_SEED_OFFSET + d + V)
        return _qwen_like(f"shape-d{d}-V{V}-N{N}", V, d, sigma, max(N // 8, 1), 8 if N >= 8 else N, 0.95,
                          SEED_BASE + 9 + N, "uniform", W_bits=W_cache[key])
    raise KeyError(name)


# ------------------------------------------------------------------------------------ serving simulation
# Inputs of the serving simulation (SURVEY §8 f NEXT-4).  The paper feeds its
# discrete-event simulation with per-sample inference times and confidences measured on MATH-500 with
# an RTX 4090; neither the benchmark nor the weights exist here, so a seeded synthetic POOL of samples
# stands in for them: per sample a prompt length, prefill / conclusion times, and per
# reasoning chunk a duration and the confidence at the ATP that ends it.  Inputs only - none of the
# method's arithmetic (no threshold, budget, EMA or queue) lives here.
def sim_pool(S: int = 500, K: int = 15, seed: int = SEED_BASE + 40) -> dict:
    """S samples x K chunks.  Confidence trajectories are polarised: low until the
    sample's solve chunk, high afterwards, with some ATPs in the band where the threshold decides."""
    rng = np.random.default_rng(seed)
    prompt = rng.integers(30, 321, size=S).astype(np.int32)
    hard = (prompt.astype(np.float64) - 30.0) / 290.0                       # longer prompt = harder
    solve = 1 + rng.geometric(0.35 - 0.2 * hard, size=S)                    # chunk index (1-based) that solves
    k = np.arange(1, K + 1)[None, :]
    low = rng.uniform(0.30, 0.90, size=(S, K))
    high = rng.uniform(0.955, 0.9995, size=(S, K))
    band = rng.uniform(0.90, 0.972, size=(S, K))
    conf = np.where(k >= solve[:, None], high, low)
    in_band = rng.random((S, K)) < 0.18
    near = (k >= solve[:, None] - 1) & (k <= solve[:, None] + 1)
    conf = np.where(in_band & near, band, conf)
    return dict(
        chunk_time=rng.uniform(0.15, 0.55, size=(S, K)).astype(np.float32),
        conf=conf.astype(np.float32),
        prompt_tokens=prompt,
        t_prefill=(0.03 + 0.0002 * prompt + rng.uniform(0, 0.02, S)).astype(np.float32),
        t_conclusion=rng.uniform(0.3, 0.8, size=S).astype(np.float32),
    )


def sim_arrivals_poisson(n_rep: int, n_req: int, qps: float, seed: int):
    """Poisson arrivals at rate qps: float64 [n_req, n_rep] (replication fastest), ascending per column."""
    rng = np.random.default_rng(seed)
    gaps = rng.exponential(1.0 / qps, size=(n_req, n_rep))
    return np.cumsum(gaps, axis=0)


def sim_arrivals_burst(n_rep: int, seed: int, phases=((600.0, 1.0), (600.0, 5.0), (600.0, 1.0))):
    """The paper's three-phase burst (10 min at 1 QPS, 10 at 5, 10 at 1): a Poisson
    process conditioned on each phase holding its expected number of arrivals (uniform order
    statistics inside the phase), so that every replication has the same request count."""
    rng = np.random.default_rng(seed)
    cols, t0 = [], 0.0
    for dur, rate in phases:
        m = int(round(dur * rate))
        cols.append(t0 + np.sort(rng.uniform(0.0, dur, size=(m, n_rep)), axis=0))
        t0 += dur
    return np.concatenate(cols, axis=0)


def sim_sample_ids(n_rep: int, n_req: int, S: int, seed: int):
    """Which pool sample each request is: int32 [n_req, n_rep]."""
    return np.random.default_rng(seed).integers(0, S, size=(n_req, n_rep)).astype(np.int32)
