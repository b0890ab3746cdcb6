"""ctypes marshalling for oracle/laser_oracle.c.  TEST INFRASTRUCTURE — see oracle/__init__.py.

No arithmetic of the method happens in this file: every number is produced by the C translation
unit.  numpy is used for buffers only.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "laser_oracle.c"
_SRCS = [_SRC, _HERE / "laser_sim_oracle.c"]
_SO = _HERE / "liblaser_oracle.so"
_lib = None


class _TauParamsC(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("lambda_base", "beta", "gamma", "l_target", "lambda_min", "lambda_max")]


class _SimPolicyC(C.Structure):
    _fields_ = ([(n, C.c_double) for n in
                 ("lambda_base", "beta", "gamma", "l_target", "lambda_min", "lambda_max", "alpha",
                  "b_base", "b_min", "f_min", "f_max", "p_min", "p_max", "budget_l_target")] +
                [(n, C.c_int32) for n in ("early_exit", "adaptive_budget", "fixed_budget", "pad_")])


class _BudgetParamsC(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("b_base", "b_min", "f_min", "f_max", "p_min", "p_max", "l_target")]


@dataclass
class TauParams:
    """Paper defaults, PAPER.md:195 (§5.1 implementation details)."""
    lambda_base: float = 0.95
    beta: float = 0.04
    gamma: float = 1.0
    l_target: float = 10.0
    lambda_min: float = 0.88
    lambda_max: float = 0.97

    def _c(self):
        return _TauParamsC(self.lambda_base, self.beta, self.gamma, self.l_target,
                           self.lambda_min, self.lambda_max)


@dataclass
class BudgetParams:
    """Paper defaults, PAPER.md:166 (f_min..p_max) and PAPER.md:195 (B_base, B_min, L_target)."""
    b_base: float = 10.0
    b_min: float = 2.0
    f_min: float = 0.6
    f_max: float = 1.5
    p_min: float = 50.0
    p_max: float = 275.0
    l_target: float = 10.0

    def _c(self):
        return _BudgetParamsC(self.b_base, self.b_min, self.f_min, self.f_max, self.p_min,
                              self.p_max, self.l_target)


@dataclass
class SimPolicy:
    """One serving policy of the simulation.  Defaults = LASER with the paper's parameters
    (PAPER.md:166, 195): adaptive threshold (Eq. 5) + budget pre-allocation (Eq. 6-8)."""
    lambda_base: float = 0.95
    beta: float = 0.04
    gamma: float = 1.0
    l_target: float = 10.0
    lambda_min: float = 0.88
    lambda_max: float = 0.97
    alpha: float = 0.3
    b_base: float = 10.0
    b_min: float = 2.0
    f_min: float = 0.6
    f_max: float = 1.5
    p_min: float = 50.0
    p_max: float = 275.0
    budget_l_target: float = 10.0
    early_exit: int = 1
    adaptive_budget: int = 1
    fixed_budget: int = 10

    def _c(self):
        return _SimPolicyC(self.lambda_base, self.beta, self.gamma, self.l_target, self.lambda_min,
                           self.lambda_max, self.alpha, self.b_base, self.b_min, self.f_min, self.f_max,
                           self.p_min, self.p_max, self.budget_l_target, self.early_exit,
                           self.adaptive_budget, self.fixed_budget, 0)


def build(force: bool = False) -> Path:
    """Compile laser_oracle.c -> liblaser_oracle.so with gcc (-O2, OpenMP, no fast-math)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < max(f.stat().st_mtime for f in _SRCS):
        tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O3", "-fopenmp", "-fno-fast-math", "-ffp-contract=off",
               "-shared", "-fPIC", "-o", str(tmp), *map(str, _SRCS), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def _L():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(str(_SO))
        dp, fp, ip, bp = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int32),
                          C.POINTER(C.c_uint8))
        i64, i32, dbl = C.c_int64, C.c_int, C.c_double
        tp, qp = C.POINTER(_TauParamsC), C.POINTER(_BudgetParamsC)
        lib.laser_oracle_num_threads.restype = i32
        lib.laser_oracle_row_stats.argtypes = [fp, fp, i64, i32, i64, dp, ip, dp, dp, dp, dp]
        lib.laser_oracle_row_stats_range.argtypes = [fp, fp, i32, i64, i64, dp, ip, dp]
        lib.laser_oracle_merge.argtypes = [dbl, C.c_int32, dbl, dbl, C.c_int32, dbl, dp, ip, dp]
        lib.laser_oracle_merge.restype = None
        lib.laser_oracle_token_prob.argtypes = [fp, fp, ip, i64, i32, i64, dp]
        lib.laser_oracle_aggregate.argtypes = [dp, ip, i64, dp]
        lib.laser_oracle_aggregate_mode.argtypes = [dp, ip, i64, i32, dp]
        lib.laser_oracle_tau_scalar.argtypes = [dbl, tp]
        lib.laser_oracle_tau_scalar.restype = dbl
        lib.laser_oracle_tau_unclamped.argtypes = [dbl, tp]
        lib.laser_oracle_tau_unclamped.restype = dbl
        lib.laser_oracle_tau.argtypes = [fp, i64, tp, dp]
        lib.laser_oracle_exit.argtypes = [dp, dp, i64, bp, dp]
        lib.laser_oracle_probe.argtypes = [fp, fp, ip, fp, tp, i64, i32, i64, i64,
                                           dp, ip, bp, dp, dp, dp, dp]
        lib.laser_oracle_ema.argtypes = [dp, i64, dbl, dbl, dp]
        lib.laser_oracle_f_diff.argtypes = [dbl, qp]
        lib.laser_oracle_f_diff.restype = dbl
        lib.laser_oracle_f_load.argtypes = [dbl, qp]
        lib.laser_oracle_f_load.restype = dbl
        lib.laser_oracle_budget.argtypes = [dp, dp, i64, qp, ip]
        lib.laser_sim_oracle_queue.argtypes = [dp, ip, i64, fp, fp, ip, fp, fp, i64, C.c_int32,
                                               C.POINTER(_SimPolicyC), dp, ip, bp, ip, dp]
        lib.laser_sim_oracle_summary.argtypes = [dp, dp, ip, i64, dbl, dp]
        _lib = lib
    return _lib


def _f32(x):
    return np.ascontiguousarray(x, dtype=np.float32)


def _ptr(a, ty):
    return a.ctypes.data_as(C.POINTER(ty)) if a is not None else None


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed (rc={rc})")


def num_threads() -> int:
    return int(_L().laser_oracle_num_threads())


def row_stats(hidden, W, want_logits: bool = False):
    """Steps 1-2 for every row of `hidden` [N,d] against W [V,d] (float32-representable values).

    Returns dict(m, a, S, pmax, gap2[, logits])."""
    hidden, W = _f32(hidden), _f32(W)
    N, d = hidden.shape
    V, d2 = W.shape
    assert d == d2
    m, S, pm, g2 = (np.empty(N, np.float64) for _ in range(4))
    a = np.empty(N, np.int32)
    lg = np.empty((N, V), np.float64) if want_logits else None
    _chk(_L().laser_oracle_row_stats(_ptr(hidden, C.c_float), _ptr(W, C.c_float), N, d, V,
                                     _ptr(m, C.c_double), _ptr(a, C.c_int32), _ptr(S, C.c_double),
                                     _ptr(pm, C.c_double), _ptr(g2, C.c_double),
                                     _ptr(lg, C.c_double)), "row_stats")
    out = dict(m=m, a=a, S=S, pmax=pm, gap2=g2)
    if want_logits:
        out["logits"] = lg
    return out


def token_prob(hidden, W, token_ids):
    """Probability of token_ids[n] under the softmax of row n (DESIGN A2) — laser_oracle_token_prob."""
    hidden, W = _f32(hidden), _f32(W)
    tok = np.ascontiguousarray(token_ids, np.int32).reshape(-1)
    N, d = hidden.shape
    V = W.shape[0]
    assert tok.shape[0] == N and W.shape[1] == d
    out = np.empty(N, np.float64)
    _chk(_L().laser_oracle_token_prob(_ptr(hidden, C.c_float), _ptr(W, C.c_float), _ptr(tok, C.c_int32),
                                      N, d, V, _ptr(out, C.c_double)), "token_prob")
    return out


def row_stats_range(hidden_row, W, v0: int, v1: int):
    hidden_row, W = _f32(hidden_row).reshape(-1), _f32(W)
    m, S, a = C.c_double(), C.c_double(), C.c_int32()
    _chk(_L().laser_oracle_row_stats_range(_ptr(hidden_row, C.c_float), _ptr(W, C.c_float),
                                           W.shape[1], v0, v1, C.byref(m), C.byref(a), C.byref(S)),
         "row_stats_range")
    return m.value, a.value, S.value


def merge(t1, t2):
    """(m,a,S) (+) (m',a',S'), first operand = lower vocab indices."""
    m, S, a = C.c_double(), C.c_double(), C.c_int32()
    _L().laser_oracle_merge(t1[0], t1[1], t1[2], t2[0], t2[1], t2[2], C.byref(m), C.byref(a),
                            C.byref(S))
    return m.value, a.value, S.value


def aggregate(pmax, req_offsets, mode: int = 0):
    pmax = np.ascontiguousarray(pmax, np.float64)
    off = np.ascontiguousarray(req_offsets, np.int32)
    R = off.shape[0] - 1
    conf = np.empty(max(R, 0), np.float64)
    _chk(_L().laser_oracle_aggregate_mode(_ptr(pmax, C.c_double), _ptr(off, C.c_int32), R, mode,
                                          _ptr(conf, C.c_double)), "aggregate")
    return conf


def tau_scalar(load: float, p: TauParams) -> float:
    return float(_L().laser_oracle_tau_scalar(float(load), C.byref(p._c())))


def tau_unclamped(load: float, p: TauParams) -> float:
    return float(_L().laser_oracle_tau_unclamped(float(load), C.byref(p._c())))


def tau(load, p: TauParams):
    load = _f32(load).reshape(-1)
    out = np.empty(load.shape[0], np.float64)
    _chk(_L().laser_oracle_tau(_ptr(load, C.c_float), load.shape[0], C.byref(p._c()),
                               _ptr(out, C.c_double)), "tau")
    return out


def exit_mask(conf, tau_):
    conf = np.ascontiguousarray(conf, np.float64)
    tau_ = np.ascontiguousarray(tau_, np.float64)
    R = conf.shape[0]
    ex = np.empty(R, np.uint8)
    mg = np.empty(R, np.float64)
    _chk(_L().laser_oracle_exit(_ptr(conf, C.c_double), _ptr(tau_, C.c_double), R,
                                _ptr(ex, C.c_uint8), _ptr(mg, C.c_double)), "exit")
    return ex, mg


@dataclass
class ProbeResult:
    conf: np.ndarray
    argmax: np.ndarray
    exit: np.ndarray
    tau: np.ndarray
    pmax: np.ndarray
    gap2: np.ndarray
    margin: np.ndarray
    seconds: float = field(default=0.0)


def probe(hidden, W, req_offsets, load, p: TauParams) -> ProbeResult:
    """Steps 1-5 (the whole hot path) — laser_oracle_probe."""
    import time
    hidden, W = _f32(hidden), _f32(W)
    off = np.ascontiguousarray(req_offsets, np.int32)
    load = _f32(load).reshape(-1)
    N, d = hidden.shape
    V = W.shape[0]
    R = off.shape[0] - 1
    assert load.shape[0] == R
    conf, tau_, mg = (np.empty(R, np.float64) for _ in range(3))
    ex = np.empty(R, np.uint8)
    am = np.empty(N, np.int32)
    pm, g2 = np.empty(N, np.float64), np.empty(N, np.float64)
    t0 = time.perf_counter()
    _chk(_L().laser_oracle_probe(_ptr(hidden, C.c_float), _ptr(W, C.c_float), _ptr(off, C.c_int32),
                                 _ptr(load, C.c_float), C.byref(p._c()), N, d, V, R,
                                 _ptr(conf, C.c_double), _ptr(am, C.c_int32), _ptr(ex, C.c_uint8),
                                 _ptr(tau_, C.c_double), _ptr(pm, C.c_double), _ptr(g2, C.c_double),
                                 _ptr(mg, C.c_double)), "probe")
    return ProbeResult(conf, am, ex, tau_, pm, g2, mg, time.perf_counter() - t0)


def ema(L, alpha: float = 0.3, lbar0: float = 0.0):
    L = np.ascontiguousarray(L, np.float64).reshape(-1)
    out = np.empty_like(L)
    _chk(_L().laser_oracle_ema(_ptr(L, C.c_double), L.shape[0], alpha, lbar0,
                               _ptr(out, C.c_double)), "ema")
    return out


def f_diff(prompt_tokens: float, q: BudgetParams) -> float:
    return float(_L().laser_oracle_f_diff(float(prompt_tokens), C.byref(q._c())))


def f_load(L: float, q: BudgetParams) -> float:
    return float(_L().laser_oracle_f_load(float(L), C.byref(q._c())))


def budget(prompt_tokens, L, q: BudgetParams):
    pt = np.ascontiguousarray(prompt_tokens, np.float64).reshape(-1)
    L = np.ascontiguousarray(L, np.float64).reshape(-1)
    out = np.empty(pt.shape[0], np.int32)
    _chk(_L().laser_oracle_budget(_ptr(pt, C.c_double), _ptr(L, C.c_double), pt.shape[0],
                                  C.byref(q._c()), _ptr(out, C.c_int32)), "budget")
    return out


def sim_queue(arrival, sample_id, pool, policy: SimPolicy):
    """Algorithm 1 over one single-server FIFO queue - laser_sim_oracle_queue.
    pool = dict(chunk_time [S,K] f32, conf [S,K] f32, prompt_tokens [S] i32, t_prefill [S] f32,
    t_conclusion [S] f32).  Returns dict(finish, chunks, exited, budget, margin)."""
    arrival = np.ascontiguousarray(arrival, np.float64).reshape(-1)
    sid = np.ascontiguousarray(sample_id, np.int32).reshape(-1)
    ct, cf = _f32(pool["chunk_time"]), _f32(pool["conf"])
    pt = np.ascontiguousarray(pool["prompt_tokens"], np.int32)
    tp_, tc = _f32(pool["t_prefill"]), _f32(pool["t_conclusion"])
    S, K = ct.shape
    n = arrival.shape[0]
    assert sid.shape[0] == n and cf.shape == (S, K) and pt.shape[0] == S
    fin, mg = np.empty(n, np.float64), np.empty(n, np.float64)
    ch, bd = np.empty(n, np.int32), np.empty(n, np.int32)
    ex = np.empty(n, np.uint8)
    _chk(_L().laser_sim_oracle_queue(_ptr(arrival, C.c_double), _ptr(sid, C.c_int32), n,
                                     _ptr(ct, C.c_float), _ptr(cf, C.c_float), _ptr(pt, C.c_int32),
                                     _ptr(tp_, C.c_float), _ptr(tc, C.c_float), S, K,
                                     C.byref(policy._c()), _ptr(fin, C.c_double), _ptr(ch, C.c_int32),
                                     _ptr(ex, C.c_uint8), _ptr(bd, C.c_int32), _ptr(mg, C.c_double)),
         "sim_queue")
    return dict(finish=fin, chunks=ch, exited=ex, budget=bd, margin=mg)


def sim_summary(arrival, finish, chunks, deadline: float = 30.0):
    """[mean latency, P95 latency (nearest rank), throughput, SLO share, mean chunks]."""
    arrival = np.ascontiguousarray(arrival, np.float64)
    finish = np.ascontiguousarray(finish, np.float64)
    chunks = np.ascontiguousarray(chunks, np.int32)
    out = np.empty(5, np.float64)
    _chk(_L().laser_sim_oracle_summary(_ptr(arrival, C.c_double), _ptr(finish, C.c_double),
                                       _ptr(chunks, C.c_int32), arrival.shape[0], deadline,
                                       _ptr(out, C.c_double)), "sim_summary")
    return out
