"""Shared helpers for the GPU parity tests: run the CUDA path through the C ABI, run the fp64 oracle
on the same seeded inputs, compare under BASELINE.json's acceptance rule.

Acceptance (BASELINE.json north_star):
  * argmax identical, except rows whose oracle top-2 logit gap is < 1e-3 (exempt, counted);
  * |conf_gpu - conf_oracle| <= 2e-3;
  * exit identical, except requests with |conf_oracle - tau_oracle| <= 2e-3 (exempt, counted).
We additionally hold the GPU to far tighter internal bounds (DESIGN.md §5 derives them from the
arithmetic: bf16 x bf16 products exact in fp32, fp32 accumulation over d <= 4096 terms, ex2.approx
2 ulp, fp32 sums): per-row |pmax| error <= 2e-4, tau error <= 2e-6.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

CONF_TOL = 2e-3
GAP_EXEMPT = 1e-3
MARGIN_EXEMPT = 2e-3
PMAX_TOL = 2e-4
TAU_TOL = 2e-6


# How run_gpu() calls the library (laser_probe_options fields + which entry point).  Test-side state:
# the fixtures of the GPU tests switch it to run the same case through every variant.
CFG = dict(mode=0, tail=0, overlap=False, use_handle=True, w_layout=0)


@dataclass
class GpuRun:
    conf: np.ndarray
    argmax: np.ndarray
    exit: np.ndarray
    tau: np.ndarray
    pmax: np.ndarray
    plan: dict


def to_device(w, device="cuda"):
    import torch
    from paper_2606_31580_b200 import binding as B
    return dict(
        hidden=B.bf16_tensor_from_bits(w.hidden_bits, device),
        W=B.bf16_tensor_from_bits(w.W_bits, device),
        off=torch.from_numpy(w.req_offsets).to(device),
        load=torch.from_numpy(w.load).to(device),
    )


def run_gpu(w, dev=None, agg=0, tau_params=None) -> GpuRun:
    import torch
    from paper_2606_31580_b200 import binding as B
    dev = dev or to_device(w)
    if CFG["w_layout"] == B.W_KBLOCKED:         # the K-block-major copy of W (laser_probe_pack_w)
        dev = dict(dev, W=B.pack_w(dev["W"]))
    probe = B.Probe(w.N_alloc, w.d, w.V, w.R, **CFG)
    # poison outputs so that unwritten entries are caught
    probe.conf.fill_(-7.0); probe.argmax.fill_(-7); probe.exit.fill_(7)
    probe.tau.fill_(-7.0); probe.pmax.fill_(-7.0)
    tp = B.TauParams(**(tau_params or w.tau_params))
    out = probe(dev["hidden"], dev["W"], dev["off"], dev["load"], tp, agg=agg)
    torch.cuda.synchronize()
    probe.close()
    return GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                  out.tau.cpu().numpy(), out.pmax.cpu().numpy(), probe.plan)


def run_oracle(w, requests=None, tau_params=None):
    """Oracle on all requests, or on a subset (list of request indices): returns (result, rows) where
    rows[i] is the global row index of the oracle's i-th row."""
    import oracle
    tp = oracle.TauParams(**(tau_params or w.tau_params))
    if requests is None:
        res = oracle.probe(w.hidden_f32(), w.W_f32(), w.req_offsets, w.load, tp)
        return res, np.arange(w.N_alloc), np.arange(w.R)
    requests = np.asarray(requests)
    rows, off = [], [0]
    for r in requests:
        b, e = int(w.req_offsets[r]), int(w.req_offsets[r + 1])
        rows.extend(range(b, e))
        off.append(len(rows))
    rows = np.asarray(rows, np.int64)
    hid = w.hidden_f32()[rows] if len(rows) else np.zeros((0, w.d), np.float32)
    res = oracle.probe(hid, w.W_f32(), np.asarray(off, np.int32), w.load[requests], tp)
    return res, rows, requests


def compare(w, g: GpuRun, ora, rows, reqs, label=""):
    """Element-by-element comparison under the acceptance rule.  Returns a dict of counters."""
    valid = ~np.isnan(ora.pmax)                     # oracle marks padding rows NaN / -1
    gr = rows[valid]
    # ---- argmax
    am_g, am_o = g.argmax[gr], ora.argmax[valid]
    gap = ora.gap2[valid]
    mism = am_g != am_o
    exempt_rows = gap < GAP_EXEMPT
    bad = mism & ~exempt_rows
    assert not bad.any(), (f"{label}: argmax mismatch on rows {gr[bad][:8]}: gpu {am_g[bad][:8]} "
                           f"oracle {am_o[bad][:8]} gap {gap[bad][:8]}")
    # ---- pmax (internal, tighter than the acceptance rule)
    dp = np.abs(g.pmax[gr].astype(np.float64) - ora.pmax[valid])
    assert np.all(dp <= PMAX_TOL), f"{label}: pmax error {dp.max():.3e} at row {gr[dp.argmax()]}"
    # ---- padding rows
    pad = rows[~valid]
    assert np.all(g.argmax[pad] == -1), f"{label}: padding rows must have argmax -1"
    # ---- conf / tau / exit
    dc = np.abs(g.conf[reqs].astype(np.float64) - ora.conf)
    nan_both = np.isnan(g.conf[reqs]) & np.isnan(ora.conf)
    assert np.all((dc <= CONF_TOL) | nan_both), f"{label}: conf error {np.nanmax(dc):.3e}"
    dt = np.abs(g.tau[reqs].astype(np.float64) - ora.tau)
    assert np.all(dt <= TAU_TOL), f"{label}: tau error {dt.max():.3e}"
    ex_m = g.exit[reqs] != ora.exit
    exempt_req = ora.margin <= MARGIN_EXEMPT
    assert not (ex_m & ~exempt_req).any(), (f"{label}: exit mismatch on requests "
                                            f"{np.asarray(reqs)[ex_m & ~exempt_req][:8]}")
    assert set(np.unique(g.exit[reqs])) <= {0, 1}
    return dict(rows=int(valid.sum()), requests=int(len(reqs)),
                argmax_mismatch_exempt=int((mism & exempt_rows).sum()),
                rows_exempt=int(exempt_rows.sum()),
                exit_mismatch_exempt=int((ex_m & exempt_req).sum()),
                requests_exempt=int(exempt_req.sum()),
                max_pmax_err=float(dp.max()) if dp.size else 0.0,
                max_conf_err=float(np.nanmax(dc)) if dc.size and not np.all(np.isnan(dc)) else 0.0,
                exits=int(ora.exit.sum()))


def check(w, requests=None, label=None, agg=0, tau_params=None):
    g = run_gpu(w, agg=agg, tau_params=tau_params)
    ora, rows, reqs = run_oracle(w, requests, tau_params=tau_params)
    if agg != 0:
        import oracle
        ora.conf = oracle.aggregate(ora.pmax, _local_offsets(w, requests), mode=agg)
        ora.exit, ora.margin = oracle.exit_mask(ora.conf, ora.tau)
    stats = compare(w, g, ora, rows, reqs, label or w.name)
    stats["plan"] = g.plan
    return stats


def _local_offsets(w, requests):
    if requests is None:
        return w.req_offsets
    off = [0]
    for r in requests:
        off.append(off[-1] + int(w.req_offsets[r + 1] - w.req_offsets[r]))
    return np.asarray(off, np.int32)
