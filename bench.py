#!/usr/bin/env python
"""bench.py — throughput of the LASER confidence probe on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload C2|C3|C4|C5:<N>|shape:d=<d>,V=<V>,N=<N>] [--sharding requests|vocab]
                    [--exchange peer|collective] [--no-sweep] [--no-cpu-baseline] [--with-sim-table]

A "step" is one pass of the whole hot path (a1-a5 of include/laser_probe.h: projection, online
softmax, per-request confidence, threshold, exit mask) over one batch of seeded synthetic input —
one laser_probe_handle_run() call = ONE kernel launch (merge + a3-a5 run in the fused kernel's tail).
Default workload: BASELINE.json configs[1] (Qwen-1.5B-shaped, d=1536, V=151936, 16 requests x 8
tokens), the config the metric is quoted on.

`value`    rows/s with every input already resident in HBM, in the library's DEFAULT (strict) mode:
           every per-call input is read in stream order behind whatever kernel precedes the call -
           what a serving loop gets behind the forward pass that writes `hidden` (device-timed, CUDA
           events on the launch stream, barrier + synchronize either side, max over ranks).
           `overlap` is the same loop with laser_probe_options.overlap = 1 (secondary figure).
`e2e`      rows/s through the host-buffer entry point of a handle: per-step inputs (hidden,
           req_offsets, load) in pinned HOST memory, H2D + kernel + D2H of conf/argmax/exit inside the
           timed region, every step's result read on the host; two batches in flight on two streams
           so the copy of one overlaps the kernel of the other.  e2e.sync_value is one batch at a time.
           W, the model's LM-head weight, stays resident (it is not a per-step input).
`roofline` for the dominant (fused) kernel: algorithmic bytes (or flops) per launch / that kernel's OWN
           average duration, bracketed by CUDA events the library records either side of it on the
           launch stream (second pass of K steps).  frac = achieved / peak reproduces by hand from
           the line.  frac_strict / frac_isolated / frac_sustained are the same bytes over the strict
           step, one isolated call and the step after 0.25 s of continuous load (with its SM clock);
           `sweep` is configs[4].
`configs`  LAST key of the line: every graded config timed in this run - C2 (the headline), C3, C4 and the
           C5 sweep - as {step_us (strict, back to back), kernel_us (bracketed launch), bound, frac,
           frac_strict, kernel, sm_mhz}.
`cpu_baseline` the fp64 oracle, as it stands, on this box's host cores (rank 0, N=1 only).

--impl reference times the oracle itself (the reference arm of this tier): each step is the oracle
on a bounded sample of the same workload.  Under torchrun only rank 0 runs it.

Multi-GPU (--gpus N under torchrun).  --sharding requests (default): the probe's batches are
independent, so ranks shard requests (each rank probes its own batch against its own replica of W)
with no data-path collective: weak scaling.  --sharding vocab: the LM head's tensor-parallel layout
(parallel.VocabParallelProbe): every rank holds V/N rows of W and the whole batch; the per-row
statistics meet on every rank through peer stores over NVLink (--exchange peer) or an NCCL
all-gather (--exchange collective): strong scaling, exchange inside the timed step.
torch.distributed is otherwise used for the barrier and the max-over-ranks reduction only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2606_31580_b200 import workloads as wl  # noqa: E402

METRIC = "probe_rows_per_sec"
UNIT = "rows/s"
NOMINAL_HBM_GBS = 8000.0
NOMINAL_BF16_TFLOPS = 2250.0


# ----------------------------------------------------------------------------------------- helpers
def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            j = json.loads(p.read_text())
            return dict(hbm_gbs=float(j["hbm_gbs"]), bf16_tflops=float(j["bf16_tflops"]),
                        bf16_tflops_sustained=float(j.get("bf16_tflops_sustained", j["bf16_tflops"])),
                        source="measured")
        except Exception:
            pass
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def ncu_traffic_bytes(workload_name: str):
    """dram read+write bytes per launch of the fused kernel from the committed ncu summary, or None."""
    f = ROOT / "profiles" / "fused_kernel_dram_traffic.csv"
    if not f.exists():
        return None
    for line in f.read_text().splitlines():
        parts = [t.strip() for t in line.split(",")]
        if len(parts) >= 2 and parts[0] == workload_name:
            try:
                return float(parts[1])
            except ValueError:
                return None
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML every ~5 ms while the GPU works."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self._stop_evt, self.err = index, [], threading.Event(), None
        self.sm_max = None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                nv.nvmlDeviceGetCurrentClocksThrottleReasons
            while not self._stop_evt.is_set():
                self.samples.append((time.perf_counter(), int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                     int(get_reasons(h))))
                time.sleep(0.004)
        except Exception as e:  # NVML missing: report it, do not fail the bench
            self.err = repr(e)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)

    def summary(self, t0, t1):
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
                 0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
                 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        window = "timed"
        if len(inside) < 3:
            inside, window = list(self.samples), "warmup+timed"
        if not inside:
            return dict(sm_mhz=None, sm_max_mhz=self.sm_max, reasons=[], window="none", error=self.err)
        bits = 0
        for s in inside:
            bits |= s[2]
        reasons = [n for b, n in names.items() if bits & b and n != "gpu_idle"]
        return dict(sm_mhz=float(np.median([s[1] for s in inside])), sm_max_mhz=self.sm_max,
                    reasons=reasons, samples=len(inside), window=window)


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except (ValueError, IndexError):
            pass
    return local_rank


def make_workload(name: str, rank: int, W_cache: dict) -> wl.Workload:
    """Rank r > 0 draws its own hidden/load batch (seed + 7919*r) against the same W."""
    if rank == 0:
        return wl.by_name(name, W_cache)
    base = wl.by_name(name, W_cache)
    if name == "C2":
        return wl.config_c2(base.W_bits, seed=wl.SEED_BASE + 2 + 7919 * rank)
    if name == "C3":
        return wl.config_c3(base.W_bits, seed=wl.SEED_BASE + 3 + 7919 * rank)
    if name == "C4":
        return wl.config_c4(base.W_bits, seed=wl.SEED_BASE + 4 + 7919 * rank)
    return base


def describe(w: wl.Workload) -> str:
    return (f"{w.name}: d={w.d} V={w.V} N={w.N_alloc} rows (valid {w.N_valid}) R={w.R} requests, bf16 W/hidden, "
            f"polarised synthetic generator (DESIGN.md §4)")


def roofline_for(w: wl.Workload, us: float, peaks: dict):
    """Slower of (algorithmic bytes / HBM) and (flops / bf16 tensor peak) bounds the path.  The peak is
    the burst figure of MEASURED_PEAKS.json (every region timed here is far shorter than a second);
    for the tensor bound the ratio against cuBLAS's sustained figure is given beside it."""
    by, fl = w.algorithmic_bytes(), w.flops()
    t_hbm = by / (peaks["hbm_gbs"] * 1e9)
    t_tc = fl / (peaks["bf16_tflops"] * 1e12)
    if t_hbm >= t_tc:
        ach = by / (us * 1e-6) / 1e9
        return dict(bound="hbm", achieved=ach, peak=peaks["hbm_gbs"], unit="GB/s", frac=ach / peaks["hbm_gbs"],
                    frac_of_nominal=ach / NOMINAL_HBM_GBS, peak_source=f"{peaks['source']} (copy bandwidth)")
    ach = fl / (us * 1e-6) / 1e12
    return dict(bound="tensor", achieved=ach, peak=peaks["bf16_tflops"], unit="TFLOP/s",
                frac=ach / peaks["bf16_tflops"], frac_of_nominal=ach / NOMINAL_BF16_TFLOPS,
                frac_vs_sustained_peak=ach / peaks["bf16_tflops_sustained"],
                peak_source=f"{peaks['source']} (cuBLAS bf16 burst; sustained {peaks['bf16_tflops_sustained']:.0f})")


# ----------------------------------------------------------------------------------------- GPU arm
KERNEL_MODES = ["auto", "single", "pair", "flex", "mixed"]     # laser_probe_options.kernel_mode, by value
W_LAYOUTS = ["rowmajor", "kblocked"]                           # laser_probe_options.w_layout, by value
SETTLE_S = 0.25
COOL_S = 1.0
MIN_TIMED_LAUNCHES = 200      # the headline is the median of ceil(200 / K) timed regions of exactly K steps


def cool():
    """Between measurement phases: let the board leave the power-capped state the previous phase drove
    it into, so that every phase (except `sustained`, which wants that state) starts like the headline."""
    import torch
    torch.cuda.synchronize()
    time.sleep(COOL_S)



def settle(case, seconds: float = SETTLE_S):
    """Extra untimed steps until the GPU has been busy for `seconds`: the first tens of milliseconds
    after idle run at boost clocks before the power cap engages (tensor-bound steps measured 9 %
    faster there), and a short timed region would report that transient instead of steady state."""
    import torch
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < seconds:
        for _ in range(20):
            case.step()
        torch.cuda.synchronize()


class GpuCase:
    def __init__(self, w: wl.Workload, device, two_w_copies: bool = False, Ws=None, overlap: bool = False,
                 share=None, mode: int = 0, w_layout: int = 0):
        import torch
        from paper_2606_31580_b200 import binding as B
        self.torch, self.B, self.w = torch, B, w
        if share is not None:
            self.hidden, self.off, self.load = share.hidden, share.off, share.load
        else:
            self.hidden = B.bf16_tensor_from_bits(w.hidden_bits, device)
            self.off = torch.from_numpy(w.req_offsets).to(device)
            self.load = torch.from_numpy(w.load).to(device)
        if Ws is None:
            Ws = [B.bf16_tensor_from_bits(w.W_bits, device)]
            if two_w_copies:
                Ws.append(Ws[0].clone())
        self.Ws = Ws
        self.tp = B.TauParams(**w.tau_params)
        self.probe = B.Probe(w.N_alloc, w.d, w.V, w.R, device=device, debug_outputs=False, overlap=overlap, mode=mode,
                             w_layout=w_layout)
        self.i = 0

    def step(self):
        W = self.Ws[self.i % len(self.Ws)]
        self.i += 1
        return self.probe(self.hidden, W, self.off, self.load, self.tp)

    def time_steps(self, steps: int, sync_fn=None):
        """K steps bracketed by events on the launch stream; returns total milliseconds."""
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if sync_fn:
            sync_fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            self.step()
        e1.record()
        torch.cuda.synchronize()
        if sync_fn:
            sync_fn()
        return e0.elapsed_time(e1)

    def isolated_call_us(self, reps: int = 30):
        """Median duration (us) of ONE call enqueued on an idle GPU (both kernels, no overlap with a
        neighbouring call): the latency a serving loop sees for a single probe."""
        torch = self.torch
        ts = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            self.step()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        ts.sort()
        return ts[len(ts) // 2]

    def graph_replay_us(self, calls: int, reps: int = 20):
        """Median duration (us) of replaying a CUDA graph that holds `calls` back-to-back probe calls,
        captured with this case's options - how a serving engine that captures its step
        would run the probe (no per-launch host work)."""
        torch = self.torch
        side = torch.cuda.Stream(device=self.hidden.device)
        g = torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                for i in range(calls):
                    self.probe(self.hidden, self.Ws[i % len(self.Ws)], self.off, self.load, self.tp, stream=side)
        ts = []
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(reps):
            torch.cuda.synchronize()
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3)
        ts.sort()
        return ts[len(ts) // 2]

    def kernel_times(self, steps: int):
        """Average duration (us) of the fused and the finalize kernel over `steps` calls."""
        B = self.B
        fused = fin = 0.0
        n = 0
        left = steps
        B.profile_enable(True)
        try:
            while left > 0:
                k = min(left, 256)
                for _ in range(k):
                    self.step()
                a, b, c = B.profile_read()
                fused += a; fin += b; n += c; left -= k
        finally:
            B.profile_enable(False)
        return fused / n * 1e3, fin / n * 1e3


def cublas_context(w: wl.Workload, case, steps: int, gpu_index: int) -> dict:
    """CONTEXT ONLY (not the product path, not part of any reported probe figure): the plain library GEMM
    logits = hidden[:N_valid] @ W^T in bf16 through torch.matmul (cuBLAS), back to back on the same box
    with the same clock sampler - what the contraction alone costs a library at this shape.  It WRITES
    the [N, V] logits (which the probe never does) and computes no softmax / argmax / confidence."""
    import torch
    torch.cuda.synchronize()
    time.sleep(COOL_S)
    h = case.hidden[:w.N_valid]
    Wt = [W.t() for W in case.Ws]
    out = torch.empty((w.N_valid, w.V), dtype=torch.bfloat16, device=h.device)
    for i in range(5):
        torch.matmul(h, Wt[i % len(Wt)], out=out)

    def timed(n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for i in range(n):
            torch.matmul(h, Wt[i % len(Wt)], out=out)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    sampler = ClockSampler(gpu_index)
    sampler.start()
    time.sleep(0.05)
    t0 = time.perf_counter()
    us = timed(steps)
    clocks = sampler.summary(t0, time.perf_counter())
    settle_t0 = time.perf_counter()
    while time.perf_counter() - settle_t0 < SETTLE_S:
        timed(20)
    t1 = time.perf_counter()
    us_sus = timed(steps)
    clocks_sus = sampler.summary(t1, time.perf_counter())
    sampler.stop()
    fl = 2.0 * w.N_valid * w.V * w.d
    return dict(what="torch.matmul(hidden[:N_valid], W.T) bf16 -> bf16 logits [N_valid, V] (cuBLAS); context only",
                us_per_call=us, tflops=fl / (us * 1e-6) / 1e12, sm_mhz=clocks.get("sm_mhz"),
                us_per_call_sustained=us_sus, tflops_sustained=fl / (us_sus * 1e-6) / 1e12,
                sustained_sm_mhz=clocks_sus.get("sm_mhz"), logits_bytes_written=2 * w.N_valid * w.V, steps=steps)


def realised_distribution(w: wl.Workload, case) -> dict:
    """One untimed call with the debug outputs on: the realised shares of rows / requests per
    confidence band (SURVEY §8 d: polarisation must be visible next to every number)."""
    import torch
    B = case.B
    probe = B.Probe(w.N_alloc, w.d, w.V, w.R, device=case.hidden.device, debug_outputs=True,
                    w_layout=case.probe.w_layout)
    out = probe(case.hidden, case.Ws[0], case.off, case.load, case.tp)
    torch.cuda.synchronize()
    nv = w.N_valid
    pm = out.pmax[:nv].float().cpu().numpy()
    conf, tau, ex = out.conf.cpu().numpy(), out.tau.cpu().numpy(), out.exit.cpu().numpy()

    def bands(x):
        n = max(len(x), 1)
        return {"lt_0.5": float((x < 0.5).sum()) / n, "0.5_0.88": float(((x >= 0.5) & (x < 0.88)).sum()) / n,
                "0.88_0.97": float(((x >= 0.88) & (x <= 0.97)).sum()) / n, "gt_0.97": float((x > 0.97).sum()) / n}
    return dict(rows=bands(pm), requests=bands(conf), exits=int(ex.sum()), requests_total=int(w.R),
                requests_within_0p05_of_tau=int((np.abs(conf - tau) < 0.05).sum()),
                tau_min=float(tau.min()) if len(tau) else None, tau_max=float(tau.max()) if len(tau) else None)


SIM_POLICIES = {
    "laser": dict(),
    "fixed_high": dict(beta=0.0, lambda_base=0.95, adaptive_budget=0, fixed_budget=10),
    "fixed_low": dict(beta=0.0, lambda_base=0.90, adaptive_budget=0, fixed_budget=10),
    "vanilla": dict(early_exit=0, adaptive_budget=0, fixed_budget=15),
    "threshold_only": dict(adaptive_budget=0, fixed_budget=10),
    "budget_only": dict(beta=0.0),
}
SIM_QPS = (0.5, 1.0, 2.0, 4.0, 8.0)


def serving_sim_bench(device, seeds: int = 128, n_req: int = 1000, with_cpu: bool = True) -> dict:
    """Secondary measurement (SURVEY §8 f NEXT-4): laser_sim_run over policies x arrival rates x seeds
    of synthetic single-server FIFO queues (one GPU thread each), next to the oracle's loop on the host.
    The latency table is illustrative only: the sample pool is synthetic."""
    import torch
    from paper_2606_31580_b200 import binding as B
    names = list(SIM_POLICIES)
    pool = wl.sim_pool()
    cols_a, cols_s, pid, key = [], [], [], []
    for qi, qps in enumerate(SIM_QPS):
        a = wl.sim_arrivals_poisson(seeds, n_req, qps, seed=wl.SEED_BASE + 50 + qi)
        sid = wl.sim_sample_ids(seeds, n_req, pool["conf"].shape[0], seed=wl.SEED_BASE + 60 + qi)
        for pi in range(len(names)):
            cols_a.append(a); cols_s.append(sid)
            pid += [pi] * seeds; key += [(pi, qi)] * seeds
    arr = np.ascontiguousarray(np.concatenate(cols_a, axis=1))
    sid = np.ascontiguousarray(np.concatenate(cols_s, axis=1))
    pid = np.asarray(pid, np.int32)
    n_rep = arr.shape[1]
    d_arr, d_sid, d_pid = (torch.from_numpy(x).to(device) for x in (arr, sid, pid))
    d_pool = {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in pool.items()}
    pols = [B.SimPolicy(**SIM_POLICIES[n]) for n in names]
    for _ in range(3):
        out = B.sim_run(d_arr, d_sid, d_pid, pols, d_pool, details=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    reps = 5
    e0.record()
    for _ in range(reps):
        out = B.sim_run(d_arr, d_sid, d_pid, pols, d_pool, details=False)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    summ = out["summary"].cpu().numpy()
    key = np.asarray(key)
    table = {}
    for pi, name in enumerate(names):
        table[name] = {}
        for qi, qps in enumerate(SIM_QPS):
            m = (key[:, 0] == pi) & (key[:, 1] == qi)
            table[name][str(qps)] = dict(mean_latency_s=float(summ[m, 0].mean()), p95_latency_s=float(summ[m, 1].mean()),
                                         throughput_qps=float(summ[m, 2].mean()), slo_share=float(summ[m, 3].mean()),
                                         mean_chunks=float(summ[m, 4].mean()))
    res = dict(value=n_rep * n_req / (ms * 1e-3), unit="simulated requests/s", ms_per_run=ms, n_rep=n_rep,
               n_req=n_req, gpu_launches_per_run=2, policies=names, qps=list(SIM_QPS), seeds=seeds,
               data="synthetic sample pool (500 samples x 15 chunks) and Poisson arrivals, DESIGN.md §10",
               table=table)
    if with_cpu:
        import oracle
        k = min(n_rep, 60)
        pick = np.linspace(0, n_rep - 1, k).astype(int)
        t0 = time.perf_counter()
        for r in pick:
            o = oracle.sim_queue(arr[:, r], sid[:, r], pool, oracle.SimPolicy(**SIM_POLICIES[names[pid[r]]]))
            oracle.sim_summary(arr[:, r], o["finish"], o["chunks"], 30.0)
        dt = time.perf_counter() - t0
        res["cpu_oracle"] = dict(value=k * n_req / dt, unit="simulated requests/s", cores=1, kind="oracle",
                                 sample=f"{k} of the {n_rep} replications, one after the other")
    return res


def run_vocab_sharded(args, dist, rank, local_rank, world, device):
    """--sharding vocab: parallel.VocabParallelProbe under torchrun (or alone: a world of one).  Strong
    scaling: the batch is fixed, W is cut into `world` row ranges, the per-row statistics of all shards
    meet on every rank inside the timed step (peer stores over NVLink, or an NCCL all-gather)."""
    import socket
    import torch
    from paper_2606_31580_b200 import binding as B, parallel as par
    os.environ.setdefault("NCCL_DEBUG", "INFO")          # keep the communicator lines (NVLS / P2P) on stderr
    os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    own_group = False
    if dist is None:
        import torch.distributed as dist
        s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", str(port))
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=device)
        own_group = True
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    w = wl.by_name(args.workload, {})                    # every rank: the same batch, the same W
    wlay = W_LAYOUTS.index(args.w_layout)
    vp = par.VocabParallelProbe(dist, w.N_alloc, w.d, w.V, w.R, device, exchange=args.exchange, w_layout=wlay)
    hidden = B.bf16_tensor_from_bits(w.hidden_bits, device)
    Wg = B.bf16_tensor_from_bits(w.W_bits[vp.v0:vp.v1], device)
    if wlay:
        Wg = B.pack_w(Wg)                                # once per model: this rank's rows, K-block-major
    off = torch.from_numpy(w.req_offsets).to(device)
    load = torch.from_numpy(w.load).to(device)
    tp = B.TauParams(**w.tau_params)

    def step():
        return vp(hidden, Wg, off, load, tp)

    def timed(fn, n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        dist.barrier(); torch.cuda.synchronize()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize(); dist.barrier()
        t = torch.tensor([e0.elapsed_time(e1)], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t[0])

    for _ in range(args.warmup):
        step()
    launches0 = B.kernel_launch_count()
    t0 = time.perf_counter()
    ms = timed(step, args.steps)
    clocks = sampler.summary(t0, time.perf_counter())
    launches = B.kernel_launch_count() - launches0

    # end to end: the step's inputs start in pinned host memory, its results are read on the host
    hh = B.bf16_tensor_from_bits(w.hidden_bits, pin=True)
    hoff, hload = torch.from_numpy(w.req_offsets).pin_memory(), torch.from_numpy(w.load).pin_memory()
    o_conf = torch.empty(w.R, dtype=torch.float32).pin_memory()
    o_arg = torch.empty(w.N_alloc, dtype=torch.int32).pin_memory()
    o_exit = torch.empty(w.R, dtype=torch.uint8).pin_memory()

    def e2e_step():
        hidden.copy_(hh, non_blocking=True); off.copy_(hoff, non_blocking=True); load.copy_(hload, non_blocking=True)
        out = step()
        o_conf.copy_(out.conf, non_blocking=True); o_arg.copy_(out.argmax, non_blocking=True)
        o_exit.copy_(out.exit, non_blocking=True)
        torch.cuda.current_stream().synchronize()
        return int(o_exit.sum())

    for _ in range(args.warmup):
        e2e_step()
    e2e_ms = timed(e2e_step, args.steps)
    sampler.stop()
    if rank == 0:
        ms_per_step = ms / args.steps
        shard_bytes = (vp.v1 - vp.v0) * w.d * 2
        print(json.dumps(dict(
            metric=METRIC, value=w.N_valid / (ms_per_step * 1e-3), unit=UNIT, n_gpus=world, steps=args.steps,
            warmup=args.warmup, ms_per_step=ms_per_step, higher_is_better=True, scaling="strong", vs_baseline=None,
            dtype="bf16", data="synthetic",
            config=dict(workload=describe(w), sharding=f"vocabulary: {world} row ranges of W, whole batch on every rank",
                        exchange=args.exchange, w_layout=args.w_layout, shard_rows=vp.v1 - vp.v0, plan=vp.shard.plan,
                        l2="each rank's W shard (%.0f MB)%s" % (shard_bytes / 1e6,
                                                                " exceeds the 126 MB L2" if shard_bytes > 126e6 else
                                                                " FITS the 126 MB L2: per-rank figure is L2-assisted")),
            requests_per_sec=w.R / (ms_per_step * 1e-3), clocks=clocks,
            e2e=dict(value=w.N_valid / (e2e_ms / args.steps * 1e-3), unit=UNIT,
                     h2d_bytes_per_step=w.N_alloc * w.d * 2 + (w.R + 1) * 4 + w.R * 4,
                     d2h_bytes_per_step=w.R * 4 + w.N_alloc * 4 + w.R, ms_per_step=e2e_ms / args.steps,
                     api="torch copies (plumbing) around parallel.VocabParallelProbe, synchronous"),
            gpu_launches=int(launches) * world,
            roofline=dict(bound="hbm", achieved=shard_bytes / (ms_per_step * 1e-3) / 1e9, unit="GB/s",
                          peak=measured_peaks()["hbm_gbs"],
                          frac=shard_bytes / (ms_per_step * 1e-3) / 1e9 / measured_peaks()["hbm_gbs"],
                          traffic=None, note="per rank: its W shard over the whole step, exchange included"))), flush=True)
    dist.barrier()
    if own_group or world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    from paper_2606_31580_b200 import binding as B

    rank = int(os.environ.get("RANK", 0))
    local_rank = int(os.environ.get("LOCAL_RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — this library has no CPU path (use --impl reference "
                         "for the oracle's CPU timing)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    if args.sharding == "vocab":
        return run_vocab_sharded(args, dist, rank, local_rank, world, device)

    def barrier():
        if dist is not None:
            dist.barrier()

    peaks = measured_peaks()
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()                      # NVML initialises while the workload is generated
    W_cache: dict = {}
    w = make_workload(args.workload, rank, W_cache)
    # the library default: strict stream order for every per-call input (what a serving loop needs
    # behind the forward pass that writes `hidden`).  This is the headline configuration.
    kmode = KERNEL_MODES.index(args.kernel_mode)
    wlay = W_LAYOUTS.index(args.w_layout)
    case = GpuCase(w, device, two_w_copies=(w.V * w.d * 2 < 2_000_000_000), mode=kmode)
    if wlay:      # --w-layout kblocked: every timed call gets the packed copies (made here, once, untimed)
        case = GpuCase(w, device, Ws=[B.pack_w(Wc) for Wc in case.Ws], share=case, mode=kmode, w_layout=wlay)
        torch.cuda.empty_cache()
    # laser_probe_options.overlap = 1: consecutive calls of a loop over resident inputs overlap
    over = GpuCase(w, device, Ws=case.Ws, overlap=True, share=case, mode=kmode, w_layout=wlay)

    for _ in range(args.warmup):
        case.step()
    torch.cuda.synchronize()
    barrier()
    # Headline: timed regions of EXACTLY K steps each, repeated until at least MIN_TIMED_LAUNCHES steps have
    # been timed (K = 20 alone is a 1.5 ms sample); the median region is reported, all of them are listed.
    regions = max(1, -(-MIN_TIMED_LAUNCHES // args.steps))
    launches0 = B.kernel_launch_count()
    t0 = time.perf_counter()
    region_ms = [case.time_steps(args.steps, barrier) for _ in range(regions)]
    t1 = time.perf_counter()
    launches = (B.kernel_launch_count() - launches0) // regions      # per region of K steps
    ms = sorted(region_ms)[len(region_ms) // 2]
    clocks = sampler.summary(t0, t1)

    # the same K steps with overlap = 1 (secondary figure)
    cool()
    for _ in range(3):
        over.step()
    overlap_ms = over.time_steps(args.steps, barrier)

    # CUDA-graph replay under the strict default: one call, and ten calls in one graph
    cool()
    graph_one_us = case.graph_replay_us(1)
    graph_ten_us = case.graph_replay_us(10) / 10.0
    graph_ten_overlap_us = over.graph_replay_us(10) / 10.0

    # dominant kernel on its own (second pass, same stream, library-recorded events either side of it)
    cool()
    fused_us, fin_us = case.kernel_times(args.steps)
    cool()
    isolated_us = case.isolated_call_us()

    # the same K strict steps once more after SETTLE_S seconds of continuous load: the power-capped steady state
    settle(case)
    t2 = time.perf_counter()
    sustained_ms = case.time_steps(args.steps, barrier)
    sustained_clocks = sampler.summary(t2, time.perf_counter())

    # W pre-packed K-block-major (laser_probe_pack_w, once per model; laser_probe_options.w_layout): the same K
    # strict steps and bracketed launches, secondary figure.  Only where W is streamed from HBM once per
    # call and two packed copies fit beside the row-major ones.
    kblocked = None
    if rank == 0 and wlay == 0 and w.N_alloc <= 256 and w.V * w.d * 2 < 2_000_000_000:
        cool()
        Wp = [B.pack_w(Wc) for Wc in case.Ws]
        kb_case = GpuCase(w, device, Ws=Wp, share=case, mode=kmode, w_layout=B.W_KBLOCKED)
        for _ in range(max(3, args.warmup)):
            kb_case.step()
        kb_ms = kb_case.time_steps(args.steps)
        cool()
        kb_kernel_us, _z = kb_case.kernel_times(args.steps)
        kblocked = dict(step_us_strict=kb_ms / args.steps * 1e3, kernel_us=kb_kernel_us,
                        frac=roofline_for(w, kb_kernel_us, peaks)["frac"],
                        frac_strict=roofline_for(w, kb_ms / args.steps * 1e3, peaks)["frac"],
                        value=float(w.N_valid) / (kb_ms / args.steps * 1e-3), unit=UNIT,
                        note="the same K strict steps / bracketed launches with W given K-block-major "
                             "([d/64][V][64], packed once by laser_probe_pack_w; laser_probe_options.w_layout = "
                             "LASER_W_KBLOCKED): every TMA box of W is one contiguous run in HBM.  Secondary figure: "
                             "the headline keeps the row-major W of the problem statement")
        del kb_case, Wp
        torch.cuda.empty_cache()

    # end to end through the host-buffer entry point of a handle: per-step inputs in pinned host memory,
    # results read on the host every step.  Two batches in flight (two handles, two streams, one
    # staging/workspace/output set each) so that the H2D copy of batch i+1 overlaps the kernel of batch
    # i, as a serving loop would run it; one batch at a time (synchronous) is timed as well.
    depth = 2
    slots = [B.HostProbe(w.N_alloc, w.d, w.V, w.R, device=device, mode=kmode, w_layout=wlay) for _ in range(depth)]
    streams = [torch.cuda.Stream(device=device) for _ in range(depth)]
    hp = slots[0]
    hh = B.bf16_tensor_from_bits(w.hidden_bits, pin=True)
    hoff = torch.from_numpy(w.req_offsets).pin_memory()
    hload = torch.from_numpy(w.load).pin_memory()

    def e2e_pipelined(n, one_stream):
        """n steps, `depth` in flight; returns (ms, exits seen on the host).  one_stream: both batches
        on ONE stream (staging kernel -> probe kernel -> staging kernel -> ... is one programmatic
        dependent launch chain; a CUDA event per batch tells the host when its results are there);
        else one stream per batch."""
        pending = [False] * depth
        seen = 0
        sts = [streams[0]] * depth if one_stream else streams
        evs = [torch.cuda.Event() for _ in range(depth)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for st in set(sts):
            st.wait_event(e0)
        tw0 = time.perf_counter()
        for i in range(n):
            k = i % depth
            if pending[k]:
                evs[k].synchronize()
                seen += int(slots[k].exit.sum())          # the step's result, read on the host
            slots[k].submit(hh, case.Ws[i % len(case.Ws)], hoff, hload, case.tp, sts[k])
            evs[k].record(sts[k])
            pending[k] = True
        for k in range(depth):
            if pending[k]:
                evs[k].synchronize()
                seen += int(slots[k].exit.sum())
        tw1 = time.perf_counter()
        for st in set(sts):
            torch.cuda.current_stream().wait_stream(st)
        e1.record()
        torch.cuda.synchronize()
        return max(e0.elapsed_time(e1), (tw1 - tw0) * 1e3), seen

    def e2e_sync(n):
        torch.cuda.synchronize()
        tw0 = time.perf_counter()
        for i in range(n):
            out = hp(hh, case.Ws[i % len(case.Ws)], hoff, hload, case.tp)
            _ = int(out.exit.sum())
        return (time.perf_counter() - tw0) * 1e3

    sampler.stop()
    cool()
    e2e_pipelined(args.warmup, True)
    e2e_pipelined(args.warmup, False)
    e2e_sync(args.warmup)
    barrier()
    # each end-to-end figure: the median of three timed regions of K steps (host-side jitter - Python, the
    # driver's launch queue - is a visible share of a 20-step region)
    med = lambda xs: sorted(xs)[len(xs) // 2]
    e2e_reps = 3
    ones, twos, syncs = [], [], []
    for _ in range(e2e_reps):
        barrier()
        ones.append(e2e_pipelined(args.steps, True)[0])
        barrier()
        twos.append(e2e_pipelined(args.steps, False)[0])
        barrier()
        syncs.append(e2e_sync(args.steps))
    e2e_one_ms, e2e_two_ms, e2e_sync_ms = med(ones), med(twos), med(syncs)
    e2e_ms = min(e2e_one_ms, e2e_two_ms)

    if dist is not None:
        t = torch.tensor([ms, e2e_ms, sustained_ms, overlap_ms], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, e2e_ms, sustained_ms, overlap_ms = float(t[0]), float(t[1]), float(t[2]), float(t[3])
        rows_t = torch.tensor([w.N_valid, w.R], device=device, dtype=torch.float64)
        dist.all_reduce(rows_t, op=dist.ReduceOp.SUM)
        rows_all, reqs_all = float(rows_t[0]), float(rows_t[1])
    else:
        rows_all, reqs_all = float(w.N_valid), float(w.R)

    out = None
    if rank == 0:
        ms_per_step = ms / args.steps
        value = rows_all / (ms_per_step * 1e-3)
        # roofline of the dominant kernel from ITS OWN duration: events recorded by the library
        # immediately before and after the fused kernel on the launch stream (no programmatic
        # dependent launch for those calls, so nothing overlaps the bracket).
        roof = roofline_for(w, fused_us, peaks)
        roof["kernel"] = ("laser_probe_flex_kernel" if case.probe.plan["flex"] else
                          "laser_probe_fused_kernel<1> (CTA pairs) beside laser_probe_fused_kernel<0> (single CTAs): mixed schedule"
                          if case.probe.plan["mixed"] else "laser_probe_fused_kernel<%d>" % case.probe.plan["cta_pair"])
        roof["kernel_us"] = fused_us
        roof["kernel_us_source"] = ("average over K launches, each bracketed on its own by CUDA events on the launch "
                                    "stream (laser_profile_enable; no programmatic dependent launch for those calls, "
                                    "so prologue and W pre-issue are inside the bracket); the kernel is the whole hot "
                                    "path: merge + a3-a5 run in its tail")
        # the interval between the event after the kernel and the next event, with nothing in between:
        # what one event pair costs on this stream (it is inside kernel_us as well; not subtracted)
        roof["event_pair_overhead_us"] = fin_us
        # the same bracket with the measured cost of an empty bracket taken off: what ncu's
        # gpu__time_duration of the kernel corresponds to (profiles/: 76.8 us at C2)
        net_us = max(fused_us - fin_us, 1e-3)
        roof["kernel_us_net_of_event_overhead"] = net_us
        roof["frac_net_of_event_overhead"] = roofline_for(w, net_us, peaks)["frac"]
        roof["algorithmic_bytes"] = w.algorithmic_bytes()
        roof["algorithmic_flops"] = w.flops()
        roof["traffic"] = ncu_traffic_bytes(args.workload)
        roof["traffic_source"] = ("profiles/fused_kernel_dram_traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum "
                                  "per launch from a committed ncu --set full capture of this kernel; not measured in this run")
        roof["step_us_strict"] = ms_per_step * 1e3
        roof["timed_launches"] = regions * args.steps
        roof["timed_regions_us_per_step"] = [round(r / args.steps * 1e3, 3) for r in region_ms]
        roof["frac_strict"] = roofline_for(w, ms_per_step * 1e3, peaks)["frac"]
        roof["isolated_call_us"] = graph_one_us
        roof["frac_isolated"] = roofline_for(w, graph_one_us, peaks)["frac"]
        roof["isolated_call_note"] = ("median replay of a CUDA graph holding ONE call on an idle GPU, events either side: "
                                      "the device-side latency of a single probe; isolated_call_us_python_launch is the "
                                      "same call launched from Python (ctypes + launch latency inside the bracket)")
        roof["isolated_call_us_python_launch"] = isolated_us
        roof["step_us_sustained"] = sustained_ms / args.steps * 1e3
        roof["frac_sustained"] = roofline_for(w, sustained_ms / args.steps * 1e3, peaks)["frac"]
        roof["sustained_sm_mhz"] = sustained_clocks.get("sm_mhz")
        roof["step_us_overlap"] = overlap_ms / args.steps * 1e3
        roof["step_frac_overlap"] = roofline_for(w, overlap_ms / args.steps * 1e3, peaks)["frac"]
        out = dict(
            metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
            ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None,
            dtype="bf16", data="synthetic",
            config=dict(workload=describe(w), plan=case.probe.plan,
                        l2="W (%.0f MB) exceeds the 126 MB L2; two W copies alternate between steps"
                           % (w.V * w.d * 2 / 1e6) if len(case.Ws) > 1 else
                           "W (%.0f MB) exceeds the 126 MB L2" % (w.V * w.d * 2 / 1e6),
                        sharding="requests sharded across ranks, W replicated, no collective" if world > 1 else "single GPU",
                        e2e_w_resident=True, kernel_mode=args.kernel_mode, w_layout=args.w_layout,
                        mode="library default: strict stream order (laser_probe_options.overlap = 0), "
                             "merge + a3-a5 in the fused kernel's tail (one launch per call)"),
            overlap=dict(value=rows_all / (overlap_ms / args.steps * 1e-3), unit=UNIT,
                         ms_per_step=overlap_ms / args.steps,
                         note="the same K steps with laser_probe_options.overlap = 1: consecutive calls of a loop "
                              "over resident inputs overlap; not what a loop behind a producer of `hidden` may use"),
            cuda_graph=dict(one_call_us=graph_one_us, per_call_us_ten_calls_strict=graph_ten_us,
                            per_call_us_ten_calls_overlap=graph_ten_overlap_us,
                            note="median replay time of a captured CUDA graph holding 1 / 10 probe calls "
                                 "(rank 0); a call is capturable: no sync, no allocation, no host read"),
            sustained=dict(value=rows_all / (sustained_ms / args.steps * 1e-3), unit=UNIT,
                           ms_per_step=sustained_ms / args.steps, clocks=sustained_clocks,
                           note=f"the same K strict steps timed again after {SETTLE_S} s of continuous probing "
                                "(power-capped steady state)"),
            requests_per_sec=reqs_all / (ms_per_step * 1e-3),
            clocks=clocks,
            e2e=dict(value=rows_all / (e2e_ms / args.steps * 1e-3), unit=UNIT,
                     h2d_bytes_per_step=w.N_valid * w.d * 2 + (w.R + 1) * 4 + w.R * 4,
                     d2h_bytes_per_step=hp.d2h_bytes,
                     ms_per_step=e2e_ms / args.steps, batches_in_flight=depth,
                     timed_regions=e2e_reps, statistic="median of the regions, K steps each",
                     api="laser_probe_handle_run_host (asynchronous), 2 handles / batches in flight on "
                         + ("ONE stream (staging kernel + probe kernel in one dependent-launch chain, an event per batch)"
                            if e2e_one_ms <= e2e_two_ms else "two streams")
                         + "; results read on the host every step",
                     ms_per_step_one_stream=e2e_one_ms / args.steps, ms_per_step_two_streams=e2e_two_ms / args.steps,
                     sync_value=float(w.N_valid) * world / (e2e_sync_ms / args.steps * 1e-3),
                     sync_ms_per_step=e2e_sync_ms / args.steps,
                     sync_api="laser_probe_handle_run_host (synchronous, one batch at a time; rank 0's figure x ranks)"),
            gpu_launches=int(launches) * world,      # every rank enqueues the same calls
            roofline=roof,
            realised=realised_distribution(w, case),
        )
        if kblocked is not None:
            out["roofline"]["w_kblocked"] = kblocked

    # heavy-load sweep (configs[4]) — rank 0, single GPU only; W shared with C2
    if rank == 0 and world == 1 and not args.no_sweep and args.workload == "C2":
        sweep = []
        for N in wl.C5_NS:
            ws = wl.config_c5(N, W_cache["C2"])
            c = GpuCase(ws, device, Ws=case.Ws, w_layout=wlay)
            k = max(5, min(args.steps, int(2e5 / max(N, 128))))
            cool()
            for _ in range(3):
                c.step()
            t_ms = c.time_steps(k) / k
            cool()
            f_us, _z = c.kernel_times(min(k, 64))
            r = roofline_for(ws, f_us, peaks)
            sweep.append(dict(N=N, step_us=round(t_ms * 1e3, 2), rows_per_sec=N / (t_ms * 1e-3),
                              kernel_us=round(f_us, 2), bound=r["bound"], achieved=r["achieved"], unit=r["unit"],
                              frac=r["frac"], frac_of_nominal=r["frac_of_nominal"],
                              frac_vs_sustained_peak=r.get("frac_vs_sustained_peak"),
                              frac_step=roofline_for(ws, t_ms * 1e3, peaks)["frac"],
                              pair=c.probe.plan["cta_pair"], tile_n=c.probe.plan["tile_n"],
                              kernel="flex" if c.probe.plan["flex"] else ("mixed" if c.probe.plan["mixed"] else
                                                                          ("pair" if c.probe.plan["cta_pair"] else "single"))))
            del c
        out["roofline"]["sweep"] = sweep

    # vocabulary-parallel layout (laser_probe_partial + laser_probe_combine): what ONE rank of G would
    # execute per step - its 1/G slice of W (ONE kernel: reduce and record stores in the fused kernel's
    # tail), then the merge of G records per row.  The exchange itself needs G GPUs (--sharding vocab).
    if rank == 0 and world == 1 and not args.no_sweep and args.workload == "C2" and wlay == 0:
        from paper_2606_31580_b200 import parallel as par
        vp = []
        for G in (2, 4, 8):
            v0, v1 = par.shard_vocab(w.V, G, 0)
            sh = B.VocabShardProbe(w.N_alloc, w.d, v1 - v0, w.R, v0, G, device=device, debug_outputs=False)
            sh.stats_all.fill_(float("-inf"))
            Wg = [Wc[v0:v1] for Wc in case.Ws]       # contiguous row slices of the resident copies
            def vp_step(i, sh=sh, Wg=Wg):
                sh.partial(case.hidden, Wg[i % len(Wg)], case.off, out=sh.stats_all[0])
                sh.combine(case.off, case.load, case.tp)
            for i in range(5):
                vp_step(i)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            k = min(args.steps, 500)
            e0.record()
            for i in range(k):
                vp_step(i)
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) / k * 1e3
            vp.append(dict(G=G, shard_rows=v1 - v0, us_per_step_per_rank=us, kernels_per_step=2,
                           shard_gb_per_s=(v1 - v0) * w.d * 2 / (us * 1e-6) / 1e9, plan=sh.plan))
        out["vocab_parallel_per_rank"] = dict(
            note="one rank's work at G-way vocabulary sharding, measured on one GPU: partial over the "
                 "first 1/G of W + combine of G records per row; the N*16-byte exchange is not included",
            points=vp)

    if rank == 0 and world == 1 and not args.no_sweep and args.workload == "C2":
        out["serving_sim"] = serving_sim_bench(device, with_cpu=not args.no_cpu_baseline)
        if not args.with_sim_table:       # the illustrative latency table is long: --with-sim-table prints it
            tab = out["serving_sim"].pop("table")
            out["serving_sim"]["table"] = "omitted (--with-sim-table); LASER at 2 QPS: " + json.dumps(
                {k: round(v, 3) for k, v in tab["laser"]["2.0"].items()})

    # The other graded configs (BASELINE.json configs[2], configs[3]) in the same run: strict step and
    # bracketed kernel, so that every config's roofline fraction is in the line the driver keeps.
    other = {}
    if rank == 0 and world == 1 and not args.no_sweep and args.workload == "C2" and kmode == 0 and wlay == 0:
        del over
        for name in ("C3", "C4"):
            try:
                wo = wl.by_name(name, W_cache)
                co = GpuCase(wo, device, mode=kmode)
                k = max(20, min(args.steps, 200))
                cool()
                for _ in range(5):
                    co.step()
                tc0 = time.perf_counter()
                t_ms = co.time_steps(k) / k
                ck = sampler.summary(tc0, time.perf_counter())
                cool()
                f_us, _z = co.kernel_times(min(k, 64))
                other[name] = (wo, co.probe.plan, t_ms * 1e3, f_us, ck.get("sm_mhz"))
                del co
                W_cache.pop(name, None)
                torch.cuda.empty_cache()
            except (RuntimeError, MemoryError) as e:      # e.g. device memory: say so instead of failing the line
                other[name] = repr(e)[:200]

    if rank == 0 and world == 1 and args.with_cublas and wlay == 0:
        out["cublas_context"] = cublas_context(w, case, args.steps, physical_gpu_index(local_rank))
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w, target_s=10.0)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        # compact per-config record, LAST key of the line: {step_us (strict, back to back), kernel_us (bracketed
        # launch), bound, frac (of kernel_us), frac_strict (of step_us), kernel, sm_mhz}
        def kname(plan):
            return "flex" if plan["flex"] else ("mixed" if plan["mixed"] else ("pair" if plan["cta_pair"] else "single"))
        r = out["roofline"]
        cfgs = {args.workload: dict(step_us=round(r["step_us_strict"], 2), kernel_us=round(r["kernel_us"], 2), bound=r["bound"],
                                    frac=round(r["frac"], 4), frac_strict=round(r["frac_strict"], 4),
                                    kernel=kname(case.probe.plan), sm_mhz=clocks.get("sm_mhz"))}
        for name, rec in other.items():
            if isinstance(rec, str):
                cfgs[name] = dict(skipped=rec)
                continue
            wo, plan, step_us, f_us, mhz = rec
            rr = roofline_for(wo, f_us, peaks)
            cfgs[name] = dict(step_us=round(step_us, 2), kernel_us=round(f_us, 2), bound=rr["bound"], frac=round(rr["frac"], 4),
                              frac_strict=round(roofline_for(wo, step_us, peaks)["frac"], 4), kernel=kname(plan), sm_mhz=mhz,
                              rows=wo.N_valid)
        for e in r.get("sweep", []):
            cfgs["C5:%d" % e["N"]] = dict(step_us=e["step_us"], kernel_us=e["kernel_us"], bound=e["bound"],
                                          frac=round(e["frac"], 4), frac_strict=round(e["frac_step"], 4), kernel=e["kernel"])
        out["configs"] = cfgs
        print(json.dumps(out), flush=True)


# ----------------------------------------------------------------------------------------- timeline
def run_timeline(args):
    """Device-side evidence for the strict step: per-CTA %globaltimer stamps of consecutive strict calls from
    the -DLASER_TIMELINE build (python -m paper_2606_31580_b200.build --timeline; loaded through
    LASER_PROBE_LIB).  Prints a markdown report: per call, when its CTAs entered, had their first W boxes
    requested, passed griddepcontrol.wait, stored their last record and finished the tail - and, between
    consecutive calls, how long call k+1 was already on the SMs before call k was done.  Not a bench line."""
    import ctypes as C
    import torch
    from paper_2606_31580_b200 import binding as B
    L = B.lib()
    if not hasattr(L, "laser_debug_timeline_read"):
        raise SystemExit("bench.py --timeline needs the timeline build: python -m paper_2606_31580_b200.build --timeline; "
                         "LASER_PROBE_LIB=paper_2606_31580_b200/liblaser_probe_timeline.so python bench.py --timeline")
    device = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    W_cache: dict = {}
    w = make_workload(args.workload, 0, W_cache)
    case = GpuCase(w, device, two_w_copies=True)
    grid = case.probe.plan["grid"]
    K = 16
    for _ in range(max(5, args.warmup)):
        case.step()
    ms = case.time_steps(K) / K                      # the last 8 of these K strict steps are what the stamps hold
    buf = np.zeros((8, 160, 8), np.uint64)
    assert L.laser_debug_timeline_read(buf.ctypes.data_as(C.c_void_p)) == 0
    t = buf[:, :grid, :].astype(np.int64)
    order = np.argsort(np.median(t[:, :, 0], axis=1))       # slots in launch order
    t = t[order]
    t0 = int(np.median(t[0, :, 0]))
    us = lambda x: (float(x) - t0) / 1e3
    q = lambda v, p: us(np.percentile(v, p))
    done = [int(np.maximum.reduce([c[:, 3], c[:, 4], c[:, 5], c[:, 6]]).max()) for c in t]   # last tail activity of any CTA
    print(f"# Timeline of 8 consecutive strict calls, {describe(w)}\n")
    print("Command: `python -m paper_2606_31580_b200.build --timeline` then `LASER_PROBE_LIB=$PWD/paper_2606_31580_b200/"
          "liblaser_probe_timeline.so python bench.py --timeline` (debug build, -DLASER_TIMELINE: per-CTA %globaltimer stamps).\n")
    print(f"Strict step of this run (CUDA events over {K} back-to-back calls): **{ms * 1e3:.2f} us**; grid {grid} CTAs on the "
          "148 SMs (one CTA per SM: 227 KB of shared memory each).  Times in us from the median CTA entry of the first call shown.  "
          "A call's CTAs do not enter together: under programmatic dependent launch CTA i of call k+1 becomes resident when a "
          "CTA of call k leaves its SM (one SM is free from the start: its CTA enters a whole call early and waits).\n")
    print("| call | CTA entry p05 / p50 / p95 | first W boxes requested p50 | griddepcontrol.wait passed (first / last CTA) "
          "| last producer done issuing | last record stored | call done (last tail activity) |")
    print("|---|---|---|---|---|---|---|")
    for k in range(8):
        c = t[k]
        print(f"| {k} | {q(c[:, 0], 5):.2f} / {q(c[:, 0], 50):.2f} / {q(c[:, 0], 95):.2f} | {q(c[:, 1], 50):.2f} | "
              f"{us(c[:, 2].min()):.2f} / {us(c[:, 2].max()):.2f} | {us(c[:, 7].max()):.2f} | {us(c[:, 3].max()):.2f} | {us(done[k]):.2f} |")
    print("\n| calls | period (done k+1 - done k) | CTAs of k+1 resident before k was done | ... with their first W boxes requested "
          "| mean head start of those requests over all CTAs (us before k was done) | k done -> last CTA of k+1 past the wait |")
    print("|---|---|---|---|---|---|")
    per, head = [], []
    for k in range(7):
        c1 = t[k + 1]
        hs = np.clip(done[k] - c1[:, 1], 0, None) / 1e3
        # the CTA that entered a whole call early on the free SM is not typical: median-based head start as well
        per.append((done[k + 1] - done[k]) / 1e3); head.append(float(np.median(hs)))
        print(f"| {k} -> {k + 1} | {per[-1]:.2f} | {int((c1[:, 0] < done[k]).sum())} of {grid} | {int((c1[:, 1] < done[k]).sum())} | "
              f"{hs.mean():.2f} (median {np.median(hs):.2f}) | {(int(c1[:, 2].max()) - done[k]) / 1e3:.2f} |")
    span = [(done[k] - int(t[k][:, 2].max())) / 1e3 for k in range(8)]
    print(f"\nMean period between completions **{np.mean(per):.2f} us** (= the strict step).  From the last CTA passing the wait to the "
          f"call's completion: {np.mean(span):.2f} us - the part of a call that cannot overlap its predecessor.  A call launched alone "
          "(roofline.kernel_us: bracketed by events, no dependent launch) additionally pays, on every SM, the CTA's start-up, "
          "prologue (barrier init, TMEM allocation, descriptor prefetch) and the latency of its first W boxes, and its last CTAs "
          "finish with most SMs idle; back to back, the median CTA of call k+1 is resident, set up and has its first ring of W "
          f"boxes requested {np.mean(head):.2f} us before call k is done, i.e. that part runs under call k's ramp-down and tail.  "
          "That head start is the difference between the bracketed kernel and the strict step.")


# ----------------------------------------------------------------------------------------- CPU arm
def oracle_sample(w: wl.Workload, gflop_budget: float):
    """Whole requests from the front of the batch worth about `gflop_budget` GFLOP of fp64 work (the
    whole batch if it is smaller): (rows, requests, hidden, offsets, load)."""
    budget_rows = max(4, int(gflop_budget * 1e9 / (2.0 * w.V * w.d)))
    reqs = 0
    while reqs < w.R and int(w.req_offsets[reqs + 1]) <= budget_rows:
        reqs += 1
    reqs = max(reqs, 1)
    rows = int(w.req_offsets[reqs])
    return rows, reqs, w.hidden_f32()[:rows], w.req_offsets[:reqs + 1], w.load[:reqs]


CPU_SAMPLE_GFLOP = 120.0      # C2: the whole 128-row batch (59.7 GFLOP)


def cpu_baseline(w: wl.Workload, target_s: float):
    """The fp64 oracle, as it stands, on this box's host cores, on the same workload (a bounded sample
    for the large configs).  bench.py's cpu_baseline / --impl reference legs are, with tests/ and
    smoke(), the only callers of oracle/ in the repo."""
    import oracle
    tp = oracle.TauParams(**w.tau_params)
    rows, reqs, hid, off, load = oracle_sample(w, CPU_SAMPLE_GFLOP)
    Wf = w.W_f32()
    best, spent, reps = None, 0.0, 0
    while spent < target_s and reps < 20:        # about target_s (10 s) of CPU work
        r = oracle.probe(hid, Wf, off, load, tp)
        best = r.seconds if best is None else min(best, r.seconds)
        spent += r.seconds
        reps += 1
    return dict(value=rows / best, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                sample=f"first {reqs} requests ({rows} rows) of {w.name}, full V and d; best of {reps} runs "
                       f"({best:.2f} s each), fp64, OpenMP over rows",
                requests_per_sec=reqs / best)


def run_reference(args):
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    if rank != 0:
        return
    import oracle
    w = wl.by_name(args.workload, {})
    tp = oracle.TauParams(**w.tau_params)
    Wf = w.W_f32()
    steps, warm = args.steps, args.warmup
    # Each step = the oracle on the sample cpu_baseline times (C2: the whole batch), as long as the
    # whole --steps/--warmup run then ends within a few minutes; otherwise a smaller sample of whole
    # requests (stated in `sample`).
    rows, reqs, hid, off, load = oracle_sample(w, CPU_SAMPLE_GFLOP)
    t_one = oracle.probe(hid, Wf, off, load, tp).seconds
    same_sample = True
    if t_one * (steps + warm) > 150.0:
        same_sample = False
        shrink = 150.0 / (t_one * (steps + warm))
        rows, reqs, hid, off, load = oracle_sample(w, CPU_SAMPLE_GFLOP * shrink * rows / max(rows, 1))
    for _ in range(warm):
        oracle.probe(hid, Wf, off, load, tp)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.probe(hid, Wf, off, load, tp)
    dt = time.perf_counter() - t0
    value = rows * steps / dt
    sample = (f"each step = fp64 oracle on the first {reqs} requests ({rows} rows) of {w.name}, full V and d"
              + (" (the cpu_baseline sample)" if same_sample else " (smaller than the cpu_baseline sample: time cap)"))
    print(json.dumps(dict(
        impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=steps, warmup=warm,
        ms_per_step=dt / steps * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
        data="synthetic", config=dict(workload=describe(w)),
        cpu_baseline=dict(value=value, unit=UNIT, cores=oracle.num_threads(), kind="oracle", sample=sample),
        e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
        gpu_launches=0)), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2")
    ap.add_argument("--sharding", default="requests", choices=["requests", "vocab"])
    ap.add_argument("--exchange", default="peer", choices=["peer", "collective"])
    ap.add_argument("--with-cublas", action="store_true",
                    help="context only: time the plain cuBLAS GEMM hidden @ W^T of the same shape beside the probe")
    ap.add_argument("--kernel-mode", default="auto", choices=KERNEL_MODES,
                    help="laser_probe_options.kernel_mode (auto = the library default; the others force a variant)")
    ap.add_argument("--w-layout", default="rowmajor", choices=W_LAYOUTS,
                    help="rowmajor (default: W as the model stores it) or kblocked (W packed once by "
                         "laser_probe_pack_w; the timed calls get the packed copy)")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--timeline", action="store_true",
                    help="debug: per-CTA timeline of consecutive strict calls (needs the --timeline build, see run_timeline)")
    ap.add_argument("--with-sim-table", action="store_true",
                    help="print the serving simulation's (illustrative) latency table in full")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    args.steps = max(args.steps, 1)
    if args.timeline:
        run_timeline(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
