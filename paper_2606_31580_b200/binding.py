"""Thin ctypes binding of include/laser_probe.h — argument marshalling only.

Every step of the path (projection, online softmax, aggregate, threshold, exit mask) runs in the CUDA
kernels of csrc/.  torch is used for device memory and streams, nothing else.  There is no CPU or
eager fallback: if liblaser_probe.so is missing this module raises on first use, and on a device
that is not sm_100 the library returns LASER_E_ARCH, which is raised as an error.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from pathlib import Path

import os

# LASER_PROBE_LIB: another build of the SAME library (the -DLASER_TIMELINE debug build, bench.py --timeline)
_SO = Path(os.environ.get("LASER_PROBE_LIB") or Path(__file__).resolve().parent / "liblaser_probe.so")
_lib = None

AGG_MEAN, AGG_GEOMEAN, AGG_MIN = 0, 1, 2
PROB_MAX, PROB_TOKEN = 0, 1
MODE_AUTO, MODE_SINGLE, MODE_PAIR, MODE_FLEX, MODE_MIXED = 0, 1, 2, 3, 4
TAIL_AUTO, TAIL_FUSED, TAIL_SEPARATE = 0, 1, 2
W_ROWMAJOR, W_KBLOCKED = 0, 1

EXPORTS = [
    "laser_tau_params_default", "laser_probe_workspace_bytes", "laser_probe_plan_query",
    "laser_probe_confidence", "laser_probe_confidence_agg", "laser_probe_staging_bytes",
    "laser_probe_confidence_host", "laser_probe_confidence_host_async", "laser_tau_from_load", "laser_ema_update",
    "laser_budget_params_default", "laser_allocate_budget", "laser_status_string",
    "laser_last_error", "laser_kernel_launch_count", "laser_shutdown", "laser_profile_enable",
    "laser_profile_read", "laser_probe_options_default", "laser_probe_plan_query_mode",
    "laser_probe_confidence_opt", "laser_probe_partial", "laser_probe_combine",
    "laser_probe_mixed_query", "laser_probe_flex_query", "laser_probe_packed_w_bytes", "laser_probe_pack_w",
    "laser_probe_handle_create", "laser_probe_handle_destroy", "laser_probe_handle_plan",
    "laser_probe_handle_workspace_bytes", "laser_probe_handle_run", "laser_probe_handle_run_host",
    "laser_sim_policy_default", "laser_sim_run", "laser_probe_confidence_static",
]


class TauParams(C.Structure):
    """laser_tau_params; defaults are the paper's."""
    _fields_ = [(n, C.c_float) for n in
                ("lambda_base", "beta", "gamma", "l_target", "lambda_min", "lambda_max")]

    def __init__(self, lambda_base=0.95, beta=0.04, gamma=1.0, l_target=10.0, lambda_min=0.88,
                 lambda_max=0.97):
        super().__init__(lambda_base, beta, gamma, l_target, lambda_min, lambda_max)


class BudgetParams(C.Structure):
    """laser_budget_params (doubles); defaults PAPER.md:166, 195."""
    _fields_ = [(n, C.c_double) for n in
                ("b_base", "b_min", "f_min", "f_max", "p_min", "p_max", "l_target")]

    def __init__(self, b_base=10.0, b_min=2.0, f_min=0.6, f_max=1.5, p_min=50.0, p_max=275.0,
                 l_target=10.0):
        super().__init__(b_base, b_min, f_min, f_max, p_min, p_max, l_target)


class Dims(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("N", "d", "V", "R")]


class Plan(C.Structure):
    _fields_ = [(n, C.c_int32) for n in
                ("num_sms", "m_tiles", "splits", "tiles_per_split", "tile_n", "k_blocks", "stages",
                 "grid", "work_items", "smem_bytes", "kernel_launches", "tile_m", "cta_pair", "ws_records", "tail_cache",
                 "mixed", "tail_tile_n", "tail_stages", "tail_smem_bytes", "tail_grid",
                 "flex", "flex_n_tok", "flex_max_tok")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


class Mixed(C.Structure):
    """laser_probe_mixed: what the mixed schedule does for n_valid rows (laser_probe_mixed_query)."""
    _fields_ = [(n, C.c_int32) for n in ("mixed", "schedule", "k_pair", "j_single", "u_pair", "u_single",
                                         "splits_pair", "splits_single")] + [("model_us", C.c_float)]


class Flex(C.Structure):
    """laser_probe_flex: what the flex kernel does for n_valid rows (laser_probe_flex_query)."""
    _fields_ = [(n, C.c_int32) for n in ("chunks", "n_tok", "splits", "tiles_per_split", "rounds")] + \
               [("model_cost", C.c_float)]


class Options(C.Structure):
    """laser_probe_options (per call: aggregate, probability, kernel variant, overlap, tail)."""
    _fields_ = [("aggregate_mode", C.c_int32), ("prob_mode", C.c_int32), ("token_ids", C.c_void_p),
                ("kernel_mode", C.c_int32), ("overlap", C.c_int32), ("tail", C.c_int32),
                ("w_layout", C.c_int32), ("w_ordered", C.c_int32)]

    def __init__(self, aggregate_mode=AGG_MEAN, prob_mode=PROB_MAX, token_ids=None, kernel_mode=MODE_AUTO,
                 overlap=0, tail=TAIL_AUTO, w_layout=0, w_ordered=0):
        super().__init__(aggregate_mode, prob_mode, token_ids, kernel_mode, int(bool(overlap)), tail, w_layout,
                         int(bool(w_ordered)))


MAX_PEERS = 16


class Peers(C.Structure):
    """laser_probe_peers (peer-push exchange of the vocabulary-parallel probe)."""
    _fields_ = [("rank", C.c_int32), ("world", C.c_int32), ("epoch", C.c_uint32),
                ("peer_stats", C.c_void_p * MAX_PEERS), ("peer_flags", C.c_void_p * MAX_PEERS)]


class SimPolicy(C.Structure):
    """laser_sim_policy (include/laser_sim.h); defaults = LASER with the paper's parameters."""
    _fields_ = ([(n, C.c_double) for n in
                 ("lambda_base", "beta", "gamma", "l_target", "lambda_min", "lambda_max", "alpha",
                  "b_base", "b_min", "f_min", "f_max", "p_min", "p_max", "budget_l_target")] +
                [(n, C.c_int32) for n in ("early_exit", "adaptive_budget", "fixed_budget", "pad_")])

    def __init__(self, lambda_base=0.95, beta=0.04, gamma=1.0, l_target=10.0, lambda_min=0.88,
                 lambda_max=0.97, alpha=0.3, b_base=10.0, b_min=2.0, f_min=0.6, f_max=1.5, p_min=50.0,
                 p_max=275.0, budget_l_target=10.0, early_exit=1, adaptive_budget=1, fixed_budget=10):
        super().__init__(lambda_base, beta, gamma, l_target, lambda_min, lambda_max, alpha, b_base, b_min,
                         f_min, f_max, p_min, p_max, budget_l_target, early_exit, adaptive_budget,
                         fixed_budget, 0)


class SimDims(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_rep", "n_req", "S", "K")]


class LaserError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"laser_probe status {status}: {text}")
        self.status = status


def lib():
    """Load liblaser_probe.so (built by paper_2606_31580_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise FileNotFoundError(
                f"{_SO} not found: run `python -m paper_2606_31580_b200.build` "
                "(there is no fallback implementation)")
        L = C.CDLL(str(_SO))
        vp, i32p, fp, u8p = C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p
        tp, dp = C.POINTER(TauParams), C.POINTER(Dims)
        L.laser_tau_params_default.argtypes = [tp]
        L.laser_probe_workspace_bytes.argtypes = [dp]
        L.laser_probe_workspace_bytes.restype = C.c_size_t
        L.laser_probe_staging_bytes.argtypes = [dp]
        L.laser_probe_staging_bytes.restype = C.c_size_t
        L.laser_probe_plan_query.argtypes = [dp, C.POINTER(Plan)]
        L.laser_probe_plan_query_mode.argtypes = [dp, C.c_int, C.POINTER(Plan)]
        L.laser_probe_options_default.argtypes = [C.POINTER(Options)]
        L.laser_probe_mixed_query.argtypes = [dp, C.c_int32, C.POINTER(Mixed)]
        L.laser_probe_flex_query.argtypes = [dp, C.c_int32, C.POINTER(Flex)]
        L.laser_probe_packed_w_bytes.argtypes = [C.c_int32, C.c_int32]
        L.laser_probe_packed_w_bytes.restype = C.c_size_t
        L.laser_probe_pack_w.argtypes = [vp, C.c_int32, C.c_int32, vp, vp]
        L.laser_probe_handle_create.argtypes = [C.POINTER(C.c_void_p), dp, C.POINTER(Options)]
        L.laser_probe_handle_destroy.argtypes = [vp]
        L.laser_probe_handle_plan.argtypes = [vp, C.POINTER(Plan)]
        L.laser_probe_handle_workspace_bytes.argtypes = [vp]
        L.laser_probe_handle_workspace_bytes.restype = C.c_size_t
        L.laser_probe_handle_run.argtypes = [vp, vp, vp, i32p, fp, tp, fp, i32p, u8p, vp, C.c_size_t, vp, fp, fp]
        L.laser_probe_handle_run_host.argtypes = [vp, vp, vp, i32p, fp, tp, fp, i32p, u8p, vp, C.c_size_t,
                                                  vp, C.c_size_t, vp, C.c_int]
        common = [vp, vp, i32p, fp, tp, fp, i32p, u8p, dp, vp, C.c_size_t, vp, fp, fp]
        L.laser_probe_confidence.argtypes = common
        L.laser_probe_confidence_agg.argtypes = common + [C.c_int]
        L.laser_probe_confidence_opt.argtypes = common + [C.POINTER(Options)]
        L.laser_probe_confidence_static.argtypes = [vp, vp, i32p, fp, tp, fp, i32p, u8p, dp, vp, fp, fp,
                                                    C.POINTER(Options)]
        L.laser_probe_partial.argtypes = [vp, vp, i32p, i32p, dp, C.c_int32, vp, C.POINTER(Peers), vp,
                                          C.c_size_t, vp, C.POINTER(Options)]
        L.laser_probe_combine.argtypes = [vp, C.c_int32, i32p, fp, tp, fp, i32p, u8p, dp, vp, fp, fp,
                                          C.POINTER(Options), vp, C.c_uint32]
        L.laser_probe_confidence_host.argtypes = [vp, vp, i32p, fp, tp, fp, i32p, u8p, dp, vp,
                                                  C.c_size_t, vp, C.c_size_t, vp]
        L.laser_probe_confidence_host_async.argtypes = L.laser_probe_confidence_host.argtypes
        L.laser_tau_from_load.argtypes = [fp, C.c_int32, tp, fp]
        L.laser_ema_update.argtypes = [fp, fp, C.c_int32, C.c_float]
        L.laser_budget_params_default.argtypes = [C.POINTER(BudgetParams)]
        L.laser_allocate_budget.argtypes = [i32p, fp, C.c_int32, C.POINTER(BudgetParams), i32p]
        L.laser_status_string.argtypes = [C.c_int]
        L.laser_status_string.restype = C.c_char_p
        L.laser_last_error.restype = C.c_char_p
        L.laser_kernel_launch_count.restype = C.c_uint64
        L.laser_profile_enable.argtypes = [C.c_int]
        L.laser_profile_read.argtypes = [C.POINTER(C.c_float), C.POINTER(C.c_float), C.POINTER(C.c_int32)]
        L.laser_sim_policy_default.argtypes = [C.POINTER(SimPolicy)]
        L.laser_sim_run.argtypes = [vp, vp, vp, C.POINTER(SimPolicy), C.c_int32, vp, vp, vp, vp, vp,
                                    C.POINTER(SimDims), C.c_double, vp, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        L = lib()
        txt = L.laser_status_string(rc).decode()
        if rc in (-7, -9):
            txt += " — " + L.laser_last_error().decode()
        raise LaserError(rc, txt)


def plan_query(N, d, V, R, mode=MODE_AUTO) -> dict:
    p = Plan()
    _check(lib().laser_probe_plan_query_mode(C.byref(Dims(N, d, V, R)), mode, C.byref(p)))
    return p.as_dict()


def mixed_query(N, d, V, R, n_valid) -> dict:
    m = Mixed()
    _check(lib().laser_probe_mixed_query(C.byref(Dims(N, d, V, R)), int(n_valid), C.byref(m)))
    return {n: getattr(m, n) for n, _ in m._fields_}


def flex_query(N, d, V, R, n_valid) -> dict:
    m = Flex()
    _check(lib().laser_probe_flex_query(C.byref(Dims(N, d, V, R)), int(n_valid), C.byref(m)))
    return {n: getattr(m, n) for n, _ in m._fields_}


def pack_w(W, stream=None):
    """laser_probe_pack_w: bf16 [V, d] device tensor -> its K-block-major copy (a flat bf16 tensor of
    laser_probe_packed_w_bytes(V, d) / 2 elements) for calls with w_layout=W_KBLOCKED.  Once per model."""
    import torch
    assert W.is_cuda and W.dtype == torch.bfloat16 and W.dim() == 2 and W.is_contiguous()
    V, d = W.shape
    nbytes = int(lib().laser_probe_packed_w_bytes(V, d))
    if nbytes == 0:
        raise LaserError(-2, "invalid W shape")
    out = torch.empty(nbytes // 2, dtype=torch.bfloat16, device=W.device)
    s = (stream or torch.cuda.current_stream(W.device)).cuda_stream
    _check(lib().laser_probe_pack_w(W.data_ptr(), V, d, out.data_ptr(), s))
    return out


def workspace_bytes(N, d, V, R) -> int:
    return int(lib().laser_probe_workspace_bytes(C.byref(Dims(N, d, V, R))))


def staging_bytes(N, d, V, R) -> int:
    return int(lib().laser_probe_staging_bytes(C.byref(Dims(N, d, V, R))))


class Handle:
    """laser_probe_handle: dims + options fixed once; plan, TMA descriptors and control slot cached."""

    def __init__(self, dims: Dims, options: Options):
        self._h = C.c_void_p()
        self._token_keepalive = None
        _check(lib().laser_probe_handle_create(C.byref(self._h), C.byref(dims), C.byref(options)))

    def plan(self) -> dict:
        p = Plan()
        _check(lib().laser_probe_handle_plan(self._h, C.byref(p)))
        return p.as_dict()

    def workspace_bytes(self) -> int:
        return int(lib().laser_probe_handle_workspace_bytes(self._h))

    def close(self):
        if self._h:
            lib().laser_probe_handle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def kernel_launch_count() -> int:
    return int(lib().laser_kernel_launch_count())


def profile_enable(on: bool):
    _check(lib().laser_profile_enable(1 if on else 0))


def profile_read():
    """-> (fused kernel ms summed, finalize kernel ms summed, calls) since the last read."""
    a, b, n = C.c_float(), C.c_float(), C.c_int32()
    _check(lib().laser_profile_read(C.byref(a), C.byref(b), C.byref(n)))
    return a.value, b.value, n.value


def tau_from_load(load, params: TauParams):
    """Host arrays (numpy float32) -> numpy float32; laser_tau_from_load."""
    import numpy as np
    load = np.ascontiguousarray(load, np.float32).reshape(-1)
    out = np.empty_like(load)
    _check(lib().laser_tau_from_load(load.ctypes.data, load.shape[0], C.byref(params), out.ctypes.data))
    return out


def ema_update(lbar, L, alpha=0.3):
    """In place on a numpy float32 array `lbar`; laser_ema_update."""
    import numpy as np
    assert lbar.dtype == np.float32 and lbar.flags.c_contiguous
    L = np.ascontiguousarray(L, np.float32).reshape(-1)
    _check(lib().laser_ema_update(lbar.ctypes.data, L.ctypes.data, lbar.shape[0], alpha))
    return lbar


def allocate_budget(prompt_tokens, L, params: BudgetParams | None = None):
    """laser_allocate_budget, Eq. 6-8."""
    import numpy as np
    pt = np.ascontiguousarray(prompt_tokens, np.int32).reshape(-1)
    L = np.ascontiguousarray(L, np.float32).reshape(-1)
    out = np.empty(pt.shape[0], np.int32)
    q = params or BudgetParams()
    _check(lib().laser_allocate_budget(pt.ctypes.data, L.ctypes.data, pt.shape[0], C.byref(q), out.ctypes.data))
    return out


@dataclass
class ProbeOutputs:
    conf: "torch.Tensor"      # float32 [R]
    argmax: "torch.Tensor"    # int32 [N]
    exit: "torch.Tensor"      # uint8 [R]
    tau: "torch.Tensor | None"
    pmax: "torch.Tensor | None"


class Probe:
    """Caller-owned buffers for repeated probe calls of one shape (device memory from torch; the
    library allocates nothing per call).  mode / overlap / tail are laser_probe_options fields, fixed
    per Probe.  use_handle=True (default) goes through laser_probe_handle_run (one handle per
    aggregate / token-id buffer, created on first use); use_handle=False through the handle-less
    laser_probe_confidence_opt."""

    def __init__(self, N, d, V, R, device="cuda", debug_outputs=True, mode=MODE_AUTO, overlap=False,
                 tail=TAIL_AUTO, use_handle=True, w_layout=W_ROWMAJOR, w_ordered=False):
        import torch
        self.torch = torch
        self.dims = Dims(N, d, V, R)
        self.device = torch.device(device)
        self.mode, self.overlap, self.tail, self.use_handle = mode, bool(overlap), tail, use_handle
        self.w_ordered = bool(w_ordered)   # W is produced on the stream: read it in stream order too
        self.w_layout = w_layout           # W_KBLOCKED: every call's W is a pack_w() copy
        wb = workspace_bytes(N, d, V, R)
        if wb == 0:
            raise LaserError(-2, "invalid dimensions")
        self.workspace = torch.empty(wb, dtype=torch.uint8, device=self.device)
        self.conf = torch.empty(R, dtype=torch.float32, device=self.device)
        self.argmax = torch.empty(N, dtype=torch.int32, device=self.device)
        self.exit = torch.empty(R, dtype=torch.uint8, device=self.device)
        self.tau = torch.empty(R, dtype=torch.float32, device=self.device) if debug_outputs else None
        self.pmax = torch.empty(N, dtype=torch.float32, device=self.device) if debug_outputs else None
        self.plan = plan_query(N, d, V, R, mode)
        fused = 2 if self.plan["mixed"] else 1
        # TAIL_AUTO: the fused tail for strict calls of up to 64 requests, else the finalize kernel (want_fused_tail)
        self.plan["kernel_launches"] = fused + (1 if (tail == TAIL_SEPARATE or (tail == TAIL_AUTO and (overlap or R > 64))) else 0)
        self._handles = {}

    def _options(self, agg, token_ids) -> Options:
        torch = self.torch
        if token_ids is None:
            return Options(agg, PROB_MAX, None, self.mode, self.overlap, self.tail, self.w_layout, self.w_ordered)
        assert token_ids.dtype == torch.int32 and token_ids.numel() == self.dims.N and token_ids.is_contiguous()
        return Options(agg, PROB_TOKEN, token_ids.data_ptr(), self.mode, self.overlap, self.tail, self.w_layout,
                       self.w_ordered)

    def __call__(self, hidden, W, req_offsets, load, params: TauParams, stream=None, agg=AGG_MEAN,
                 token_ids=None):
        """hidden bf16 [N,d], W bf16 [V,d], req_offsets int32 [R+1], load float32 [R] — device
        tensors.  Enqueues on `stream` (default: torch's current stream); does not synchronise.
        token_ids (device int32 [N]) selects LASER_PROB_TOKEN: the aggregate runs over the
        probabilities of those tokens instead of the row maxima."""
        torch = self.torch
        d = self.dims
        assert hidden.dtype == torch.bfloat16 and W.dtype == torch.bfloat16
        assert hidden.is_contiguous() and W.is_contiguous()
        assert tuple(hidden.shape) == (d.N, d.d)
        if self.w_layout == W_KBLOCKED:
            assert W.numel() * 2 == lib().laser_probe_packed_w_bytes(d.V, d.d)    # a pack_w() copy
        else:
            assert tuple(W.shape) == (d.V, d.d)
        assert req_offsets.dtype == torch.int32 and req_offsets.numel() == d.R + 1
        assert load.dtype == torch.float32 and load.numel() == d.R
        s = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        tau = self.tau.data_ptr() if self.tau is not None else None
        pmax = self.pmax.data_ptr() if self.pmax is not None else None
        if self.use_handle:
            key = (agg, token_ids.data_ptr() if token_ids is not None else None)
            h = self._handles.get(key)
            if h is None:
                h = self._handles[key] = Handle(d, self._options(agg, token_ids))
                h._token_keepalive = token_ids
            _check(lib().laser_probe_handle_run(
                h._h, hidden.data_ptr(), W.data_ptr(), req_offsets.data_ptr(), load.data_ptr(),
                C.byref(params), self.conf.data_ptr(), self.argmax.data_ptr(), self.exit.data_ptr(),
                self.workspace.data_ptr(), self.workspace.numel(), s, tau, pmax))
        else:
            opt = self._options(agg, token_ids)
            _check(lib().laser_probe_confidence_opt(
                hidden.data_ptr(), W.data_ptr(), req_offsets.data_ptr(), load.data_ptr(),
                C.byref(params), self.conf.data_ptr(), self.argmax.data_ptr(), self.exit.data_ptr(),
                C.byref(d), self.workspace.data_ptr(), self.workspace.numel(), s, tau, pmax, C.byref(opt)))
        return ProbeOutputs(self.conf, self.argmax, self.exit, self.tau, self.pmax)

    def close(self):
        for h in self._handles.values():
            h.close()
        self._handles = {}


STATIC_SCRATCH_BYTES = 4 << 20     # LASER_STATIC_SCRATCH_BYTES


def probe_static(hidden, W, req_offsets, load, params: TauParams, out_conf, out_argmax, out_exit,
                 stream=None, out_tau=None, out_pmax=None, options: Options | None = None):
    """laser_probe_confidence_static: the probe for callers that have their input and output tensors
    and nothing else - no device workspace to pass and no way to allocate one (a plug-in inside an engine
    whose memory pool owns the GPU, a serving loop that must stay off the driver's allocation lock).

    The statistics records go to a 4 MiB array built into the library (STATIC_SCRATCH_BYTES per GPU,
    held until the process exits); a batch whose workspace_bytes(N, d, V, R) is larger raises LaserError
    with status -9 and launches nothing.  This wrapper allocates nothing either: every tensor, outputs
    included, is the caller's.  All calls on one GPU share that array - keep them in one stream order,
    calls that overlap on the GPU corrupt each other silently.  The first call on a device sets the
    array's address up; make it before any stream capture.  Asynchronous on `stream`."""
    import torch
    assert hidden.is_cuda and hidden.dtype == torch.bfloat16 and hidden.dim() == 2 and hidden.is_contiguous()
    assert W.dtype == torch.bfloat16 and W.is_contiguous()
    N, d = hidden.shape
    R = load.numel()
    w_layout = options.w_layout if options is not None else W_ROWMAJOR
    V = W.shape[0] if w_layout == W_ROWMAJOR else W.numel() // (64 * ((d + 63) // 64))
    assert req_offsets.dtype == torch.int32 and req_offsets.numel() == R + 1
    assert load.dtype == torch.float32
    assert out_conf.dtype == torch.float32 and out_conf.numel() == R
    assert out_argmax.dtype == torch.int32 and out_argmax.numel() == N
    assert out_exit.dtype == torch.uint8 and out_exit.numel() == R
    assert out_tau is None or (out_tau.dtype == torch.float32 and out_tau.numel() == R)
    assert out_pmax is None or (out_pmax.dtype == torch.float32 and out_pmax.numel() == N)
    s = (stream or torch.cuda.current_stream(hidden.device)).cuda_stream
    _check(lib().laser_probe_confidence_static(
        hidden.data_ptr(), W.data_ptr(), req_offsets.data_ptr(), load.data_ptr(), C.byref(params),
        out_conf.data_ptr(), out_argmax.data_ptr(), out_exit.data_ptr(), C.byref(Dims(N, d, V, R)), s,
        out_tau.data_ptr() if out_tau is not None else None,
        out_pmax.data_ptr() if out_pmax is not None else None,
        C.byref(options) if options is not None else None))


class VocabShardProbe:
    """Vocabulary-parallel probe, one instance per GPU (rank g of G): laser_probe_partial over this
    GPU's rows of W, exchange of the 16-byte row records, laser_probe_combine.

    stats_all is the gathered buffer [G, N, 4] (float32 view of laser_row_stats).  `partial` writes
    this rank's records to stats_local [N, 4]; the caller all-gathers them into stats_all (see
    parallel.VocabParallelProbe) and calls `combine`.  With `peers` (parallel.PeerExchange) partial
    pushes the records into every rank's gathered buffer itself and combine waits for the flags."""

    def __init__(self, N, d, V_shard, R, v_offset, world, device="cuda", debug_outputs=True, mode=MODE_AUTO,
                 overlap=False, tail=TAIL_AUTO, w_layout=W_ROWMAJOR):
        import torch
        self.torch = torch
        self.options = Options(AGG_MEAN, PROB_MAX, None, mode, overlap, tail, w_layout)
        self.dims = Dims(N, d, V_shard, R)
        self.v_offset, self.world = int(v_offset), int(world)
        self.device = torch.device(device)
        wb = workspace_bytes(N, d, V_shard, R)
        if wb == 0:
            raise LaserError(-2, "invalid dimensions")
        self.workspace = torch.empty(wb, dtype=torch.uint8, device=self.device)
        self.stats_local = torch.empty((N, 4), dtype=torch.float32, device=self.device)
        self.stats_all = torch.empty((world, N, 4), dtype=torch.float32, device=self.device)
        self.conf = torch.empty(R, dtype=torch.float32, device=self.device)
        self.argmax = torch.empty(N, dtype=torch.int32, device=self.device)
        self.exit = torch.empty(R, dtype=torch.uint8, device=self.device)
        self.tau = torch.empty(R, dtype=torch.float32, device=self.device) if debug_outputs else None
        self.pmax = torch.empty(N, dtype=torch.float32, device=self.device) if debug_outputs else None
        self.plan = plan_query(N, d, V_shard, R, mode)

    def _stream(self, stream):
        return (stream or self.torch.cuda.current_stream(self.device)).cuda_stream

    def partial(self, hidden, W_shard, req_offsets, token_ids=None, stream=None, out=None, peers: Peers | None = None):
        """a1 + a2 over this shard -> stats_local (or `out`, a [N, 4] float32 tensor)."""
        torch, d = self.torch, self.dims
        assert hidden.dtype == torch.bfloat16 and W_shard.dtype == torch.bfloat16
        assert hidden.is_contiguous() and W_shard.is_contiguous()
        assert tuple(hidden.shape) == (d.N, d.d)
        if self.options.w_layout == W_KBLOCKED:
            assert W_shard.numel() * 2 == lib().laser_probe_packed_w_bytes(d.V, d.d)   # pack_w() of the shard
        else:
            assert tuple(W_shard.shape) == (d.V, d.d)
        assert req_offsets.dtype == torch.int32 and req_offsets.numel() == d.R + 1
        if token_ids is not None:
            assert token_ids.dtype == torch.int32 and token_ids.numel() == d.N
        out = self.stats_local if out is None else out
        assert out.dtype == torch.float32 and out.numel() == d.N * 4 and out.is_contiguous()
        _check(lib().laser_probe_partial(
            hidden.data_ptr(), W_shard.data_ptr(), req_offsets.data_ptr(),
            token_ids.data_ptr() if token_ids is not None else None, C.byref(d), self.v_offset,
            out.data_ptr(), C.byref(peers) if peers is not None else None,
            self.workspace.data_ptr(), self.workspace.numel(), self._stream(stream), C.byref(self.options)))
        return out

    def combine(self, req_offsets, load, params: TauParams, stats_all=None, agg=AGG_MEAN, token_prob=False,
                stream=None, wait_flags=None, epoch=0):
        """Merge of the G records per row + a3-a5 -> ProbeOutputs."""
        torch, d = self.torch, self.dims
        st = self.stats_all if stats_all is None else stats_all
        assert st.dtype == torch.float32 and st.numel() == self.world * d.N * 4 and st.is_contiguous()
        opt = Options(agg, PROB_TOKEN if token_prob else PROB_MAX, None)
        _check(lib().laser_probe_combine(
            st.data_ptr(), self.world, req_offsets.data_ptr(), load.data_ptr(), C.byref(params),
            self.conf.data_ptr(), self.argmax.data_ptr(), self.exit.data_ptr(), C.byref(d),
            self._stream(stream), self.tau.data_ptr() if self.tau is not None else None,
            self.pmax.data_ptr() if self.pmax is not None else None, C.byref(opt),
            wait_flags.data_ptr() if wait_flags is not None else None, epoch))
        return ProbeOutputs(self.conf, self.argmax, self.exit, self.tau, self.pmax)


class HostProbe:
    """Host-buffer entry points: per-step tensors in pinned HOST memory, W resident on device.
    use_handle=True: laser_probe_handle_run_host; False: laser_probe_confidence_host[_async]."""

    def __init__(self, N, d, V, R, device="cuda", use_handle=True, mode=MODE_AUTO, tail=TAIL_AUTO,
                 w_layout=W_ROWMAJOR, overlap=False, w_ordered=False):
        import torch
        self.torch = torch
        self.dims = Dims(N, d, V, R)
        self.device = torch.device(device)
        self.workspace = torch.empty(workspace_bytes(N, d, V, R), dtype=torch.uint8, device=self.device)
        self.staging = torch.empty(staging_bytes(N, d, V, R), dtype=torch.uint8, device=self.device)
        self.conf = torch.empty(R, dtype=torch.float32).pin_memory()
        self.argmax = torch.empty(N, dtype=torch.int32).pin_memory()
        self.exit = torch.empty(R, dtype=torch.uint8).pin_memory()
        self.h2d_bytes = N * d * 2 + (R + 1) * 4 + R * 4   # upper bound: only valid rows are copied
        self.d2h_bytes = R * 4 + N * 4 + R
        assert use_handle or w_layout == W_ROWMAJOR      # the handle-less host entry points take row-major W
        assert use_handle or not overlap
        self.handle = (Handle(self.dims, Options(kernel_mode=mode, tail=tail, w_layout=w_layout, overlap=overlap,
                                                 w_ordered=w_ordered))
                       if use_handle else None)

    def _call(self, sync, h_hidden, W, h_req_offsets, h_load, params, stream):
        torch = self.torch
        assert not h_hidden.is_cuda and W.is_cuda
        s = (stream or torch.cuda.current_stream(self.device)).cuda_stream
        common = (h_hidden.data_ptr(), W.data_ptr(), h_req_offsets.data_ptr(), h_load.data_ptr(),
                  C.byref(params), self.conf.data_ptr(), self.argmax.data_ptr(), self.exit.data_ptr())
        tail = (self.workspace.data_ptr(), self.workspace.numel(), self.staging.data_ptr(),
                self.staging.numel(), s)
        if self.handle is not None:
            _check(lib().laser_probe_handle_run_host(self.handle._h, *common, *tail, 1 if sync else 0))
        else:
            fn = lib().laser_probe_confidence_host if sync else lib().laser_probe_confidence_host_async
            _check(fn(*common, C.byref(self.dims), *tail))
        return ProbeOutputs(self.conf, self.argmax, self.exit, None, None)

    def __call__(self, h_hidden, W, h_req_offsets, h_load, params: TauParams, stream=None):
        """Synchronous: results are in the returned host tensors on return."""
        return self._call(True, h_hidden, W, h_req_offsets, h_load, params, stream)

    def submit(self, h_hidden, W, h_req_offsets, h_load, params: TauParams, stream):
        """Asynchronous: enqueue on `stream` and return; the outputs are valid after
        stream.synchronize().  One HostProbe per in-flight batch."""
        return self._call(False, h_hidden, W, h_req_offsets, h_load, params, stream)


def bf16_tensor_from_bits(bits, device=None, pin=False):
    """numpy uint16 bf16 bit patterns -> torch.bfloat16 tensor (no value conversion)."""
    import numpy as np
    import torch
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    if pin:
        t = t.pin_memory()
    return t.to(device) if device is not None else t


def sim_run(arrival, sample_id, policy_id, policies, pool, deadline=30.0, stream=None, details=True):
    """laser_sim_run: many single-server FIFO queues served by Algorithm 1, one per GPU thread.

    arrival float64 [n_req, n_rep], sample_id int32 [n_req, n_rep], policy_id int32 [n_rep] - CUDA
    tensors; policies: list of SimPolicy; pool: dict of CUDA tensors chunk_time / conf float32 [S, K],
    prompt_tokens int32 [S], t_prefill / t_conclusion float32 [S].
    Returns dict(finish, chunks, exited, budget, summary [n_rep, 5]) of CUDA tensors; asynchronous."""
    import torch
    n_req, n_rep = arrival.shape
    S, K = pool["chunk_time"].shape
    dev = arrival.device
    assert arrival.dtype == torch.float64 and arrival.is_contiguous()
    assert sample_id.dtype == torch.int32 and tuple(sample_id.shape) == (n_req, n_rep) and sample_id.is_contiguous()
    assert policy_id.dtype == torch.int32 and policy_id.numel() == n_rep
    for k, dt in (("chunk_time", torch.float32), ("conf", torch.float32), ("prompt_tokens", torch.int32),
                  ("t_prefill", torch.float32), ("t_conclusion", torch.float32)):
        assert pool[k].dtype == dt and pool[k].is_contiguous() and pool[k].device == dev
    pols = (SimPolicy * len(policies))(*policies)
    out = dict(finish=torch.empty((n_req, n_rep), dtype=torch.float64, device=dev),
               chunks=torch.empty((n_req, n_rep), dtype=torch.int32, device=dev),
               exited=torch.empty((n_req, n_rep), dtype=torch.uint8, device=dev) if details else None,
               budget=torch.empty((n_req, n_rep), dtype=torch.int32, device=dev) if details else None,
               summary=torch.empty((n_rep, 5), dtype=torch.float64, device=dev))
    s = (stream or torch.cuda.current_stream(dev)).cuda_stream
    _check(lib().laser_sim_run(
        arrival.data_ptr(), sample_id.data_ptr(), policy_id.data_ptr(), pols, len(policies),
        pool["chunk_time"].data_ptr(), pool["conf"].data_ptr(), pool["prompt_tokens"].data_ptr(),
        pool["t_prefill"].data_ptr(), pool["t_conclusion"].data_ptr(), C.byref(SimDims(n_rep, n_req, S, K)),
        float(deadline), out["finish"].data_ptr(), out["chunks"].data_ptr(),
        out["exited"].data_ptr() if details else None, out["budget"].data_ptr() if details else None,
        out["summary"].data_ptr(), s))
    return out
