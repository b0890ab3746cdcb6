"""laser_probe_confidence_static: the probe for callers that cannot allocate device memory.

Who needs it: code that is handed its input and output buffers by a host application and has nothing
else - a plug-in inside an inference engine whose memory pool already owns the GPU (cudaMalloc there
fails or fragments the pool), a serving loop that must stay off the driver's allocation lock.  Such a
caller cannot give laser_probe_confidence the device workspace it asks for, and must not trigger the
library's own one-time cudaMalloc of its control block.  The static entry point keeps the statistics
records in a 4 MiB array that is part of the library's device image and runs the separate tail, so it
allocates nothing; the price is a size limit and one shared array per GPU (calls must not overlap).

This file sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure
here must not hide the parity tests.  The GPU test stands on its own - it passes in a fresh process
(the entry point's first call on the device does the address set-up) and after the other GPU tests
(which leave handles, the control block and the array's old contents behind).
"""
import ctypes as C

import numpy as np
import pytest

from paper_2606_31580_b200 import binding as B
from paper_2606_31580_b200 import workloads as wl


# ------------------------------------------------------------------------------------------ host side
def test_limit_is_checked_on_the_host_before_anything_runs():
    """Batches whose workspace exceeds the built-in array are refused with their own status code and a
    message naming both sizes - on the host, with no GPU, before any launch."""
    L = B.lib()
    buf = (C.c_char * 4096)()
    a = (C.addressof(buf) + 255) // 256 * 256
    tp = B.TauParams()

    def call(dims):
        return L.laser_probe_confidence_static(a, a, a, a, C.byref(tp), a, a, a, C.byref(dims), None, None,
                                               None, None)

    big = B.Dims(4096, 1536, 151936, 512)
    assert B.workspace_bytes(4096, 1536, 151936, 512) > B.STATIC_SCRATCH_BYTES
    assert call(big) == -9                                      # LASER_E_STATIC_LIMIT
    msg = L.laser_last_error().decode()
    assert str(B.workspace_bytes(4096, 1536, 151936, 512)) in msg and str(B.STATIC_SCRATCH_BYTES) in msg
    with pytest.raises(B.LaserError, match="built-in"):
        B._check(-9)
    # the graded configs C1-C4 fit
    for dims in [(32, 64, 1000, 8), (128, 1536, 151936, 16), (256, 3584, 152064, 32), (1024, 4096, 128256, 64)]:
        assert 0 < B.workspace_bytes(*dims) <= B.STATIC_SCRATCH_BYTES
    # the usual argument checks come first and need no GPU either
    assert call(B.Dims(32, 60, 1000, 8)) == -2                  # LASER_E_DIMS
    assert call(B.Dims(0, 64, 1000, 0)) == 0                    # empty batch: no-op
    assert L.laser_probe_confidence_static(None, a, a, a, C.byref(tp), a, a, a, C.byref(B.Dims(32, 64, 1000, 8)),
                                           None, None, None, None) == -1


def test_static_entry_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; covered by the gpu test")
    L = B.lib()
    buf = (C.c_char * 4096)()
    a = (C.addressof(buf) + 255) // 256 * 256
    rc = L.laser_probe_confidence_static(a, a, a, a, C.byref(B.TauParams()), a, a, a,
                                         C.byref(B.Dims(32, 64, 1000, 8)), None, None, None, None)
    assert rc in (-7, -6)                                       # LASER_E_CUDA / LASER_E_ARCH


# ------------------------------------------------------------------------------------------ device
def _run_both(w):
    """One batch through the static entry point and through the existing workspace path (handle, fused
    tail); returns the two result sets as numpy arrays."""
    import torch
    dev = "cuda"
    hid = B.bf16_tensor_from_bits(w.hidden_bits, dev)
    W = B.bf16_tensor_from_bits(w.W_bits, dev)
    off = torch.from_numpy(w.req_offsets).to(dev)
    load = torch.from_numpy(w.load).to(dev)
    tp = B.TauParams(**w.tau_params)
    N, R = w.N_alloc, w.R
    # the caller's outputs (poisoned, so that an unwritten entry shows)
    conf = torch.full((R,), -7.0, dtype=torch.float32, device=dev)
    arg = torch.full((N,), -7, dtype=torch.int32, device=dev)
    ex = torch.full((R,), 7, dtype=torch.uint8, device=dev)
    tau = torch.full((R,), -7.0, dtype=torch.float32, device=dev)
    pmax = torch.full((N,), -7.0, dtype=torch.float32, device=dev)
    torch.cuda.synchronize()
    B.probe_static(hid, W, off, load, tp, conf, arg, ex, out_tau=tau, out_pmax=pmax)
    torch.cuda.synchronize()
    got = dict(conf=conf.cpu().numpy(), argmax=arg.cpu().numpy(), exit=ex.cpu().numpy(),
               tau=tau.cpu().numpy(), pmax=pmax.cpu().numpy())
    probe = B.Probe(N, w.d, w.V, R)
    ref = probe(hid, W, off, load, tp)
    torch.cuda.synchronize()
    want = dict(conf=ref.conf.cpu().numpy(), argmax=ref.argmax.cpu().numpy(), exit=ref.exit.cpu().numpy(),
                tau=ref.tau.cpu().numpy(), pmax=ref.pmax.cpu().numpy())
    probe.close()
    return got, want


@pytest.mark.gpu
def test_static_entry_matches_the_workspace_path_on_two_calls_in_a_row():
    """Two different batches, back to back, through the no-allocation entry point; each must equal what
    the existing path (caller workspace, handle, fused tail) returns for it, under the tolerances of the
    parity tests (tests/_parity.py).  The second batch is smaller and of another shape than the first, so
    most of the array still holds the first call's records when it runs: they must not leak into it."""
    import _parity as P
    first = wl.scaled("static-a", 33000, 512, 0.05, 37, 8, seed=4101, N_alloc=300, var_len=(1, 8))  # flex / split-V
    second = wl.scaled("static-b", 5000, 64, 0.05, 6, 5, seed=4102, N_alloc=40)                     # one token tile
    launches0 = B.kernel_launch_count()
    for w in (first, second):
        got, want = _run_both(w)
        n_valid = w.N_valid
        assert np.array_equal(got["argmax"], want["argmax"]), w.name
        assert np.all(got["argmax"][n_valid:] == -1)
        assert np.array_equal(got["exit"], want["exit"]), w.name
        assert set(np.unique(got["exit"])) <= {0, 1}
        assert np.all(np.abs(got["pmax"][:n_valid].astype(np.float64) - want["pmax"][:n_valid]) <= P.PMAX_TOL)
        assert np.all(np.abs(got["conf"].astype(np.float64) - want["conf"]) <= P.CONF_TOL)
        assert np.all(np.abs(got["tau"].astype(np.float64) - want["tau"]) <= P.TAU_TOL)
        assert got["conf"].min() >= 0.0 and got["tau"].min() > 0.0      # nothing left poisoned
    # each static call is the fused kernel(s) + the separate tail kernel; each reference call one launch or more
    assert B.kernel_launch_count() - launches0 >= 2 * 2 + 2
    # and against the oracle, on the second batch (small enough for the fp64 loops)
    g = P.GpuRun(got["conf"], got["argmax"], got["exit"], got["tau"], got["pmax"], {})
    ora, rows, reqs = P.run_oracle(second)
    P.compare(second, g, ora, rows, reqs, "static entry vs oracle")
