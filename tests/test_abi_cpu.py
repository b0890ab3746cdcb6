"""CPU-only checks of the C-ABI library: it loads without a GPU, exports every symbol the header
declares, validates arguments, plans launches sanely, and refuses (loudly) to compute without a
B200.  The host-side scalar helpers (tau, EMA, budget) are compared with the oracle."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

import oracle
from paper_2606_31580_b200 import binding as B
from paper_2606_31580_b200 import build as build_mod

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module", autouse=True)
def _built():
    build_mod.build()


def test_header_symbols_all_exported():
    hdr = "".join(f.read_text() for f in sorted((ROOT / "include").glob("*.h")))
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(laser_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations found"
    L = B.lib()
    missing = [s for s in sorted(declared) if not hasattr(L, s)]
    assert not missing, missing
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)


def test_library_is_sm100a_with_tcgen05_and_tma():
    """The shipped binary holds sm_100a SASS with the Blackwell tensor / TMA instructions."""
    import shutil, subprocess
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    so = ROOT / "paper_2606_31580_b200" / "liblaser_probe.so"
    sass = subprocess.run(["cuobjdump", "-sass", str(so)], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    for mnemonic in ("UTCHMMA", "LDTM", "UTMALDG"):
        assert mnemonic in sass, mnemonic
    assert "HMMA." not in sass.replace("UTCHMMA", "")       # no legacy mma.sync path


@pytest.mark.parametrize("dims", [(128, 1536, 151936, 16), (256, 3584, 152064, 32), (1024, 4096, 128256, 64),
                                  (32, 64, 1000, 8), (8, 1536, 151936, 1), (64, 1536, 151936, 8),
                                  (512, 1536, 151936, 64), (4096, 1536, 151936, 512),
                                  (16384, 1536, 151936, 2048), (1, 8, 1, 1), (300, 72, 70001, 20),
                                  (640, 4096, 128256, 64), (1300, 1536, 151936, 100)])
def test_plan_invariants(dims):
    N, d, V, R = dims
    p = B.plan_query(*dims)
    # AUTO: the flex kernel for 129..1024 rows except exactly 256 (checked in test_flex_plan_invariants)
    # unless its fixed 256-row vocabulary tiles quantise badly (test_auto_avoids_flex_for_badly_quantised_vocabularies)
    narrow = d < 768 or (d < 1280 and N > 384)          # narrow hidden sizes: epilogue-bound, see make_plan
    assert p["flex"] == (1 if (128 < N <= 1024 and N != 256 and not narrow) else 0)
    if p["flex"]:
        p = B.plan_query(*dims, mode=B.MODE_MIXED)
    assert p["flex"] == 0
    bn, T, S = p["tile_n"], p["tiles_per_split"], p["splits"]
    pair, tm = p["cta_pair"], p["tile_m"]
    t128 = -(-N // 128)
    mixed = p["mixed"]
    # AUTO outside the flex range / MIXED: one single-CTA kernel up to 128 rows, one CTA-pair kernel up to
    # 256, above that the mixed schedule (single-CTA tail-tile kernel + pair kernel, the tail in whichever
    # has the work)
    assert (pair, mixed) == ((0, 0) if t128 <= 1 else ((1, 0) if t128 == 2 else (1, 1))) and tm == (256 if pair else 128)
    assert p["kernel_launches"] == (2 if mixed else 1)
    assert bn % (32 if pair else 16) == 0 and 16 <= bn <= 256
    assert S * T * bn >= V and (S - 1) * T * bn < V          # splits tile the vocabulary exactly once
    assert p["m_tiles"] == max(1, -(-N // tm)) and p["k_blocks"] == -(-d // 64)
    units = p["num_sms"] // 2 if pair else p["num_sms"]
    assert p["work_items"] == p["m_tiles"] * S
    assert p["grid"] == ((2 * units) if mixed else (2 if pair else 1) * min(units, p["work_items"]))
    assert 2 <= p["stages"] <= 8
    b_rows = bn // 2 if pair else bn                          # W rows one CTA stages per tile
    pipe = p["stages"] * (16384 + b_rows * 128) + 1280        # stages + alignment slack + barrier block
    assert 0 <= p["tail_cache"] <= 512
    assert pipe + (8 * (p["tail_cache"] + 1) if p["tail_cache"] else 0) == p["smem_bytes"] <= 227 * 1024
    if mixed:
        assert p["tail_tile_n"] % 16 == 0 and 16 <= p["tail_tile_n"] <= 256 and p["tail_grid"] == p["num_sms"]
        assert 2 <= p["tail_stages"] <= 8 and p["tail_smem_bytes"] <= 227 * 1024
        assert p["ws_records"] >= N                            # at least one record per row
    else:
        # packed records: at least the full batch's, at most 2x it (a re-plan for fewer token items may
        # use more splits per row, never more than the units allow)
        full = p["m_tiles"] * tm * S
        assert full <= p["ws_records"] <= 2 * full and (p["ws_records"] == full or p["m_tiles"] > 1)
    both = [B.plan_query(*dims, mode=m)["ws_records"] for m in (B.MODE_SINGLE, B.MODE_PAIR)]
    assert B.workspace_bytes(*dims) >= max(16, 16 * max(both + [p["ws_records"]]))
    # the busiest unit does at most ~8 % more than an even share of W rows (+ one tile of slack)
    busy = min(units, p["work_items"])
    rounds = -(-p["work_items"] // busy)
    assert rounds * T * bn <= 1.08 * (p["m_tiles"] * V / busy) + bn


@pytest.mark.parametrize("dims", [(136, 1536, 151936, 17), (256, 3584, 152064, 32), (320, 1536, 151936, 40),
                                  (1024, 4096, 128256, 64), (400, 512, 33000, 40), (130, 64, 1000, 3),
                                  (4096, 1536, 151936, 512), (17, 8, 17, 2), (2000, 256, 300, 9)])
def test_flex_plan_invariants(dims):
    """The flex kernel's plan and its device-side table (one entry per count of 16-row groups)."""
    N, d, V, R = dims
    p = B.plan_query(*dims, mode=B.MODE_FLEX)
    assert p["flex"] == 1 and p["mixed"] == 0 and p["cta_pair"] == 1 and p["kernel_launches"] == 1
    assert p["tile_n"] == 256 and p["grid"] == 2 * (p["num_sms"] // 2) and p["k_blocks"] == -(-d // 64)
    pairs, tiles = p["num_sms"] // 2, -(-V // 256)
    assert p["flex_n_tok"] % 16 == 0 and 16 <= p["flex_n_tok"] <= p["flex_max_tok"] <= 256
    assert p["m_tiles"] * p["flex_n_tok"] >= N and p["splits"] * p["tiles_per_split"] >= tiles
    assert 2 <= p["stages"] <= 8 and 0 <= p["tail_cache"] <= 512
    pipe = p["stages"] * (16384 + p["flex_max_tok"] // 2 * 128) + 1280 + 16384   # ring + slack + transpose blocks
    assert pipe + (8 * (p["tail_cache"] + 1) if p["tail_cache"] else 0) == p["smem_bytes"] <= 227 * 1024
    assert B.workspace_bytes(*dims) >= 16 * p["ws_records"]
    for n_valid in sorted({1, 15, 16, 17, 128, 129, 255, 256, 257, N // 2, N - 1, N} & set(range(1, N + 1))):
        f = B.flex_query(*dims, n_valid)
        C_, nt, S = f["chunks"], f["n_tok"], f["splits"]
        assert nt % 16 == 0 and 16 <= nt <= p["flex_max_tok"]
        assert C_ * nt >= n_valid and (C_ - 1) * nt < n_valid + 16 * C_   # the chunks cover the rows, padding < 16 per chunk
        assert S * f["tiles_per_split"] >= tiles and 1 <= S <= max(4 * pairs, 1)
        assert (C_ * S) % pairs == 0 or S == tiles or C_ * S < pairs      # whole rounds unless V is tiny
        assert min(C_ * nt, N) * 2 * S <= p["ws_records"]                  # 2 S records per row fit the workspace
        assert f["rounds"] == -(-C_ * S // pairs)
    # outside the table's range FLEX falls back to what AUTO does
    if N <= 4096:
        assert B.plan_query(5000, d, V, R, mode=B.MODE_FLEX)["flex"] == 0


def test_packed_w_size_and_argument_checks():
    """K-block-major W (laser_probe_pack_w): size formula and argument validation (no GPU needed)."""
    L = B.lib()
    assert L.laser_probe_packed_w_bytes(151936, 1536) == 24 * 151936 * 128 == 151936 * 1536 * 2
    assert L.laser_probe_packed_w_bytes(1000, 72) == 2 * 1000 * 128          # d padded to the next 64 columns
    assert L.laser_probe_packed_w_bytes(0, 64) == 0 and L.laser_probe_packed_w_bytes(10, 60) == 0
    buf = (C.c_char * 4096)()
    a = C.addressof(buf)
    assert L.laser_probe_pack_w(None, 10, 64, a, None) == -1 and L.laser_probe_pack_w(a, 10, 64, None, None) == -1
    assert L.laser_probe_pack_w(a, 10, 60, a + 2048, None) == -2 and L.laser_probe_pack_w(a, 0, 64, a + 2048, None) == -2
    assert L.laser_probe_pack_w(a + 4, 10, 64, a + 2048, None) == -3


def test_auto_avoids_flex_for_badly_quantised_vocabularies():
    """AUTO keeps the pair / mixed schedule when whole 256-row tiles would leave the busiest pair more than
    15 % above an even share: a G = 8 vocabulary shard of C2 is 75 tiles for 74 pairs."""
    for N in (200, 400, 640, 1024):
        p = B.plan_query(N, 1536, 18992, 16)
        assert p["flex"] == 0 and p["cta_pair"] == 1, (N, p)
        assert B.plan_query(N, 1536, 18992, 16, mode=B.MODE_FLEX)["flex"] == 1        # still available when forced
        assert B.plan_query(N, 1536, 151936, 16)["flex"] == 1                          # the whole vocabulary: 12 % at worst
        assert B.plan_query(N, 1536, 1000, 16)["flex"] == 1                            # fewer tiles than pairs: nothing to balance
    # narrow hidden sizes (the epilogue bounds a tile): flex only where the mixed schedule would pad, or not at all
    assert B.plan_query(320, 1024, 151936, 40)["flex"] == 1 and B.plan_query(512, 1024, 151936, 64)["flex"] == 0
    assert B.plan_query(320, 512, 151936, 40)["flex"] == 0 and B.plan_query(512, 1280, 151936, 64)["flex"] == 1


def test_forced_modes_plan():
    p = B.plan_query(32, 64, 1000, 8, mode=B.MODE_PAIR)
    assert p["cta_pair"] == 1 and p["tile_m"] == 256 and p["grid"] % 2 == 0 and p["tile_n"] % 32 == 0
    p = B.plan_query(4096, 1536, 151936, 512, mode=B.MODE_SINGLE)
    assert p["cta_pair"] == 0 and p["tile_m"] == 128 and p["m_tiles"] == 32
    with pytest.raises(B.LaserError):
        B.plan_query(32, 64, 1000, 8, mode=5)
    # the N = 16384 workspace is tens of MB, not the 77 MB of a max-split stride (round-1 advice)
    assert B.workspace_bytes(16384, 1536, 151936, 2048) < 40e6


def test_options_are_per_call_and_validated():
    """kernel variant, overlap and tail travel in laser_probe_options (no process-wide setters)."""
    L = B.lib()
    o = B.Options(7, 7, None, 7, 1, 7, 1, 1)
    assert L.laser_probe_options_default(C.byref(o)) == 0
    assert (o.aggregate_mode, o.prob_mode, o.token_ids, o.kernel_mode, o.overlap, o.tail, o.w_layout, o.w_ordered) == \
        (0, 0, None, 0, 0, 0, 0, 0)
    assert not hasattr(L, "laser_probe_set_mode") and not hasattr(L, "laser_probe_set_overlap")
    buf = (C.c_char * 4096)()
    a = C.addressof(buf)
    tp, d = B.TauParams(), B.Dims(32, 64, 1000, 8)
    call = lambda opt: L.laser_probe_confidence_opt(a, a, a, a, C.byref(tp), a, a, a, C.byref(d), a, 4096, None,
                                                    None, None, C.byref(opt))
    for bad in (B.Options(kernel_mode=5), B.Options(tail=3), B.Options(aggregate_mode=3), B.Options(prob_mode=2)):
        assert call(bad) == -8                                              # LASER_E_MODE
    o = B.Options(); o.overlap = 2
    assert call(o) == -8
    o = B.Options(); o.w_layout = 2
    assert call(o) == -8
    o = B.Options(); o.w_ordered = 2
    assert call(o) == -8
    assert call(B.Options(prob_mode=B.PROB_TOKEN)) == -1                    # token ids missing
    h = C.c_void_p()
    assert L.laser_probe_handle_create(C.byref(h), C.byref(B.Dims(32, 60, 1000, 8)), None) == -2
    assert L.laser_probe_handle_create(C.byref(h), C.byref(d), C.byref(B.Options(tail=9))) == -8
    assert L.laser_probe_handle_create(None, C.byref(d), None) == -1
    assert L.laser_probe_handle_run(None, a, a, a, a, C.byref(tp), a, a, a, a, 4096, None, None, None) == -1
    assert L.laser_probe_handle_destroy(None) == 0 and L.laser_probe_handle_workspace_bytes(None) == 0


def test_c2_plan_is_the_documented_one():
    p = B.plan_query(128, 1536, 151936, 16)
    assert (p["splits"], p["tiles_per_split"], p["tile_n"], p["stages"], p["grid"]) == (147, 5, 208, 5, 147)


def test_argument_validation_needs_no_gpu():
    L = B.lib()
    tp = B.TauParams()
    assert B.workspace_bytes(128, 1537, 1000, 4) == 0                      # d % 8 != 0
    assert B.workspace_bytes(128, 0, 1000, 4) == 0 and B.workspace_bytes(-1, 64, 1000, 4) == 0
    buf = (C.c_char * 4096)()
    a = C.addressof(buf)
    args = lambda dims, t=tp, mode=0: (a, a, a, a, C.byref(t), a, a, a, C.byref(dims), a, 4096, None, None, None, mode)
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 60, 1000, 8))) == -2    # LASER_E_DIMS
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 64, 1000, 8), B.TauParams(l_target=0.0))) == -4
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 64, 1000, 8), B.TauParams(lambda_min=0.98))) == -4
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 64, 1000, 8), B.TauParams(beta=float("nan")))) == -4
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 64, 1000, 8), tp, 7)) == -8     # LASER_E_MODE
    assert L.laser_probe_confidence_agg(*args(B.Dims(0, 64, 1000, 0))) == 0             # empty batch: no-op
    bad = list(args(B.Dims(32, 64, 1000, 8))); bad[0] = None
    assert L.laser_probe_confidence_agg(*bad) == -1                                     # LASER_E_NULL
    assert L.laser_probe_confidence_agg(*args(B.Dims(32, 64, 1000, 8))[:0], *[a + 2] + list(args(B.Dims(32, 64, 1000, 8)))[1:]) == -3
    for code in range(-9, 1):
        assert L.laser_status_string(code)


def test_shutdown_is_idempotent_and_leaves_the_host_side_usable():
    """laser_shutdown drops cached handles / control blocks (nothing to drop without a GPU) and the
    library stays usable: the host-side queries answer as before."""
    L = B.lib()
    before = B.plan_query(128, 1536, 151936, 16)
    assert L.laser_shutdown() == 0 and L.laser_shutdown() == 0
    assert B.plan_query(128, 1536, 151936, 16) == before
    assert B.workspace_bytes(128, 1536, 151936, 16) > 0


def test_no_cpu_fallback():
    """Without a B200 the compute entry point must fail loudly, never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; covered by the gpu tests")
    L = B.lib()
    buf = (C.c_char * (1 << 20))()
    a = (C.addressof(buf) + 255) // 256 * 256
    rc = L.laser_probe_confidence(a, a, a, a, C.byref(B.TauParams()), a, a, a, C.byref(B.Dims(32, 64, 1000, 8)),
                                  a, 1 << 19, None, None, None)
    assert rc in (-7, -6)                                                  # LASER_E_CUDA / LASER_E_ARCH
    with pytest.raises(B.LaserError):
        B._check(rc)


def test_tau_from_load_matches_oracle():
    rng = np.random.default_rng(0)
    for kw in (dict(), dict(l_target=0.5), dict(beta=0.1, gamma=2.0, l_target=8.0), dict(beta=0.0, lambda_base=0.9)):
        load = (rng.random(257) * 4 * kw.get("l_target", 10.0)).astype(np.float32)
        got = B.tau_from_load(load, B.TauParams(**kw))
        want = oracle.tau(load, oracle.TauParams(**kw))
        np.testing.assert_allclose(got, want, atol=2e-7)
        assert got.min() >= np.float32(0.88) and got.max() <= np.float32(0.97)
    d = B.TauParams()
    B.lib().laser_tau_params_default(C.byref(d))
    assert [round(getattr(d, f), 6) for f, _ in d._fields_] == [0.95, 0.04, 1.0, 10.0, 0.88, 0.97]


def test_ema_and_budget_match_oracle():
    rng = np.random.default_rng(1)
    L = (rng.random((50, 6)) * 30).astype(np.float32)
    lbar = np.zeros(6, np.float32)                                        # Alg. 1 line 1: Lbar <- 0
    traj = []
    for t in range(50):
        B.ema_update(lbar, L[t], alpha=0.3)
        traj.append(lbar.copy())
    traj = np.stack(traj)
    for j in range(6):
        np.testing.assert_allclose(traj[:, j], oracle.ema(L[:, j].astype(np.float64), 0.3), rtol=2e-6)
    pt = rng.integers(1, 600, 500)
    Lr = (rng.random(500) * 60).astype(np.float32)
    got = B.allocate_budget(pt, Lr)
    # the ABI's parameters are doubles: the oracle gets the same unrounded defaults
    want = oracle.budget(pt.astype(np.float64), Lr.astype(np.float64), oracle.BudgetParams())
    assert np.array_equal(got, want)
    assert got.min() >= 2 and got.max() <= 15
    # the whole integer grid, including the points where the exact product of Eq. 6 is an integer
    ps, Ls = np.meshgrid(np.arange(1, 600), np.arange(0, 61), indexing="ij")
    got = B.allocate_budget(ps.ravel(), Ls.ravel().astype(np.float32))
    want = oracle.budget(ps.ravel().astype(np.float64), Ls.ravel().astype(np.float64), oracle.BudgetParams())
    assert np.array_equal(got, want)
    assert list(B.allocate_budget([100, 65], np.asarray([5, 11], np.float32))) == [8, 6]


def test_partial_combine_validation_needs_no_gpu():
    import ctypes as C
    from paper_2606_31580_b200 import binding as B
    L = B.lib()
    d = B.Dims(8, 64, 100, 1)
    tp = B.TauParams()
    assert L.laser_probe_partial(None, None, None, None, C.byref(d), 0, None, None, None, 0, None, None) == -1
    assert L.laser_probe_partial(None, None, None, None, C.byref(d), -1, None, None, None, 0, None, None) == -2
    assert L.laser_probe_combine(None, 0, None, None, C.byref(tp), None, None, None, C.byref(d), None, None,
                                 None, None, None, 0) == -2
    assert L.laser_probe_combine(None, 17, None, None, C.byref(tp), None, None, None, C.byref(d), None, None,
                                 None, None, None, 0) == -2
    assert L.laser_probe_combine(None, 2, None, None, C.byref(tp), None, None, None, C.byref(d), None, None,
                                 None, None, None, 0) == -1


def test_sim_validation_needs_no_gpu():
    L = B.lib()
    pol = B.SimPolicy()
    assert L.laser_sim_policy_default(C.byref(pol)) == 0
    assert (pol.lambda_base, pol.beta, pol.alpha, pol.b_base, pol.p_max) == (0.95, 0.04, 0.3, 10.0, 275.0)
    d = B.SimDims(4, 10, 5, 3)
    args = [None] * 3 + [C.byref(pol), 1] + [None] * 5 + [C.byref(d), 30.0] + [None] * 6
    assert L.laser_sim_run(*args) == -1                      # NULL arrays
    bad = B.SimDims(4, 10, 0, 3)
    args[10] = C.byref(bad)
    assert L.laser_sim_run(*args) == -2
    args[10] = C.byref(d); args[4] = 17
    assert L.laser_sim_run(*args) == -2                      # too many policies
    args[4] = 1
    pol.alpha = 1.5
    assert L.laser_sim_run(*args) == -4
    empty = B.SimDims(0, 10, 5, 3)
    pol.alpha = 0.3
    args[10] = C.byref(empty)
    assert L.laser_sim_run(*args) == 0                       # nothing to simulate


def test_headers_are_plain_c_and_link(tmp_path):
    """include/*.h compile as C99 (no C++-isms, no torch types) and a C program links against the
    library and calls host-only entry points."""
    import shutil, subprocess
    if not shutil.which("gcc"):
        pytest.skip("gcc not on PATH")
    src = tmp_path / "abi.c"
    src.write_text(r'''
#include <stdio.h>
#include "laser_probe.h"
#include "laser_sim.h"
int main(void) {
    laser_tau_params t; laser_sim_policy sp; laser_probe_dims d = {128, 1536, 151936, 16}; laser_probe_plan pl;
    laser_probe_options opt; laser_probe_handle* h = 0; laser_budget_params bp; int rc;
    int32_t prompt[2] = {100, 65}, budget[2]; float L[2] = {5.0f, 11.0f};
    float load[3] = {0.0f, 10.0f, 20.0f}, tau[3];
    if (laser_tau_params_default(&t) != LASER_OK || laser_sim_policy_default(&sp) != LASER_OK) return 1;
    if (laser_tau_from_load(load, 3, &t, tau) != LASER_OK) return 2;
    if (laser_probe_plan_query(&d, &pl) != LASER_OK || laser_probe_workspace_bytes(&d) == 0) return 3;
    if (laser_probe_confidence(0, 0, 0, 0, &t, 0, 0, 0, &d, 0, 0, 0, 0, 0) != LASER_E_NULL) return 4;
    /* the handle API: per-call options; without a B200 creation must fail loudly, never fall back */
    if (laser_probe_options_default(&opt) != LASER_OK) return 5;
    opt.kernel_mode = LASER_MODE_SINGLE; opt.tail = LASER_TAIL_FUSED;
    rc = laser_probe_handle_create(&h, &d, &opt);
    if (rc == LASER_OK) {
        if (laser_probe_handle_plan(h, &pl) != LASER_OK || laser_probe_handle_workspace_bytes(h) == 0) return 6;
        if (laser_probe_handle_run(h, 0, 0, 0, 0, &t, 0, 0, 0, 0, 0, 0, 0, 0) != LASER_E_NULL) return 7;
        if (laser_probe_handle_destroy(h) != LASER_OK) return 8;
    } else if (rc != LASER_E_CUDA && rc != LASER_E_ARCH) return 9;
    if (laser_budget_params_default(&bp) != LASER_OK) return 10;
    if (laser_allocate_budget(prompt, L, 2, &bp, budget) != LASER_OK || budget[0] != 8 || budget[1] != 6) return 11;
    printf("%.6f %.6f %.6f %d %s\n", tau[0], tau[1], tau[2], pl.splits, laser_status_string(LASER_E_ARCH));
    return 0;
}
''')
    exe = tmp_path / "abi"
    so_dir = ROOT / "paper_2606_31580_b200"
    subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", str(ROOT / "include"), str(src),
                    "-o", str(exe), f"-L{so_dir}", "-llaser_probe", f"-Wl,-rpath,{so_dir}"], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert out[:3] == ["0.970000", "0.950000", "0.919536"] and int(out[3]) == 147
