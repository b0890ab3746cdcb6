"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  All tests need a B200 (`-m gpu`)."""
import json
import os
from pathlib import Path

import numpy as np
import pytest

from paper_2606_31580_b200 import workloads as wl

pytestmark = pytest.mark.gpu

OUT = Path(os.environ.get("GRAFT_REPO_ROOT", Path(__file__).resolve().parent.parent)) / "gpurun_out"


def _log(name, stats):
    try:
        OUT.mkdir(exist_ok=True)
        with open(OUT / "parity_stats.jsonl", "a") as f:
            f.write(json.dumps(dict(case=name, **stats)) + "\n")
    except OSError:
        pass
    print(name, stats)


@pytest.fixture(scope="module")
def P():
    import _parity as p
    return p


_ORACLE_CACHE = {}


def _oracle_once(P, key, w):
    """The full oracle of an unmodified seeded workload, computed once per session."""
    if key not in _ORACLE_CACHE:
        _ORACLE_CACHE[key] = P.run_oracle(w)
    return _ORACLE_CACHE[key]


# ------------------------------------------------------------------ the five BASELINE.json configs
def test_c1_tiny(P):
    w = wl.config_c1()
    st = P.check(w)
    _log("C1", st)
    assert st["exits"] >= 1                                   # the mask is exercised (DESIGN A16)


@pytest.mark.parametrize("w_layout", [0, 1])
def test_c2_qwen15b_full(P, c2_W_bits, w_layout):
    """The graded config, every row and request, in the launch configuration bench.py times (W row-major,
    and its K-block-major copy from laser_probe_pack_w)."""
    w = wl.config_c2(c2_W_bits)
    P.CFG["w_layout"] = w_layout
    try:
        g = P.run_gpu(w)
    finally:
        P.CFG["w_layout"] = 0
    ora, rows, reqs = _oracle_once(P, "C2", w)
    st = P.compare(w, g, ora, rows, reqs, f"C2/w_layout{w_layout}")
    _log("C2" if w_layout == 0 else "C2/kblocked", st)
    assert st["rows"] == 128 and st["requests"] == 16 and 0 < st["exits"] < 16


@pytest.mark.parametrize("mode", [0, 3])
def test_c3_qwen7b_full(P, force_mode, mode):
    """Every row and request of C3 against the oracle: AUTO (pair kernel, one 256-row item per split) and
    the flex kernel (one 256-token chunk)."""
    force_mode(mode)
    w = wl.config_c3()
    g = P.run_gpu(w)
    assert g.plan["flex"] == (1 if mode == 3 else 0)
    ora, rows, reqs = _oracle_once(P, "C3", w)
    st = P.compare(w, g, ora, rows, reqs, f"C3/mode{mode}")
    _log(f"C3/mode{mode}", st)
    assert st["rows"] == w.N_valid == 256 and st["requests"] == 32


@pytest.mark.parametrize("mode", [0, 4])
def test_c4_llama8b_full(P, force_mode, mode):
    """Every valid row and every request of C4 (variable lengths, padded allocation) against the oracle:
    AUTO (the flex kernel: chunks and splits decided on the device from req_offsets[R], the W boxes
    requested under the dense guess dropped) and the mixed schedule (device-side split of the SMs)."""
    force_mode(mode)
    w = wl.config_c4()
    assert w.N_alloc == 1024 and w.N_valid < 1024
    g = P.run_gpu(w)
    assert g.plan["flex"] == (1 if mode == 0 else 0) and g.plan["mixed"] == (1 if mode == 4 else 0)
    ora, rows, reqs = _oracle_once(P, "C4", w)
    st = P.compare(w, g, ora, rows, reqs, f"C4/mode{mode}")
    _log(f"C4/mode{mode}", st)
    assert st["rows"] == w.N_valid and st["requests"] == w.R == 64
    assert np.all(g.argmax[w.N_valid:] == -1)                 # padding rows (DESIGN A11)
    assert np.all(g.argmax[:w.N_valid] >= 0)


def _stratified_requests(w, item_rows=256, per_half=2, seed=0):
    """Requests sampled so that every item of `item_rows` token rows - and both 128-row halves of it
    (the two CTAs of a pair) - is covered: per_half requests from each half of each item."""
    rng = np.random.default_rng(seed)
    starts = w.req_offsets[:-1]
    pick = []
    for lo in range(0, w.N_valid, item_rows // 2):
        cand = np.flatnonzero((starts >= lo) & (starts < lo + item_rows // 2))
        if len(cand):
            pick.extend(rng.choice(cand, size=min(per_half, len(cand)), replace=False).tolist())
    return np.sort(np.asarray(pick))


@pytest.mark.parametrize("N", wl.C5_NS)
def test_c5_sweep(P, c2_W_bits, N):
    """configs[4]: every row against the oracle up to N = 4096; at N = 16384 (64 items of 256 rows) a
    stratified 2048-row sample that covers every item and both CTAs of every pair."""
    w = wl.config_c5(N, c2_W_bits)
    g = P.run_gpu(w)
    sample = None if N <= 4096 else _stratified_requests(w, 256, 2, seed=N)
    ora, rows, reqs = _oracle_once(P, f"C5:{N}", w) if sample is None else P.run_oracle(w, sample)
    st = P.compare(w, g, ora, rows, reqs, f"C5:{N}")
    _log(f"C5:{N}", st)
    if sample is None:
        assert st["rows"] == N
    else:
        assert st["rows"] >= 2048
        items = set((rows // 128).tolist())
        assert items == set(range(N // 128))                  # every 128-row half of every item
    # properties that hold at any size: planted tokens win; conf within [0,1]; exit is 0/1
    pl = w.planted >= 0
    assert np.all(g.argmax[pl] == w.planted[pl])
    assert np.all((g.conf >= 0) & (g.conf <= 1.0 + 1e-6))
    assert np.all((g.pmax > 0) & (g.pmax <= 1.0))


def test_c5_4096_flex(P, force_mode, c2_W_bits):
    """The flex kernel at the top of its range (16 chunks of 256 tokens), every row against the oracle."""
    force_mode(3)
    w = wl.config_c5(4096, c2_W_bits)
    g = P.run_gpu(w)
    assert g.plan["flex"] == 1 and g.plan["m_tiles"] == 16
    ora, rows, reqs = _oracle_once(P, "C5:4096", w)
    st = P.compare(w, g, ora, rows, reqs, "C5:4096/flex")
    _log("C5:4096/flex", st)
    assert st["rows"] == 4096


# ------------------------------------------------------------------ stress inputs (not timed)
def test_s1_tau_band(P, c2_W_bits):
    """Requests planted around the band where tau(load) decides: the mask depends on load."""
    w = wl.tau_band_stress(c2_W_bits, 0.02, R=40, L=8)
    st = P.check(w)
    _log("S1", st)
    assert 0 < st["exits"] < w.R


def test_literal_generator_flat(P):
    """BASELINE.json's generator taken literally: flat distributions, tiny top-2 gaps."""
    w = wl.literal(151936, 1536, 0.02, 8, 8, seed=wl.SEED_BASE + 7)
    st = P.check(w)
    _log("literal", st)
    assert st["exits"] == 0


@pytest.mark.parametrize("V,d,R,L,n_alloc,var_len", [
    (5000, 256, 12, 8, None, None),        # several tiles, V not a multiple of 16
    (4099, 200, 9, 5, None, None),         # d not a multiple of 64 (k tail), odd V
    (33000, 512, 40, None, 400, (1, 16)),  # 3 token tiles, CSR with padding rows
    (70001, 128, 20, None, 300, (0, 24)),  # empty requests, ragged everything
    (1000, 64, 3, 130, None, None),        # a request longer than one token tile
    (17, 8, 2, 3, None, None),             # V smaller than one tile, d smaller than one k-block
])
def test_scaled_shapes(P, path, V, d, R, L, n_alloc, var_len):
    w = wl.scaled(f"scaled-V{V}-d{d}", V, d, 0.05, R, L, seed=V + d, N_alloc=n_alloc, var_len=var_len)
    st = P.check(w)
    _log(f"{w.name}/{path}", st)


# ------------------------------------------------------------------ both kernel variants on every shape class
@pytest.fixture
def force_mode(P):
    """Force the single-CTA or the CTA-pair kernel (laser_probe_options.kernel_mode) for run_gpu()."""
    def _set(mode):
        P.CFG["mode"] = mode
    yield _set
    P.CFG["mode"] = 0


PATHS = {"auto-handle": dict(tail=0, use_handle=True),       # a3-a5 in the fused kernel's tail up to 64 requests, else the finalize kernel
         "fused-handle": dict(tail=1, use_handle=True),      # fused tail whatever R is (at most 32 finalizer CTAs)
         "separate-handle": dict(tail=2, use_handle=True),   # finalize kernel (LASER_TAIL_SEPARATE)
         "auto-implicit": dict(tail=0, use_handle=False)}    # handle-less entry point, implicit handle


@pytest.fixture(params=list(PATHS))
def path(P, request):
    """Run the test once per call path: fused tail / separate finalize kernel / handle-less ABI."""
    P.CFG.update(PATHS[request.param])
    yield request.param
    P.CFG.update(tail=0, use_handle=True)


@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("V,d,R,L,n_alloc,var_len", [
    (5000, 256, 12, 8, None, None),        # N = 96: the pair's second CTA holds only padding rows
    (33000, 512, 40, None, 400, (1, 16)),  # N = 400: two 256-row items, second one ragged
    (70001, 128, 20, None, 300, (0, 24)),  # empty requests, odd V
    (1000, 64, 3, 130, None, None),        # a request that straddles the two CTAs of a pair
    (17, 8, 2, 3, None, None),             # V smaller than half a tile
])
def test_forced_variants(P, force_mode, path, mode, V, d, R, L, n_alloc, var_len):
    force_mode(mode)
    w = wl.scaled(f"mode{mode}-V{V}-d{d}", V, d, 0.05, R, L, seed=V + d + mode, N_alloc=n_alloc, var_len=var_len)
    st = P.check(w)
    assert st["plan"]["cta_pair"] == (1 if mode >= 2 else 0) and st["plan"]["flex"] == (1 if mode == 3 else 0)
    _log(w.name, st)


@pytest.mark.parametrize("mode", [1, 2, 3, 4])
def test_forced_variants_c5_512(P, force_mode, c2_W_bits, mode):
    force_mode(mode)
    w = wl.config_c5(512, c2_W_bits)
    g = P.run_gpu(w)
    assert g.plan["cta_pair"] == (1 if mode >= 2 else 0) and g.plan["flex"] == (1 if mode == 3 else 0)
    assert g.plan["mixed"] == (1 if mode == 4 else 0)
    ora, rows, reqs = _oracle_once(P, "C5:512", w)
    st = P.compare(w, g, ora, rows, reqs, f"C5:512/mode{mode}")
    assert st["rows"] == 512
    _log(f"C5:512/mode{mode}", st)
    pl = w.planted >= 0
    assert np.all(g.argmax[pl] == w.planted[pl])


@pytest.mark.parametrize("mode", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("R,L,var_len,n_alloc", [
    (20, None, (1, 16), 1000),   # ~170 valid rows of 1000: most token tiles are padding
    (32, 8, None, 1024),         # exactly 256 valid rows: boundary of a pair item
    (33, 8, None, 1024),         # 264 valid rows: one row group into the next item
    (5, 0, None, 700),           # every request empty, several token tiles allocated
])
def test_padding_tiles_are_skipped_and_replanned(P, force_mode, path, mode, R, L, var_len, n_alloc):
    """req_offsets[R] < N leaves whole token tiles of padding: the kernels skip them and re-deal the
    vocabulary over the tiles that hold rows (device-side plan_splits); results must not change."""
    force_mode(mode)
    w = wl.scaled(f"pad-m{mode}-R{R}", 33000, 512, 0.05, R, L, seed=R + 17, N_alloc=n_alloc, var_len=var_len)
    assert w.N_valid < w.N_alloc
    st = P.check(w)
    assert st["plan"]["m_tiles"] > 1
    _log(w.name, st)


@pytest.mark.parametrize("R,L,var_len,n_alloc", [
    (40, 8, None, None),         # N = 320: one pair item + a half-filled tail tile
    (48, 8, None, None),         # N = 384: one pair item + a full tail tile
    (80, 8, None, None),         # N = 640: two pair items + a tail tile
    (9, 8, None, 1024),          # 72 valid rows of 1024: the tail-tile kernel alone, on every SM
    (32, 8, None, 1024),         # 256 valid rows: the pair kernel alone
    (33, 8, None, 1024),         # 264 valid rows: one pair item + a tail tile holding 8 rows
    (74, None, (1, 16), 1024),   # ragged, ~600 valid rows (C4-like)
    (3, 0, None, 700),           # every request empty: neither part has work
])
def test_mixed_schedule_odd_tile_counts(P, force_mode, path, R, L, var_len, n_alloc):
    """Mixed schedule (AUTO above 1024 rows, LASER_MODE_MIXED anywhere above 256): 256-row items on CTA
    pairs, an odd last 128-row tile on single CTAs in a second kernel beside them; which part takes what
    is decided on the device from req_offsets[R].  Requests that straddle the two parts are merged from
    both kernels' records."""
    force_mode(4)
    w = wl.scaled(f"mixed-R{R}-L{L}-N{n_alloc}", 33000, 512, 0.05, R, L, seed=R + 31, N_alloc=n_alloc, var_len=var_len)
    st = P.check(w)
    separate = path == "separate-handle" or (path.startswith("auto") and R > 64)     # AUTO: fused tail up to 64 requests
    assert st["plan"]["mixed"] == 1 and st["plan"]["kernel_launches"] == (3 if separate else 2)
    _log(f"{w.name}/{path}", st)


def test_mixed_schedule_ties_across_the_two_kernels(P, force_mode):
    """Duplicate W rows whose logits tie exactly, for a row of the pair part and a row of the tail tile:
    the lowest index must win in both kernels (different tile heights, different split counts)."""
    from paper_2606_31580_b200 import binding as B
    force_mode(4)
    V, d, N = 40000, 128, 384
    plan = B.plan_query(N, d, V, 3, mode=B.MODE_MIXED)
    assert plan["mixed"] == 1
    rng = np.random.default_rng(19)
    Wf = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((N, d)).astype(np.float32)
    for row in (10, 200, 300):                     # leader CTA, peer CTA, tail-tile kernel
        big = (h[row] * 0.5).astype(np.float32)
        for v1, v2 in [(255, 256), (1000, 30000), (plan["tile_n"] - 1, plan["tile_n"])]:
            W2 = Wf.copy(); W2[v1] = big; W2[v2] = big
            w = wl.Workload("ties-mixed", wl.bf16_bits(W2), wl.bf16_bits(h), wl.fixed_offsets(3, 128),
                            np.array([0.3, 0.7, 0.5], np.float32))
            g = P.run_gpu(w)
            assert g.argmax[row] == v1, (row, v1, v2, g.argmax[row])
            ora, rows, reqs = P.run_oracle(w)
            assert ora.argmax[row] == v1 and ora.gap2[row] == 0.0
            P.compare(w, g, ora, rows, reqs, "ties-mixed")


def test_ties_in_pair_mode(P, force_mode):
    """Duplicate W rows across the two halves of a pair's vocabulary tile, across tiles and splits."""
    from paper_2606_31580_b200 import binding as B
    force_mode(2)
    V, d, N = 20000, 128, 200
    plan = B.plan_query(N, d, V, 2, mode=B.MODE_PAIR)
    assert plan["cta_pair"] == 1 and plan["flex"] == 0
    bn, T, S = plan["tile_n"], plan["tiles_per_split"], plan["splits"]
    assert T >= 2 and S >= 2
    rng = np.random.default_rng(9)
    Wf = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((N, d)).astype(np.float32)
    for row in (0, 150):                            # a row of the leader CTA, a row of the peer CTA
        big = (h[row] * 0.5).astype(np.float32)
        for v1, v2 in [(bn // 2 - 1, bn // 2), (bn - 1, bn), (T * bn - 1, T * bn), (5, S * bn + 7),
                       (5, 3 * bn + 7)]:   # round-robin deal: (5, S*bn+7) = consecutive tiles of split 0
            W2 = Wf.copy(); W2[v1] = big; W2[v2] = big
            w = wl.Workload("ties-pair", wl.bf16_bits(W2), wl.bf16_bits(h), wl.fixed_offsets(2, 100),
                            np.array([0.3, 0.7], np.float32))
            g = P.run_gpu(w)
            assert g.argmax[row] == v1, (row, v1, v2, g.argmax[row], plan)
            ora, rows, reqs = P.run_oracle(w)
            assert ora.argmax[row] == v1 and ora.gap2[row] == 0.0
            P.compare(w, g, ora, rows, reqs, "ties-pair")


def test_ties_in_flex_mode(P, force_mode):
    """Flex kernel: duplicate W rows across the vocabulary quarters of the four epilogue warps (31 | 32),
    the two CTAs of a pair (127 | 128), tiles, consecutive tiles of one split and different splits - for a
    row of the first chunk, of the second chunk, and of a chunk's last 16-token group."""
    from paper_2606_31580_b200 import binding as B
    force_mode(3)
    V, d, N = 20000, 128, 304
    f = B.flex_query(N, d, V, 2, N)
    C_, nt, S = f["chunks"], f["n_tok"], f["splits"]
    assert C_ == 2 and nt == 160 and S >= 2 and f["tiles_per_split"] >= 2
    rng = np.random.default_rng(10)
    Wf = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((N, d)).astype(np.float32)
    for row in (3, 150, 170, 300):                  # chunk 0 (first / last 16-token group), chunk 1 (first / last group)
        big = (h[row] * 0.5).astype(np.float32)
        for v1, v2 in [(31, 32), (127, 128), (255, 256), (5, S * 256 + 7), (5, 3 * 256 + 7), (200, 19999)]:
            W2 = Wf.copy(); W2[v1] = big; W2[v2] = big
            w = wl.Workload("ties-flex", wl.bf16_bits(W2), wl.bf16_bits(h), wl.fixed_offsets(2, 152),
                            np.array([0.3, 0.7], np.float32))
            g = P.run_gpu(w)
            assert g.plan["flex"] == 1
            assert g.argmax[row] == v1, (row, v1, v2, g.argmax[row], f)
            ora, rows, reqs = P.run_oracle(w)
            assert ora.argmax[row] == v1 and ora.gap2[row] == 0.0
            P.compare(w, g, ora, rows, reqs, "ties-flex")


# ------------------------------------------------------------------ closed forms on the GPU
@pytest.mark.parametrize("R,mode", [(4, 0), (40, 3), (40, 4)])      # single kernel / flex (N = 320) / mixed
def test_uniform_logits_gpu(P, force_mode, R, mode):
    """P1 on the device: hidden = 0 -> pmax = 1/V, argmax 0 (lowest index), conf = 1/V."""
    force_mode(mode)
    w = wl.scaled("uniform", 40000, 256, 0.05, R, 8, seed=5)
    w.hidden_bits[:] = 0
    g = P.run_gpu(w)
    assert g.plan["flex"] == (1 if mode == 3 else 0)
    assert np.all(g.argmax == 0)
    np.testing.assert_allclose(g.pmax, 1.0 / w.V, rtol=2e-5)
    np.testing.assert_allclose(g.conf, 1.0 / w.V, rtol=2e-5)
    assert np.all(g.exit == 0)


@pytest.mark.parametrize("reps,mode", [(1, 0), (20, 3), (20, 4)])    # N = 8: single kernel; N = 160: flex / mixed
def test_one_hot_confidence_one(P, force_mode, reps, mode):
    """P2 on the device: W = 40*I, hidden = e_j -> conf = 1 (to fp32), argmax = j, exit."""
    force_mode(mode)
    V = d = 256
    W = wl.bf16_bits((40.0 * np.eye(V)).astype(np.float32))
    js = np.tile(np.array([0, 17, 255, 128, 127, 31, 32, 200]), reps)
    w = wl.Workload("onehot", W, wl.bf16_bits(np.eye(V, dtype=np.float32)[js]),
                    wl.fixed_offsets(2 * reps, 4), np.tile(np.array([0.0, 1.0], np.float32), reps))
    g = P.run_gpu(w)
    assert g.plan["flex"] == (1 if mode == 3 else 0)
    assert np.array_equal(g.argmax, js)
    np.testing.assert_allclose(g.conf, 1.0, atol=1e-6)
    assert np.all(g.exit == 1)


def test_ties_across_tile_and_split_boundaries(P):
    """P3 on the device: duplicate W rows give bit-identical logits; the lowest index must survive the
    in-thread, cross-tile and cross-split merges."""
    from paper_2606_31580_b200 import binding as B
    V, d, N = 80000, 128, 16
    plan = B.plan_query(N, d, V, 2)
    bn, T, S = plan["tile_n"], plan["tiles_per_split"], plan["splits"]
    assert T >= 2 and S >= 2
    rng = np.random.default_rng(8)
    Wf = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((N, d)).astype(np.float32)
    big = (h[0] * 0.5).astype(np.float32)          # strong match for row 0 only
    # tiles are dealt round-robin: split sp owns tiles sp, sp + S, ...
    pairs = [(bn - 1, bn),                         # adjacent tiles = neighbouring splits
             (T * bn - 1, T * bn),
             (5, S * bn + 7),                      # same split, consecutive tiles of it (in-thread merge)
             (bn + 3, (S + 1) * bn + 1),           # same split (1), consecutive tiles
             (5, 3 * bn + 7),                      # different splits
             (31, 32)]                             # same tile, adjacent 32-column chunks
    for v1, v2 in pairs:
        W2 = Wf.copy(); W2[v1] = big; W2[v2] = big
        w = wl.Workload("ties", wl.bf16_bits(W2), wl.bf16_bits(h), wl.fixed_offsets(2, 8),
                        np.array([0.3, 0.7], np.float32))
        g = P.run_gpu(w)
        assert g.argmax[0] == v1, (v1, v2, g.argmax[0], plan)
        ora, rows, reqs = P.run_oracle(w)
        assert ora.argmax[0] == v1 and ora.gap2[0] == 0.0
        P.compare(w, g, ora, rows, reqs, "ties")


@pytest.mark.parametrize("tail,mode", [(1, 1), (1, 2), (2, 4), (0, 0), (1, 4), (2, 3), (0, 3), (1, 3)])   # fused tail on either variant / mixed: separate, auto, fused / flex
@pytest.mark.parametrize("overlap", [True, False])
def test_back_to_back_calls_share_a_workspace(P, overlap, tail, mode):
    """Stream order under programmatic dependent launch: calls enqueued back to back on one stream,
    all on ONE workspace, with alternating inputs.  The fused kernel of call k+1 may start while the
    tail of call k still reads the workspace (laser_probe_options.overlap), and all calls go through
    ONE handle, i.e. one control slot whose counters call k resets just before call k+1 counts;
    every call must still produce its own batch's result."""
    import torch
    from paper_2606_31580_b200 import binding as B
    V, d, R, L = 1000, 64, 48, 8          # short fused kernel, long finalize kernel: the tightest race
    ws = [wl.scaled(f"b2b{i}", V, d, 0.05, R, L, seed=900 + i) for i in range(2)]
    devs = [P.to_device(w) for w in ws]
    oras = [P.run_oracle(w) for w in ws]
    K = 24
    probes = [B.Probe(R * L, d, V, R, overlap=overlap, tail=tail, mode=mode) for _ in range(K)]
    for p in probes[1:]:
        p.workspace = probes[0].workspace
        p._handles = probes[0]._handles          # one handle (one control slot) for all calls
    tp = B.TauParams(**ws[0].tau_params)
    torch.cuda.synchronize()
    n0 = B.kernel_launch_count()
    for k, p in enumerate(probes):
        dv = devs[k % 2]
        p(dv["hidden"], dv["W"], dv["off"], dv["load"], tp)
    assert B.kernel_launch_count() - n0 == K * probes[0].plan["kernel_launches"]
    # N = 384 rows at d = 64: MIXED - and AUTO, which avoids the flex kernel at so narrow a hidden size - is
    # two fused kernels, FLEX one; the merge is one more launch when it is asked for (tail 2) or when AUTO
    # avoids the fused tail (overlap)
    assert probes[0].plan["flex"] == (1 if mode == 3 else 0)
    assert probes[0].plan["kernel_launches"] == (2 if mode in (0, 4) else 1) + (1 if (tail == 2 or (tail == 0 and overlap)) else 0)
    torch.cuda.synchronize()
    for k, p in enumerate(probes):
        g = P.GpuRun(p.conf.cpu().numpy(), p.argmax.cpu().numpy(), p.exit.cpu().numpy(),
                     p.tau.cpu().numpy(), p.pmax.cpu().numpy(), p.plan)
        ora, rows, reqs = oras[k % 2]
        P.compare(ws[k % 2], g, ora, rows, reqs, f"b2b call {k}")
    # the two batches differ, so a call that read the other batch's partials cannot pass
    assert not np.array_equal(oras[0][0].argmax, oras[1][0].argmax)


def test_c2_in_the_configuration_bench_times(P, c2_W_bits):
    """The launch configuration of bench.py's timed regions at full C2 size: strict (the headline) and
    overlap, calls enqueued back to back on one stream through one handle, two resident copies of W
    alternating between calls, one workspace.  Every call's outputs (kept in separate buffers) are
    compared with the oracle."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.config_c2(c2_W_bits)
    dev = P.to_device(w)
    Ws = [dev["W"], dev["W"].clone()]
    ora, rows, reqs = P.run_oracle(w)
    K = 6
    tp = B.TauParams(**w.tau_params)
    for overlap in (False, True):
        probes = [B.Probe(w.N_alloc, w.d, w.V, w.R, overlap=overlap) for _ in range(K)]
        for p in probes[1:]:
            p.workspace = probes[0].workspace
            p._handles = probes[0]._handles
        for p in probes:
            p.conf.fill_(-7.0); p.argmax.fill_(-7); p.exit.fill_(7); p.pmax.fill_(-7.0)
        torch.cuda.synchronize()
        n0 = B.kernel_launch_count()
        for k, p in enumerate(probes):
            p(dev["hidden"], Ws[k % 2], dev["off"], dev["load"], tp)
        assert B.kernel_launch_count() - n0 == K * probes[0].plan["kernel_launches"]
        assert probes[0].plan["kernel_launches"] == (2 if overlap else 1)   # strict: one launch per call
        torch.cuda.synchronize()
        for k, p in enumerate(probes):
            g = P.GpuRun(p.conf.cpu().numpy(), p.argmax.cpu().numpy(), p.exit.cpu().numpy(),
                         p.tau.cpu().numpy(), p.pmax.cpu().numpy(), p.plan)
            st = P.compare(w, g, ora, rows, reqs, f"c2 bench configuration, overlap={overlap}, call {k}")
        _log(f"c2-bench-config/overlap={overlap}", st)


# ------------------------------------------------------------------ semantics fixed at the boundary
@pytest.mark.parametrize("L,mode", [(4, 0), (60, 3), (60, 4), (60, 2)])   # single kernel / flex / mixed / pair
def test_nan_row_poisons_only_its_request(P, force_mode, L, mode):
    """DESIGN A12 through every kernel: a NaN in one row makes that row's pmax and its request's conf NaN
    (exit 0) and leaves the other requests alone."""
    force_mode(mode)
    w = wl.scaled("nan", 3000, 64, 0.05, 3, L, seed=11)
    row = L + 1                                      # a row of request 1
    hf = w.hidden_f32().copy(); hf[row, 7] = np.nan
    w.hidden_bits = wl.bf16_bits(hf)
    g = P.run_gpu(w)
    assert g.plan["flex"] == (1 if mode == 3 else 0)
    assert np.isnan(g.conf[1]) and g.exit[1] == 0 and np.isnan(g.pmax[row])
    assert np.isfinite(g.conf[0]) and np.isfinite(g.conf[2])
    assert np.isfinite(np.delete(g.pmax, row)).all()
    ora, _, _ = P.run_oracle(w)
    np.testing.assert_allclose(g.conf[[0, 2]], ora.conf[[0, 2]], atol=2e-3)


def test_empty_batches_and_requests(P):
    import torch
    from paper_2606_31580_b200 import binding as B
    tp = B.TauParams(l_target=0.5)
    # R = 0, N = 0: no-op, no launch
    before = B.kernel_launch_count()
    pr = B.Probe(0, 64, 1000, 0)
    z16 = torch.empty((0, 64), dtype=torch.bfloat16, device="cuda")
    W = torch.zeros((1000, 64), dtype=torch.bfloat16, device="cuda")
    pr(z16, W, torch.zeros(1, dtype=torch.int32, device="cuda"),
       torch.empty(0, dtype=torch.float32, device="cuda"), tp)
    assert B.kernel_launch_count() == before
    # R = 0, N = 4: all rows are padding
    pr = B.Probe(4, 64, 1000, 0)
    pr.argmax.fill_(5)
    pr(torch.zeros((4, 64), dtype=torch.bfloat16, device="cuda"), W,
       torch.zeros(1, dtype=torch.int32, device="cuda"), torch.empty(0, dtype=torch.float32, device="cuda"), tp)
    torch.cuda.synchronize()
    assert pr.argmax.cpu().tolist() == [-1] * 4
    # all requests empty: conf 0, exit 0, tau defined
    w = wl.scaled("emptyreq", 2000, 64, 0.05, 3, 0, seed=12, N_alloc=8)
    g = P.run_gpu(w)
    assert np.all(g.conf == 0) and np.all(g.exit == 0) and np.all(g.argmax == -1)
    assert np.all((g.tau >= 0.88) & (g.tau <= 0.97))


def test_exit_is_strict_on_device(P):
    """conf == tau must not exit: beta = 0, lambda_base = the GPU's own conf of a one-row request."""
    from paper_2606_31580_b200 import binding as B
    V = d = 64
    W = wl.bf16_bits((3.0 * np.eye(V)).astype(np.float32))
    w = wl.Workload("strict", W, wl.bf16_bits(np.eye(V, dtype=np.float32)[[2]]),
                    wl.fixed_offsets(1, 1), np.array([0.3], np.float32))
    c = float(P.run_gpu(w).conf[0])
    for lam, want in [(c, 0), (np.nextafter(np.float32(c), np.float32(0)), 1),
                      (np.nextafter(np.float32(c), np.float32(1)), 0)]:
        tp = dict(lambda_base=float(lam), beta=0.0, gamma=1.0, l_target=0.5, lambda_min=0.0, lambda_max=1.0)
        g = P.run_gpu(w, tau_params=tp)
        assert g.tau[0] == np.float32(lam) and g.exit[0] == want


def test_lower_clamp_and_fixed_threshold(P):
    """beta = 0.1 reaches lambda_min (DESIGN A8); beta = 0 is the Fixed-High baseline (P9)."""
    w = wl.config_c1()
    for tp in (dict(wl.TAU_DEFAULTS_NORMALISED, beta=0.1), dict(wl.TAU_DEFAULTS_NORMALISED, beta=0.0)):
        w.load = np.linspace(0, 3, w.R).astype(np.float32)
        st = P.check(w, tau_params=tp)
    g = P.run_gpu(w, tau_params=dict(wl.TAU_DEFAULTS_NORMALISED, beta=0.1))
    assert g.tau.min() == np.float32(0.88) and g.tau.max() == np.float32(0.97)


@pytest.mark.parametrize("agg", [1, 2])
def test_aggregate_modes(P, path, agg):
    """NEXT-1: geometric mean / min over the request's tokens in the same fused reduction."""
    w = wl.scaled("agg", 12000, 256, 0.05, 10, None, seed=21, var_len=(1, 9))
    st = P.check(w, agg=agg)
    _log(f"agg{agg}", st)


def test_deterministic_and_host_entry(P, c2_W_bits):
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.config_c5(64, c2_W_bits)
    dev = P.to_device(w)
    a = P.run_gpu(w, dev)
    b = P.run_gpu(w, dev)
    for f in ("conf", "argmax", "exit", "pmax"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    hp = B.HostProbe(w.N_alloc, w.d, w.V, w.R)
    hh = B.bf16_tensor_from_bits(w.hidden_bits, pin=True)
    out = hp(hh, dev["W"], torch.from_numpy(w.req_offsets).pin_memory(),
             torch.from_numpy(w.load).pin_memory(), B.TauParams(**w.tau_params))
    assert np.array_equal(out.conf.numpy(), a.conf) and np.array_equal(out.argmax.numpy(), a.argmax)
    assert np.array_equal(out.exit.numpy(), a.exit)
    # asynchronous form: two batches in flight on two streams, results valid after the stream sync
    hps = [B.HostProbe(w.N_alloc, w.d, w.V, w.R) for _ in range(2)]
    sts = [torch.cuda.Stream() for _ in range(2)]
    w2 = wl.config_c5(64, c2_W_bits)
    w2.load = (1.0 - w.load).astype(np.float32)                 # second batch: other thresholds
    a2 = P.run_gpu(w2, dev=dict(dev, load=torch.from_numpy(w2.load).cuda()))
    ins = [(hh, torch.from_numpy(w.req_offsets).pin_memory(), torch.from_numpy(w.load).pin_memory()),
           (hh, torch.from_numpy(w2.req_offsets).pin_memory(), torch.from_numpy(w2.load).pin_memory())]
    for rep in range(3):
        for k in range(2):
            hps[k].submit(ins[k][0], dev["W"], ins[k][1], ins[k][2], B.TauParams(**w.tau_params), sts[k])
        for k, want in enumerate((a, a2)):
            sts[k].synchronize()
            assert np.array_equal(hps[k].conf.numpy(), want.conf) and np.array_equal(hps[k].exit.numpy(), want.exit)
            assert np.array_equal(hps[k].argmax.numpy(), want.argmax)
    # pageable host buffers take the staged-copy path; same results
    hp2 = B.HostProbe(w.N_alloc, w.d, w.V, w.R)
    hp2.conf, hp2.argmax, hp2.exit = (torch.full((w.R,), -7.0), torch.full((w.N_alloc,), -7, dtype=torch.int32),
                                      torch.full((w.R,), 7, dtype=torch.uint8))
    out2 = hp2(B.bf16_tensor_from_bits(w.hidden_bits), dev["W"], torch.from_numpy(w.req_offsets.copy()),
               torch.from_numpy(w.load.copy()), B.TauParams(**w.tau_params))
    assert np.array_equal(out2.conf.numpy(), a.conf) and np.array_equal(out2.argmax.numpy(), a.argmax)
    assert np.array_equal(out2.exit.numpy(), a.exit)


@pytest.mark.parametrize("pinned", [True, False])
def test_host_entry_through_an_overlap_handle(P, pinned):
    """laser_probe_handle_run_host stages `hidden` on the stream just ahead of the fused kernel (its own
    staging kernel for pinned memory, a copy otherwise).  A handle created with overlap = 1 lets the fused
    kernel read its inputs while the kernel ahead still runs - which here is that producer: the host entry
    must order the read behind it regardless.  Two batches alternate through one handle and one staging
    buffer, so a kernel that read early would see the other batch's rows."""
    import torch
    from paper_2606_31580_b200 import binding as B
    V, d, R, L = 20000, 256, 12, 8
    ws = [wl.scaled(f"hostovl{i}", V, d, 0.05, R, L, seed=300 + i) for i in range(2)]
    ws[1].W_bits = ws[0].W_bits                  # one resident W; the per-step tensors differ
    W = B.bf16_tensor_from_bits(ws[0].W_bits, "cuda")
    wants = [P.run_gpu(w, dev=dict(P.to_device(w), W=W)) for w in ws]
    assert not np.array_equal(wants[0].argmax, wants[1].argmax)
    hp = B.HostProbe(R * L, d, V, R, overlap=True)
    if not pinned:
        hp.conf, hp.argmax, hp.exit = (torch.empty(R), torch.empty(R * L, dtype=torch.int32),
                                       torch.empty(R, dtype=torch.uint8))
    ins = []
    for w in ws:
        t = (B.bf16_tensor_from_bits(w.hidden_bits, pin=pinned), torch.from_numpy(w.req_offsets.copy()),
             torch.from_numpy(w.load.copy()))
        ins.append(tuple(x.pin_memory() for x in t) if pinned else t)
    for k in range(20):
        out = hp(*ins[k % 2][:1], W, *ins[k % 2][1:], B.TauParams(**ws[0].tau_params))
        want = wants[k % 2]
        assert np.array_equal(out.argmax.numpy(), want.argmax), f"call {k}"
        # (an overlap handle's AUTO tail is the finalize kernel: eight warps sum a request's rows instead of four,
        # so conf may differ from the fused tail's in the last place)
        assert np.allclose(out.conf.numpy(), want.conf, rtol=0, atol=1e-6) and np.array_equal(out.exit.numpy(), want.exit), f"call {k}"


@pytest.mark.parametrize("mode", [0, 2, 3])        # single-CTA kernel / CTA pairs / flex: the three places W is requested early
def test_w_produced_on_the_stream(P, mode):
    """laser_probe_options.w_ordered = 1: W is read in stream order like every other input.  Here W is
    WRITTEN on the stream just ahead of the probe by a kernel that lets its dependents start at once -
    the library's own staging kernel (griddepcontrol.launch_dependents at entry), pointed at W: the host
    entry's staging buffer is the W buffer itself, so each call copies the step's `hidden` rows from
    pinned memory over W's first rows and then probes `hidden` against that W.  Two batches alternate;
    every call must see the rows written for it (a W box requested ahead of the wait would hold the other
    batch's).  Reference: the same W assembled with torch, through the default path."""
    import torch
    from paper_2606_31580_b200 import binding as B
    V, d, R, L = 9000, 256, (12 if mode == 0 else 36), 8
    N = R * L
    ws = [wl.scaled(f"wprod{i}", V, d, 0.05, R, L, seed=500 + i) for i in range(2)]
    W0 = B.bf16_tensor_from_bits(ws[0].W_bits, "cuda")
    tp = B.TauParams(**ws[0].tau_params)
    wants = []
    for w in ws:
        hid = B.bf16_tensor_from_bits(w.hidden_bits, "cuda")
        Wk = W0.clone()
        Wk[:N] = hid                                   # what the staging kernel will have written
        pr = B.Probe(N, d, V, R, mode=mode)
        o = pr(hid, Wk, torch.from_numpy(w.req_offsets).cuda(), torch.from_numpy(w.load).cuda(), tp)
        torch.cuda.synchronize()
        wants.append((o.argmax.cpu().numpy().copy(), o.conf.cpu().numpy().copy(), o.exit.cpu().numpy().copy()))
        pr.close()
    # row n of such a W is hidden row n, so with the rows written for THIS call argmax[n] = n for nearly every row
    # (|h_n|^2 beats every other logit unless another row shares its planted token with a larger shift); against
    # the other batch's rows - what an early W box would hold - it cannot be: the check below is sensitive
    assert all(np.mean(wt[0] == np.arange(N)) > 0.9 for wt in wants)
    assert not np.array_equal(ws[0].hidden_bits, ws[1].hidden_bits)
    Wbuf = W0.clone()
    assert Wbuf.data_ptr() % 256 == 0 and B.staging_bytes(N, d, V, R) <= Wbuf.numel() * 2
    hp = B.HostProbe(N, d, V, R, mode=mode, w_ordered=True)
    # the staging buffer IS W: hidden lands in its first N rows (with pinned offsets / load / outputs the host
    # entry stages nothing else)
    hp.staging = Wbuf.view(torch.uint8).view(-1)
    ins = [(B.bf16_tensor_from_bits(w.hidden_bits, pin=True), torch.from_numpy(w.req_offsets.copy()).pin_memory(),
            torch.from_numpy(w.load.copy()).pin_memory()) for w in ws]
    st = torch.cuda.Stream()
    for k in range(24):
        hp.submit(ins[k % 2][0], Wbuf, ins[k % 2][1], ins[k % 2][2], tp, st)
        if k % 3 == 2 or k == 23:                      # mostly back to back: the calls chain under dependent launch
            st.synchronize()
            want = wants[k % 2]
            assert np.array_equal(hp.argmax.numpy(), want[0]), f"call {k}"
            assert np.array_equal(hp.conf.numpy(), want[1]) and np.array_equal(hp.exit.numpy(), want[2]), f"call {k}"
    # and w_ordered changes nothing else: same results as the default on resident weights
    w = ws[0]
    dev = P.to_device(w)
    a = B.Probe(N, d, V, R, mode=mode)(dev["hidden"], dev["W"], dev["off"], dev["load"], tp)
    b = B.Probe(N, d, V, R, mode=mode, w_ordered=True)(dev["hidden"], dev["W"], dev["off"], dev["load"], tp)
    torch.cuda.synchronize()
    assert torch.equal(a.argmax, b.argmax) and torch.equal(a.conf, b.conf) and torch.equal(a.exit, b.exit)


def test_shutdown_then_use_again(P):
    """laser_shutdown drops the implicit handles and, with no handle left, the control block; the next
    call sets everything up again and gives the same result (implicit and explicit handles, fused tail)."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.scaled("shutdown", 9000, 128, 0.05, 10, 8, seed=77)
    P.CFG.update(use_handle=False)
    try:
        a = P.run_gpu(w)
        torch.cuda.synchronize()
        assert B.lib().laser_shutdown() == 0 and B.lib().laser_shutdown() == 0
        b = P.run_gpu(w)
    finally:
        P.CFG.update(use_handle=True)
    c = P.run_gpu(w)                         # explicit handle after the shutdown
    for f in ("conf", "argmax", "exit", "pmax", "tau"):
        assert np.array_equal(getattr(a, f), getattr(b, f)) and np.array_equal(getattr(a, f), getattr(c, f)), f


def test_error_codes_on_device(P):
    import torch
    from paper_2606_31580_b200 import binding as B
    w = wl.config_c1()
    dev = P.to_device(w)
    pr = B.Probe(w.N_alloc, w.d, w.V, w.R)
    tp = B.TauParams(l_target=0.5)
    with pytest.raises(B.LaserError) as e:
        pr.workspace = pr.workspace[:64]
        pr(dev["hidden"], dev["W"], dev["off"], dev["load"], tp)
    assert e.value.status == -5
    pr = B.Probe(w.N_alloc, w.d, w.V, w.R)
    with pytest.raises(B.LaserError) as e:
        pr(dev["hidden"], dev["W"], dev["off"], dev["load"], B.TauParams(lambda_min=0.99, lambda_max=0.9))
    assert e.value.status == -4
    mis = torch.empty(w.V * w.d + 8, dtype=torch.bfloat16, device="cuda")[1:1 + w.V * w.d].view(w.V, w.d)
    with pytest.raises(B.LaserError) as e:
        pr(dev["hidden"], mis, dev["off"], dev["load"], tp)
    assert e.value.status == -3


def test_cuda_graph_capture_and_replay(P, c2_W_bits):
    """A serving engine captures its decode step in a CUDA graph: the probe call (one kernel launch
    with the programmatic-dependent-launch attribute, no synchronisation, no allocation) must be
    capturable, and a replay must read the CURRENT contents of the input buffers."""
    import torch
    from paper_2606_31580_b200 import binding as B
    w1 = wl.config_c2(c2_W_bits)
    w2 = wl.config_c2(c2_W_bits, seed=wl.SEED_BASE + 2 + 7919)          # another batch, same shapes
    d1, d2 = P.to_device(w1), P.to_device(w2)
    hidden, off, load = d1["hidden"].clone(), d1["off"].clone(), d1["load"].clone()
    probe = B.Probe(w1.N_alloc, w1.d, w1.V, w1.R)
    tp = B.TauParams(**w1.tau_params)
    probe(hidden, d1["W"], off, load, tp)                               # warm-up outside capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            probe(hidden, d1["W"], off, load, tp, stream=side)
    for w, d in ((w1, d1), (w2, d2), (w1, d1)):
        hidden.copy_(d["hidden"]); off.copy_(d["off"]); load.copy_(d["load"])
        probe.conf.fill_(-7.0); probe.argmax.fill_(-7); probe.exit.fill_(7)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        run = P.GpuRun(probe.conf.cpu().numpy(), probe.argmax.cpu().numpy(), probe.exit.cpu().numpy(),
                       probe.tau.cpu().numpy(), probe.pmax.cpu().numpy(), probe.plan)
        ora, rows, reqs = P.run_oracle(w)
        P.compare(w, run, ora, rows, reqs, f"graph replay {w.name}")
    # replay latency of one captured call, for the record
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ts = []
    for _ in range(20):
        torch.cuda.synchronize(); e0.record(); g.replay(); e1.record(); torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    print("graph replay, one call: median %.1f us" % sorted(ts)[len(ts) // 2])


def test_cuda_graph_replay_replans_the_flex_kernel(P):
    """The flex kernel decides chunks and splits from req_offsets[R] on the device, so ONE captured graph
    serves batches with different numbers of valid rows in the same allocation: a dense batch (the guess
    its W boxes are requested under holds), a half-empty one and a nearly empty one (the guess is dropped)."""
    import torch
    from paper_2606_31580_b200 import binding as B
    V, d, n_alloc = 33000, 512, 640
    w0 = wl.scaled("graph-flex-dense", V, d, 0.05, 80, 8, seed=61, N_alloc=n_alloc)
    mk = lambda name, seed, var_len: wl._qwen_like(name, V, d, 0.05, 80, None, 0.9, seed, "uniform", W_bits=w0.W_bits,
                                                   N_alloc=n_alloc, var_len=var_len)     # the same W: it is in the graph
    ws = [w0, mk("graph-flex-half", 62, (1, 8)), mk("graph-flex-few", 63, (0, 1))]
    assert ws[0].N_valid == n_alloc and ws[1].N_valid < 400 and ws[2].N_valid < 100
    chunks = {B.flex_query(n_alloc, d, V, 80, w.N_valid)["chunks"] for w in ws}
    assert len(chunks) >= 2                                   # the replays really take different decompositions
    devs = [P.to_device(w) for w in ws]
    hidden, off, load = devs[0]["hidden"].clone(), devs[0]["off"].clone(), devs[0]["load"].clone()
    probe = B.Probe(n_alloc, d, V, 80, mode=B.MODE_FLEX)
    assert probe.plan["flex"] == 1
    tp = B.TauParams(**ws[0].tau_params)
    probe(hidden, devs[0]["W"], off, load, tp)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            probe(hidden, devs[0]["W"], off, load, tp, stream=side)
    for k in (0, 1, 2, 1, 0):
        w, dv = ws[k], devs[k]
        hidden.copy_(dv["hidden"]); off.copy_(dv["off"]); load.copy_(dv["load"])
        probe.conf.fill_(-7.0); probe.argmax.fill_(-7); probe.exit.fill_(7); probe.pmax.fill_(-7.0)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        run = P.GpuRun(probe.conf.cpu().numpy(), probe.argmax.cpu().numpy(), probe.exit.cpu().numpy(),
                       probe.tau.cpu().numpy(), probe.pmax.cpu().numpy(), probe.plan)
        ora, rows, reqs = P.run_oracle(w)
        P.compare(w, run, ora, rows, reqs, f"flex graph replay {w.name}")


def test_flex_back_to_back_with_changing_row_counts(P):
    """Stress of the flex kernel's guess-and-drop protocol under programmatic dependent launch: 10 x 48 calls
    enqueued back to back through ONE handle and ONE workspace, cycling over batches whose valid-row count
    makes the kernel keep (dense) or drop (padded) the W boxes it requested ahead of the wait, with a
    different decomposition from one call to the next.  Every call's outputs must be bit-identical to those
    of the same batch run alone, which are checked against the oracle."""
    import torch
    from paper_2606_31580_b200 import binding as B
    V, d, n_alloc, R = 33000, 512, 640, 80
    w0 = wl.scaled("stress-flex-dense", V, d, 0.05, R, 8, seed=71, N_alloc=n_alloc)
    mk = lambda name, seed, var_len: wl._qwen_like(name, V, d, 0.05, R, None, 0.9, seed, "uniform", W_bits=w0.W_bits,
                                                   N_alloc=n_alloc, var_len=var_len)
    ws = [w0, mk("stress-flex-half", 72, (1, 8)), mk("stress-flex-few", 73, (0, 2)), mk("stress-flex-most", 74, (4, 8))]
    devs = [P.to_device(w) for w in ws]
    tp = B.TauParams(**ws[0].tau_params)
    ref = []
    for w, dv in zip(ws, devs):                  # each batch alone, against the oracle
        pr = B.Probe(n_alloc, d, V, R, mode=B.MODE_FLEX)
        assert pr.plan["flex"] == 1
        out = pr(dv["hidden"], devs[0]["W"], dv["off"], dv["load"], tp)
        torch.cuda.synchronize()
        g = P.GpuRun(out.conf.cpu().numpy(), out.argmax.cpu().numpy(), out.exit.cpu().numpy(),
                     out.tau.cpu().numpy(), out.pmax.cpu().numpy(), pr.plan)
        ora, rows, reqs = P.run_oracle(w)
        P.compare(w, g, ora, rows, reqs, w.name)
        ref.append((out.conf.clone(), out.argmax.clone(), out.exit.clone()))
    K = 48
    probes = [B.Probe(n_alloc, d, V, R, debug_outputs=False, mode=B.MODE_FLEX) for _ in range(K)]
    for p in probes[1:]:
        p.workspace = probes[0].workspace
        p._handles = probes[0]._handles
    rng = np.random.default_rng(5)
    for rnd in range(10):
        order = rng.integers(0, len(ws), size=K)
        for p in probes:
            p.conf.fill_(-7.0); p.argmax.fill_(-7); p.exit.fill_(7)
        torch.cuda.synchronize()
        for k, p in enumerate(probes):
            dv = devs[order[k]]
            p(dv["hidden"], devs[0]["W"], dv["off"], dv["load"], tp)
        torch.cuda.synchronize()
        for k, p in enumerate(probes):
            c, a, e = ref[order[k]]
            nv = ws[order[k]].N_valid
            assert torch.equal(p.conf, c) and torch.equal(p.exit, e), (rnd, k, int(order[k]))
            assert torch.equal(p.argmax, a), (rnd, k, int(order[k]), nv)


@pytest.mark.parametrize("n_valid", [1, 13, 16, 17, 29, 45, 64, 77, 96, 109, 125, 141, 157, 173, 192, 205, 221, 237, 253, 256,
                                     257, 300, 511, 513, 769, 1000, 1024])
def test_flex_every_chunk_height(P, force_mode, n_valid):
    """The flex kernel at every chunk height (16 ... 256 token rows: 16 hidden tensor maps, the 16-token
    last group of a chunk, one to four chunks) in one 1024-row allocation: n_valid rows in a single request
    plus empty ones, so that the decomposition comes from req_offsets[R] alone."""
    from paper_2606_31580_b200 import binding as B
    force_mode(3)
    V, d, n_alloc, R = 5000, 64, 1024, 3
    rng = np.random.default_rng(1000 + n_valid)
    W_bits = wl.make_W(V, d, 0.05, 4321)                       # one W for the whole sweep
    hb = np.zeros((n_alloc, d), np.uint16)
    hb[:n_valid] = wl.bf16_bits(rng.standard_normal((n_valid, d)).astype(np.float32) * 2.0)
    off = np.array([0, n_valid // 2, n_valid // 2, n_valid], np.int32)    # a request, an empty one, a request
    w = wl.Workload(f"flex-height-{n_valid}", W_bits, hb, off, rng.random(R).astype(np.float32))
    f = B.flex_query(n_alloc, d, V, R, n_valid)
    assert f["chunks"] * f["n_tok"] >= n_valid > (f["chunks"] - 1) * f["n_tok"] - 16 * f["chunks"]
    st = P.check(w)
    assert st["plan"]["flex"] == 1 and st["rows"] == n_valid
    print(w.name, f["chunks"], f["n_tok"], f["splits"], {k: v for k, v in st.items() if k != "plan"})

