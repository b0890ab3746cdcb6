"""Pins of the fp64 oracle (steps 1-3 and 5) against what the mathematics fixes — DESIGN.md §5 P1-P4,
P8, P10-P14.  None of these re-types the oracle's formula or re-calls its routine: they use closed
forms, invariants, brute force in a different formulation, a library routine, and the statistical
closed forms of the synthetic generator.  CPU only."""
import math

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle
from paper_2606_31580_b200 import workloads as wl


def _probe(h, W, off, load, p):
    return oracle.probe(np.asarray(h, np.float32), np.asarray(W, np.float32), off, load, p)


# ------------------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("V,d", [(1000, 64), (7, 8), (1, 8), (4099, 24)])
def test_P1_uniform_logits(V, d, tau_norm):
    """hidden = 0 => every logit 0 => pmax = 1/V exactly, argmax 0 (tie -> lowest index), C = 1/V."""
    rng = np.random.default_rng(1)
    W = rng.standard_normal((V, d)).astype(np.float32)
    r = _probe(np.zeros((6, d)), W, [0, 2, 6], [0.1, 0.9], tau_norm)
    assert np.all(r.argmax == 0)
    np.testing.assert_allclose(r.pmax, 1.0 / V, rtol=0, atol=1e-15)
    np.testing.assert_allclose(r.conf, 1.0 / V, rtol=1e-15)
    if V > 1:
        assert np.all(r.gap2 == 0.0)
    # W = 0 instead of hidden = 0
    r = _probe(rng.standard_normal((3, d)), np.zeros((V, d)), [0, 3], [0.5], tau_norm)
    assert np.all(r.argmax == 0) and np.allclose(r.pmax, 1.0 / V, rtol=1e-15)


# ------------------------------------------------------------------------------------------ P2
@pytest.mark.parametrize("M", [0.0, 1.0, 5.0, 40.0])
def test_P2_scaled_identity(M, tau_norm):
    """V = d, W = M*I, hidden = e_j  =>  pmax = 1 / (1 + (V-1) e^{-M}), argmax = j.
    M = 40 is BASELINE.json's 'one-hot hidden states give confidence 1'."""
    V = 64
    W = (M * np.eye(V)).astype(np.float32)
    js = np.array([0, 5, 63, 17])
    h = np.eye(V, dtype=np.float32)[js]
    r = _probe(h, W, [0, 4], [0.5], tau_norm)
    expect = 1.0 / (1.0 + (V - 1) * math.exp(-M))
    np.testing.assert_allclose(r.pmax, expect, rtol=1e-14)
    np.testing.assert_allclose(r.conf, expect, rtol=1e-14)
    if M > 0:
        assert np.array_equal(r.argmax, js)
        np.testing.assert_allclose(r.gap2, M, rtol=1e-15)
    else:
        assert np.all(r.argmax == 0)
    if M == 40.0:
        assert abs(r.conf[0] - 1.0) < 1e-14 and r.exit[0] == 1


# ------------------------------------------------------------------------------------------ P3
def test_P3_ties_lowest_index():
    rng = np.random.default_rng(3)
    V, d = 300, 16
    W = (rng.standard_normal((V, d)) * 0.1).astype(np.float32)
    h = rng.standard_normal((1, d)).astype(np.float32)
    base = oracle.row_stats(h, W, want_logits=True)
    # plant a row that wins, and an exact duplicate of it further on (also across index 128/256)
    big = (h[0] * 2.0).astype(np.float32)
    for v1, v2 in [(5, 200), (127, 128), (100, 256), (0, 299)]:
        W2 = W.copy(); W2[v1] = big; W2[v2] = big
        r = oracle.row_stats(h, W2, want_logits=True)
        assert r["a"][0] == v1
        assert r["gap2"][0] == 0.0
        lg = r["logits"][0]
        assert lg[v1] == lg[v2] == lg.max()
        rest = np.exp(np.delete(lg, [v1, v2]) - lg[v1]).sum()
        np.testing.assert_allclose(r["pmax"][0], 1.0 / (2.0 + rest), rtol=1e-13)
    assert base["gap2"][0] > 0


# ------------------------------------------------------------------------------------------ P4
def test_P4_shift_and_permutation_invariance():
    rng = np.random.default_rng(4)
    V, d, N = 513, 32, 5
    # values on a coarse grid so that W + u is exact in float32
    W = (rng.integers(-64, 64, (V, d)) / 64.0).astype(np.float32)
    h = (rng.integers(-32, 32, (N, d)) / 8.0).astype(np.float32)
    u = (rng.integers(-64, 64, d) / 64.0).astype(np.float32)
    r0 = oracle.row_stats(h, W)
    r1 = oracle.row_stats(h, W + u[None, :])
    np.testing.assert_allclose(r1["pmax"], r0["pmax"], rtol=1e-12)
    keep = r0["gap2"] > 1e-9
    assert np.array_equal(r1["a"][keep], r0["a"][keep])
    np.testing.assert_allclose(r1["m"] - r0["m"], h.astype(np.float64) @ u.astype(np.float64), atol=1e-12)
    perm = rng.permutation(V)
    r2 = oracle.row_stats(h, W[perm])
    np.testing.assert_allclose(r2["pmax"], r0["pmax"], rtol=1e-12)
    assert np.array_equal(perm[r2["a"]][keep], r0["a"][keep])
    assert np.all(r0["pmax"] >= 1.0 / V) and np.all(r0["pmax"] <= 1.0)


@settings(max_examples=40, deadline=None)
@given(st.integers(1, 400), st.lists(st.integers(1, 399), max_size=6), st.integers(0, 2 ** 31 - 1))
def test_P4_merge_associativity(V, cuts, seed):
    """Split V at arbitrary points, take the definition on each chunk, fold with (+): identical to
    the single pass (argmax exactly, S to rounding), whatever the chunking."""
    rng = np.random.default_rng(seed)
    d = 8
    W = (rng.integers(-8, 9, (V, d)) / 4.0).astype(np.float32)     # coarse grid -> real ties occur
    h = (rng.integers(-8, 9, (1, d)) / 4.0).astype(np.float32)
    full = oracle.row_stats(h, W)
    bounds = sorted({0, V, *[c for c in cuts if c < V]})
    acc = (-math.inf, -1, 0.0)
    for v0, v1 in zip(bounds[:-1], bounds[1:]):
        acc = oracle.merge(acc, oracle.row_stats_range(h[0], W, v0, v1))
    assert acc[1] == full["a"][0]
    assert acc[0] == full["m"][0]
    np.testing.assert_allclose(acc[2], full["S"][0], rtol=1e-13)


def test_P4_merge_chunk_sizes_1_7_128():
    rng = np.random.default_rng(44)
    V, d = 1000, 64
    W = (rng.standard_normal((V, d)) * 0.05).astype(np.float32)
    h = rng.standard_normal((1, d)).astype(np.float32)
    full = oracle.row_stats(h, W)
    for cs in (1, 7, 128, V):
        acc = (-math.inf, -1, 0.0)
        for v0 in range(0, V, cs):
            acc = oracle.merge(acc, oracle.row_stats_range(h[0], W, v0, min(V, v0 + cs)))
        assert acc[1] == full["a"][0] and acc[0] == full["m"][0]
        np.testing.assert_allclose(acc[2], full["S"][0], rtol=1e-13)


# ------------------------------------------------------------------------------------------ P8
def test_P8_exit_is_strict(tau_norm):
    """conf == tau => no exit; one ulp above => exit.  beta = 0 makes tau = lambda_base (P9); V = d,
    W = M*I, one-row requests give conf = 1/(1+(V-1)e^-M) which we read back and use as lambda_base."""
    V = 16
    W = (3.0 * np.eye(V)).astype(np.float32)
    h = np.eye(V, dtype=np.float32)[[2]]
    c = oracle.row_stats(h, W)["pmax"][0]
    for lam, want in [(c, 0), (np.nextafter(c, 0.0), 1), (np.nextafter(c, 1.0), 0)]:
        p = oracle.TauParams(lambda_base=float(lam), beta=0.0, lambda_min=0.0, lambda_max=1.0, l_target=0.5)
        r = _probe(h, W, [0, 1], [0.3], p)
        assert r.tau[0] == lam and r.conf[0] == c
        assert r.exit[0] == want
    ex, mg = oracle.exit_mask([0.5, np.nan, 0.96], [0.5, 0.1, 0.95])
    assert list(ex) == [0, 0, 1]


# ------------------------------------------------------------------------------------------ P10
def test_P10_bruteforce_tiny_pipeline(tau_norm):
    """Whole pipeline against a deliberately different formulation: exact rational dot products,
    the full probability vector exp(l)/sum(exp(l)) in long double WITHOUT max subtraction."""
    from fractions import Fraction
    rng = np.random.default_rng(10)
    for trial in range(5):
        d, V, R = int(rng.integers(1, 9)), int(rng.integers(2, 17)), int(rng.integers(1, 4))
        lens = rng.integers(0, 4, R)
        off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        N = int(off[-1]) + 2                       # two padding rows
        W = (rng.integers(-16, 17, (V, d)) / 8.0).astype(np.float32)
        h = (rng.integers(-16, 17, (N, d)) / 8.0).astype(np.float32)
        load = rng.random(R).astype(np.float32)
        r = _probe(h, W, off, load, tau_norm)
        for n in range(int(off[-1])):
            lg = [sum(Fraction(float(h[n, k])) * Fraction(float(W[v, k])) for k in range(d)) for v in range(V)]
            e = np.array([np.exp(np.longdouble(float(x))) for x in lg], dtype=np.longdouble)
            prob = e / e.sum()
            assert r.argmax[n] == min(v for v in range(V) if lg[v] == max(lg))
            assert abs(float(prob.max()) - r.pmax[n]) < 1e-14
        assert np.all(r.argmax[int(off[-1]):] == -1)
        for q in range(R):
            rows = r.pmax[off[q]:off[q + 1]]
            want = float(np.sum(rows.astype(np.longdouble)) / len(rows)) if len(rows) else 0.0
            assert abs(r.conf[q] - want) < 1e-15
            assert r.exit[q] == (1 if want > r.tau[q] else 0) or abs(want - r.tau[q]) < 1e-14


# ------------------------------------------------------------------------------------------ P11
def test_P11_library_crosscheck_c1(tau_norm):
    import torch
    w = wl.config_c1()
    r = oracle.row_stats(w.hidden_f32(), w.W_f32())
    lg = torch.from_numpy(w.hidden_f32()).double() @ torch.from_numpy(w.W_f32()).double().T
    pm, am = torch.softmax(lg, -1).max(-1)
    np.testing.assert_allclose(r["pmax"], pm.numpy(), rtol=1e-12, atol=1e-15)
    keep = r["gap2"] > 1e-9
    assert np.array_equal(r["a"][keep], am.numpy()[keep])


def test_P11_library_crosscheck_c2_slice(c2_W_bits):
    import torch
    w = wl.config_c2(c2_W_bits)
    h = w.hidden_f32()[:8]
    r = oracle.row_stats(h, w.W_f32())
    lg = torch.from_numpy(h).double() @ torch.from_numpy(w.W_f32()).double().T
    pm, am = torch.softmax(lg, -1).max(-1)
    np.testing.assert_allclose(r["pmax"], pm.numpy(), rtol=1e-11, atol=1e-15)
    assert np.array_equal(r["a"], am.numpy())


# ------------------------------------------------------------------------------------------ P12
def test_P12_segmented_mean():
    pm = np.array([0.25, 0.5, 1.0, 0.125, 0.75, 0.3])
    off = np.array([0, 0, 1, 3, 3, 6], np.int32)     # len 0, 1, 2, 0, 3
    c = oracle.aggregate(pm, off)
    assert c[0] == 0.0 and c[3] == 0.0
    assert c[1] == pm[0]                             # single-row request: bit-for-bit
    assert c[2] == 0.75
    np.testing.assert_allclose(c[4], (0.125 + 0.75 + 0.3) / 3, rtol=1e-15)
    # (v) conf lies within [min, max] of its rows
    rng = np.random.default_rng(12)
    pm = rng.random(200); off = np.concatenate([[0], np.cumsum(rng.integers(1, 9, 30))]).astype(np.int32)
    c = oracle.aggregate(pm, off)
    for q in range(30):
        seg = pm[off[q]:off[q + 1]]
        assert seg.min() - 1e-15 <= c[q] <= seg.max() + 1e-15
    # NEXT-1 aggregates: geometric mean and min
    g = oracle.aggregate(np.array([0.5, 0.125, 1.0, 1.0]), np.array([0, 2, 4], np.int32), mode=1)
    np.testing.assert_allclose(g, [0.25, 1.0], rtol=1e-15)
    mn = oracle.aggregate(np.array([0.5, 0.125, 1.0, 0.9]), np.array([0, 2, 4], np.int32), mode=2)
    assert list(mn) == [0.125, 0.9]


# ------------------------------------------------------------------------------------------ P13
def test_P13_full_vocab_logsumexp_lln(c2_W_bits):
    """Flat rows at the REAL vocabulary size: m - ln(pmax) = ln sum_v e^{l_v} ~ ln V + d sigma^2 / 2
    (law of large numbers; hidden RMS-normalised so |h|^2 = d).  Catches dropped tail tiles / wrong
    v ranges that tiny cases cannot."""
    V, d = c2_W_bits.shape
    rng = np.random.default_rng(13)
    hb, _ = wl.polarised_hidden(c2_W_bits, 48, rng, q=0.0, c_lo=4, c_hi=10, kap=0.0)
    r = oracle.row_stats(wl.bits_to_f32(hb), wl.bits_to_f32(c2_W_bits))
    lse = r["m"] - np.log(r["pmax"])
    predicted = math.log(V) + d * 0.02 ** 2 / 2
    assert abs(lse.mean() - predicted) < 0.01, (lse.mean(), predicted)
    assert np.all(np.abs(lse - predicted) < 0.05)


# ------------------------------------------------------------------------------------------ P14
def test_P14_targeted_rows_real_vocab(c2_W_bits, tau_norm):
    """S1 generator: rows planted so that the analytically PREDICTED pmax is p*.  The oracle must land
    on p* (median error ~3e-4, max ~3e-3 per DESIGN §4) and on the planted token."""
    s1 = wl.tau_band_stress(c2_W_bits, 0.02, R=24, L=8)
    r = oracle.probe(s1.hidden_f32(), s1.W_f32(), s1.req_offsets, s1.load, tau_norm)
    err = np.abs(r.pmax - s1.target_pmax)
    assert np.median(err) < 8e-4 and err.max() < 5e-3, (np.median(err), err.max())
    assert np.array_equal(r.argmax, s1.planted)
    # the set does what it is for: both exit outcomes occur
    assert 0 < r.exit.sum() < s1.R


def test_nan_rows_poison_conf_not_exit(tau_norm):
    """DESIGN A12: NaN in a request's rows -> conf NaN, exit 0; other requests untouched."""
    rng = np.random.default_rng(99)
    W = (rng.standard_normal((50, 8))).astype(np.float32)
    h = rng.standard_normal((4, 8)).astype(np.float32)
    h[1, 3] = np.nan
    r = _probe(h, W, [0, 2, 4], [0.5, 0.5], tau_norm)
    assert np.isnan(r.conf[0]) and r.exit[0] == 0 and np.isfinite(r.conf[1])


# ------------------------------------------------------------------------------------------ P15
# Probability of a GIVEN token (DESIGN A2 alternative, NEXT-1): oracle.token_prob.
@pytest.mark.parametrize("M", [0.0, 1.0, 5.0, 40.0])
def test_P15_token_prob_scaled_identity(M):
    """W = M*I, hidden = e_j: the planted token has 1/(1+(V-1)e^-M), any other e^-M/(1+(V-1)e^-M)."""
    V = 48
    W = (M * np.eye(V)).astype(np.float32)
    js = np.array([0, 5, 47, 17])
    h = np.eye(V, dtype=np.float32)[js]
    den = 1.0 + (V - 1) * math.exp(-M)
    np.testing.assert_allclose(oracle.token_prob(h, W, js), 1.0 / den, rtol=1e-14)
    others = (js + 3) % V
    np.testing.assert_allclose(oracle.token_prob(h, W, others), math.exp(-M) / den, rtol=1e-14)


def test_P15_token_prob_is_a_distribution_and_matches_library():
    """Sum over every token of a row's probabilities is 1 (brute force over the whole vocabulary);
    the entries equal torch.softmax's; the argmax token's probability is step 2's pmax bit for bit;
    a token outside the vocabulary has probability 0."""
    import torch
    rng = np.random.default_rng(15)
    V, d = 257, 24
    W = wl.bits_to_f32(wl.bf16_bits(rng.standard_normal((V, d)) * 0.7))
    h1 = wl.bits_to_f32(wl.bf16_bits(rng.standard_normal((1, d)) * 1.5))
    h = np.repeat(h1, V, axis=0)
    p = oracle.token_prob(h, W, np.arange(V))
    assert abs(p.sum() - 1.0) < 1e-13 and np.all(p > 0)
    ref = torch.softmax(torch.from_numpy(h1).double() @ torch.from_numpy(W).double().T, -1)[0].numpy()
    np.testing.assert_allclose(p, ref, rtol=1e-12)
    rs = oracle.row_stats(h1, W)
    assert oracle.token_prob(h1, W, rs["a"])[0] == rs["pmax"][0]
    assert np.all(oracle.token_prob(np.repeat(h1, 3, axis=0), W, [-1, V, 2**31 - 1]) == 0.0)
    # uniform logits: every token has 1/V
    np.testing.assert_allclose(oracle.token_prob(np.zeros((4, d), np.float32), W, [0, 1, 100, 256]), 1.0 / V,
                               rtol=1e-15)
