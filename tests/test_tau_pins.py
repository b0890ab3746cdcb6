"""Pins of the oracle's threshold (step 4: Eq. 5 + clamp) and of the NEXT-2 control-plane helpers
(EMA, budget Eq. 6-8) — DESIGN.md §5 P5-P7, P9.  The expected values come from tests/golden/
tau_closed_form.txt (Eq. 5 evaluated by hand from tabulated tanh) and from a tanh written as
expm1(2x)/(expm1(2x)+2), not from the oracle.  CPU only."""
import math
from pathlib import Path

import numpy as np
import pytest

import oracle

GOLD = Path(__file__).parent / "golden" / "tau_closed_form.txt"


def _tanh_alt(x):
    e = math.expm1(2.0 * x)
    return e / (e + 2.0)


def _rows():
    out = []
    for line in GOLD.read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            out.append(tuple(float(t) for t in line.split()))
    return out


def test_P5_closed_form_paper_units(tau_defaults):
    rows = _rows()
    assert len(rows) == 7
    for L, unclamped, clamped in rows:
        assert abs(oracle.tau_unclamped(L, tau_defaults) - unclamped) < 5e-15
        assert abs(oracle.tau_scalar(L, tau_defaults) - clamped) < 5e-15
    assert oracle.tau_scalar(10.0, tau_defaults) == 0.95          # exactly: tanh(0) = 0
    assert abs(oracle.tau_scalar(1e9, tau_defaults) - 0.91) < 1e-12   # L -> inf: lambda_base - beta


def test_P6_normalised_units_and_scale_invariance(tau_norm, tau_defaults):
    assert oracle.tau_scalar(0.5, tau_norm) == 0.95
    assert abs(oracle.tau_scalar(1.0, tau_norm) - 0.919536233761769) < 5e-15
    assert oracle.tau_scalar(0.2, tau_norm) == 0.97               # unclamped 0.97148 -> clamp
    assert abs(oracle.tau_unclamped(0.2, tau_norm) - (0.95 - 0.04 * _tanh_alt(-0.6))) < 5e-15
    assert abs(oracle.tau_scalar(0.9, tau_norm) - (0.95 - 0.04 * _tanh_alt(0.8))) < 5e-15
    # tau(load, L_t) = tau(c*load, c*L_t): only the ratio enters Eq. 5
    for load in np.linspace(0, 3, 31):
        a = oracle.tau_scalar(load * 0.5, tau_norm)
        b = oracle.tau_scalar(load * 10.0, tau_defaults)
        assert abs(a - b) < 1e-14
    # the upper clamp binds exactly below L = L_t * (1 - atanh(0.5))   (DESIGN A8)
    Lc = 10.0 * (1.0 - math.atanh(0.5))
    assert abs(Lc - 4.50694) < 1e-5
    assert oracle.tau_scalar(Lc - 1e-6, tau_defaults) == 0.97
    assert oracle.tau_scalar(Lc + 1e-6, tau_defaults) < 0.97


@pytest.mark.parametrize("beta", [0.02, 0.03, 0.04, 0.05, 0.06, 0.1])
@pytest.mark.parametrize("l_t", [5.0, 8.0, 10.0, 15.0, 20.0])
@pytest.mark.parametrize("gamma", [0.5, 1.0, 2.0])
def test_P7_monotone_and_in_range(beta, l_t, gamma):
    """threshold decreases when load > target, increases when below; always inside
    [lambda_min, lambda_max] (Eq. 4).  Grid = Table 3's swept ranges
    plus beta = 0.1, which is the only way to reach the lower clamp (DESIGN A8)."""
    p = oracle.TauParams(beta=beta, l_target=l_t, gamma=gamma)
    loads = np.linspace(0.0, 8.0 * l_t, 801).astype(np.float32)
    t = oracle.tau(loads, p)
    assert np.all(np.diff(t) <= 0.0)
    assert np.all(t >= p.lambda_min) and np.all(t <= p.lambda_max)
    un = np.array([oracle.tau_unclamped(float(x), p) for x in loads])
    expect = np.array([0.95 - beta * _tanh_alt(gamma * (float(x) - l_t) / l_t) for x in loads])
    np.testing.assert_allclose(un, expect, rtol=0, atol=1e-15)
    assert np.all(un[loads > l_t] < 0.95) and np.all(un[loads < l_t] > 0.95)
    assert np.all(np.abs(un - 0.95) < beta)                        # tanh bounded in (-1, 1)
    if beta == 0.1:
        assert t.min() == 0.88 and un.min() < 0.88                 # lower clamp binds
    if beta == 0.02:
        assert np.array_equal(t, np.clip(un, 0.88, 0.97)) and t.max() < 0.97   # no clamp ever


def test_P9_fixed_threshold_special_case():
    """beta = 0 => tau = clamp(lambda_base) for every load: the Fixed-High (0.95) and Fixed-Low
    (0.90) baselines."""
    loads = np.linspace(0, 50, 101).astype(np.float32)
    for lam in (0.95, 0.90):
        t = oracle.tau(loads, oracle.TauParams(lambda_base=lam, beta=0.0))
        assert np.all(t == lam)
    assert np.all(oracle.tau(loads, oracle.TauParams(lambda_base=0.99, beta=0.0)) == 0.97)
    assert np.all(oracle.tau(loads, oracle.TauParams(lambda_base=0.5, beta=0.0)) == 0.88)


# ------------------------------------------------------------------------------------ NEXT-2 helpers
def test_ema_closed_form():
    """Lbar(t) = alpha L + (1-alpha) Lbar(t-1), Lbar(0) = 0.  Constant input L:
    Lbar(t) = L (1 - (1-alpha)^t)."""
    out = oracle.ema(np.full(20, 7.0), alpha=0.3)
    want = 7.0 * (1.0 - 0.7 ** np.arange(1, 21))
    np.testing.assert_allclose(out, want, rtol=1e-14)
    imp = oracle.ema([1.0] + [0.0] * 5, alpha=0.5)                 # impulse response alpha(1-alpha)^t
    np.testing.assert_allclose(imp, 0.5 * 0.5 ** np.arange(6), rtol=1e-15)


def test_budget_eq6_to_8_pins():
    q = oracle.BudgetParams()
    assert oracle.f_diff(50, q) == 0.6 and oracle.f_diff(275, q) == 1.5       # end points of Eq. 7
    assert oracle.f_diff(10, q) == 0.6 and oracle.f_diff(1000, q) == 1.5      # clip
    assert abs(oracle.f_diff(162.5, q) - 1.05) < 1e-15                        # midpoint
    assert oracle.f_load(0, q) == 1.0 and oracle.f_load(10, q) == 1.0         # L <= L_target
    assert oracle.f_load(20, q) == 0.5 and oracle.f_load(0.5, q) == 1.0       # max(1, L)
    B = oracle.budget([50, 275, 275, 162.5, 50, 275], [0, 0, 20, 30, 100, 1000], q)
    #   floor(10*.6*1)=6, floor(10*1.5)=15, floor(15*.5)=7, floor(10*1.05/3)=3, max(2, floor(.6))=2, 2
    assert list(B) == [6, 15, 7, 3, 2, 2]


def test_budget_floor_is_that_of_the_exact_product():
    """Eq. 6 floors a real-number product.  Exact rational arithmetic (a different
    formulation from the oracle's doubles) over the whole grid |p| < 600, L <= 60 with the paper's
    defaults: the oracle must agree everywhere, in particular at the points where
    the exact product IS an integer and binary evaluation lands one ulp below it (DESIGN A19)."""
    from fractions import Fraction as Fr
    q = oracle.BudgetParams()
    f_min, f_max, p_min, p_max, b_base, b_min, l_t = Fr(3, 5), Fr(3, 2), 50, 275, 10, 2, 10
    ps, Ls = np.meshgrid(np.arange(1, 600), np.arange(0, 61), indexing="ij")
    got = oracle.budget(ps.ravel().astype(np.float64), Ls.ravel().astype(np.float64), q)
    want = []
    for p_, L_ in zip(ps.ravel().tolist(), Ls.ravel().tolist()):
        fd = min(max(f_min + Fr(p_ - p_min, p_max - p_min) * (f_max - f_min), f_min), f_max)
        fl = min(Fr(1), Fr(l_t, max(1, L_)))
        want.append(max(b_min, (b_base * fd * fl).__floor__()))
    want = np.asarray(want)
    assert np.array_equal(got, want), np.flatnonzero(got != want)[:10]
    # the two interior exact-integer points named in the review of round 1
    assert list(oracle.budget([100.0, 65.0], [5.0, 11.0], q)) == [8, 6]
