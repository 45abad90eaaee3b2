"""Pins of the oracle's other pair potentials (reading f1: Gaussian, Yukawa, Morse in their
textbook forms through the V(r), -(1/r) dV/dr functor of PAPER.md:284, with the cutoff treatments of PAPER.md:105,
314, 355-367) to closed forms, finite differences and an independent numpy pair sum.  CPU only."""
import math

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl

POTS = {"gauss": (2.0, 0.9, 0.0), "yukawa": (3.0, 1.7, 0.0), "morse": (1.5, 2.2, 1.1), "lj": (1.0, 1.0, 0.0)}


def test_closed_forms(orc):
    """Values that can be read off the formulas: Gaussian at r = sigma, Yukawa at r = 1/kappa, Morse at its minimum
    r0 (depth -D0, zero force) and at r0 + ln 2 / a (V = -3/4 D0, F = -a D0 / 2)."""
    e = math.e
    V, f = orc.pair_generic("gauss", 0.9, 2.0, 0.9, 0, 9, 9, 0)
    assert V == pytest.approx(2.0 / math.sqrt(e), rel=1e-14) and f * 0.9 == pytest.approx(V / 0.9, rel=1e-14)
    V, f = orc.pair_generic("yukawa", 1 / 1.7, 3.0, 1.7, 0, 9, 9, 0)
    assert V == pytest.approx(3.0 * 1.7 / e, rel=1e-14) and f / 1.7 == pytest.approx(2 * 1.7 * V, rel=1e-14)
    V, f = orc.pair_generic("morse", 1.1, 1.5, 2.2, 1.1, 9, 9, 0)
    assert V == pytest.approx(-1.5, rel=1e-15) and abs(f) < 1e-15
    r = 1.1 + math.log(2) / 2.2
    V, f = orc.pair_generic("morse", r, 1.5, 2.2, 1.1, 9, 9, 0)
    assert V == pytest.approx(-0.75 * 1.5, rel=1e-13) and f * r == pytest.approx(-2.2 * 1.5 / 2, rel=1e-13)
    assert orc.pair_generic("lj", 1.5, 1, 1, 0, 9, 9, 0) == orc.lj_pair(1.5, 1, 1, 9, 0)


@pytest.mark.parametrize("pot", list(POTS))
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_force_is_minus_gradient_and_cutoff_treatments(orc, pot, mode):
    eps, sig, p2 = POTS[pot]
    rc, ron = 2.5, 1.6
    h = 1e-6
    for r in np.concatenate([np.linspace(0.8, rc - 1e-3, 70), [ron - 3e-7, ron, ron + 3e-7]]):
        Vp, _ = orc.pair_generic(pot, r + h, eps, sig, p2, rc, ron, mode)
        Vm, _ = orc.pair_generic(pot, r - h, eps, sig, p2, rc, ron, mode)
        _, f = orc.pair_generic(pot, r, eps, sig, p2, rc, ron, mode)
        assert f * r == pytest.approx(-(Vp - Vm) / (2 * h), rel=3e-6, abs=3e-8)
    V0, f0 = orc.pair_generic(pot, 1.3, eps, sig, p2, rc, ron, 0)
    Vc, fc = orc.pair_generic(pot, rc - 1e-9, eps, sig, p2, rc, ron, mode)
    assert orc.pair_generic(pot, rc, eps, sig, p2, rc, ron, mode) == (0.0, 0.0)
    if mode == 1:
        V1, f1 = orc.pair_generic(pot, 1.3, eps, sig, p2, rc, ron, 1)
        assert f1 == f0 and abs(Vc) < 1e-8 and V1 == pytest.approx(V0 - orc.pair_generic(pot, rc - 1e-12, eps, sig, p2, rc, ron, 0)[0], rel=1e-9)
    if mode == 2:
        assert orc.pair_generic(pot, 1.3, eps, sig, p2, rc, ron, 2) == (V0, f0)      # below r_on
        assert abs(Vc) < 1e-15 and abs(fc) < 1e-7


def _pair_sum_numpy(pos, typ, L, p, pot):
    N = len(pos)
    i, j = np.triu_indices(N, 1)
    d = pos[i] - pos[j]
    d -= L * np.round(d / L)
    r = np.sqrt((d * d).sum(1))
    k = typ[i] * p.ntypes + typ[j]
    e, s, q, rc = p.eps[k], p.sigma[k], p.p2[k], p.rcut[k]
    v = {"gauss": lambda x: e * np.exp(-x * x / (2 * s * s)), "yukawa": lambda x: e * np.exp(-s * x) / x,
         "morse": lambda x: e * (np.exp(-2 * s * (x - q)) - 2 * np.exp(-s * (x - q)))}[pot]
    return np.where(r < rc, v(r) - v(rc), 0.0).sum()


@pytest.mark.parametrize("pot", ["gauss", "yukawa", "morse"])
def test_force_sums_with_other_potentials(orc, pot):
    """Two types, per-pair tables, energy shift: list sums == brute force, Newton III, sum U_i == numpy pair sum,
    tr W == -dU/dlambda under uniform scaling."""
    w = wl.scaled(wl.CONFIGS["ka_1m"], 1200)
    s = wl.make_state(w)
    pos = s.pos.astype(np.float64)
    eps, sig = [1.0, 1.5, 1.5, 0.5], [1.0, 0.8, 0.8, 0.88]
    p2 = [1.1, 0.9, 0.9, 1.0]
    if pot == "yukawa":
        sig = [1.5, 2.0, 2.0, 1.2]
    if pot == "morse":
        sig = [2.0, 2.5, 2.5, 3.0]
    p = orc.Params(2, eps, sig, w.rcut, 1, pot=pot, p2=p2)
    Fb, Ub, Wb = orc.compute_lj_brute(pos, s.type, s.L, p)
    c, r, n = orc.nlist_cells(pos, s.L, w.r_max)
    Fl, Ul, Wl, _ = orc.compute_lj_nlist(pos, s.type, s.L, p, c, r, n)
    assert np.allclose(Fb, Fl, rtol=1e-12, atol=1e-12) and np.allclose(Ub, Ul, rtol=1e-12, atol=1e-13)
    assert np.linalg.norm(Fb.sum(0)) / np.abs(Fb).sum() < 1e-10
    assert Ub.sum() == pytest.approx(_pair_sum_numpy(pos, s.type, s.L, p, pot), rel=1e-11)
    h = 1e-6
    Up = orc.compute_lj_brute(pos * (1 + h), s.type, s.L * (1 + h), p)[1].sum()
    Um = orc.compute_lj_brute(pos * (1 - h), s.type, s.L * (1 - h), p)[1].sum()
    trW = Wb[:, 0].sum() + Wb[:, 3].sum() + Wb[:, 5].sum()
    assert trW == pytest.approx(-(Up - Um) / (2 * h), rel=5e-5)
    # and the LJ sums are what they were when the potential is switched back
    plj = orc.Params.of(w)
    assert np.array_equal(orc.compute_lj_brute(pos, s.type, s.L, plj)[0], orc.compute_lj_brute(pos, s.type, s.L, orc.Params.of(w))[0])
