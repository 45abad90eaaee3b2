"""GPU parity of the XPLOR-smoothed pair functor: V = V_lj S(r) with
r_on per type pair, through the C ABI (hb_set_ron_pair + hb_compute_lj(HB_XPLOR)), against the oracle's
orc_lj_pair_xplor sums on identical seeded snapshots, at the tolerances of tests/parity.py.  Needs a B200."""
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

CASES = {
    "lj_20k": wl.scaled(wl.CONFIGS["lj_64k"], 19_683),
    "ka_10k": wl.scaled(wl.CONFIGS["ka_1m"], 10_001),
    "table2_5k": wl.Workload("table2", 5000, 0.4, 1.0, 1, (1.0,), (1.0,), (2.5,), 0.4, 0.005, 0, 1, 0),
}


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _ron(w, frac=0.6):
    return [float(np.float32(frac * rc)) for rc in w.rcut]     # 1.5 sigma at r_cut = 2.5 sigma: the paper's test value


@pytest.mark.parametrize("case", ["lj_20k", "ka_10k"])
def test_xplor_forces_energy_virial(hb, orc, case):
    w = CASES[case]
    s = wl.make_state(w)
    ron = _ron(w)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.set_ron_pair(ron)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(hb.HB_XPLOR)
        f4, w6 = g.get_forces()
        th = g.thermo()
        # the shift modes still work after the smoothed one (the pair table is rebuilt per mode)
        g.compute_lj(hb.HB_SHIFT_ENERGY)
        f4s, w6s = g.get_forces()
    pos64 = s.pos.astype(np.float64)
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    p = orc.Params(w.ntypes, w.eps, w.sigma, w.rcut, 2, ron=ron)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=parity.BAND)
    assert A.max() < 1e-9          # V and F are continuous at r_cut: a cutoff flip changes nothing
    parity.assert_forces_close(F, U, W, A, f4, w6)
    parity.assert_energy_close(U.sum(), th["U"])
    ps = orc.Params(w.ntypes, w.eps, w.sigma, w.rcut, 1)
    Fs, Us, Ws, As = orc.compute_lj_nlist(pos64, s.type, s.L, ps, *lst, band=parity.BAND)
    parity.assert_forces_close(Fs, Us, Ws, As, f4s, w6s)
    assert np.abs(F - Fs).max() > 1e-3 * np.abs(F).max()      # and the two functors do differ


def test_xplor_ron_beyond_rcut_is_the_plain_truncated_potential(hb, orc):
    """reading x1: r_on >= r_cut leaves no switching interval."""
    w = CASES["lj_20k"]
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.set_ron_pair([3.0])
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(hb.HB_XPLOR)
        f4, w6 = g.get_forces()
        g.compute_lj(hb.HB_SHIFT_NONE)
        f4n, w6n = g.get_forces()
    assert np.array_equal(f4[:, :3], f4n[:, :3]) and np.allclose(f4[:, 3], f4n[:, 3], rtol=1e-6, atol=1e-7)
    pos64 = s.pos.astype(np.float64)
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    p = orc.Params(1, w.eps, w.sigma, w.rcut, 2, ron=[3.0])
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=parity.BAND)
    A0 = orc.compute_lj_nlist(pos64, s.type, s.L, orc.Params(1, w.eps, w.sigma, w.rcut, 0), *lst, band=parity.BAND)[3]
    parity.assert_forces_close(F, U, W, A0, f4, w6)


def test_xplor_two_particles_against_the_hand_worked_values(hb):
    """The CUDA path against tests/golden/xplor_closed_form.txt without the oracle in between."""
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", "xplor_closed_form.txt")) as f:
        for ln in f:
            if ln.strip() and not ln.startswith("#"):
                a = [int(x) for x in ln.split()]
                rows.append((Fraction(a[0], a[1]), Fraction(a[2], a[3]), Fraction(a[4], a[5])))
    L = float(np.float32(20.0))
    for r, S, dS in rows:
        if r >= Fraction(5, 2):
            continue
        Vlj = 4 * (1 / r ** 12 - 1 / r ** 6)
        Flj = (48 / r ** 12 - 24 / r ** 6) / r
        V, F = float(Vlj * S), float(Flj * S - Vlj * dS)
        pos = np.array([[0.25, -0.5, 1.0], [0.25 + float(r), -0.5, 1.0]], dtype=np.float32)
        with hb.System(2, L, 1, [1.0], [1.0]) as g:
            g.set_state(pos, np.zeros(2, dtype=np.int32), np.zeros_like(pos))
            g.set_ron_pair([1.5])
            g.build_nlist(2.5, 0.4)
            g.compute_lj(hb.HB_XPLOR)
            f4, w6 = g.get_forces()
        assert float(f4[1, 0]) == pytest.approx(F, rel=2e-5, abs=2e-6)       # force on the right particle along +x
        assert float(f4[0, 0]) == pytest.approx(-F, rel=2e-5, abs=2e-6)
        assert 2.0 * float(f4[0, 3]) == pytest.approx(V, rel=2e-5, abs=2e-7)


@pytest.mark.parametrize("mode", ["step", "run"])
def test_xplor_trajectory_and_conservation(hb, orc, mode):
    """Table 2's system (N = 5000, rho = 0.4, r_cut = 2.5, r_on = 1.5, dt = 0.005) through hb_step_nve / the fused
    kernels of hb_run_nve: 10 steps against the oracle's trajectory (<= 1e-5 absolute, as for config 1), then
    400 more: the total energy stays where the oracle's stays, and forces agree stage-wise on the reached state."""
    w = CASES["table2_5k"]
    s = wl.make_state(w)
    p = orc.Params(1, w.eps, w.sigma, w.rcut, 2, ron=[1.5])
    ref = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 10, log=True)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.set_ron_pair([1.5])
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(hb.HB_XPLOR)
        E0 = g.thermo()
        if mode == "step":
            for _ in range(10):
                g.step_nve(w.dt)
        else:
            g.run_nve(w.dt, 10, 0)
        out = g.get_state()
        th = g.thermo()
        g.run_nve(w.dt, 400, 0)
        out2 = g.get_state()
        f4, w6 = g.get_forces()
        th2 = g.thermo()
    d = out["pos"].astype(np.float64) + out["image"] * s.L - (ref["pos"] + ref["image"] * s.L)
    assert np.abs(d).max() <= 1e-5
    assert th["K"] + th["U"] == pytest.approx(ref["KU"][-1].sum(), rel=2e-5)
    assert E0["K"] + E0["U"] == pytest.approx(ref["KU"][0].sum(), rel=1e-6)
    long = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 410, log=True)
    assert th2["K"] + th2["U"] == pytest.approx(long["KU"][-1].sum(), abs=2e-5 * long["KU"][-1, 0])
    pos_g = out2["pos"].astype(np.float64)
    lst = orc.nlist_cells(pos_g, s.L, w.r_max)
    F, U, W, A = orc.compute_lj_nlist(pos_g, s.type, s.L, p, *lst, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6)
    parity.assert_energy_close(U.sum(), th2["U"])
