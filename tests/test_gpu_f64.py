"""GPU parity of the binary64 variant (PAPER.md:125, 353, 373 and Table 2): the same neighbor
list, force sums and velocity Verlet in binary64 (tunable precision = 64).  Against the fp64 oracle the agreement is at
rounding level (1e-12), which checks the list handling and the functors far more sharply than the binary32 path can;
the conservation properties are the ones Table 2 reports for the double-precision builds.  Needs a B200."""
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


def _dp_system(hb, w, s, **tun):
    g = hb.System.from_workload(w)
    g.set_tunable("precision", 64)
    for k, v in tun.items():
        g.set_tunable(k, v)
    g.set_state(s.pos, s.type, s.vel, s.image)
    g.build_nlist(0.0, w.r_buff)
    return g


@pytest.mark.parametrize("case,mode", [("lj_20k", 1), ("lj_20k", 0), ("lj_20k", 2), ("ka_10k", 1), ("ka_10k", 2)])
def test_f64_forces_energy_virial(hb, orc, case, mode):
    w = CASES[case]
    s = wl.make_state(w)
    ron = [float(np.float32(0.6 * rc)) for rc in w.rcut]
    with _dp_system(hb, w, s) as g:
        g.set_ron_pair(ron)
        g.compute_lj(mode)
        f4, w6 = g.get_forces_f64()
        f4s, _ = g.get_forces()
        th = g.thermo()
    pos64 = s.pos.astype(np.float64)
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    p = orc.Params(w.ntypes, w.eps, w.sigma, w.rcut, mode, ron=ron)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=1e-12)
    Fmax = np.abs(F).max()
    assert (np.abs(f4[:, :3] - F).max(1) <= 1e-12 * Fmax + A[:, 0]).all()
    assert (np.abs(f4[:, 3] - U) <= 1e-12 * np.abs(U).max() + A[:, 1]).all()
    assert (np.abs(w6 - W).max(1) <= 1e-12 * np.abs(W).max() + A[:, 2]).all()
    assert th["U"] == pytest.approx(U.sum(), rel=1e-13, abs=A[:, 1].sum())
    assert np.allclose(th["W"], W.sum(0), rtol=0, atol=1e-12 * np.abs(W).sum())
    assert np.array_equal(f4s, f4.astype(np.float32))          # the binary32 accessor returns the same sums, rounded


@pytest.mark.parametrize("pot", ["gauss", "yukawa", "morse"])
def test_f64_functors(hb, orc, pot):
    e, sg, q = {"gauss": (2.0, 0.9, 0.0), "yukawa": (3.0, 1.7, 0.0), "morse": (1.5, 2.2, 1.1)}[pot]
    f32 = lambda x: float(np.float32(x))
    base = CASES["lj_20k"]
    w = wl.Workload(pot, base.N, base.rho, base.T, 1, (f32(e),), (f32(sg),), (2.5,), 0.4, 0.005, 0, 1, 0)
    s = wl.make_state(w)
    with _dp_system(hb, w, s) as g:
        g.set_pair_potential(pot, [f32(q)])
        g.compute_lj(1)
        f4, w6 = g.get_forces_f64()
    pos64 = s.pos.astype(np.float64)
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    p = orc.Params(1, w.eps, w.sigma, w.rcut, 1, pot=pot, p2=[f32(q)])
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=1e-12)
    assert np.abs(f4[:, :3] - F).max() <= 1e-12 * np.abs(F).max() + A[:, 0].max()
    assert np.abs(f4[:, 3] - U).max() <= 1e-12 * np.abs(U).max() + A[:, 1].max()


def test_f64_trajectory_matches_the_oracle(hb, orc):
    """Config 1, 10 steps: the binary32 path agrees with the oracle to 1e-5; this one to 1e-11 (both sides binary64,
    different order of summation).  A sort in between: the binary64 arrays live by tag."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    p = orc.Params.of(w)
    ref = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 10)
    with _dp_system(hb, w, s) as g:
        g.compute_lj(w.shift)
        g.run_nve(w.dt, 6, 0)
        g.sort()
        g.run_nve(w.dt, 3, 0)
        g.step_nve(w.dt)
        out = g.get_state_f64()
        out32 = g.get_state()
        th = g.thermo()
    assert np.abs(out["pos"] + out["image"] * s.L - (ref["pos"] + ref["image"] * s.L)).max() <= 1e-11
    assert np.abs(out["vel"] - ref["vel"]).max() <= 1e-11
    assert np.array_equal(out32["pos"], out["pos"].astype(np.float32)) and np.array_equal(out32["image"], out["image"])
    t = orc.thermo(ref["vel"], ref["U"], ref["W"], s.L)
    assert th["K"] == pytest.approx(t["K"], rel=1e-11) and th["U"] == pytest.approx(t["U"], rel=1e-11)
    assert th["P"] == pytest.approx(t["P"], rel=1e-10)


def test_f64_state_in_and_out(hb, orc):
    """hb_set_state_f64 keeps all 53 bits; in binary32 mode it rounds, and hb_get_state_f64 widens."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    pos = s.pos.astype(np.float64) + 1e-9 * wl.counter_uniform(5, 1, np.arange(3 * w.N)).reshape(-1, 3)
    vel = s.vel.astype(np.float64) * (1 + 1e-10)
    with hb.System.from_workload(w) as g:
        g.set_tunable("precision", 64)
        g.set_state_f64(pos, s.type, vel, s.image)
        o = g.get_state_f64()
        assert np.array_equal(o["pos"], pos) and np.array_equal(o["vel"], vel) and np.array_equal(o["image"], s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        f4, _ = g.get_forces_f64()
        lst = orc.nlist_cells(pos, s.L, w.r_max)
        F, U, W, A = orc.compute_lj_nlist(pos, s.type, s.L, orc.Params.of(w), *lst, band=1e-12)
        assert np.abs(f4[:, :3] - F).max() <= 1e-12 * np.abs(F).max() + A[:, 0].max()
        g.set_tunable("precision", 32)
        g.set_state_f64(pos, s.type, vel, s.image)
        o = g.get_state_f64()
        assert np.array_equal(o["pos"], pos.astype(np.float32).astype(np.float64))
        with pytest.raises(hb.HBError):
            g.get_forces_f64()
        bad = pos.copy()
        bad[3, 1] = s.L
        with pytest.raises(hb.HBError) as e:
            g.set_state_f64(bad, s.type, vel, s.image)
        assert e.value.code == hb.HB_ENAN


def test_f64_conservation_against_f32(hb):
    """PAPER.md Table 2 (N = 5000, rho = 0.4, r_cut = 2.5, XPLOR, dt = 0.005): the double-precision build conserves
    momentum to round-off (1e-19 per particle against 1e-10) and drifts less in energy.  Same start, same list, 1500 steps
    each: the binary64 momentum per particle moves by less than 1e-15 (the start carries the 1e-9 the binary32 input
    velocities sum to), the binary32 one walks away by orders of magnitude more; the energy fluctuates alike in both."""
    w = CASES["table2_5k"]
    s = wl.make_state(w)
    res = {}
    for prec in (32, 64):
        with hb.System.from_workload(w) as g:
            g.set_tunable("precision", prec)
            g.set_state(s.pos, s.type, s.vel, s.image)
            g.build_nlist(0.0, w.r_buff)
            g.compute_lj(hb.HB_XPLOR)
            g.run_nve(w.dt, 500, 0)
            E, P = [], []
            for _ in range(5):
                t = g.thermo()
                E.append(t["K"] + t["U"])
                P.append(np.array([t["px"], t["py"], t["pz"]]) / w.N)
                g.run_nve(w.dt, 200, 0)
            P = np.array(P)
            res[prec] = (np.array(E), np.abs(P - P[0]).max(), g.stats()["rebuilds"])
    E32, dP32, _ = res[32]
    E64, dP64, nb = res[64]
    assert nb > 50
    assert dP64 < 1e-15 and dP32 > 1000 * dP64, (dP64, dP32)
    # the energy FLUCTUATION is the integrator's and the same for both precisions (Table 2, first column: 1.9e-5);
    # a drift difference needs the paper's long runs to show and is not asserted here
    for E in (E32, E64):
        assert np.std(E) / abs(np.mean(E)) < 6e-5
    assert abs(E64[0] - E32[0]) < 1e-3 * abs(E64[0])


def test_f64_refuses_thermostats(hb):
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    with _dp_system(hb, w, s) as g:
        g.compute_lj(w.shift)
        with pytest.raises(hb.HBError) as e:
            g.run_nvt(w.dt, 5, 1.0, 0.5)
        assert e.value.code == hb.HB_EINVAL
