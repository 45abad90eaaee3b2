"""GPU parity of the other pair functors and of per-particle mass (PAPER.md:105, 111, 125,
284; reading f1): Gaussian, Yukawa and Morse through the same step kernel with the three cutoff treatments
(hb_set_pair_potential + hb_compute_lj), masses through hb_set_mass into the integrators, the thermostats and
hb_thermo -- against the oracle on identical seeded snapshots, at the tolerances of tests/parity.py.  Needs a B200."""
import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

# (eps, sigma, p2) per potential, the values the oracle's own pins use (tests/test_oracle_potentials.py)
POTS = {"gauss": (2.0, 0.9, 0.0), "yukawa": (3.0, 1.7, 0.0), "morse": (1.5, 2.2, 1.1)}


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _f32(x):
    return float(np.float32(x))


def _one_type(pot, N=19_683):
    """The LJ-liquid geometry (rho* = 0.382, r_cut 3.0 -> here 2.5, r_buff 0.4) with another potential's parameters."""
    e, s, q = POTS[pot]
    base = wl.scaled(wl.CONFIGS["lj_64k"], N)
    return wl.Workload(pot, N, base.rho, base.T, 1, (_f32(e),), (_f32(s),), (2.5,), 0.4, 0.005, 0, 1, 0), (_f32(q),)


def _two_types(pot, N=10_001):
    """Kob-Andersen geometry and 80:20 type mix, per-pair parameter tables and cutoffs."""
    e, s, q = POTS[pot]
    base = wl.scaled(wl.CONFIGS["ka_1m"], N)
    eps = tuple(_f32(e * f) for f in (1.0, 1.5, 1.5, 0.5))
    sig = tuple(_f32(s * f) for f in (1.0, 0.8, 0.8, 0.88))
    rcut = (2.5, 2.0, 2.0, 2.2)
    p2 = tuple(_f32(q * f) for f in (1.0, 0.9, 0.9, 0.8))
    return wl.Workload(pot + "2", N, base.rho, base.T, 2, eps, sig, rcut, 0.3, 0.002, 0, 1, 0, frac_A=base.frac_A), p2


@pytest.mark.parametrize("pot", list(POTS))
@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("types", [1, 2])
def test_functor_forces_energy_virial(hb, orc, pot, mode, types):
    w, p2 = _one_type(pot) if types == 1 else _two_types(pot)
    s = wl.make_state(w)
    ron = [_f32(0.7 * rc) for rc in w.rcut]
    with hb.System.from_workload(w) as g:
        g.set_pair_potential(pot, p2)
        g.set_ron_pair(ron)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(mode)
        f4, w6 = g.get_forces()
        th = g.thermo()
    pos64 = s.pos.astype(np.float64)
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    p = orc.Params(w.ntypes, w.eps, w.sigma, w.rcut, mode, ron=ron, pot=pot, p2=p2)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=parity.BAND)
    assert np.abs(F).max() > 0.1
    parity.assert_forces_close(F, U, W, A, f4, w6)
    parity.assert_energy_close(U.sum(), th["U"], A[:, 1].sum())
    Wt = W.sum(0)
    assert np.allclose(th["W"], Wt, rtol=0, atol=1e-5 * np.abs(Wt).max() + A[:, 2].sum())


def test_potential_switches_back_to_lj(hb, orc):
    """hb_set_pair_potential(HB_POT_LJ) after a generic functor gives the LJ numbers again (tables are rebuilt)."""
    w = wl.scaled(wl.CONFIGS["lj_64k"], 8_000)
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(1)
        a, _ = g.get_forces()
        g.set_pair_potential("morse", [1.1])
        g.compute_lj(1)
        b, _ = g.get_forces()
        g.set_pair_potential("lj")
        g.compute_lj(1)
        c, _ = g.get_forces()
        with pytest.raises(hb.HBError):
            g.set_pair_potential(7)
    assert np.array_equal(a, c) and not np.array_equal(a, b)


@pytest.mark.parametrize("pot", ["morse", "gauss"])
def test_functor_nve_conserves_energy(hb, pot):
    """350 steps of hb_run_nve with a smoothed generic functor (V and F continuous at r_cut): device-side rebuilds,
    total energy conserved at the 1e-4 level of the kinetic energy (dt = 0.0025: the Morse well with a = 2.2 is
    stiffer than LJ's, the velocity-Verlet error goes with dt^2)."""
    w, p2 = _one_type(pot, 8_000)
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        g.set_pair_potential(pot, p2)
        g.set_ron_pair([_f32(0.7 * rc) for rc in w.rcut])
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(2)
        dt = 0.0025
        g.run_nve(dt, 50, 0)
        E = []
        for _ in range(6):
            t = g.thermo()
            E.append(t["K"] + t["U"])
            g.run_nve(dt, 50, 0)
        st = g.stats()
    assert st["rebuilds"] >= 3
    assert np.ptp(E) < 2e-4 * 1.5 * w.N * w.T, np.ptp(E)


# ---- per-particle mass ----

def _masses(N):
    return (0.5 + 3.0 * wl.counter_uniform(3, 9, np.arange(N))).astype(np.float32)


def _unwrapped(o, L):
    return o["pos"].astype(np.float64) + o["image"] * L


@pytest.mark.parametrize("tun", [dict(), dict(graph_mode=0), dict(fuse_nve=0), dict(thermo_every=1)])
def test_mass_nve_trajectory_and_thermo(hb, orc, tun):
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    m = _masses(w.N)
    p = orc.Params.of(w)
    ref = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 10, mass=m.astype(np.float64))
    with hb.System.from_workload(w) as g:
        for k, v in tun.items():
            g.set_tunable(k, v)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.set_mass(m)
        assert np.array_equal(g.get_mass(), m)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        g.run_nve(w.dt, 6, 0)
        g.sort()                                   # a reorder in between: the masses travel with the particles
        g.run_nve(w.dt, 4, 0)
        out = g.get_state()
        th = g.thermo()
        assert np.array_equal(g.get_mass(), m)
    assert np.abs(_unwrapped(out, s.L) - (ref["pos"] + ref["image"] * s.L)).max() <= 1e-5
    assert np.abs(out["vel"].astype(np.float64) - ref["vel"]).max() <= 1e-5 * max(1.0, np.abs(ref["vel"]).max())
    v = out["vel"].astype(np.float64)
    t = orc.thermo(v, ref["U"], ref["W"], s.L, mass=m.astype(np.float64))
    assert th["K"] == pytest.approx(t["K"], rel=1e-12)
    for a in ("px", "py", "pz"):
        assert th[a] == pytest.approx(t[a], abs=1e-9 * w.N)
    # the heavy and the light particles do move differently from the m = 1 run
    one = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 10)
    assert np.abs(one["vel"] - ref["vel"]).max() > 1e-2


def test_unit_mass_is_the_default_path_bit_for_bit(hb):
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    outs = []
    for setm in (False, True):
        with hb.System.from_workload(w) as g:
            g.set_state(s.pos, s.type, s.vel, s.image)
            if setm:
                g.set_mass(np.ones(w.N, np.float32))
            g.build_nlist(0.0, w.r_buff)
            g.compute_lj(w.shift)
            g.run_nve(w.dt, 20, 0)
            outs.append(g.get_state())
    assert np.array_equal(outs[0]["pos"], outs[1]["pos"]) and np.array_equal(outs[0]["vel"], outs[1]["vel"])


def test_mass_thermostats_match_the_oracle(hb, orc):
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    m = _masses(w.N)
    p = orc.Params.of(w)
    m64 = m.astype(np.float64)
    T, tau, gamma, seed = 1.0, 0.5, 2.0, 99
    ref_n = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 12, T, tau, mass=m64)
    ref_l = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 12, T, gamma, seed, mass=m64)
    for kind, ref in (("nvt", ref_n), ("lang", ref_l)):
        with hb.System.from_workload(w) as g:
            g.set_state(s.pos, s.type, s.vel, s.image)
            g.set_mass(m)
            g.build_nlist(0.0, w.r_buff)
            g.compute_lj(w.shift)
            if kind == "nvt":
                g.run_nvt(w.dt, 12, T, tau)
                ts = g.get_thermostat()
                assert ts["xi"] == pytest.approx(ref["state"][0], abs=2e-6) and ts["eta"] == pytest.approx(ref["state"][1], abs=2e-6)
            else:
                g.run_langevin(w.dt, 12, T, gamma, seed)
            out = g.get_state()
        assert np.abs(_unwrapped(out, s.L) - (ref["pos"] + ref["image"] * s.L)).max() <= 2e-5, kind
        assert np.abs(out["vel"].astype(np.float64) - ref["vel"]).max() <= 2e-5 * max(1.0, np.abs(ref["vel"]).max()), kind


def test_mass_errors(hb):
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        with pytest.raises(hb.HBError) as e:
            g.set_mass(np.ones(w.N, np.float32))          # no state yet
        assert e.value.code == hb.HB_ESTATE
        g.set_state(s.pos, s.type, s.vel, s.image)
        bad = np.ones(w.N, np.float32)
        bad[17] = 0.0
        with pytest.raises(hb.HBError) as e:
            g.set_mass(bad)
        assert e.value.code == hb.HB_EINVAL
        g.set_mass(np.full(w.N, 2.0, np.float32))
        g.set_state(s.pos, s.type, s.vel, s.image)        # resets the masses
        assert np.array_equal(g.get_mass(), np.ones(w.N, np.float32))
