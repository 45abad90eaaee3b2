"""GPU parity of the thermostatted integrators (readings n1, n2): hb_run_nvt and
hb_run_langevin through the C ABI against the oracle's orc_run_thermostat on identical seeded inputs: short
trajectories particle by particle (as for config 1), thermostat variables, long-run behaviour by invariants.
Needs a B200."""
import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _system(hb, w, s, **tun):
    g = hb.System.from_workload(w)
    for k, v in tun.items():
        g.set_tunable(k, v)
    g.set_state(s.pos, s.type, s.vel, s.image)
    g.build_nlist(0.0, w.r_buff)
    g.compute_lj(w.shift)
    return g


def _unwrapped(o, L):
    return o["pos"].astype(np.float64) + o["image"] * L


@pytest.mark.parametrize("tun", [dict(), dict(graph_mode=0), dict(fuse_nve=0), dict(graph_steps=4), dict(graph_mode=2)])
def test_nvt_trajectory_matches_the_oracle(hb, orc, tun):
    """config-1 fluid, 10 Nose-Hoover steps at T = 0.9, tau = 0.5: positions <= 1e-5, velocities, xi and eta."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    p = orc.Params.of(w)
    T, tau = 0.9, 0.5
    ref = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 10, T, tau, log=True)
    with _system(hb, w, s, **tun) as g:
        g.run_nvt(w.dt, 10, T, tau)
        out = g.get_state()
        ts = g.get_thermostat()
        th = g.thermo()
    assert np.abs(_unwrapped(out, s.L) - (ref["pos"] + ref["image"] * s.L)).max() <= 1e-5
    assert np.abs(out["vel"].astype(np.float64) - ref["vel"]).max() <= 1e-5 * max(1.0, np.abs(ref["vel"]).max())
    assert ts["xi"] == pytest.approx(ref["state"][0], rel=1e-5, abs=1e-8)
    assert ts["eta"] == pytest.approx(ref["state"][1], rel=1e-5, abs=1e-9)
    assert abs(ref["state"][0]) > 1e-3                     # the thermostat did act
    assert th["K"] == pytest.approx(ref["log"][-1, 0], rel=2e-5)


def test_nvt_reaches_the_set_temperature_and_conserves_its_invariant(hb, orc):
    """20,000-particle fluid from the hot melting lattice to T = 1.0: T_k within 3 %, and over the following 600
    steps H' = K + U + g T (tau^2 xi^2 / 2 + eta) stays put at the level the oracle keeps it."""
    w = wl.scaled(wl.CONFIGS["lj_64k"], 19_683)
    s = wl.make_state(w)
    T, tau, g_ = 1.0, 0.5, 3 * w.N - 3
    with _system(hb, w, s) as g:
        g.run_nvt(w.dt, 1500, T, tau, sort_period=500)
        H = []
        for _ in range(7):
            th, ts = g.thermo(), g.get_thermostat()
            H.append(th["K"] + th["U"] + g_ * T * (0.5 * tau * tau * ts["xi"] ** 2 + ts["eta"]))
            Tk = 2 * th["K"] / g_
            g.run_nvt(w.dt, 100, T, tau)
        st = g.stats()
    assert Tk == pytest.approx(T, rel=0.03)
    assert st["rebuilds"] > 50 and st["sorts"] >= 3
    assert np.ptp(H) < 3e-4 * 1.5 * w.N * T, np.ptp(H)


@pytest.mark.parametrize("tun", [dict(), dict(graph_mode=0), dict(fuse_nve=0), dict(graph_steps=4)])
def test_langevin_trajectory_matches_the_oracle(hb, orc, tun):
    """The same generator on both sides (orc_uniform_pm1 / hb_uniform_pm1): 10 Langevin steps agree particle by
    particle, then 7 more in a second call (the step counter carries on)."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    p = orc.Params.of(w)
    T, gamma, seed = 0.8, 2.0, 12345
    ref = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 17, T, gamma, seed)
    with _system(hb, w, s, **tun) as g:
        g.run_langevin(w.dt, 10, T, gamma, seed)
        g.sort()                                   # a reorder in between: the generator follows the tags
        g.run_langevin(w.dt, 7, T, gamma, seed)
        out = g.get_state()
        ts = g.get_thermostat()
    assert ts["langevin_steps"] == 17
    assert np.abs(_unwrapped(out, s.L) - (ref["pos"] + ref["image"] * s.L)).max() <= 2e-5
    assert np.abs(out["vel"].astype(np.float64) - ref["vel"]).max() <= 2e-5 * max(1.0, np.abs(ref["vel"]).max())
    nve = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 17)
    assert np.abs(ref["vel"] - nve["vel"]).max() > 0.05   # the noise is not a no-op


@pytest.mark.parametrize("tun", [dict(), dict(fuse_nve=0), dict(graph_mode=2)])
def test_langevin_after_a_graph_run_and_a_single_step(hb, orc, tun):
    """hb_run_nve, then hb_step_nve, then hb_run_langevin: the single step leaves its own step offset in the handle,
    and the graphs captured for the new ensemble must not inherit it -- the generator's stream is the number of the
    Langevin step since hb_set_state (hb.h), whatever was called before."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    p = orc.Params.of(w)
    T, gamma, seed = 0.8, 2.0, 99
    nve = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 4)
    ref = orc.run_langevin(nve["pos"], nve["vel"], nve["image"], s.type, s.L, p, w.r_buff, w.dt, 10, T, gamma, seed)
    with _system(hb, w, s, **tun) as g:
        g.run_nve(w.dt, 3, 0)
        g.step_nve(w.dt)
        g.run_langevin(w.dt, 10, T, gamma, seed)
        out = g.get_state()
        ts = g.get_thermostat()
    assert ts["langevin_steps"] == 10
    assert np.abs(_unwrapped(out, s.L) - (ref["pos"] + ref["image"] * s.L)).max() <= 2e-5
    assert np.abs(out["vel"].astype(np.float64) - ref["vel"]).max() <= 2e-5 * max(1.0, np.abs(ref["vel"]).max())


def test_langevin_free_particles_and_thermalisation(hb, orc):
    """eps = 0: stationary <v^2> = T / (1 - gamma dt / 2) per component (the closed form that pins the oracle);
    the interacting fluid settles at the set temperature."""
    N, L = 20_000, 60.0
    s = wl.uniform_random_state(N, L, 1.0, seed=4)
    T, gamma, dt = 1.5, 10.0, 0.01
    with hb.System(N, L, 1, [0.0], [1.0]) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(2.5, 0.4)
        g.compute_lj(0)
        g.run_langevin(dt, 300, T, gamma, 7)
        acc = []
        for _ in range(6):
            g.run_langevin(dt, 50, T, gamma, 7)
            acc.append((g.get_state()["vel"].astype(np.float64) ** 2).mean())
    assert np.mean(acc) == pytest.approx(T / (1 - gamma * dt / 2), rel=0.01)
    w = wl.scaled(wl.CONFIGS["lj_64k"], 19_683)
    s = wl.make_state(w)
    with _system(hb, w, s) as g:
        g.run_langevin(w.dt, 2500, 0.9, 1.0, 3, sort_period=1000)
        Tk = []
        for _ in range(5):
            g.run_langevin(w.dt, 100, 0.9, 1.0, 3)
            Tk.append(2 * g.thermo()["K"] / (3 * w.N))
        out = g.get_state()
    assert np.mean(Tk) == pytest.approx(0.9, rel=0.03)
    assert np.array_equal(np.sort(out["order"]), np.arange(w.N))


def test_nve_is_unchanged_by_the_thermostat_code(hb, orc):
    """hb_run_nve after thermostatted runs integrates NVE again; tau -> huge and gamma = 0 reproduce it bit for bit."""
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    outs = []
    for mode in ("nve", "nvt", "lang"):
        with _system(hb, w, s) as g:
            if mode == "nve":
                g.run_nve(w.dt, 20, 0)
            elif mode == "nvt":
                g.run_nvt(w.dt, 20, 1.0, 1e18)
            else:
                g.run_langevin(w.dt, 20, 1.0, 0.0, 1)
            outs.append(g.get_state())
    assert np.array_equal(outs[0]["pos"], outs[2]["pos"]) and np.array_equal(outs[0]["vel"], outs[2]["vel"])
    assert np.abs(outs[0]["pos"] - outs[1]["pos"]).max() <= 1e-6 and np.abs(outs[0]["vel"] - outs[1]["vel"]).max() <= 1e-6
