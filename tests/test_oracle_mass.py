"""Pins of per-particle mass in the oracle's integrators: m = 1 is the pinned
path bit for bit, dynamical similarity under a uniform rescaling of the masses, momentum conservation with mixed
masses, K = 1/2 sum m v^2, equipartition under Langevin dynamics.  CPU only."""
import math

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl


def _lj(N=729):
    w = wl.scaled(wl.CONFIGS["lj_64k"], N)
    return w, wl.make_state(w)


def test_unit_masses_are_the_pinned_path(orc):
    w, s = _lj()
    p = orc.Params.of(w)
    a = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 20)
    b = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 20, mass=np.ones(w.N))
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["vel"], b["vel"])


def test_mass_rescaling_is_a_change_of_time_unit(orc):
    """All masses times lambda, velocities times 1/sqrt(lambda), time step times sqrt(lambda): the same path in
    space (Newton's equations are invariant); catches F*m instead of F/m and a mass applied to one half kick only."""
    w, s = _lj()
    p = orc.Params.of(w)
    lam = 4.0
    a = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 30, log=True)
    b = orc.run_nve(s.pos, s.vel.astype(np.float64) / math.sqrt(lam), s.image, s.type, s.L, p, w.r_buff, w.dt * math.sqrt(lam), 30,
                    mass=np.full(w.N, lam), log=True)
    assert np.abs(a["pos"] + a["image"] * s.L - b["pos"] - b["image"] * s.L).max() < 1e-10
    assert np.abs(a["vel"] - b["vel"] * math.sqrt(lam)).max() < 1e-10
    assert np.allclose(a["KU"], b["KU"], rtol=1e-10)             # K = 1/2 sum m v^2 is the same number


def test_mixed_masses_conserve_momentum_and_energy(orc):
    w, s = _lj()
    p = orc.Params.of(w)
    m = 0.5 + 3.0 * wl.counter_uniform(3, 9, np.arange(w.N))
    o = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, 0.002, 400, mass=m, log=True)
    P0 = (m[:, None] * s.vel.astype(np.float64)).sum(0)
    P1 = (m[:, None] * o["vel"]).sum(0)
    assert np.abs(P1 - P0).max() < 1e-10
    E = o["KU"].sum(1)
    assert E.std() < 2e-4 * abs(o["KU"][:, 0].mean())
    t = orc.thermo(o["vel"], o["U"], o["W"], s.L, mass=m)
    assert t["K"] == pytest.approx(0.5 * (m[:, None] * o["vel"] ** 2).sum(), rel=1e-13)
    assert [t["px"], t["py"], t["pz"]] == pytest.approx(P1.tolist(), abs=1e-10)
    # the heavy particles are the slow ones after the exchange of energy: equipartition within the statistics
    light, heavy = m < 1.5, m > 2.5
    vv = (o["vel"] ** 2).sum(1)
    assert vv[light].mean() > 1.5 * vv[heavy].mean()


def test_langevin_equipartition_with_masses(orc):
    """Free particles of two masses: <m v^2> per component = T / (1 - gamma dt / (2 m)) for each species (the fixed
    point of v <- v (1 - gamma dt / m) + sqrt(6 gamma T dt) u / m)."""
    N, L = 2000, 30.0
    s = wl.uniform_random_state(N, L, 1.0, seed=4)
    p = orc.Params(1, [0.0], [1.0], [2.5], 0)
    m = np.where(np.arange(N) % 2 == 0, 1.0, 5.0)
    T, gamma, dt = 1.2, 10.0, 0.01
    o = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, 0.4, dt, 600, T, gamma, seed=2, mass=m)
    acc = {1.0: [], 5.0: []}
    for _ in range(10):
        o = orc.run_langevin(o["pos"], o["vel"], o["image"], s.type, s.L, p, 0.4, dt, 100, T, gamma, seed=2,
                             step0=int(o["state"][0]), forces=(o["F"], o["U"], o["W"]), mass=m)
        for mm in acc:
            acc[mm].append((mm * o["vel"][m == mm] ** 2).mean())
    for mm in acc:
        assert np.mean(acc[mm]) == pytest.approx(T / (1 - gamma * dt / (2 * mm)), rel=0.02)


def test_nose_hoover_with_masses_is_reversible(orc):
    w, s = _lj(N=512)
    p = orc.Params.of(w)
    m = 0.5 + 3.0 * wl.counter_uniform(3, 9, np.arange(w.N))
    a = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 30, 0.8, 0.5, xi=0.2, mass=m)
    b = orc.run_nvt(a["pos"], -a["vel"], a["image"], s.type, s.L, p, w.r_buff, w.dt, 30, 0.8, 0.5, xi=-a["state"][0],
                    eta=a["state"][1], forces=(a["F"], a["U"], a["W"]), mass=m)
    assert np.abs(b["pos"] + b["image"] * s.L - s.pos - s.image * s.L).max() < 1e-9
    assert np.abs(b["vel"] + s.vel).max() < 1e-9
