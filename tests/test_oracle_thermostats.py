"""Pins of the oracle's thermostatted integrators (readings n1, n2 in DESIGN.md) to things
other than themselves: limits that reduce to the pinned NVE loop, time reversibility, the conserved quantity of the
Nose-Hoover equations, closed forms of the Langevin velocity recursion for free particles, and the Python statement
of the counter-based generator in workloads.py.  CPU only."""
import math

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl


def _lj(N=1000, T=1.2, seed=0):
    w = wl.scaled(wl.CONFIGS["lj_64k"], N)
    w = wl.dataclasses.replace(w, T=T)
    return w, wl.make_state(w, seed=seed)


def test_counter_generator_matches_its_python_statement(orc):
    """n2: orc_counter_u64 == workloads.counter_u64 (an independent implementation) bit for bit; the uniform is
    exact in binary32, strictly inside (-1, 1), with mean 0 and variance 1/3."""
    rng = np.random.default_rng(0)
    for _ in range(200):
        seed, stream, index = (int(x) for x in rng.integers(0, 2 ** 62, size=3))
        assert orc.counter_u64(seed, stream, index) == int(wl.counter_u64(seed, stream, np.array([index], dtype=np.uint64))[0])
    u = np.array([orc.uniform_pm1(3, 17, i) for i in range(100_000)])
    assert np.array_equal(u, u.astype(np.float32).astype(np.float64))
    assert np.abs(u).max() < 1.0 and abs(u.mean()) < 6e-3 and u.var() == pytest.approx(1 / 3, rel=0.01)
    k = wl.counter_u64(3, 17, np.arange(1000, dtype=np.uint64)) >> np.uint64(41)
    assert np.array_equal(u[:1000], (2.0 * k.astype(np.float64) + 1.0 - 2 ** 23) / 2 ** 23)
    assert orc.uniform_pm1(3, 18, 5) != orc.uniform_pm1(3, 17, 5) != orc.uniform_pm1(4, 17, 5)


def test_thermostats_reduce_to_nve(orc):
    """n1 with tau = infinity and n2 with gamma = 0 are the NVE loop of c7, bit for bit."""
    w, s = _lj()
    p = orc.Params.of(w)
    ref = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 25)
    a = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 25, 1.0, math.inf)
    b = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 25, 1.0, 0.0, seed=9)
    for o in (a, b):
        assert np.array_equal(o["pos"], ref["pos"]) and np.array_equal(o["vel"], ref["vel"]) and np.array_equal(o["image"], ref["image"])
    assert a["state"].tolist() == [0.0, 0.0] and b["state"][0] == 25


def test_nose_hoover_is_time_reversible_and_keeps_momentum(orc):
    """n1: k steps, then (v, xi) -> (-v, -xi), k steps: back at the start to round-off (a wrong order of the
    half steps, or friction applied explicitly in both, breaks this); sum of v stays 0."""
    w, s = _lj(N=512)
    p = orc.Params.of(w)
    a = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 40, 0.8, 0.5, xi=0.3)
    assert abs(a["state"][0] - 0.3) > 1e-3
    # dP/dt = -xi P for the total momentum: a start with P = 0 (here ~1e-6 from the binary32 rounding of v) stays there
    assert np.abs(a["vel"].sum(0)).max() < 2 * max(1e-9, np.abs(s.vel.astype(np.float64).sum(0)).max())
    b = orc.run_nvt(a["pos"], -a["vel"], a["image"], s.type, s.L, p, w.r_buff, w.dt, 40, 0.8, 0.5,
                    xi=-a["state"][0], eta=a["state"][1], forces=(a["F"], a["U"], a["W"]))
    d = b["pos"] + b["image"] * s.L - (s.pos.astype(np.float64) + s.image * s.L)
    assert np.abs(d).max() < 1e-9
    assert np.abs(b["vel"] + s.vel.astype(np.float64)).max() < 1e-9
    assert b["state"][0] == pytest.approx(-0.3, abs=1e-10)


def test_nose_hoover_conserved_quantity_and_temperature(orc):
    """n1: H' = K + U + g T (tau^2 xi^2 / 2 + eta), g = 3N - 3, has no drift and fluctuates as dt^2;
    a fluid started at T_k ~ 1.9 (melting lattice) is brought to the set temperature."""
    w, s = _lj(N=1000, T=1.2)
    p = orc.Params.of(w)
    T, tau, g = 1.0, 0.5, 3 * 1000 - 3
    eq = orc.run_nvt(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, 0.005, 1500, T, tau)

    def hprime(dt, n):
        o = orc.run_nvt(eq["pos"], eq["vel"], eq["image"], s.type, s.L, p, w.r_buff, dt, n, T, tau,
                        xi=eq["state"][0], eta=eq["state"][1], forces=(eq["F"], eq["U"], eq["W"]), log=True)
        K, U, xi, eta = o["log"].T
        return K + U + g * T * (0.5 * tau * tau * xi * xi + eta), 2 * K / g

    H1, Tk = hprime(0.005, 800)
    H2, _ = hprime(0.0025, 1600)
    K0 = 1.5 * 1000 * T
    assert np.abs(H1 - H1[0]).max() < 2e-3 * K0                       # vs O(1) K0 swings of K + U alone
    ratio = (H1 - H1.mean()).std() / (H2 - H2.mean()).std()
    assert 2.5 < ratio < 6.5, ratio
    assert Tk[200:].mean() == pytest.approx(T, rel=0.04)
    # without the thermostat the same start stays hot
    nve = orc.run_nve(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, 0.005, 1500, log=True)
    assert 2 * nve["KU"][-300:, 0].mean() / g > 1.3


def test_langevin_free_particles_closed_forms(orc):
    """n2 with V = 0 (eps = 0): without noise v_n = v_0 (1 - gamma dt)^n exactly; with noise the stationary
    <v^2> per component is T / (1 - gamma dt / 2) (the recursion's fixed point), not T."""
    N, L = 2000, 30.0
    s = wl.uniform_random_state(N, L, 1.0, seed=4)
    p = orc.Params(1, [0.0], [1.0], [2.5], 0)
    gamma, dt = 10.0, 0.01
    o = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, 0.4, dt, 37, 0.0, gamma, seed=1)
    assert np.abs(o["vel"] - s.vel.astype(np.float64) * (1 - gamma * dt) ** 37).max() < 1e-13
    T = 1.5
    acc, n = 0.0, 0
    st = dict(pos=s.pos, vel=s.vel, image=s.image, step=0)
    o = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, 0.4, dt, 300, T, gamma, seed=7)
    for _ in range(12):
        o = orc.run_langevin(o["pos"], o["vel"], o["image"], s.type, s.L, p, 0.4, dt, 100, T, gamma, seed=7,
                             step0=int(o["state"][0]), forces=(o["F"], o["U"], o["W"]))
        acc += (o["vel"] ** 2).mean()
        n += 1
    assert acc / n == pytest.approx(T / (1 - gamma * dt / 2), rel=0.012)
    assert abs(acc / n - T) > 0.03 * T


def test_langevin_thermalises_the_lj_fluid_and_restarts_exactly(orc):
    """n2 on the interacting fluid: T_k settles at the set temperature (within the O(gamma dt) of the scheme);
    a run split in two calls (forces and step counter handed over) equals the uninterrupted run to round-off."""
    w, s = _lj(N=1000, T=1.2)
    p = orc.Params.of(w)
    T, gamma = 0.9, 1.0
    o = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 2500, T, gamma, seed=5, log=True)
    Tk = 2 * o["log"][1200:, 0] / (3 * 1000)
    assert Tk.mean() == pytest.approx(T, rel=0.05)
    a = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 30, T, gamma, seed=5)
    b = orc.run_langevin(a["pos"], a["vel"], a["image"], s.type, s.L, p, w.r_buff, w.dt, 30, T, gamma, seed=5,
                         step0=30, forces=(a["F"], a["U"], a["W"]))
    c = orc.run_langevin(s.pos, s.vel, s.image, s.type, s.L, p, w.r_buff, w.dt, 60, T, gamma, seed=5)
    # (the second call rebuilds its list at its first step: another order of the sums, round-off level differences)
    assert np.abs(b["vel"] - c["vel"]).max() < 1e-10 and np.abs(b["pos"] - c["pos"]).max() < 1e-11
    d = orc.run_langevin(a["pos"], a["vel"], a["image"], s.type, s.L, p, w.r_buff, w.dt, 30, T, gamma, seed=5,
                         step0=0, forces=(a["F"], a["U"], a["W"]))
    assert np.abs(d["vel"] - c["vel"]).max() > 1e-3      # the step counter does select the random numbers
