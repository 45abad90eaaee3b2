"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py
times (default tunables, hb_run_nve's graphs), on SAMPLED outputs: for a seeded
sample of particles the oracle computes the neighbor row and the force, energy
and virial by brute force over all N particles (O(S N), seconds), and the cell
membership of every particle (O(N)).  Needs a B200.

Two snapshots per config: the seeded start (lattice + jitter) and the state the
GPU itself reaches after `steps` NVE steps with device-side rebuilds and a sort,
downloaded and handed to the oracle -- so the reordered, rebuilt, fused path is
what is compared, not just the first build.
"""
import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

# config -> NVE steps run before the second snapshot (enough for several rebuilds; the sort period is cut to fit)
CASES = {"lj_64k": 120, "lj_1m": 40, "wca_256k": 60, "ka_1m": 40}
SAMPLE = 192


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _sampled_parity(hb, orc, w, g, pos32, typ, L, rng):
    N = w.N
    pos64 = pos32.astype(np.float64)
    p = orc.Params.of(w)
    sample = np.sort(rng.choice(N, size=SAMPLE, replace=False)).astype(np.int64)
    # cells: every particle (the oracle's canonical binary32 formula is O(N))
    g.build_cells()                      # no-op: the cell list of these positions is in place
    m, start, tags = g.get_cells()
    assert m == orc.cell_dim(L, w.r_max)
    parity.assert_cells_equal(orc, pos32, L, m, start, tags)
    # neighbor rows of the sample against brute force over all N
    rs, nbr = g.get_nlist()
    cnt_ref, rs_ref, nbr_ref = orc.nlist_brute_sample(pos64, L, w.r_max, sample)
    bad = 0
    for k, i in enumerate(sample):
        got = set(nbr[rs[i]:rs[i + 1]].tolist())
        ref = set(nbr_ref[rs_ref[k]:rs_ref[k + 1]].tolist())
        assert len(got) == rs[i + 1] - rs[i], "duplicate entries in a row"
        assert i not in got, "self in list"
        for j in got ^ ref:
            d = pos64[i] - pos64[j]
            d -= L * np.rint(d / L)
            dist = float(np.sqrt((d * d).sum()))
            assert abs(dist - w.r_max) <= parity.BAND, f"row {i}: pair with d = {dist} on one side only"
            bad += 1
    # forces, energies, virials of the sample
    f4, w6 = g.get_forces()
    F, U, W, A = orc.compute_lj_brute_sample(pos64, typ, L, p, sample, band=parity.BAND)
    # max |F| over the sample stands in for max over all particles (it is smaller or equal: a stricter test)
    worst = parity.assert_forces_close(F, U, W, A, f4, w6, rows=sample)
    return worst, bad


@pytest.mark.parametrize("case", list(CASES))
def test_fullsize_sampled_parity(hb, orc, case):
    w = wl.CONFIGS[case]
    s = wl.make_state(w)
    rng = np.random.default_rng(1234)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        worst0, _ = _sampled_parity(hb, orc, w, g, s.pos, s.type, s.L, rng)
        # the path bench.py times: graphs, device-side rebuild decisions, fused step kernel, one sort on the way
        steps = CASES[case]
        g.run_nve(w.dt, steps, max(1, steps // 2))
        st = g.stats()
        assert st["rebuilds"] >= 3 and st["sorts"] >= 1 and st["steps"] == steps
        out = g.get_state()
        assert np.array_equal(np.sort(out["order"]), np.arange(w.N)), "a particle was lost or duplicated"
        assert np.array_equal(out["type"], s.type)
        assert np.all(out["pos"] >= -s.L / 2) and np.all(out["pos"] <= s.L / 2)
        # the list in use must still hold every pair inside r_cut of the sample (reading c3's invariant) ...
        pos64 = out["pos"].astype(np.float64)
        sample = np.sort(rng.choice(w.N, size=SAMPLE, replace=False)).astype(np.int64)
        rs, nbr = g.get_nlist()
        _, rs_need, nbr_need = orc.nlist_brute_sample(pos64, s.L, w.r_cut_max, sample)
        for k, i in enumerate(sample):
            have = set(nbr[rs[i]:rs[i + 1]].tolist())
            assert set(nbr_need[rs_need[k]:rs_need[k + 1]].tolist()) <= have, f"row {i} misses a pair inside r_cut"
        # ... and the forces of the final state (computed by the graph's last kernel over that older list) must
        # agree with brute force on that state
        f4, w6 = g.get_forces()
        F, U, W, A = orc.compute_lj_brute_sample(pos64, s.type, s.L, orc.Params.of(w), sample, band=parity.BAND)
        parity.assert_forces_close(F, U, W, A, f4, w6, rows=sample)
        # a fresh build on that state: cells, rows, forces again
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        worst1, _ = _sampled_parity(hb, orc, w, g, out["pos"], s.type, s.L, rng)
    assert max(worst0, worst1) <= parity.F_TOL


def test_four_million_particles(hb, orc):
    """Beyond BASELINE's sizes: N = 160^3 = 4,096,000 (262,144 cells, 16,384 tiles, 128 scan tiles): the index
    arithmetic, the cell scan across many scan tiles and the tables of the tile kernels at a size where a 32-bit
    slip would show; sampled forces against brute force over all N after 30 steps with rebuilds and two sorts."""
    w = wl.scaled(wl.CONFIGS["lj_64k"], 160 ** 3)
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        g.run_nve(w.dt, 30, 15)
        st = g.stats()
        out = g.get_state()
        f4, w6 = g.get_forces()
        th = g.thermo()
    assert st["rebuilds"] >= 3 and st["sorts"] == 2 and st["overflow_retries"] == 0
    assert np.array_equal(np.sort(out["order"]), np.arange(w.N))
    assert max(abs(th["px"]), abs(th["py"]), abs(th["pz"])) / w.N < 1e-6
    pos64 = out["pos"].astype(np.float64)
    sample = np.sort(np.random.default_rng(7).choice(w.N, size=128, replace=False)).astype(np.int64)
    F, U, W, A = orc.compute_lj_brute_sample(pos64, s.type, s.L, orc.Params.of(w), sample, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6, rows=sample)
