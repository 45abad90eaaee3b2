"""GPU parity on seeded RANDOM small systems: box sizes from 3 cells per axis up, densities from a dilute gas
to a dense liquid, one to three types with random symmetric tables and per-pair cutoffs, both shift modes,
random tile shapes.  Every case is compared stage by stage with the oracle (cells bit-exact, neighbor sets,
forces / energies / virials); the lattice-based ones are also run for a few steps through hb_run_nve and the
list in use is checked to hold every pair inside r_cut (reading c3's invariant).  Needs a B200.

The point is breadth of geometry: tiles clipped at the box faces, tiles wider than the box (the same cell staged
under two periodic images), the image rule by tile centre and the one by cell centre, cells with zero to
dozens of particles, rows of length zero.
"""

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity

pytestmark = pytest.mark.gpu

NCASES = 60


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _f32(x):
    return float(np.float32(x))


def _random_case(k):
    rng = np.random.default_rng(1000 + k)
    for _ in range(100):
        ntypes = int(rng.integers(1, 4))
        gas = bool(rng.integers(0, 2)) or ntypes == 3        # make_state knows two types; three come from the gas generator
        N = int(rng.integers(60, 4000))
        rho = float(rng.uniform(0.08, 1.1)) if not gas else float(rng.uniform(0.05, 0.6))
        eps = np.ones((ntypes, ntypes))
        sig = np.ones((ntypes, ntypes))
        rc = np.ones((ntypes, ntypes))
        for a in range(ntypes):
            for b in range(a, ntypes):
                eps[a, b] = eps[b, a] = _f32(rng.uniform(0.5, 1.5))
                sig[a, b] = sig[b, a] = _f32(rng.uniform(0.8, 1.1))
                rc[a, b] = rc[b, a] = _f32(rng.uniform(1.3, 3.0) * sig[a, b])
        r_buff = _f32(rng.uniform(0.1, 0.5))
        w = wl.Workload(f"rand{k}", N, rho, float(rng.uniform(0.5, 1.5)), ntypes, tuple(eps.ravel()), tuple(sig.ravel()),
                        tuple(rc.ravel()), r_buff, _f32(0.002), 20, int(rng.integers(0, 2)), 0,
                        frac_A=float(rng.uniform(0.3, 0.9)), jitter=float(rng.uniform(0.0, 0.25)), seed=k)
        if w.L >= 3.0 * w.r_max * 1.001:
            tiles = [int(rng.integers(0, 5)) for _ in range(3)]
            if 0 in tiles:
                tiles = [0, 0, 0]
            return w, gas, tiles
    raise AssertionError("no admissible case drawn")


@pytest.mark.parametrize("k", range(NCASES))
def test_random_system(hb, orc, k):
    w, gas, tiles = _random_case(k)
    s = wl.uniform_random_state(w.N, w.L, w.T, seed=k, ntypes=w.ntypes) if gas else wl.make_state(w)
    pos64 = s.pos.astype(np.float64)
    p = orc.Params.of(w)
    with hb.System.from_workload(w) as g:
        for name, v in zip(("tile_x", "tile_y", "tile_z"), tiles):
            g.set_tunable(name, v)
        g.set_tunable("graph_steps", 7)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.build_cells()
        m, start, tags = g.get_cells()
        assert m == orc.cell_dim(s.L, w.r_max) and m >= 3
        parity.assert_cells_equal(orc, s.pos, s.L, m, start, tags)
        rs, nbr = g.get_nlist()
        lst = orc.nlist_cells(pos64, s.L, w.r_max)
        parity.assert_nlist_equal(pos64, s.L, w.r_max, lst[1], lst[2], rs, nbr)
        g.compute_lj(w.shift)
        f4, w6 = g.get_forces()
        F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=parity.BAND)
        parity.assert_forces_close(F, U, W, A, f4, w6)
        if gas:
            return      # overlapping particles: no sensible dynamics
        g.run_nve(w.dt, w.steps, 9)
        out = g.get_state()
        rs, nbr = g.get_nlist()
        f4, w6 = g.get_forces()
    assert np.array_equal(np.sort(out["order"]), np.arange(w.N)) and np.array_equal(out["type"], s.type)
    pos64 = out["pos"].astype(np.float64)
    need = orc.nlist_cells(pos64, s.L, w.r_cut_max)
    kg = np.sort(parity.rows_as_keys(rs, nbr))
    kn = parity.rows_as_keys(need[1], need[2])
    assert np.isin(kn, kg, assume_unique=True).all(), "the list in use misses a pair inside r_cut"
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, *lst, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6)
