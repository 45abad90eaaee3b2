"""GPU parity of the neighbor list with per-type-pair list cutoffs (reading
t1; tunable nlist_pair_rcut): neighbor sets against the oracle's typed Algorithm 3, forces unchanged, the rebuild
invariant through hb_run_nve.  Needs a B200."""
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


def _rlist(w):
    return np.array([np.float32(np.float32(rc) + np.float32(w.r_buff)) for rc in w.rcut], dtype=np.float64)


def _per_pair(typ, rlist, nt):
    return lambda keys: rlist[typ[keys >> 32] * nt + typ[keys & 0xFFFFFFFF]]


@pytest.mark.parametrize("coop", [0, 1, 2])
def test_typed_list_sets_and_forces(hb, orc, coop):
    w = wl.scaled(wl.CONFIGS["ka_1m"], 20_000)
    s = wl.make_state(w)
    rl = _rlist(w)
    pos64 = s.pos.astype(np.float64)
    with hb.System.from_workload(w) as g:
        g.set_tunable("coop_rebuild", coop)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        n_single = g.get_nlist_sizes()[-1]
        g.compute_lj(w.shift)
        f_single, _ = g.get_forces()
        g.set_tunable("nlist_pair_rcut", 1)
        g.build_nlist(0.0, w.r_buff)
        rs, nbr = g.get_nlist()
        g.compute_lj(w.shift)
        f4, w6 = g.get_forces()
        th = g.thermo()
        st = g.stats()
    c, r, n = orc.nlist_cells_typed(pos64, s.type, s.L, w.ntypes, rl)
    parity.assert_nlist_equal(pos64, s.L, _per_pair(s.type, rl, w.ntypes), r, n, rs, nbr)
    assert st["max_nbrs"] == np.diff(rs).max()
    assert rs[-1] < 0.9 * n_single                      # the B rows got shorter (AB 2.0, BB 2.2 against AA 2.5 sigma)
    p = orc.Params.of(w)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, c, r, n, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6)
    parity.assert_energy_close(U.sum(), th["U"], A[:, 1].sum())
    # the same physics as with the single list cutoff (summation order aside)
    assert np.abs(f4[:, :3] - f_single[:, :3]).max() <= 1e-4 * np.abs(F).max()


def test_typed_list_through_run_nve(hb, orc):
    """Device-side rebuilds with the typed criterion: after 150 steps the list in use holds every pair inside its own
    r_cut (reading c3's invariant) and no pair beyond its own r_list plus what a particle may have moved."""
    w = wl.scaled(wl.CONFIGS["ka_1m"], 20_000)
    s = wl.make_state(w)
    rl = _rlist(w)
    with hb.System.from_workload(w) as g:
        g.set_tunable("nlist_pair_rcut", 1)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        E0 = g.thermo()
        g.run_nve(w.dt, 150, 50)
        out = g.get_state()
        rs, nbr = g.get_nlist()
        f4, w6 = g.get_forces()
        E1 = g.thermo()
        st = g.stats()
    assert st["rebuilds"] >= 3
    pos64 = out["pos"].astype(np.float64)
    rc = np.array(w.rcut, dtype=np.float64)
    need = orc.nlist_cells_typed(pos64, s.type, s.L, w.ntypes, rc)
    kg = np.sort(parity.rows_as_keys(rs, nbr))
    assert np.isin(parity.rows_as_keys(need[1], need[2]), kg, assume_unique=True).all(), "the list in use misses a pair inside r_cut"
    d = parity.pair_dist(pos64, s.L, kg)
    assert (d < _per_pair(s.type, rl, w.ntypes)(kg) + w.r_buff + 1e-4).all()
    lst = orc.nlist_cells(pos64, s.L, w.r_max)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, orc.Params.of(w), *lst, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6)
    # the dense lattice start melts violently (U = +6 per particle turns into kinetic energy within these steps):
    # the velocity-Verlet error of that transient is what is left, 2e-3 of the kinetic energy reached
    assert abs((E1["K"] + E1["U"]) - (E0["K"] + E0["U"])) < 2e-3 * E1["K"]


def test_one_type_ignores_the_tunable(hb, orc):
    w = wl.scaled(wl.CONFIGS["lj_64k"], 8_000)
    s = wl.make_state(w)
    with hb.System.from_workload(w) as g:
        g.set_tunable("nlist_pair_rcut", 1)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        rs, nbr = g.get_nlist()
    pos64 = s.pos.astype(np.float64)
    c, r, n = orc.nlist_cells(pos64, s.L, w.r_max)
    parity.assert_nlist_equal(pos64, s.L, w.r_max, r, n, rs, nbr)


@pytest.mark.parametrize("typed", [0, 1])
def test_raising_rcut_after_a_build_rebuilds_with_the_new_radius(hb, orc, typed):
    """hb_set_rcut_pair on a handle that already has a list, then straight to hb_thermo / hb_run_nve with no explicit
    hb_build_nlist: the list the library rebuilds on its own must use the NEW r_max, cell count and per-pair table,
    or the pairs between the old list radius and the new cutoff are silently missing from the forces."""
    w = wl.scaled(wl.CONFIGS["ka_1m"], 20_000)
    s = wl.make_state(w)
    pos64 = s.pos.astype(np.float64)
    short = tuple(0.8 * rc for rc in w.rcut)             # the first list: every cutoff 20 % shorter
    with hb.System(w.N, w.L, w.ntypes, w.eps, w.sigma) as g:
        g.set_tunable("nlist_pair_rcut", typed)
        g.set_rcut_pair(short)
        g.set_state(s.pos, s.type, s.vel, s.image)
        g.build_nlist(0.0, w.r_buff)
        g.compute_lj(w.shift)
        m_short = g.stats()["cells_per_axis"]
        g.set_rcut_pair(w.rcut)                          # raise them; no hb_build_nlist after this
        th = g.thermo()                                  # rebuilds the list and the forces by itself
        m_full = g.stats()["cells_per_axis"]
        rs, nbr = g.get_nlist()
        f4, w6 = g.get_forces()
        g.run_nve(w.dt, 20, 0)                           # and the graphs are captured for the new geometry
        E1 = g.thermo()
    assert m_full < m_short                              # wider cells: the geometry was reconfigured
    rl = _rlist(w)
    if typed:
        c, r, n = orc.nlist_cells_typed(pos64, s.type, s.L, w.ntypes, rl)
        parity.assert_nlist_equal(pos64, s.L, _per_pair(s.type, rl, w.ntypes), r, n, rs, nbr)
    else:
        c, r, n = orc.nlist_cells(pos64, s.L, w.r_max)
        parity.assert_nlist_equal(pos64, s.L, w.r_max, r, n, rs, nbr)
    p = orc.Params.of(w)
    F, U, W, A = orc.compute_lj_nlist(pos64, s.type, s.L, p, c, r, n, band=parity.BAND)
    parity.assert_forces_close(F, U, W, A, f4, w6)
    parity.assert_energy_close(U.sum(), th["U"], A[:, 1].sum())
    # the dense lattice start melts violently: same bound as test_typed_list_through_run_nve (the velocity-Verlet error
    # of that transient); a run whose graphs still held the short cutoff would lose far more than this
    E0 = th["K"] + th["U"]
    assert abs(E1["K"] + E1["U"] - E0) <= 2e-3 * E1["K"]
