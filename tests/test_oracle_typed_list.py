"""Pins of the oracle's neighbor list with per-type-pair list cutoffs (
reading t1: N(i) = { j != i : d_ij < r_cut(type i, type j) + r_buff }).  CPU only."""
import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl
from tests import parity


def _ka(N=1500):
    w = wl.scaled(wl.CONFIGS["ka_1m"], N)
    s = wl.make_state(w)
    rlist = np.array([np.float32(np.float32(rc) + np.float32(w.r_buff)) for rc in w.rcut], dtype=np.float64)
    return w, s, rlist


def _keys(rs, nbr):
    return np.sort(parity.rows_as_keys(rs, nbr))


def test_uniform_table_is_the_single_cutoff_list(orc):
    w, s, _ = _ka()
    pos = s.pos.astype(np.float64)
    a = orc.nlist_brute(pos, s.L, w.r_max)
    b = orc.nlist_brute_typed(pos, s.type, s.L, 2, [w.r_max] * 4)
    c = orc.nlist_cells_typed(pos, s.type, s.L, 2, [w.r_max] * 4)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[2], b[2])
    assert np.array_equal(_keys(a[1], a[2]), _keys(c[1], c[2]))


def test_typed_list_against_numpy_and_the_cell_path(orc):
    """Independent numpy statement of the definition (all pairs, minimum image, the pair's own cutoff); a wrong table
    index (type j for type i, a transposed table entry used asymmetrically) or the global cutoff fails it."""
    w, s, rlist = _ka(900)
    pos = s.pos.astype(np.float64)
    d = pos[:, None, :] - pos[None, :, :]
    d -= s.L * np.round(d / s.L)
    r = np.sqrt((d * d).sum(-1))
    rl = rlist.reshape(2, 2)[s.type[:, None], s.type[None, :]]
    want = (r < rl) & ~np.eye(len(pos), dtype=bool)
    c, rs, nbr = orc.nlist_brute_typed(pos, s.type, s.L, 2, rlist)
    got = np.zeros_like(want)
    got[np.repeat(np.arange(len(pos)), c), nbr] = True
    assert np.array_equal(got, want)
    assert np.array_equal(got, got.T)                        # full list: i in N(j) iff j in N(i)
    c2, rs2, nbr2 = orc.nlist_cells_typed(pos, s.type, s.L, 2, rlist)
    assert np.array_equal(_keys(rs, nbr), _keys(rs2, nbr2))
    # it is a proper subset of the single-cutoff list, and the B rows are the ones that got shorter
    full = orc.nlist_brute(pos, s.L, float(rlist.max()))
    assert np.isin(_keys(rs, nbr), _keys(full[1], full[2]), assume_unique=True).all()
    assert c.sum() < full[0].sum() and (c[s.type == 1] < full[0][s.type == 1]).mean() > 0.9


def test_forces_over_the_typed_list_are_the_forces(orc):
    """Every pair inside its r_cut is in the typed list (r_list >= r_cut), so the force sums over it equal the
    O(N^2) definition: bit for bit the sums over the single-cutoff list when the order of j is the same."""
    w, s, rlist = _ka()
    pos = s.pos.astype(np.float64)
    p = orc.Params.of(w)
    F0, U0, W0 = orc.compute_lj_brute(pos, s.type, s.L, p)
    lt = orc.nlist_brute_typed(pos, s.type, s.L, 2, rlist)
    F1, U1, W1, _ = orc.compute_lj_nlist(pos, s.type, s.L, p, *lt)
    assert np.array_equal(F0, F1) and np.array_equal(U0, U1) and np.array_equal(W0, W1)


def test_small_box_is_rejected(orc):
    w, s, rlist = _ka(200)
    with pytest.raises(RuntimeError):
        orc.nlist_brute_typed(s.pos.astype(np.float64), s.type, s.L, 2, rlist * 4)
