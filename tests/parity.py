"""Comparison helpers shared by the GPU parity tests.  Tolerances are the ones
BASELINE.json's north_star states:
  * cell membership and neighbor sets bit-exact, pairs whose distance is within
    1e-5 sigma of r_cut + r_buff excluded;
  * per-particle force: max |dF| / max |F| <= 1e-4 (fp32 GPU vs fp64 oracle), plus
    the cutoff-flip allowance of reading c6.ii for pairs within 1e-5 of r_cut;
  * total potential energy within 1e-5 relative.
"""
import numpy as np

BAND = 1e-5          # sigma; exclusion band around r_max (lists) and r_cut (force flips)
F_TOL = 1e-4         # max|dF| / max|F|
U_TOL = 1e-5         # relative, total potential energy


def assert_cells_equal(orc, pos32, L, m, start_gpu, tags_gpu):
    """Bit-exact membership: every particle sits in the cell the oracle's canonical
    binary32 formula (reading c1.iv) gives; order inside a cell is free."""
    cell = orc.cell_index_f32(pos32, L, m)
    start, _ = orc.build_cells(cell, m)
    assert start_gpu[0] == 0 and start_gpu[-1] == len(pos32)
    assert np.array_equal(start, start_gpu.astype(np.int64)), "cell occupancies differ"
    assert np.array_equal(np.sort(tags_gpu), np.arange(len(pos32), dtype=tags_gpu.dtype)), "a tag is missing or repeated"
    cell_gpu = np.empty(len(pos32), dtype=np.int32)
    cell_gpu[tags_gpu.astype(np.int64)] = np.repeat(np.arange(m ** 3, dtype=np.int32), np.diff(start_gpu))
    assert np.array_equal(cell, cell_gpu), f"{(cell != cell_gpu).sum()} particles in the wrong cell"


def rows_as_keys(row_start, nbr):
    """Every (i, j) entry as one int64 key i * 2^32 + j."""
    counts = np.diff(row_start)
    i = np.repeat(np.arange(len(counts), dtype=np.int64), counts)
    return (i << 32) | nbr.astype(np.int64)


def pair_dist(pos, L, keys):
    i, j = keys >> 32, keys & 0xFFFFFFFF
    d = pos[i] - pos[j]
    d -= L * np.rint(d / L)
    return np.sqrt((d * d).sum(1))


def assert_nlist_equal(pos64, L, r_max, rs_ref, nbr_ref, rs_gpu, nbr_gpu):
    """Set equality of (i, j) entries except pairs within BAND of r_max (a number, or a function of the int64 keys
    i * 2^32 + j that returns each pair's own list cutoff); no duplicates, no self.
    Exact at any size: rows whose (length, sum j, sum j^2) differ are compared entry by entry as sets,
    all the others must make identical sorted key arrays."""
    kr = np.sort(rows_as_keys(rs_ref, nbr_ref))
    kg = np.sort(rows_as_keys(rs_gpu, nbr_gpu))
    assert not np.any(kg[1:] == kg[:-1]), "duplicate neighbor entries"
    assert not np.any((kg >> 32) == (kg & 0xFFFFFFFF)), "self in list"
    if len(kr) == len(kg) and np.array_equal(kr, kg):
        return 0
    n = len(rs_ref) - 1

    def row_sums(k):
        i, j = k >> 32, (k & 0xFFFFFFFF).astype(np.float64)
        return (np.bincount(i, minlength=n), np.bincount(i, weights=j, minlength=n), np.bincount(i, weights=j * j, minlength=n))

    a, b = row_sums(kr), row_sums(kg)
    odd = (a[0] != b[0]) | (a[1] != b[1]) | (a[2] != b[2])
    keep_r, keep_g = ~odd[kr >> 32], ~odd[kg >> 32]
    assert np.array_equal(kr[keep_r], kg[keep_g]), "rows with equal checksums differ"
    only_ref = np.setdiff1d(kr[~keep_r], kg[~keep_g], assume_unique=True)
    only_gpu = np.setdiff1d(kg[~keep_g], kr[~keep_r], assume_unique=True)
    for name, ks in (("missing from GPU list", only_ref), ("extra in GPU list", only_gpu)):
        if len(ks):
            d = pair_dist(pos64, L, ks)
            rm = r_max(ks) if callable(r_max) else r_max       # per-type-pair list cutoffs: a function of the (i, j) keys
            bad = np.abs(d - rm) > BAND
            assert not bad.any(), f"{bad.sum()} pairs {name}, e.g. d = {d[bad][:3]} vs r_max = {rm if np.isscalar(rm) else rm[bad][:3]}"
    return len(only_ref) + len(only_gpu)


def assert_forces_close(F_ref, U_ref, W_ref, allow, f4, w6, rows=None):
    """f4 [N][4] = (F, U_i), w6 [N][6] from the GPU (by tag); rows selects a sample."""
    if rows is not None:
        f4, w6 = f4[rows], (w6[rows] if w6 is not None else None)
    Fmax = np.abs(F_ref).max()
    dF = np.abs(f4[:, :3].astype(np.float64) - F_ref).max(1)
    lim = F_TOL * Fmax + (allow[:, 0] if allow is not None else 0.0)
    worst = (dF / lim).max()
    assert worst <= 1.0, f"force mismatch: max |dF| = {dF.max():.3e}, max |F| = {Fmax:.3e}, worst ratio {worst:.2f}"
    if w6 is not None:
        Wmax = np.abs(W_ref).max()
        dW = np.abs(w6.astype(np.float64) - W_ref).max(1)
        limW = F_TOL * Wmax + (allow[:, 2] if allow is not None else 0.0)
        assert (dW / limW).max() <= 1.0, f"virial mismatch: max |dW| = {dW.max():.3e}, max |W| = {Wmax:.3e}"
    dU = np.abs(f4[:, 3].astype(np.float64) - U_ref)
    limU = F_TOL * np.abs(U_ref).max() + (allow[:, 1] if allow is not None else 0.0)
    assert (dU / limU).max() <= 1.0, f"per-particle energy mismatch: {dU.max():.3e}"
    return float(dF.max() / Fmax)


def assert_energy_close(U_ref_total, U_gpu_total, allow_total=0.0):
    err = abs(U_gpu_total - U_ref_total)
    assert err <= U_TOL * abs(U_ref_total) + allow_total, f"U: gpu {U_gpu_total!r} vs oracle {U_ref_total!r}"
    return err / abs(U_ref_total)
