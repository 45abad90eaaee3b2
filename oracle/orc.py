"""ctypes front end of the oracle (oracle/orc.c).  TEST INFRASTRUCTURE ONLY.

Argument marshalling and nothing else: every number comes out of orc.c.
May be imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs -- never by the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orc.c")
_LIB = os.path.join(_HERE, "liborc.so")
_lib = None

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_fp = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")
_up = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
_vp = C.c_void_p


def build(force: bool = False) -> str:
    """gcc -O2, IEEE arithmetic (no fast-math, no FMA contraction), OpenMP over i."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off",
                               "-Wall", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_cell_dim.restype = C.c_int
        L.orc_cell_dim.argtypes = [C.c_double, C.c_double]
        L.orc_cell_index_f32.argtypes = [_fp, C.c_int64, C.c_float, C.c_int, _ip]
        L.orc_cell_index_f64.argtypes = [_dp, C.c_int64, C.c_double, C.c_int, _ip, _vp]
        L.orc_build_cells.argtypes = [_ip, C.c_int64, C.c_int, _lp, _ip]
        L.orc_nlist_brute.argtypes = [_dp, C.c_int64, C.c_double, C.c_double, _ip, _vp, _vp]
        L.orc_nlist_brute_sample.argtypes = [_dp, C.c_int64, C.c_double, C.c_double, _lp, C.c_int64, _ip, _vp, _vp]
        L.orc_nlist_cells.argtypes = [_dp, C.c_int64, C.c_double, C.c_double, C.c_int, _ip, _lp, _ip, _ip, _vp, _vp]
        L.orc_nlist_brute_typed.argtypes = [_dp, _ip, C.c_int64, C.c_double, C.c_int, _dp, _ip, _vp, _vp]
        L.orc_nlist_cells_typed.argtypes = [_dp, _ip, C.c_int64, C.c_double, C.c_int, _dp, C.c_int, _ip, _lp, _ip, _ip, _vp, _vp]
        L.orc_max_disp2.restype = C.c_double
        L.orc_max_disp2.argtypes = [_dp, _dp, C.c_int64, C.c_double]
        L.orc_lj_pair.argtypes = [C.c_double] * 4 + [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_lj_pair_xplor.argtypes = [C.c_double] * 5 + [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_pair_generic.argtypes = [C.c_int] + [C.c_double] * 6 + [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_set_p2.argtypes = [_vp, C.c_int]
        L.orc_set_mass.argtypes = [_vp, C.c_int64]
        L.orc_compute_lj_brute.argtypes = [_dp, _ip, C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp]
        L.orc_compute_lj_brute_sample.argtypes = [_dp, _ip, C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, _dp, C.c_int,
                                                  _lp, C.c_int64, C.c_double, _dp, _dp, _dp, _vp]
        L.orc_compute_lj_nlist.argtypes = [_dp, _ip, C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, _dp, C.c_int,
                                           _ip, _lp, _ip, C.c_double, _dp, _dp, _dp, _vp]
        L.orc_nve_step1.argtypes = [_dp, _dp, _dp, _ip, C.c_int64, C.c_double, C.c_double]
        L.orc_nve_step2.argtypes = [_dp, _dp, C.c_int64, C.c_double]
        L.orc_thermo.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double, _dp]
        L.orc_hilbert_key.restype = C.c_uint32
        L.orc_hilbert_key.argtypes = [C.c_uint32] * 3 + [C.c_int]
        L.orc_sfc_keys.argtypes = [_fp, C.c_int64, C.c_float, C.c_int, _up]
        L.orc_sort_perm.argtypes = [_up, C.c_int64, C.c_int, _lp]
        L.orc_run_nve.argtypes = [_dp, _dp, _ip, _ip, C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, _dp, C.c_int,
                                  C.c_double, C.c_double, C.c_int64, C.c_int, _dp, _dp, _dp, _vp, _vp]
        L.orc_counter_u64.restype = C.c_uint64
        L.orc_counter_u64.argtypes = [C.c_uint64] * 3
        L.orc_uniform_pm1.restype = C.c_double
        L.orc_uniform_pm1.argtypes = [C.c_uint64] * 3
        L.orc_run_thermostat.argtypes = [C.c_int, _dp, _dp, _ip, _ip, C.c_int64, C.c_double, C.c_int, _dp, _dp, _dp, _dp, C.c_int,
                                         C.c_double, C.c_double, C.c_int64, C.c_double, C.c_double, C.c_uint64, _dp,
                                         C.c_int, _dp, _dp, _dp, _vp, _vp]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


class Params:
    """Per-type-pair tables as fp64 arrays (values already fp32-representable)."""

    POTS = {"lj": 0, "gauss": 1, "yukawa": 2, "morse": 3}

    def __init__(self, ntypes, eps, sigma, rcut, shift, ron=None, pot="lj", p2=None):
        """shift: 0 plain, 1 energy shift, 2 XPLOR smoothing (needs ron per type pair).  pot: the potential whose
        parameters the eps / sigma / p2 tables hold (see orc_pair_bare)."""
        self.ntypes = int(ntypes)
        self.eps, self.sigma, self.rcut = _d(eps).ravel(), _d(sigma).ravel(), _d(rcut).ravel()
        self.ron = self.rcut.copy() if ron is None else _d(ron).ravel()
        self.p2 = np.zeros_like(self.eps) if p2 is None else _d(p2).ravel()
        self.mode, self.pot = int(shift), self.POTS[pot]
        assert self.eps.size == self.sigma.size == self.rcut.size == self.ron.size == self.p2.size == self.ntypes ** 2

    @property
    def shift(self):
        """What the C sums take: cutoff treatment in the low two bits, the potential above them; the p2 table goes
        in through orc_set_p2 every time the value is read for a call."""
        lib().orc_set_p2(_ptr(self.p2), self.p2.size)
        return self.mode + 4 * self.pot

    @classmethod
    def of(cls, w):
        return cls(w.ntypes, w.eps, w.sigma, w.rcut, w.shift)


def cell_dim(L, r_max):
    return lib().orc_cell_dim(float(L), float(r_max))


def cell_index_f32(pos32, L, m):
    pos32 = np.ascontiguousarray(pos32, dtype=np.float32)
    out = np.empty(len(pos32), dtype=np.int32)
    lib().orc_cell_index_f32(pos32, len(pos32), float(L), int(m), out)
    return out


def cell_index_f64(pos, L, m):
    pos = _d(pos)
    out = np.empty(len(pos), dtype=np.int32)
    margin = np.empty(len(pos), dtype=np.float64)
    lib().orc_cell_index_f64(pos, len(pos), float(L), int(m), out, _ptr(margin))
    return out, margin


def build_cells(cell, m):
    cell = np.ascontiguousarray(cell, dtype=np.int32)
    start = np.empty(m ** 3 + 1, dtype=np.int64)
    members = np.empty(len(cell), dtype=np.int32)
    lib().orc_build_cells(cell, len(cell), int(m), start, members)
    return start, members


def _two_pass(call, nrows):
    count = np.empty(nrows, dtype=np.int32)
    _check(call(count, None, None), "nlist count")
    row_start = np.zeros(nrows + 1, dtype=np.int64)
    np.cumsum(count, out=row_start[1:])
    nbr = np.empty(max(int(row_start[-1]), 1), dtype=np.int32)
    _check(call(count, _ptr(row_start), _ptr(nbr)), "nlist fill")
    return count, row_start, nbr[: row_start[-1]]


def nlist_brute(pos, L, r_max):
    pos = _d(pos)
    return _two_pass(lambda c, r, n: lib().orc_nlist_brute(pos, len(pos), float(L), float(r_max), c, r, n), len(pos))


def nlist_brute_sample(pos, L, r_max, sample):
    pos = _d(pos)
    sample = np.ascontiguousarray(sample, dtype=np.int64)
    return _two_pass(lambda c, r, n: lib().orc_nlist_brute_sample(pos, len(pos), float(L), float(r_max),
                                                                  sample, len(sample), c, r, n), len(sample))


def nlist_cells(pos, L, r_max, m=None, cell=None):
    """Algorithm 2 + Algorithm 3.  cell defaults to the fp64 binning."""
    pos = _d(pos)
    m = cell_dim(L, r_max) if m is None else m
    if cell is None:
        cell, _ = cell_index_f64(pos, L, m)
    start, members = build_cells(cell, m)
    return _two_pass(lambda c, r, n: lib().orc_nlist_cells(pos, len(pos), float(L), float(r_max), int(m), cell,
                                                           start, members, c, r, n), len(pos))


def nlist_brute_typed(pos, typ, L, ntypes, rlist):
    """Definition of the list with per-type-pair list cutoffs rlist[ntypes*ntypes] (reading t1)."""
    pos, rlist = _d(pos), _d(rlist).ravel()
    typ = np.ascontiguousarray(typ, dtype=np.int32)
    return _two_pass(lambda c, r, n: lib().orc_nlist_brute_typed(pos, typ, len(pos), float(L), int(ntypes), rlist, c, r, n), len(pos))


def nlist_cells_typed(pos, typ, L, ntypes, rlist):
    """Algorithm 2 + 3 over the cells of the largest list cutoff, each pair tested against its own."""
    pos, rlist = _d(pos), _d(rlist).ravel()
    typ = np.ascontiguousarray(typ, dtype=np.int32)
    m = cell_dim(L, float(rlist.max()))
    cell, _ = cell_index_f64(pos, L, m)
    start, members = build_cells(cell, m)
    return _two_pass(lambda c, r, n: lib().orc_nlist_cells_typed(pos, typ, len(pos), float(L), int(ntypes), rlist, int(m), cell,
                                                                 start, members, c, r, n), len(pos))


def max_disp2(pos, pos_build, L):
    return lib().orc_max_disp2(_d(pos), _d(pos_build), len(pos), float(L))


def lj_pair(r, eps, sigma, r_cut, shift):
    V, f = C.c_double(), C.c_double()
    lib().orc_lj_pair(float(r), float(eps), float(sigma), float(r_cut), int(shift), C.byref(V), C.byref(f))
    return V.value, f.value


def pair_generic(pot, r, eps, sigma, p2, r_cut, r_on, mode):
    V, f = C.c_double(), C.c_double()
    lib().orc_pair_generic(Params.POTS[pot], float(r), float(eps), float(sigma), float(p2), float(r_cut), float(r_on), int(mode),
                           C.byref(V), C.byref(f))
    return V.value, f.value


def lj_pair_xplor(r, eps, sigma, r_cut, r_on):
    V, f = C.c_double(), C.c_double()
    lib().orc_lj_pair_xplor(float(r), float(eps), float(sigma), float(r_cut), float(r_on), C.byref(V), C.byref(f))
    return V.value, f.value


def compute_lj_brute(pos, typ, L, p: Params):
    pos, typ = _d(pos), np.ascontiguousarray(typ, dtype=np.int32)
    N = len(pos)
    F, U, W = np.empty((N, 3)), np.empty(N), np.empty((N, 6))
    _check(lib().orc_compute_lj_brute(pos, typ, N, float(L), p.ntypes, p.eps, p.sigma, p.rcut, p.ron, p.shift, F, U, W), "lj brute")
    return F, U, W


def compute_lj_brute_sample(pos, typ, L, p: Params, sample, band=0.0):
    pos, typ = _d(pos), np.ascontiguousarray(typ, dtype=np.int32)
    sample = np.ascontiguousarray(sample, dtype=np.int64)
    S = len(sample)
    F, U, W, A = np.empty((S, 3)), np.empty(S), np.empty((S, 6)), np.empty((S, 3))
    _check(lib().orc_compute_lj_brute_sample(pos, typ, len(pos), float(L), p.ntypes, p.eps, p.sigma, p.rcut, p.ron, p.shift,
                                             sample, S, float(band), F, U, W, _ptr(A)), "lj brute sample")
    return F, U, W, A


def compute_lj_nlist(pos, typ, L, p: Params, count, row_start, nbr, band=0.0):
    pos, typ = _d(pos), np.ascontiguousarray(typ, dtype=np.int32)
    N = len(pos)
    nbr = np.ascontiguousarray(nbr, dtype=np.int32)
    if nbr.size == 0:
        nbr = np.zeros(1, dtype=np.int32)
    F, U, W, A = np.empty((N, 3)), np.empty(N), np.empty((N, 6)), np.empty((N, 3))
    _check(lib().orc_compute_lj_nlist(pos, typ, N, float(L), p.ntypes, p.eps, p.sigma, p.rcut, p.ron, p.shift,
                                      np.ascontiguousarray(count, dtype=np.int32),
                                      np.ascontiguousarray(row_start, dtype=np.int64), nbr,
                                      float(band), F, U, W, _ptr(A)), "lj nlist")
    return F, U, W, A


class _Mass:
    """with _Mass(mass): ... -- the per-particle masses of the integrator calls inside (None: m = 1)."""

    def __init__(self, mass):
        self.m = None if mass is None else _d(mass).copy()

    def __enter__(self):
        lib().orc_set_mass(_ptr(self.m), 0 if self.m is None else len(self.m))

    def __exit__(self, *a):
        lib().orc_set_mass(None, 0)


def nve_step1(pos, vel, F, image, L, dt):
    """In place on float64 pos/vel and int32 image."""
    lib().orc_nve_step1(pos, vel, _d(F), image, len(pos), float(L), float(dt))


def nve_step2(vel, F, dt):
    lib().orc_nve_step2(vel, _d(F), len(vel), float(dt))


THERMO_FIELDS = ("K", "U", "Wxx", "Wxy", "Wxz", "Wyy", "Wyz", "Wzz", "P", "px", "py", "pz")


def thermo(vel, U, W, L, mass=None):
    out = np.empty(12)
    with _Mass(mass):
        lib().orc_thermo(_d(vel), _d(U), _d(W), len(vel), float(L), out)
    return dict(zip(THERMO_FIELDS, out))


def hilbert_key(ix, iy, iz, B):
    return lib().orc_hilbert_key(int(ix), int(iy), int(iz), int(B))


def sfc_keys(pos32, L, B=8):
    pos32 = np.ascontiguousarray(pos32, dtype=np.float32)
    key = np.empty(len(pos32), dtype=np.uint32)
    lib().orc_sfc_keys(pos32, len(pos32), float(L), int(B), key)
    return key


def sort_perm(key, B=8):
    key = np.ascontiguousarray(key, dtype=np.uint32)
    perm = np.empty(len(key), dtype=np.int64)
    _check(lib().orc_sort_perm(key, len(key), int(B), perm), "sort_perm")
    return perm


def run_nve(pos, vel, image, typ, L, p: Params, r_buff, dt, nsteps, forces=None, log=False, mass=None):
    """Whole loop; returns dict(pos, vel, image, F, U, W, KU, builds, max_nbrs)."""
    pos, vel = _d(pos).copy(), _d(vel).copy()
    image = np.ascontiguousarray(image, dtype=np.int32).copy()
    typ = np.ascontiguousarray(typ, dtype=np.int32)
    N = len(pos)
    if forces is None:
        F, U, W, have = np.zeros((N, 3)), np.zeros(N), np.zeros((N, 6)), 0
    else:
        F, U, W = (_d(x).copy() for x in forces)
        have = 1
    KU = np.zeros((nsteps + 1, 2)) if log else None
    stats = np.zeros(2, dtype=np.int64)
    with _Mass(mass):
        _check(lib().orc_run_nve(pos, vel, image, typ, N, float(L), p.ntypes, p.eps, p.sigma, p.rcut, p.ron, p.shift,
                                 float(r_buff), float(dt), int(nsteps), have, F, U, W, _ptr(KU), _ptr(stats)), "run_nve")
    return dict(pos=pos, vel=vel, image=image, F=F, U=U, W=W, KU=KU, builds=int(stats[0]), max_nbrs=int(stats[1]))


def counter_u64(seed, stream, index):
    return int(lib().orc_counter_u64(int(seed), int(stream), int(index)))


def uniform_pm1(seed, stream, index):
    return lib().orc_uniform_pm1(int(seed), int(stream), int(index))


def _run_thermostat(mode, pos, vel, image, typ, L, p, r_buff, dt, nsteps, T, par, seed, state, forces, log, mass=None):
    pos, vel = _d(pos).copy(), _d(vel).copy()
    image = np.ascontiguousarray(image, dtype=np.int32).copy()
    typ = np.ascontiguousarray(typ, dtype=np.int32)
    N = len(pos)
    if forces is None:
        F, U, W, have = np.zeros((N, 3)), np.zeros(N), np.zeros((N, 6)), 0
    else:
        F, U, W = (_d(x).copy() for x in forces)
        have = 1
    lg = np.zeros((nsteps + 1, 4)) if log else None
    stats = np.zeros(2, dtype=np.int64)
    st = np.array(state, dtype=np.float64)
    with _Mass(mass):
        _check(lib().orc_run_thermostat(mode, pos, vel, image, typ, N, float(L), p.ntypes, p.eps, p.sigma, p.rcut, p.ron, p.shift,
                                        float(r_buff), float(dt), int(nsteps), float(T), float(par), int(seed), st, have,
                                        F, U, W, _ptr(lg), _ptr(stats)), "run_thermostat")
    return dict(pos=pos, vel=vel, image=image, F=F, U=U, W=W, log=lg, state=st, builds=int(stats[0]))


def run_nvt(pos, vel, image, typ, L, p: Params, r_buff, dt, nsteps, T, tau, xi=0.0, eta=0.0, forces=None, log=False, mass=None):
    """Nose-Hoover (reading n1); returns dict(pos, vel, image, F, U, W, log[K, U, xi, eta], state=[xi, eta])."""
    return _run_thermostat(1, pos, vel, image, typ, L, p, r_buff, dt, nsteps, T, tau, 0, [xi, eta], forces, log, mass)


def run_langevin(pos, vel, image, typ, L, p: Params, r_buff, dt, nsteps, T, gamma, seed, step0=0, forces=None, log=False, mass=None):
    """Langevin (reading n2); state[0] = number of the next time step."""
    return _run_thermostat(2, pos, vel, image, typ, L, p, r_buff, dt, nsteps, T, gamma, seed, [float(step0), 0.0], forces, log, mass)


def num_threads():
    return lib().orc_num_threads()
