"""Thin ctypes binding of libhb (include/hb.h): same names, argument marshalling
only -- every step of the path runs in the CUDA kernels of csrc/.

There is NO CPU fallback: if libhb.so is missing or no CUDA device is present,
the calls raise.  Arrays may be numpy (host pointers, copied by the library) or
torch CUDA tensors (device pointers, used in place).  PyTorch is used only for
device memory and streams: `System(..., use_torch_allocator=True)` makes the
library allocate through torch's caching allocator, and work is enqueued on
torch's current CUDA stream.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhb.so")

HB_OK, HB_EINVAL, HB_ECUDA, HB_ENOMEM, HB_EBOX, HB_ESTATE, HB_ENAN = 0, -1, -2, -3, -4, -5, -6
HB_SHIFT_NONE, HB_SHIFT_ENERGY, HB_XPLOR = 0, 1, 2
HB_POT_LJ, HB_POT_GAUSS, HB_POT_YUKAWA, HB_POT_MORSE = 0, 1, 2, 3
POTS = {"lj": HB_POT_LJ, "gauss": HB_POT_GAUSS, "yukawa": HB_POT_YUKAWA, "morse": HB_POT_MORSE}
THERMO_STATIC_MAX_N = 16_777_216   # HB_THERMO_STATIC_MAX_N
_ERR_NAMES = {-1: "HB_EINVAL", -2: "HB_ECUDA", -3: "HB_ENOMEM", -4: "HB_EBOX", -5: "HB_ESTATE", -6: "HB_ENAN"}

EXPORTS = ["hb_create", "hb_destroy", "hb_set_state", "hb_get_state", "hb_set_state_f64", "hb_get_state_f64", "hb_get_forces_f64", "hb_set_rcut_pair", "hb_set_ron_pair",
           "hb_set_pair_potential", "hb_set_mass", "hb_get_mass", "hb_build_cells",
           "hb_build_nlist", "hb_needs_rebuild", "hb_compute_lj", "hb_step_nve", "hb_run_nve", "hb_run_nvt", "hb_run_langevin",
           "hb_get_thermostat", "hb_set_thermostat", "hb_sort",
           "hb_thermo", "hb_thermo_static", "hb_get_cells", "hb_get_nlist", "hb_get_forces", "hb_stats", "hb_set_tunable",
           "hb_get_tunable", "hb_time_stage", "hb_measure_peak", "hb_last_error", "hb_version"]


class HBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class hb_allocator(C.Structure):
    _fields_ = [("alloc", C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)),
                ("free", C.CFUNCTYPE(None, C.c_void_p, C.c_void_p, C.c_void_p)),
                ("user", C.c_void_p)]


class hb_thermo_t(C.Structure):
    _fields_ = [("K", C.c_double), ("U", C.c_double), ("W", C.c_double * 6), ("P", C.c_double),
                ("px", C.c_double), ("py", C.c_double), ("pz", C.c_double)]


class hb_stats_t(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("steps", "rebuilds", "sorts", "overflow_retries", "max_nbrs", "row_pitch",
                                         "cells_per_axis", "graph_launches", "kernel_launches", "graph_builds")]


_lib = None


def load():
    """dlopen libhb.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1308_5587_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    L.hb_create.argtypes = [C.POINTER(vp), i64, dbl, i32, vp, vp, vp, vp]
    L.hb_destroy.argtypes = [vp]
    L.hb_set_state.argtypes = [vp, vp, vp, vp, vp, i32]
    L.hb_get_state.argtypes = [vp, vp, vp, vp, vp, vp, i32]
    L.hb_set_state_f64.argtypes = [vp, vp, vp, vp, vp, i32]
    L.hb_get_state_f64.argtypes = [vp, vp, vp, vp, i32]
    L.hb_get_forces_f64.argtypes = [vp, vp, vp, i32]
    L.hb_set_rcut_pair.argtypes = [vp, vp]
    L.hb_set_ron_pair.argtypes = [vp, vp]
    L.hb_set_pair_potential.argtypes = [vp, i32, vp]
    L.hb_set_mass.argtypes = [vp, vp, i32]
    L.hb_get_mass.argtypes = [vp, vp, i32]
    L.hb_build_cells.argtypes = [vp]
    L.hb_build_nlist.argtypes = [vp, dbl, dbl]
    L.hb_needs_rebuild.argtypes = [vp, C.POINTER(i32)]
    L.hb_compute_lj.argtypes = [vp, i32]
    L.hb_step_nve.argtypes = [vp, dbl]
    L.hb_run_nve.argtypes = [vp, dbl, i64, i64]
    L.hb_run_nvt.argtypes = [vp, dbl, i64, i64, dbl, dbl]
    L.hb_run_langevin.argtypes = [vp, dbl, i64, i64, dbl, dbl, C.c_uint64]
    L.hb_get_thermostat.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i64)]
    L.hb_set_thermostat.argtypes = [vp, dbl, dbl, i64]
    L.hb_sort.argtypes = [vp]
    L.hb_thermo.argtypes = [vp, C.POINTER(hb_thermo_t)]
    L.hb_thermo_static.argtypes = [vp, vp, vp, vp, i64, dbl, vp, vp, C.c_char_p, C.c_size_t]
    L.hb_get_cells.argtypes = [vp, vp, vp, vp, i32]
    L.hb_get_nlist.argtypes = [vp, vp, vp, i32]
    L.hb_get_forces.argtypes = [vp, vp, vp, i32]
    L.hb_stats.argtypes = [vp, C.POINTER(hb_stats_t)]
    L.hb_set_tunable.argtypes = [vp, C.c_char_p, i32]
    L.hb_get_tunable.argtypes = [vp, C.c_char_p, C.POINTER(i32)]
    L.hb_time_stage.argtypes = [vp, C.c_char_p, i32, i64, C.POINTER(dbl)]
    L.hb_measure_peak.argtypes = [vp, C.c_char_p, C.POINTER(dbl)]
    L.hb_last_error.argtypes = [vp]
    L.hb_last_error.restype = C.c_char_p
    L.hb_version.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("hb_last_error", "hb_version"):
            getattr(L, name).restype = i32
    _lib = L
    return L


def _is_torch(a):
    return a is not None and type(a).__module__.startswith("torch")


def _ptr(a, dtype):
    """(pointer, on_device) of a numpy array or a torch CUDA tensor; None -> NULL."""
    if a is None:
        return None, None
    if _is_torch(a):
        import torch
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int32: torch.int32, np.uint32: torch.int32, np.int64: torch.int64}[dtype]
        if a.dtype != want or not a.is_contiguous() or not a.is_cuda:
            raise TypeError(f"torch argument must be a contiguous CUDA tensor of {want}")
        return C.c_void_p(a.data_ptr()), 1
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise TypeError(f"numpy argument must be C-contiguous {np.dtype(dtype)}")
    return a.ctypes.data_as(C.c_void_p), 0


def _where(*flags):
    s = {f for f in flags if f is not None}
    if len(s) > 1:
        raise TypeError("all arrays of one call must live on the same side (host or device)")
    return s.pop() if s else 0


class System:
    """One hb_system handle.  Methods are the C calls without the `hb_` prefix."""

    def __init__(self, N, L, ntypes=1, eps=(1.0,), sigma=(1.0,), stream=None, use_torch_allocator=False):
        self._lib = load()
        self._h = C.c_void_p()
        self.N, self.L, self.ntypes = int(N), float(L), int(ntypes)
        eps = np.ascontiguousarray(eps, dtype=np.float64).ravel()
        sigma = np.ascontiguousarray(sigma, dtype=np.float64).ravel()
        if eps.size != ntypes * ntypes or sigma.size != ntypes * ntypes:
            raise ValueError("eps and sigma must have ntypes*ntypes entries")
        if stream is None:
            try:
                import torch
                if torch.cuda.is_available():
                    stream = torch.cuda.current_stream().cuda_stream
            except ImportError:
                stream = None
        self._alloc = None
        alloc_ptr = None
        if use_torch_allocator:
            import torch
            dev = torch.cuda.current_device()

            def _alloc(nbytes, strm, user):
                return torch.cuda.caching_allocator_alloc(int(nbytes), dev, strm or 0)

            def _free(ptr, strm, user):
                torch.cuda.caching_allocator_delete(ptr)

            self._alloc = hb_allocator(hb_allocator._fields_[0][1](_alloc), hb_allocator._fields_[1][1](_free), None)
            alloc_ptr = C.cast(C.pointer(self._alloc), C.c_void_p)
        rc = self._lib.hb_create(C.byref(self._h), self.N, self.L, self.ntypes, eps.ctypes.data_as(C.c_void_p),
                                 sigma.ctypes.data_as(C.c_void_p), C.c_void_p(stream or 0), alloc_ptr)
        if rc != HB_OK:
            msg = self._lib.hb_last_error(self._h).decode() if self._h else "hb_create failed"
            if self._h:
                self._lib.hb_destroy(self._h)
                self._h = C.c_void_p()
            raise HBError(rc, msg)

    @classmethod
    def from_workload(cls, w, **kw):
        s = cls(w.N, w.L, w.ntypes, w.eps, w.sigma, **kw)
        s.set_rcut_pair(w.rcut)
        return s

    def _ck(self, rc):
        if rc != HB_OK:
            raise HBError(rc, self._lib.hb_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.hb_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- state ----
    def set_state(self, pos, type=None, vel=None, image=None):
        if vel is None:
            vel = np.zeros((self.N, 3), dtype=np.float32) if not _is_torch(pos) else pos.new_zeros((self.N, 3))
        p, d1 = _ptr(pos, np.float32)
        t, d2 = _ptr(type, np.int32)
        v, d3 = _ptr(vel, np.float32)
        im, d4 = _ptr(image, np.int32)
        self._ck(self._lib.hb_set_state(self._h, p, t, v, im, _where(d1, d2, d3, d4)))

    def get_state(self, device=False):
        """dict(pos, type, vel, image, order) BY TAG; numpy, or torch CUDA tensors if device."""
        N = self.N
        if device:
            import torch
            o = dict(pos=torch.empty((N, 3), dtype=torch.float32, device="cuda"),
                     type=torch.empty(N, dtype=torch.int32, device="cuda"),
                     vel=torch.empty((N, 3), dtype=torch.float32, device="cuda"),
                     image=torch.empty((N, 3), dtype=torch.int32, device="cuda"),
                     order=torch.empty(N, dtype=torch.int32, device="cuda"))
            ptrs = [C.c_void_p(o[k].data_ptr()) for k in ("pos", "type", "vel", "image", "order")]
        else:
            o = dict(pos=np.empty((N, 3), np.float32), type=np.empty(N, np.int32), vel=np.empty((N, 3), np.float32),
                     image=np.empty((N, 3), np.int32), order=np.empty(N, np.uint32))
            ptrs = [o[k].ctypes.data_as(C.c_void_p) for k in ("pos", "type", "vel", "image", "order")]
        self._ck(self._lib.hb_get_state(self._h, *ptrs, 1 if device else 0))
        return o

    def get_state_into(self, pos=None, type=None, vel=None, image=None, order=None):
        p, d1 = _ptr(pos, np.float32)
        t, d2 = _ptr(type, np.int32)
        v, d3 = _ptr(vel, np.float32)
        im, d4 = _ptr(image, np.int32)
        o, d5 = _ptr(order, np.uint32)
        self._ck(self._lib.hb_get_state(self._h, p, t, v, im, o, _where(d1, d2, d3, d4, d5)))

    # ---- the binary64 variant (tunable precision = 64) ----
    def set_state_f64(self, pos, type=None, vel=None, image=None):
        if vel is None:
            vel = np.zeros((self.N, 3), dtype=np.float64)
        p, d1 = _ptr(pos, np.float64)
        t, d2 = _ptr(type, np.int32)
        v, d3 = _ptr(vel, np.float64)
        im, d4 = _ptr(image, np.int32)
        self._ck(self._lib.hb_set_state_f64(self._h, p, t, v, im, _where(d1, d2, d3, d4)))

    def get_state_f64(self):
        """dict(pos, vel float64 [N][3], image int32 [N][3]) BY TAG."""
        o = dict(pos=np.empty((self.N, 3), np.float64), vel=np.empty((self.N, 3), np.float64), image=np.empty((self.N, 3), np.int32))
        self._ck(self._lib.hb_get_state_f64(self._h, *(o[k].ctypes.data_as(C.c_void_p) for k in ("pos", "vel", "image")), 0))
        return o

    def get_forces_f64(self, virial=True):
        """(F_xyz_U float64[N][4], W float64[N][6] or None) BY TAG, of the binary64 sums."""
        f = np.empty((self.N, 4), np.float64)
        w = np.empty((self.N, 6), np.float64) if virial else None
        self._ck(self._lib.hb_get_forces_f64(self._h, f.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p) if virial else None, 0))
        return f, w

    # ---- the hot path ----
    def set_rcut_pair(self, rcut):
        rcut = np.ascontiguousarray(rcut, dtype=np.float64).ravel()
        if rcut.size != self.ntypes ** 2:
            raise ValueError("rcut must have ntypes*ntypes entries")
        self._ck(self._lib.hb_set_rcut_pair(self._h, rcut.ctypes.data_as(C.c_void_p)))

    def set_ron_pair(self, ron):
        ron = np.ascontiguousarray(ron, dtype=np.float64).ravel()
        if ron.size != self.ntypes ** 2:
            raise ValueError("ron must have ntypes*ntypes entries")
        self._ck(self._lib.hb_set_ron_pair(self._h, ron.ctypes.data_as(C.c_void_p)))

    def set_pair_potential(self, pot, p2=None):
        """pot: HB_POT_* or one of "lj", "gauss", "yukawa", "morse"; p2: third parameter table (Morse r0)."""
        pot = POTS[pot] if isinstance(pot, str) else int(pot)
        ptr = None
        if p2 is not None:
            p2 = np.ascontiguousarray(p2, dtype=np.float64).ravel()
            if p2.size != self.ntypes ** 2:
                raise ValueError("p2 must have ntypes*ntypes entries")
            ptr = p2.ctypes.data_as(C.c_void_p)
        self._ck(self._lib.hb_set_pair_potential(self._h, pot, ptr))

    def set_mass(self, mass):
        m, d = _ptr(mass, np.float32)
        self._ck(self._lib.hb_set_mass(self._h, m, d))

    def get_mass(self):
        m = np.empty(self.N, np.float32)
        self._ck(self._lib.hb_get_mass(self._h, m.ctypes.data_as(C.c_void_p), 0))
        return m

    def build_cells(self):
        self._ck(self._lib.hb_build_cells(self._h))

    def build_nlist(self, r_cut, r_buff):
        self._ck(self._lib.hb_build_nlist(self._h, float(r_cut), float(r_buff)))

    def needs_rebuild(self):
        need = C.c_int()
        self._ck(self._lib.hb_needs_rebuild(self._h, C.byref(need)))
        return bool(need.value)

    def compute_lj(self, shift_mode=HB_SHIFT_ENERGY):
        self._ck(self._lib.hb_compute_lj(self._h, int(shift_mode)))

    def step_nve(self, dt):
        self._ck(self._lib.hb_step_nve(self._h, float(dt)))

    def run_nve(self, dt, nsteps, sort_period=0):
        self._ck(self._lib.hb_run_nve(self._h, float(dt), int(nsteps), int(sort_period)))

    def run_nvt(self, dt, nsteps, T, tau, sort_period=0):
        self._ck(self._lib.hb_run_nvt(self._h, float(dt), int(nsteps), int(sort_period), float(T), float(tau)))

    def run_langevin(self, dt, nsteps, T, gamma, seed, sort_period=0):
        self._ck(self._lib.hb_run_langevin(self._h, float(dt), int(nsteps), int(sort_period), float(T), float(gamma), int(seed)))

    def get_thermostat(self):
        xi, eta, n = C.c_double(), C.c_double(), C.c_int64()
        self._ck(self._lib.hb_get_thermostat(self._h, C.byref(xi), C.byref(eta), C.byref(n)))
        return dict(xi=xi.value, eta=eta.value, langevin_steps=n.value)

    def set_thermostat(self, xi=0.0, eta=0.0, langevin_steps=0):
        self._ck(self._lib.hb_set_thermostat(self._h, float(xi), float(eta), int(langevin_steps)))

    def sort(self):
        self._ck(self._lib.hb_sort(self._h))

    def thermo(self):
        t = hb_thermo_t()
        self._ck(self._lib.hb_thermo(self._h, C.byref(t)))
        return dict(K=t.K, U=t.U, W=list(t.W), P=t.P, px=t.px, py=t.py, pz=t.pz)

    @staticmethod
    def thermo_static(vel, mass, f_xyz_u, virial6, L, out, stream=None):
        """hb_thermo_static: the sums of thermo() from the caller's own CUDA tensors, for callers that must not
        allocate device memory (include/hb.h says who and why).  No handle is involved.  vel float32 [N][3];
        mass [N], f_xyz_u [N][4], virial6 [N][6] float32 or None; out: a CUDA float64 tensor of 12 elements that
        receives (K, U, W[6], P, px, py, pz) once the two kernels enqueued on `stream` (default: torch's current
        stream) have run -- this call does not wait for them.  N <= THERMO_STATIC_MAX_N."""
        lib = load()
        N = int(vel.shape[0])
        ptrs = []
        for a in (vel, mass, f_xyz_u, virial6):
            p, d = _ptr(a, np.float32)
            if d == 0:
                raise TypeError("hb_thermo_static takes device arrays (torch CUDA tensors) only")
            ptrs.append(p)
        o, d = _ptr(out, np.float64)
        if d != 1 or out.numel() != 12:
            raise TypeError("out must be a CUDA float64 tensor of 12 elements")
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        err = C.create_string_buffer(512)
        rc = lib.hb_thermo_static(*ptrs, N, float(L), o, C.c_void_p(stream or 0), err, len(err))
        if rc != HB_OK:
            raise HBError(rc, err.value.decode())

    # ---- accessors (BY TAG) ----
    def get_cells(self):
        """(m, cell_start int32[m^3+1], cell_tags uint32[N])."""
        m3 = np.empty(3, np.int32)
        self._ck(self._lib.hb_get_cells(self._h, m3.ctypes.data_as(C.c_void_p), None, None, 0))
        m = int(m3[0])
        start = np.empty(m ** 3 + 1, np.int32)
        tags = np.empty(self.N, np.uint32)
        self._ck(self._lib.hb_get_cells(self._h, None, start.ctypes.data_as(C.c_void_p), tags.ctypes.data_as(C.c_void_p), 0))
        return m, start, tags

    def get_nlist(self):
        """(row_start int64[N+1], nbr_tags uint32[row_start[N]]) BY TAG."""
        rs = np.empty(self.N + 1, np.int64)
        self._ck(self._lib.hb_get_nlist(self._h, rs.ctypes.data_as(C.c_void_p), None, 0))
        nbr = np.empty(max(int(rs[-1]), 1), np.uint32)
        self._ck(self._lib.hb_get_nlist(self._h, rs.ctypes.data_as(C.c_void_p), nbr.ctypes.data_as(C.c_void_p), 0))
        return rs, nbr[: rs[-1]]

    def get_nlist_sizes(self):
        """row_start int64[N+1] BY TAG without the entries."""
        rs = np.empty(self.N + 1, np.int64)
        self._ck(self._lib.hb_get_nlist(self._h, rs.ctypes.data_as(C.c_void_p), None, 0))
        return rs

    def get_forces(self, virial=True):
        """(F_xyz_U float32[N][4], W float32[N][6] or None) BY TAG."""
        f = np.empty((self.N, 4), np.float32)
        w = np.empty((self.N, 6), np.float32) if virial else None
        self._ck(self._lib.hb_get_forces(self._h, f.ctypes.data_as(C.c_void_p),
                                         w.ctypes.data_as(C.c_void_p) if virial else None, 0))
        return f, w

    def stats(self):
        s = hb_stats_t()
        self._ck(self._lib.hb_stats(self._h, C.byref(s)))
        return {n: getattr(s, n) for n, _ in hb_stats_t._fields_}

    def time_stage(self, stage, reps=20, flush_l2_bytes=0):
        """Mean milliseconds per launch of one stage (CUDA events on the system's stream)."""
        ms = C.c_double()
        self._ck(self._lib.hb_time_stage(self._h, stage.encode(), int(reps), int(flush_l2_bytes), C.byref(ms)))
        return ms.value

    def measure_peak(self, which):
        """Measured roofline denominator: "fp32_tflops", "l2_gbs" or "smem_gbs"."""
        v = C.c_double()
        self._ck(self._lib.hb_measure_peak(self._h, which.encode(), C.byref(v)))
        return v.value

    def set_tunable(self, name, value):
        self._ck(self._lib.hb_set_tunable(self._h, name.encode(), int(value)))

    def get_tunable(self, name):
        v = C.c_int()
        self._ck(self._lib.hb_get_tunable(self._h, name.encode(), C.byref(v)))
        return v.value


def version():
    return load().hb_version().decode()
