"""hb_thermo_static -- the thermodynamic sums for callers that cannot allocate device memory -- against hb_thermo.

Some users of this library run where device allocation is off the table: the whole GPU was given to a memory pool
at start-up (so cudaMalloc can fail, or is forbidden by the host program's rules), or they are a logging / analysis
hook inside someone else's time-step loop, which a cudaMalloc or cudaFree would stall because both synchronise the
device.  They cannot call hb_create (it allocates every array of a system) and therefore not hb_thermo either.
hb_thermo_static is the one entry point for them: no handle, the caller's own device arrays in, one hb_thermo_t
out, and the partial sums of the reduction in a fixed 360,448-byte array that is part of the library image
(include/hb.h, "hb_thermo_static", has the contract: limit of 16,777,216 particles, one array per GPU shared by all
calls, first call per device does the address look-up).

What is checked here: on the same per-particle arrays the new entry point reports the same K, U, W, P and momentum as
the existing path (hb_thermo on a handle), to the 1e-12 relative agreement the other tests ask of binary64 sums --
the two add the same binary32 terms in binary64, only in a different order.  The calls are made back to back, a
large system, then a small one, then the large one again after it has moved, because every call reuses the one
array and finds in it whatever the previous call left: a result that depended on stale partial sums, or on the
array starting out as zeros, would show up in the second or third call.

This file sorts last on purpose (pytest -x stops at the first failure; a problem here must not hide the other
tests), and it has to pass both on its own in a fresh process and after everything else has run.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1308_5587_b200 import workloads as wl

REL = 1e-12     # the agreement tests/test_gpu_parity.py asks of K (binary64 sums of the same binary32 terms)


@pytest.fixture(scope="module")
def hb():
    from paper_1308_5587_b200 import hb as _hb
    _hb.load()
    return _hb


def _device_arrays(g):
    """The caller's side: its own device arrays, in the layouts the accessors write (by tag)."""
    import torch
    st = g.get_state()
    f4, w6 = g.get_forces()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return dev(st["vel"]), dev(g.get_mass()), dev(f4), dev(w6)


def _check(hb, g, L, with_mass=True):
    """One hb_thermo_static call on the arrays of g, compared with g.thermo()."""
    import torch
    ref = g.thermo()                                   # the existing path: reads the handle's arrays
    vel, mass, f4, w6 = _device_arrays(g)
    out = torch.full((12,), float("nan"), dtype=torch.float64, device="cuda")
    hb.System.thermo_static(vel, mass if with_mass else None, f4, w6, L, out)
    got = out.cpu().numpy()                            # orders the read after the two kernels (same stream)
    assert np.isfinite(got).all(), got

    # Sums with cancellation (momentum, off-diagonal virial) are compared on the scale of their terms.
    v = vel.cpu().numpy().astype(np.float64)
    m = mass.cpu().numpy().astype(np.float64) if with_mass else np.ones(len(v))
    w = w6.cpu().numpy().astype(np.float64)
    u = f4.cpu().numpy().astype(np.float64)[:, 3]
    k_scale = (0.5 * m * (v * v).sum(axis=1)).sum()
    assert abs(got[0] - ref["K"]) <= REL * k_scale
    assert abs(got[1] - ref["U"]) <= REL * np.abs(u).sum()
    for c in range(6):
        assert abs(got[2 + c] - ref["W"][c]) <= REL * np.abs(w[:, c]).sum(), c
    p_scale = (2.0 * k_scale + np.abs(w[:, [0, 3, 5]]).sum()) / (3.0 * L ** 3)
    assert abs(got[8] - ref["P"]) <= REL * p_scale
    for c, key in enumerate(("px", "py", "pz")):
        assert abs(got[9 + c] - ref[key]) <= REL * np.abs(m * v[:, c]).sum(), key
    return got


@pytest.mark.gpu
def test_thermo_static_matches_hb_thermo_call_after_call(hb):
    big = wl.scaled(wl.CONFIGS["lj_64k"], 19_683)      # 27^3: four full blocks of 4096 particles and a ragged fifth
    small = wl.CONFIGS["lj_1k"]                        # one partly filled block
    sb, ss = wl.make_state(big), wl.make_state(small)
    masses = (0.5 + 1.5 * wl.counter_uniform(7, 3, np.arange(big.N))).astype(np.float32)
    with hb.System.from_workload(big) as gb, hb.System.from_workload(small) as gs:
        gb.set_state(sb.pos, sb.type, sb.vel, sb.image)
        gb.set_mass(masses)
        gb.build_nlist(0.0, big.r_buff)
        gb.compute_lj(big.shift)
        gs.set_state(ss.pos, ss.type, ss.vel, ss.image)
        gs.build_nlist(0.0, small.r_buff)
        gs.compute_lj(small.shift)

        first = _check(hb, gb, sb.L)                   # call 1: five blocks' partial sums land in the shared array
        _check(hb, gs, ss.L, with_mass=False)          # call 2: one block; the other four still hold call 1's sums
        gb.run_nve(big.dt, 25, 0)                      # the large system moves on, so call 3 has new answers
        third = _check(hb, gb, sb.L)                   # call 3: over call 2's leftovers
        assert third[0] != first[0] and third[1] != first[1]     # really a new state, not a replay of call 1


@pytest.mark.gpu
def test_thermo_static_optional_inputs(hb):
    """mass = NULL means unit masses, f_xyz_u / virial6 = NULL report U = 0 and W = 0 (P is then 2K / 3V)."""
    import torch
    w = wl.CONFIGS["lj_1k"]
    s = wl.make_state(w)
    vel = torch.from_numpy(s.vel).cuda()
    out = torch.empty(12, dtype=torch.float64, device="cuda")
    hb.System.thermo_static(vel, None, None, None, s.L, out)
    got = out.cpu().numpy()
    v = s.vel.astype(np.float64)
    K = 0.5 * (v * v).sum()
    assert abs(got[0] - K) <= REL * K
    assert got[1] == 0.0 and (got[2:8] == 0.0).all()
    assert abs(got[8] - 2.0 * K / (3.0 * s.L ** 3)) <= REL * K
    assert np.abs(got[9:12] - v.sum(axis=0)).max() <= REL * np.abs(v).sum()


def test_thermo_static_refuses_more_particles_than_the_fixed_array_serves(hb):
    """Over the limit the call must say so and launch nothing (so this needs no GPU: no pointer is touched)."""
    lib = hb.load()
    dummy = (C.c_float * 4)()
    out = (C.c_double * 12)()
    err = C.create_string_buffer(512)
    too_many = hb.THERMO_STATIC_MAX_N + 1
    rc = lib.hb_thermo_static(C.cast(dummy, C.c_void_p), None, None, None, too_many, 10.0,
                              C.cast(out, C.c_void_p), None, err, len(err))
    assert rc == hb.HB_EINVAL
    msg = err.value.decode()
    assert str(hb.THERMO_STATIC_MAX_N) in msg and str(too_many) in msg and "HB_THERMO_STATIC_MAX_N" in msg
    for bad_n in (0, -5):
        assert lib.hb_thermo_static(C.cast(dummy, C.c_void_p), None, None, None, bad_n, 10.0,
                                    C.cast(out, C.c_void_p), None, err, len(err)) == hb.HB_EINVAL
    assert lib.hb_thermo_static(None, None, None, None, 10, 10.0, C.cast(out, C.c_void_p), None, None, 0) == hb.HB_EINVAL


def test_header_limit_and_binding_limit_agree():
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    text = open(os.path.join(root, "include", "hb.h")).read()
    from paper_1308_5587_b200 import hb as _hb
    assert int(re.search(r"#define HB_THERMO_STATIC_MAX_N (\d+)", text).group(1)) == _hb.THERMO_STATIC_MAX_N
