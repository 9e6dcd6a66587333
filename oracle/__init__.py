"""fp64 CPU oracle for the short-range PP path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It never imports
`paper_1411_3396_b200` (the CUDA path) and shares no code with it; the only
common module is the seeded input generator, which holds no arithmetic of
the method.

The arithmetic lives in `srpp_oracle.c` (plain C, fp64, OpenMP over targets;
see its header for the passages of PAPER.md / readings of SURVEY.md 8(c) it
follows).  This file only marshals numpy arrays into it through ctypes.
`default_poly.py` re-derives the default polynomial coefficients (SURVEY.md
Appendix A).

Pins (tests/test_oracle_pins.py): P1 two-particle closed form, P2 zero beyond
the cutoff, P3 unit lattice (122 neighbours, zero net force), P4 momentum
conservation, P5 8-particle worked example, P6 brute force vs cell list,
P7 config-1 soft pins, P8 binning worked example, P9/P10 coefficient table,
P11 permutation invariance; the R9 allowance band (constructed near-cutoff
neighbours), the R18 metric (hand-computed vectors) and the sub-cycle
`orc_subcycle` (two-particle step worked by hand from P1's printed values,
composition, momentum, time reversal).  Unpinned: fidelity of the DEFAULT polynomial to
the real HACC grid force ("parity unpinned": PAPER.md prints nothing to
compare with; both sides take poly[6] as data, so GPU-vs-oracle parity does
not depend on it).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "srpp_oracle.c")
_LIB = os.path.join(_HERE, "libsrpp_oracle.so")

# SURVEY.md Appendix A, fp32 bit patterns of c0..c5 (re-derived by default_poly.py, pin P10)
DEFAULT_POLY_BITS = (0x3EDEAD5D, 0xBE36288A, 0x3D2403BC, 0xBBB0860A, 0x39CFCFAA, 0xB74AC976)
DEFAULT_POLY = np.array(DEFAULT_POLY_BITS, dtype=np.uint32).view(np.float32)


class Params(C.Structure):
    _fields_ = [("box", C.c_float * 3), ("rcut", C.c_float), ("eps", C.c_float), ("poly", C.c_float * 6),
                ("periodic", C.c_int32 * 3)]


def make_params(box, rcut=3.0, eps=0.1, poly=None, periodic=(1, 1, 1)) -> Params:
    """periodic[a] = 0 makes axis a open: plain coordinate differences, no neighbours across the faces (the
    overloaded node volume of PAPER.md:65); the default is the periodic box of BASELINE.json."""
    p = Params()
    for a in range(3):
        p.periodic[a] = 1 if periodic[a] else 0
    for a in range(3):
        p.box[a] = float(box[a])
    p.rcut = float(rcut)
    p.eps = float(eps)
    poly = DEFAULT_POLY if poly is None else np.asarray(poly, dtype=np.float32)
    for k in range(6):
        p.poly[k] = float(poly[k])
    return p


def build(force: bool = False) -> str:
    """Compile srpp_oracle.c -> libsrpp_oracle.so with gcc (fp contraction off, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        f32p, u32p = C.POINTER(C.c_float), C.POINTER(C.c_uint32)
        f64p, i64p, i32p = C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_int32)
        L.orc_num_threads.restype = C.c_int32
        L.orc_cell_ids.restype = C.c_int32
        L.orc_cell_ids.argtypes = [f32p, C.c_int64, f32p, i32p, u32p]
        L.orc_build_mesh.restype = C.c_int32
        L.orc_build_mesh.argtypes = [f32p, C.c_int64, f32p, i32p, u32p, u32p, f32p]
        L.orc_pair_factor.restype = C.c_double
        L.orc_pair_factor.argtypes = [C.POINTER(Params), C.c_double]
        L.orc_poly.restype = C.c_double
        L.orc_poly.argtypes = [C.POINTER(Params), C.c_double]
        L.orc_accel_bruteforce.restype = None
        L.orc_accel_bruteforce.argtypes = [f32p, C.c_int64, C.POINTER(Params), f64p, i64p, f64p]
        L.orc_accel.restype = C.c_int32
        L.orc_accel.argtypes = [f32p, C.c_int64, C.POINTER(Params), i64p, C.c_int64, f64p, i64p, f64p,
                                f64p, i64p]
        L.orc_kick.restype = None
        L.orc_kick.argtypes = [f32p, f32p, C.c_float, C.c_int64]
        L.orc_stream.restype = None
        L.orc_stream.argtypes = [f32p, f32p, C.c_float, f32p, C.c_int64]
        L.orc_subcycle.restype = C.c_int32
        L.orc_subcycle.argtypes = [f32p, f32p, C.c_int64, C.POINTER(Params), C.c_float, C.c_float, C.c_int32, f32p]
        L.orc_mbp.restype = None
        L.orc_mbp.argtypes = [f32p, C.c_int64, C.POINTER(C.c_int64), C.c_int64, C.c_float, C.POINTER(C.c_double),
                              C.POINTER(C.c_int64)]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def _pm(pos_mass):
    a = np.ascontiguousarray(pos_mass, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4, "pos_mass must be float32 [n,4] (x,y,z,m)"
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def cell_ids(pos_mass, box, ncell) -> np.ndarray:
    """uint32 linear cell id per particle (R10, R11). Raises ValueError on a DOMAIN violation (R13)."""
    a, ap = _pm(pos_mass)
    b, bp = _f32(box)
    nc = np.ascontiguousarray(ncell, dtype=np.int32)
    out = np.empty(a.shape[0], dtype=np.uint32)
    rc = lib().orc_cell_ids(ap, a.shape[0], bp, nc.ctypes.data_as(C.POINTER(C.c_int32)),
                            out.ctypes.data_as(C.POINTER(C.c_uint32)))
    if rc != 0:
        raise ValueError("DOMAIN: a position is outside [0, L) or not finite")
    return out


def build_mesh(pos_mass, box, ncell):
    """Stable counting sort by cell id (R12) -> (cell_start uint32[ncells+1], perm uint32[n], sorted f32[n,4])."""
    a, ap = _pm(pos_mass)
    b, bp = _f32(box)
    nc = np.ascontiguousarray(ncell, dtype=np.int32)
    ncells = int(nc[0]) * int(nc[1]) * int(nc[2])
    n = a.shape[0]
    cell_start = np.empty(ncells + 1, dtype=np.uint32)
    perm = np.empty(n, dtype=np.uint32)
    srt = np.empty((n, 4), dtype=np.float32)
    rc = lib().orc_build_mesh(ap, n, bp, nc.ctypes.data_as(C.POINTER(C.c_int32)),
                              cell_start.ctypes.data_as(C.POINTER(C.c_uint32)),
                              perm.ctypes.data_as(C.POINTER(C.c_uint32)),
                              srt.ctypes.data_as(C.POINTER(C.c_float)))
    if rc == -3:
        raise ValueError("DOMAIN: a position is outside [0, L) or not finite")
    if rc != 0:
        raise MemoryError("oracle build_mesh failed (%d)" % rc)
    return cell_start, perm, srt


def pair_factor(params: Params, s: float) -> float:
    """f(s) = (s+eps^2)^(-3/2) - P(s) for s < rc^2, else 0."""
    return float(lib().orc_pair_factor(C.byref(params), float(s)))


def poly(params: Params, s: float) -> float:
    return float(lib().orc_poly(C.byref(params), float(s)))


def accel_bruteforce(pos_mass, params: Params, stats: bool = False):
    """O(N^2) plain definition. Returns acc f64 [n,3] (and n_in, sum_abs if stats)."""
    a, ap = _pm(pos_mass)
    n = a.shape[0]
    acc = np.zeros((n, 3), dtype=np.float64)
    n_in = np.zeros(n, dtype=np.int64)
    sa = np.zeros(n, dtype=np.float64)
    lib().orc_accel_bruteforce(ap, n, C.byref(params), acc.ctypes.data_as(C.POINTER(C.c_double)),
                               n_in.ctypes.data_as(C.POINTER(C.c_int64)),
                               sa.ctypes.data_as(C.POINTER(C.c_double)))
    return (acc, n_in, sa) if stats else acc


def accel(pos_mass, params: Params, targets=None, stats: bool = False):
    """Cell-list evaluation of the same sum, for `targets` (default: all).

    Returns acc f64 [nt,3]; with stats=True also a dict with n_in, sum_abs,
    allowance (R9) and n_cand (candidates of the oracle's own cell list).
    """
    a, ap = _pm(pos_mass)
    n = a.shape[0]
    if targets is None:
        tp, nt = None, n
    else:
        t = np.ascontiguousarray(targets, dtype=np.int64)
        assert t.size == 0 or (t.min() >= 0 and t.max() < n)
        tp, nt = t.ctypes.data_as(C.POINTER(C.c_int64)), t.shape[0]
    acc = np.zeros((nt, 3), dtype=np.float64)
    n_in = np.zeros(nt, dtype=np.int64)
    sa = np.zeros(nt, dtype=np.float64)
    al = np.zeros(nt, dtype=np.float64)
    nc = np.zeros(nt, dtype=np.int64)
    rc = lib().orc_accel(ap, n, C.byref(params), tp, nt, acc.ctypes.data_as(C.POINTER(C.c_double)),
                         n_in.ctypes.data_as(C.POINTER(C.c_int64)),
                         sa.ctypes.data_as(C.POINTER(C.c_double)),
                         al.ctypes.data_as(C.POINTER(C.c_double)),
                         nc.ctypes.data_as(C.POINTER(C.c_int64)))
    if rc != 0:
        raise MemoryError("oracle accel failed (%d)" % rc)
    if stats:
        return acc, {"n_in": n_in, "sum_abs": sa, "allowance": al, "n_cand": nc}
    return acc


def kick(vel, acc, kdt: float) -> np.ndarray:
    """v <- fmaf(a, kdt, v) per component in fp32 (R16). vel, acc: float32 [n,4]; returns new vel."""
    v = np.array(vel, dtype=np.float32, order="C", copy=True)
    a, ap = _f32(acc)
    lib().orc_kick(v.ctypes.data_as(C.POINTER(C.c_float)), ap, float(kdt), v.shape[0])
    return v


def stream(pos_mass, vel, dt: float, box) -> np.ndarray:
    """x <- wrap(fmaf(v, dt, x)) in fp32 (R13, R17). Returns new pos_mass."""
    x = np.array(pos_mass, dtype=np.float32, order="C", copy=True)
    v, vp = _f32(vel)
    b, bp = _f32(box)
    lib().orc_stream(x.ctypes.data_as(C.POINTER(C.c_float)), vp, float(dt), bp, x.shape[0])
    return x


def subcycle(pos_mass, vel, params: Params, dt: float, kdt: float, nsub: int = 1):
    """nsub x { stream(dt/2); a = accel (fp64 sum rounded once to fp32); kick(kdt); stream(dt/2) } (R20).
    Returns new (pos_mass, vel, acc) as float32 [n,4] arrays; acc = accelerations of the last sub-step."""
    x = np.array(pos_mass, dtype=np.float32, order="C", copy=True)
    v = np.array(vel, dtype=np.float32, order="C", copy=True)
    assert x.ndim == 2 and x.shape[1] == 4 and v.shape == x.shape
    a = np.zeros_like(x)
    f32p = C.POINTER(C.c_float)
    rc = lib().orc_subcycle(x.ctypes.data_as(f32p), v.ctypes.data_as(f32p), x.shape[0], C.byref(params),
                            C.c_float(dt), C.c_float(kdt), int(nsub), a.ctypes.data_as(f32p))
    if rc != 0:
        raise MemoryError("oracle subcycle failed (%d)" % rc)
    return x, v, a


def error_norms(a_test, a_ref, allowance=None):
    """R18 error metrics. Returns (per_particle_rel [n], global_rel_l2).

    per-particle: |a_test - a_ref|_2 / max(|a_ref|_2, 1e-4 * rms|a_ref|), with the R9 allowance
    subtracted from the numerator first (never below 0); global: sqrt(sum|diff|^2 / sum|a_ref|^2).
    """
    a_test = np.asarray(a_test, dtype=np.float64)[:, :3]
    a_ref = np.asarray(a_ref, dtype=np.float64)[:, :3]
    diff = np.linalg.norm(a_test - a_ref, axis=1)
    ref = np.linalg.norm(a_ref, axis=1)
    rms = float(np.sqrt(np.mean(ref * ref))) if ref.size else 0.0
    if allowance is not None:
        diff_pp = np.maximum(0.0, diff - np.asarray(allowance, dtype=np.float64))
    else:
        diff_pp = diff
    floor = max(1e-4 * rms, 1e-300)
    per = diff_pp / np.maximum(ref, floor)
    tot = float(np.sum(ref * ref))
    glob = float(np.sqrt(np.sum(diff * diff) / tot)) if tot > 0 else float(np.sqrt(np.sum(diff * diff)))
    return per, glob


def mbp(pos_mass, halo_start, eps: float):
    """Most bound particle of every halo (reading R19).  halo_start: int64 [nhalo+1], halo h is the
    run pos_mass[halo_start[h]:halo_start[h+1]].  Returns (phi f64 [n], index int64 [nhalo])."""
    a, ap = _pm(pos_mass)
    hs = np.ascontiguousarray(halo_start, dtype=np.int64)
    nh = hs.shape[0] - 1
    assert nh >= 0 and (nh == 0 or (hs[0] >= 0 and hs[-1] <= a.shape[0] and np.all(np.diff(hs) >= 0)))
    phi = np.zeros(a.shape[0], dtype=np.float64)
    idx = np.full(max(nh, 0), -1, dtype=np.int64)
    lib().orc_mbp(ap, a.shape[0], hs.ctypes.data_as(C.POINTER(C.c_int64)), nh, C.c_float(eps),
                  phi.ctypes.data_as(C.POINTER(C.c_double)), idx.ctypes.data_as(C.POINTER(C.c_int64)))
    return phi, idx
