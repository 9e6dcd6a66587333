"""Thin ctypes binding over libsrpp.so (include/srpp.h).  Argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used here for
device memory and streams, nothing else.  There is NO CPU fallback: if libsrpp.so is missing
or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsrpp.so")

SRPP_OK = 0
STATUS_NAMES = {0: "OK", -1: "INVALID_ARG", -2: "GEOMETRY", -3: "DOMAIN", -4: "WORKSPACE", -5: "STATE", -6: "CUDA", -7: "LIMIT"}
MBP_STATIC_MAX_N, MBP_STATIC_MAX_HALOS = 1 << 20, 1 << 16      # include/srpp.h

EXPORTS = ("srpp_version", "srpp_default_poly", "srpp_workspace_bytes", "srpp_create", "srpp_destroy",
           "srpp_build_mesh", "srpp_get_mesh", "srpp_accel", "srpp_accel_kick", "srpp_get_stats", "srpp_kick", "srpp_stream",
           "srpp_step_host", "srpp_strerror", "srpp_last_cuda_error", "srpp_set_timing", "srpp_get_timings",
           "srpp_probe_fp32", "srpp_set_boundary", "srpp_mbp_workspace_bytes", "srpp_mbp", "srpp_mbp_static", "srpp_subcycle",
           "srpp_blocks_workspace_bytes", "srpp_blocks_init", "srpp_accel_blocks", "srpp_get_blocks")


class SrppParams(C.Structure):
    _fields_ = [("box", C.c_float * 3), ("ncell", C.c_int32 * 3), ("rcut", C.c_float), ("eps", C.c_float),
                ("poly", C.c_float * 6)]


class SrppStats(C.Structure):
    _fields_ = [("work_items", C.c_uint64), ("pair_slots", C.c_uint64), ("candidate_pairs", C.c_uint64),
                ("max_cell_count", C.c_uint32), ("uniform_mass", C.c_uint32), ("kernel_launches", C.c_uint64),
                ("rebins_incremental", C.c_uint64), ("rebins_full", C.c_uint64), ("last_movers", C.c_uint64)]


class SrppBlockInfo(C.Structure):
    _fields_ = [("x0", C.c_float), ("x1", C.c_float), ("level", C.c_int32), ("pad_", C.c_int32), ("n_active", C.c_int64),
                ("n_total", C.c_int64), ("candidate_pairs", C.c_uint64), ("ms", C.c_float), ("pad2_", C.c_float)]


SRPP_MAX_BLOCKS = 64


class SrppTimings(C.Structure):
    _fields_ = [("mesh_ms", C.c_float), ("accel_ms", C.c_float), ("force_ms", C.c_float), ("rebin_ms", C.c_float),
                ("kick_stream_ms", C.c_float)]


class SrppError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        name = STATUS_NAMES.get(status, str(status))
        super().__init__("%s failed: SRPP_ERR_%s (%d) %s" % (where, name, status, detail))


_lib = None


def load() -> C.CDLL:
    """dlopen libsrpp.so and declare the prototypes of include/srpp.h.  Raises if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libsrpp.so is not built (%s): run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "or `python paper_1411_3396_b200/build.py`; there is no CPU fallback" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
    L.srpp_version.restype = i32
    L.srpp_default_poly.restype = i32
    L.srpp_default_poly.argtypes = [C.POINTER(C.c_float)]
    L.srpp_workspace_bytes.restype = i32
    L.srpp_workspace_bytes.argtypes = [C.POINTER(SrppParams), i64, C.POINTER(C.c_size_t)]
    L.srpp_create.restype = i32
    L.srpp_create.argtypes = [C.POINTER(vp), C.POINTER(SrppParams), vp, C.c_size_t, vp]
    L.srpp_destroy.restype = None
    L.srpp_destroy.argtypes = [vp]
    L.srpp_build_mesh.restype = i32
    L.srpp_build_mesh.argtypes = [vp, vp, i64]
    L.srpp_get_mesh.restype = i32
    L.srpp_get_mesh.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.srpp_accel.restype = i32
    L.srpp_accel.argtypes = [vp, vp]
    L.srpp_accel_kick.restype = i32
    L.srpp_accel_kick.argtypes = [vp, vp, vp, f32]
    L.srpp_get_stats.restype = i32
    L.srpp_get_stats.argtypes = [vp, C.POINTER(SrppStats)]
    L.srpp_kick.restype = i32
    L.srpp_kick.argtypes = [vp, vp, vp, f32, i64]
    L.srpp_stream.restype = i32
    L.srpp_stream.argtypes = [vp, vp, vp, f32, i64]
    L.srpp_blocks_workspace_bytes.restype = i32
    L.srpp_blocks_workspace_bytes.argtypes = [C.POINTER(SrppParams), i64, C.POINTER(C.c_size_t)]
    L.srpp_blocks_init.restype = i32
    L.srpp_blocks_init.argtypes = [vp, i32]
    L.srpp_accel_blocks.restype = i32
    L.srpp_accel_blocks.argtypes = [vp, vp, i64, vp, vp, C.c_size_t]
    L.srpp_get_blocks.restype = i32
    L.srpp_get_blocks.argtypes = [vp, C.POINTER(SrppBlockInfo), i32, C.POINTER(i32)]
    L.srpp_subcycle.restype = i32
    L.srpp_subcycle.argtypes = [vp, vp, vp, vp, f32, f32, i32, i64]
    L.srpp_step_host.restype = i32
    L.srpp_step_host.argtypes = [vp, vp, vp, vp, f32, i64, vp, C.c_size_t]
    L.srpp_set_timing.restype = i32
    L.srpp_set_timing.argtypes = [vp, i32]
    L.srpp_get_timings.restype = i32
    L.srpp_get_timings.argtypes = [vp, C.POINTER(SrppTimings)]
    L.srpp_mbp_workspace_bytes.restype = i32
    L.srpp_mbp_workspace_bytes.argtypes = [i64, i64, C.POINTER(C.c_size_t)]
    L.srpp_mbp.restype = i32
    L.srpp_mbp.argtypes = [vp, vp, i64, C.POINTER(i64), i64, vp, vp, vp, vp, C.c_size_t]
    L.srpp_mbp_static.restype = i32
    L.srpp_mbp_static.argtypes = [vp, i64, C.POINTER(i64), i64, f32, vp, vp, vp, vp]
    L.srpp_set_boundary.restype = i32
    L.srpp_set_boundary.argtypes = [vp, C.POINTER(i32), C.POINTER(C.c_float), C.POINTER(C.c_float)]
    L.srpp_probe_fp32.restype = i32
    L.srpp_probe_fp32.argtypes = [vp, i32, i32, C.POINTER(C.c_double)]
    L.srpp_strerror.restype = C.c_char_p
    L.srpp_strerror.argtypes = [i32]
    L.srpp_last_cuda_error.restype = C.c_char_p
    L.srpp_last_cuda_error.argtypes = [vp]
    _lib = L
    return L


def default_poly() -> np.ndarray:
    out = (C.c_float * 6)()
    rc = load().srpp_default_poly(out)
    if rc != SRPP_OK:
        raise SrppError(rc, "srpp_default_poly")
    return np.array(list(out), dtype=np.float32)


def make_params(box, ncell, rcut=3.0, eps=0.1, poly=None) -> SrppParams:
    p = SrppParams()
    poly = default_poly() if poly is None else np.asarray(poly, dtype=np.float32)
    for a in range(3):
        p.box[a] = float(box[a])
        p.ncell[a] = int(ncell[a])
    p.rcut, p.eps = float(rcut), float(eps)
    for k in range(6):
        p.poly[k] = float(poly[k])
    return p


def workspace_bytes(params: SrppParams, n: int) -> int:
    out = C.c_size_t(0)
    rc = load().srpp_workspace_bytes(C.byref(params), int(n), C.byref(out))
    if rc != SRPP_OK:
        raise SrppError(rc, "srpp_workspace_bytes")
    return int(out.value)


def strerror(status: int) -> str:
    return load().srpp_strerror(int(status)).decode()


def mbp_static(pos_mass, halo_start, eps: float, idx, pmin=None, phi=None, stream=None) -> None:
    """srpp_mbp_static: the most bound particle of every halo with the library's built-in scratch array -- no workspace,
    no context, no device allocation.  The caller passes every output: idx int64 [nhalo], pmin float32 [nhalo] or None,
    phi float32 [n] or None (CUDA tensors).  halo_start: host int64 sequence [nhalo+1].  Raises SrppError (status -7 =
    LIMIT above MBP_STATIC_MAX_N members or MBP_STATIC_MAX_HALOS halos)."""
    hs = np.ascontiguousarray(halo_start, dtype=np.int64)
    nh, n = int(hs.shape[0]) - 1, int(pos_mass.shape[0])
    if stream is None:
        import torch
        stream = torch.cuda.current_stream(pos_mass.device)
    st = stream.cuda_stream
    rc = load().srpp_mbp_static(pos_mass.data_ptr(), n, hs.ctypes.data_as(C.POINTER(C.c_int64)), nh, float(eps),
                                phi.data_ptr() if phi is not None else None, idx.data_ptr() if nh > 0 else None,
                                pmin.data_ptr() if pmin is not None else None, st)
    if rc != SRPP_OK:
        raise SrppError(rc, "srpp_mbp_static", strerror(rc))


class Solver:
    """One srpp_ctx plus the torch-owned workspace it points into.

    box, ncell, rcut, eps, poly -> srpp_params; n_max sizes the workspace; `stream` is a
    torch.cuda.Stream (default: the current stream at construction).
    """

    def __init__(self, box, ncell, rcut=3.0, eps=0.1, poly=None, n_max: int = 0, device="cuda:0", stream=None):
        import torch
        self._torch = torch
        self.lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the srpp path has no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.params = make_params(box, ncell, rcut, eps, poly)
        self.n_max = int(n_max)
        nbytes = workspace_bytes(self.params, self.n_max)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._ctx = C.c_void_p()
        rc = self.lib.srpp_create(C.byref(self._ctx), C.byref(self.params), self.workspace.data_ptr(), nbytes,
                                  self.stream.cuda_stream)
        if rc != SRPP_OK:
            raise SrppError(rc, "srpp_create")
        self.n = -1
        self.ncells = int(ncell[0]) * int(ncell[1]) * int(ncell[2])

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, rc: int, where: str):
        if rc != SRPP_OK:
            detail = self.lib.srpp_last_cuda_error(self._ctx).decode() if rc == -6 else strerror(rc)
            raise SrppError(rc, where, detail)

    def _f4(self, t, name):
        torch = self._torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                and t.dim() == 2 and t.shape[1] == 4):
            raise TypeError("%s must be a contiguous CUDA float32 tensor of shape [n, 4]" % name)
        return t

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.srpp_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/srpp.h ----------------------------------------------------------
    def build_mesh(self, pos_mass):
        self._f4(pos_mass, "pos_mass")
        n = pos_mass.shape[0]
        self.n = -1
        self._check(self.lib.srpp_build_mesh(self._ctx, pos_mass.data_ptr(), n), "srpp_build_mesh")
        self.n = n
        self._pos_ref = pos_mass   # keep the caller's tensor alive while views exist

    def get_mesh(self):
        """(cell_start uint32[ncells+1], perm uint32[n], sorted float32[n,4]) as torch CLONES of the views."""
        torch = self._torch
        cs, pm, so = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self.lib.srpp_get_mesh(self._ctx, C.byref(cs), C.byref(pm), C.byref(so)), "srpp_get_mesh")
        base = self.workspace.data_ptr()

        def view(ptr, nbytes):
            off = ptr.value - base
            assert 0 <= off and off + nbytes <= self.workspace.numel()
            return self.workspace[off: off + nbytes]
        n = self.n
        with torch.cuda.stream(self.stream):
            cell_start = view(cs, 4 * (self.ncells + 1)).view(torch.int32).clone()
            perm = view(pm, 4 * n).view(torch.int32).clone() if n else torch.empty(0, dtype=torch.int32, device=self.device)
            srt = (view(so, 16 * n).view(torch.float32).view(n, 4).clone() if n
                   else torch.empty((0, 4), dtype=torch.float32, device=self.device))
        return cell_start, perm, srt

    def accel(self, acc=None):
        torch = self._torch
        if self.n < 0:
            self._check(-5, "srpp_accel")
        if acc is None:
            acc = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        self._f4(acc, "acc")
        if acc.shape[0] != self.n:
            raise ValueError("acc has %d rows, mesh has %d particles" % (acc.shape[0], self.n))
        self._check(self.lib.srpp_accel(self._ctx, acc.data_ptr()), "srpp_accel")
        return acc

    def accel_kick(self, vel, kdt: float, acc=None):
        """srpp_accel_kick: accelerations (caller's order) and v <- fmaf(a, kdt, v) in one call; returns acc."""
        torch = self._torch
        if self.n < 0:
            self._check(-5, "srpp_accel_kick")
        if acc is None:
            acc = torch.empty((self.n, 4), dtype=torch.float32, device=self.device)
        self._f4(acc, "acc"), self._f4(vel, "vel")
        if acc.shape[0] != self.n or vel.shape[0] != self.n:
            raise ValueError("acc / vel rows differ from the mesh's %d particles" % self.n)
        self._check(self.lib.srpp_accel_kick(self._ctx, acc.data_ptr(), vel.data_ptr(), float(kdt)), "srpp_accel_kick")
        return acc

    def get_stats(self) -> dict:
        s = SrppStats()
        self._check(self.lib.srpp_get_stats(self._ctx, C.byref(s)), "srpp_get_stats")
        return {k: int(getattr(s, k)) for k, _ in SrppStats._fields_}

    def set_timing(self, enable: bool = True):
        self._check(self.lib.srpp_set_timing(self._ctx, 1 if enable else 0), "srpp_set_timing")

    def get_timings(self) -> dict:
        """Device milliseconds of the last build_mesh / accel / force kernel (synchronises)."""
        t = SrppTimings()
        self._check(self.lib.srpp_get_timings(self._ctx, C.byref(t)), "srpp_get_timings")
        return {k: float(getattr(t, k)) for k, _ in SrppTimings._fields_}

    def mbp(self, pos_mass, halo_start, want_phi: bool = True):
        """srpp_mbp: most bound particle of every halo.  halo_start: host int64 sequence [nhalo+1].
        Returns (index int64 [nhalo], phi_min float32 [nhalo], phi float32 [n] or None), device tensors."""
        import numpy as np
        torch = self._torch
        hs = np.ascontiguousarray(halo_start, dtype=np.int64)
        nh, n = int(hs.shape[0]) - 1, int(pos_mass.shape[0])
        nbytes = C.c_size_t(0)
        self._check(self.lib.srpp_mbp_workspace_bytes(n, nh, C.byref(nbytes)), "srpp_mbp_workspace_bytes")
        with torch.cuda.stream(self.stream):           # allocated (and zeroed) on the stream the kernels run on
            ws = torch.empty(max(int(nbytes.value), 256), dtype=torch.uint8, device=self.device)
            idx = torch.empty(max(nh, 1), dtype=torch.int64, device=self.device)[:nh]
            pmin = torch.empty(max(nh, 1), dtype=torch.float32, device=self.device)[:nh]
            phi = torch.zeros(max(n, 1), dtype=torch.float32, device=self.device)[:n] if want_phi else None
        self._check(self.lib.srpp_mbp(self._ctx, pos_mass.data_ptr(), n, hs.ctypes.data_as(C.POINTER(C.c_int64)), nh,
                                      phi.data_ptr() if want_phi else None, idx.data_ptr(), pmin.data_ptr(),
                                      ws.data_ptr(), int(nbytes.value)), "srpp_mbp")
        self._mbp_ws = ws                                  # keep the workspace alive until the stream has run
        return idx, pmin, phi

    def set_boundary(self, periodic=(1, 1, 1), active_lo=None, active_hi=None) -> None:
        """srpp_set_boundary: open (non-periodic) axes and the active box of an overloaded node volume."""
        per = (C.c_int32 * 3)(*[1 if v else 0 for v in periodic])
        lo = (C.c_float * 3)(*[float(v) for v in active_lo]) if active_lo is not None else None
        hi = (C.c_float * 3)(*[float(v) for v in active_hi]) if active_hi is not None else None
        self._check(self.lib.srpp_set_boundary(self._ctx, per, lo, hi), "srpp_set_boundary")

    def probe_fp32(self, variant: int = 1, trips: int = 2000) -> float:
        """Sustained FP32 flop/s of a register-only FMA stream (0 = FFMA, 1 = packed FFMA2)."""
        out = C.c_double(0.0)
        self._check(self.lib.srpp_probe_fp32(self._ctx, int(variant), int(trips), C.byref(out)), "srpp_probe_fp32")
        return float(out.value)

    def kick(self, vel, acc, kdt: float):
        self._f4(vel, "vel"), self._f4(acc, "acc")
        if vel.shape != acc.shape:
            raise ValueError("vel and acc shapes differ")
        self._check(self.lib.srpp_kick(self._ctx, vel.data_ptr(), acc.data_ptr(), float(kdt), vel.shape[0]), "srpp_kick")
        return vel

    def stream_positions(self, pos_mass, vel, dt: float):
        self._f4(pos_mass, "pos_mass"), self._f4(vel, "vel")
        if vel.shape != pos_mass.shape:
            raise ValueError("pos_mass and vel shapes differ")
        self._check(self.lib.srpp_stream(self._ctx, pos_mass.data_ptr(), vel.data_ptr(), float(dt), vel.shape[0]),
                    "srpp_stream")
        return pos_mass

    def blocks_init(self, nblocks: int) -> None:
        """srpp_blocks_init: start the block plan with nblocks equal x-ranges."""
        self._check(self.lib.srpp_blocks_init(self._ctx, int(nblocks)), "srpp_blocks_init")

    def accel_blocks(self, pos_mass, acc=None):
        """srpp_accel_blocks: accelerations block by block (extract, own mesh, force, reconcile); refines the plan for the
        next call by the x2 rule.  Returns (acc, blocks) with blocks = list of dicts (srpp_block_info)."""
        torch = self._torch
        self._f4(pos_mass, "pos_mass")
        n = pos_mass.shape[0]
        if acc is None:
            acc = torch.empty((n, 4), dtype=torch.float32, device=self.device)
        self._f4(acc, "acc")
        nbytes = C.c_size_t(0)
        self._check(self.lib.srpp_blocks_workspace_bytes(C.byref(self.params), n, C.byref(nbytes)), "srpp_blocks_workspace_bytes")
        if getattr(self, "_blocks_ws", None) is None or self._blocks_ws.numel() < nbytes.value:
            self._blocks_ws = torch.empty(int(nbytes.value), dtype=torch.uint8, device=self.device)
        self._check(self.lib.srpp_accel_blocks(self._ctx, pos_mass.data_ptr(), n, acc.data_ptr(), self._blocks_ws.data_ptr(),
                                               self._blocks_ws.numel()), "srpp_accel_blocks")
        info = (SrppBlockInfo * SRPP_MAX_BLOCKS)()
        cnt = C.c_int32(0)
        self._check(self.lib.srpp_get_blocks(self._ctx, info, SRPP_MAX_BLOCKS, C.byref(cnt)), "srpp_get_blocks")
        blocks = [{k: getattr(info[b], k) for k in ("x0", "x1", "level", "n_active", "n_total", "candidate_pairs", "ms")}
                  for b in range(cnt.value)]
        return acc, blocks

    def subcycle(self, pos_mass, vel, dt: float, kdt: float = None, nsub: int = 1, acc=None):
        """srpp_subcycle: nsub x {stream(dt/2), accel, kick(kdt), stream(dt/2)}; pos_mass and vel are updated in place.
        Returns acc (accelerations of the last sub-step).  kdt defaults to dt."""
        torch = self._torch
        self._f4(pos_mass, "pos_mass"), self._f4(vel, "vel")
        if vel.shape != pos_mass.shape:
            raise ValueError("pos_mass and vel shapes differ")
        n = pos_mass.shape[0]
        if acc is None:
            acc = torch.zeros((n, 4), dtype=torch.float32, device=self.device)
        self._f4(acc, "acc")
        self.n = -1
        self._check(self.lib.srpp_subcycle(self._ctx, pos_mass.data_ptr(), vel.data_ptr(), acc.data_ptr(), float(dt),
                                           float(dt if kdt is None else kdt), int(nsub), n), "srpp_subcycle")
        self.n = n
        self._pos_ref = pos_mass
        return acc

    def step_host(self, pos_mass_host, vel_host, acc_host, kdt: float, scratch):
        """End-to-end call on HOST (ideally pinned) float32 [n,4] tensors/arrays; `scratch` is a CUDA uint8 tensor
        of >= 48 n bytes.  vel_host may be None (no kick)."""
        def hptr(a):
            if a is None:
                return None
            if hasattr(a, "data_ptr"):
                assert not a.is_cuda and a.is_contiguous()
                return a.data_ptr()
            assert a.flags["C_CONTIGUOUS"] and a.dtype == np.float32
            return a.ctypes.data
        n = int(pos_mass_host.shape[0])
        self.n = -1
        rc = self.lib.srpp_step_host(self._ctx, hptr(pos_mass_host), hptr(vel_host), hptr(acc_host), float(kdt), n,
                                     scratch.data_ptr(), scratch.numel())
        self._check(rc, "srpp_step_host")
        self.n = n
        return acc_host
