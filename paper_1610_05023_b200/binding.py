"""Thin ctypes binding of include/dg_habc.h — argument marshalling only; every step of the path runs in the
CUDA kernels of libdg_habc.so.  torch is used for the device workspace and the stream (dg_options)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None


class DgError(RuntimeError):
    pass


class _Mesh(C.Structure):
    _fields_ = [("nverts", C.c_int32), ("xyz", C.POINTER(C.c_double)), ("ntets", C.c_int32),
                ("tets", C.POINTER(C.c_int32))]


class _Options(C.Structure):
    _fields_ = [("precision", C.c_int32), ("cfl", C.c_double), ("dt", C.c_double), ("stream", C.c_void_p),
                ("device", C.c_int32), ("workspace_dev", C.c_void_p), ("workspace_bytes", C.c_uint64),
                ("use_graph", C.c_int32), ("kernel", C.c_int32), ("face_bc", C.c_int32 * 6), ("time_kernels", C.c_int32)]


class _Info(C.Structure):
    _fields_ = [("N", C.c_int32), ("J", C.c_int32), ("K", C.c_int32), ("Np", C.c_int32), ("Nfp", C.c_int32),
                ("T", C.c_int32), ("E", C.c_int32), ("C", C.c_int32), ("precision", C.c_int32),
                ("launches_per_step", C.c_int32), ("dt", C.c_double), ("device_bytes", C.c_uint64),
                ("kernel", C.c_int32), ("kernel_name", C.c_char * 44)]


class _DeviceView(C.Structure):
    _fields_ = [("elem_bytes", C.c_int32), ("reserved", C.c_int32), ("q", C.c_void_p), ("face_aux", C.c_void_p),
                ("face_S", C.c_void_p), ("edge_aux", C.c_void_p)]


EXPORTS = ["dg_workspace_bytes", "dg_create", "dg_get_info", "dg_get_nodes", "dg_set_initial", "dg_set_source", "dg_step",
           "dg_get_fields", "dg_get_face_map", "dg_get_edge_map", "dg_reference_element", "dg_mesh_counts",
           "dg_profile_step", "dg_last_step_kernel_ms", "dg_set_time_kernels", "dg_get_device_ptrs", "dg_get_aux_fields_noalloc", "dg_last_error",
           "dg_destroy"]


def lib() -> C.CDLL:
    """Load (building if the sources are newer) the C-ABI library.  Fails loudly if it cannot be had."""
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if _build.is_stale():
            path = _build.build()
        _LIB = C.CDLL(path)
        _LIB.dg_last_error.restype = C.c_char_p
        _LIB.dg_destroy.restype = None
        for name in EXPORTS:
            getattr(_LIB, name)
    return _LIB


def _check(rc: int):
    if rc != 0:
        raise DgError(f"[{rc}] " + lib().dg_last_error().decode())


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_int32))


def _mesh(verts, tets):
    verts = np.ascontiguousarray(verts, dtype=np.float64)
    tets = np.ascontiguousarray(tets, dtype=np.int32)
    return _Mesh(verts.shape[0], _dp(verts), tets.shape[0], _ip(tets)), (verts, tets)


def dg_reference_element(dim: int, N: int):
    """(rst [Np,dim], D [dim,Np,Np], LIFT [Np,Nfaces*Nfp], Fmask [Nfaces,Nfp]) as the library computes them."""
    Np = {1: N + 1, 2: (N + 1) * (N + 2) // 2, 3: (N + 1) * (N + 2) * (N + 3) // 6}[dim]
    Nfp = {1: 1, 2: N + 1, 3: (N + 1) * (N + 2) // 2}[dim]
    nf = dim + 1
    rst, D = np.empty((Np, dim)), np.empty((dim, Np, Np))
    LIFT, Fm = np.empty((Np, nf * Nfp)), np.empty((nf, Nfp), dtype=np.int32)
    npo = C.c_int32(0)
    _check(lib().dg_reference_element(dim, N, _dp(rst), _dp(D), _dp(LIFT), _ip(Fm), C.byref(npo)))
    assert npo.value == Np
    return rst, D, LIFT, Fm


_BC_CODES = {"habc": 0, "dirichlet": 1, "rigid": 2}
# dg_options.kernel (DG_KERNEL_* of include/dg_habc.h)
KERNEL_AUTO, KERNEL_SCALAR, KERNEL_MMA, KERNEL_WS, KERNEL_TF32, KERNEL_TPG, KERNEL_ELEM = range(7)


def _face_bc_codes(face_bc):
    codes = np.zeros(6, dtype=np.int32)
    for (axis, sign), kind in (face_bc or {}).items():
        codes[axis * 2 + (1 if sign > 0 else 0)] = _BC_CODES[kind]
    return codes


def dg_mesh_counts(verts, tets, face_bc=None):
    m, keep = _mesh(verts, tets)
    out = np.zeros(4, dtype=np.int32)
    _check(lib().dg_mesh_counts(C.byref(m), _ip(_face_bc_codes(face_bc)), _ip(out)))
    return tuple(int(x) for x in out)


class Solver:
    """dg_create / dg_set_initial / dg_step / dg_get_fields / dg_destroy of the C ABI."""

    def __init__(self, verts, tets, N: int, J: int, c, rho, precision: int = 64, cfl: float = 1.0,
                 dt: float = 0.0, device: int = 0, use_graph: bool = True, torch_workspace: bool = True,
                 kernel: int = 0, face_bc=None, time_kernels: bool = False, default_stream: bool = False):
        """face_bc: None (HABC everywhere) or {(axis, sign): "habc" | "dirichlet" | "rigid"} for some of the six domain
        faces (axis 0..2, sign -1/+1) -- dg_options.face_bc.  torch_workspace = False: dg_options.workspace_dev = NULL,
        the library allocates with cudaMalloc.  default_stream = True: dg_options.stream = NULL, the legacy default
        stream (plain launches, no CUDA graph)."""
        import torch                                          # device memory + stream only
        if not torch.cuda.is_available():
            raise DgError("no CUDA device: the DG+HABC path has no CPU fallback")
        L = lib()
        m, self._keep = _mesh(verts, tets)
        c = np.ascontiguousarray(c, dtype=np.float64)
        rho = np.ascontiguousarray(rho, dtype=np.float64)
        opt = _Options()
        opt.precision, opt.cfl, opt.dt, opt.device, opt.use_graph = precision, cfl, dt, device, int(use_graph)
        opt.kernel = int(kernel)
        opt.time_kernels = int(time_kernels)
        for i, code in enumerate(_face_bc_codes(face_bc)):
            opt.face_bc[i] = int(code)
        self._torch = torch
        torch.cuda.set_device(device)
        # a dedicated (capturable) torch stream: the solver's kernels and CUDA graph run on it
        self._stream = torch.cuda.default_stream(device) if default_stream else torch.cuda.Stream(device=device)
        self.stream = self._stream
        opt.stream = None if default_stream else self._stream.cuda_stream
        self._ws = None
        if torch_workspace:
            nbytes = C.c_uint64(0)
            _check(L.dg_workspace_bytes(C.byref(m), N, J, precision, C.byref(nbytes)))
            self._ws = torch.empty(int(nbytes.value), dtype=torch.uint8, device=f"cuda:{device}")
            opt.workspace_dev, opt.workspace_bytes = self._ws.data_ptr(), nbytes.value
        self._h = C.c_void_p()
        _check(L.dg_create(C.byref(m), N, J, _dp(c), _dp(rho), C.byref(opt), C.byref(self._h)))
        info = _Info()
        _check(L.dg_get_info(self._h, C.byref(info)))
        self.info = self._info_dict(info)
        for k, v in self.info.items():
            setattr(self, k, v)

    # ---- boundary calls
    def get_nodes(self):
        x = np.empty((3, self.K, self.Np))
        _check(lib().dg_get_nodes(self._h, _dp(x[0]), _dp(x[1]), _dp(x[2])))
        return x[0], x[1], x[2]

    def set_initial(self, p, u, v, w):
        a = [np.ascontiguousarray(f, dtype=np.float64).reshape(self.K, self.Np) for f in (p, u, v, w)]
        _check(lib().dg_set_initial(self._h, *[_dp(f) for f in a]))

    def set_source(self, xyz, f_peak: float, t_s: float, amplitude: float = 1.0):
        xyz = np.ascontiguousarray(xyz, dtype=np.float64).reshape(3)
        L = lib()
        L.dg_set_source.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_double, C.c_double, C.c_double]
        _check(L.dg_set_source(self._h, _dp(xyz), float(f_peak), float(t_s), float(amplitude)))
        self.launches_per_step = self.info["launches_per_step"] = self._refresh_info()["launches_per_step"]

    @staticmethod
    def _info_dict(info):
        d = {k: getattr(info, k) for k, _ in _Info._fields_}
        d["kernel_name"] = d["kernel_name"].decode()
        return d

    def _refresh_info(self):
        info = _Info()
        _check(lib().dg_get_info(self._h, C.byref(info)))
        return self._info_dict(info)

    def step(self, nsteps: int = 1):
        _check(lib().dg_step(self._h, int(nsteps)))

    def get_fields(self, aux: bool = True, out=None):
        """(q [4,K,Np], face_aux, edge_aux).  `out`: optional preallocated float64 C-contiguous [4,K,Np] array for q
        (e.g. backed by pinned host memory) -- written in place and returned."""
        q = np.empty((4, self.K, self.Np)) if out is None else out
        if q.dtype != np.float64 or q.shape != (4, self.K, self.Np) or not q.flags["C_CONTIGUOUS"]:
            raise DgError("get_fields(out=...): need a C-contiguous float64 array of shape (4, K, Np)")
        fa = np.zeros((self.T, self.J, 3, self.Nfp)) if aux else None
        ea = np.zeros((self.E, self.J * self.J, 2, self.N + 1)) if aux else None
        _check(lib().dg_get_fields(self._h, _dp(q[0]), _dp(q[1]), _dp(q[2]), _dp(q[3]), _dp(fa), _dp(ea)))
        return q, fa, ea

    NOALLOC_MAX_VALUES = 1 << 19                              # DG_NOALLOC_MAX_VALUES of include/dg_habc.h

    def get_aux_fields_noalloc(self):
        """dg_get_aux_fields_noalloc: (face_aux, edge_aux) exactly as get_fields() returns them, but staged on the GPU
        through a fixed 4 MiB array built into libdg_habc.so instead of the solver's workspace, so the call never asks
        for device memory.  It is meant for hosts that cannot allocate when they want the data -- all device memory
        already given to another pool, another thread in a global-mode stream capture, a loop that cannot afford
        cudaMalloc's device-wide synchronisation.  Solvers with more than NOALLOC_MAX_VALUES auxiliary values
        (T*J*3*Nfp + E*J*J*2*(N+1)) raise DgError [-4].  The first call on a device looks up the array's address and
        should come before any stream capture; calls are serialised inside the library because they share the array."""
        fa = np.zeros((self.T, self.J, 3, self.Nfp))
        ea = np.zeros((self.E, self.J * self.J, 2, self.N + 1))
        _check(lib().dg_get_aux_fields_noalloc(self._h, _dp(fa), _dp(ea)))
        return fa, ea

    def device_view(self):
        """dg_get_device_ptrs: raw device addresses of the current state in the library's layout (q [K][Np][4], face
        auxiliary state [T][J][3][Nfp] + closure sum S [T][Nfp], edge auxiliary state [E][J*J][2][N+1]) and the element
        size in bytes.  Valid until the next step() flips the buffers; order reads after `self.stream`."""
        v = _DeviceView()
        _check(lib().dg_get_device_ptrs(self._h, C.byref(v)))
        return {k: getattr(v, k) for k, _ in _DeviceView._fields_ if k != "reserved"}

    def get_face_map(self):
        tet, face, axis, sign = (np.empty(self.T, dtype=np.int32) for _ in range(4))
        xyz = np.empty((self.T, self.Nfp, 3))
        _check(lib().dg_get_face_map(self._h, _ip(tet), _ip(face), _ip(axis), _ip(sign), _dp(xyz)))
        return tet, face, axis, sign, xyz

    def get_edge_map(self):
        axis = np.empty(self.E, dtype=np.int32)
        nax, sg = np.empty((self.E, 2), dtype=np.int32), np.empty((self.E, 2), dtype=np.int32)
        xyz = np.empty((self.E, self.N + 1, 3))
        _check(lib().dg_get_edge_map(self._h, _ip(axis), _ip(nax), _ip(sg), _dp(xyz)))
        return axis, nax, sg, xyz

    def last_step_kernel_ms(self):
        """dg_last_step_kernel_ms: device time of the 3D kernel in the five stages of the last step, from events recorded
        inside the step itself (Solver(..., time_kernels=True))."""
        ms = np.zeros(5)
        _check(lib().dg_last_step_kernel_ms(self._h, _dp(ms)))
        return ms

    def set_time_kernels(self, on: bool):
        """dg_set_time_kernels: switch the per-stage kernel events of dg_options.time_kernels on or off."""
        _check(lib().dg_set_time_kernels(self._h, int(bool(on))))

    def profile_step(self):
        ms = np.zeros(6)
        _check(lib().dg_profile_step(self._h, _dp(ms)))
        return dict(zip(("vol3d", "face2d", "edge1d", "close_face", "close_edge", "close_corner"), ms.tolist()))

    def synchronize(self):
        self._stream.synchronize()

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._stream.synchronize()          # dg_step is asynchronous: finish before the workspace goes back to torch
            lib().dg_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
