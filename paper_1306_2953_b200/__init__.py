"""Thin Python binding of librs.so (include/rs.h): argument marshalling only.

Every step of the path -- mesh enumeration, neighbour tables, pack/unpack, the fused stencil +
potential -- runs inside the library (C++ host code and hand-written sm_100a CUDA kernels).  PyTorch
appears only as the owner of device memory and streams: tensors are passed as raw pointers.

There is no CPU fallback: importing this package without a loadable librs.so raises, and the
compute calls raise RsError(RS_ERR_CUDA) when no CUDA device is present.

Function names mirror the C ABI (rs_mesh_create, rs_block_pack, rs_block_unpack,
rs_hamiltonian_apply, ...); see include/rs.h for the meaning of every argument and for the
passages of the paper that define each operation.
"""
from __future__ import annotations

import ctypes as C
import os
import shutil

import numpy as np

from . import build as _build

RS_OK, RS_ERR_INVALID_ARG, RS_ERR_ALLOC, RS_ERR_CUDA, RS_ERR_UNSUPPORTED = range(5)
RS_REAL64, RS_COMPLEX128 = 0, 1
RS_ORDER_BRICK, RS_ORDER_LEX, RS_ORDER_TILE = 0, 1, 2
RS_KERNEL_AUTO, RS_KERNEL_GATHER, RS_KERNEL_SWEEP = 0, 1, 2
RS_MAX_FD_ORDER = 8
RS_MAX_BLOCK = 64

_STATUS_NAMES = {0: "RS_OK", 1: "RS_ERR_INVALID_ARG", 2: "RS_ERR_ALLOC", 3: "RS_ERR_CUDA", 4: "RS_ERR_UNSUPPORTED"}

# every symbol include/rs.h declares (tests check that the library exports all of them)
EXPORTS = (
    "rs_mesh_create", "rs_mesh_create_ordered", "rs_mesh_create_box", "rs_mesh_destroy", "rs_mesh_npoints",
    "rs_mesh_spacing", "rs_mesh_nbricks", "rs_mesh_get_points", "rs_mesh_get_index_map", "rs_block_bytes",
    "rs_block_pack", "rs_block_unpack", "rs_hamiltonian_apply", "rs_hamiltonian_apply_v",
    "rs_hamiltonian_apply_states_host", "rs_last_error", "rs_kernel_name", "rs_kernel_table_bytes", "rs_version",
    "rs_sweep_options_default", "rs_mesh_set_sweep_options", "rs_hamiltonian_prepare",
    "rs_block_dot", "rs_block_expectation", "rs_block_expectation_static", "rs_block_axpy", "rs_block_copy", "rs_hamiltonian_apply_ex", "rs_block_overlap",
    "rs_nonlocal_create", "rs_nonlocal_destroy", "rs_nonlocal_sphere_size", "rs_nonlocal_get_sphere", "rs_nonlocal_set_projectors",
    "rs_nonlocal_ncolors", "rs_nonlocal_get_colors", "rs_nonlocal_prepare", "rs_nonlocal_apply",
    "rs_workspace_create", "rs_workspace_destroy", "rs_workspace_bytes", "rs_hamiltonian_apply_states_stream",
    "rs_sweep_selfcheck", "rs_sweep_stats", "rs_hamiltonian_autotune",
)


class SweepOptions(C.Structure):
    """rs_sweep_options of include/rs.h (per-mesh options of the plane-sweep kernel's work dealing)."""
    _fields_ = [("planes", C.c_int), ("planes_tuned", C.c_int), ("ctas", C.c_int), ("force_tensor", C.c_int),
                ("min_split", C.c_int), ("tune_rounds", C.c_int)]


class RsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


def _load() -> C.CDLL:
    so = _build.SO
    if _build.needs_build():
        if shutil.which(os.environ.get("NVCC", "nvcc")) is None:
            raise ImportError(f"{so} is missing or stale and nvcc is not available to build it; "
                              "there is no fallback path")
        _build.build(force=True, verbose=bool(os.environ.get("RS_BUILD_VERBOSE")))
    L = C.CDLL(so)
    vp, dp, i32p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.rs_mesh_create.argtypes = [dp, C.c_int, C.c_double, C.c_double, C.c_int, C.POINTER(vp)]
    L.rs_mesh_create_ordered.argtypes = [dp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.POINTER(vp)]
    L.rs_mesh_create_box.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.POINTER(vp)]
    L.rs_mesh_destroy.argtypes = [vp]
    L.rs_mesh_npoints.argtypes = [vp]
    L.rs_mesh_npoints.restype = C.c_int64
    L.rs_mesh_spacing.argtypes = [vp]
    L.rs_mesh_spacing.restype = C.c_double
    L.rs_mesh_nbricks.argtypes = [vp]
    L.rs_mesh_nbricks.restype = C.c_int64
    L.rs_mesh_get_points.argtypes = [vp, i32p]
    L.rs_mesh_get_index_map.argtypes = [vp, C.c_int, i32p]
    L.rs_block_bytes.argtypes = [vp, C.c_int, C.c_int]
    L.rs_block_bytes.restype = C.c_size_t
    L.rs_block_pack.argtypes = [vp, vp, C.c_int64, C.c_int, C.c_int, C.c_int, vp, C.c_int, vp]
    L.rs_block_unpack.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int64, C.c_int, C.c_int, vp]
    L.rs_hamiltonian_apply.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int, C.c_int, vp]
    L.rs_hamiltonian_autotune.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int, C.c_int, vp]
    L.rs_hamiltonian_apply_v.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int, C.c_int, vp, C.c_int]
    L.rs_hamiltonian_apply_states_host.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int64, C.c_int, C.c_int, C.c_int]
    L.rs_block_dot.argtypes = [vp, vp, vp, C.c_int, C.c_int, vp, vp]
    L.rs_block_expectation.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, vp, vp]
    L.rs_block_expectation_static.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, vp, vp]
    L.rs_block_axpy.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, vp]
    L.rs_nonlocal_create.argtypes = [vp, dp, C.c_int, C.c_double, C.c_int, C.POINTER(vp)]
    L.rs_nonlocal_destroy.argtypes = [vp]
    L.rs_nonlocal_sphere_size.argtypes = [vp, C.c_int]
    L.rs_nonlocal_sphere_size.restype = C.c_int64
    L.rs_nonlocal_get_sphere.argtypes = [vp, C.c_int, i32p]
    L.rs_nonlocal_set_projectors.argtypes = [vp, C.c_int, dp]
    L.rs_nonlocal_ncolors.argtypes = [vp]
    L.rs_nonlocal_get_colors.argtypes = [vp, i32p]
    L.rs_nonlocal_prepare.argtypes = [vp]
    L.rs_nonlocal_apply.argtypes = [vp, vp, vp, C.c_int, C.c_int, vp]
    L.rs_block_overlap.argtypes = [vp, vp, vp, C.c_int, C.c_int, vp, vp]
    L.rs_block_copy.argtypes = [vp, vp, vp, C.c_int, C.c_int, vp]
    L.rs_hamiltonian_apply_ex.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int, C.c_int, vp, vp, vp]
    L.rs_workspace_create.argtypes = [vp, C.c_int, C.c_int, C.c_int64, C.c_int, C.POINTER(vp)]
    L.rs_workspace_destroy.argtypes = [vp]
    L.rs_workspace_bytes.argtypes = [vp]
    L.rs_workspace_bytes.restype = C.c_size_t
    L.rs_hamiltonian_apply_states_stream.argtypes = [vp, C.c_int, dp, vp, vp, vp, C.c_int]
    L.rs_last_error.restype = C.c_char_p
    L.rs_kernel_name.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int]
    L.rs_kernel_name.restype = C.c_char_p
    L.rs_kernel_table_bytes.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int]
    L.rs_kernel_table_bytes.restype = C.c_int64
    L.rs_version.restype = C.c_int
    L.rs_sweep_options_default.argtypes = [C.POINTER(SweepOptions)]
    L.rs_mesh_set_sweep_options.argtypes = [vp, C.POINTER(SweepOptions)]
    L.rs_hamiltonian_prepare.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.rs_sweep_stats.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64), C.c_int64]
    L.rs_sweep_stats.restype = C.c_int64
    L.rs_sweep_selfcheck.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64)]
    return L


_lib = _load()
LIBRARY_PATH = _build.SO


def _check(status: int) -> None:
    if status != RS_OK:
        raise RsError(status, (_lib.rs_last_error() or b"").decode())


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ptr(t) -> int:
    """Raw address of a torch tensor (device or host) or a numpy array."""
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream) -> int:
    """cudaStream_t as an integer: None -> torch's current stream, int -> as given, torch Stream -> its handle."""
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _dtype_of(t) -> int:
    s = str(t.dtype)
    if s.endswith("float64"):
        return RS_REAL64
    if s.endswith("complex128"):
        return RS_COMPLEX128
    raise TypeError(f"unsupported element type {t.dtype}: the path computes in fp64 (real or complex)")


class Mesh:
    """Owner of an rs_mesh handle (host tables + device tables)."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.rs_mesh_destroy(h)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise RsError(RS_ERR_INVALID_ARG, "mesh already destroyed")
        return self._h

    @property
    def npoints(self) -> int:
        return int(_lib.rs_mesh_npoints(self.handle))

    @property
    def spacing(self) -> float:
        return float(_lib.rs_mesh_spacing(self.handle))

    @property
    def nbricks(self) -> int:
        return int(_lib.rs_mesh_nbricks(self.handle))

    def points(self) -> np.ndarray:
        return rs_mesh_get_points(self)

    def index_map(self, fd_order: int) -> np.ndarray:
        return rs_mesh_get_index_map(self, fd_order)


def rs_version() -> int:
    return int(_lib.rs_version())


def rs_sweep_options_default() -> SweepOptions:
    o = SweepOptions()
    _check(_lib.rs_sweep_options_default(C.byref(o)))
    return o


def rs_mesh_set_sweep_options(mesh, options: SweepOptions | None = None, **fields) -> None:
    """Set the mesh's plane-sweep options (defaults, overridden by `fields`); tables built so far are dropped."""
    o = options if options is not None else rs_sweep_options_default()
    for k, v in fields.items():
        if k not in dict(SweepOptions._fields_):
            raise RsError(RS_ERR_INVALID_ARG, f"unknown sweep option {k}")
        setattr(o, k, int(v))
    _check(_lib.rs_mesh_set_sweep_options(mesh.handle, C.byref(o)))


def rs_hamiltonian_prepare(mesh, fd_order: int, nst: int, dtype: int = RS_REAL64) -> None:
    """Build and upload the neighbour structure for (fd_order, nst, dtype) now; later applies allocate nothing."""
    _check(_lib.rs_hamiltonian_prepare(mesh.handle, fd_order, nst, dtype))


def rs_sweep_stats(mesh, fd_order: int, nst: int, dtype: int = RS_REAL64, max_ctas: int = 4096) -> np.ndarray:
    """[nctas][5] int64: {clock ticks of the last launch, steps, pieces, modelled load x1000, full warp-steps} per CTA."""
    out = np.zeros((max_ctas, 5), dtype=np.int64)
    n = _lib.rs_sweep_stats(mesh.handle, fd_order, nst, dtype, out.ctypes.data_as(C.POINTER(C.c_int64)), max_ctas)
    return out[:n]


def rs_sweep_selfcheck(mesh, fd_order: int, nst: int, dtype: int = RS_REAL64, max_planes: int = 32, nctas: int = 148) -> dict:
    """Host-only replay of the plane-sweep records against the plain neighbour table; raises on a discrepancy."""
    st = (C.c_int64 * 8)()
    _check(_lib.rs_sweep_selfcheck(mesh.handle, fd_order, nst, dtype, max_planes, nctas, st))
    return {"nctas": st[0], "records": st[1], "pieces": st[2], "cost_max": st[3] / 1000.0, "cost_mean": st[4] / 1000.0,
            "table_bytes": st[5], "fill_slots": st[6], "copy_runs": st[7]}


def rs_mesh_create(centers, radius: float, spacing: float, max_fd_order: int = 4,
                   ordering: int = RS_ORDER_LEX) -> Mesh:
    c = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1, 3)
    out = C.c_void_p()
    _check(_lib.rs_mesh_create_ordered(_dptr(c), c.shape[0], radius, spacing, max_fd_order, ordering, C.byref(out)))
    return Mesh(out.value)


def rs_mesh_create_box(nx: int, ny: int, nz: int, spacing: float, max_fd_order: int = 4, periodic: bool = False,
                       ordering: int = RS_ORDER_LEX) -> Mesh:
    out = C.c_void_p()
    _check(_lib.rs_mesh_create_box(nx, ny, nz, spacing, max_fd_order, int(periodic), ordering, C.byref(out)))
    return Mesh(out.value)


def rs_mesh_destroy(mesh: Mesh) -> None:
    h, mesh._h = mesh._h, None
    if h:
        _check(_lib.rs_mesh_destroy(h))


def rs_mesh_npoints(mesh: Mesh) -> int:
    return mesh.npoints


def rs_mesh_get_points(mesh: Mesh) -> np.ndarray:
    ijk = np.empty((mesh.npoints, 3), dtype=np.int32)
    _check(_lib.rs_mesh_get_points(mesh.handle, ijk.ctypes.data_as(C.POINTER(C.c_int32))))
    return ijk


def rs_mesh_get_index_map(mesh: Mesh, fd_order: int) -> np.ndarray:
    m = np.empty((mesh.npoints, 6 * fd_order), dtype=np.int32)
    _check(_lib.rs_mesh_get_index_map(mesh.handle, fd_order, m.ctypes.data_as(C.POINTER(C.c_int32))))
    return m


def rs_block_bytes(mesh: Mesh, block_size: int, dtype: int = RS_REAL64) -> int:
    return int(_lib.rs_block_bytes(mesh.handle, block_size, dtype))


def rs_block_pack(mesh: Mesh, states, ist0: int, nst_in_block: int, block_size: int, block, stream=None,
                  ld: int | None = None) -> None:
    """states: device tensor [nst_total][ld]; block: device tensor of rs_block_bytes() bytes."""
    ld = int(states.shape[-1]) if ld is None else ld
    _check(_lib.rs_block_pack(mesh.handle, _ptr(states), ld, ist0, nst_in_block, block_size, _ptr(block),
                              _dtype_of(states), _stream(stream)))


def rs_block_unpack(mesh: Mesh, block, block_size: int, nst_in_block: int, states, ist0: int, stream=None,
                    ld: int | None = None) -> None:
    ld = int(states.shape[-1]) if ld is None else ld
    _check(_lib.rs_block_unpack(mesh.handle, _ptr(block), block_size, nst_in_block, _ptr(states), ld, ist0,
                                _dtype_of(states), _stream(stream)))


def rs_hamiltonian_apply(mesh: Mesh, fd_order: int, coeffs, vloc, psi, hpsi, nst: int, dtype: int | None = None,
                         stream=None, kernel: int = RS_KERNEL_AUTO) -> None:
    """hpsi <- -1/2 Lap psi + vloc psi on one block of width nst (device tensors); asynchronous on `stream`."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    if c.shape != (fd_order + 1,):
        raise RsError(RS_ERR_INVALID_ARG, "coeffs must hold c_0..c_n")
    dtype = _dtype_of(psi) if dtype is None else dtype
    _check(_lib.rs_hamiltonian_apply_v(mesh.handle, fd_order, _dptr(c), _ptr(vloc), _ptr(psi), _ptr(hpsi), nst,
                                       dtype, _stream(stream), kernel))


def rs_hamiltonian_autotune(mesh: Mesh, fd_order: int, coeffs, vloc, psi, hpsi, nst: int, dtype: int | None = None,
                            stream=None) -> None:
    """Once per (mesh, order, width): measure the plane-sweep kernel's per-step costs on these buffers and re-deal the
    work to the CTAs accordingly (synchronises the stream; hpsi receives H psi)."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    if c.shape != (fd_order + 1,):
        raise RsError(RS_ERR_INVALID_ARG, "coeffs must hold c_0..c_n")
    dtype = _dtype_of(psi) if dtype is None else dtype
    _check(_lib.rs_hamiltonian_autotune(mesh.handle, fd_order, _dptr(c), _ptr(vloc), _ptr(psi), _ptr(hpsi), nst, dtype,
                                        _stream(stream)))


def rs_hamiltonian_apply_states_host(mesh: Mesh, fd_order: int, coeffs, vloc_host, states_host, hstates_host,
                                     block_size: int) -> None:
    """Whole path on HOST arrays [nst_total][ld] (numpy or CPU torch tensors): H2D, pack/apply/unpack per block, D2H."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    nst_total, ld = int(states_host.shape[0]), int(states_host.shape[1])
    _check(_lib.rs_hamiltonian_apply_states_host(mesh.handle, fd_order, _dptr(c), _ptr(vloc_host), _ptr(states_host),
                                                 _ptr(hstates_host), ld, nst_total, block_size,
                                                 _dtype_of(states_host)))


def rs_block_dot(mesh: Mesh, a, b, nst: int, out, stream=None) -> None:
    """out[j] = sum_p conj(a[p][j]) b[p][j] (device tensors; out: nst elements of the blocks' dtype)."""
    _check(_lib.rs_block_dot(mesh.handle, _ptr(a), _ptr(b), nst, _dtype_of(a), _ptr(out), _stream(stream)))


def rs_block_expectation(mesh: Mesh, psi, hpsi, eps, nst: int, out, stream=None) -> None:
    """out[3][nst] float64 = Re<psi|hpsi>, |psi|^2, |hpsi - eps psi|^2 per orbital (eps: device float64 [nst] or None)."""
    _check(_lib.rs_block_expectation(mesh.handle, _ptr(psi), _ptr(hpsi), _ptr(eps) if eps is not None else None, nst,
                                     _dtype_of(psi), _ptr(out), _stream(stream)))


def rs_block_expectation_static(mesh: Mesh, psi, hpsi, eps, nst: int, out, stream=None) -> None:
    """rs_block_expectation without any allocation: partial sums in the library's static device array (<= 64 real
    columns; calls that overlap on the GPU race).  Same output, bit for bit."""
    _check(_lib.rs_block_expectation_static(mesh.handle, _ptr(psi), _ptr(hpsi), _ptr(eps) if eps is not None else None, nst,
                                            _dtype_of(psi), _ptr(out), _stream(stream)))


def rs_block_axpy(mesh: Mesh, alpha, x, y, nst: int, stream=None) -> None:
    """y[p][j] += alpha[j] x[p][j] (alpha: device tensor of nst elements of the blocks' dtype)."""
    _check(_lib.rs_block_axpy(mesh.handle, _ptr(alpha), _ptr(x), _ptr(y), nst, _dtype_of(x), _stream(stream)))


def rs_block_overlap(mesh: Mesh, a, b, nst: int, M, stream=None) -> None:
    """M[j][k] = sum_p conj(a[p][j]) b[p][k] (device tensors; M: [nst][nst] of the blocks' dtype): eqs. 5 / 7."""
    _check(_lib.rs_block_overlap(mesh.handle, _ptr(a), _ptr(b), nst, _dtype_of(a), _ptr(M), _stream(stream)))


def rs_block_copy(mesh: Mesh, src, dst, nst: int, stream=None) -> None:
    _check(_lib.rs_block_copy(mesh.handle, _ptr(src), _ptr(dst), nst, _dtype_of(src), _stream(stream)))


def rs_hamiltonian_apply_ex(mesh: Mesh, fd_order: int, coeffs, vloc, psi, hpsi, nst: int, eps, sums, stream=None) -> None:
    """rs_hamiltonian_apply plus sums[3][nst] = Re<psi|H psi>, |psi|^2, |H psi - eps psi|^2 from the same call."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    if c.shape != (fd_order + 1,):
        raise RsError(RS_ERR_INVALID_ARG, "coeffs must hold c_0..c_n")
    _check(_lib.rs_hamiltonian_apply_ex(mesh.handle, fd_order, _dptr(c), _ptr(vloc), _ptr(psi), _ptr(hpsi), nst,
                                        _dtype_of(psi), _stream(stream), _ptr(eps) if eps is not None else None, _ptr(sums)))


class NonLocal:
    """Owner of an rs_nonlocal handle (projector spheres, colouring, device tables); keeps its mesh alive."""

    def __init__(self, mesh: Mesh, centers, rc: float, nlm: int):
        c = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1, 3)
        out = C.c_void_p()
        _check(_lib.rs_nonlocal_create(mesh.handle, _dptr(c), c.shape[0], rc, nlm, C.byref(out)))
        self._h, self.mesh, self.natoms, self.nlm = out, mesh, c.shape[0], nlm

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.rs_nonlocal_destroy(h)

    def sphere(self, atom: int) -> np.ndarray:
        """mesh indices (ascending) of the atom's sphere points = the row order of its projector table."""
        n = int(_lib.rs_nonlocal_sphere_size(self._h, atom))
        if n < 0:
            raise RsError(RS_ERR_INVALID_ARG, "bad atom index")
        idx = np.empty(n, dtype=np.int32)
        _check(_lib.rs_nonlocal_get_sphere(self._h, atom, idx.ctypes.data_as(C.POINTER(C.c_int32))))
        return idx

    def set_projectors(self, atom: int, gamma) -> None:
        g = np.ascontiguousarray(gamma, dtype=np.float64)
        if g.shape != (int(_lib.rs_nonlocal_sphere_size(self._h, atom)), self.nlm):
            raise RsError(RS_ERR_INVALID_ARG, "projector table must be [sphere points][nlm]")
        _check(_lib.rs_nonlocal_set_projectors(self._h, atom, _dptr(g)))

    @property
    def ncolors(self) -> int:
        return int(_lib.rs_nonlocal_ncolors(self._h))

    def colors(self) -> np.ndarray:
        c = np.empty(self.natoms, dtype=np.int32)
        _check(_lib.rs_nonlocal_get_colors(self._h, c.ctypes.data_as(C.POINTER(C.c_int32))))
        return c

    def prepare(self) -> None:
        _check(_lib.rs_nonlocal_prepare(self._h))


def rs_nonlocal_create(mesh: Mesh, centers, rc: float, nlm: int) -> NonLocal:
    return NonLocal(mesh, centers, rc, nlm)


def rs_nonlocal_apply(nl: NonLocal, psi, hpsi, nst: int, stream=None) -> None:
    """hpsi += V_nl psi on one block (eq. 4 of the paper); device tensors."""
    _check(_lib.rs_nonlocal_apply(nl._h, _ptr(psi), _ptr(hpsi), nst, _dtype_of(psi), _stream(stream)))


class Workspace:
    """Owner of an rs_workspace handle (ring of block-sized device windows + streams); keeps its mesh alive."""

    def __init__(self, mesh: Mesh, block_size: int, dtype: int, ld: int, nbuf: int = 3):
        out = C.c_void_p()
        _check(_lib.rs_workspace_create(mesh.handle, block_size, dtype, ld, nbuf, C.byref(out)))
        self._h, self.mesh, self.block_size, self.dtype, self.ld = out, mesh, block_size, dtype, ld

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _lib is not None:
            _lib.rs_workspace_destroy(h)

    @property
    def nbytes(self) -> int:
        return int(_lib.rs_workspace_bytes(self._h))


def rs_workspace_create(mesh: Mesh, block_size: int, dtype: int, ld: int, nbuf: int = 3) -> Workspace:
    return Workspace(mesh, block_size, dtype, ld, nbuf)


def rs_hamiltonian_apply_states_stream(ws: Workspace, fd_order: int, coeffs, vloc_host, states_host, hstates_host) -> None:
    """Whole path on HOST arrays [nst_total][ld] through a workspace created once (no allocation per call)."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    nst_total, ld = int(states_host.shape[0]), int(states_host.shape[1])
    if ld != ws.ld or _dtype_of(states_host) != ws.dtype:
        raise RsError(RS_ERR_INVALID_ARG, "states do not match the workspace (leading dimension / dtype)")
    _check(_lib.rs_hamiltonian_apply_states_stream(ws._h, fd_order, _dptr(c), _ptr(vloc_host), _ptr(states_host),
                                                   _ptr(hstates_host), nst_total))


def rs_kernel_name(mesh: Mesh, fd_order: int, nst: int, dtype: int = RS_REAL64, kernel: int = RS_KERNEL_AUTO) -> str:
    return _lib.rs_kernel_name(mesh.handle, fd_order, nst, dtype, kernel).decode()


def rs_kernel_table_bytes(mesh: Mesh, fd_order: int, nst: int, dtype: int = RS_REAL64,
                          kernel: int = RS_KERNEL_AUTO) -> int:
    return int(_lib.rs_kernel_table_bytes(mesh.handle, fd_order, nst, dtype, kernel))
