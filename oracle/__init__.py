"""Python face of the CPU oracle (oracle/oracle.c) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports the CUDA package and shares no code with it.
Every function cites the passage it follows in oracle.c's header.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_SRC_NEXT = os.path.join(_HERE, "oracle_next.c")      # SURVEY.md section 8(f) rows (block BLAS-1, overlap, non-local)
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (-O2, no FMA contraction so the summation order is the source's)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_NEXT)):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99",
               "-o", _SO, _SRC, _SRC_NEXT, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, u8p, i64p = (C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_uint8),
                             C.POINTER(C.c_int64))
        L.orc_fd_coeffs.argtypes = [C.c_int, dp]
        L.orc_fd_coeffs.restype = C.c_int
        L.orc_bbox.argtypes = [dp, C.c_int, C.c_double, C.c_double, ip, ip]
        L.orc_bbox.restype = None
        L.orc_mask.argtypes = [dp, C.c_int, C.c_double, C.c_double, ip, ip, u8p]
        L.orc_mask.restype = C.c_int64
        L.orc_count_outside_arms.argtypes = [C.c_int, ip, u8p]
        L.orc_count_outside_arms.restype = C.c_int64
        L.orc_vloc.argtypes = [dp, dp, C.c_int, dp, C.c_int64, dp]
        L.orc_vloc.restype = None
        L.orc_hpsi_dense.argtypes = [C.c_int, dp, C.c_double, ip, C.c_int, u8p, dp, dp, dp, C.c_int]
        L.orc_hpsi_dense.restype = None
        L.orc_hpsi_states.argtypes = [C.c_int, dp, C.c_double, ip, C.c_int, u8p, dp, i64p, C.c_int64, dp, dp,
                                      C.c_int, C.c_int, C.c_int, dp]
        L.orc_hpsi_states.restype = C.c_int
        L.orc_block_pack.argtypes = [dp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int64, C.c_int64, dp, C.c_int]
        L.orc_block_pack.restype = None
        L.orc_block_unpack.argtypes = [dp, C.c_int, C.c_int, C.c_int64, dp, C.c_int64, C.c_int, C.c_int]
        L.orc_block_unpack.restype = None
        i32p = C.POINTER(C.c_int32)
        L.orc_block_dot.argtypes = [dp, dp, C.c_int64, C.c_int, C.c_int, dp]
        L.orc_block_dot.restype = None
        L.orc_block_axpy.argtypes = [dp, dp, dp, C.c_int64, C.c_int, C.c_int]
        L.orc_block_axpy.restype = None
        L.orc_block_residual.argtypes = [dp, dp, dp, C.c_int64, C.c_int, C.c_int, dp]
        L.orc_block_residual.restype = None
        L.orc_overlap.argtypes = [dp, C.c_int, dp, C.c_int, C.c_int64, C.c_int, dp]
        L.orc_overlap.restype = None
        L.orc_sphere_points.argtypes = [i32p, C.c_int64, C.c_double, dp, C.c_double, i64p]
        L.orc_sphere_points.restype = C.c_int64
        L.orc_nonlocal.argtypes = [C.c_int, i64p, i64p, i64p, dp, C.c_int, C.c_double, dp, dp, C.c_int64, C.c_int, C.c_int]
        L.orc_nonlocal.restype = None
        _lib = L
    return _lib


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def fd_coeffs(n: int) -> np.ndarray:
    """c_0..c_n of the half-width-n central second-derivative stencil (reading S1)."""
    c = np.zeros(n + 1)
    if lib().orc_fd_coeffs(n, _p(c, C.c_double)) != 0:
        raise ValueError("bad order")
    return c


@dataclass
class Mesh:
    """The oracle's own mesh: bounding lattice + in-domain mask; canonical order = lexicographic
    (i, j, k) over in-domain points = ascending dense index."""
    lo: np.ndarray       # [3] int32, lattice index of dense (0,0,0)
    dims: np.ndarray     # [3] int32
    spacing: float
    mask: np.ndarray     # [nx*ny*nz] uint8
    periodic: bool = False

    def __post_init__(self):
        self.canon = np.flatnonzero(self.mask).astype(np.int64)   # canonical ip -> dense index
        self.npoints = int(self.canon.size)

    @property
    def nbox(self) -> int:
        return int(np.prod(self.dims.astype(np.int64)))

    def ijk(self) -> np.ndarray:
        """[np][3] int32 lattice indices of the canonical points."""
        nx, ny, nz = (int(d) for d in self.dims)
        q = self.canon
        out = np.empty((q.size, 3), dtype=np.int32)
        out[:, 0] = q // (ny * nz) + self.lo[0]
        out[:, 1] = (q // nz) % ny + self.lo[1]
        out[:, 2] = q % nz + self.lo[2]
        return out

    def xyz(self) -> np.ndarray:
        return self.ijk().astype(np.float64) * self.spacing

    def dense_index_of(self, ijk: np.ndarray) -> np.ndarray:
        """dense index of arbitrary lattice points (must lie in the bounding box)."""
        rel = ijk.astype(np.int64) - self.lo.astype(np.int64)
        if (rel < 0).any() or (rel >= self.dims.astype(np.int64)).any():
            raise ValueError("point outside the oracle's bounding box")
        return (rel[:, 0] * int(self.dims[1]) + rel[:, 1]) * int(self.dims[2]) + rel[:, 2]

    def canonical_rank_of(self, ijk: np.ndarray) -> np.ndarray:
        """canonical index of the given in-domain lattice points (raises if any is outside Omega)."""
        q = self.dense_index_of(ijk)
        if not self.mask[q].all():
            raise ValueError("point outside the oracle's domain")
        rank = np.cumsum(self.mask, dtype=np.int64) - 1
        return rank[q]

    def to_dense(self, f_canon: np.ndarray) -> np.ndarray:
        d = np.zeros(self.nbox, dtype=f_canon.dtype)
        d[self.canon] = f_canon
        return d


def mesh_from_spheres(centers: np.ndarray, radius: float, spacing: float) -> Mesh:
    """Union of closed balls on the lattice h*Z^3 (readings S3/S4)."""
    centers = np.ascontiguousarray(centers, dtype=np.float64)
    lo = np.zeros(3, dtype=np.int32)
    dims = np.zeros(3, dtype=np.int32)
    lib().orc_bbox(_p(centers, C.c_double), centers.shape[0], radius, spacing, _p(lo, C.c_int), _p(dims, C.c_int))
    mask = np.zeros(int(np.prod(dims.astype(np.int64))), dtype=np.uint8)
    n = lib().orc_mask(_p(centers, C.c_double), centers.shape[0], radius, spacing, _p(lo, C.c_int),
                       _p(dims, C.c_int), _p(mask, C.c_uint8))
    m = Mesh(lo, dims, spacing, mask)
    assert m.npoints == n
    return m


def mesh_box(nx: int, ny: int, nz: int, spacing: float, periodic: bool) -> Mesh:
    """Full rectangular test box, lattice indices 0..n-1 (pins P2, P3, P5, P7)."""
    dims = np.array([nx, ny, nz], dtype=np.int32)
    return Mesh(np.zeros(3, dtype=np.int32), dims, spacing, np.ones(nx * ny * nz, dtype=np.uint8), periodic)


def mesh_from_mask(mask3d: np.ndarray, spacing: float) -> Mesh:
    dims = np.array(mask3d.shape, dtype=np.int32)
    return Mesh(np.zeros(3, dtype=np.int32), dims, spacing, np.ascontiguousarray(mask3d, dtype=np.uint8).ravel())


def count_outside_arms(mesh: Mesh, n: int) -> int:
    return int(lib().orc_count_outside_arms(n, _p(mesh.dims, C.c_int), _p(mesh.mask, C.c_uint8)))


def vloc(centers: np.ndarray, charges: np.ndarray, xyz: np.ndarray) -> np.ndarray:
    centers = np.ascontiguousarray(centers, dtype=np.float64)
    charges = np.ascontiguousarray(charges, dtype=np.float64)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    v = np.zeros(xyz.shape[0])
    lib().orc_vloc(_p(centers, C.c_double), _p(charges, C.c_double), centers.shape[0], _p(xyz, C.c_double),
                   xyz.shape[0], _p(v, C.c_double))
    return v


def hpsi_dense(mesh: Mesh, n: int, coeffs: np.ndarray, v_dense: np.ndarray, psi_dense: np.ndarray) -> np.ndarray:
    """H psi for ONE orbital given on the dense bounding lattice (real or complex)."""
    lanes = 2 if np.iscomplexobj(psi_dense) else 1
    psi_dense = np.ascontiguousarray(psi_dense)
    out = np.zeros_like(psi_dense)
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    v = np.ascontiguousarray(v_dense, dtype=np.float64)
    lib().orc_hpsi_dense(n, _p(c, C.c_double), mesh.spacing, _p(mesh.dims, C.c_int), int(mesh.periodic),
                         _p(mesh.mask, C.c_uint8), _p(v, C.c_double),
                         psi_dense.ctypes.data_as(C.POINTER(C.c_double)),
                         out.ctypes.data_as(C.POINTER(C.c_double)), lanes)
    return out


def hpsi(mesh: Mesh, n: int, coeffs: np.ndarray, v_canon: np.ndarray, psi_canon: np.ndarray,
         nthreads: int = 1) -> np.ndarray:
    """H psi for psi_canon[nst][np] (canonical point order), one orbital at a time."""
    psi_canon = np.ascontiguousarray(psi_canon)
    if psi_canon.ndim == 1:
        return hpsi(mesh, n, coeffs, v_canon, psi_canon[None, :], nthreads)[0]
    lanes = 2 if np.iscomplexobj(psi_canon) else 1
    nst, npts = psi_canon.shape
    assert npts == mesh.npoints
    out = np.zeros_like(psi_canon)
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    vd = mesh.to_dense(np.ascontiguousarray(v_canon, dtype=np.float64))
    nthreads = max(1, min(nthreads, nst))
    scratch = np.empty(nthreads * 2 * mesh.nbox * lanes)
    lib().orc_hpsi_states(n, _p(c, C.c_double), mesh.spacing, _p(mesh.dims, C.c_int), int(mesh.periodic),
                          _p(mesh.mask, C.c_uint8), _p(vd, C.c_double), _p(mesh.canon, C.c_int64), npts,
                          psi_canon.ctypes.data_as(C.POINTER(C.c_double)),
                          out.ctypes.data_as(C.POINTER(C.c_double)), nst, lanes, nthreads,
                          _p(scratch, C.c_double))
    return out


def block_pack(states: np.ndarray, ist0: int, nst_in_block: int, B: int, npts: int, nrows: int) -> np.ndarray:
    """Fig. 4: [nst][ld] -> [nrows][B], orbital index fastest; padding = 0."""
    states = np.ascontiguousarray(states)
    lanes = 2 if np.iscomplexobj(states) else 1
    blk = np.empty((nrows, B), dtype=states.dtype)
    lib().orc_block_pack(states.ctypes.data_as(C.POINTER(C.c_double)), states.shape[1], ist0, nst_in_block, B,
                         npts, nrows, blk.ctypes.data_as(C.POINTER(C.c_double)), lanes)
    return blk


def block_unpack(block: np.ndarray, nst_in_block: int, npts: int, states: np.ndarray, ist0: int) -> None:
    lanes = 2 if np.iscomplexobj(block) else 1
    assert states.flags.c_contiguous and block.flags.c_contiguous and states.dtype == block.dtype
    lib().orc_block_unpack(block.ctypes.data_as(C.POINTER(C.c_double)), block.shape[1], nst_in_block, npts,
                           states.ctypes.data_as(C.POINTER(C.c_double)), states.shape[1], ist0, lanes)


# ---- oracle_next.c ---------------------------------------------------------------
def _as2d(a):
    a = np.ascontiguousarray(a)
    return a[None, :] if a.ndim == 1 else a


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def block_dot(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """out[j] = sum_p conj(a[j][p]) b[j][p]   (sec. VIII; plain sums, reading S11)."""
    a, b = _as2d(a), _as2d(b)
    assert a.shape == b.shape and a.dtype == b.dtype
    lanes = 2 if np.iscomplexobj(a) else 1
    out = np.zeros(a.shape[0], dtype=a.dtype)
    lib().orc_block_dot(_dp(a), _dp(b), a.shape[1], a.shape[0], lanes, _dp(out))
    return out


def block_axpy(alpha: np.ndarray, x: np.ndarray, y: np.ndarray) -> np.ndarray:
    """returns y + alpha_j x_j per orbital (linear combination)."""
    x = _as2d(x)
    y = np.array(_as2d(y), copy=True, order="C")
    assert x.shape == y.shape and x.dtype == y.dtype
    lanes = 2 if np.iscomplexobj(x) else 1
    alpha = np.ascontiguousarray(alpha, dtype=x.dtype)
    assert alpha.shape == (x.shape[0],)
    lib().orc_block_axpy(_dp(alpha), _dp(x), _dp(y), x.shape[1], x.shape[0], lanes)
    return y


def block_residual(hpsi_: np.ndarray, psi: np.ndarray, eps: np.ndarray) -> np.ndarray:
    """r_j = (H psi)_j - eps_j psi_j, eps real (RMM-DIIS residual)."""
    hpsi_, psi = _as2d(hpsi_), _as2d(psi)
    assert hpsi_.shape == psi.shape and hpsi_.dtype == psi.dtype
    lanes = 2 if np.iscomplexobj(psi) else 1
    eps = np.ascontiguousarray(eps, dtype=np.float64)
    assert eps.shape == (psi.shape[0],)
    r = np.empty_like(psi)
    lib().orc_block_residual(_dp(hpsi_), _dp(psi), _dp(eps), psi.shape[1], psi.shape[0], lanes, _dp(r))
    return r


def overlap(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """M[j][k] = sum_p conj(a[j][p]) b[k][p]: S (eq. 5, b = a) or h (eq. 7, b = H a)."""
    a, b = _as2d(a), _as2d(b)
    assert a.shape[1] == b.shape[1] and a.dtype == b.dtype
    lanes = 2 if np.iscomplexobj(a) else 1
    M = np.zeros((a.shape[0], b.shape[0]), dtype=a.dtype)
    lib().orc_overlap(_dp(a), a.shape[0], _dp(b), b.shape[0], a.shape[1], lanes, _dp(M))
    return M


@dataclass
class Projectors:
    """Non-local projector data in the oracle's canonical point order (eq. 4)."""
    off: np.ndarray      # [natoms] int64 offsets into idx / gamma
    npts: np.ndarray     # [natoms] int64 sphere sizes
    idx: np.ndarray      # [sum npts] int64 canonical point indices, ascending per atom
    gamma: np.ndarray    # [sum npts][nlm] float64 projector values (INPUT)
    nlm: int


def sphere_points(mesh: Mesh, center, rc: float) -> np.ndarray:
    """canonical indices of the mesh points in the closed ball of radius rc around `center` (ascending)."""
    ijk = np.ascontiguousarray(mesh.ijk(), dtype=np.int32)
    ctr = np.ascontiguousarray(center, dtype=np.float64)
    n = lib().orc_sphere_points(ijk.ctypes.data_as(C.POINTER(C.c_int32)), mesh.npoints, mesh.spacing, _dp(ctr), rc, None)
    idx = np.empty(n, dtype=np.int64)
    lib().orc_sphere_points(ijk.ctypes.data_as(C.POINTER(C.c_int32)), mesh.npoints, mesh.spacing, _dp(ctr), rc,
                            idx.ctypes.data_as(C.POINTER(C.c_int64)))
    return idx


def make_projectors(mesh: Mesh, centers: np.ndarray, rc: float, values_at) -> Projectors:
    """values_at(xyz_relative [n][3]) -> [n][nlm]: the projector values are an input supplied by the caller."""
    centers = np.ascontiguousarray(centers, dtype=np.float64).reshape(-1, 3)
    xyz = mesh.xyz()
    idxs, gam = [], []
    for A in range(centers.shape[0]):
        ix = sphere_points(mesh, centers[A], rc)
        idxs.append(ix)
        gam.append(np.ascontiguousarray(values_at(xyz[ix] - centers[A]), dtype=np.float64).reshape(ix.size, -1))
    npts = np.array([i.size for i in idxs], dtype=np.int64)
    off = np.concatenate([[0], np.cumsum(npts)[:-1]]).astype(np.int64)
    nlm = gam[0].shape[1]
    return Projectors(off, npts, np.concatenate(idxs).astype(np.int64), np.ascontiguousarray(np.concatenate(gam, axis=0)), nlm)


def nonlocal_apply(mesh: Mesh, proj: Projectors, psi: np.ndarray, out: np.ndarray | None = None) -> np.ndarray:
    """out + V_nl psi (eq. 4; integral = h^3 * lattice sum); out defaults to zeros."""
    psi = _as2d(psi)
    lanes = 2 if np.iscomplexobj(psi) else 1
    res = np.zeros_like(psi) if out is None else np.array(_as2d(out), copy=True, order="C")
    lib().orc_nonlocal(int(proj.off.size), proj.off.ctypes.data_as(C.POINTER(C.c_int64)),
                       proj.npts.ctypes.data_as(C.POINTER(C.c_int64)), proj.idx.ctypes.data_as(C.POINTER(C.c_int64)),
                       _dp(proj.gamma), proj.nlm, mesh.spacing ** 3, _dp(psi), _dp(res), psi.shape[1], psi.shape[0], lanes)
    return res
