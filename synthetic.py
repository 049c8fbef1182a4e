"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the tests, the bench, the oracle harness and the CUDA
harness.  It holds NONE of the method's arithmetic (no stencil, no mesh
enumeration, no neighbour map, no layout transform): it only produces the
*inputs* of the path -- atom centres, charges, the synthetic local potential
sampled at caller-supplied coordinates, and N(0,1) orbitals in canonical
(lexicographic i,j,k) point order.

Recipe (BASELINE.json "configs"):
  * config 0: one centre at the origin, Z=4, R=4.0, h=0.30, nst=4 real, seed 0.
  * config 1: benzene-shaped, 6 centres Z=4 on a hexagon of radius 2.64 bohr and
    6 centres Z=1 at radius 4.68 bohr on the same rays (angles 0,60,..; z=0),
    R=5.0, h=0.20, nst=16 real, seed 1.
  * config 2: 100 centres uniform in a 20-bohr cube, rejection-sampled to a
    minimum separation of 2.5 bohr, Z from {1,4,5,6}, seed 2; R=5.0, h=0.20;
    nst=256 real.
  * config 3: config 2's mesh and potential, nst=128 complex, seed 3.
  * config 4: 500 centres in a 35-bohr cube, min separation 2.3 bohr, seed 4;
    R=4.5, h=0.25; nst=1024 real; fd orders 4 and 6.
They stand in for the paper's molecules (beta-cyclodextrin 260k points / 256
orbitals; Table I set), whose geometries and
pseudopotentials are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SOFT = 0.5  # bohr; V(r) = -Z erf(r/SOFT)/r   (BASELINE.json config 0)


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    centers: np.ndarray  # [nc][3] float64, bohr
    charges: np.ndarray  # [nc] float64
    radius: float
    spacing: float
    fd_orders: tuple
    nst: int
    is_complex: bool
    seed: int
    block_sizes: tuple
    np_expected: int | None = None  # survey scratch count, informational
    extra: dict = field(default_factory=dict)


def _hexagon(radius: float) -> np.ndarray:
    ang = np.deg2rad(60.0 * np.arange(6))
    return np.stack([radius * np.cos(ang), radius * np.sin(ang), np.zeros(6)], axis=1)


def benzene_centers() -> tuple[np.ndarray, np.ndarray]:
    c = np.concatenate([_hexagon(2.64), _hexagon(4.68)], axis=0)
    z = np.concatenate([np.full(6, 4.0), np.full(6, 1.0)])
    return c, z


def cluster_centers(n: int, box: float, dmin: float, seed: int) -> tuple[np.ndarray, np.ndarray]:
    """Rejection-sample n centres uniform in [0,box]^3 with pair distance >= dmin,
    then draw Z from {1,4,5,6} (proposed procedure)."""
    rng = np.random.default_rng(seed)
    acc: list[np.ndarray] = []
    while len(acc) < n:
        p = rng.uniform(0.0, box, 3)
        if all(np.linalg.norm(p - q) >= dmin for q in acc):
            acc.append(p)
    z = rng.choice(np.array([1.0, 4.0, 5.0, 6.0]), n)
    return np.array(acc), z


def config(i: int) -> Config:
    if i == 0:
        return Config(0, "tiny-atom", np.zeros((1, 3)), np.array([4.0]), 4.0, 0.30, (4,), 4, False, 0,
                      (4,), 9843)
    if i == 1:
        c, z = benzene_centers()
        return Config(1, "benzene-shaped", c, z, 5.0, 0.20, (4,), 16, False, 1, (1, 2, 4, 8, 16), 261987)
    if i in (2, 3):
        c, z = cluster_centers(100, 20.0, 2.5, 2)
        if i == 2:
            return Config(2, "100-atom", c, z, 5.0, 0.20, (4,), 256, False, 2, (1, 2, 4, 8, 16, 32, 64), 1959454)
        return Config(3, "100-atom-complex", c, z, 5.0, 0.20, (4,), 128, True, 3, (1, 2, 4, 8, 16, 32), 1959454)
    if i == 4:
        c, z = cluster_centers(500, 35.0, 2.3, 4)
        return Config(4, "500-atom", c, z, 4.5, 0.25, (4, 6), 1024, False, 4, (16, 32, 64), 3803534)
    raise ValueError(f"no config {i}")


def vloc_at(xyz: np.ndarray, centers: np.ndarray, charges: np.ndarray, chunk: int = 1 << 18) -> np.ndarray:
    """Synthetic local potential V(r) = sum_A -Z_A erf(rho_A/0.5)/rho_A at the given
    coordinates (every centre contributes everywhere; rho -> 0 limit -Z*2/(0.5*sqrt(pi))).
    It is an INPUT of the path, not part of the method."""
    from scipy.special import erf

    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    out = np.zeros(xyz.shape[0])
    lim = 2.0 / (SOFT * math.sqrt(math.pi))
    for s in range(0, xyz.shape[0], chunk):
        p = xyz[s:s + chunk]
        v = np.zeros(p.shape[0])
        for a in range(centers.shape[0]):
            rho = np.sqrt(((p - centers[a]) ** 2).sum(axis=1))
            small = rho < 1e-12
            safe = np.where(small, 1.0, rho)
            term = np.where(small, lim, erf(safe / SOFT) / safe)
            v -= charges[a] * term
        out[s:s + chunk] = v
    return out


def projector_values(xyz_rel: np.ndarray, lmax: int = 1, sigma: float = 0.7) -> np.ndarray:
    """Synthetic stand-ins for the pseudopotential projectors gamma_lm(r - R_A) of PAPER.md:181 (eq. 4), whose real
    data are not available: a Gaussian exp(-r^2/(2 sigma^2)) times the real solid harmonics up to lmax <= 3
    (1; x, y, z; xy, yz, zx, x^2-y^2, 3z^2-r^2; the seven cubic ones), unnormalised.  An INPUT of the path, sampled at caller-supplied coordinates
    relative to the atom; the caller decides which points lie inside the cut-off sphere.  Returns [n][(lmax+1)^2]."""
    p = np.ascontiguousarray(xyz_rel, dtype=np.float64).reshape(-1, 3)
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    r2 = x * x + y * y + z * z
    g = np.exp(-r2 / (2.0 * sigma * sigma))
    cols = [np.ones_like(x)]
    if lmax >= 1:
        cols += [x, y, z]
    if lmax >= 2:
        cols += [x * y, y * z, z * x, x * x - y * y, 3.0 * z * z - r2]
    if lmax >= 3:
        cols += [z * (5.0 * z * z - 3.0 * r2), x * (5.0 * z * z - r2), y * (5.0 * z * z - r2), z * (x * x - y * y), x * y * z,
                 x * (x * x - 3.0 * y * y), y * (3.0 * x * x - y * y)]
    if lmax > 3:
        raise ValueError("lmax <= 3")
    return np.stack(cols, axis=1) * g[:, None]


def orbital(seed: int, ist: int, npts: int, is_complex: bool = False) -> np.ndarray:
    """Orbital `ist` as i.i.d. N(0,1) values in canonical (lexicographic i,j,k) point order;
    complex: a second draw of npts for the imaginary part."""
    rng = np.random.default_rng([seed, ist])
    re = rng.standard_normal(npts)
    if not is_complex:
        return re
    im = rng.standard_normal(npts)
    return re + 1j * im


def orbitals(seed: int, ist0: int, nst: int, npts: int, is_complex: bool = False) -> np.ndarray:
    """[nst][npts] array of orbitals ist0 .. ist0+nst-1 (canonical point order)."""
    out = np.empty((nst, npts), dtype=np.complex128 if is_complex else np.float64)
    for j in range(nst):
        out[j] = orbital(seed, ist0 + j, npts, is_complex)
    return out


def shard_orbitals(nst_total: int, block: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range [ist0, ist1) of orbitals owned by `rank`: whole blocks, dealt out as
    evenly as possible (orbitals are independent, no exchange)."""
    nblk = (nst_total + block - 1) // block
    lo = (nblk * rank) // world
    hi = (nblk * (rank + 1)) // world
    return min(lo * block, nst_total), min(hi * block, nst_total)


def rank_orbital_ids(rank: int, nst: int) -> range:
    """Weak scaling of bench.py (--gpus N): every rank owns its own nst orbitals of the same mesh, ids rank*nst ..
    (rank+1)*nst - 1; no rank ever needs another rank's orbitals (orbitals are independent)."""
    return range(rank * nst, (rank + 1) * nst)


def canonical_rank(ijk: np.ndarray) -> np.ndarray:
    """rank[ip] = position of mesh point ip in the canonical (lexicographic i, j, k) order of the same
    point set.  `ijk` is whatever enumeration a mesh builder publishes; orbitals generated in
    canonical order are brought to that enumeration with  psi_mesh = psi_canon[..., rank]  and back
    with  out_canon[..., rank] = out_mesh.  Pure index bookkeeping on inputs/outputs."""
    ijk = np.asarray(ijk)
    order = np.lexsort((ijk[:, 2], ijk[:, 1], ijk[:, 0]))  # canonical position -> mesh index
    rank = np.empty(order.size, dtype=np.int64)
    rank[order] = np.arange(order.size, dtype=np.int64)
    return rank
