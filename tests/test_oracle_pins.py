"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each expected value is a
closed form, an exact rational identity, a brute-force construction from the definition, or a
number the paper prints.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
import synthetic

GOLD = os.path.join(os.path.dirname(__file__), "golden")
EPS = np.finfo(np.float64).eps


def golden_coeffs():
    rows = {}
    for line in open(os.path.join(GOLD, "fd_coeffs.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, rest = line.split(":")
        rows[int(n)] = [Fraction(t) for t in rest.split()]
    return rows


# ---- P1: coefficient table -------------------------------------------------------------------
@pytest.mark.parametrize("n", [4, 6])
def test_P1_coeffs_match_textbook_rationals(n):
    gold = golden_coeffs()[n]
    c = oracle.fd_coeffs(n)
    for k in range(n + 1):
        assert abs(c[k] - float(gold[k])) <= 4 * EPS * abs(float(gold[k])), (n, k)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 8])
def test_P1_moment_identities_exact(n):
    """sum_k c_k = 0, sum_k c_k k^2 = 2, sum_k c_k k^(2j) = 0 (j=2..n) in exact rationals, with the
    closed form S1 written independently here in Fractions; the oracle's doubles must round to it."""
    cf = [Fraction(0)] * (n + 1)
    for m in range(1, n + 1):
        cf[m] = Fraction(2 * (-1) ** (m + 1) * math.factorial(n) ** 2,
                         m * m * math.factorial(n - m) * math.factorial(n + m))
    cf[0] = -2 * sum(cf[1:])
    full = {k: cf[abs(k)] for k in range(-n, n + 1)}
    assert sum(full.values()) == 0
    assert sum(v * k ** 2 for k, v in full.items()) == 2
    for j in range(2, n + 1):
        assert sum(v * k ** (2 * j) for k, v in full.items()) == 0
    c = oracle.fd_coeffs(n)
    for k in range(n + 1):
        assert abs(c[k] - float(cf[k])) <= 8 * EPS * abs(float(cf[k]))


def _apply(mesh, n, psi, v=None):
    c = oracle.fd_coeffs(n)
    v = np.zeros(mesh.npoints) if v is None else v
    return oracle.hpsi(mesh, n, c, v, psi)


# ---- P2: constants are annihilated (periodic box) ---------------------------------------------
@pytest.mark.parametrize("n", [4, 6])
def test_P2_constants(n):
    h = 0.25
    mesh = oracle.mesh_box(24, 24, 24, h, periodic=True)
    out = _apply(mesh, n, np.ones(mesh.npoints))
    c = oracle.fd_coeffs(n)
    sum_abs_w = 0.5 / h ** 2 * (3 * abs(c[0]) + 6 * np.abs(c[1:]).sum())
    assert np.abs(out).max() <= 64 * EPS * sum_abs_w


# ---- P3: polynomials up to total degree 2n+1 are differentiated exactly (interior points) ------
@pytest.mark.parametrize("n", [4, 6])
def test_P3_polynomials(n):
    h = 0.25
    N = 24
    mesh = oracle.mesh_box(N, N, N, h, periodic=False)
    ijk = mesh.ijk().astype(np.float64)
    x, y, z = [(ijk[:, a] - N / 2) * h for a in range(3)]
    interior = np.all((mesh.ijk() >= n) & (mesh.ijk() < N - n), axis=1)
    rng = np.random.default_rng(5)
    deg = 2 * n + 1
    monos = [(a, b, c) for a in range(deg + 1) for b in range(deg + 1 - a) for c in range(deg + 1 - a - b)]
    picks = [monos[i] for i in rng.choice(len(monos), 12, replace=False)] + [(deg, 0, 0), (0, deg - 1, 1), (3, 3, deg - 6)]
    for (a, b, c) in picks:
        p = x ** a * y ** b * z ** c
        lap = np.zeros_like(p)
        if a >= 2:
            lap += a * (a - 1) * x ** (a - 2) * y ** b * z ** c
        if b >= 2:
            lap += b * (b - 1) * x ** a * y ** (b - 2) * z ** c
        if c >= 2:
            lap += c * (c - 1) * x ** a * y ** b * z ** (c - 2)
        out = _apply(mesh, n, p)          # = -1/2 Lap p   (V = 0)
        err = np.abs(-2.0 * out - lap)[interior].max()
        # rounding: each of the 6n+1 products carries ~eps * |w_k| * max|p| of error
        tol = 64 * EPS * (6 * n + 1) * np.abs(p).max() / h ** 2 * 4 + 1e-13 * max(1.0, np.abs(lap).max())
        assert err <= tol, ((a, b, c), err, tol)


# ---- P4: first degree that is NOT exact: leading truncation term, closed form -----------------
@pytest.mark.parametrize("n,deg,coef,offset", [(4, 10, 90, -1152.0), (6, 14, 182, -1036800.0)])
def test_P4_leading_truncation_term(n, deg, coef, offset):
    """1-D: FD[x^(2n+2)] = (2n+2)(2n+1) x^(2n) + offset * h^(2n), offset = 2*sum_k c_k k^(2n+2) is a
    constant (n=4: -1152; n=6: -1 036 800), independent of x."""
    gold = golden_coeffs()[n]
    assert 2 * sum(gold[k] * k ** (2 * n + 2) for k in range(1, n + 1)) == Fraction(int(offset))
    h = 0.25
    N = 32
    mesh = oracle.mesh_box(N, 1 + 2 * n, 1 + 2 * n, h, periodic=False)
    ijk = mesh.ijk()
    x = (ijk[:, 0].astype(np.float64) - N / 2) * h
    p = x ** deg
    out = -2.0 * _apply(mesh, n, p)
    interior = (ijk[:, 0] >= n) & (ijk[:, 0] < N - n) & (ijk[:, 1] == n) & (ijk[:, 2] == n)
    expect = coef * x ** (deg - 2) + offset * h ** (2 * n)
    scale = np.abs(p).max() / h ** 2
    assert np.abs(out - expect)[interior].max() <= 512 * EPS * scale


# ---- P5: plane wave on a periodic box vs the closed-form FD symbol ----------------------------
def golden_symbol():
    vals = {}
    for line in open(os.path.join(GOLD, "fd_symbol.txt")):
        if line.startswith("#"):
            continue
        n, name, v = line.split()
        vals[(int(n), name)] = float(v)
    return vals


@pytest.mark.parametrize("n", [4, 6])
def test_P5_symbol_spot_values(n):
    """The golden symbol values must be reproduced by the oracle applied to cos(theta * i) in 1-D."""
    gold = golden_symbol()
    for name, theta, N in (("pi/8", math.pi / 8, 16), ("pi/2", math.pi / 2, 16), ("pi", math.pi, 16)):
        h = 1.0
        mesh = oracle.mesh_box(N, 1, 1, h, periodic=True)
        i = mesh.ijk()[:, 0].astype(np.float64)
        psi = np.cos(theta * i) + 1j * np.sin(theta * i)
        out = _apply(mesh, n, psi)
        # y and z arms see the same value (1-point periodic axes): they add 2*(c_0 + 2 sum c_k) = 0.
        lam = -2.0 * out / psi
        assert np.abs(lam - gold[(n, name)]).max() <= 1e-13 * 8


@pytest.mark.parametrize("n", [4, 6])
def test_P5_plane_wave_3d(n):
    h, N, m = 0.25, 24, (2, 3, 5)
    mesh = oracle.mesh_box(N, N, N, h, periodic=True)
    ijk = mesh.ijk().astype(np.float64)
    q = [2 * math.pi * ma / (N * h) for ma in m]
    phase = sum(q[a] * ijk[:, a] * h for a in range(3))
    psi = np.exp(1j * phase)
    gold = golden_coeffs()[n]
    lam = [(float(gold[0]) + 2 * sum(float(gold[k]) * math.cos(k * q[a] * h) for k in range(1, n + 1))) / h ** 2
           for a in range(3)]
    expect = -0.5 * sum(lam) * psi
    out = _apply(mesh, n, psi)
    assert np.abs(out - expect).max() / np.abs(expect).max() <= 1e-13
    # and with a constant potential added
    out2 = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), np.full(mesh.npoints, 0.75), psi)
    assert np.abs(out2 - (expect + 0.75 * psi)).max() / np.abs(expect).max() <= 1e-13


# ---- P6: Hermiticity on the molecule-shaped meshes --------------------------------------------
@pytest.mark.parametrize("cfg_i,is_complex", [(0, False), (0, True), (1, False), (1, True)])
def test_P6_hermiticity(cfg_i, is_complex):
    cfg = synthetic.config(cfg_i)
    mesh = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    v = synthetic.vloc_at(mesh.xyz(), cfg.centers, cfg.charges)
    phi = synthetic.orbital(100 + cfg_i, 0, mesh.npoints, is_complex)
    psi = synthetic.orbital(100 + cfg_i, 1, mesh.npoints, is_complex)
    n = 4
    c = oracle.fd_coeffs(n)
    hphi, hpsi = oracle.hpsi(mesh, n, c, v, np.stack([phi, psi]))
    lhs = np.vdot(phi, hpsi)
    rhs = np.vdot(hphi, psi)
    assert abs(lhs - rhs) / (np.linalg.norm(phi) * np.linalg.norm(hpsi)) <= 1e-13


# ---- P7: dense brute-force matrix on a 6^3 cube (and on a sphere-shaped subset) ---------------
def _dense_H(points, n, h, v, coeffs_frac):
    """H_ij from the definition: w_|d| if i, j differ along exactly one axis by |d| <= n; diagonal
    3 w_0 + V_i; w_k = -1/2 c_k / h^2.  `points` [np][3] ints."""
    w = [-0.5 * float(ck) / h ** 2 for ck in coeffs_frac]
    npts = len(points)
    H = np.zeros((npts, npts))
    for i in range(npts):
        for j in range(npts):
            d = points[j] - points[i]
            nzs = np.flatnonzero(d)
            if nzs.size == 0:
                H[i, j] = 3 * w[0] + v[i]
            elif nzs.size == 1 and abs(d[nzs[0]]) <= n:
                H[i, j] = w[abs(d[nzs[0]])]
    return H


@pytest.mark.parametrize("shape", ["cube", "sphere"])
def test_P7_dense_bruteforce(shape):
    n, h = 4, 0.3
    N = 6
    g = np.arange(N)
    I, J, K = np.meshgrid(g, g, g, indexing="ij")
    if shape == "cube":
        mask = np.ones((N, N, N), dtype=np.uint8)
    else:
        mask = (((I - 2.5) ** 2 + (J - 2.5) ** 2 + (K - 2.5) ** 2) <= 2.6 ** 2).astype(np.uint8)
    mesh = oracle.mesh_from_mask(mask, h)
    pts = mesh.ijk().astype(np.int64)
    rng = np.random.default_rng(7)
    v = rng.standard_normal(mesh.npoints)
    H = _dense_H(pts, n, h, v, golden_coeffs()[n])
    assert np.array_equal(H, H.T)
    for is_complex in (False, True):
        psi = rng.standard_normal(mesh.npoints) + (1j * rng.standard_normal(mesh.npoints) if is_complex else 0)
        ref = H @ psi
        out = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), v, psi)
        assert np.abs(out - ref).max() / np.abs(ref).max() <= 1e-14


# ---- P8: delta response = the star itself ------------------------------------------------------
def test_P8_delta_response():
    n, h, N = 4, 0.2, 13
    mesh = oracle.mesh_box(N, N, N, h, periodic=False)
    rng = np.random.default_rng(8)
    v = rng.standard_normal(mesh.npoints)
    ctr = np.array([6, 6, 6])
    ijk = mesh.ijk()
    ic = int(np.flatnonzero((ijk == ctr).all(axis=1))[0])
    psi = np.zeros(mesh.npoints)
    psi[ic] = 1.0
    out = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), v, psi)
    gold = [float(f) for f in golden_coeffs()[n]]
    expect = np.zeros(mesh.npoints)
    for p in range(mesh.npoints):
        d = ijk[p] - ctr
        nzs = np.flatnonzero(d)
        if nzs.size == 0:
            expect[p] = -0.5 * 3 * gold[0] / h ** 2 + v[p]
        elif nzs.size == 1 and abs(d[nzs[0]]) <= n:
            expect[p] = -0.5 * gold[abs(d[nzs[0]])] / h ** 2
    assert np.abs(out - expect).max() <= 16 * EPS * np.abs(expect).max()
    assert np.count_nonzero(out) == 6 * n + 1


# ---- P9: mesh builder vs the paper's Table I and the continuum volume -------------------------
def test_P9_benzene_grid_size_table1():
    """Benzene-shaped centres at R=5.5, h=0.41 -> Table I prints 37.3k points."""
    table = {}
    for line in open(os.path.join(GOLD, "table1_grid_sizes.txt")):
        if not line.startswith("#"):
            k, v = line.split()
            table[k] = float(v)
    c, _ = synthetic.benzene_centers()
    mesh = oracle.mesh_from_spheres(c, 5.5, 0.41)
    assert abs(mesh.npoints / 1000.0 - table["benzene"]) <= 0.15   # within the table's rounding + geometry
    assert mesh.npoints == 37295                                    # SURVEY.md section 4 scratch count


def test_P9_single_sphere_count_and_symmetry():
    cfg = synthetic.config(0)
    mesh = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    cont = 4.0 / 3.0 * math.pi * cfg.radius ** 3 / cfg.spacing ** 3
    assert abs(mesh.npoints - cont) / cont < 0.02
    assert mesh.npoints == 9843                                     # brute force below must agree too
    # brute force, independent formula: integer test i^2+j^2+k^2 <= (R/h)^2
    m = int(cfg.radius / cfg.spacing) + 2
    g = np.arange(-m, m + 1)
    I, J, K = np.meshgrid(g, g, g, indexing="ij")
    assert int(((I * I + J * J + K * K) <= (cfg.radius / cfg.spacing) ** 2).sum()) == mesh.npoints
    # the point set is symmetric under i -> -i etc. and contains the origin
    pts = set(map(tuple, mesh.ijk().tolist()))
    assert (0, 0, 0) in pts
    assert all((-i, j, k) in pts and (i, -j, k) in pts and (i, j, -k) in pts and (j, i, k) in pts for (i, j, k) in pts)


def test_P9_union_is_union_of_single_spheres():
    cfg = synthetic.config(1)
    whole = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    pts = set()
    for a in range(cfg.centers.shape[0]):
        one = oracle.mesh_from_spheres(cfg.centers[a:a + 1], cfg.radius, cfg.spacing)
        pts |= set(map(tuple, one.ijk().tolist()))
    assert pts == set(map(tuple, whole.ijk().tolist()))
    assert whole.npoints == cfg.np_expected


# ---- P10: Fig. 4 layout example ----------------------------------------------------------------
def test_P10_fig4_layout():
    """4 orbitals x 5 coefficients: element (orbital j, coefficient p) sits at j*5+p in the standard
    layout and at p*4+j in the blocked layout."""
    dims = dict(line.split() for line in open(os.path.join(GOLD, "fig4_layout.txt")) if not line.startswith("#"))
    norb, ncoef = int(dims["norbitals"]), int(dims["ncoeff"])
    assert (norb, ncoef) == (4, 5)                                # the figure's own sizes
    states = np.arange(norb * ncoef, dtype=np.float64).reshape(norb, ncoef)   # value = standard-layout address
    blk = oracle.block_pack(states, 0, norb, norb, ncoef, ncoef)
    flat = blk.ravel()
    for j in range(norb):
        for p in range(ncoef):
            assert flat[p * norb + j] == j * ncoef + p
    # the arrows of Fig. 4: first coefficient of orbital j moves from address 5j to address j
    assert [int(flat[j]) for j in range(4)] == [0, 5, 10, 15]


@pytest.mark.parametrize("B", [1, 2, 4, 8, 16, 32, 64])
def test_P10_pack_unpack_roundtrip(B):
    rng = np.random.default_rng(10)
    nst, npts, ld = 11, 37, 41
    for dtype in (np.float64, np.complex128):
        states = rng.standard_normal((nst, ld)).astype(dtype)
        if dtype is np.complex128:
            states = states + 1j * rng.standard_normal((nst, ld))
        back = np.full_like(states, -7.0)
        for ist0 in range(0, nst, B):
            nb = min(B, nst - ist0)
            blk = oracle.block_pack(states, ist0, nb, B, npts, npts + 1)
            assert np.all(blk[npts] == 0) and np.all(blk[:, nb:] == 0)
            assert np.array_equal(blk[:npts, :nb], states[ist0:ist0 + nb, :npts].T)
            oracle.block_unpack(blk, nb, npts, back, ist0)
        assert np.array_equal(back[:, :npts], states[:, :npts])
        assert np.all(back[:, npts:] == -7.0)


# ---- P12: the synthetic potential ---------------------------------------------------------------
def test_P12_vloc_closed_forms():
    z4 = -4.0 * 2.0 / (0.5 * math.sqrt(math.pi))
    assert abs(z4 - (-9.0270333367641)) < 1e-12
    c = np.zeros((1, 3))
    q = np.array([4.0])
    for fn in (lambda xyz: synthetic.vloc_at(xyz, c, q), lambda xyz: oracle.vloc(c, q, xyz)):
        v = fn(np.array([[0.0, 0.0, 0.0], [30.0, 0.0, 0.0], [0.0, 0.5, 0.0]]))
        assert abs(v[0] - z4) < 1e-13
        assert abs(v[1] - (-4.0 / 30.0)) < 1e-15                # far field -> -Z/r
        assert abs(v[2] - (-4.0 * math.erf(1.0) / 0.5)) < 1e-14
    cfg = synthetic.config(1)
    xyz = np.random.default_rng(12).uniform(-6, 6, (500, 3))
    a = synthetic.vloc_at(xyz, cfg.centers, cfg.charges)
    b = oracle.vloc(cfg.centers, cfg.charges, xyz)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()
    far = np.array([[400.0, 300.0, 0.0]])
    assert abs(synthetic.vloc_at(far, cfg.centers, cfg.charges)[0] + cfg.charges.sum() / 500.0) < 1e-4


# ---- P11 (oracle side): the count of outside arms has a closed form on a full box -------------
def test_P11_outside_arm_count_closed_form():
    n = 4
    nx, ny, nz = 7, 9, 11
    mesh = oracle.mesh_box(nx, ny, nz, 0.3, periodic=False)
    # along an axis of length L every point loses sum_{m=1..n} [i-m<0] + [i+m>=L] arms
    def lost(L):
        return sum((1 if i - m < 0 else 0) + (1 if i + m >= L else 0) for i in range(L) for m in range(1, n + 1))
    expect = lost(nx) * ny * nz + lost(ny) * nx * nz + lost(nz) * nx * ny
    assert oracle.count_outside_arms(mesh, n) == expect


def test_cluster_generator_recipe():
    c, z = synthetic.cluster_centers(100, 20.0, 2.5, 2)
    assert c.shape == (100, 3) and (c >= 0).all() and (c <= 20).all()
    d = np.linalg.norm(c[:, None, :] - c[None, :, :], axis=2) + np.eye(100) * 99
    assert d.min() >= 2.5
    assert set(np.unique(z)) <= {1.0, 4.0, 5.0, 6.0}
    c2, z2 = synthetic.cluster_centers(100, 20.0, 2.5, 2)
    assert np.array_equal(c, c2) and np.array_equal(z, z2)
