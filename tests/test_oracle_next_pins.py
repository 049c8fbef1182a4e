"""Pins of oracle/oracle_next.c against what the paper and the mathematics fix:
closed forms on plane waves, exact small-integer cases, Hermiticity / positivity invariants, dense brute force on a
6^3 mesh, special cases that reduce to a one-line formula.  No pin re-types the oracle's own loop: the dense checks
go through matrices built from the definition (test_oracle_pins._dense_H for H, an explicit h^3 sum_A,lm g g^T
matrix for V_nl) and numpy's matrix product."""
import math

import numpy as np
import pytest

import oracle
import synthetic
from test_oracle_pins import _dense_H, golden_coeffs


def plane_waves(N, h, ms):
    mesh = oracle.mesh_box(N, N, N, h, periodic=True)
    ijk = mesh.ijk().astype(np.float64)
    qs = [[2 * math.pi * ma / (N * h) for ma in m] for m in ms]
    psi = np.stack([np.exp(1j * sum(q[a] * ijk[:, a] * h for a in range(3))) for q in qs])
    return mesh, qs, psi


def fd_lambda(n, q, h):
    c = golden_coeffs()[n]
    return sum((float(c[0]) + 2 * sum(float(c[k]) * math.cos(k * q[a] * h) for k in range(1, n + 1))) / h ** 2 for a in range(3))


# ---- f1: block dot products, linear combinations, residuals ---------------------------
def test_F1_dot_small_integers_exact():
    """<a|b> with the conjugate on the LEFT: 2 orbitals x 3 points of small Gaussian integers, values by hand."""
    a = np.array([[1 + 2j, 3 - 1j, -2 + 0j], [0 + 1j, 2 + 2j, 1 - 3j]])
    b = np.array([[2 - 1j, 1 + 1j, 4 + 2j], [3 + 0j, -1 + 2j, 2 + 1j]])
    # conj(1+2i)(2-i) = (1-2i)(2-i) = -5i ; conj(3-i)(1+i) = (3+i)(1+i) = 2+4i ; conj(-2)(4+2i) = -8-4i  -> -6 - 5i
    # conj(i)(3) = -3i ; conj(2+2i)(-1+2i) = (2-2i)(-1+2i) = 2+6i ; conj(1-3i)(2+i) = (1+3i)(2+i) = -1+7i -> 1 + 10i
    assert np.array_equal(oracle.block_dot(a, b), np.array([-6 - 5j, 1 + 10j]))
    assert np.array_equal(oracle.block_dot(b, a), np.conj(np.array([-6 - 5j, 1 + 10j])))      # conjugate symmetry
    ar = np.array([[1.0, -2.0, 3.0]])
    assert np.array_equal(oracle.block_dot(ar, ar), np.array([14.0]))


def test_F1_dot_plane_wave_orthogonality():
    """sum_p conj(e^{iq.r}) e^{iq'.r} = N^3 delta_qq' on the periodic box (a dropped conjugate gives 0 on the diagonal)."""
    N, h = 12, 0.25
    mesh, _, psi = plane_waves(N, h, [(1, 2, 3), (2, 0, 5), (1, 2, 3)])
    d = oracle.block_dot(psi, psi)
    assert np.abs(d - N ** 3).max() <= 1e-12 * N ** 3
    x = oracle.block_dot(psi[:2], psi[1:])            # <pw0|pw1> = 0, <pw1|pw2> = 0
    assert np.abs(x).max() <= 1e-12 * N ** 3


@pytest.mark.parametrize("is_complex", [False, True])
def test_F1_expectation_value_is_real_and_matches_dense(is_complex):
    """<psi|H psi> is real for Hermitian H (to 1e-13 of |psi||H psi|) and equals psi^dagger H psi with the dense 6^3
    matrix built from the definition."""
    n, h, N = 4, 0.3, 6
    mesh = oracle.mesh_box(N, N, N, h, periodic=False)
    rng = np.random.default_rng(5)
    v = rng.standard_normal(mesh.npoints)
    psi = rng.standard_normal((3, mesh.npoints)) + (1j * rng.standard_normal((3, mesh.npoints)) if is_complex else 0)
    hp = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), v, psi)
    e = oracle.block_dot(psi, hp)
    scale = np.linalg.norm(psi, axis=1) * np.linalg.norm(hp, axis=1)
    assert np.abs(np.imag(e)).max() <= 1e-13 * scale.max()
    H = _dense_H(mesh.ijk().astype(np.int64), n, h, v, golden_coeffs()[n])
    ref = np.einsum("jp,pq,jq->j", np.conj(psi), H, psi)
    assert np.abs(e - ref).max() <= 1e-13 * scale.max()


def test_F1_axpy_exact_and_residual_of_an_exact_eigenpair():
    x = np.array([[1.0, 2.0, 3.0], [4.0, 5.0, 6.0]])
    y = np.array([[10.0, 20.0, 30.0], [1.0, 1.0, 1.0]])
    assert np.array_equal(oracle.block_axpy(np.array([2.0, -1.0]), x, y), np.array([[12.0, 24.0, 36.0], [-3.0, -4.0, -5.0]]))
    xc = np.array([[1 + 1j, 2 - 1j]])
    yc = np.array([[0 + 0j, 1 + 0j]])
    # (2 - i)(1 + i) = 3 + i ; (2 - i)(2 - i) = 3 - 4i
    assert np.array_equal(oracle.block_axpy(np.array([2 - 1j]), xc, yc), np.array([[3 + 1j, 4 - 4j]]))
    # residual: plane waves are exact eigenvectors of the periodic FD Hamiltonian with constant V
    n, N, h, v0 = 4, 12, 0.25, 0.75
    mesh, qs, psi = plane_waves(N, h, [(1, 2, 3), (0, 4, 1)])
    hp = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), np.full(mesh.npoints, v0), psi)
    eps = np.array([-0.5 * fd_lambda(n, q, h) + v0 for q in qs])
    r = oracle.block_residual(hp, psi, eps)
    assert np.abs(r).max() <= 64 * np.finfo(float).eps * np.abs(hp).max()
    # and a wrong eigenvalue leaves exactly (eps - eps') psi
    r2 = oracle.block_residual(hp, psi, eps + np.array([0.5, -0.25]))
    assert np.abs(r2 - (np.array([-0.5, 0.25])[:, None] * psi)).max() <= 64 * np.finfo(float).eps * np.abs(hp).max()
    # real data, small integers: exact
    assert np.array_equal(oracle.block_residual(np.array([[5.0, 7.0]]), np.array([[1.0, 2.0]]), np.array([3.0])), np.array([[2.0, 1.0]]))


# ---- f2: overlap and subspace matrices (eqs. 5 and 7) ------------------------------------------
def test_F2_overlap_of_plane_waves_is_N3_identity_and_h_is_diagonal():
    n, N, h, v0 = 4, 12, 0.25, -0.4
    ms = [(1, 2, 3), (2, 0, 5), (0, 0, 0), (3, 3, 1)]
    mesh, qs, psi = plane_waves(N, h, ms)
    S = oracle.overlap(psi, psi)
    assert np.abs(S - N ** 3 * np.eye(4)).max() <= 1e-12 * N ** 3
    hp = oracle.hpsi(mesh, n, oracle.fd_coeffs(n), np.full(mesh.npoints, v0), psi)
    hm = oracle.overlap(psi, hp)
    lam = np.array([-0.5 * fd_lambda(n, q, h) + v0 for q in qs])
    assert np.abs(hm - N ** 3 * np.diag(lam)).max() <= 1e-12 * N ** 3 * np.abs(lam).max()


@pytest.mark.parametrize("is_complex", [False, True])
def test_F2_overlap_is_hermitian_and_matches_dense_matrices(is_complex):
    """S = Psi^dagger Psi, h = Psi^dagger H Psi with H the dense 6^3 matrix from the definition; rectangular case too."""
    n, h, N = 4, 0.3, 6
    mesh = oracle.mesh_box(N, N, N, h, periodic=False)
    rng = np.random.default_rng(11)
    v = rng.standard_normal(mesh.npoints)
    A = rng.standard_normal((5, mesh.npoints)) + (1j * rng.standard_normal((5, mesh.npoints)) if is_complex else 0)
    Bm = rng.standard_normal((3, mesh.npoints)) + (1j * rng.standard_normal((3, mesh.npoints)) if is_complex else 0)
    S = oracle.overlap(A, A)
    assert np.abs(S - np.conj(S.T)).max() <= 1e-13 * np.abs(S).max()
    assert np.abs(S - np.conj(A) @ A.T).max() <= 1e-13 * np.abs(S).max()
    R = oracle.overlap(A, Bm)                            # [5][3]: row index = the conjugated (left) orbital
    assert R.shape == (5, 3) and np.abs(R - np.conj(A) @ Bm.T).max() <= 1e-13 * np.abs(R).max()
    H = _dense_H(mesh.ijk().astype(np.int64), n, h, v, golden_coeffs()[n])
    hm = oracle.overlap(A, oracle.hpsi(mesh, n, oracle.fd_coeffs(n), v, A))
    ref = np.conj(A) @ H @ A.T
    assert np.abs(hm - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(hm - np.conj(hm.T)).max() <= 1e-12 * np.abs(hm).max()          # Hermitian subspace Hamiltonian
    assert np.all(np.linalg.eigvalsh(S) > 0)                                    # Gram matrix of independent vectors


def test_F2_small_integers_exact():
    a = np.array([[1.0, 2.0, 3.0], [0.0, 1.0, -1.0]])
    b = np.array([[1.0, 0.0, 2.0], [2.0, 2.0, 2.0], [-1.0, 1.0, 0.0]])
    assert np.array_equal(oracle.overlap(a, b), np.array([[7.0, 12.0, 1.0], [-2.0, 0.0, 1.0]]))


# ---- f3: non-local potential, eq. (4) ---------------------------------------------------------------
def _small_problem(lmax=1, rc=0.95, h=0.3):
    N = 6
    mesh = oracle.mesh_box(N, N, N, h, periodic=False)
    centers = np.array([[0.6, 0.6, 0.75], [1.0, 0.9, 0.6], [0.3, 1.2, 1.2]])       # overlapping spheres on purpose
    proj = oracle.make_projectors(mesh, centers, rc, lambda p: synthetic.projector_values(p, lmax, 0.5))
    return mesh, centers, proj


def _dense_vnl(mesh, proj):
    V = np.zeros((mesh.npoints, mesh.npoints))
    for A in range(proj.off.size):
        sl = slice(int(proj.off[A]), int(proj.off[A] + proj.npts[A]))
        ix = proj.idx[sl]
        for lm in range(proj.nlm):
            g = np.zeros(mesh.npoints)
            g[ix] = proj.gamma[sl, lm]
            V += mesh.spacing ** 3 * np.outer(g, g)
    return V


def test_F3_sphere_membership_counts():
    """closed ball on the lattice: one centre on a lattice point, radius 2h: 1 + 6 + 12 + 8 + 6 = 33 points (|d|^2 <= 4)."""
    mesh = oracle.mesh_box(9, 9, 9, 0.5, periodic=False)
    ix = oracle.sphere_points(mesh, [2.0, 2.0, 2.0], 1.0)
    assert ix.size == 33 and np.all(np.diff(ix) > 0)
    d = mesh.ijk()[ix] - np.array([4, 4, 4])
    assert ((d ** 2).sum(axis=1) <= 4).all()
    assert oracle.sphere_points(mesh, [2.0, 2.0, 2.0], 0.49).size == 1
    assert oracle.sphere_points(mesh, [-3.0, 0.0, 0.0], 1.0).size == 0              # sphere outside the mesh


@pytest.mark.parametrize("is_complex", [False, True])
def test_F3_matches_the_dense_matrix_and_is_symmetric_psd(is_complex):
    mesh, centers, proj = _small_problem()
    assert proj.nlm == 4 and (proj.npts > 10).all()
    rng = np.random.default_rng(3)
    psi = rng.standard_normal((3, mesh.npoints)) + (1j * rng.standard_normal((3, mesh.npoints)) if is_complex else 0)
    phi = rng.standard_normal((3, mesh.npoints)) + (1j * rng.standard_normal((3, mesh.npoints)) if is_complex else 0)
    V = _dense_vnl(mesh, proj)
    out = oracle.nonlocal_apply(mesh, proj, psi)
    ref = psi @ V.T
    assert np.abs(out - ref).max() <= 1e-13 * np.abs(ref).max()
    # accumulation into an existing H psi
    base = rng.standard_normal(psi.shape).astype(psi.dtype)
    assert np.abs(oracle.nonlocal_apply(mesh, proj, psi, base) - (base + ref)).max() <= 1e-13 * np.abs(ref).max()
    # <phi|V psi> = <V phi|psi>, <psi|V psi> >= 0
    vphi = oracle.nonlocal_apply(mesh, proj, phi)
    lhs, rhs = oracle.block_dot(phi, out), oracle.block_dot(vphi, psi)
    assert np.abs(lhs - rhs).max() <= 1e-13 * np.abs(lhs).max()
    e = oracle.block_dot(psi, out)
    assert (np.real(e) > 0).all() and np.abs(np.imag(e)).max() <= 1e-13 * np.abs(e).max()


def test_F3_single_projector_closed_form_and_locality():
    """One atom, one projector (lmax = 0): V g = g * h^3 sum g^2 for psi = g; psi supported outside the sphere gives 0;
    psi orthogonal to g gives 0."""
    h = 0.3
    mesh = oracle.mesh_box(7, 7, 7, h, periodic=False)
    ctr = np.array([[0.9, 0.9, 0.9]])
    proj = oracle.make_projectors(mesh, ctr, 0.7, lambda p: synthetic.projector_values(p, 0, 0.4))
    g = np.zeros(mesh.npoints)
    g[proj.idx] = proj.gamma[:, 0]
    norm2 = h ** 3 * float(np.sum(proj.gamma[:, 0] ** 2))
    out = oracle.nonlocal_apply(mesh, proj, g)
    assert np.abs(out - norm2 * g).max() <= 1e-14 * np.abs(out).max()
    outside = np.ones(mesh.npoints)
    outside[proj.idx] = 0.0
    assert np.array_equal(oracle.nonlocal_apply(mesh, proj, outside), np.zeros((1, mesh.npoints)))
    rng = np.random.default_rng(0)
    w = rng.standard_normal(mesh.npoints)
    w -= g * (g @ w) / (g @ g)
    assert np.abs(oracle.nonlocal_apply(mesh, proj, w)).max() <= 1e-13 * np.abs(w).max() * norm2 * 10


def test_F3_synthetic_projector_shapes():
    """The INPUT generator: (lmax+1)^2 columns, s / p / d parity under inversion, Gaussian envelope."""
    p = np.array([[0.1, -0.2, 0.3], [0.0, 0.0, 0.0]])
    for lmax, nlm in ((0, 1), (1, 4), (2, 9)):
        g = synthetic.projector_values(p, lmax, 0.7)
        gm = synthetic.projector_values(-p, lmax, 0.7)
        assert g.shape == (2, nlm)
        assert np.allclose(g[:, 0], gm[:, 0])
        if lmax >= 1:
            assert np.allclose(g[:, 1:4], -gm[:, 1:4])
        if lmax >= 2:
            assert np.allclose(g[:, 4:9], gm[:, 4:9])
    assert synthetic.projector_values(p, 0, 0.7)[1, 0] == 1.0
    assert math.isclose(synthetic.projector_values(p, 0, 0.7)[0, 0], math.exp(-0.14 / (2 * 0.49)), rel_tol=1e-15)
