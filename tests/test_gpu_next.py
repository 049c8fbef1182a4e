"""GPU parity of the SURVEY.md section 8(f) rows against oracle/oracle_next.c (through the C ABI):
f1 block dot / expectation / axpy / copy and the fused apply_ex, f2 overlap and subspace matrices, f3 non-local potential.

Tolerances: a sum of np products accumulated in another order differs by at
most ~np^(1/2..1) eps relative to sum |a||b| <= |a|_2 |b|_2; the tests bound it by 1e-12 |a_j|_2 |b_k|_2 (np <= 4 M,
eps = 1.1e-16: 4e6 eps = 4.4e-10 worst case, sqrt-law typical 2e-13)."""
import numpy as np
import pytest

import oracle
import synthetic
import paper_1306_2953_b200 as rs
from harness import EPS, Problem, check

pytestmark = pytest.mark.gpu
_cache = {}


def problem(i):
    if i not in _cache:
        _cache[i] = Problem.from_config(i)
    return _cache[i]


def to_block(p, f_canon, B):
    """per-orbital canonical arrays [nst <= B][np] -> device block [np+1][B] through rs_block_pack."""
    import torch

    st = torch.from_numpy(p.to_mesh(f_canon)).cuda()
    blk = torch.empty((p.np + 1, B), dtype=st.dtype, device="cuda")
    rs.rs_block_pack(p.mesh, st, 0, f_canon.shape[0], B, blk)
    return blk


def from_block(p, blk, nst):
    import torch

    out = torch.empty((nst, p.np), dtype=blk.dtype, device="cuda")
    rs.rs_block_unpack(p.mesh, blk, blk.shape[1], nst, out, 0)
    return p.to_canon(out.cpu().numpy())


def rand_orbitals(seed, nst, npts, is_complex):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((nst, npts))
    return a + 1j * rng.standard_normal((nst, npts)) if is_complex else a


# ---- f1 ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("is_complex", [False, True])
@pytest.mark.parametrize("B,nst", [(1, 1), (2, 2), (4, 3), (16, 16), (32, 19), (64, 64)])
def test_block_dot_and_expectation(B, nst, is_complex):
    import torch

    p = problem(1)
    a = rand_orbitals(B, nst, p.np, is_complex)
    b = rand_orbitals(B + 100, nst, p.np, is_complex)
    A, Bk = to_block(p, a, B), to_block(p, b, B)
    out = torch.full((B,), -3.0, dtype=A.dtype, device="cuda")
    rs.rs_block_dot(p.mesh, A, Bk, B, out)
    g = out.cpu().numpy()
    o = oracle.block_dot(a, b)
    scale = np.linalg.norm(a, axis=1) * np.linalg.norm(b, axis=1)
    assert (np.abs(g[:nst] - o) <= 1e-12 * scale).all()
    assert np.all(g[nst:] == 0)                                   # padding columns are zero columns
    eps = np.linspace(-1.0, 2.0, B)
    sums = torch.full((3, B), -3.0, dtype=torch.float64, device="cuda")
    rs.rs_block_expectation(p.mesh, A, Bk, torch.from_numpy(eps).cuda(), B, sums)
    s = sums.cpu().numpy()
    r = oracle.block_residual(b, a, eps[:nst])
    assert (np.abs(s[0, :nst] - np.real(o)) <= 1e-12 * scale).all()
    assert (np.abs(s[1, :nst] - np.real(oracle.block_dot(a, a))) <= 1e-12 * np.linalg.norm(a, axis=1) ** 2).all()
    assert (np.abs(s[2, :nst] - np.real(oracle.block_dot(r, r))) <= 1e-12 * np.linalg.norm(r, axis=1) ** 2).all()
    rs.rs_block_expectation(p.mesh, A, Bk, None, B, sums)          # eps = NULL: |hpsi|^2
    assert (np.abs(sums.cpu().numpy()[2, :nst] - np.real(oracle.block_dot(b, b))) <= 1e-12 * np.linalg.norm(b, axis=1) ** 2).all()
    out2 = torch.empty_like(out)
    rs.rs_block_dot(p.mesh, A, Bk, B, out2)
    assert torch.equal(out, out2)                                  # deterministic: same bits on a second call


@pytest.mark.parametrize("is_complex", [False, True])
@pytest.mark.parametrize("B,nst", [(1, 1), (8, 5), (16, 16), (64, 33)])
def test_block_axpy_and_copy(B, nst, is_complex):
    import torch

    p = problem(0)
    x = rand_orbitals(B, nst, p.np, is_complex)
    y = rand_orbitals(B + 7, nst, p.np, is_complex)
    alpha = rand_orbitals(B + 9, 1, B, is_complex)[0]
    X, Y = to_block(p, x, B), to_block(p, y, B)
    Ycopy = torch.full_like(Y, 9.0)
    rs.rs_block_copy(p.mesh, Y, Ycopy, B)
    assert torch.equal(Y, Ycopy)
    rs.rs_block_axpy(p.mesh, torch.from_numpy(alpha).cuda(), X, Y, B)
    g = from_block(p, Y, nst)
    o = oracle.block_axpy(alpha[:nst], x, y)
    bound = 4 * EPS * (np.abs(y) + np.abs(alpha[:nst])[:, None] * np.abs(x)) * (2 if is_complex else 1)
    assert (np.abs(g - o) <= bound).all()
    assert torch.all(Y[p.np] == 0)                                  # the zero slot stays zero


@pytest.mark.parametrize("cfg_i,B,is_complex", [(1, 4, False), (1, 16, False), (1, 32, False), (1, 8, True), (2, 16, False)])
def test_apply_ex_sums_match_the_oracle(cfg_i, B, is_complex):
    """H psi and the per-orbital sums of one eigensolver step from ONE call (config 1; config 2 at full size): gather kernel
    (B = 4) or plane-sweep kernel (B >= 16 real columns) followed by the streaming reduction kernel."""
    import torch

    p = problem(cfg_i)
    n = 4
    psi = synthetic.orbitals(77, 0, B, p.np, is_complex=is_complex)
    blk = to_block(p, psi, B)
    hblk = torch.empty_like(blk)
    v = torch.from_numpy(p.v_mesh).cuda()
    o = p.oracle_hpsi(psi, n, nthreads=16)
    e_o = np.real(oracle.block_dot(psi, o))
    n_o = np.real(oracle.block_dot(psi, psi))
    eps = e_o / n_o                                               # Rayleigh quotients
    r = oracle.block_residual(o, psi, eps)
    sums = torch.empty((3, B), dtype=torch.float64, device="cuda")
    rs.rs_hamiltonian_apply_ex(p.mesh, n, oracle.fd_coeffs(n), v, blk, hblk, B, torch.from_numpy(eps).cuda(), sums)
    check(from_block(p, hblk, B), o, p.cond_denominator(psi, n), f"apply_ex B={B}")
    s = sums.cpu().numpy()
    scale = np.linalg.norm(psi, axis=1) * np.linalg.norm(o, axis=1)
    assert (np.abs(s[0] - e_o) <= 1e-12 * scale).all()
    assert (np.abs(s[1] - n_o) <= 1e-12 * n_o).all()
    r2 = np.real(oracle.block_dot(r, r))
    assert (np.abs(s[2] - r2) <= 1e-11 * np.linalg.norm(o, axis=1) ** 2).all()


# ---- f2 ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("is_complex", [False, True])
@pytest.mark.parametrize("B,nst", [(1, 1), (2, 2), (4, 3), (8, 8), (16, 13), (32, 32), (64, 64)])
def test_block_overlap_matches_the_oracle(B, nst, is_complex):
    """S-type (b = a, same buffer) and rectangular-type (b != a) blocks on config 1 (262 k points: ~2000 point tiles with a
    ragged last one, every kernel shape 8..128 real columns); the oracle's triple loop is O(nst^2 np), so the widest
    cases compare a seeded sample of matrix rows."""
    import torch

    p = problem(1)
    a = rand_orbitals(3 * B, nst, p.np, is_complex)
    b = rand_orbitals(3 * B + 1, nst, p.np, is_complex)
    A, Bk = to_block(p, a, B), to_block(p, b, B)
    na, nb = np.linalg.norm(a, axis=1), np.linalg.norm(b, axis=1)
    rows = list(range(nst)) if nst <= 16 else sorted(np.random.default_rng(B).choice(nst, 6, replace=False).tolist())
    for X, Y, x, y, ny in ((A, A, a, a, na), (A, Bk, a, b, nb)):
        M = torch.full((B, B), 7.0, dtype=A.dtype, device="cuda")
        rs.rs_block_overlap(p.mesh, X, Y, B, M)
        g = M.cpu().numpy()
        o = oracle.overlap(x[rows], y)
        assert (np.abs(g[rows][:, :nst] - o) <= 1e-12 * np.outer(na[rows], ny)).all()
        assert np.all(g[nst:] == 0) and np.all(g[:, nst:] == 0)          # padding columns
        if X is Y:
            assert np.abs(g - np.conj(g.T)).max() <= 1e-12 * (na.max() ** 2)
        M2 = torch.empty_like(M)
        rs.rs_block_overlap(p.mesh, X, Y, B, M2)
        assert torch.equal(M, M2)                                       # deterministic


def test_subspace_hamiltonian_of_plane_waves_is_diagonal():
    """eq. 7 end to end on the CUDA path: h = Psi^dagger (H Psi) for plane waves on the periodic box = N^3 diag(lambda(q))."""
    import math
    import torch

    n, h, N, v0 = 4, 0.25, 16, 0.3
    p = Problem(None, None, None, h, max_n=4, box=(N, N, N), periodic=True)
    p.v_canon[:] = v0
    p.v_mesh[:] = v0
    ijk = p.omesh.ijk().astype(np.float64)
    ms = [(1, 2, 3), (2, 0, 5), (0, 0, 0), (3, 3, 1)]
    qs = [[2 * math.pi * ma / (N * h) for ma in m] for m in ms]
    psi = np.stack([np.exp(1j * sum(q[a] * ijk[:, a] * h for a in range(3))) for q in qs])
    B = 4
    blk = to_block(p, psi, B)
    hblk = torch.empty_like(blk)
    c = np.array([-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560])
    rs.rs_hamiltonian_apply(p.mesh, n, c, torch.from_numpy(p.v_mesh).cuda(), blk, hblk, B)
    S = torch.empty((B, B), dtype=torch.complex128, device="cuda")
    Hm = torch.empty_like(S)
    rs.rs_block_overlap(p.mesh, blk, blk, B, S)
    rs.rs_block_overlap(p.mesh, blk, hblk, B, Hm)
    lam = np.array([-0.5 * sum((c[0] + 2 * sum(c[k] * math.cos(k * q[a] * h) for k in range(1, n + 1))) / h ** 2 for a in range(3)) + v0
                    for q in qs])
    assert np.abs(S.cpu().numpy() - N ** 3 * np.eye(B)).max() <= 1e-12 * N ** 3
    assert np.abs(Hm.cpu().numpy() - N ** 3 * np.diag(lam)).max() <= 1e-12 * N ** 3 * np.abs(lam).max()


# ---- f3 ----------------------------------------------------------------------------------------------------------
def make_nonlocal(p, centers, rc, lmax, sigma=0.7, oracle_atoms=None):
    """The same INPUT (synthetic.projector_values) on both sides: the library samples it at the sphere points it
    publishes, the oracle at its own; the two point sets are compared first.  oracle_atoms: the atoms the oracle is
    given (an atom whose sphere holds no mesh point adds nothing to eq. 4, and the oracle's helper wants >= 1 point)."""
    nlm = (lmax + 1) ** 2
    nl = rs.rs_nonlocal_create(p.mesh, centers, rc, nlm)
    h = p.mesh.spacing
    for A in range(len(centers)):
        idx = nl.sphere(A)
        assert np.array_equal(np.sort(p.rank[idx]), oracle.sphere_points(p.omesh, centers[A], rc))
        nl.set_projectors(A, synthetic.projector_values(p.ijk[idx].astype(np.float64) * h - centers[A], lmax, sigma))
    oc = centers if oracle_atoms is None else centers[oracle_atoms]
    proj = oracle.make_projectors(p.omesh, oc, rc, lambda x: synthetic.projector_values(x, lmax, sigma))
    return nl, proj


@pytest.mark.parametrize("B,nst,is_complex,lmax", [(1, 1, False, 0), (4, 3, False, 1), (16, 16, False, 1), (16, 9, True, 1),
                                                   (32, 32, False, 2), (64, 64, False, 1), (64, 40, True, 0)])
def test_nonlocal_apply_matches_the_oracle(B, nst, is_complex, lmax):
    """eq. 4 on config 1: 12 atoms with overlapping projector spheres (several colours), accumulated into an existing H psi."""
    import torch

    p = problem(1)
    centers = p.cfg.centers
    key = ("nl", lmax)
    if key not in _cache:
        _cache[key] = make_nonlocal(p, centers, 2.0, lmax)
    nl, proj = _cache[key]
    assert nl.ncolors >= 2
    psi = rand_orbitals(40 + B, nst, p.np, is_complex)
    base = rand_orbitals(41 + B, nst, p.np, is_complex)
    blk, hblk = to_block(p, psi, B), to_block(p, base, B)
    rs.rs_nonlocal_apply(nl, blk, hblk, B)
    g = from_block(p, hblk, nst)
    o = oracle.nonlocal_apply(p.omesh, proj, psi, base)
    vn = oracle.nonlocal_apply(p.omesh, proj, np.abs(psi.real) + (np.abs(psi.imag) if is_complex else 0.0))   # no cancellation: scale
    assert np.abs(g - o).max() <= 1e-12 * np.abs(o).max()
    assert (np.abs(g - o) <= 1e-12 * (np.abs(vn).max() + np.abs(base))).all()
    hb2 = to_block(p, base, B)
    rs.rs_nonlocal_apply(nl, blk, hb2, B)
    assert torch.equal(hblk, hb2)                                   # deterministic
    assert torch.all(hblk[p.np] == 0)


@pytest.mark.parametrize("lmax", [0, 3])
def test_nonlocal_crowded_and_empty_spheres(lmax):
    """Five atoms within one bohr of each other (up to five spheres over one point: the further-pairs path of the
    gather), an atom whose sphere misses the mesh, one at the mesh edge; large spheres (many chunks per atom, the
    persistent CTAs of part 1 change atom in mid-range); 1 and 16 projectors; one handle reused at several widths."""
    import torch

    p = problem(1)
    c0 = p.cfg.centers[0]
    rng = np.random.default_rng(7)
    centers = np.concatenate([c0 + rng.uniform(-0.5, 0.5, (5, 3)), [c0 + 60.0], [p.cfg.centers[-1] + [p.cfg.radius * 0.9, 0.0, 0.0]]])
    nl, proj = make_nonlocal(p, centers, 3.0, lmax, sigma=1.1, oracle_atoms=[0, 1, 2, 3, 4, 6])
    assert nl.sphere(5).size == 0 and nl.sphere(0).size > 5000
    for B, nst, is_complex in ((1, 1, False), (2, 2, False), (16, 16, False), (8, 8, True), (64, 33, False)):
        psi = rand_orbitals(50 + B, nst, p.np, is_complex)
        base = rand_orbitals(51 + B, nst, p.np, is_complex)
        blk, hblk = to_block(p, psi, B), to_block(p, base, B)
        rs.rs_nonlocal_apply(nl, blk, hblk, B)
        g = from_block(p, hblk, nst)
        o = oracle.nonlocal_apply(p.omesh, proj, psi, base)
        vn = oracle.nonlocal_apply(p.omesh, proj, np.abs(psi.real) + (np.abs(psi.imag) if is_complex else 0.0))
        assert (np.abs(g - o) <= 1e-12 * (np.abs(vn).max() + np.abs(base))).all(), (B, nst)
        hb2 = to_block(p, base, B)
        rs.rs_nonlocal_apply(nl, blk, hb2, B)
        assert torch.equal(hblk, hb2)


def test_full_hamiltonian_with_nonlocal_term_is_hermitian_on_gpu():
    """H = -1/2 Lap + V_loc + V_nl through the CUDA path: <phi|H psi> = <H phi|psi> (all three terms)."""
    import torch

    p = problem(1)
    key = ("nl", 1)
    if key not in _cache:
        _cache[key] = make_nonlocal(p, p.cfg.centers, 2.0, 1)
    nl, _ = _cache[key]
    B = 2
    f = rand_orbitals(5, 2, p.np, True)
    blk = to_block(p, f, B)
    hblk = torch.empty_like(blk)
    rs.rs_hamiltonian_apply(p.mesh, 4, oracle.fd_coeffs(4), torch.from_numpy(p.v_mesh).cuda(), blk, hblk, B)
    rs.rs_nonlocal_apply(nl, blk, hblk, B)
    M = torch.empty((B, B), dtype=torch.complex128, device="cuda")
    rs.rs_block_overlap(p.mesh, blk, hblk, B, M)                     # M[0][1] = <phi|H psi>, M[1][0] = <psi|H phi>
    m = M.cpu().numpy()
    hp = from_block(p, hblk, 2)
    assert abs(m[0, 1] - np.conj(m[1, 0])) <= 1e-13 * np.linalg.norm(f[0]) * np.linalg.norm(hp[1])
