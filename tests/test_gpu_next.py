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


@pytest.mark.parametrize("B,is_complex", [(4, False), (16, False), (32, False), (8, True)])
def test_apply_ex_sums_match_the_oracle(B, is_complex):
    """H psi and the per-orbital sums of one eigensolver step from ONE call, config 1 (gather and plane-sweep kernels)."""
    import torch

    p = problem(1)
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
