"""rs_block_expectation_static: the allocation-free variant of rs_block_expectation (partial sums in a file-scope
device array of the library) against the existing path and the oracle, on two calls in a row.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests:
it builds its own mesh, so no scratch of another test is involved, and the array it shares keeps whatever the last
call left there."""
import numpy as np
import pytest

import oracle
import paper_1306_2953_b200 as rs
from harness import Problem

pytestmark = pytest.mark.gpu


def rand_orbitals(seed, nst, npts, is_complex):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((nst, npts))
    return a + 1j * rng.standard_normal((nst, npts)) if is_complex else a


def to_block(p, f_canon, B):
    import torch

    st = torch.from_numpy(p.to_mesh(f_canon)).cuda()
    blk = torch.empty((p.np + 1, B), dtype=st.dtype, device="cuda")
    rs.rs_block_pack(p.mesh, st, 0, f_canon.shape[0], B, blk)
    return blk


def test_static_scratch_expectation_matches_the_allocating_path_twice_in_a_row():
    import torch

    p = Problem.from_config(1)                       # a mesh of its own: rs_block_expectation never ran on it
    cases = []
    # call 1 fills the widest slots the array has (64 real columns), call 2 is a narrow complex block with other data:
    # whatever call 1 left in the array must not reach call 2's sums
    for seed, B, nst, is_complex in ((1, 64, 64, False), (2, 4, 3, True)):
        a, b = rand_orbitals(seed, nst, p.np, is_complex), rand_orbitals(seed + 50, nst, p.np, is_complex)
        eps = np.linspace(-0.5, 1.5, B)
        cases.append(dict(B=B, nst=nst, a=a, b=b, eps=eps, A=to_block(p, a, B), Bk=to_block(p, b, B),
                          eps_d=torch.from_numpy(eps).cuda(),
                          out=torch.full((3, B), -7.0, dtype=torch.float64, device="cuda"),
                          ref=torch.full((3, B), -9.0, dtype=torch.float64, device="cuda")))
    # the first call per device resolves the array's address and loads the kernels: warm up, then watch free memory
    c0 = cases[0]
    rs.rs_block_expectation_static(p.mesh, c0["A"], c0["Bk"], c0["eps_d"], c0["B"], c0["out"])
    c0["out"].fill_(-7.0)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for c in cases:                                  # two calls in a row, same stream
        rs.rs_block_expectation_static(p.mesh, c["A"], c["Bk"], c["eps_d"], c["B"], c["out"])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "rs_block_expectation_static allocated device memory"

    for c in cases:
        rs.rs_block_expectation(p.mesh, c["A"], c["Bk"], c["eps_d"], c["B"], c["ref"])      # the existing path (allocates its scratch)
    torch.cuda.synchronize()
    for c in cases:
        g, r, nst = c["out"].cpu().numpy(), c["ref"].cpu().numpy(), c["nst"]
        a, b = c["a"], c["b"]
        na, nb = np.linalg.norm(a, axis=1), np.linalg.norm(b, axis=1)
        res = oracle.block_residual(b, a, c["eps"][:nst])
        scale = np.stack([na * nb, na ** 2, np.linalg.norm(res, axis=1) ** 2])
        # the tolerance of the f1 tests (tests/test_gpu_next.py): 1e-12 |a_j| |b_j| ...
        assert (np.abs(g[:, :nst] - r[:, :nst]) <= 1e-12 * scale).all()
        # ... and in fact the same bits: same kernels, same grid, same order of the sums
        assert np.array_equal(g, r)
        assert np.all(g[:, nst:] == 0)               # padding columns are zero columns
        o = np.stack([np.real(oracle.block_dot(a, b)), np.real(oracle.block_dot(a, a)), np.real(oracle.block_dot(res, res))])
        assert (np.abs(g[:, :nst] - o) <= 1e-12 * scale).all()

    # a second round over the same inputs, now after the allocating path ran: still the same bits
    for c in cases:
        again = torch.empty_like(c["out"])
        rs.rs_block_expectation_static(p.mesh, c["A"], c["Bk"], c["eps_d"], c["B"], again)
        assert torch.equal(again, c["out"])
    # eps = NULL
    c = cases[1]
    rs.rs_block_expectation_static(p.mesh, c["A"], c["Bk"], None, c["B"], c["out"])
    rs.rs_block_expectation(p.mesh, c["A"], c["Bk"], None, c["B"], c["ref"])
    assert torch.equal(c["out"], c["ref"])


def test_static_scratch_rejects_blocks_beyond_its_size():
    import torch

    p = Problem.from_config(0)
    B = 64                                           # complex: 128 real columns > the 64 the static array holds
    blk = torch.zeros((p.np + 1, B), dtype=torch.complex128, device="cuda")
    out = torch.zeros((3, B), dtype=torch.float64, device="cuda")
    with pytest.raises(rs.RsError) as e:
        rs.rs_block_expectation_static(p.mesh, blk, blk.clone(), None, B, out)
    assert e.value.status == rs.RS_ERR_INVALID_ARG and "64" in str(e.value) and "static scratch" in str(e.value)
    half = torch.zeros((p.np + 1, 32), dtype=torch.complex128, device="cuda")              # 64 real columns: the limit itself
    rs.rs_block_expectation_static(p.mesh, half, half.clone(), None, 32, out[:, :32].contiguous())
    raw = torch.zeros((p.np + 1) * 4 + 2, dtype=torch.float64, device="cuda")
    with pytest.raises(rs.RsError) as e:                                                     # misaligned block
        rs.rs_block_expectation_static(p.mesh, raw[1:1 + (p.np + 1) * 4], raw[1:1 + (p.np + 1) * 4].clone(), None, 4, out)
    assert e.value.status == rs.RS_ERR_INVALID_ARG
    torch.cuda.synchronize()
