"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the same seeded
inputs, element by element (configs 0-1 and small boxes: several tiles, ragged tails, every block
size, both enumerations, every kernel, real and complex, orders 1..8)."""
import numpy as np
import pytest

import oracle
import synthetic
import paper_1306_2953_b200 as rs
from harness import EPS, Problem, check

pytestmark = pytest.mark.gpu

KERNELS = {"auto": rs.RS_KERNEL_AUTO, "gather": rs.RS_KERNEL_GATHER, "sweep": rs.RS_KERNEL_SWEEP}
_cache = {}


def problem(i, ordering=rs.RS_ORDER_LEX):
    key = (i, ordering)
    if key not in _cache:
        _cache[key] = Problem.from_config(i, ordering=ordering)
    return _cache[key]


def _run(p, psi, n, B, kernel):
    try:
        return p.gpu_hpsi(psi, n, B, kernel=KERNELS[kernel])
    except rs.RsError as e:
        if e.status == rs.RS_ERR_UNSUPPORTED and kernel != "auto":
            pytest.skip(f"{kernel} kernel does not serve this call: {e}")
        raise


# ---- config 0: tiny atom, nst=4, B=4 (BASELINE.json configs[0]) ---------------------------------
@pytest.mark.parametrize("kernel", ["auto", "gather", "sweep"])
@pytest.mark.parametrize("ordering", [rs.RS_ORDER_BRICK, rs.RS_ORDER_LEX, rs.RS_ORDER_TILE])
def test_config0(kernel, ordering):
    p = problem(0, ordering)
    cfg = p.cfg
    psi = synthetic.orbitals(cfg.seed, 0, cfg.nst, p.np)
    g = _run(p, psi, 4, 4, kernel)
    o = p.oracle_hpsi(psi, 4)
    check(g, o, p.cond_denominator(psi, 4), "config0")


# ---- config 1: benzene-shaped, nst=16, every block size 1..64 (padded) --------------------------
@pytest.mark.parametrize("kernel", ["auto", "gather", "sweep"])
@pytest.mark.parametrize("B", [1, 2, 4, 8, 16, 32, 64])
def test_config1_real(B, kernel):
    p = problem(1)
    cfg = p.cfg
    psi = synthetic.orbitals(cfg.seed, 0, cfg.nst, p.np)
    g = _run(p, psi, 4, B, kernel)
    o = p.oracle_hpsi(psi, 4)
    check(g, o, p.cond_denominator(psi, 4), f"config1 B={B}")


@pytest.mark.parametrize("kernel", ["auto", "gather", "sweep"])
@pytest.mark.parametrize("B", [1, 2, 8, 32, 64])
def test_config1_complex(B, kernel):
    p = problem(1)
    psi = synthetic.orbitals(31, 0, 6, p.np, is_complex=True)      # 6 orbitals: ragged last block for B=4..
    g = _run(p, psi, 4, B, kernel)
    o = p.oracle_hpsi(psi, 4)
    check(g, o, p.cond_denominator(psi, 4), f"config1 complex B={B}")


@pytest.mark.parametrize("kernel", ["auto", "gather"])
@pytest.mark.parametrize("n", [1, 2, 3, 5, 6, 7, 8])
def test_other_orders(n, kernel):
    cfg = synthetic.config(0)
    key = ("orders", 8)
    if key not in _cache:
        _cache[key] = Problem(cfg.centers, cfg.charges, cfg.radius, cfg.spacing, max_n=8)
    p = _cache[key]
    psi = synthetic.orbitals(5, 0, 5, p.np)
    g = _run(p, psi, n, 4, kernel)                                  # 5 orbitals in blocks of 4: 4 + 1 (padded)
    o = p.oracle_hpsi(psi, n)
    check(g, o, p.cond_denominator(psi, n), f"order {n}")


@pytest.mark.parametrize("knob", [("force_tensor", 1), ("planes", 8), ("planes", 100), ("ctas", 7), ("ctas", 1000)])
def test_sweep_kernel_variants(knob):
    """The plane-sweep kernel under its per-mesh options: 2-D tensor-map copies for 16 columns, thin and thick slabs,
    few CTAs (long chains of work pieces through one CTA) and more CTAs than work."""
    cfg = synthetic.config(1)
    p = Problem(cfg.centers, cfg.charges, cfg.radius, cfg.spacing, max_n=4)      # fresh mesh: its own options
    rs.rs_mesh_set_sweep_options(p.mesh, **{knob[0]: knob[1]})
    psi = synthetic.orbitals(cfg.seed, 0, cfg.nst, p.np)
    g = p.gpu_hpsi(psi, 4, 16, kernel=rs.RS_KERNEL_SWEEP)
    assert rs.rs_kernel_name(p.mesh, 4, 16, kernel=rs.RS_KERNEL_SWEEP).startswith("sweep[")
    assert rs.rs_kernel_name(problem(1).mesh, 4, 16, kernel=rs.RS_KERNEL_SWEEP).count("tma2d") == 0   # other meshes keep the defaults
    o = problem(1).oracle_hpsi(psi, 4)
    check(g, o, problem(1).cond_denominator(psi, 4), f"sweep variant {knob}")


@pytest.mark.parametrize("B,is_complex", [(16, False), (64, False), (8, True)])
def test_sweep_kernel_order6(B, is_complex):
    """fd_order 6 through the plane-sweep kernel's 8 x 16 / 2 x 4 shape (config 1 mesh; ragged last block)."""
    key = ("c1n6",)
    if key not in _cache:
        cfg = synthetic.config(1)
        _cache[key] = Problem(cfg.centers, cfg.charges, cfg.radius, cfg.spacing, max_n=6)
    p = _cache[key]
    psi = synthetic.orbitals(61, 0, B + 3, p.np, is_complex=is_complex)
    g = _run(p, psi, 6, B, "sweep")
    assert rs.rs_kernel_name(p.mesh, 6, B, rs.RS_COMPLEX128 if is_complex else rs.RS_REAL64, rs.RS_KERNEL_SWEEP).startswith("sweep[n6")
    o = p.oracle_hpsi(psi, 6)
    check(g, o, p.cond_denominator(psi, 6), f"sweep n=6 B={B}")


def test_autotune_keeps_parity():
    """rs_hamiltonian_autotune re-deals the plane-sweep work from measured step costs: same results, kernel still the sweep."""
    import torch

    cfg = synthetic.config(1)
    p = Problem(cfg.centers, cfg.charges, cfg.radius, cfg.spacing, max_n=4)      # fresh mesh: its tables get replaced
    B = 16
    psi = synthetic.orbitals(cfg.seed, 0, B, p.np)
    dev = torch.device("cuda:0")
    states = torch.from_numpy(p.to_mesh(psi)).to(dev)
    v = torch.from_numpy(p.v_mesh).to(dev)
    blk = torch.empty((p.np + 1, B), dtype=torch.float64, device=dev)
    hblk = torch.full((p.np + 1, B), 3.0, dtype=torch.float64, device=dev)
    rs.rs_block_pack(p.mesh, states, 0, B, B, blk)
    rs.rs_hamiltonian_autotune(p.mesh, 4, oracle.fd_coeffs(4), v, blk, hblk, B)
    out = torch.empty_like(states)
    rs.rs_block_unpack(p.mesh, hblk, B, B, out, 0)
    o = problem(1).oracle_hpsi(psi, 4)
    check(p.to_canon(out.cpu().numpy()), o, problem(1).cond_denominator(psi, 4), "autotune call itself")
    g = p.gpu_hpsi(psi, 4, B, kernel=rs.RS_KERNEL_SWEEP)                          # re-dealt tables
    check(g, o, problem(1).cond_denominator(psi, 4), "after autotune")
    st = rs.rs_sweep_stats(p.mesh, 4, B)
    assert st.shape[0] > 0 and st[:, 0].max() > 0
    # per-CTA regressors of the cost model (the "full warp-steps" column read record 0 for every step)
    assert st[:, 4].sum() > 0 and (st[:, 4] <= 8 * st[:, 1]).all() and len(set(st[:, 4].tolist())) > 1


@pytest.mark.parametrize("seed,n,B", [(0, 4, 16), (1, 4, 32), (2, 6, 16), (3, 6, 32), (4, 4, 8), (5, 6, 8)])
def test_sweep_kernel_ragged_clusters(seed, n, B):
    """Small spheres scattered so that z-rows break into several copy runs of odd lengths and most tiles are nearly
    empty: 1-D bulk copies (B = 16), overlapping 2-D tensor boxes (B = 32) and boxes wider than the block's rows
    (B = 8: half a slice, the copy unit zero-fills the other half), before and after the autotuned re-deal."""
    rng = np.random.default_rng(seed)
    nc = int(rng.integers(4, 12))
    centers = rng.uniform(0.0, 9.0, (nc, 3))
    charges = rng.choice(np.array([1.0, 4.0, 6.0]), nc)
    p = Problem(centers, charges, float(rng.uniform(1.3, 2.6)), 0.3, max_n=6)
    psi = rng.standard_normal((B + 5, p.np))
    o = p.oracle_hpsi(psi, n)
    den = p.cond_denominator(psi, n)
    check(_run(p, psi, n, B, "sweep"), o, den, f"ragged seed {seed} n={n} B={B}")
    import torch
    blk = torch.zeros((p.np + 1, B), dtype=torch.float64, device="cuda")
    hblk = torch.empty_like(blk)
    v = torch.from_numpy(p.v_mesh).cuda()
    rs.rs_mesh_set_sweep_options(p.mesh, planes_tuned=7)   # short pieces after the re-deal as well
    rs.rs_hamiltonian_autotune(p.mesh, n, oracle.fd_coeffs(n), v, blk, hblk, B)
    check(_run(p, psi, n, B, "sweep"), o, den, f"ragged seed {seed} n={n} B={B} after autotune")


def test_sweep_kernel_dirichlet_boxes():
    """Non-periodic boxes through the plane-sweep kernel: sizes that are not multiples of the 16 x 16 tile."""
    for box in [(24, 24, 24), (7, 9, 10), (1, 1, 37), (13, 1, 5), (40, 17, 33)]:
        p = Problem(None, None, None, 0.25, max_n=4, box=box, periodic=False)
        rng = np.random.default_rng(23)
        psi = rng.standard_normal((16, p.np))
        g = _run(p, psi, 4, 16, "sweep")
        o = p.oracle_hpsi(psi, 4)
        check(g, o, p.cond_denominator(psi, 4), f"sweep box {box}")


def test_config1_order6_lex_ordering():
    p = problem(1, rs.RS_ORDER_LEX)
    psi = synthetic.orbitals(2, 0, 3, p.np)
    g = p.gpu_hpsi(psi, 6, 2, ld_pad=5)
    o = p.oracle_hpsi(psi, 6)
    check(g, o, p.cond_denominator(psi, 6), "config1 lex n=6")


# ---- test boxes: Dirichlet and periodic, sizes that are not multiples of the brick / tile -------
@pytest.mark.parametrize("kernel", ["auto", "gather"])
@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("box", [(24, 24, 24), (7, 9, 10), (1, 1, 37), (13, 1, 5)])
def test_boxes(box, periodic, kernel):
    n = 4
    if periodic and min(box) == 1:
        n = 2
    p = Problem(None, None, None, 0.25, max_n=4, box=box, periodic=periodic)
    rng = np.random.default_rng(17)
    psi = rng.standard_normal((3, p.np)) + 1j * rng.standard_normal((3, p.np))
    g = _run(p, psi, n, 2, kernel)
    o = p.oracle_hpsi(psi, n)
    check(g, o, p.cond_denominator(psi, n), f"box {box} periodic={periodic}")


def test_plane_wave_closed_form_on_gpu():
    """P5 on the CUDA path itself: periodic 24^3 box, plane wave, closed-form FD symbol."""
    import math

    n, h, N, m = 4, 0.25, 24, (2, 3, 5)
    p = Problem(None, None, None, h, max_n=4, box=(N, N, N), periodic=True)
    p.v_canon[:] = 0.75
    p.v_mesh[:] = 0.75
    ijk = p.omesh.ijk().astype(np.float64)
    q = [2 * math.pi * ma / (N * h) for ma in m]
    psi = np.exp(1j * sum(q[a] * ijk[:, a] * h for a in range(3)))[None, :]
    c = [-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560]
    lam = [(c[0] + 2 * sum(c[k] * math.cos(k * q[a] * h) for k in range(1, n + 1))) / h ** 2 for a in range(3)]
    expect = (-0.5 * sum(lam) + 0.75) * psi
    g = p.gpu_hpsi(psi, n, 1, coeffs=np.array(c))
    assert np.abs(g - expect).max() / np.abs(expect).max() <= 1e-13


def test_delta_response_on_gpu():
    """P8 on the CUDA path: H delta = the star itself (validates every arm of the neighbour structure)."""
    p = problem(0)
    n = 4
    c = oracle.fd_coeffs(n)
    ijk = p.omesh.ijk()
    for ctr in ((0, 0, 0), (3, -2, 5), (0, 0, 13), (-9, 4, 2)):
        ic = int(np.flatnonzero((ijk == np.array(ctr)).all(axis=1))[0])
        psi = np.zeros((1, p.np))
        psi[0, ic] = 1.0
        g = p.gpu_hpsi(psi, n, 1)[0]
        h = p.cfg.spacing
        expect = np.zeros(p.np)
        d = ijk - np.array(ctr)
        for a in range(3):
            on_axis = (np.delete(d, a, axis=1) == 0).all(axis=1)
            for k in range(1, n + 1):
                expect[on_axis & (np.abs(d[:, a]) == k)] = -0.5 * c[k] / h ** 2
        expect[ic] = -0.5 * 3 * c[0] / h ** 2 + p.v_canon[ic]
        assert np.abs(g - expect).max() <= 16 * EPS * np.abs(expect).max(), ctr


def test_hermiticity_on_gpu():
    p = problem(1)
    phi = synthetic.orbital(101, 0, p.np, True)
    psi = synthetic.orbital(101, 1, p.np, True)
    hphi, hpsi = p.gpu_hpsi(np.stack([phi, psi]), 4, 2)
    assert abs(np.vdot(phi, hpsi) - np.vdot(hphi, psi)) / (np.linalg.norm(phi) * np.linalg.norm(hpsi)) <= 1e-13


# ---- pack / unpack: bit-exact against the oracle's layout transform -----------------------------
@pytest.mark.parametrize("is_complex", [False, True])
@pytest.mark.parametrize("B", [1, 2, 4, 8, 16, 32, 64])
def test_pack_unpack_bit_exact(B, is_complex):
    import torch

    p = problem(0)
    npts = p.np
    nst, ld = 11, npts + 3
    rng = np.random.default_rng(B)
    st = rng.standard_normal((nst, ld))
    if is_complex:
        st = st + 1j * rng.standard_normal((nst, ld))
    dst = torch.from_numpy(st).cuda()
    back = torch.full_like(dst, -7.0)
    tdt = torch.complex128 if is_complex else torch.float64
    for ist0 in range(0, nst, B):
        nb = min(B, nst - ist0)
        blk = torch.full((npts + 1, B), 5.0, dtype=tdt, device="cuda")
        rs.rs_block_pack(p.mesh, dst, ist0, nb, B, blk)
        want = oracle.block_pack(st, ist0, nb, B, npts, npts + 1)
        assert np.array_equal(blk.cpu().numpy(), want)            # zero slot row and padding columns included
        rs.rs_block_unpack(p.mesh, blk, B, nb, back, ist0)
    res = back.cpu().numpy()
    assert np.array_equal(res[:, :npts], st[:, :npts]) and np.all(res[:, npts:] == -7.0)


def test_fig4_worked_example_on_gpu():
    """PAPER.md:107 (Fig. 4): 4 orbitals x 5 coefficients, blocked address = p*4 + j."""
    import torch

    m = rs.rs_mesh_create_box(5, 1, 1, 1.0, 1, False, rs.RS_ORDER_LEX)
    st = torch.arange(20, dtype=torch.float64, device="cuda").reshape(4, 5)
    blk = torch.empty((6, 4), dtype=torch.float64, device="cuda")
    rs.rs_block_pack(m, st, 0, 4, 4, blk)
    flat = blk.cpu().numpy().ravel()
    for j in range(4):
        for pt in range(5):
            assert flat[pt * 4 + j] == j * 5 + pt
    assert np.all(flat[20:] == 0)


def test_states_host_entry_point():
    """Whole path on host buffers (step a7) = per-block device path = oracle."""
    p = problem(0)
    psi = synthetic.orbitals(9, 0, 7, p.np, is_complex=True)
    st = p.to_mesh(psi)
    out = np.zeros_like(st)
    rs.rs_hamiltonian_apply_states_host(p.mesh, 4, oracle.fd_coeffs(4), p.v_mesh, st, out, 4)
    o = p.oracle_hpsi(psi, 4)
    check(p.to_canon(out), o, p.cond_denominator(psi, 4), "states_host")


@pytest.mark.parametrize("B,nst,is_complex,ld_pad", [(4, 22, False, 3), (16, 70, False, 5), (64, 265, False, 0),
                                                     (16, 70, True, 1), (4, 22, True, 0)])
def test_states_stream_many_blocks(B, nst, is_complex, ld_pad):
    """a7 on config 1 with >= 5 blocks and a ragged last one: every window of the 3-deep ring is reused (block 3
    re-enters window 0), uploads / computes / downloads overlap on three streams, sweep kernel for B >= 16 real columns;
    padded leading dimension: the caller's padding columns must come back untouched.  Second call on the same
    workspace (nothing allocated) with other inputs."""
    p = problem(1)
    dt = rs.RS_COMPLEX128 if is_complex else rs.RS_REAL64
    ld = p.np + ld_pad
    ws = rs.rs_workspace_create(p.mesh, B, dt, ld)
    assert ws.nbytes == 3 * 2 * (B * ld * (16 if is_complex else 8) + rs.rs_block_bytes(p.mesh, B, dt)) + 8 * p.np
    for seed in (71, 72):
        psi = synthetic.orbitals(seed, 0, nst, p.np, is_complex=is_complex)
        st = np.full((nst, ld), 123.0, dtype=psi.dtype)
        st[:, :p.np] = p.to_mesh(psi)
        out = np.full((nst, ld), -7.0, dtype=psi.dtype)
        rs.rs_hamiltonian_apply_states_stream(ws, 4, oracle.fd_coeffs(4), p.v_mesh, st, out)
        assert np.all(out[:, p.np:] == -7.0)
        o = p.oracle_hpsi(psi, 4, nthreads=16)
        check(p.to_canon(out[:, :p.np]), o, p.cond_denominator(psi, 4), f"states_stream B={B} nst={nst} seed={seed}")
    if B == 16 and not is_complex:                        # the convenience form (workspace per call) gives the same bits
        out2 = np.full((nst, ld), -7.0, dtype=psi.dtype)
        rs.rs_hamiltonian_apply_states_host(p.mesh, 4, oracle.fd_coeffs(4), p.v_mesh, st, out2, B)
        assert np.array_equal(out, out2)


def test_warm_apply_allocates_nothing():
    """after rs_hamiltonian_prepare, apply / pack / unpack allocate nothing (free device memory
    unchanged across many calls, also for a new psi buffer of a wide block whose tensor maps are host-side only)."""
    import torch

    p = problem(1)
    dev = torch.device("cuda:0")
    v = torch.from_numpy(p.v_mesh).to(dev)
    c = oracle.fd_coeffs(4)
    for B in (8, 16, 32):
        bufs = [torch.zeros((p.np + 1, B), dtype=torch.float64, device=dev) for _ in range(4)]
        rs.rs_hamiltonian_prepare(p.mesh, 4, B)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for k in range(6):
            rs.rs_hamiltonian_apply(p.mesh, 4, c, v, bufs[k % 2], bufs[2 + k % 2], B)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, f"apply allocated device memory (B={B})"


def test_misaligned_block_pointers_are_rejected():
    """psi / hpsi must be 16-byte aligned on every kernel path: an offset view returns RS_ERR_INVALID_ARG
    instead of faulting in a bulk copy."""
    import torch

    p = problem(1)
    dev = torch.device("cuda:0")
    v = torch.from_numpy(p.v_mesh).to(dev)
    for B in (1, 16, 32):
        raw = torch.zeros((p.np + 1) * B + 2, dtype=torch.float64, device=dev)
        ok = torch.zeros((p.np + 1) * B, dtype=torch.float64, device=dev)
        off = raw[1:1 + (p.np + 1) * B]
        assert off.data_ptr() % 16 == 8
        for psi, hpsi in ((off, ok), (ok, off)):
            with pytest.raises(rs.RsError) as e:
                rs.rs_hamiltonian_apply(p.mesh, 4, oracle.fd_coeffs(4), v, psi, hpsi, B)
            assert e.value.status == rs.RS_ERR_INVALID_ARG
    torch.cuda.synchronize()                              # no sticky fault


def test_kernel_choice_is_reported():
    p = problem(1)
    name = rs.rs_kernel_name(p.mesh, 4, 16)
    assert name == "gather" or name.startswith("sweep[")
    assert rs.rs_kernel_table_bytes(p.mesh, 4, 16, kernel=rs.RS_KERNEL_GATHER) == p.np * 24 * 4


# ---- full-size configs (BASELINE.json configs[2..4]) in the launch configuration bench.py times -----------
# One block of orbitals through pack -> apply -> unpack on the full mesh, every output compared with the
# oracle (the oracle does a whole orbital of these meshes in a fraction of a second per core).
@pytest.mark.parametrize("B", [1, 2, 4, 8, 16, 32, 64])
def test_config2_full_mesh_block(B):
    """Every block size BASELINE.json configs[2] names, on the full 1.96 M-point mesh (B = 8: half a 16-column slice of the
    plane-sweep kernel; B < 8: the gather kernel)."""
    p = problem(2)
    cfg = p.cfg
    nst = B + 3 if B == 16 else B                       # B = 16: a second, ragged block as well
    psi = synthetic.orbitals(cfg.seed, 0, nst, p.np)
    g = _run(p, psi, 4, B, "auto")
    assert rs.rs_kernel_name(p.mesh, 4, B).startswith("sweep[" if B >= 8 else "gather")
    o = p.oracle_hpsi(psi, 4, nthreads=16)
    check(g, o, p.cond_denominator(psi, 4), f"config2 B={B}")


@pytest.mark.parametrize("B", [1, 2, 4, 8, 16, 32])
def test_config3_complex_full_mesh_block(B):
    """Every block size BASELINE.json configs[3] names (complex: 2 B real columns; B < 4: the gather kernel)."""
    p = problem(2)                                       # config 3 = config 2's mesh and potential, complex orbitals
    cfg = synthetic.config(3)
    psi = synthetic.orbitals(cfg.seed, 0, B, p.np, is_complex=True)
    g = _run(p, psi, 4, B, "auto")
    assert rs.rs_kernel_name(p.mesh, 4, B, rs.RS_COMPLEX128).startswith("sweep[" if B >= 4 else "gather")
    o = p.oracle_hpsi(psi, 4, nthreads=16)
    check(g, o, p.cond_denominator(psi, 4), f"config3 complex B={B}")


@pytest.mark.parametrize("n,B", [(4, 16), (4, 32), (4, 64), (6, 16), (6, 32), (6, 64)])
def test_config4_full_mesh_block(n, B):
    """BASELINE.json configs[4]: blocks of 16 / 32 / 64 REAL orbitals (no padding columns), orders 4 and 6."""
    p = problem(4)                                       # 500 centres, 3.8 M points
    cfg = p.cfg
    psi = synthetic.orbitals(cfg.seed, 0, B, p.np)
    g = _run(p, psi, n, B, "auto")
    assert rs.rs_kernel_name(p.mesh, n, B).startswith(f"sweep[n{n}")
    o = p.oracle_hpsi(psi, n, nthreads=16)
    check(g, o, p.cond_denominator(psi, n), f"config4 n={n} B={B}")


def test_config4_streamed_at_its_stated_size():
    """BASELINE.json configs[4] end to end: 1024 real orbitals streamed through HBM in blocks of 64, fd_order 4, through
    the a7 workspace (3 windows: the device never holds more than 3 blocks).  Orbitals are generated chunk by chunk on
    the host (neither side holds the 31 GB set); one sampled orbital per 128 is compared with the oracle."""
    p = problem(4)
    cfg = p.cfg
    B, chunk, n = 64, 128, 4
    ws = rs.rs_workspace_create(p.mesh, B, rs.RS_REAL64, p.np)
    c = oracle.fd_coeffs(n)
    rng = np.random.default_rng(4)
    worst = 0.0
    for ist0 in range(0, cfg.nst, chunk):
        psi = synthetic.orbitals(cfg.seed, ist0, chunk, p.np)
        st = p.to_mesh(psi)
        out = np.empty_like(st)
        rs.rs_hamiltonian_apply_states_stream(ws, n, c, p.v_mesh, st, out)
        j = int(rng.integers(0, chunk))                  # a seeded sample: orbital ist0 + j
        o = p.oracle_hpsi(psi[j:j + 1], n, nthreads=16)
        worst = max(worst, check(p.to_canon(out[j:j + 1]), o, p.cond_denominator(psi[j:j + 1], n), f"config4 orbital {ist0 + j}"))
        assert np.isfinite(out).all()
    assert worst <= 1e-12
