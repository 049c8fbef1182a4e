"""Host-side checks of librs.so that need no GPU: the library loads and exports every symbol of
include/rs.h; the mesh builder (steps a1-a3) agrees with the oracle's own mask as a point SET and
arm by arm; argument errors are reported as include/rs.h says.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import synthetic
import paper_1306_2953_b200 as rs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "rs.h")).read()
    body = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(rs_[a-z_0-9]+)\s*\(", body))
    assert declared == set(rs.EXPORTS), declared ^ set(rs.EXPORTS)
    lib = C.CDLL(rs.LIBRARY_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert rs.rs_version() >= 100


def test_binding_never_imports_oracle():
    src = open(os.path.join(ROOT, "paper_1306_2953_b200", "__init__.py")).read()
    src += open(os.path.join(ROOT, "paper_1306_2953_b200", "build.py")).read()
    assert "oracle" not in src
    for f in os.listdir(os.path.join(ROOT, "paper_1306_2953_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_1306_2953_b200", "csrc", f)).read().lower(), f
    osrc = (open(os.path.join(ROOT, "oracle", "oracle.c")).read() + open(os.path.join(ROOT, "oracle", "oracle_next.c")).read() +
            open(os.path.join(ROOT, "oracle", "__init__.py")).read())
    assert "rs.h" not in osrc and "import paper_1306" not in osrc and "librs" not in osrc


def _sets_equal(lib_ijk, omesh):
    a = set(map(tuple, lib_ijk.tolist()))
    b = set(map(tuple, omesh.ijk().tolist()))
    return a == b, (a - b, b - a)


@pytest.mark.parametrize("ordering", [rs.RS_ORDER_BRICK, rs.RS_ORDER_LEX, rs.RS_ORDER_TILE])
@pytest.mark.parametrize("cfg_i", [0, 1])
def test_mesh_point_set_equals_oracle(cfg_i, ordering):
    cfg = synthetic.config(cfg_i)
    m = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 6, ordering)
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    assert m.npoints == om.npoints == cfg.np_expected
    ijk = m.points()
    assert len(set(map(tuple, ijk.tolist()))) == m.npoints          # no duplicates
    ok, diff = _sets_equal(ijk, om)
    assert ok, diff
    if ordering == rs.RS_ORDER_LEX:
        assert np.array_equal(ijk, om.ijk())
        assert np.array_equal(synthetic.canonical_rank(ijk), np.arange(m.npoints))
    elif ordering == rs.RS_ORDER_TILE:
        # i decreases only where the enumeration moves on to the next tile column (the tile origin is the library's)
        ext = ijk.max(axis=0) - ijk.min(axis=0) + 1
        ncols = (ext[1] // 16 + 2) * (ext[2] // 16 + 2)
        assert (np.diff(ijk[:, 0]) < 0).sum() < ncols and m.nbricks == 0
        same_plane = np.diff(ijk[:, 0]) == 0                   # inside a tile plane: (j, k) ascending, within 16 x 16
        dj, dk = np.diff(ijk[:, 1])[same_plane], np.diff(ijk[:, 2])[same_plane]
        assert ((dj > 0) | ((dj == 0) & (dk > 0))).all() and np.abs(dj).max() < 16 and np.abs(dk).max() < 16
    else:
        assert m.nbricks > 0
    # canonical_rank agrees with the oracle's own ranking of the same points
    assert np.array_equal(synthetic.canonical_rank(ijk), om.canonical_rank_of(ijk))


def test_mesh_table1_benzene_count():
    c, _ = synthetic.benzene_centers()
    assert rs.rs_mesh_create(c, 5.5, 0.41, 4).npoints == 37295      # PAPER.md:513 prints 37.3k


def test_mesh_off_lattice_centres_and_negative_coordinates():
    rng = np.random.default_rng(3)
    c = rng.uniform(-3.0, 3.0, (5, 3)) + np.array([-7.3, 2.1, 0.4])
    m = rs.rs_mesh_create(c, 2.7, 0.33, 4)
    om = oracle.mesh_from_spheres(c, 2.7, 0.33)
    ok, diff = _sets_equal(m.points(), om)
    assert ok, diff


def _bruteforce_map(ijk, n, periodic_box=None):
    """neighbour table from the definition, through a python dict (independent of both builders)."""
    lut = {tuple(p): i for i, p in enumerate(ijk.tolist())}
    npts = len(lut)
    out = np.full((npts, 6 * n), npts, dtype=np.int32)
    for ip, p in enumerate(ijk.tolist()):
        for a in range(3):
            for k in range(1, n + 1):
                for sgn, d in ((0, k), (1, -k)):
                    q = list(p)
                    q[a] += d
                    if periodic_box is not None:
                        q[a] %= periodic_box[a]
                    out[ip, a * 2 * n + 2 * (k - 1) + sgn] = lut.get(tuple(q), npts)
    return out


@pytest.mark.parametrize("ordering", [rs.RS_ORDER_BRICK, rs.RS_ORDER_LEX, rs.RS_ORDER_TILE])
@pytest.mark.parametrize("n", [1, 4, 6])
def test_index_map_matches_definition_and_invariants(n, ordering):
    cfg = synthetic.config(0)
    m = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 6, ordering)
    npts = m.npoints
    mp = m.index_map(n)
    assert mp.shape == (npts, 6 * n)
    assert mp.min() >= 0 and mp.max() <= npts
    assert np.array_equal(mp, _bruteforce_map(m.points(), n))
    # P11: map(map(ip,+k),-k) == ip wherever the forward entry is a real point
    for a in range(3):
        for k in range(1, n + 1):
            fwd = mp[:, a * 2 * n + 2 * (k - 1)]
            real = fwd < npts
            back = mp[fwd[real], a * 2 * n + 2 * (k - 1) + 1]
            assert np.array_equal(back, np.flatnonzero(real))
    # P11: number of zero-slot entries == the oracle's count of star arms leaving the domain
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    assert int((mp == npts).sum()) == oracle.count_outside_arms(om, n)


@pytest.mark.parametrize("periodic", [False, True])
def test_box_mesh_and_map(periodic):
    nx, ny, nz, n = 7, 9, 10, 4
    m = rs.rs_mesh_create_box(nx, ny, nz, 0.3, n, periodic)
    assert m.npoints == nx * ny * nz
    ijk = m.points()
    assert ijk.min() == 0 and tuple(ijk.max(axis=0)) == (nx - 1, ny - 1, nz - 1)
    mp = m.index_map(n)
    assert np.array_equal(mp, _bruteforce_map(ijk, n, (nx, ny, nz) if periodic else None))
    if periodic:
        assert mp.max() < m.npoints            # no arm ever leaves a periodic box
    else:
        om = oracle.mesh_box(nx, ny, nz, 0.3, False)
        assert int((mp == m.npoints).sum()) == oracle.count_outside_arms(om, n)


def test_block_bytes_and_argument_errors():
    m = rs.rs_mesh_create(np.zeros((1, 3)), 2.0, 0.5, 4)
    npts = m.npoints
    assert rs.rs_block_bytes(m, 16, rs.RS_REAL64) == (npts + 1) * 16 * 8
    assert rs.rs_block_bytes(m, 8, rs.RS_COMPLEX128) == (npts + 1) * 8 * 16
    assert rs.rs_block_bytes(m, 3, rs.RS_REAL64) == 0 and rs.rs_block_bytes(m, 128, rs.RS_REAL64) == 0
    with pytest.raises(rs.RsError) as e:
        rs.rs_mesh_create(np.zeros((1, 3)), -1.0, 0.5, 4)
    assert e.value.status == rs.RS_ERR_INVALID_ARG
    with pytest.raises(rs.RsError):
        rs.rs_mesh_create(np.zeros((1, 3)), 2.0, 0.5, rs.RS_MAX_FD_ORDER + 1)
    with pytest.raises(rs.RsError):
        m.index_map(5)                         # > max_fd_order of this mesh
    with pytest.raises(rs.RsError) as e:
        rs.rs_mesh_create(np.array([[100.2, 0.2, 0.2]]), 0.01, 0.5, 4)   # sphere holds no lattice point
    assert e.value.status == rs.RS_ERR_INVALID_ARG


def test_compute_calls_validate_arguments_before_touching_the_device():
    """Argument errors come back as RS_ERR_INVALID_ARG with or without a GPU (no launch is made)."""
    m = rs.rs_mesh_create(np.zeros((1, 3)), 2.0, 0.5, 4)
    npts = m.npoints
    c = np.array([-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560])
    v = np.zeros(npts)
    a = np.zeros((npts + 1) * 4)
    b = np.zeros((npts + 1) * 4)
    for bad in (dict(nst=3), dict(nst=128), dict(fd_order=0), dict(fd_order=5), dict(alias=True)):
        nst = bad.get("nst", 4)
        n = bad.get("fd_order", 4)
        cc = c if n == 4 else np.zeros(n + 1)
        with pytest.raises(rs.RsError) as e:
            rs.rs_hamiltonian_apply(m, n, cc, v, a, a if bad.get("alias") else b, nst, rs.RS_REAL64, stream=0)
        assert e.value.status == rs.RS_ERR_INVALID_ARG, bad
    st = np.zeros((2, npts))
    with pytest.raises(rs.RsError) as e:
        rs.rs_block_pack(m, st, 0, 5, 4, a, stream=0)           # nst_in_block > block_size
    assert e.value.status == rs.RS_ERR_INVALID_ARG
    with pytest.raises(rs.RsError) as e:
        rs.rs_block_unpack(m, a, 4, 2, st, 0, stream=0, ld=npts - 1)   # ld < np
    assert e.value.status == rs.RS_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    m = rs.rs_mesh_create(np.zeros((1, 3)), 2.0, 0.5, 4)
    npts = m.npoints
    c = np.array([-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560])
    a = np.zeros((npts + 1) * 4)
    b = np.zeros((npts + 1) * 4)
    with pytest.raises(rs.RsError) as e:
        rs.rs_hamiltonian_apply(m, 4, c, np.zeros(npts), a, b, 4, rs.RS_REAL64, stream=0)
    assert e.value.status == rs.RS_ERR_CUDA
    assert np.all(b == 0)
    with pytest.raises(rs.RsError) as e:
        rs.rs_hamiltonian_apply_states_host(m, 4, c, np.zeros(npts), np.zeros((4, npts)), np.zeros((4, npts)), 4)
    assert e.value.status == rs.RS_ERR_CUDA


def test_misaligned_block_pointers_are_rejected_without_a_device():
    """Argument checks come before the device check: a psi / hpsi pointer that is not 16-byte aligned (an offset view)
    is RS_ERR_INVALID_ARG on every kernel path (rs.h "Alignment")."""
    m = rs.rs_mesh_create_box(8, 8, 8, 0.25, 4)
    npts = m.npoints
    c = np.array([-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560])
    for B in (1, 16, 32):
        raw = np.zeros((npts + 1) * B + 4)
        base = 0 if raw.ctypes.data % 16 == 0 else 1
        ok, off = raw[base:base + (npts + 1) * B], raw[base + 1:base + 1 + (npts + 1) * B]
        other = np.zeros((npts + 1) * B + 2)
        other = other[(0 if other.ctypes.data % 16 == 0 else 1):][:(npts + 1) * B]
        assert off.ctypes.data % 16 == 8 and ok.ctypes.data % 16 == 0 and other.ctypes.data % 16 == 0
        for psi, hpsi in ((off, other), (other, off)):
            with pytest.raises(rs.RsError) as e:
                rs.rs_hamiltonian_apply(m, 4, c, np.zeros(npts), psi, hpsi, B, rs.RS_REAL64, stream=0)
            assert e.value.status == rs.RS_ERR_INVALID_ARG


# ---- plane-sweep kernel's compact records: host replay against the plain neighbour table (reading S15) ----
@pytest.mark.parametrize("cfg_i,nst,dtype,planes,nctas", [
    (0, 16, rs.RS_REAL64, 32, 148), (0, 16, rs.RS_REAL64, 8, 3), (1, 16, rs.RS_REAL64, 32, 148),
    (1, 32, rs.RS_REAL64, 32, 148), (1, 64, rs.RS_REAL64, 16, 132), (1, 8, rs.RS_COMPLEX128, 32, 148),
    (1, 16, rs.RS_REAL64, 100, 1), (1, 16, rs.RS_REAL64, 12, 1000),
])
def test_sweep_records_expand_to_the_plain_table(cfg_i, nst, dtype, planes, nctas):
    cfg = synthetic.config(cfg_i)
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 4)
    st = rs.rs_sweep_selfcheck(mesh, 4, nst, dtype, planes, nctas)
    assert st["nctas"] == nctas and st["records"] > 0 and st["cost_max"] >= st["cost_mean"] > 0


@pytest.mark.parametrize("cfg_i,n,nst", [(0, 6, 16), (1, 6, 16), (1, 6, 64)])
def test_sweep_records_order6_shape(cfg_i, n, nst):
    """fd_order 6 runs on its own kernel shape (8 x 16 tiles, 2 x 4 patches)."""
    cfg = synthetic.config(cfg_i)
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 6)
    st = rs.rs_sweep_selfcheck(mesh, n, nst, rs.RS_REAL64, 32, 148)
    assert st["records"] > 0


def test_sweep_options_are_per_mesh():
    """No process-global tuning state: options live in the mesh handle."""
    d = rs.rs_sweep_options_default()
    assert (d.planes, d.planes_tuned, d.ctas, d.force_tensor, d.min_split, d.tune_rounds) == (32, 1 << 20, 0, 0, 3, 3)
    a = rs.rs_mesh_create_box(24, 24, 24, 0.25, 4)
    b = rs.rs_mesh_create_box(24, 24, 24, 0.25, 4)
    rs.rs_mesh_set_sweep_options(a, force_tensor=1, ctas=5)
    assert "tma2d" in rs.rs_kernel_name(a, 4, 16, kernel=rs.RS_KERNEL_SWEEP)
    assert "tma1d" in rs.rs_kernel_name(b, 4, 16, kernel=rs.RS_KERNEL_SWEEP)
    with pytest.raises(rs.RsError) as e:
        rs.rs_mesh_set_sweep_options(a, planes=0)
    assert e.value.status == rs.RS_ERR_INVALID_ARG
    with pytest.raises(rs.RsError):
        rs.rs_mesh_set_sweep_options(a, no_such_field=1)


def test_sweep_selfcheck_on_boxes_and_unsupported_calls():
    for box in [(24, 24, 24), (7, 9, 10), (1, 1, 37), (40, 17, 33)]:
        mesh = rs.rs_mesh_create_box(*box, 0.25, 4, False, rs.RS_ORDER_LEX)
        rs.rs_sweep_selfcheck(mesh, 4, 16, rs.RS_REAL64, 32, 148)
    mesh = rs.rs_mesh_create_box(8, 8, 8, 0.25, 4, True, rs.RS_ORDER_LEX)          # periodic: gather kernel only
    with pytest.raises(rs.RsError) as e:
        rs.rs_sweep_selfcheck(mesh, 4, 16)
    assert e.value.status == rs.RS_ERR_UNSUPPORTED
    mesh = rs.rs_mesh_create_box(8, 8, 8, 0.25, 5, False, rs.RS_ORDER_LEX)
    with pytest.raises(rs.RsError) as e:
        rs.rs_sweep_selfcheck(mesh, 4, 4)                                           # 4 real columns: gather kernel only
    assert e.value.status == rs.RS_ERR_UNSUPPORTED
    rs.rs_sweep_selfcheck(mesh, 4, 8)                                               # 8 real columns: half a 16-column slice
    rs.rs_sweep_selfcheck(mesh, 4, 4, rs.RS_COMPLEX128)
    with pytest.raises(rs.RsError) as e:
        rs.rs_sweep_selfcheck(mesh, 5, 16)                                          # fd_order 5: gather kernel only
    assert e.value.status == rs.RS_ERR_UNSUPPORTED


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_sweep_records_on_random_sparse_clusters(seed):
    """Ragged meshes: small spheres scattered so that z-rows break into several runs, tiles are mostly empty and
    pieces are short; the record replay must still expand to the plain table (both kernel shapes, odd CTA counts)."""
    rng = np.random.default_rng(seed)
    nc = int(rng.integers(3, 12))
    centers = rng.uniform(0.0, 9.0, (nc, 3))
    radius = float(rng.uniform(1.1, 2.6))
    mesh = rs.rs_mesh_create(centers, radius, 0.3, 6)
    for n in (4, 6):
        for nst, planes, nctas in ((16, int(rng.integers(4, 40)), int(rng.integers(1, 200))), (32, 1 << 20, 148)):
            st = rs.rs_sweep_selfcheck(mesh, n, nst, rs.RS_REAL64, planes, nctas)
            assert st["records"] > 0


# ---- f3: non-local potential, host side (spheres, colouring) -- no device needed ------------------------------------
def test_nonlocal_spheres_equal_the_oracles_and_colours_are_race_free():
    """The library's projector spheres (closed ball on the mesh) are the oracle's point sets, and no two atoms of one
    colour share a mesh point ("groups whose spheres do not overlap")."""
    cfg = synthetic.config(1)                                   # 12 centres, heavily overlapping spheres at rc = 2.0
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 4)
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    rank = synthetic.canonical_rank(mesh.points())
    rc = 2.0
    nl = rs.rs_nonlocal_create(mesh, cfg.centers, rc, 4)
    sets = []
    for A in range(cfg.centers.shape[0]):
        idx = nl.sphere(A)
        assert np.all(np.diff(idx) > 0)
        assert np.array_equal(np.sort(rank[idx]), oracle.sphere_points(om, cfg.centers[A], rc))
        sets.append(set(idx.tolist()))
    col = nl.colors()
    assert col.min() == 0 and col.max() + 1 == nl.ncolors and nl.ncolors >= 2
    for A in range(len(sets)):
        for Bq in range(A):
            if col[A] == col[Bq]:
                assert not (sets[A] & sets[Bq]), (A, Bq)
    # greedy: every atom of colour c > 0 conflicts with some atom of every lower colour
    for A in range(len(sets)):
        for c in range(col[A]):
            assert any(col[Bq] == c and (sets[A] & sets[Bq]) for Bq in range(len(sets)))
    # far-apart atoms: one colour; a sphere outside the mesh: empty
    far = rs.rs_nonlocal_create(mesh, np.array([[0.0, 0.0, 0.0], [100.0, 0.0, 0.0]]), 1.0, 1)
    assert far.ncolors == 1 and far.sphere(1).size == 0 and far.sphere(0).size > 0
    with pytest.raises(rs.RsError) as e:
        rs.rs_nonlocal_create(mesh, cfg.centers, rc, 17)
    assert e.value.status == rs.RS_ERR_INVALID_ARG


def test_next_row_entry_points_check_arguments_without_a_device():
    """f1-f3 entry points: bad arguments -> RS_ERR_INVALID_ARG, good arguments on a host-only handle -> RS_ERR_CUDA (no fallback)."""
    import ctypes as C

    m = rs.rs_mesh_create_box(8, 8, 8, 0.25, 4)
    npts = m.npoints

    def aligned(n):
        raw = np.zeros(n + 2)
        return raw[(0 if raw.ctypes.data % 16 == 0 else 1):][:n]

    a, b = aligned((npts + 1) * 4), aligned((npts + 1) * 4)
    out = np.zeros(16)
    L, h = rs._lib, m.handle
    ptr = lambda x: C.c_void_p(x.ctypes.data)
    assert L.rs_block_dot(h, ptr(a), ptr(b), 3, rs.RS_REAL64, ptr(out), None) == rs.RS_ERR_INVALID_ARG          # width not a power of two
    assert L.rs_block_dot(h, ptr(a), None, 4, rs.RS_REAL64, ptr(out), None) == rs.RS_ERR_INVALID_ARG
    assert L.rs_block_dot(h, ptr(a[1:]), ptr(b), 4, rs.RS_REAL64, ptr(out), None) == rs.RS_ERR_INVALID_ARG      # misaligned block
    assert L.rs_block_axpy(h, ptr(out), ptr(a), ptr(a), 4, rs.RS_REAL64, None) == rs.RS_ERR_INVALID_ARG         # x == y
    assert L.rs_block_overlap(h, ptr(a), ptr(b), 4, 7, ptr(out), None) == rs.RS_ERR_INVALID_ARG                 # bad dtype
    assert L.rs_block_expectation(h, ptr(a), ptr(b), None, 4, rs.RS_REAL64, None, None) == rs.RS_ERR_INVALID_ARG
    c = np.array([-205 / 72, 8 / 5, -1 / 5, 8 / 315, -1 / 560])
    assert L.rs_hamiltonian_apply_ex(h, 4, c.ctypes.data_as(C.POINTER(C.c_double)), ptr(out), ptr(a), ptr(b), 4, rs.RS_REAL64, None,
                                     None, None) == rs.RS_ERR_INVALID_ARG
    # the allocation-free expectation sums: 64 real columns at most, whatever the device
    wide = aligned((npts + 1) * 128)
    assert L.rs_block_expectation_static(h, ptr(wide), ptr(wide), None, 64, rs.RS_COMPLEX128, ptr(out), None) == rs.RS_ERR_INVALID_ARG
    assert b"static scratch" in L.rs_last_error()
    assert L.rs_block_expectation_static(h, ptr(a[1:]), ptr(b), None, 4, rs.RS_REAL64, ptr(out), None) == rs.RS_ERR_INVALID_ARG
    assert L.rs_block_expectation_static(h, ptr(a), ptr(b), None, 3, rs.RS_REAL64, ptr(out), None) == rs.RS_ERR_INVALID_ARG
    nl0 = rs.rs_nonlocal_create(m, np.zeros((1, 3)), 0.6, 1)
    nl0.set_projectors(0, np.ones((nl0.sphere(0).size, 1)))
    assert L.rs_nonlocal_apply(nl0._h, ptr(a[1:]), ptr(b), 4, rs.RS_REAL64, None) == rs.RS_ERR_INVALID_ARG      # misaligned block
    assert L.rs_nonlocal_apply(nl0._h, ptr(a), ptr(a), 4, rs.RS_REAL64, None) == rs.RS_ERR_INVALID_ARG          # in place
    import torch
    if not torch.cuda.is_available():
        for call in (lambda: L.rs_block_dot(h, ptr(a), ptr(b), 4, rs.RS_REAL64, ptr(out), None),
                     lambda: L.rs_block_expectation_static(h, ptr(a), ptr(b), None, 4, rs.RS_REAL64, ptr(out), None),
                     lambda: L.rs_block_overlap(h, ptr(a), ptr(b), 4, rs.RS_REAL64, ptr(out), None),
                     lambda: L.rs_block_axpy(h, ptr(out), ptr(a), ptr(b), 4, rs.RS_REAL64, None),
                     lambda: L.rs_block_copy(h, ptr(a), ptr(b), 4, rs.RS_REAL64, None),
                     lambda: L.rs_hamiltonian_prepare(h, 4, 4, rs.RS_REAL64)):
            assert call() == rs.RS_ERR_CUDA
        nl = rs.rs_nonlocal_create(m, np.zeros((1, 3)), 0.6, 1)
        nl.set_projectors(0, np.ones((nl.sphere(0).size, 1)))
        with pytest.raises(rs.RsError) as e:
            rs.rs_nonlocal_apply(nl, a, b, 4, stream=0)
        assert e.value.status == rs.RS_ERR_CUDA
        with pytest.raises(rs.RsError) as e:
            rs.rs_workspace_create(m, 4, rs.RS_REAL64, npts)
        assert e.value.status == rs.RS_ERR_CUDA
    with pytest.raises(rs.RsError) as e:
        rs.rs_workspace_create(m, 4, rs.RS_REAL64, npts - 1)            # ld < np
    assert e.value.status == rs.RS_ERR_INVALID_ARG
