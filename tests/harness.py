"""Shared plumbing of the GPU parity tests: build one problem on both sides (library mesh + oracle
mesh), move seeded canonical-order inputs into the library's enumeration, run the CUDA path through
the C ABI, bring results back to canonical order and compare with the oracle.

Tolerances:
  NORMWISE  max|g - o| / max|o| <= 1e-12        -- north_star's "max relative error 1e-12"
  CONDWISE  |g - o|_i <= 64 eps * (sum_k |w_k||psi_nbr| + |V psi|)_i   -- elementwise, conditioning-aware
"""
from __future__ import annotations

import numpy as np

import oracle
import synthetic
import paper_1306_2953_b200 as rs

NORMWISE_TOL = 1e-12
EPS = np.finfo(np.float64).eps


class Problem:
    def __init__(self, centers, charges, radius, spacing, max_n=6, ordering=rs.RS_ORDER_LEX, box=None,
                 periodic=False):
        if box is None:
            self.mesh = rs.rs_mesh_create(centers, radius, spacing, max_n, ordering)
            self.omesh = oracle.mesh_from_spheres(centers, radius, spacing)
        else:
            self.mesh = rs.rs_mesh_create_box(*box, spacing, max_n, periodic, ordering)
            self.omesh = oracle.mesh_box(*box, spacing, periodic)
        self.np = self.mesh.npoints
        assert self.np == self.omesh.npoints
        self.ijk = self.mesh.points()
        self.rank = synthetic.canonical_rank(self.ijk)        # mesh index -> canonical index
        assert np.array_equal(self.rank, self.omesh.canonical_rank_of(self.ijk))   # same point SET
        if centers is not None:
            self.v_canon = synthetic.vloc_at(self.omesh.xyz(), np.asarray(centers, float), np.asarray(charges, float))
        else:
            self.v_canon = np.random.default_rng(99).standard_normal(self.np)
        self.v_mesh = self.v_canon[self.rank]

    @classmethod
    def from_config(cls, i, **kw):
        cfg = synthetic.config(i)
        p = cls(cfg.centers, cfg.charges, cfg.radius, cfg.spacing, **kw)
        p.cfg = cfg
        return p

    def to_mesh(self, f_canon):
        return np.ascontiguousarray(f_canon[..., self.rank])

    def to_canon(self, f_mesh):
        out = np.empty_like(f_mesh)
        out[..., self.rank] = f_mesh
        return out

    # ---- the CUDA path, through the binding (pack -> apply -> unpack per block) ------------------
    def gpu_hpsi(self, psi_canon, n, B, kernel=rs.RS_KERNEL_AUTO, coeffs=None, ld_pad=0):
        import torch

        coeffs = oracle.fd_coeffs(n) if coeffs is None else coeffs   # coefficients are an INPUT of the C ABI
        nst = psi_canon.shape[0]
        is_c = np.iscomplexobj(psi_canon)
        tdt = torch.complex128 if is_c else torch.float64
        ld = self.np + ld_pad
        st_host = np.zeros((nst, ld), dtype=psi_canon.dtype)
        st_host[:, :self.np] = self.to_mesh(psi_canon)
        dev = torch.device("cuda:0")
        states = torch.from_numpy(st_host).to(dev)
        out = torch.full((nst, ld), -7.0, dtype=tdt, device=dev)
        v = torch.from_numpy(self.v_mesh).to(dev)
        blk = torch.empty((self.np + 1, B), dtype=tdt, device=dev)
        hblk = torch.full((self.np + 1, B), 3.0, dtype=tdt, device=dev)
        assert blk.numel() * blk.element_size() == rs.rs_block_bytes(self.mesh, B, rs.RS_COMPLEX128 if is_c else rs.RS_REAL64)
        for ist0 in range(0, nst, B):
            nb = min(B, nst - ist0)
            rs.rs_block_pack(self.mesh, states, ist0, nb, B, blk)
            rs.rs_hamiltonian_apply(self.mesh, n, coeffs, v, blk, hblk, B, kernel=kernel)
            rs.rs_block_unpack(self.mesh, hblk, B, nb, out, ist0)
        torch.cuda.synchronize()
        assert torch.all(hblk[self.np] == 3.0)          # apply never writes the zero-slot row
        res = out.cpu().numpy()
        if ld_pad:
            assert np.all(res[:, self.np:] == -7.0)     # unpack never writes beyond np
        return self.to_canon(res[:, :self.np])

    def oracle_hpsi(self, psi_canon, n, nthreads=8):
        return oracle.hpsi(self.omesh, n, oracle.fd_coeffs(n), self.v_canon, psi_canon, nthreads=nthreads)

    def cond_denominator(self, psi_canon, n):
        """sum_k |w_k| |psi_nbr| + |V psi| per output: the oracle applied to |psi| with coefficients -|c_k|
        (so that -1/2 c_k/h^2 becomes +|w_k|) and potential |V|.  Complex: |re| + |im| bounds both lanes."""
        absn = np.abs(psi_canon.real) + (np.abs(psi_canon.imag) if np.iscomplexobj(psi_canon) else 0.0)
        return oracle.hpsi(self.omesh, n, -np.abs(oracle.fd_coeffs(n)), np.abs(self.v_canon), absn, nthreads=8)


def check(g, o, denom=None, what=""):
    """normwise bound always; conditioning-aware elementwise bound when `denom` is given."""
    scale = np.abs(o).max()
    err = np.abs(g - o).max() / scale
    assert err <= NORMWISE_TOL, f"{what}: normwise error {err:.3e} > {NORMWISE_TOL}"
    if denom is not None:
        bad = np.abs(g - o) > 64 * EPS * denom + 1e-300
        assert not bad.any(), f"{what}: {int(bad.sum())} outputs beyond 64 eps * conditioning"
    return err
