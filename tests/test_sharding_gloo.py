"""Multi-GPU path on CPU (world_size 2, gloo): the path shards over orbital blocks with no exchange
(orbitals are independent).  Each rank takes the contiguous range of
whole blocks that synthetic.shard_orbitals deals it, computes H psi for that range with the oracle standing in
for the device (no GPU here), and the gathered result must equal the unsharded one; the max-over-ranks timing
reduction bench.py uses is exercised too.  What runs of the product here: every rank builds its own replica of the
mesh through librs.so (host tables only: mesh, plane-sweep records and their replay) and the replicas must be
identical; the kernels themselves need a device.  No multi-GPU run exists (gpurun gives one GPU)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import synthetic


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nst, block, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = synthetic.config(0)
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    v = synthetic.vloc_at(om.xyz(), cfg.centers, cfg.charges)
    lo, hi = synthetic.shard_orbitals(nst, block, rank, world)
    mine = np.zeros((nst, om.npoints))
    if hi > lo:
        psi = synthetic.orbitals(cfg.seed, lo, hi - lo, om.npoints)
        mine[lo:hi] = oracle.hpsi(om, 4, oracle.fd_coeffs(4), v, psi, nthreads=1)
    t = torch.from_numpy(mine)
    dist.all_reduce(t)                                   # test-side gather only: disjoint ranges, so the sum is the union
    ms = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)            # bench.py's max-over-ranks timing
    ranges = [None] * world
    dist.all_gather_object(ranges, (lo, hi))
    # the product's replicated set-up: each rank builds the mesh and the sweep records itself
    import hashlib
    import paper_1306_2953_b200 as rs
    mesh = rs.rs_mesh_create(cfg.centers, cfg.radius, cfg.spacing, 4)
    st = rs.rs_sweep_selfcheck(mesh, 4, 16)
    digest = hashlib.sha256(mesh.points().tobytes()).hexdigest() + f":{st['records']}:{st['table_bytes']}"
    digests = [None] * world
    dist.all_gather_object(digests, digest)
    assert len(set(digests)) == 1 and mesh.npoints == om.npoints
    ids = [None] * world
    dist.all_gather_object(ids, list(synthetic.rank_orbital_ids(rank, nst)))
    assert sorted(sum(ids, [])) == list(range(world * nst))          # bench.py's weak-scaling ownership: disjoint, complete
    if rank == 0:
        np.savez(out_path, h=t.numpy(), ms=ms.numpy(), ranges=np.array(ranges))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("nst,block", [(10, 4), (3, 2), (1, 4)])
def test_orbital_block_sharding_world2(tmp_path, nst, block):
    out = str(tmp_path / "gathered.npz")
    mp.spawn(_worker, args=(2, _free_port(), nst, block, out), nprocs=2, join=True)
    got = np.load(out)
    cfg = synthetic.config(0)
    om = oracle.mesh_from_spheres(cfg.centers, cfg.radius, cfg.spacing)
    v = synthetic.vloc_at(om.xyz(), cfg.centers, cfg.charges)
    ref = oracle.hpsi(om, 4, oracle.fd_coeffs(4), v, synthetic.orbitals(cfg.seed, 0, nst, om.npoints), nthreads=2)
    assert np.array_equal(got["h"], ref)                 # same arithmetic, same order: bit-identical
    assert got["ms"][0] == 2.0
    r = got["ranges"]
    assert r[0][0] == 0 and r[0][1] == r[1][0] and r[1][1] == nst          # contiguous, disjoint, complete
    assert all(lo % block == 0 for lo, _ in r if lo < nst)                  # whole blocks


def test_shard_orbitals_properties():
    for nst, block, world in [(256, 16, 8), (1024, 64, 8), (7, 4, 3), (5, 8, 2)]:
        spans = [synthetic.shard_orbitals(nst, block, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == nst
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        sizes = [(hi - lo + block - 1) // block for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1
