"""N > 1 path on CPU (gloo, world_size 2): transducers are sharded, H needs no exchange, H^T's partial
volumes are summed by one all-reduce.  The operator here is the oracle -- what is
under test is the host-side sharding / reduction logic of paper_1304_2017_b200.shard."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1304_2017_b200 import shard, workloads as wl


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 64, 9216):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                lo, hi = shard.shard_range(n, r, world)
                assert 0 <= lo <= hi <= n
                seen += list(range(lo, hi))
            assert seen == list(range(n))
            sizes = [shard.shard_range(n, r, world)[1] - shard.shard_range(n, r, world)[0] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def test_weak_replicas_are_rotations_about_z():
    tr = wl.arc_array(4, 6, 65.0)
    r1 = shard.weak_replica_transducers(tr, 1, 2, 6)
    assert np.allclose(np.linalg.norm(r1, axis=1), 65.0)
    assert np.allclose(r1[:, 2], tr[:, 2])
    assert not np.allclose(r1, tr)
    assert np.allclose(shard.weak_replica_transducers(tr, 0, 2, 6), tr)
    # two half-steps make one full view step: rank-1 positions of view v rotated again land on view v+1
    r2 = shard.weak_replica_transducers(r1, 1, 2, 6)
    assert np.allclose(r2.reshape(4, 6, 3)[:, :-1], tr.reshape(4, 6, 3)[:, 1:], atol=1e-9)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from dataclasses import replace
    from oracle import oat_oracle as orc
    w = wl.small(n=10, q=5, nt=30, kband=8)
    x = w.phantom().astype(np.float64)
    y = w.data_noise().astype(np.float64)
    lo, hi = shard.shard_range(w.n_trans, rank, world)
    ws = replace(w, trans_xyz=shard.shard_transducers(w.trans_xyz, rank, world))
    hx_local = orc.project(ws, x)                                   # H: this rank's rows, no exchange
    part = torch.from_numpy(orc.backproject(ws, y[lo:hi], n_threads=1))
    shard.allreduce_volume(part)                                    # H^T: one all-reduce
    rows = torch.zeros((w.n_trans, w.nt), dtype=torch.float64)      # only to CHECK the rows (uneven shards: 3 + 2)
    rows[lo:hi] = torch.from_numpy(hx_local)
    dist.all_reduce(rows)
    # the same split serves the spherical-voxel pair (the paper's own multi-GPU case, Algs. 7-12): rows of H_sph are
    # per transducer, H_sph† sums over transducers
    from oracle import oat_sph as osph
    nf, f0, df = 7, 0.1, 0.3
    rng = np.random.default_rng(5)
    u = rng.standard_normal((w.n_trans, nf)) + 1j * rng.standard_normal((w.n_trans, nf))
    su_local = osph.project(ws, x, f0, df, nf)
    spart = torch.from_numpy(osph.backproject(ws, u[lo:hi], f0, df, nf))
    shard.allreduce_volume(spart)
    srows = torch.zeros((w.n_trans, nf, 2), dtype=torch.float64)
    srows[lo:hi] = torch.from_numpy(np.stack([su_local.real, su_local.imag], axis=-1))
    dist.all_reduce(srows)
    if rank == 0:
        full_su = osph.project(w, x, f0, df, nf)
        full_sx = osph.backproject(w, u, f0, df, nf)
        out["su"] = float(np.abs(srows.numpy()[..., 0] + 1j * srows.numpy()[..., 1] - full_su).max() / np.abs(full_su).max())
        out["sx"] = float(np.abs(spart.numpy() - full_sx).max() / np.abs(full_sx).max())
        full_hx = orc.project(w, x)
        full_xb = orc.backproject(w, y)
        out["hx"] = float(np.abs(rows.numpy() - full_hx).max() / np.abs(full_hx).max())
        out["xb"] = float(np.abs(part.numpy() - full_xb).max() / np.abs(full_xb).max())
    dist.destroy_process_group()


def test_two_rank_gloo_sharded_operators():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mgr = mp.Manager(); out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out["hx"] <= 1e-13 and out["xb"] <= 1e-12, dict(out)
    assert out["su"] <= 1e-13 and out["sx"] <= 1e-12, dict(out)
