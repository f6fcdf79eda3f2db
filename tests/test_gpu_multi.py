"""Row NEXT-4 / SURVEY.md section 8(e) on the CUDA operators: transducers (rows of H) are sharded, H needs no exchange, H^T's
partial volumes are summed.

  * test_shards_on_one_device: the strong split executed shard after shard on cuda:0 (no collective): rows of H of every
    shard equal the rows of the unsharded operator, the partial volumes of H^T add up to the unsharded H^T y; same for
    the spherical-voxel pair.  Runs on one GPU.
  * test_two_ranks_nccl: two processes, one GPU each, NCCL all-reduce of the partial volumes (paper_1304_2017_b200.shard),
    against the single-GPU result.  Skipped unless two CUDA devices are visible.
"""
import os
import socket
from dataclasses import replace

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)                   # real volumes / data or complex spectra
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_shards_on_one_device():
    import torch
    from paper_1304_2017_b200 import binding as oat, build, shard, workloads as wl
    build.build()
    w = wl.small(n=20, q=11, nt=96, kband=32, h=0.25)
    x = torch.from_numpy(w.phantom()).cuda()
    y = torch.from_numpy(w.data_noise()).cuda()
    g = oat.oat_geometry_create(w)
    hx = oat.oat_project(g, x).clone()
    hty = oat.oat_backproject(g, y).clone()
    nf = 24
    oat.oat_sph_set(g, nf, 0.05, 0.09)
    rng = np.random.default_rng(3)
    u = torch.from_numpy((rng.standard_normal((w.n_trans, nf)) + 1j * rng.standard_normal((w.n_trans, nf))).astype(np.complex64)).cuda()
    sx = oat.oat_sph_project(g, x).clone()
    stu = oat.oat_sph_backproject(g, u).clone()
    g.close()
    for world in (2, 3):
        part = torch.zeros_like(hty); spart = torch.zeros_like(stu)
        for rank in range(world):
            lo, hi = shard.shard_range(w.n_trans, rank, world)
            ws = replace(w, trans_xyz=shard.shard_transducers(w.trans_xyz, rank, world))
            gs = oat.oat_geometry_create(ws)
            rows = oat.oat_project(gs, x)
            assert rel_l2(rows.cpu().numpy(), hx[lo:hi].cpu().numpy()) <= 1e-6       # H: this rank's rows, no exchange
            part += oat.oat_backproject(gs, y[lo:hi].contiguous())                   # H^T: partial volume
            oat.oat_sph_set(gs, nf, 0.05, 0.09)
            assert rel_l2(oat.oat_sph_project(gs, x).cpu().numpy(), sx[lo:hi].cpu().numpy()) <= 1e-6
            spart += oat.oat_sph_backproject(gs, u[lo:hi].contiguous())
            gs.close()
        assert rel_l2(part.cpu().numpy(), hty.cpu().numpy()) <= 2e-6
        assert rel_l2(spart.cpu().numpy(), stu.cpu().numpy()) <= 2e-6


def _rank_main(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    from paper_1304_2017_b200 import binding as oat, shard, workloads as wl
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ.setdefault("NCCL_DEBUG", "INFO")                 # the communicator log shows both ranks
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = wl.small(n=20, q=11, nt=96, kband=32, h=0.25)
    lo, hi = shard.shard_range(w.n_trans, rank, world)
    ws = replace(w, trans_xyz=shard.shard_transducers(w.trans_xyz, rank, world))
    g = oat.oat_geometry_create(ws, rank)                        # a second device in the same test session
    x = torch.from_numpy(w.phantom()).cuda()
    y = torch.from_numpy(w.data_noise()[lo:hi].copy()).cuda()
    rows = oat.oat_project(g, x)
    part = oat.oat_backproject(g, y)
    shard.allreduce_volume(part)                                 # the path's one exchange step
    torch.cuda.synchronize()
    np.save(os.path.join(out_dir, f"rows{rank}.npy"), rows.cpu().numpy())
    if rank == 0:
        np.save(os.path.join(out_dir, "hty.npy"), part.cpu().numpy())
    g.close()
    dist.destroy_process_group()


def test_two_ranks_nccl(tmp_path):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip(f"needs 2 CUDA devices for the NCCL path, {torch.cuda.device_count()} visible (this pool leases 1 GPU)")
    import torch.multiprocessing as mp
    from paper_1304_2017_b200 import binding as oat, build, shard, workloads as wl
    build.build()
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mp.spawn(_rank_main, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    w = wl.small(n=20, q=11, nt=96, kband=32, h=0.25)
    g = oat.oat_geometry_create(w)
    hx = oat.oat_project(g, torch.from_numpy(w.phantom()).cuda()).cpu().numpy()
    hty = oat.oat_backproject(g, torch.from_numpy(w.data_noise()).cuda()).cpu().numpy()
    g.close()
    rows = np.concatenate([np.load(tmp_path / "rows0.npy"), np.load(tmp_path / "rows1.npy")])
    assert rel_l2(rows, hx) <= 1e-6
    assert rel_l2(np.load(tmp_path / "hty.npy"), hty) <= 2e-6
