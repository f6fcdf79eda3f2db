"""Full-size parity: BASELINE.json configs 3 and 5 in the launch configuration bench.py times (the
complete transducer set on the GPU), checked on sampled outputs the oracle can compute one by one.

  H   : the GPU projects with ALL Q transducers; the rows of a seeded subset are compared with the
        oracle run on that subset (rows of H are independent of each other).
  H^T : y is non-zero only in the subset's rows on BOTH sides; exact, because H^T is a sum over
        transducers.  The GPU still runs its full-size geometry and launch.
Tolerance: rel-L2 <= 1e-4 (north_star).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
TOL = 1e-4


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.mark.parametrize("cfg,nsub", [(3, 8), (5, 4)])
def test_fullsize_sampled_rows(cfg, nsub):
    import torch
    from oracle import oat_oracle as orc
    from paper_1304_2017_b200 import binding as oat, build, workloads as wl
    build.build()
    w = wl.config(cfg)
    idx, ws = w.seeded_subset(nsub)
    x = w.phantom()
    g = oat.oat_geometry_create(w)
    xd = torch.from_numpy(x).cuda()
    y = oat.oat_project(g, xd)
    torch.cuda.synchronize()
    y_rows = y[torch.from_numpy(idx).cuda()].cpu().numpy()
    ref_rows = orc.project(ws, x.astype(np.float64))
    e_h = rel_l2(y_rows, ref_rows)
    # H^T with data only in the sampled rows
    rng = np.random.default_rng(cfg + 500)
    ysub = rng.standard_normal((nsub, w.nt)).astype(np.float32)
    yfull = torch.zeros((w.n_trans, w.nt), dtype=torch.float32, device="cuda")
    yfull[torch.from_numpy(idx).cuda()] = torch.from_numpy(ysub).cuda()
    xb = oat.oat_backproject(g, yfull)
    torch.cuda.synchronize()
    ref_xb = orc.backproject(ws, ysub.astype(np.float64))
    e_t = rel_l2(xb.cpu().numpy(), ref_xb)
    # adjoint identity at full size (properties that hold at any size)
    yn = torch.from_numpy(rng.standard_normal((w.n_trans, w.nt)).astype(np.float32)).cuda() if cfg == 3 else yfull
    lhs, rhs, rel = oat.oat_adjoint_check(g, xd, yn)
    print(f"config {cfg}: H rows {e_h:.2e}, H^T {e_t:.2e}, adjoint {rel:.2e}, samples/op {oat.oat_num_surface_samples(g):.4g}")
    g.close()
    assert e_h <= TOL and e_t <= TOL and rel <= TOL
