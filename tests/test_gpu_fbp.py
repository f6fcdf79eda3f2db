"""GPU parity tests of row NEXT-2 (filtered backprojection, Eq. 27) through the C ABI against the fp64 oracle
oracle/oat_fbp.py on the same seeded inputs.

Tolerance: the integer decision k = floor(k~) is taken in fp64 on both sides; the brackets, the interpolation and the
sum over transducers are fp32 (chunk sums of 256 terms, fp64 total): rel-L2 <= 2e-5."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oat_fbp as ofbp, oat_oracle as orc
    from paper_1304_2017_b200 import binding as oat, build, workloads as wl
    build.build()
    assert torch.cuda.is_available()
    return torch, ofbp, orc, oat, wl


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def gpu_fbp(torch, oat, w, p, wq):
    g = oat.oat_geometry_create(w)
    x = oat.oat_fbp(g, torch.from_numpy(np.ascontiguousarray(p, dtype=np.float32)).cuda(),
                    torch.from_numpy(np.ascontiguousarray(wq, dtype=np.float32)).cuda())
    torch.cuda.synchronize()
    out = x.cpu().numpy()
    g.close()
    return out


@pytest.mark.parametrize("n,q,nt", [(13, 7, 200), (8, 300, 160), (21, 64, 333)])
def test_small_problems_random_data(env, n, q, nt):
    """Noise data (the hardest case for the interval decision), ragged tiles (n not a multiple of 8 / 4), more
    transducers than one shared-memory chunk (q = 300 > 256)."""
    torch, ofbp, orc, oat, wl = env
    w = wl.small(n=n, q=q, nt=nt, kband=32)
    rng = np.random.default_rng(n * q)
    p = rng.standard_normal((q, nt)).astype(np.float32)
    wq = rng.standard_normal(q).astype(np.float32)
    got = gpu_fbp(torch, oat, w, p, wq)
    ref = ofbp.fbp(w, p.astype(np.float64), wq.astype(np.float64))
    assert np.count_nonzero(ref) > 0.5 * ref.size
    # nodes where some k~ is an integer to rounding (the grid centre is equidistant from the whole Fibonacci sphere) are
    # ties between two correct intervals of the discontinuous Eq. (27): compare what is unique
    uniq = (ofbp.interval_margin(w, ofbp.node_positions(w).reshape(-1, 3)) > 1e-9).reshape(ref.shape)
    assert uniq.sum() >= ref.size - 8
    assert rel_l2(got[uniq], ref[uniq]) <= TOL


def test_non_cubic_grid_record_edges_and_degenerate_sizes(env):
    torch, ofbp, orc, oat, wl = env
    tr = wl.fibonacci_sphere(9, 14.0)
    w = wl.Workload("fbp-nc", 11, 6, 17, 0.4, (-1.0, -2.0, -3.5), tr[:3], c=1.5, t0=7.9, dt=0.05, nt=30, surf_step=0.4, kband=32)
    rng = np.random.default_rng(2)
    p = rng.standard_normal((3, 30)).astype(np.float32)            # the record covers only part of the grid (reading G25)
    wq = np.linspace(-1.0, 2.0, 3).astype(np.float32)
    ref = ofbp.fbp(w, p.astype(np.float64), wq.astype(np.float64))
    assert 0 < np.count_nonzero(ref) < ref.size
    got = gpu_fbp(torch, oat, w, p, wq)
    uniq = (ofbp.interval_margin(w, ofbp.node_positions(w).reshape(-1, 3)) > 1e-9).reshape(ref.shape)
    assert rel_l2(got[uniq], ref[uniq]) <= TOL
    assert np.all(got[(ref == 0.0) & uniq] == 0.0)
    # K = 1: no pair has both k and k+1 inside the record
    w1 = wl.Workload("fbp-k1", 5, 5, 5, 0.4, (-1.0, -1.0, -1.0), tr, c=1.5, t0=9.0, dt=0.05, nt=1, surf_step=0.4, kband=32)
    assert np.all(gpu_fbp(torch, oat, w1, np.ones((9, 1), np.float32), np.ones(9, np.float32)) == 0.0)


def test_transducer_on_a_grid_node(env):
    """Reading G25: a voxel that coincides with a transducer gets no term from that transducer (and no NaN)."""
    torch, ofbp, orc, oat, wl = env
    tr = np.array([[0.5, -0.5, 1.0], [9.0, 2.0, -3.0], [-7.0, 6.0, 4.0]])          # the first one sits on node (5, 3, 6)
    w = wl.Workload("fbp-on-node", 9, 9, 9, 0.5, (-2.0, -2.0, -2.0), tr, c=1.5, t0=0.0, dt=0.05, nt=300, surf_step=0.5, kband=32)
    assert np.allclose(ofbp.node_positions(w)[6, 3, 5], tr[0])
    rng = np.random.default_rng(3)
    p = rng.standard_normal((3, 300)).astype(np.float32)
    wq = np.array([1.0, -0.5, 2.0], dtype=np.float32)
    got = gpu_fbp(torch, oat, w, p, wq)
    ref = ofbp.fbp(w, p.astype(np.float64), wq.astype(np.float64))
    assert np.all(np.isfinite(got))
    uniq = (ofbp.interval_margin(w, ofbp.node_positions(w).reshape(-1, 3)) > 1e-9).reshape(ref.shape)
    uniq[6, 3, 5] = True                                    # the node on the transducer is compared too
    assert rel_l2(got[uniq], ref[uniq]) <= TOL
    assert abs(got[6, 3, 5] - ref[6, 3, 5]) <= TOL * np.abs(ref).max()


def test_config1_fbp_of_projected_phantom(env):
    """Config 1 end to end: p = H x from the library, FBP with the Fibonacci patch weights, against the oracle's
    FBP of the same p; and the image correlates with the phantom (limited by the 64-transducer aperture)."""
    torch, ofbp, orc, oat, wl = env
    w = wl.config(1)
    x = w.phantom()
    g = oat.oat_geometry_create(w)
    pd = oat.oat_project(g, torch.from_numpy(x).cuda())
    areas = wl.patch_areas_equal(w.trans_xyz, w.centre)
    wq = oat.oat_fbp_weights(g, areas)                      # the library's weights of Eq. (27) ...
    wq_ref = ofbp.weights(w, areas)                         # ... against the oracle's, computed independently
    assert np.allclose(wq, wq_ref, rtol=2e-7)
    img = oat.oat_fbp(g, pd, torch.from_numpy(wq).cuda()).cpu().numpy()
    p = pd.cpu().numpy()
    g.close()
    ref = ofbp.fbp(w, p.astype(np.float64), wq_ref)
    uniq = (ofbp.interval_margin(w, ofbp.node_positions(w).reshape(-1, 3)) > 1e-9).reshape(ref.shape)
    assert uniq.sum() >= ref.size - 8
    assert rel_l2(img[uniq], ref[uniq]) <= TOL
    c = np.corrcoef(img.ravel(), x.ravel())[0, 1]
    assert c > 0.5, c


@pytest.mark.parametrize("cfg", [3, 5])
def test_fullsize_sampled_voxels(env, cfg):
    """Full configs 3 and 5 in the launch configuration bench.py times: the whole image on the GPU, the oracle on 48
    seeded nodes (Eq. 27 voxel by voxel); smooth band-limited data so that the record is realistic."""
    torch, ofbp, orc, oat, wl = env
    w = wl.config(cfg)
    rng = np.random.default_rng(cfg)
    t = np.arange(w.nt)
    ph = rng.uniform(0, 2 * np.pi, size=(w.n_trans, 1)); f = rng.uniform(0.01, 0.05, size=(w.n_trans, 1))
    p = (np.sin(2 * np.pi * f * t[None, :] + ph) * np.exp(-((t[None, :] - w.nt / 2) / (0.3 * w.nt)) ** 2)).astype(np.float32)
    areas = wl.patch_areas_arc(64, 144, 65.0) if cfg == 3 else wl.patch_areas_equal(w.trans_xyz, w.centre)
    g = oat.oat_geometry_create(w)
    wq = oat.oat_fbp_weights(g, areas)
    g.close()
    assert np.allclose(wq, ofbp.weights(w, areas), rtol=2e-7)
    got = gpu_fbp(torch, oat, w, p, wq)
    idx = rng.integers(0, [w.nz, w.ny, w.nx], size=(48, 3))
    idx[0] = (0, 0, 0); idx[1] = (w.nz - 1, w.ny - 1, w.nx - 1)
    o = np.asarray(w.origin)
    pts = o[None, :] + w.spacing * idx[:, ::-1].astype(np.float64)
    ref = ofbp.fbp_points(w, p.astype(np.float64), wq.astype(np.float64), pts)
    val = got[idx[:, 0], idx[:, 1], idx[:, 2]]
    uniq = ofbp.interval_margin(w, pts) > 1e-9
    assert np.linalg.norm(ref) > 0 and uniq.sum() >= 40
    assert rel_l2(val[uniq], ref[uniq]) <= TOL
