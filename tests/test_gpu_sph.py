"""GPU parity tests of row NEXT-3 (spherical-voxel model H_sph, Eq. 17-19, and its adjoint, Eq. 24) through the C ABI
against the complex128 oracle oracle/oat_sph.py on the same seeded inputs.

Tolerance: distances and phase reduction are fp64 on the GPU; phasors come from sincospif and a 16-step fp32 complex
recurrence (error ~ 16 eps), amplitudes and sums are fp32: rel-L2 <= 2e-5 for H_sph and H_sph†, adjoint identity
Re<Hx,u> = <x,H†u> <= 1e-4."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oat_sph as osph
    from paper_1304_2017_b200 import binding as oat, build, workloads as wl
    build.build()
    assert torch.cuda.is_available()
    return torch, osph, oat, wl


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def run_pair(env, w, nf, f0, df, he=None, seed=0, sparse=False, aperture=0.0, m=1):
    torch, osph, oat, wl = env
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((w.nz, w.ny, w.nx)).astype(np.float32)
    if sparse:
        x[rng.random(x.shape) < 0.9] = 0.0
    u = (rng.standard_normal((w.n_trans, nf)) + 1j * rng.standard_normal((w.n_trans, nf))).astype(np.complex64)
    g = oat.oat_geometry_create(w)
    oat.oat_sph_set(g, nf, f0, df, he)
    if aperture:
        oat.oat_sph_set_aperture(g, aperture, m)
    hx = oat.oat_sph_project(g, torch.from_numpy(x).cuda()).cpu().numpy()
    htu = oat.oat_sph_backproject(g, torch.from_numpy(u).cuda()).cpu().numpy()
    g.close()
    he128 = None if he is None else np.asarray(he, dtype=np.complex64).astype(np.complex128)
    rx = osph.project(w, x.astype(np.float64), f0, df, nf, he128, aperture, m)
    ru = osph.backproject(w, u.astype(np.complex128), f0, df, nf, he128, aperture, m)
    e1, e2 = rel_l2(hx, rx), rel_l2(htu, ru)
    lhs = float(np.real(np.vdot(u.astype(np.complex128), hx.astype(np.complex128))))
    rhs = float(np.vdot(x.astype(np.float64), htu.astype(np.float64)))
    return e1, e2, abs(lhs - rhs) / max(abs(lhs), abs(rhs))


@pytest.mark.parametrize("n,q,nf,f0,df", [(9, 5, 40, 0.0, 0.05), (14, 3, 16, 0.4, 0.11), (7, 37, 23, 0.05, 0.02), (20, 4, 100, 0.0, 0.03)])
def test_small_problems(env, n, q, nf, f0, df):
    """Ragged frequency groups (nf not a multiple of 16), f0 = 0 (p~0(0) = 0), several voxel chunks (20^3 > 2048), more
    (transducer, group) pairs than one block."""
    torch, osph, oat, wl = env
    w = wl.small(n=n, q=q, nt=8, kband=8)
    e1, e2, adj = run_pair(env, w, nf, f0, df, seed=n + q)
    assert e1 <= TOL and e2 <= TOL and adj <= 1e-4, (e1, e2, adj)


def test_eir_spectrum_sparse_volume_and_non_cubic_grid(env):
    torch, osph, oat, wl = env
    tr = wl.fibonacci_sphere(6, 25.0) + np.array([0.2, -0.1, 0.3])
    w = wl.Workload("sph-nc", 11, 6, 17, 0.3, (-1.0, -2.0, -3.5), tr, c=1.5, t0=0.0, dt=0.05, nt=8, surf_step=0.3, kband=8, gain=0.7)
    nf = 48
    f = 0.1 + 0.07 * np.arange(nf)
    he = (np.exp(-((f - 2.0) / 1.5) ** 2) * np.exp(-2j * np.pi * f * 0.3)).astype(np.complex64)
    e1, e2, adj = run_pair(env, w, nf, 0.1, 0.07, he=he, seed=5, sparse=True)
    assert e1 <= TOL and e2 <= TOL and adj <= 1e-4, (e1, e2, adj)


def test_high_frequencies_and_long_distances(env):
    """Phases of ~1e3 cycles (f up to 20 MHz, d/c ~ 45 us): the case that needs the fp64 phase reduction."""
    torch, osph, oat, wl = env
    tr = wl.fibonacci_sphere(4, 65.0)
    w = wl.Workload("sph-hf", 10, 10, 10, 0.25, (-8.0, 3.0, -1.0), tr, c=1.5, t0=0.0, dt=0.05, nt=8, surf_step=0.25, kband=8)
    e1, e2, adj = run_pair(env, w, 64, 16.0, 0.0625, seed=9)
    assert e1 <= TOL and e2 <= TOL and adj <= 1e-4, (e1, e2, adj)


def test_errors_and_empty(env):
    torch, osph, oat, wl = env
    w = wl.small(n=6, q=2, nt=8, kband=8)
    g = oat.oat_geometry_create(w)
    x = torch.zeros((6, 6, 6), dtype=torch.float32, device="cuda")
    with pytest.raises(oat.OatError):
        oat.oat_sph_project(g, x)                          # no frequency grid
    oat.oat_sph_set(g, 8, 0.0, 0.1)
    assert torch.all(oat.oat_sph_project(g, x) == 0)       # zero volume -> zero data (all-zero chunks are skipped)
    with pytest.raises(oat.OatError):
        oat.oat_sph_set(g, 8, -1.0, 0.1)
    g.close()


@pytest.mark.parametrize("mu_rel", [0.0, 0.05])
def test_pls_sph_cg_first_iterations_match_the_oracle(env, mu_rel):
    """Eq. (30): 3 CG iterations on a small problem against the oracle's PLS-Sph loop; curves and iterate must match."""
    torch, osph, oat, wl = env
    from oracle import oat_pls as opls
    w = wl.small(n=10, q=6, nt=8, kband=8)
    nf, f0, df = 32, 0.05, 0.06
    rng = np.random.default_rng(12)
    xt = w.phantom().astype(np.float64)
    ut = osph.project(w, xt, f0, df, nf)
    u = (ut + 0.02 * np.abs(ut).max() * (rng.standard_normal(ut.shape) + 1j * rng.standard_normal(ut.shape))).astype(np.complex64)
    b = osph.backproject(w, u.astype(np.complex128), f0, df, nf)
    mu = mu_rel * float(np.linalg.norm(osph.backproject(w, osph.project(w, b, f0, df, nf), f0, df, nf)) / np.linalg.norm(opls.penalty_apply(b))) if mu_rel else 0.0
    g = oat.oat_geometry_create(w)
    oat.oat_sph_set(g, nf, f0, df)
    x, obj, grad = oat.oat_sph_pls_cg(g, torch.from_numpy(u).cuda(), 3, mu)
    g.close()
    xo, objo, grado = osph.pls_cg(w, u.astype(np.complex128), 3, mu, f0, df, nf)
    assert np.allclose(obj, objo, rtol=5e-4)
    assert np.allclose(grad, grado, rtol=3e-3)
    assert rel_l2(x.cpu().numpy(), xo) <= 1e-3
    assert np.all(np.diff(obj) < 0)


# ---------------------------------------------------------------- finite aperture (Eq. 18, reading G30)
@pytest.mark.parametrize("n,q,nf,aperture,m", [(9, 5, 40, 2.0, 2), (12, 3, 23, 2.0, 3), (7, 6, 16, 0.7, 4)])
def test_finite_aperture(env, n, q, nf, aperture, m):
    torch, osph, oat, wl = env
    w = wl.small(n=n, q=q, nt=8, kband=8)
    e1, e2, adj = run_pair(env, w, nf, 0.05, 0.07, seed=n * m, aperture=aperture, m=m)
    assert e1 <= TOL and e2 <= TOL and adj <= 1e-4, (e1, e2, adj)
    # the aperture changes the operator (the test would also pass for a kernel that ignored it otherwise)
    rng = np.random.default_rng(n * m)
    x = rng.standard_normal((w.nz, w.ny, w.nx)).astype(np.float32)
    g = oat.oat_geometry_create(w)
    oat.oat_sph_set(g, nf, 0.05, 0.07)
    a = oat.oat_sph_project(g, torch.from_numpy(x).cuda()).cpu().numpy()
    oat.oat_sph_set_aperture(g, aperture, m)
    b = oat.oat_sph_project(g, torch.from_numpy(x).cuda()).cpu().numpy()
    oat.oat_sph_set_aperture(g, 0.0, 1)
    c = oat.oat_sph_project(g, torch.from_numpy(x).cuda()).cpu().numpy()
    g.close()
    assert rel_l2(b, a) > 1e-3 and np.array_equal(a, c)


@pytest.mark.parametrize("aperture,m", [(0.0, 1), (2.0, 2)])
def test_bench_shape_sampled_rows_and_voxels(env, aperture, m):
    """The shape bench.py times (config 3's 240^3 grid, 256 seeded transducers, 64 frequencies), in full on the GPU;
    the oracle evaluates 2 sampled rows of H_sph x (dense N(0,1) volume) and 24 sampled voxels of H_sph† u."""
    torch, osph, oat, wl = env
    w = wl.config(3)
    _, ws = w.seeded_subset(256)
    nf, f0, df = 64, 0.0, 0.078125
    rng = np.random.default_rng(77)
    x = rng.standard_normal((ws.nz, ws.ny, ws.nx)).astype(np.float32)
    u = (rng.standard_normal((ws.n_trans, nf)) + 1j * rng.standard_normal((ws.n_trans, nf))).astype(np.complex64)
    g = oat.oat_geometry_create(ws)
    oat.oat_sph_set(g, nf, f0, df)
    oat.oat_sph_set_aperture(g, aperture, m)
    hx = oat.oat_sph_project(g, torch.from_numpy(x).cuda()).cpu().numpy()
    htu = oat.oat_sph_backproject(g, torch.from_numpy(u).cuda()).cpu().numpy()
    g.close()
    rows = [5, 200] if m == 1 else [131]
    ref_rows = osph.project_rows(ws, x.astype(np.float64), rows, f0, df, nf, None, aperture, m)
    idx = rng.integers(0, [ws.nz, ws.ny, ws.nx], size=(24, 3))
    pts = np.asarray(ws.origin)[None, :] + ws.spacing * idx[:, ::-1].astype(np.float64)
    ref_vox = osph.backproject_points(ws, u.astype(np.complex128), pts, f0, df, nf, None, aperture, m)
    e1 = rel_l2(hx[rows], ref_rows)
    e2 = rel_l2(htu[idx[:, 0], idx[:, 1], idx[:, 2]], ref_vox)
    print(f"H_sph at 240^3 x 256 x 64 (aperture {aperture} mm, m = {m}): rows {e1:.2e}, voxels {e2:.2e}")
    assert e1 <= 2 * TOL and e2 <= TOL, (e1, e2)
