"""GPU parity tests of row NEXT-1 (EIR operator, smoothness penalty, PLS-CG) through the C ABI against the
fp64 oracle oracle/oat_pls.py on the same seeded inputs.

Tolerances: the EIR is an L-term fp32 FMA chain per output (error ~ eps sqrt(L)), the penalty a 6-term stencil:
rel-L2 <= 1e-5 for both; adjoint identities <= 1e-5; H^e D G and its transpose inherit the 1e-4 of H / H^T;
PLS-CG curves like the CGLS test of row C1."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oat_oracle as orc, oat_pls as pls
    from paper_1304_2017_b200 import binding as oat, build, workloads as wl
    build.build()
    assert torch.cuda.is_available()
    return torch, orc, pls, oat, wl


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def eir_taps(n, dt, seed=0):
    """A damped band-pass pulse, the shape of a measured transducer EIR (the paper's own is not printed)."""
    t = np.arange(n) * dt
    return (dt * np.exp(-t / (0.15 * n * dt)) * np.sin(2 * np.pi * 2.5 * t + 0.3 * seed)).astype(np.float32)


@pytest.mark.parametrize("K,L,Q", [(300, 37, 5), (256, 256, 3), (1000, 300, 2), (40, 64, 4), (513, 1, 2), (40, 5, 70000)])
def test_eir_forward_and_adjoint_match_the_oracle(env, K, L, Q):
    """Eq. (14) / Eq. (21) on ragged tiles (K not a multiple of the 256-output tile), L > K, L = 1, and more transducers
    than a grid's y dimension can hold (Q = 70 000 > 65 535: the rows are on grid.x)."""
    torch, orc, pls, oat, wl = env
    w = wl.small(n=8, q=Q, nt=K, kband=32)
    rng = np.random.default_rng(K + L)
    he = rng.standard_normal(L).astype(np.float32)
    p = rng.standard_normal((Q, K)).astype(np.float32)
    g = oat.oat_geometry_create(w)
    oat.oat_eir_set(g, he)
    pd = torch.from_numpy(p).cuda()
    u = oat.oat_eir_apply(g, pd).cpu().numpy()
    ut = oat.oat_eir_apply(g, pd, adjoint=True).cpu().numpy()
    g.close()
    assert rel_l2(u, pls.eir_apply(he.astype(np.float64), p)) <= 1e-5
    assert rel_l2(ut, pls.eir_adjoint(he.astype(np.float64), p)) <= 1e-5
    assert np.all(u[:, 0] == 0.0)                        # one-sample delay of Eq. (14) (reading G20)
    lhs = np.vdot(u.astype(np.float64), p); rhs = np.vdot(p.astype(np.float64), ut)   # <H^e p, p> = <p, H^e† p>
    assert abs(lhs - rhs) <= 1e-5 * max(abs(lhs), abs(rhs), 1e-30)


def test_eir_requires_taps_and_distinct_buffers(env):
    torch, orc, pls, oat, wl = env
    w = wl.small(n=8, q=2, nt=64, kband=32)
    g = oat.oat_geometry_create(w)
    p = torch.zeros((2, 64), dtype=torch.float32, device="cuda")
    with pytest.raises(oat.OatError):
        oat.oat_eir_apply(g, p)                          # no taps set
    oat.oat_eir_set(g, np.ones(3, dtype=np.float32))
    with pytest.raises(oat.OatError):
        oat.oat_eir_apply(g, p, out=p)                   # in place
    oat.oat_eir_set(g, np.zeros(0, dtype=np.float32))    # removes the EIR again
    with pytest.raises(oat.OatError):
        oat.oat_eir_apply(g, p)
    g.close()


@pytest.mark.parametrize("shape", [(7, 5, 9), (1, 1, 6), (33, 40, 17)])
def test_penalty_matches_the_oracle(env, shape):
    torch, orc, pls, oat, wl = env
    nz, ny, nx = shape
    w = wl.Workload("pen", nx, ny, nz, 0.5, (-1.0, -1.0, -1.0), np.array([[30.0, 1.0, 2.0]]), c=1.5, t0=1.0, dt=0.1, nt=8,
                    surf_step=0.5, kband=8)
    rng = np.random.default_rng(nx * 100 + nz)
    x = rng.standard_normal(shape).astype(np.float32)
    g = oat.oat_geometry_create(w)
    xd = torch.from_numpy(x).cuda()
    lx = oat.oat_penalty_apply(g, xd).cpu().numpy()
    r = oat.oat_penalty_value(g, xd)
    g.close()
    assert rel_l2(lx, pls.penalty_apply(x.astype(np.float64))) <= 1e-5
    ref = pls.penalty_value(x.astype(np.float64))
    assert abs(r - ref) <= 1e-5 * ref
    assert abs(np.vdot(x.astype(np.float64), lx) - ref) <= 1e-5 * ref      # R(x) = x^T L x


def test_full_operator_with_eir_matches_the_oracle(env):
    """u = H^e D G x and x = G^T D^T H^e† u on config 1 against the oracle, and their adjoint identity."""
    torch, orc, pls, oat, wl = env
    w = wl.config(1)
    he = eir_taps(48, w.dt)
    x, u = w.phantom(), w.data_noise()
    g = oat.oat_geometry_create(w)
    oat.oat_eir_set(g, he)
    xd, ud = torch.from_numpy(x).cuda(), torch.from_numpy(u).cuda()
    hx = oat.oat_project_eir(g, xd).cpu().numpy()
    htu = oat.oat_backproject_eir(g, ud).cpu().numpy()
    g.close()
    he64 = he.astype(np.float64)
    assert rel_l2(hx, pls.project_full(w, x.astype(np.float64), he64)) <= 1e-4
    assert rel_l2(htu, pls.backproject_full(w, u.astype(np.float64), he64)) <= 1e-4
    lhs = np.vdot(hx.astype(np.float64), u); rhs = np.vdot(x.astype(np.float64), htu)
    assert abs(lhs - rhs) <= 1e-4 * max(abs(lhs), abs(rhs))


@pytest.mark.parametrize("with_eir,mu_rel", [(True, 0.05), (False, 0.0), (True, 0.0)])
def test_pls_cg_first_iterations_match_the_oracle(env, with_eir, mu_rel):
    """Eq. (29): first 3 CG iterations on a config-2-shaped problem (6 transducers so the oracle finishes in
    seconds) against the oracle's PLS-CG; objective and gradient curves must match and the objective decrease."""
    torch, orc, pls, oat, wl = env
    w = wl.config(4)
    _, ws = w.seeded_subset(6)
    he = eir_taps(40, ws.dt) * 20.0 if with_eir else None
    he64 = None if he is None else he.astype(np.float64)
    xt = w.phantom()
    utrue = pls.project_full(ws, xt.astype(np.float64), he64)
    rng = np.random.default_rng(4)
    u = (utrue + rng.standard_normal(utrue.shape) * 0.05 * np.abs(utrue).max()).astype(np.float32)
    # scale mu to the operator: mu_rel * ||H^T u|| / ||L H^T u|| makes the penalty term comparable to H^T H
    b = pls.backproject_full(ws, u.astype(np.float64), he64)
    mu = mu_rel * float(np.linalg.norm(pls.backproject_full(ws, pls.project_full(ws, b, he64), he64)) / np.linalg.norm(pls.penalty_apply(b))) if mu_rel else 0.0
    g = oat.oat_geometry_create(ws)
    if with_eir:
        oat.oat_eir_set(g, he)
    x, obj, grad = oat.oat_pls_cg(g, torch.from_numpy(u).cuda(), 3, mu)
    g.close()
    xo, objo, grado = pls.pls_cg(ws, u.astype(np.float64), 3, mu, he64)
    assert np.allclose(obj, objo, rtol=5e-4)
    assert np.allclose(grad, grado, rtol=3e-3)
    assert rel_l2(x.cpu().numpy(), xo) <= 1e-3
    assert np.all(np.diff(obj) < 0)
