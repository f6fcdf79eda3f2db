"""Pins of the NEXT-1 oracle (oracle/oat_pls.py: EIR operator, smoothness penalty, PLS-CG) against things other
than itself: numpy's library convolution, the impulse response, the graph Laplacian built edge by edge,
finite differences, closed forms, and a dense direct solve.  CPU only."""
import numpy as np
import pytest

from oracle import oat_oracle as orc
from oracle import oat_pls as pls
from paper_1304_2017_b200 import workloads as wl


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


# ---------------------------------------------------------------- H^e (Eq. 14) and H^e† (Eq. 21)
@pytest.mark.parametrize("K,L", [(64, 9), (50, 50), (16, 40), (7, 1)])
def test_eir_is_numpy_convolution_delayed_by_one_sample(K, L):
    """Eq. (14): u[k] = sum_kappa he[k-1-kappa] p[kappa] = (he * p)[k-1]: the library's full linear
    convolution shifted by the one-sample delay of the paper's index (reading G20), cut to K samples."""
    rng = np.random.default_rng(K * 100 + L)
    he, p = rng.standard_normal(L), rng.standard_normal((3, K))
    u = pls.eir_apply(he, p)
    for q in range(3):
        full = np.convolve(he, p[q])                     # full[n] = sum_m he[m] p[n-m]
        expect = np.concatenate([[0.0], full])[:K]       # u[k] = full[k-1], u[0] = 0
        assert np.allclose(u[q], expect, rtol=1e-13, atol=1e-13)


def test_eir_impulse_response_and_causality():
    he = np.array([0.5, -1.0, 0.25, 2.0])
    p = np.zeros((1, 12)); p[0, 3] = 1.0
    u = pls.eir_apply(he, p)[0]
    assert np.all(u[:4] == 0.0)                          # nothing before kappa0 + 1 (one-sample delay, G20)
    assert np.array_equal(u[4:8], he) and np.all(u[8:] == 0.0)


def test_eir_adjoint_identity_and_explicit_transpose():
    rng = np.random.default_rng(5)
    K, L = 40, 13
    he = rng.standard_normal(L)
    p, u = rng.standard_normal((4, K)), rng.standard_normal((4, K))
    lhs = np.vdot(pls.eir_apply(he, p), u); rhs = np.vdot(p, pls.eir_adjoint(he, u))
    assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), abs(rhs))
    # explicit K x K matrix of Eq. (14) from unit vectors; Eq. (21) must be its transpose, entry by entry
    T = np.stack([pls.eir_apply(he, np.eye(K)[k][None])[0] for k in range(K)], axis=1)
    Tt = np.stack([pls.eir_adjoint(he, np.eye(K)[k][None])[0] for k in range(K)], axis=1)
    assert np.array_equal(Tt, T.T)
    assert np.all(np.triu(T) == 0.0)                     # strictly lower triangular: causal with the delay
    assert np.allclose(np.diag(T, -1), he[0]) and np.allclose(np.diag(T, -3), he[2])


# ---------------------------------------------------------------- R (Eq. 34)
def laplacian_edge_by_edge(nz, ny, nx):
    """Graph Laplacian of the 6-neighbour grid: one pass over the edges (n, n-before) of Eq. (34)."""
    N = nz * ny * nx
    Lm = np.zeros((N, N))
    idx = lambda z, y, x: (z * ny + y) * nx + x
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                n = idx(z, y, x)
                for (dz, dy, dx) in ((0, 0, 1), (0, 1, 0), (1, 0, 0)):
                    zz, yy, xx = z - dz, y - dy, x - dx
                    if zz < 0 or yy < 0 or xx < 0:
                        continue                          # reading G21: no neighbour before -> term omitted
                    m = idx(zz, yy, xx)
                    Lm[n, n] += 1; Lm[m, m] += 1; Lm[n, m] -= 1; Lm[m, n] -= 1
    return Lm


def test_penalty_matches_the_graph_laplacian_and_is_psd():
    rng = np.random.default_rng(11)
    nz, ny, nx = 3, 4, 5
    x = rng.standard_normal((nz, ny, nx))
    Lm = laplacian_edge_by_edge(nz, ny, nx)
    assert np.allclose(pls.penalty_apply(x).ravel(), Lm @ x.ravel(), rtol=1e-13, atol=1e-13)
    assert abs(pls.penalty_value(x) - x.ravel() @ Lm @ x.ravel()) <= 1e-12 * pls.penalty_value(x)
    assert np.allclose(Lm, Lm.T) and np.linalg.eigvalsh(Lm).min() > -1e-12
    assert np.all(pls.penalty_apply(np.full((nz, ny, nx), 3.7)) == 0.0)      # constants are in the null space


def test_penalty_closed_forms_and_gradient():
    nz, ny, nx = 6, 5, 7
    a, b, c = 0.3, -1.1, 2.0
    zz, yy, xx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ramp = a * xx + b * yy + c * zz
    exact = a * a * (nx - 1) * ny * nz + b * b * nx * (ny - 1) * nz + c * c * nx * ny * (nz - 1)
    assert abs(pls.penalty_value(ramp) - exact) <= 1e-12 * exact
    # a single spike of height s has 6 (interior) differences of size s: once as "n" and once as "the neighbour before"
    spike = np.zeros((nz, ny, nx)); spike[2, 2, 3] = 1.5
    assert abs(pls.penalty_value(spike) - 6 * 1.5 ** 2) <= 1e-13
    corner = np.zeros((nz, ny, nx)); corner[0, 0, 0] = 1.0
    assert abs(pls.penalty_value(corner) - 3.0) <= 1e-13
    # grad R = 2 L x by central finite differences along a random direction
    rng = np.random.default_rng(2)
    x, d = rng.standard_normal((nz, ny, nx)), rng.standard_normal((nz, ny, nx))
    eps = 1e-6
    fd = (pls.penalty_value(x + eps * d) - pls.penalty_value(x - eps * d)) / (2 * eps)
    assert abs(fd - 2.0 * np.vdot(d, pls.penalty_apply(x))) <= 1e-7 * abs(fd)


# ---------------------------------------------------------------- PLS-CG (Eq. 29)
@pytest.fixture(scope="module")
def tiny_full():
    tr = np.array([[6.0, 1.0, 2.0], [-1.5, -5.0, 4.0], [0.5, 5.5, -3.0]])
    w = wl.Workload("tiny", 5, 4, 3, 0.5, (-1.0, -0.75, -0.5), tr, c=1.5, t0=2.6, dt=0.1, nt=22,
                    surf_step=0.4, kband=4, gain=1.0)
    he = np.array([0.2, 0.7, -0.4, 0.1])
    N = w.n_voxels
    # dense H = H^e D G column by column (D G is pinned by P5 in test_oracle_pins.py, H^e above)
    M = np.stack([pls.project_full(w, np.eye(N)[n].reshape(w.nz, w.ny, w.nx), he).ravel() for n in range(N)], axis=1)
    return w, he, M


def test_full_operator_adjoint_identity(tiny_full):
    w, he, M = tiny_full
    rng = np.random.default_rng(21)
    x, u = rng.random((w.nz, w.ny, w.nx)), rng.standard_normal((w.n_trans, w.nt))
    lhs = np.vdot(pls.project_full(w, x, he), u); rhs = np.vdot(x, pls.backproject_full(w, u, he))
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))
    assert np.allclose(pls.backproject_full(w, u, he).ravel(), M.T @ u.ravel(), rtol=1e-11, atol=1e-13)


def test_pls_cg_matches_textbook_cg_and_the_direct_solve(tiny_full):
    w, he, M = tiny_full
    rng = np.random.default_rng(8)
    xt = rng.random(w.n_voxels)
    u = (M @ xt + 0.01 * rng.standard_normal(M.shape[0])).reshape(w.n_trans, w.nt)
    mu = 0.05 * np.linalg.norm(M, 2) ** 2
    Lm = laplacian_edge_by_edge(w.nz, w.ny, w.nx)
    A = M.T @ M + mu * Lm; b = M.T @ u.ravel()
    # textbook CG (Shewchuk) on the dense system
    xc = np.zeros_like(b); r = b.copy(); p = r.copy(); xs = []
    for _ in range(10):
        Ap = A @ p; al = (r @ r) / (p @ Ap); xc = xc + al * p
        rn = r - al * Ap; be = (rn @ rn) / (r @ r); p = rn + be * p; r = rn
        xs.append(xc.copy())
    x3, obj3, grad3 = pls.pls_cg(w, u, 3, mu, he)
    assert np.allclose(x3.ravel(), xs[2], rtol=1e-8, atol=1e-10)
    x10, obj, grad = pls.pls_cg(w, u, 10, mu, he)
    assert np.allclose(x10.ravel(), xs[9], rtol=1e-6, atol=1e-9)
    # the objective of Eq. (29) is evaluated honestly and decreases monotonically (CG minimises it over Krylov spaces)
    phi = lambda x: np.sum((u.ravel() - M @ x) ** 2) + mu * x @ Lm @ x
    assert abs(obj[0] - phi(np.zeros_like(b))) <= 1e-12 * obj[0]
    assert abs(obj[10] - phi(xs[9])) <= 1e-9 * obj[10]
    assert np.all(np.diff(obj) <= 1e-12 * obj[0])
    # converges to the unique minimiser of Eq. (29): (M^T M + mu L) x = M^T u
    xd = np.linalg.solve(A, b)
    x60, obj60, grad60 = pls.pls_cg(w, u, 60, mu, he)
    assert np.linalg.norm(x60.ravel() - xd) <= 1e-7 * np.linalg.norm(xd)
    assert grad60[-1] <= 1e-8 * grad60[0]


def test_pls_cg_without_eir_and_penalty_is_cg_on_the_normal_equations(tiny_full):
    """mu = 0, no EIR: the iterates equal those of the CGLS oracle of row C1 (same Krylov spaces)."""
    w, _, _ = tiny_full
    rng = np.random.default_rng(3)
    y = rng.standard_normal((w.n_trans, w.nt))
    xa, _, _ = pls.pls_cg(w, y, 4, 0.0, None)
    xb, _, _ = orc.cgls(w, y, 4)
    assert rel_l2(xa, xb) <= 1e-9
