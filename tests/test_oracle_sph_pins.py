"""Pins of the NEXT-3 oracle (oracle/oat_sph.py: spherical-voxel model H_sph, Eq. 17-19, and its adjoint, Eq. 24)
against things other than itself: the time-domain N-wave of a uniform sphere (closed form from Eq. 2-3) recovered by
an inverse Fourier sum, the small-f series of Eq. (19), and the adjoint identity.  CPU only."""
import math

import numpy as np

from oracle import oat_sph as sph
from paper_1304_2017_b200 import workloads as wl


def problem(n=3, ds=0.5, q=3, rs=20.0, kappa=1.0):
    tr = wl.fibonacci_sphere(max(q, 2), rs)[:q] + np.array([0.3, -0.2, 0.1])
    o = -(n - 1) * ds / 2.0
    return wl.Workload("sph-pin", n, n, n, ds, (o, o, o), tr, c=1.5, t0=0.0, dt=0.05, nt=8, surf_step=ds, kband=8, gain=kappa)


def test_single_voxel_is_the_n_wave_of_a_uniform_sphere():
    """One spherical voxel of radius ds/2 and unit amplitude: the inverse Fourier sum of Eq. (17) over a dense frequency
    grid must give p(t) = kappa (-2 pi c^2 (ct - d)/d) for |ct - d| < ds/2 and 0 outside (Eq. 2-3 L59-63 for a ball; pin
    P6 of the interpolation model).  Pins Eq. (19) -- sign, the factor 4 pi kappa = beta/C_p, cos/sin terms -- and the
    Green's function exp(-j 2 pi f d/c)/(2 pi d) of Eq. (18)."""
    w = problem(kappa=1.7)
    x = np.zeros((w.nz, w.ny, w.nx)); x[1, 2, 0] = 1.0
    node = np.asarray(w.origin) + w.spacing * np.array([0, 2, 1])
    df, nf = 0.02, 10000                                  # 0 .. 200 MHz, period 50 us > d/c + a/c
    f = sph.freqs(0.0, df, nf)
    u = sph.project(w, x, 0.0, df, nf)
    a = w.spacing / 2.0
    taper = 0.5 * (1.0 + np.cos(np.pi * f / f[-1]))       # smooths p(t) over ~0.01 us; a linear ramp is unchanged by it
    for q in range(w.n_trans):
        d = np.linalg.norm(w.trans_xyz[q] - node)
        s = np.array([-0.6, -0.3, 0.0, 0.25, 0.55]) * a    # ct - d, inside the N-wave
        t = (d + s) / w.c
        pt = 2.0 * df * np.real(np.exp(2j * np.pi * np.outer(t, f)) @ (u[q] * taper))   # real signal, P(0) = 0
        exact = w.gain * (-2.0 * math.pi * w.c ** 2 * s / d)
        assert np.allclose(pt, exact, rtol=2e-3, atol=2e-3 * abs(exact).max()), (q, pt, exact)
        t_out = (d + np.array([-2.5, 1.8, 4.0]) * a) / w.c
        p_out = 2.0 * df * np.real(np.exp(2j * np.pi * np.outer(t_out, f)) @ (u[q] * taper))
        assert np.all(np.abs(p_out) < 5e-3 * abs(exact).max())


def test_p0_small_frequency_series_and_dc():
    """Eq. (19) near f = 0: bracket = (x cos x - sin x)/omega ~ -omega^2 T^3/3, T = ds/2c  =>  p~0 ~ +j (16 pi^3/3) kappa c^3 T^3 f."""
    w = problem(kappa=0.8)
    T = w.spacing / (2.0 * w.c)
    f = np.array([0.0, 1e-3, 2e-3])
    p0 = sph.p0_tilde(w, f)
    assert p0[0] == 0.0
    lead = 1j * (16.0 * math.pi ** 3 / 3.0) * w.gain * w.c ** 3 * T ** 3 * f[1:]
    assert np.allclose(p0[1:], lead, rtol=1e-4)
    assert np.all(np.abs(p0.real) < 1e-12 * np.abs(p0.imag).max())          # purely imaginary without an EIR
    he = np.array([1.0, 2.0 - 1.0j, 0.5j])
    assert np.allclose(sph.p0_tilde(w, f, he), p0 * he)


def test_adjoint_identity_and_linearity():
    w = problem(n=4, q=5)
    rng = np.random.default_rng(0)
    f0, df, nf = 0.3, 0.17, 23
    x = rng.standard_normal((w.nz, w.ny, w.nx))
    u = rng.standard_normal((w.n_trans, nf)) + 1j * rng.standard_normal((w.n_trans, nf))
    he = rng.standard_normal(nf) + 1j * rng.standard_normal(nf)
    hx = sph.project(w, x, f0, df, nf, he)
    htu = sph.backproject(w, u, f0, df, nf, he)
    lhs = np.real(np.vdot(u, hx))                          # Re <u, Hx> = Re sum conj(u) Hx
    rhs = np.vdot(x, htu)
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))
    x2 = rng.standard_normal(x.shape)
    assert np.allclose(sph.project(w, 2 * x - 3 * x2, f0, df, nf, he), 2 * hx - 3 * sph.project(w, x2, f0, df, nf, he), rtol=1e-12, atol=1e-14)
    # dense matrix column: one voxel, one transducer, written out from Eq. (17)-(18)
    e = np.zeros_like(x); e[2, 1, 3] = 1.0
    node = np.asarray(w.origin) + w.spacing * np.array([3, 1, 2])
    d = np.linalg.norm(w.trans_xyz[4] - node)
    fl = f0 + df * 7
    col = sph.project(w, e, f0, df, nf, he)[4, 7]
    assert np.allclose(col, sph.p0_tilde(w, np.array([fl]))[0] * he[7] * np.exp(-2j * np.pi * fl * d / w.c) / (2 * np.pi * d), rtol=1e-12)


def laplacian_edge_by_edge(nz, ny, nx):
    """Graph Laplacian of the 6-neighbour grid, one pass over the edges (n, n-before) of Eq. (34) (reading G21)."""
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
                        continue
                    m = idx(zz, yy, xx)
                    Lm[n, n] += 1; Lm[m, m] += 1; Lm[n, m] -= 1; Lm[m, n] -= 1
    return Lm


def test_pls_sph_cg_matches_the_dense_real_system():
    """Eq. (30): stack real and imaginary parts of the dense H_sph (built column by column) into a real matrix M; the CG
    iterates must equal textbook CG on (M^T M + mu L) x = M^T u_stacked and converge to numpy.linalg.solve."""
    w = problem(n=3, q=4)
    f0, df, nf = 0.2, 0.35, 9
    N = w.n_voxels
    Hc = np.stack([sph.project(w, np.eye(N)[n].reshape(w.nz, w.ny, w.nx), f0, df, nf).ravel() for n in range(N)], axis=1)
    M = np.vstack([Hc.real, Hc.imag])
    rng = np.random.default_rng(4)
    xt = rng.random(N)
    uc = (Hc @ xt).reshape(w.n_trans, nf) * (1.0 + 0.01 * rng.standard_normal((w.n_trans, nf)))
    us = np.concatenate([uc.ravel().real, uc.ravel().imag])
    Lm = laplacian_edge_by_edge(w.nz, w.ny, w.nx)
    mu = 0.02 * np.linalg.norm(M, 2) ** 2
    A = M.T @ M + mu * Lm; b = M.T @ us
    assert np.allclose(sph.backproject(w, uc, f0, df, nf).ravel(), b, rtol=1e-11, atol=1e-14 * np.abs(b).max())
    xc = np.zeros(N); r = b.copy(); p = r.copy(); xs = []
    for _ in range(6):
        Ap = A @ p; al = (r @ r) / (p @ Ap); xc = xc + al * p
        rn = r - al * Ap; p = rn + ((rn @ rn) / (r @ r)) * p; r = rn
        xs.append(xc.copy())
    x3, obj, grad = sph.pls_cg(w, uc, 3, mu, f0, df, nf)
    assert np.allclose(x3.ravel(), xs[2], rtol=1e-8, atol=1e-11 * np.abs(xs[2]).max())
    phi = lambda x: np.sum((us - M @ x) ** 2) + mu * x @ Lm @ x
    assert abs(obj[3] - phi(xs[2])) <= 1e-9 * obj[3] and np.all(np.diff(obj) < 0)
    x80, _, g80 = sph.pls_cg(w, uc, 80, mu, f0, df, nf)
    xd = np.linalg.solve(A, b)
    assert np.linalg.norm(x80.ravel() - xd) <= 1e-6 * np.linalg.norm(xd)


# ---------------------------------------------------------------- finite aperture (Eq. 18, reading G30)
def test_aperture_with_one_sub_element_is_the_point_like_model():
    w = problem(n=4, q=3)
    rng = np.random.default_rng(11)
    x = rng.standard_normal((w.nz, w.ny, w.nx))
    u = rng.standard_normal((w.n_trans, 12)) + 1j * rng.standard_normal((w.n_trans, 12))
    a = sph.project(w, x, 0.1, 0.3, 12)
    assert np.array_equal(a, sph.project(w, x, 0.1, 0.3, 12, aperture=2.0, m=1))
    assert np.array_equal(a, sph.project(w, x, 0.1, 0.3, 12, aperture=0.0, m=4))
    b = sph.backproject(w, u, 0.1, 0.3, 12)
    assert np.array_equal(b, sph.backproject(w, u, 0.1, 0.3, 12, aperture=2.0, m=1))


def test_sub_elements_tile_a_square_facing_the_grid_centre():
    """Reading G30: the m x m midpoints lie in the plane through r_q normal to (centre - r_q), inside a square of side a
    whose sides follow e_x, e_y of reading S1; their mean is r_q and their second moments are those of the midpoint rule."""
    w = problem(n=3, q=3)
    a, m = 2.0, 4
    for q in range(w.n_trans):
        pts = sph.element_points(w, q, a, m)
        assert pts.shape == (m * m, 3)
        rq = w.trans_xyz[q]
        n = (w.centre - rq) / np.linalg.norm(w.centre - rq)
        assert np.allclose((pts - rq) @ n, 0.0, atol=1e-12)                 # in the plane facing the centre
        assert np.allclose(pts.mean(axis=0), rq, atol=1e-12)
        ex, ey, ez = sph.element_frame(w, q)
        assert np.allclose(ez, n) and abs(ex @ ey) < 1e-12 and abs(ex @ ez) < 1e-12 and np.isclose(np.linalg.norm(ex), 1.0)
        assert abs(ey[2]) < 1e-12                                             # y^tr is horizontal (e_z x z^)
        lx, ly = (pts - rq) @ ex, (pts - rq) @ ey
        assert np.all(np.abs(lx) < a / 2) and np.all(np.abs(ly) < a / 2)
        assert np.isclose(np.mean(lx ** 2), a * a / 12.0 * (1.0 - 1.0 / m ** 2))   # midpoint rule on [-a/2, a/2]
        assert np.isclose(np.mean(ly ** 2), a * a / 12.0 * (1.0 - 1.0 / m ** 2))


def test_far_field_of_the_aperture_is_the_sinc_pattern():
    """Fraunhofer limit of Eq. (18): for a source far from a flat a x a element, (1/S_q) h~_q = G(d) sinc(k a s_x / 2)
    sinc(k a s_y / 2), k = 2 pi f / c, (s_x, s_y) = components of the unit vector element -> source along the element's
    sides.  The element (2 mm, m = 24 sub-elements per side) faces the centre of a coarse 3^3 grid 400 mm away, so the
    grid's off-centre nodes sample the pattern well off its axis (|k a s / 2| up to ~5); the residual is the Fresnel term
    ~ k a^2 / (8 d) <= 1.6e-2 rad, hence the 1.2e-2 gate.  The voxel size enters only through the common factor p~0."""
    ds, a, m = 150.0, 2.0, 24
    tr = np.array([[400.0, 30.0, -20.0]])
    o = -1.0 * ds
    w = wl.Workload("sph-ff", 3, 3, 3, ds, (o, o, o), tr, c=1.5, t0=0.0, dt=0.05, nt=8, surf_step=ds, kband=8, gain=1.0)
    f0, df, nf = 0.5, 0.5, 6                                       # 0.5 .. 3 MHz: lambda 3 .. 0.5 mm
    f = sph.freqs(f0, df, nf)
    ex, ey, ez = sph.element_frame(w, 0)
    p0 = sph.p0_tilde(w, f)
    k = 2.0 * np.pi * f / w.c
    strongest = 1.0
    for (iz, iy, ix) in [(1, 1, 1), (1, 2, 1), (0, 1, 1), (2, 2, 0), (0, 0, 2)]:
        x = np.zeros((3, 3, 3)); x[iz, iy, ix] = 1.0
        node = np.asarray(w.origin) + ds * np.array([ix, iy, iz])
        u = sph.project(w, x, f0, df, nf, aperture=a, m=m)[0]
        v = node - tr[0]
        d = np.linalg.norm(v)
        sx, sy = (v / d) @ ex, (v / d) @ ey
        pat = np.sinc(k * a * sx / 2.0 / np.pi) * np.sinc(k * a * sy / 2.0 / np.pi)      # np.sinc(t) = sin(pi t)/(pi t)
        exp = p0 * np.exp(-1j * k * d) / (2.0 * np.pi * d) * pat
        scale = np.abs(p0 / (2.0 * np.pi * d))
        assert np.all(np.abs(u - exp) <= 1.2e-2 * scale), ((iz, iy, ix), np.abs(u - exp) / scale)
        strongest = min(strongest, np.abs(pat).min())
        if (iz, iy, ix) != (1, 1, 1):                              # off axis the point-like response is clearly different
            up = sph.project(w, x, f0, df, nf)[0]
            assert np.abs(up - u).max() > 0.2 * np.abs(up).max()
    assert strongest < 0.1                                         # the pattern was sampled down to its side lobes


def test_adjoint_identity_with_aperture():
    w = problem(n=4, q=3)
    rng = np.random.default_rng(12)
    x = rng.standard_normal((w.nz, w.ny, w.nx))
    u = rng.standard_normal((w.n_trans, 9)) + 1j * rng.standard_normal((w.n_trans, 9))
    he = rng.standard_normal(9) + 1j * rng.standard_normal(9)
    hx = sph.project(w, x, 0.2, 0.4, 9, he, aperture=1.5, m=3)
    htu = sph.backproject(w, u, 0.2, 0.4, 9, he, aperture=1.5, m=3)
    lhs, rhs = np.real(np.vdot(hx, u)), float(np.vdot(x, htu))
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))


def test_row_and_point_evaluations_equal_the_full_operators():
    """project_rows / backproject_points (used for sampled parity at the bench's sizes) are the same sums as project /
    backproject."""
    w = problem(n=5, q=4)
    rng = np.random.default_rng(13)
    x = rng.standard_normal((w.nz, w.ny, w.nx))
    u = rng.standard_normal((w.n_trans, 7)) + 1j * rng.standard_normal((w.n_trans, 7))
    full = sph.project(w, x, 0.1, 0.2, 7, aperture=1.0, m=2)
    rows = sph.project_rows(w, x, [3, 1], 0.1, 0.2, 7, aperture=1.0, m=2, chunk=17)
    assert np.allclose(rows, full[[3, 1]], rtol=1e-12, atol=1e-15)
    xb = sph.backproject(w, u, 0.1, 0.2, 7, aperture=1.0, m=2)
    from oracle.oat_fbp import node_positions
    pts = node_positions(w)[[0, 4, 2], [1, 3, 2], [4, 0, 2]]
    assert np.allclose(sph.backproject_points(w, u, pts, 0.1, 0.2, 7, aperture=1.0, m=2), xb[[0, 4, 2], [1, 3, 2], [4, 0, 2]], rtol=1e-12, atol=1e-15)
