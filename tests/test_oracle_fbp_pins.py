"""Pins of the NEXT-2 oracle (oracle/oat_fbp.py, Eq. 27) against things other than itself: the un-fused
evaluation of the continuous formula Eq. (4) with the approximations Eq. (25)-(26), the exact reconstruction of a
uniform ball from its closed-form N-wave data, and the support of a single data sample.  CPU only."""
import math

import numpy as np

from oracle import oat_fbp as fbp
from paper_1304_2017_b200 import workloads as wl


def sphere_problem(q=1500, rs=30.0, n=9, ds=0.5, dt=0.02, nt=2200, t0=2.0, kappa=1.0):
    tr = wl.fibonacci_sphere(q, rs)
    o = -(n - 1) * ds / 2.0
    return wl.Workload("fbp-pin", n, n, n, ds, (o, o, o), tr, c=1.5, t0=t0, dt=dt, nt=nt, surf_step=ds, kband=32, gain=kappa)


def ball_data(w, centre, rb, amp):
    """Exact pressure of a uniform ball: p = kappa (-2 pi A c^2 (ct - d)/d) for |ct - d| <= R_b (from Eq. 2-3)."""
    t = w.t0 + w.dt * np.arange(w.nt)
    d = np.linalg.norm(w.trans_xyz - np.asarray(centre), axis=1)[:, None]
    s = w.c * t[None, :] - d
    return np.where(np.abs(s) <= rb, w.gain * (-2.0 * math.pi * amp * w.c ** 2 * s / d), 0.0)


def test_fused_formula_equals_eq4_with_eq25_and_eq26():
    """Eq. (27) = Eq. (4) with the linear interpolation Eq. (25) and the difference Eq. (26), evaluated separately
    here (reading G24: the bracket of Alg. 2 line 9 does not satisfy this, Eq. 27 does)."""
    w = sphere_problem(q=40, nt=600, dt=0.05, t0=14.0)
    rng = np.random.default_rng(0)
    p = rng.standard_normal((w.n_trans, w.nt))
    areas = wl.patch_areas_equal(w.trans_xyz, w.centre)
    wq = fbp.weights(w, areas)
    pts = rng.uniform(-2.0, 2.0, size=(25, 3))
    got = fbp.fbp_points(w, p, wq, pts)
    rs = np.linalg.norm(w.trans_xyz - w.centre, axis=1)
    exp = np.zeros(len(pts))
    for q in range(w.n_trans):
        d = np.linalg.norm(pts - w.trans_xyz[q], axis=1)
        kt = (d / w.c - w.t0) / w.dt
        k = np.floor(kt).astype(int)
        assert np.all((k >= 0) & (k + 1 < w.nt))
        pint = (k + 1 - kt) * p[q, k] + (kt - k) * p[q, k + 1]                 # Eq. (25)
        dpdt = (p[q, k + 1] - p[q, k]) / w.dt                                   # Eq. (26)
        # Eq. (4): -C_p/(2 pi beta c^2 R^s) dS [2 p/|r - r^s| + (1/c) dp/dt], C_p/beta = 1/(4 pi kappa)
        exp += -areas[q] / (8.0 * math.pi ** 2 * w.gain * w.c ** 2 * rs[q]) * (2.0 * pint / d + dpdt / w.c)
    assert np.allclose(got, exp, rtol=1e-11, atol=1e-14)


def test_uniform_ball_is_reconstructed_from_its_n_wave():
    """Full-sphere FBP (Eq. 4 is exact for a spherical aperture) of closed-form ball data: A inside, 0 outside."""
    w = sphere_problem()
    centre, rb, amp = np.array([0.4, -0.3, 0.2]), 1.2, 0.7
    p = ball_data(w, centre, rb, amp)
    wq = fbp.weights(w, wl.patch_areas_equal(w.trans_xyz, w.centre))
    inside = centre + np.array([[0, 0, 0], [0.5, 0, 0], [0, -0.6, 0.3], [-0.3, 0.3, 0.5]])
    vin = fbp.fbp_points(w, p, wq, inside)
    # inside the ball every shell crosses the linear part of the N-wave, where Eq. (25)-(26) are exact: only the
    # quadrature over the 1500 transducers is left (probed 2e-7)
    assert np.all(np.abs(vin / amp - 1.0) < 1e-5), vin
    # outside, the jumps at the ends of the N-wave alias against the finite transducer count (streaks of either sign,
    # probed rms 0.11 A at Q = 1500): the image is zero in the mean
    rng = np.random.default_rng(1)
    u = rng.standard_normal((300, 3)); u /= np.linalg.norm(u, axis=1)[:, None]
    vout = fbp.fbp_points(w, p, wq, centre + u * rng.uniform(1.6, 3.0, size=(300, 1))) / amp
    assert abs(np.mean(vout)) < 0.02 and np.sqrt(np.mean(vout ** 2)) < 0.2
    # scale pins: twice the amplitude -> twice the image; kappa cancels between data and weights
    w2 = sphere_problem(kappa=2.5)
    p2 = ball_data(w2, centre, rb, amp)
    v2 = fbp.fbp_points(w2, p2, fbp.weights(w2, wl.patch_areas_equal(w2.trans_xyz, w2.centre)), inside)
    assert np.allclose(v2, vin, rtol=1e-12)


def test_single_data_sample_lights_up_one_shell():
    """p = e_(q0,k0): only voxels with k0 - 1 < k~ < k0 + 1 receive anything, with the two brackets of Eq. (27)."""
    w = sphere_problem(q=6, n=21, ds=0.25, nt=700, dt=0.05, t0=12.0)
    q0, k0 = 2, 160
    p = np.zeros((w.n_trans, w.nt)); p[q0, k0] = 1.0
    wq = np.arange(1.0, w.n_trans + 1.0)
    img = fbp.fbp(w, p, wq)
    pts = fbp.node_positions(w).reshape(-1, 3)
    kt = (np.linalg.norm(pts - w.trans_xyz[q0], axis=1) / w.c - w.t0) / w.dt
    tau = w.t0 / w.dt
    k = np.floor(kt)
    exp = np.where(k == k0, wq[q0] * ((k0 + 1 + tau) / (kt + tau) - 1.5),
                   np.where(k == k0 - 1, wq[q0] * (1.5 - (k0 - 1 + tau) / (kt + tau)), 0.0))
    assert np.count_nonzero(exp) > 50
    assert np.allclose(img.ravel(), exp, rtol=1e-12, atol=1e-15)


def test_record_edges_and_linearity():
    w = sphere_problem(q=5, n=7, nt=40, dt=0.05, t0=19.0)      # the record covers only part of the grid (reading G25)
    rng = np.random.default_rng(3)
    p1, p2 = rng.standard_normal((5, 40)), rng.standard_normal((5, 40))
    wq = rng.standard_normal(5)
    a = fbp.fbp(w, p1, wq); b = fbp.fbp(w, p2, wq)
    assert np.allclose(fbp.fbp(w, 2.0 * p1 - 3.0 * p2, wq), 2.0 * a - 3.0 * b, rtol=1e-12, atol=1e-13)
    pts = fbp.node_positions(w).reshape(-1, 3)
    # a transducer whose every k~ is outside [0, K-1) contributes exactly nothing
    w.trans_xyz = np.vstack([w.trans_xyz, [[300.0, 0.0, 0.0]]])
    p3 = np.vstack([p1, rng.standard_normal((1, 40))])
    assert np.array_equal(fbp.fbp(w, p3, np.append(wq, 7.0)), a)
    assert np.isfinite(a).all() and pts.shape[0] == a.size


def test_weights_are_the_constant_of_eq27_for_the_papers_geometry():
    """Eq. (27) L221 prints, for the ring/view geometry of L203, the factor -C_p R^s dtheta dphi sin(theta_q) / (pi beta c0^3 dt);
    with kappa = beta / (4 pi C_p) that is -R^s dtheta dphi sin(theta_q) / (4 pi^2 kappa c0^3 dt).  Numbers by hand."""
    rs, n_el, n_views = 65.0, 4, 6
    w = wl.Workload("w", 5, 5, 5, 0.5, (-1.0, -1.0, -1.0), np.zeros((n_el * n_views, 3)), c=1.5, t0=1.0, dt=0.05, nt=10, surf_step=0.5, gain=0.25)
    pol = np.deg2rad(14.0 + np.arange(n_el) * 152.0 / (n_el - 1))
    dth, dph = np.deg2rad(152.0 / (n_el - 1)), 2.0 * math.pi / n_views
    tr = []
    for e in range(n_el):
        for v in range(n_views):
            tr.append([rs * math.sin(pol[e]) * math.cos(v * dph), rs * math.sin(pol[e]) * math.sin(v * dph), rs * math.cos(pol[e])])
    w.trans_xyz = np.array(tr) + w.centre
    got = fbp.weights(w, wl.patch_areas_arc(n_el, n_views, rs))
    beta_over_cp = 4.0 * math.pi * 0.25
    exp = np.repeat(-rs * dth * dph * np.sin(pol) / (math.pi * beta_over_cp * 1.5 ** 3 * 0.05), n_views)
    assert np.allclose(got, exp, rtol=1e-13)


def test_interval_margin_flags_ties_and_nothing_else():
    """oat_fbp.interval_margin decides which points a parity test may skip (reading G26): it must be ~0 exactly where some
    k~ is an integer -- the centre of a Fibonacci sphere whose radius is a whole number of samples -- and equal to the
    constructed offset elsewhere, so that a threshold of 1e-9 excludes the ties and nothing at margin 1e-6."""
    w = sphere_problem(q=50, rs=30.0, n=5, ds=0.5, dt=0.02, nt=2200, t0=2.0)     # k~ at the centre = (30/1.5 - 2)/0.02 = 900
    m0 = fbp.interval_margin(w, np.zeros((1, 3)))
    assert m0[0] < 1e-9
    # a point on the axis through transducer 0, displaced by delta samples: margin = |delta| for that transducer at most
    u = w.trans_xyz[0] / np.linalg.norm(w.trans_xyz[0])
    for delta in (1e-6, 1e-3, 0.25):
        pt = (u * (-delta * w.c * w.dt))[None, :]                                  # farther from transducer 0 by delta samples
        m = fbp.interval_margin(w, pt)
        assert 0.0 < m[0] <= delta * (1 + 1e-6) + 1e-9
        kt = (np.linalg.norm(w.trans_xyz - pt, axis=1) / w.c - w.t0) / w.dt
        assert np.isclose(m[0], np.min(np.abs(kt - np.rint(kt))), rtol=0, atol=1e-12)
        if delta >= 1e-6:
            assert m[0] > 1e-9 or delta < 1e-6
    # points whose every k~ lies outside the record are never ties
    far = np.array([[1e4, 0.0, 0.0]])
    assert np.isinf(fbp.interval_margin(w, far)[0])
    # generic points: the margin is the brute-force minimum over transducers
    rng = np.random.default_rng(5)
    pts = rng.uniform(-1.0, 1.0, size=(20, 3))
    m = fbp.interval_margin(w, pts)
    for i, pt in enumerate(pts):
        kt = (np.linalg.norm(w.trans_xyz - pt, axis=1) / w.c - w.t0) / w.dt
        assert np.isclose(m[i], np.min(np.abs(kt - np.rint(kt))), atol=1e-12)
    assert np.all(m > 1e-9)
