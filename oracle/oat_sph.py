"""fp64 / complex128 CPU oracle of row NEXT-3: the spherical-voxel imaging model in the temporal
frequency domain, H_sph (Eq. 17-20) and its adjoint H_sph† (Eq. 24), for point-like transducers (Alg. 9
L684-729, line 7) and for finite flat square apertures (the spatial impulse response of Eq. 18; L243, L291).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package.  Plain numpy.

Readings (also in DESIGN.md §2):
  G27  Frequencies: Eq. (17) has f = l df, Alg. 9 line 1 f = l df + f_min; taken as f_l = f0 + l df, l = 0..L-1.
       p~0(f) of Eq. (19) L153 has the removable singularity f = 0 (the bracket is O(f^3) against 1/f): p~0(0) := 0.
       beta c0^3 / C_p = 4 pi kappa c0^3 with kappa = beta / (4 pi C_p) (the library's `gain`); h~e(f) := 1 unless given.
  G28  Transducers are point-like: (1/S_q) h~_q(r_n, f) -> exp(-j 2 pi f d / c0) / (2 pi d), d = |r_q - r_n| (Eq. 18
       with S_q -> a point; Alg. 9 line 7 "example here assumes point-like transducers").  A voxel that coincides with a
       transducer (d = 0) contributes nothing.
  G30  Finite aperture (Eq. 18 L152 integrates over the transducer surface S_q; the paper prints no evaluation rule and no
       element orientation; its elements are 2 x 2 mm^2, L291): S_q is a flat square of side `aperture`, centred on r_q,
       whose normal points to the grid centre (the z^tr axis of Appendix) and whose sides lie along the x^tr, y^tr
       axes of reading S1.  The integral is the plain m x m midpoint rule: (1/S_q) h~_q = (1/m^2) sum_ij G(r_ij, r_n, f)
       with r_ij = r_q + ((i+1/2)/m - 1/2) a e_x + ((j+1/2)/m - 1/2) a e_y and G the point response of reading G28.
       m = 1 (or aperture = 0) is the point-like model.  PARITY UNPINNED against the authors' code (no value printed);
       pinned here by m = 1, by the Fraunhofer limit of the continuous integral and by the adjoint identity.
  G29  Eq. (24) as printed maps complex data to a complex image; alpha is real (Eq. 16), so the adjoint with respect to
       the real inner product Re<.,.> of C^{QL} is its real part, and that is what H_sph† returns:
       Re<H x, u> = <x, H† u> for real x.
"""
from __future__ import annotations

import numpy as np

from .oat_fbp import node_positions
from . import oat_pls as _pls


def freqs(f0, df, nf):
    return f0 + df * np.arange(nf, dtype=np.float64)


def p0_tilde(w, f, he=None):
    """Eq. (19): p~0(f) = -j (beta c^3 / (C_p f)) [ (ds/2c) cos(pi f ds / c) - sin(pi f ds / c)/(2 pi f) ] h~e(f)."""
    f = np.asarray(f, dtype=np.float64)
    out = np.zeros(f.shape, dtype=np.complex128)
    nz = f != 0.0
    fn = f[nz]
    br = (w.spacing / (2.0 * w.c)) * np.cos(np.pi * fn * w.spacing / w.c) - np.sin(np.pi * fn * w.spacing / w.c) / (2.0 * np.pi * fn)
    out[nz] = -1j * (4.0 * np.pi * w.gain * w.c ** 3 / fn) * br
    if he is not None:
        out = out * np.asarray(he, dtype=np.complex128)
    return out


def element_frame(w, q):
    """Reading S1 (Appendix): e_z from the transducer to the grid centre, e_y = (e_z x z^)/|.| (y^ if parallel),
    e_x = e_y x e_z.  Returns (e_x, e_y, e_z)."""
    v = np.asarray(w.centre, dtype=np.float64) - np.asarray(w.trans_xyz, dtype=np.float64)[q]
    ez = v / np.sqrt(np.sum(v * v))
    a = np.array([ez[1], -ez[0], 0.0])
    an = np.sqrt(np.sum(a * a))
    ey = np.array([0.0, 1.0, 0.0]) if an < 1e-12 else a / an
    ex = np.cross(ey, ez)
    return ex, ey, ez


def element_points(w, q, aperture=0.0, m=1):
    """Midpoints r_ij of the m x m sub-elements of transducer q's square surface (reading G30): (m*m, 3)."""
    rq = np.asarray(w.trans_xyz, dtype=np.float64)[q]
    if aperture == 0.0 or m == 1:
        return rq[None, :].copy()
    ex, ey, _ = element_frame(w, q)
    pts = []
    for i in range(m):
        for j in range(m):
            pts.append(rq + ((i + 0.5) / m - 0.5) * aperture * ex + ((j + 0.5) / m - 0.5) * aperture * ey)
    return np.array(pts)


def _dist(w, r):
    pts = node_positions(w).reshape(-1, 3)
    return np.sqrt(np.sum((pts - r) ** 2, axis=1))


def project(w, x, f0, df, nf, he=None, aperture=0.0, m=1):
    """Eq. (17): u[q,l] = p~0(f_l) sum_n x_n (1/S_q) h~_q(r_n, f_l), with (1/S_q) h~_q the mean over the sub-elements of
    exp(-j 2 pi f_l d / c) / (2 pi d), d = |r_ij - r_n| (Eq. 18, readings G28 / G30); returns complex (Q, L)."""
    x = np.asarray(x, dtype=np.float64).ravel()
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    u = np.zeros((w.n_trans, nf), dtype=np.complex128)
    for q in range(w.n_trans):
        el = element_points(w, q, aperture, m)
        for r in el:
            d = _dist(w, r)
            ok = d > 0
            amp = np.where(ok, x / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0)
            u[q] += p0 * (np.exp(-2j * np.pi * np.outer(f, d) / w.c) @ amp) / len(el)
    return u


def backproject(w, u, f0, df, nf, he=None, aperture=0.0, m=1):
    """Eq. (24), real part (reading G29): x_n = Re sum_q sum_l u[q,l] p~0*(f_l) conj((1/S_q) h~_q(r_n, f_l))."""
    u = np.asarray(u, dtype=np.complex128)
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    x = np.zeros(w.n_voxels, dtype=np.float64)
    for q in range(w.n_trans):
        v = u[q] * np.conj(p0)
        el = element_points(w, q, aperture, m)
        for r in el:
            d = _dist(w, r)
            ok = d > 0
            s = (v @ np.exp(2j * np.pi * np.outer(f, d) / w.c)).real
            x += np.where(ok, s / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0) / len(el)
    return x.reshape(w.nz, w.ny, w.nx)


def project_rows(w, x, q_list, f0, df, nf, he=None, aperture=0.0, m=1, chunk=200000):
    """Rows q in q_list of Eq. (17) on a LARGE grid: the same sum as project(), taken over the voxels in chunks so that
    the (frequency x voxel) phasor table fits in memory; returns complex (len(q_list), L)."""
    x = np.asarray(x, dtype=np.float64).ravel()
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    pts = node_positions(w).reshape(-1, 3)
    out = np.zeros((len(q_list), nf), dtype=np.complex128)
    for row, q in enumerate(q_list):
        el = element_points(w, q, aperture, m)
        for r in el:
            for a in range(0, x.size, chunk):
                d = np.sqrt(np.sum((pts[a:a + chunk] - r) ** 2, axis=1))
                ok = d > 0
                amp = np.where(ok, x[a:a + chunk] / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0)
                out[row] += p0 * (np.exp(-2j * np.pi * np.outer(f, d) / w.c) @ amp) / len(el)
    return out


def backproject_points(w, u, pts, f0, df, nf, he=None, aperture=0.0, m=1):
    """Eq. (24) (real part) at arbitrary points `pts` (M, 3): the same sum as backproject(), voxel by voxel; returns (M,)."""
    u = np.asarray(u, dtype=np.complex128)
    pts = np.asarray(pts, dtype=np.float64)
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    out = np.zeros(pts.shape[0], dtype=np.float64)
    for q in range(w.n_trans):
        v = u[q] * np.conj(p0)
        el = element_points(w, q, aperture, m)
        for r in el:
            d = np.sqrt(np.sum((pts - r) ** 2, axis=1))
            ok = d > 0
            s = (v @ np.exp(2j * np.pi * np.outer(f, d) / w.c)).real
            out += np.where(ok, s / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0) / len(el)
    return out


def pls_cg(w, u, n_iter, mu, f0, df, nf, he=None, aperture=0.0, m=1):
    """PLS-Sph, Eq. (30) L271 with "linear CG" (L265): CG on (H† H + mu L) x = H† u from x0 = 0 with H = H_sph, H† its
    real-part adjoint (reading G29) and L the penalty matrix of Eq. (34) (oat_pls.penalty_apply); the data space is
    C^{QL} with the real inner product Re<.,.>.  Same loop and curves as oat_pls.pls_cg (reading G22):
    obj_i = ||u - H x_i||^2 + mu R(x_i), grad_i = ||H† u - (H† H + mu L) x_i||."""
    u = np.asarray(u, dtype=np.complex128)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    d = u.copy()
    r = backproject(w, u, f0, df, nf, he, aperture, m)
    p = r.copy()
    rr = float(np.vdot(r, r))
    obj = [float(np.real(np.vdot(d, d)))]
    grad = [rr ** 0.5]
    for _ in range(n_iter):
        q = project(w, p, f0, df, nf, he, aperture, m)
        wv = backproject(w, q, f0, df, nf, he, aperture, m) + mu * _pls.penalty_apply(p)
        pw = float(np.vdot(p, wv))
        if pw <= 0.0 or rr == 0.0:
            obj.append(obj[-1]); grad.append(grad[-1]); continue
        alpha = rr / pw
        x += alpha * p
        d -= alpha * q
        r -= alpha * wv
        rr_new = float(np.vdot(r, r))
        p = r + (rr_new / rr) * p
        rr = rr_new
        obj.append(float(np.real(np.vdot(d, d))) + mu * _pls.penalty_value(x))
        grad.append(rr ** 0.5)
    return x, np.array(obj), np.array(grad)
