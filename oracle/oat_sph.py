"""fp64 / complex128 CPU oracle of row NEXT-3: the spherical-voxel imaging model in the temporal
frequency domain, H_sph (Eq. 17-20) and its adjoint H_sph† (Eq. 24), for point-like transducers (Alg. 9
L684-729, line 7).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package.  Plain numpy.

Readings (also in DESIGN.md §2):
  G27  Frequencies: Eq. (17) has f = l df, Alg. 9 line 1 f = l df + f_min; taken as f_l = f0 + l df, l = 0..L-1.
       p~0(f) of Eq. (19) L153 has the removable singularity f = 0 (the bracket is O(f^3) against 1/f): p~0(0) := 0.
       beta c0^3 / C_p = 4 pi kappa c0^3 with kappa = beta / (4 pi C_p) (the library's `gain`); h~e(f) := 1 unless given.
  G28  Transducers are point-like: (1/S_q) h~_q(r_n, f) -> exp(-j 2 pi f d / c0) / (2 pi d), d = |r_q - r_n| (Eq. 18
       with S_q -> a point; Alg. 9 line 7 "example here assumes point-like transducers").  A voxel that coincides with a
       transducer (d = 0) contributes nothing.
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


def _dist(w, q):
    pts = node_positions(w).reshape(-1, 3)
    return np.sqrt(np.sum((pts - np.asarray(w.trans_xyz, dtype=np.float64)[q]) ** 2, axis=1))


def project(w, x, f0, df, nf, he=None):
    """Eq. (17): u[q,l] = p~0(f_l) sum_n x_n exp(-j 2 pi f_l d_qn / c) / (2 pi d_qn); returns complex (Q, L)."""
    x = np.asarray(x, dtype=np.float64).ravel()
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    u = np.zeros((w.n_trans, nf), dtype=np.complex128)
    for q in range(w.n_trans):
        d = _dist(w, q)
        ok = d > 0
        amp = np.where(ok, x / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0)
        u[q] = p0 * (np.exp(-2j * np.pi * np.outer(f, d) / w.c) @ amp)
    return u


def backproject(w, u, f0, df, nf, he=None):
    """Eq. (24), real part (reading G29): x_n = Re sum_q sum_l u[q,l] p~0*(f_l) exp(+j 2 pi f_l d_qn / c) / (2 pi d_qn)."""
    u = np.asarray(u, dtype=np.complex128)
    f = freqs(f0, df, nf)
    p0 = p0_tilde(w, f, he)
    x = np.zeros(w.n_voxels, dtype=np.float64)
    for q in range(w.n_trans):
        d = _dist(w, q)
        ok = d > 0
        v = u[q] * np.conj(p0)
        s = (v @ np.exp(2j * np.pi * np.outer(f, d) / w.c)).real
        x += np.where(ok, s / (2.0 * np.pi * np.where(ok, d, 1.0)), 0.0)
    return x.reshape(w.nz, w.ny, w.nx)


def pls_cg(w, u, n_iter, mu, f0, df, nf, he=None):
    """PLS-Sph, Eq. (30) L271 with "linear CG" (L265): CG on (H† H + mu L) x = H† u from x0 = 0 with H = H_sph, H† its
    real-part adjoint (reading G29) and L the penalty matrix of Eq. (34) (oat_pls.penalty_apply); the data space is
    C^{QL} with the real inner product Re<.,.>.  Same loop and curves as oat_pls.pls_cg (reading G22):
    obj_i = ||u - H x_i||^2 + mu R(x_i), grad_i = ||H† u - (H† H + mu L) x_i||."""
    u = np.asarray(u, dtype=np.complex128)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    d = u.copy()
    r = backproject(w, u, f0, df, nf, he)
    p = r.copy()
    rr = float(np.vdot(r, r))
    obj = [float(np.real(np.vdot(d, d)))]
    grad = [rr ** 0.5]
    for _ in range(n_iter):
        q = project(w, p, f0, df, nf, he)
        wv = backproject(w, q, f0, df, nf, he) + mu * _pls.penalty_apply(p)
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
