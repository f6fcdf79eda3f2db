"""fp64 CPU oracle of row NEXT-1: the electrical impulse response operator H^e / H^e†,
the quadratic smoothness penalty R, and the penalised least-squares CG loop "PLS-Int" of the paper.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package.  Plain numpy, fp64,
written in the paper's order and notation; citations are PAPER.md line numbers.

Readings taken where the paper is silent (also listed in DESIGN.md §2):
  G20  Eq. (14) L129 / Eq. (21) L170 index the impulse response with k-1-kappa (a one-sample delay); taken
       literally.  [h^e]_m = dt * h^e(m dt) is given for m = 0..L-1 and is zero for every other m (causal,
       finite), and the sums run over kappa = 0..K-1 only (zero extension of p outside the record).
  G21  Eq. (34): n_x, n_y, n_z are "the neighboring voxels before the n-th voxel"; a voxel on the low
       face of the grid has no such neighbour and that term is omitted.
  G22  Eq. (29) L267 with "linear CG" (L265): CG on the normal equations (H^T H + mu L) x = H^T u from
       x0 = 0 with a fixed iteration count, where H = H^e D G and L is the symmetric matrix with
       R(x) = x^T L x (so grad(mu R) = 2 mu L x and grad ||u - Hx||^2 = -2 H^T (u - Hx)).  One H and one H^T
       per iteration (L273).  Curves: objective ||u - H x_i||^2 + mu R(x_i) and ||H^T u - (H^T H + mu L) x_i||.
"""
from __future__ import annotations

import numpy as np

from . import oat_oracle as _orc


def eir_apply(he, p):
    """Eq. (14):  u[q,k] = sum_{kappa=0}^{K-1} he[k-1-kappa] p[q,kappa]   (reading G20)."""
    he = np.asarray(he, dtype=np.float64)
    p = np.asarray(p, dtype=np.float64)
    K = p.shape[-1]
    u = np.zeros_like(p)
    for m in range(he.size):                 # tap m = k-1-kappa  <=>  kappa = k-1-m
        sh = m + 1                           # u[k] += he[m] p[k-sh]
        if sh >= K:
            break
        u[..., sh:] += he[m] * p[..., :K - sh]
    return u


def eir_adjoint(he, u):
    """Eq. (21):  p'[q,k] = sum_{kappa=0}^{K-1} he[kappa-1-k] u[q,kappa]."""
    he = np.asarray(he, dtype=np.float64)
    u = np.asarray(u, dtype=np.float64)
    K = u.shape[-1]
    pp = np.zeros_like(u)
    for m in range(he.size):                 # tap m = kappa-1-k  <=>  kappa = k+1+m
        sh = m + 1
        if sh >= K:
            break
        pp[..., :K - sh] += he[m] * u[..., sh:]
    return pp


def penalty_value(x):
    """Eq. (34): R = sum_n (x_n - x_{n_x})^2 + (x_n - x_{n_y})^2 + (x_n - x_{n_z})^2 (reading G21).
    x has shape (nz, ny, nx)."""
    x = np.asarray(x, dtype=np.float64)
    r = 0.0
    for ax in range(3):
        d = np.diff(x, axis=ax)              # x_n - x_{n before} for every n that has a neighbour before it
        r += float(np.sum(d * d))
    return r


def penalty_apply(x):
    """L x with R(x) = x^T L x:  (L x)_n = sum over axes of (x_n - x_before) [if it exists] + (x_n - x_after) [if it exists]."""
    x = np.asarray(x, dtype=np.float64)
    out = np.zeros_like(x)
    for ax in range(3):
        d = np.diff(x, axis=ax)
        lo = [slice(None)] * 3; hi = [slice(None)] * 3
        lo[ax] = slice(0, x.shape[ax] - 1); hi[ax] = slice(1, x.shape[ax])
        out[tuple(hi)] += d                  # (x_n - x_before) at n
        out[tuple(lo)] -= d                  # (x_n - x_after) at the neighbour before
    return out


def project_full(w, x, he=None, **kw):
    """H x = H^e D G x (Eq. 11); he = None leaves the EIR out."""
    y = _orc.project(w, x, **kw)
    return y if he is None else eir_apply(he, y)


def backproject_full(w, u, he=None, **kw):
    """H^T u = G^T D^T H^e† u (L168)."""
    u = np.asarray(u, dtype=np.float64)
    return _orc.backproject(w, u if he is None else eir_adjoint(he, u), **kw)


def pls_cg(w, u, n_iter, mu, he=None, **kw):
    """Reading G22: linear CG on (H^T H + mu L) x = H^T u from x0 = 0 (Eq. 29).

    r = H^T u; p = r; loop { q = H p; w = H^T q + mu L p; alpha = <r,r>/<p,w>; x += alpha p; d -= alpha q;
    r -= alpha w; beta = <r,r>_new/<r,r>_old; p = r + beta p } with d = u - H x tracked alongside.
    Returns x and the curves obj_i = ||d_i||^2 + mu R(x_i), grad_i = ||r_i||, i = 0..n_iter.
    """
    u = np.asarray(u, dtype=np.float64)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    d = u.copy()
    r = backproject_full(w, u, he, **kw)
    p = r.copy()
    rr = float(np.vdot(r, r))
    obj = [float(np.vdot(d, d))]
    grad = [rr ** 0.5]
    for _ in range(n_iter):
        q = project_full(w, p, he, **kw)
        wv = backproject_full(w, q, he, **kw) + mu * penalty_apply(p)
        pw = float(np.vdot(p, wv))
        if pw <= 0.0 or rr == 0.0:
            obj.append(obj[-1]); grad.append(grad[-1]); continue
        alpha = rr / pw
        x += alpha * p
        d -= alpha * q
        r -= alpha * wv
        rr_new = float(np.vdot(r, r))
        beta = rr_new / rr
        rr = rr_new
        p = r + beta * p
        obj.append(float(np.vdot(d, d)) + mu * penalty_value(x))
        grad.append(rr ** 0.5)
    return x, np.array(obj), np.array(grad)
