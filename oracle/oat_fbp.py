"""fp64 CPU oracle of row NEXT-2: the discretised filtered backprojection of the paper,
Eq. (27) L221 (continuous form Eq. 4; approximations Eq. 25-26; Algs. 1-2 L457-499).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the CUDA package.  Plain numpy, fp64.

Readings (also in DESIGN.md §2):
  G23  Eq. (27) is printed for the ring/view geometry of L203 with the patch area (R^s)^2 dtheta dphi sin(theta_q).
       The operator here takes ONE WEIGHT PER TRANSDUCER,
           w_q = -C_p dS_q / (pi beta c0^3 dt R^s)  =  -dS_q / (4 pi^2 kappa c0^3 dt R^s),   kappa = beta/(4 pi C_p),
       with dS_q the transducer's patch area, so that any sampling of the sphere can be used; for the paper's
       geometry dS_q = (R^s)^2 dtheta dphi sin(theta_q) reproduces Eq. (27) exactly.
  G24  Alg. 2 L491 (line 9) prints the bracket with k where Eq. (27) has k+1 and with the two samples swapped; Eq. (27)
       is the one that follows from Eq. (4) with Eq. (25)-(26) (checked in the pins) and is the one implemented.
  G25  Samples outside the record: a voxel/transducer pair whose k = floor(k~) is < 0 or whose k+1 is > K-1
       contributes nothing (the paper is silent; its texture fetch would clamp).  A voxel that coincides with a
       transducer (k~ + t_min/dt = 0) contributes nothing.
"""
from __future__ import annotations

import numpy as np


def node_positions(w):
    """(nz, ny, nx, 3) positions of the grid nodes, node (ix,iy,iz) at origin + spacing (ix,iy,iz) (L203)."""
    o = np.asarray(w.origin, dtype=np.float64)
    xs = o[0] + w.spacing * np.arange(w.nx)
    ys = o[1] + w.spacing * np.arange(w.ny)
    zs = o[2] + w.spacing * np.arange(w.nz)
    zz, yy, xx = np.meshgrid(zs, ys, xs, indexing="ij")
    return np.stack([xx, yy, zz], axis=-1)


def fbp_points(w, p, weights, pts):
    """Eq. (27) at arbitrary points `pts` (M, 3): returns (M,) values.

    alpha = sum_q w_q { (1.5 - (k+tau)/(k~+tau)) p[q,k+1] + ((k+1+tau)/(k~+tau) - 1.5) p[q,k] },
    k~ = (|r_q - r|/c0 - t_min)/dt, k = floor(k~), tau = t_min/dt.
    """
    p = np.asarray(p, dtype=np.float64)
    wq = np.asarray(weights, dtype=np.float64)
    pts = np.asarray(pts, dtype=np.float64)
    tr = np.asarray(w.trans_xyz, dtype=np.float64)
    K = w.nt
    tau = w.t0 / w.dt
    out = np.zeros(pts.shape[0], dtype=np.float64)
    for q in range(tr.shape[0]):
        d = np.sqrt(np.sum((pts - tr[q]) ** 2, axis=1))
        kt = (d / w.c - w.t0) / w.dt
        k = np.floor(kt)
        den = kt + tau
        ok = (k >= 0) & (k + 1 <= K - 1) & (den > 0)             # reading G25
        ki = np.where(ok, k, 0).astype(np.int64)
        dn = np.where(ok, den, 1.0)
        a1 = 1.5 - (ki + tau) / dn
        a0 = (ki + 1 + tau) / dn - 1.5
        out += np.where(ok, wq[q] * (a1 * p[q, ki + 1] + a0 * p[q, ki]), 0.0)
    return out


def fbp(w, p, weights):
    """Eq. (27) on every node of the grid: returns (nz, ny, nx)."""
    pts = node_positions(w).reshape(-1, 3)
    return fbp_points(w, p, weights, pts).reshape(w.nz, w.ny, w.nx)


def weights(w, areas):
    """Reading G23: w_q = -dS_q / (4 pi^2 kappa c0^3 dt R_q), the constant of Eq. (27) L221 with kappa = beta/(4 pi C_p)
    (Eq. 3) and R_q = |r_q - centre| the radius of the measurement sphere (L203); `areas` = the patch areas dS_q."""
    tr = np.asarray(w.trans_xyz, dtype=np.float64)
    r = np.sqrt(np.sum((tr - np.asarray(w.centre, dtype=np.float64)) ** 2, axis=1))
    return -np.asarray(areas, dtype=np.float64) / (4.0 * np.pi ** 2 * w.gain * w.c ** 3 * w.dt * r)


def interval_margin(w, pts):
    """min over transducers of |k~ - nearest integer| at each point (M,): where it is below the rounding noise of k~
    (~1e-12) the choice of interval k = floor(k~) is a tie -- Eq. (27) is discontinuous across integer k~, both
    neighbouring intervals are correct results -- and a parity test compares only the points where it is not."""
    pts = np.asarray(pts, dtype=np.float64)
    tr = np.asarray(w.trans_xyz, dtype=np.float64)
    m = np.full(pts.shape[0], np.inf)
    for q in range(tr.shape[0]):
        kt = (np.sqrt(np.sum((pts - tr[q]) ** 2, axis=1)) / w.c - w.t0) / w.dt
        inrec = (kt > -1.0) & (kt < w.nt)
        m = np.minimum(m, np.where(inrec, np.abs(kt - np.rint(kt)), np.inf))
    return m
