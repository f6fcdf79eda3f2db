"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the fp64 oracle's tests and the CUDA path's tests and
bench.  It holds none of the method's arithmetic: it only produces the problem
statement of the paper (voxel grid, spacing, transducer
positions, c, t0, dt, Nt) and seeded phantoms / data vectors.  The arrays made
here are handed unchanged to both sides, so no random stream has to match
across languages.

Stand-in statement: the paper's own numerical phantom (nine
blurred spheres whose parameters are never printed) and its live-mouse data set
(L291) are not available; these inputs take their shapes, sizes and value
structure (smooth-edged spheres, sparse vessel-like absorbers, 65 mm spherical /
arc aperture, 20 MHz sampling, 0.2-0.5 mm grids).

Layout conventions (SURVEY.md §8 notation): volumes are float32 arrays of shape
(nz, ny, nx), x fastest; data vectors have shape (Q, K), time fastest
(index q*K + k).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np


# --------------------------------------------------------------------------
# problem statement
# --------------------------------------------------------------------------
@dataclass
class Workload:
    """One acquisition geometry + reconstruction grid."""
    name: str
    nx: int
    ny: int
    nz: int
    spacing: float            # Delta_s, mm
    origin: tuple             # position of node (0,0,0) = (x_min, y_min, z_min), mm
    trans_xyz: np.ndarray     # (Q, 3) float64 transducer positions r_q^s, mm
    c: float                  # speed of sound, mm/us
    t0: float                 # time of sample k = 0 (t_min), us
    dt: float                 # sampling interval, us
    nt: int                   # K
    surf_step: float          # h: surface-patch size of Eq. (37), mm
    kband: int = 32           # B: time samples sharing one angular rule (reading G11)
    gain: float = 1.0         # kappa = beta / (4 pi C_p)
    seed: int = 0
    phantom_spec: dict = field(default_factory=dict)

    @property
    def n_trans(self) -> int:
        return int(self.trans_xyz.shape[0])

    @property
    def n_voxels(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def centre(self) -> np.ndarray:
        o = np.asarray(self.origin, dtype=np.float64)
        n = np.array([self.nx, self.ny, self.nz], dtype=np.float64)
        return o + self.spacing * (n - 1.0) / 2.0

    def subset(self, idx) -> "Workload":
        """Same problem restricted to the transducers ``idx`` (rows of H)."""
        idx = np.asarray(idx, dtype=np.int64)
        return replace(self, name=f"{self.name}[sub{len(idx)}]",
                       trans_xyz=np.ascontiguousarray(self.trans_xyz[idx]))

    def seeded_subset(self, n: int) -> tuple:
        """Seeded transducer subset of SURVEY.md §8(d): rng(seed+1000).choice."""
        rng = np.random.default_rng(self.seed + 1000)
        idx = np.sort(rng.choice(self.n_trans, size=min(n, self.n_trans), replace=False))
        return idx, self.subset(idx)

    def phantom(self) -> np.ndarray:
        return make_phantom(self)

    def data_noise(self, seed: Optional[int] = None) -> np.ndarray:
        """Seeded N(0,1) data vector (Q, K) for the adjoint test."""
        rng = np.random.default_rng(self.seed + 100 if seed is None else seed)
        return rng.standard_normal((self.n_trans, self.nt)).astype(np.float32)


# --------------------------------------------------------------------------
# transducer layouts
# --------------------------------------------------------------------------
def fibonacci_sphere(q: int, radius: float) -> np.ndarray:
    """z_i = 1 - (2i+1)/Q, phi_i = i*pi*(3 - sqrt 5)."""
    i = np.arange(q, dtype=np.float64)
    z = 1.0 - (2.0 * i + 1.0) / q
    phi = i * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return radius * np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def arc_array(n_elem: int, n_views: int, radius: float,
              polar0_deg: float = 14.0, span_deg: float = 152.0) -> np.ndarray:
    """n_elem elements on an arc in the x-z plane, rotated about z over n_views
    equally spaced views; q = e * n_views + v."""
    e = np.arange(n_elem, dtype=np.float64)
    pol = np.deg2rad(polar0_deg + e * span_deg / max(1, n_elem - 1))
    v = np.arange(n_views, dtype=np.float64)
    az = 2.0 * math.pi * v / n_views
    pol_g, az_g = np.meshgrid(pol, az, indexing="ij")          # (e, v)
    xyz = np.stack([radius * np.sin(pol_g) * np.cos(az_g),
                    radius * np.sin(pol_g) * np.sin(az_g),
                    radius * np.cos(pol_g)], axis=-1)
    return np.ascontiguousarray(xyz.reshape(-1, 3))


def patch_areas_equal(trans_xyz: np.ndarray, centre) -> np.ndarray:
    """Patch area dS_q of an (almost) uniform sampling of a full sphere, e.g. the Fibonacci layout: 4 pi R_q^2 / Q."""
    r = np.linalg.norm(np.asarray(trans_xyz, dtype=np.float64) - np.asarray(centre, dtype=np.float64), axis=1)
    return 4.0 * math.pi * r * r / max(1, len(r))


def patch_areas_arc(n_elem: int, n_views: int, radius: float, polar0_deg: float = 14.0, span_deg: float = 152.0) -> np.ndarray:
    """Patch area of the ring/view layout of `arc_array` (L203, L211): (R^s)^2 dtheta dphi sin(theta_q), q = e * n_views + v."""
    e = np.arange(n_elem, dtype=np.float64)
    pol = np.deg2rad(polar0_deg + e * span_deg / max(1, n_elem - 1))
    dth = np.deg2rad(span_deg / max(1, n_elem - 1))
    dph = 2.0 * math.pi / n_views
    return np.repeat(radius * radius * dth * dph * np.sin(pol), n_views)


def default_t0(trans_xyz: np.ndarray, n: int, spacing: float, c: float, dt: float) -> float:
    """t0 = dt * max(1, floor((min_q |r_q - C| - R_pad)/(c dt)) - 1) with
    R_pad = sqrt(3) * ((N-1) spacing / 2 + spacing); grid centred at the origin."""
    r_pad = math.sqrt(3.0) * ((n - 1) * spacing / 2.0 + spacing)
    dmin = float(np.min(np.linalg.norm(trans_xyz, axis=1)))
    return dt * max(1, math.floor((dmin - r_pad) / (c * dt)) - 1)


# --------------------------------------------------------------------------
# phantoms (rasterised on the nodes, Eq. (9), one-voxel soft edge)
# --------------------------------------------------------------------------
def _axes(w: Workload):
    ox, oy, oz = w.origin
    x = ox + w.spacing * np.arange(w.nx, dtype=np.float64)
    y = oy + w.spacing * np.arange(w.ny, dtype=np.float64)
    z = oz + w.spacing * np.arange(w.nz, dtype=np.float64)
    return x, y, z


def _box(axis: np.ndarray, lo: float, hi: float):
    i0 = int(np.searchsorted(axis, lo, side="left"))
    i1 = int(np.searchsorted(axis, hi, side="right"))
    return max(0, i0), min(len(axis), i1)


def _soft(d_inside: np.ndarray, spacing: float) -> np.ndarray:
    """clamp(0.5 + (R - dist)/spacing, 0, 1) with d_inside = R - dist."""
    return np.clip(0.5 + d_inside / spacing, 0.0, 1.0)


def add_ball(vol, w: Workload, centre, radius, amp):
    x, y, z = _axes(w)
    m = radius + w.spacing
    sx = _box(x, centre[0] - m, centre[0] + m)
    sy = _box(y, centre[1] - m, centre[1] + m)
    sz = _box(z, centre[2] - m, centre[2] + m)
    if sx[0] >= sx[1] or sy[0] >= sy[1] or sz[0] >= sz[1]:
        return
    zz, yy, xx = np.meshgrid(z[sz[0]:sz[1]], y[sy[0]:sy[1]], x[sx[0]:sx[1]], indexing="ij")
    dist = np.sqrt((xx - centre[0]) ** 2 + (yy - centre[1]) ** 2 + (zz - centre[2]) ** 2)
    vol[sz[0]:sz[1], sy[0]:sy[1], sx[0]:sx[1]] += amp * _soft(radius - dist, w.spacing)


def add_gaussian(vol, w: Workload, centre, sigma, amp):
    x, y, z = _axes(w)
    m = 5.0 * sigma
    sx = _box(x, centre[0] - m, centre[0] + m)
    sy = _box(y, centre[1] - m, centre[1] + m)
    sz = _box(z, centre[2] - m, centre[2] + m)
    if sx[0] >= sx[1] or sy[0] >= sy[1] or sz[0] >= sz[1]:
        return
    zz, yy, xx = np.meshgrid(z[sz[0]:sz[1]], y[sy[0]:sy[1]], x[sx[0]:sx[1]], indexing="ij")
    d2 = (xx - centre[0]) ** 2 + (yy - centre[1]) ** 2 + (zz - centre[2]) ** 2
    vol[sz[0]:sz[1], sy[0]:sy[1], sx[0]:sx[1]] += amp * np.exp(-d2 / (2.0 * sigma * sigma))


def add_cylinder(vol, w: Workload, mid, axis, radius, length, amp):
    x, y, z = _axes(w)
    axis = np.asarray(axis, dtype=np.float64)
    axis = axis / np.linalg.norm(axis)
    half = length / 2.0
    ext = np.abs(axis) * half + radius + w.spacing
    sx = _box(x, mid[0] - ext[0], mid[0] + ext[0])
    sy = _box(y, mid[1] - ext[1], mid[1] + ext[1])
    sz = _box(z, mid[2] - ext[2], mid[2] + ext[2])
    if sx[0] >= sx[1] or sy[0] >= sy[1] or sz[0] >= sz[1]:
        return
    zz, yy, xx = np.meshgrid(z[sz[0]:sz[1]], y[sy[0]:sy[1]], x[sx[0]:sx[1]], indexing="ij")
    dx, dy, dz = xx - mid[0], yy - mid[1], zz - mid[2]
    along = dx * axis[0] + dy * axis[1] + dz * axis[2]
    perp = np.sqrt(np.maximum(0.0, dx * dx + dy * dy + dz * dz - along * along))
    val = _soft(radius - perp, w.spacing) * _soft(half - np.abs(along), w.spacing)
    vol[sz[0]:sz[1], sy[0]:sy[1], sx[0]:sx[1]] += amp * val


def _unit_vectors(rng, n):
    v = rng.standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def make_phantom(w: Workload) -> np.ndarray:
    """Seeded non-negative phantom described by ``w.phantom_spec``; float32 (nz, ny, nx)."""
    spec = w.phantom_spec
    rng = np.random.default_rng(w.seed)
    vol = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    side = 0.7 * w.spacing * (min(w.nx, w.ny, w.nz) - 1)
    cen = w.centre

    def centres(n):
        if "centre_ball_mm" in spec:                     # config 1: within 5 mm of the origin
            r = spec["centre_ball_mm"] * rng.random(n) ** (1.0 / 3.0)
            return cen + r[:, None] * _unit_vectors(rng, n)
        return cen + side * (rng.random((n, 3)) - 0.5)

    nb = spec.get("balls", 0)
    if nb:
        c = centres(nb)
        lo, hi = spec.get("ball_radius", (1.0, 3.0))
        rad = rng.uniform(lo, hi, nb)
        amp = rng.uniform(0.5, 1.0, nb)
        for i in range(nb):
            add_ball(vol, w, c[i], rad[i], amp[i])
    ng = spec.get("gaussians", 0)
    if ng:
        c = centres(ng)
        lo, hi = spec.get("gauss_sigma", (0.3, 1.5))
        sig = rng.uniform(lo, hi, ng)
        amp = rng.uniform(0.3, 1.0, ng)
        for i in range(ng):
            add_gaussian(vol, w, c[i], sig[i], amp[i])
    nc = spec.get("cylinders", 0)
    if nc:
        c = centres(nc)
        ax = _unit_vectors(rng, nc)
        lo, hi = spec.get("cyl_radius", (0.2, 1.0))
        rad = rng.uniform(lo, hi, nc)
        l0, l1 = spec.get("cyl_length", (5.0, 30.0))
        ln = rng.uniform(l0, l1, nc)
        amp = rng.uniform(0.3, 1.0, nc)
        for i in range(nc):
            add_cylinder(vol, w, c[i], ax[i], rad[i], ln[i], amp[i])
    return np.ascontiguousarray(vol.astype(np.float32))


# --------------------------------------------------------------------------
# the five configs of BASELINE.json (readings of SURVEY.md §8(d))
# --------------------------------------------------------------------------
def _centred_origin(n: int, spacing: float) -> tuple:
    o = -(n - 1) * spacing / 2.0
    return (o, o, o)


def config(index: int) -> Workload:
    """index 1..5 as in BASELINE.json ``configs`` (config 4 = config-2 geometry,
    used for the CG loop)."""
    if index == 1:
        n, ds = 32, 0.5
        tr = fibonacci_sphere(64, 30.0)
        return Workload("cfg1-tiny", n, n, n, ds, _centred_origin(n, ds), tr,
                        c=1.5, t0=14.0, dt=0.05, nt=256, surf_step=0.25, seed=1,
                        phantom_spec=dict(balls=3, ball_radius=(1.0, 3.0), centre_ball_mm=5.0))
    if index in (2, 4):
        n, ds = 128, 0.2
        tr = fibonacci_sphere(1024, 40.0)
        t0 = default_t0(tr, n, ds, 1.5, 0.05)
        return Workload("cfg2-mid" if index == 2 else "cfg4-cg", n, n, n, ds,
                        _centred_origin(n, ds), tr, c=1.5, t0=t0, dt=0.05, nt=1024,
                        surf_step=ds, seed=2,
                        phantom_spec=dict(balls=20, ball_radius=(0.5, 4.0), gaussians=10,
                                          gauss_sigma=(0.3, 1.5)))
    if index == 3:
        n, ds = 240, 0.25
        tr = arc_array(64, 144, 65.0, 14.0, 152.0)
        t0 = default_t0(tr, n, ds, 1.5, 0.05)
        return Workload("cfg3-arc", n, n, n, ds, _centred_origin(n, ds), tr,
                        c=1.5, t0=t0, dt=0.05, nt=2048, surf_step=ds, seed=3,
                        phantom_spec=dict(cylinders=40, cyl_radius=(0.2, 1.0),
                                          cyl_length=(5.0, 30.0), balls=5,
                                          ball_radius=(1.0, 3.0)))
    if index == 5:
        n, ds = 256, 0.2
        tr = fibonacci_sphere(4096, 50.0)
        t0 = default_t0(tr, n, ds, 1.5, 0.025)
        return Workload("cfg5-stress", n, n, n, ds, _centred_origin(n, ds), tr,
                        c=1.5, t0=t0, dt=0.025, nt=4096, surf_step=ds, seed=5,
                        phantom_spec=dict(balls=60, ball_radius=(0.5, 4.0), gaussians=30,
                                          gauss_sigma=(0.3, 1.5), cylinders=40,
                                          cyl_radius=(0.2, 1.0), cyl_length=(5.0, 30.0)))
    raise ValueError(f"no such config: {index}")


def small(n: int = 12, q: int = 3, nt: int = 48, spacing: float = 0.5, radius: float = 12.0,
          h: Optional[float] = None, kband: int = 8, seed: int = 7, dt: float = 0.1,
          c: float = 1.5) -> Workload:
    """A small non-cubic-friendly test problem (ragged tails: nt not a multiple
    of kband is allowed) whose shells cover the whole grid."""
    tr = fibonacci_sphere(max(q, 1), radius)[:q]
    t0 = default_t0(tr, n, spacing, c, dt)
    return Workload(f"small{n}", n, n, n, spacing, _centred_origin(n, spacing), tr,
                    c=c, t0=t0, dt=dt, nt=nt, surf_step=spacing if h is None else h,
                    kband=kband, seed=seed,
                    phantom_spec=dict(balls=2, ball_radius=(0.8, 2.0),
                                      centre_ball_mm=0.25 * n * spacing,
                                      gaussians=1, gauss_sigma=(0.5, 1.0)))
