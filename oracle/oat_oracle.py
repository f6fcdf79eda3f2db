"""ctypes front end of the fp64 CPU oracle (oracle/oat_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from the CUDA package; problems are passed in as plain
attributes (nx, ny, nz, spacing, origin, trans_xyz, c, t0, dt, nt, surf_step,
kband, gain) -- e.g. a ``workloads.Workload``.

All arrays are float64 on the host.  Volumes have shape (nz, ny, nx), data
vectors (Q, K).  Passages followed are cited in oat_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oat_oracle.c"
_LIB = _HERE / "liboat_oracle.so"
_lib = None


class _Desc(ctypes.Structure):
    _fields_ = [
        ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
        ("spacing", ctypes.c_double),
        ("origin", ctypes.c_double * 3),
        ("n_trans", ctypes.c_int32),
        ("trans_xyz", ctypes.POINTER(ctypes.c_double)),
        ("c", ctypes.c_double), ("t0", ctypes.c_double), ("dt", ctypes.c_double),
        ("nt", ctypes.c_int32),
        ("surf_step", ctypes.c_double),
        ("kband", ctypes.c_int32),
        ("gain", ctypes.c_double),
        ("literal", ctypes.c_int32),
        ("n_threads", ctypes.c_int32),
    ]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain C, OpenMP over transducers)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=gnu11",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        dp = ctypes.POINTER(ctypes.c_double)
        pd = ctypes.POINTER(_Desc)
        for name in ("oat_ref_srt", "oat_ref_srt_adjoint", "oat_ref_diff", "oat_ref_diff_adjoint",
                     "oat_ref_project", "oat_ref_backproject"):
            fn = getattr(lib, name)
            fn.argtypes = [pd, dp, dp]
            fn.restype = ctypes.c_int
        lib.oat_ref_count_samples.argtypes = [pd, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)]
        lib.oat_ref_count_samples.restype = ctypes.c_int
        lib.oat_ref_weight_sum.argtypes = [pd, ctypes.c_int, dp, ctypes.POINTER(ctypes.c_int64)]
        lib.oat_ref_weight_sum.restype = ctypes.c_int
        lib.oat_ref_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oat_ref_max_threads())


def _desc(w, literal=False, n_threads=0, kband=None, surf_step=None):
    tr = np.ascontiguousarray(np.asarray(w.trans_xyz, dtype=np.float64).reshape(-1, 3))
    d = _Desc()
    d.nx, d.ny, d.nz = int(w.nx), int(w.ny), int(w.nz)
    d.spacing = float(w.spacing)
    d.origin = (ctypes.c_double * 3)(*[float(v) for v in w.origin])
    d.n_trans = int(tr.shape[0])
    d.trans_xyz = tr.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    d.c, d.t0, d.dt = float(w.c), float(w.t0), float(w.dt)
    d.nt = int(w.nt)
    d.surf_step = float(w.surf_step if surf_step is None else surf_step)
    d.kband = int(w.kband if kband is None else kband)
    d.gain = float(getattr(w, "gain", 1.0))
    d.literal = 1 if literal else 0
    d.n_threads = int(n_threads)
    return d, tr          # keep ``tr`` alive while ``d`` is in use


def _ptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def _vol(w, x):
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    assert x.size == w.nx * w.ny * w.nz, "volume size"
    return x


def _dat(w, y):
    q = np.asarray(w.trans_xyz).reshape(-1, 3).shape[0]
    y = np.ascontiguousarray(np.asarray(y, dtype=np.float64))
    assert y.size == q * w.nt, "data size"
    return y, q


def srt(w, x, **kw):
    """g = G x (S5)."""
    d, keep = _desc(w, **kw); x = _vol(w, x)
    g = np.zeros((d.n_trans, w.nt), dtype=np.float64)
    _check(_load().oat_ref_srt(ctypes.byref(d), _ptr(x), _ptr(g)), "srt")
    return g


def srt_adjoint(w, gp, **kw):
    """x = G^T g' (S8)."""
    d, keep = _desc(w, **kw); gp, _ = _dat(w, gp)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    _check(_load().oat_ref_srt_adjoint(ctypes.byref(d), _ptr(gp), _ptr(x)), "srt_adjoint")
    return x


def diff(w, g, **kw):
    """p = D g (S6)."""
    d, keep = _desc(w, **kw); g, q = _dat(w, g)
    p = np.zeros((q, w.nt), dtype=np.float64)
    _check(_load().oat_ref_diff(ctypes.byref(d), _ptr(g), _ptr(p)), "diff")
    return p


def diff_adjoint(w, y, **kw):
    """g' = D^T y (S7)."""
    d, keep = _desc(w, **kw); y, q = _dat(w, y)
    gp = np.zeros((q, w.nt), dtype=np.float64)
    _check(_load().oat_ref_diff_adjoint(ctypes.byref(d), _ptr(y), _ptr(gp)), "diff_adjoint")
    return gp


def project(w, x, **kw):
    """y = H x = D G x."""
    d, keep = _desc(w, **kw); x = _vol(w, x)
    y = np.zeros((d.n_trans, w.nt), dtype=np.float64)
    _check(_load().oat_ref_project(ctypes.byref(d), _ptr(x), _ptr(y)), "project")
    return y


def backproject(w, y, **kw):
    """x = H^T y = G^T D^T y."""
    d, keep = _desc(w, **kw); y, _ = _dat(w, y)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    _check(_load().oat_ref_backproject(ctypes.byref(d), _ptr(y), _ptr(x)), "backproject")
    return x


def count_samples(w, per_qk=False, **kw):
    """In-box quadrature samples: total, or an int64 (Q, K) array."""
    d, keep = _desc(w, **kw)
    tot = ctypes.c_int64(0)
    arr = np.zeros((d.n_trans, w.nt), dtype=np.int64) if per_qk else None
    p = arr.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)) if per_qk else None
    _check(_load().oat_ref_count_samples(ctypes.byref(d), p, ctypes.byref(tot)), "count_samples")
    return arr if per_qk else int(tot.value)


def weight_sum(w, k, **kw):
    """(sum of solid-angle weights over the whole sphere, number of directions) for k's band."""
    d, keep = _desc(w, **kw)
    s = ctypes.c_double(0); n = ctypes.c_int64(0)
    _check(_load().oat_ref_weight_sum(ctypes.byref(d), int(k), ctypes.byref(s), ctypes.byref(n)), "weight_sum")
    return float(s.value), int(n.value)


def cgls(w, y, n_iter, **kw):
    """Row C1 / reading G15: CGLS on min ||y - Hx||^2 from x0 = 0, fixed n_iter.

    r = y - Hx; s = H^T r; p = s; loop { q = Hp; alpha = |s|^2/|q|^2; x += alpha p;
    r -= alpha q; s = H^T r; beta = |s|^2_new/|s|^2_old; p = s + beta p }
    (the paper names only "linear CG" with refs, L265, L429-430).
    Returns x and the curves ||y - H x_i|| / ||y|| and ||H^T (y - H x_i)||, i = 0..n_iter.
    """
    y = np.asarray(y, dtype=np.float64)
    x = np.zeros((w.nz, w.ny, w.nx), dtype=np.float64)
    r = y.copy()
    s = backproject(w, r, **kw)
    p = s.copy()
    gamma = float(np.vdot(s, s))
    ynorm = float(np.linalg.norm(y))
    res = [float(np.linalg.norm(r)) / ynorm]
    grad = [gamma ** 0.5]
    for _ in range(n_iter):
        q = project(w, p, **kw)
        qq = float(np.vdot(q, q))
        if qq == 0.0:
            res.append(res[-1]); grad.append(grad[-1]); continue
        alpha = gamma / qq
        x += alpha * p
        r -= alpha * q
        s = backproject(w, r, **kw)
        gamma_new = float(np.vdot(s, s))
        beta = gamma_new / gamma if gamma > 0 else 0.0
        gamma = gamma_new
        p = s + beta * p
        res.append(float(np.linalg.norm(r)) / ynorm)
        grad.append(gamma ** 0.5)
    return x, np.array(res), np.array(grad)
