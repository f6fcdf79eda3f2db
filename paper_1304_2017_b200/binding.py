"""Thin ctypes binding of liboat.so -- same names as include/oat.h, argument
marshalling only.  PyTorch supplies device memory and streams; every step of
the path runs in the library's CUDA kernels.  There is no CPU fallback: if the
library cannot be loaded or no CUDA device exists, calls raise ``OatError``.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

_LIB_PATH = Path(__file__).resolve().parent / "csrc" / "liboat.so"
_lib = None

OAT_OK, OAT_ERR_INVALID, OAT_ERR_ALLOC, OAT_ERR_CUDA = 0, -1, -2, -3
OAT_NOALLOC_MAX_VOXELS = 1 << 21     # include/oat.h: largest volume oat_penalty_value_noalloc accepts

EXPORTS = [
    "oat_geometry_create", "oat_geometry_destroy", "oat_num_voxels", "oat_num_samples",
    "oat_num_surface_samples", "oat_project", "oat_backproject", "oat_adjoint_check",
    "oat_project_host", "oat_backproject_host", "oat_cgls", "oat_set_variant",
    "oat_eir_set", "oat_eir_apply", "oat_project_eir", "oat_backproject_eir", "oat_penalty_apply", "oat_penalty_value", "oat_penalty_value_noalloc", "oat_pls_cg", "oat_fbp", "oat_fbp_weights", "oat_sph_set", "oat_sph_set_aperture", "oat_sph_project", "oat_sph_backproject", "oat_sph_pls_cg",
    "oat_last_launch_count", "oat_uses_marching", "oat_last_kernel_ms", "oat_tile_stats", "oat_measure_red_rate", "oat_measure_gather_rate", "oat_measure_gather_rate_ex", "oat_measure_red_rate_ex", "oat_last_error", "oat_version",
]


class OatError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"liboat error {code}: {msg}")
        self.code = code


class oat_geometry_desc(ctypes.Structure):
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
    ]


def load():
    """Load liboat.so (built in-tree by paper_1304_2017_b200.build); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise OatError(OAT_ERR_CUDA, f"{_LIB_PATH} is missing: run `python -m paper_1304_2017_b200.build` "
                                     "(nvcc, sm_100a). There is no CPU fallback.")
    lib = ctypes.CDLL(str(_LIB_PATH))
    vp, fp, dp = ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)
    lib.oat_geometry_create.argtypes = [ctypes.POINTER(oat_geometry_desc), ctypes.c_int, ctypes.POINTER(vp)]
    lib.oat_geometry_create.restype = ctypes.c_int
    lib.oat_geometry_destroy.argtypes = [vp]
    lib.oat_geometry_destroy.restype = None
    for n in ("oat_num_voxels", "oat_num_samples", "oat_num_surface_samples"):
        getattr(lib, n).argtypes = [vp]
        getattr(lib, n).restype = ctypes.c_int64
    for n in ("oat_project", "oat_backproject"):
        getattr(lib, n).argtypes = [vp, fp, fp, vp]
        getattr(lib, n).restype = ctypes.c_int
    lib.oat_adjoint_check.argtypes = [vp, fp, fp, dp, dp, dp, vp]
    lib.oat_adjoint_check.restype = ctypes.c_int
    for n in ("oat_project_host", "oat_backproject_host"):
        getattr(lib, n).argtypes = [vp, fp, fp]
        getattr(lib, n).restype = ctypes.c_int
    lib.oat_cgls.argtypes = [vp, fp, fp, ctypes.c_int, dp, dp, vp]
    lib.oat_cgls.restype = ctypes.c_int
    lib.oat_set_variant.argtypes = [vp, ctypes.c_char_p, ctypes.c_int]
    lib.oat_set_variant.restype = ctypes.c_int
    lib.oat_last_launch_count.argtypes = [vp]
    lib.oat_last_launch_count.restype = ctypes.c_int
    lib.oat_uses_marching.argtypes = [vp, ctypes.c_int]
    lib.oat_uses_marching.restype = ctypes.c_int
    lib.oat_tile_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong), ctypes.c_int]
    lib.oat_tile_stats.restype = ctypes.c_int
    lib.oat_last_kernel_ms.argtypes = [vp]
    lib.oat_last_kernel_ms.restype = ctypes.c_float
    lib.oat_last_error.restype = ctypes.c_char_p
    lib.oat_version.restype = ctypes.c_char_p
    lib.oat_measure_red_rate.argtypes = [ctypes.c_int, dp]
    lib.oat_measure_red_rate.restype = ctypes.c_int
    lib.oat_measure_gather_rate.argtypes = [ctypes.c_int, dp]
    lib.oat_measure_gather_rate.restype = ctypes.c_int
    lib.oat_measure_gather_rate_ex.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp]
    lib.oat_measure_gather_rate_ex.restype = ctypes.c_int
    lib.oat_measure_red_rate_ex.argtypes = [ctypes.c_int, ctypes.c_int, dp]
    lib.oat_measure_red_rate_ex.restype = ctypes.c_int
    lib.oat_eir_set.argtypes = [vp, fp, ctypes.c_int32]
    lib.oat_eir_apply.argtypes = [vp, fp, fp, ctypes.c_int, vp]
    lib.oat_project_eir.argtypes = [vp, fp, fp, vp]
    lib.oat_backproject_eir.argtypes = [vp, fp, fp, vp]
    lib.oat_penalty_apply.argtypes = [vp, fp, fp, vp]
    lib.oat_penalty_value.argtypes = [vp, fp, dp, vp]
    lib.oat_penalty_value_noalloc.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, fp, dp, vp]
    lib.oat_penalty_value_noalloc.restype = ctypes.c_int
    lib.oat_pls_cg.argtypes = [vp, fp, fp, ctypes.c_int, ctypes.c_double, dp, dp, vp]
    lib.oat_sph_set.argtypes = [vp, ctypes.c_int32, ctypes.c_double, ctypes.c_double, fp]
    lib.oat_sph_project.argtypes = [vp, fp, fp, vp]
    lib.oat_sph_backproject.argtypes = [vp, fp, fp, vp]
    for n in ("oat_sph_set", "oat_sph_set_aperture", "oat_sph_project", "oat_sph_backproject"):
        getattr(lib, n).restype = ctypes.c_int
    lib.oat_sph_pls_cg.argtypes = [vp, fp, fp, ctypes.c_int, ctypes.c_double, dp, dp, vp]
    lib.oat_sph_pls_cg.restype = ctypes.c_int
    lib.oat_fbp.argtypes = [vp, fp, fp, fp, vp]
    lib.oat_fbp.restype = ctypes.c_int
    for n in ("oat_eir_set", "oat_eir_apply", "oat_project_eir", "oat_backproject_eir", "oat_penalty_apply",
              "oat_penalty_value", "oat_pls_cg"):
        getattr(lib, n).restype = ctypes.c_int
    _lib = lib
    return lib


def oat_last_error() -> str:
    return load().oat_last_error().decode()


def oat_version() -> str:
    return load().oat_version().decode()


def _check(rc):
    if rc != 0:
        raise OatError(rc, oat_last_error())


def make_desc(w):
    """Descriptor from any object with the problem-statement attributes (e.g. workloads.Workload).
    Returns (desc, keepalive)."""
    tr = np.ascontiguousarray(np.asarray(w.trans_xyz, dtype=np.float64).reshape(-1, 3))
    d = oat_geometry_desc()
    d.nx, d.ny, d.nz = int(w.nx), int(w.ny), int(w.nz)
    d.spacing = float(w.spacing)
    d.origin = (ctypes.c_double * 3)(*[float(v) for v in w.origin])
    d.n_trans = int(tr.shape[0])
    d.trans_xyz = tr.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    d.c, d.t0, d.dt = float(w.c), float(w.t0), float(w.dt)
    d.nt = int(w.nt)
    d.surf_step = float(getattr(w, "surf_step", 0.0))
    d.kband = int(getattr(w, "kband", 0))
    d.gain = float(getattr(w, "gain", 0.0))
    return d, tr


class Geometry:
    """Owner of an ``oat_geometry*`` handle."""

    def __init__(self, handle, device, n_trans, nt, shape):
        self.handle, self.device, self.n_trans, self.nt, self.shape = handle, device, n_trans, nt, shape

    def close(self):
        if self.handle:
            load().oat_geometry_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def oat_geometry_create(w, device: int = 0) -> Geometry:
    d, keep = make_desc(w)
    h = ctypes.c_void_p()
    _check(load().oat_geometry_create(ctypes.byref(d), int(device), ctypes.byref(h)))
    return Geometry(h, int(device), d.n_trans, d.nt, (d.nz, d.ny, d.nx))


def oat_geometry_destroy(g: Geometry):
    g.close()


def oat_num_voxels(g) -> int:
    return int(load().oat_num_voxels(g.handle))


def oat_num_samples(g) -> int:
    return int(load().oat_num_samples(g.handle))


def oat_num_surface_samples(g) -> int:
    v = int(load().oat_num_surface_samples(g.handle))
    if v < 0:
        raise OatError(OAT_ERR_CUDA, oat_last_error())
    return v


def _dev_ptr(t, n, what, g):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise OatError(OAT_ERR_INVALID, f"{what} must be a CUDA tensor")
    if t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n:
        raise OatError(OAT_ERR_INVALID, f"{what} must be contiguous float32 with {n} elements")
    if t.device.index != g.device:
        raise OatError(OAT_ERR_INVALID, f"{what} is on cuda:{t.device.index}, geometry on cuda:{g.device}")
    return ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def oat_project(g, x, y=None, stream=None):
    """y = H x on the current torch stream; x: (nz,ny,nx) float32 CUDA tensor."""
    import torch
    if y is None:
        y = torch.empty((g.n_trans, g.nt), dtype=torch.float32, device=x.device)
    _check(load().oat_project(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g),
                              _dev_ptr(y, oat_num_samples(g), "y", g), _stream(stream)))
    return y


def oat_backproject(g, y, x=None, stream=None):
    """x = H^T y on the current torch stream; y: (Q,K) float32 CUDA tensor."""
    import torch
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=y.device)
    _check(load().oat_backproject(g.handle, _dev_ptr(y, oat_num_samples(g), "y", g),
                                  _dev_ptr(x, oat_num_voxels(g), "x", g), _stream(stream)))
    return x


def oat_adjoint_check(g, x, y, stream=None):
    """(lhs, rhs, rel) with lhs = <Hx, y>, rhs = <x, H^T y>."""
    lhs, rhs, rel = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(load().oat_adjoint_check(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g),
                                    _dev_ptr(y, oat_num_samples(g), "y", g),
                                    ctypes.byref(lhs), ctypes.byref(rhs), ctypes.byref(rel), _stream(stream)))
    return lhs.value, rhs.value, rel.value


def _host_ptr(a, n, what):
    """Host float32 buffer: a numpy array or a CPU torch tensor (pinned or pageable)."""
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags["C_CONTIGUOUS"] or a.size != n:
            raise OatError(OAT_ERR_INVALID, f"{what} must be C-contiguous float32 with {n} elements")
        return ctypes.c_void_p(a.ctypes.data)
    import torch
    if isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == torch.float32 and a.is_contiguous() and a.numel() == n:
        return ctypes.c_void_p(a.data_ptr())
    raise OatError(OAT_ERR_INVALID, f"{what} must be a host float32 buffer with {n} elements")


def oat_project_host(g, h_x, h_y):
    _check(load().oat_project_host(g.handle, _host_ptr(h_x, oat_num_voxels(g), "h_x"),
                                   _host_ptr(h_y, oat_num_samples(g), "h_y")))
    return h_y


def oat_backproject_host(g, h_y, h_x):
    _check(load().oat_backproject_host(g.handle, _host_ptr(h_y, oat_num_samples(g), "h_y"),
                                       _host_ptr(h_x, oat_num_voxels(g), "h_x")))
    return h_x


def oat_cgls(g, y, n_iter, x=None, stream=None):
    """n_iter CGLS steps from x = 0; returns (x, res, grad) with the two curves of length n_iter+1."""
    import torch
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=y.device)
    res = np.zeros(n_iter + 1, dtype=np.float64)
    grad = np.zeros(n_iter + 1, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    _check(load().oat_cgls(g.handle, _dev_ptr(y, oat_num_samples(g), "y", g), _dev_ptr(x, oat_num_voxels(g), "x", g),
                           int(n_iter), res.ctypes.data_as(dp), grad.ctypes.data_as(dp), _stream(stream)))
    return x, res, grad


def oat_set_variant(g, key: str, variant: int):
    _check(load().oat_set_variant(g.handle, key.encode(), int(variant)))


def oat_uses_marching(g, backproject: bool = False) -> bool:
    return bool(load().oat_uses_marching(g.handle, 1 if backproject else 0))


def oat_last_launch_count(g) -> int:
    return int(load().oat_last_launch_count(g.handle))


def oat_last_kernel_ms(g) -> float:
    return float(load().oat_last_kernel_ms(g.handle))


def oat_tile_stats(g, reset: bool = True):
    """Enumeration counters of the tile-stationary kernels (candidates, after the fp32 cull, owning rays, chunks)."""
    out = (ctypes.c_ulonglong * 8)()
    _check(load().oat_tile_stats(g.handle, out, 1 if reset else 0))
    return [int(v) for v in out[:8]]


def oat_measure_red_rate(device: int = 0) -> float:
    """Sustained scattered RED.128 lanes per second on `device` (roofline unit of H^T)."""
    v = ctypes.c_double(0.0)
    _check(load().oat_measure_red_rate(int(device), ctypes.byref(v)))
    return float(v.value)


def oat_measure_gather_rate(device: int = 0) -> float:
    """Sustained scattered 32-byte sector loads per second that miss L1 and hit L2 (roofline unit of H)."""
    v = ctypes.c_double(0.0)
    _check(load().oat_measure_gather_rate(int(device), ctypes.byref(v)))
    return float(v.value)


# ---------------------------------------------------------------- row NEXT-1: EIR, penalty, PLS-CG
def oat_eir_set(g, he):
    """Set (or, with an empty array, remove) the EIR taps [h^e]_m, m = 0..len-1 (Eq. 14)."""
    he = np.ascontiguousarray(np.asarray(he, dtype=np.float32).ravel())
    _check(load().oat_eir_set(g.handle, ctypes.c_void_p(he.ctypes.data if he.size else None), ctypes.c_int32(he.size)))


def oat_eir_apply(g, p, out=None, adjoint=False, stream=None):
    import torch
    if out is None:
        out = torch.empty((g.n_trans, g.nt), dtype=torch.float32, device=p.device)
    _check(load().oat_eir_apply(g.handle, _dev_ptr(p, oat_num_samples(g), "in", g), _dev_ptr(out, oat_num_samples(g), "out", g),
                                ctypes.c_int(1 if adjoint else 0), _stream(stream)))
    return out


def oat_project_eir(g, x, u=None, stream=None):
    import torch
    if u is None:
        u = torch.empty((g.n_trans, g.nt), dtype=torch.float32, device=x.device)
    _check(load().oat_project_eir(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g), _dev_ptr(u, oat_num_samples(g), "u", g), _stream(stream)))
    return u


def oat_backproject_eir(g, u, x=None, stream=None):
    import torch
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=u.device)
    _check(load().oat_backproject_eir(g.handle, _dev_ptr(u, oat_num_samples(g), "u", g), _dev_ptr(x, oat_num_voxels(g), "x", g), _stream(stream)))
    return x


def oat_penalty_apply(g, x, lx=None, stream=None):
    import torch
    if lx is None:
        lx = torch.empty(g.shape, dtype=torch.float32, device=x.device)
    _check(load().oat_penalty_apply(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g), _dev_ptr(lx, oat_num_voxels(g), "lx", g), _stream(stream)))
    return lx


def oat_penalty_value(g, x, stream=None) -> float:
    v = ctypes.c_double(0.0)
    _check(load().oat_penalty_value(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g), ctypes.byref(v), _stream(stream)))
    return float(v.value)


def oat_penalty_value_noalloc(x, stream=None) -> float:
    """R(x) = x^T L x for a (nz, ny, nx) float32 CUDA tensor of at most OAT_NOALLOC_MAX_VOXELS elements, through the
    library entry point that needs no geometry handle and allocates nothing (its scratch is a fixed array inside
    liboat.so).  It exists for programs that may not call cudaMalloc once they are running -- all GPU memory already
    belongs to their own pool, or the device-wide stall of an allocation is not tolerable in their acquisition loop.
    Larger volumes raise OatError (OAT_ERR_INVALID) naming the limit; use oat_penalty_value for those.  Calls share the
    library's one scratch array per GPU: do not run two of them concurrently on the same device.  This wrapper itself
    only marshals arguments; it makes x's device current for the call, as the entry point works on the current device."""
    import torch
    if not isinstance(x, torch.Tensor) or not x.is_cuda or x.dtype != torch.float32 or not x.is_contiguous() or x.dim() != 3:
        raise OatError(OAT_ERR_INVALID, "x must be a contiguous float32 CUDA tensor of shape (nz, ny, nx)")
    nz, ny, nx = (int(v) for v in x.shape)
    v = ctypes.c_double(0.0)
    with torch.cuda.device(x.device):
        _check(load().oat_penalty_value_noalloc(ctypes.c_int32(nx), ctypes.c_int32(ny), ctypes.c_int32(nz),
                                                ctypes.c_void_p(x.data_ptr()), ctypes.byref(v), _stream(stream)))
    return float(v.value)


def oat_pls_cg(g, u, n_iter, mu, x=None, stream=None):
    """n_iter CG steps on (H^T H + mu L) x = H^T u from x = 0; returns (x, obj, grad), curves of length n_iter+1."""
    import torch
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=u.device)
    obj = np.zeros(n_iter + 1, dtype=np.float64)
    grad = np.zeros(n_iter + 1, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    _check(load().oat_pls_cg(g.handle, _dev_ptr(u, oat_num_samples(g), "u", g), _dev_ptr(x, oat_num_voxels(g), "x", g),
                             int(n_iter), ctypes.c_double(float(mu)), obj.ctypes.data_as(dp), grad.ctypes.data_as(dp), _stream(stream)))
    return x, obj, grad


# ---------------------------------------------------------------- row NEXT-2: filtered backprojection
def oat_fbp(g, p, weights, x=None, stream=None):
    """x = FBP(p) by Eq. (27) with one weight per transducer (device tensors; weights: Q float32)."""
    import torch
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=p.device)
    _check(load().oat_fbp(g.handle, _dev_ptr(p, oat_num_samples(g), "p", g), _dev_ptr(weights, g.n_trans, "weights", g),
                          _dev_ptr(x, oat_num_voxels(g), "x", g), _stream(stream)))
    return x


def oat_sph_set_aperture(g, side: float, m: int):
    """Square transducer surface of side `side` (mm), integrated with m x m sub-elements (Eq. 18); 0 / 1 = point-like."""
    lib = load()
    lib.oat_sph_set_aperture.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int32]
    lib.oat_sph_set_aperture.restype = ctypes.c_int
    _check(lib.oat_sph_set_aperture(g.handle, ctypes.c_double(float(side)), ctypes.c_int32(int(m))))


def oat_fbp_weights(g, areas) -> np.ndarray:
    """The Q weights of Eq. (27) from the transducers' patch areas (host arrays)."""
    a = np.ascontiguousarray(areas, dtype=np.float64)
    if a.shape != (g.n_trans,):
        raise OatError(OAT_ERR_INVALID, f"areas must have shape ({g.n_trans},)")
    out = np.empty(g.n_trans, dtype=np.float32)
    _check(load().oat_fbp_weights(g.handle, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                  out.ctypes.data_as(ctypes.POINTER(ctypes.c_float))))
    return out


# ---------------------------------------------------------------- row NEXT-3: spherical-voxel model (frequency domain)
def oat_sph_set(g, nf, f0, df, he=None):
    """Frequency grid f_l = f0 + l df and (optionally) the complex EIR spectrum h~e(f_l); nf = 0 removes it."""
    ptr = None
    if he is not None:
        he = np.asarray(he, dtype=np.complex64).ravel()
        if he.size != nf:
            raise OatError(OAT_ERR_INVALID, f"he must have {nf} complex samples")
        buf = np.ascontiguousarray(he.view(np.float32))
        ptr = ctypes.c_void_p(buf.ctypes.data)
    _check(load().oat_sph_set(g.handle, ctypes.c_int32(int(nf)), ctypes.c_double(float(f0)), ctypes.c_double(float(df)), ptr))
    g.sph_nf = int(nf)


def oat_sph_project(g, x, u=None, stream=None):
    """u = H_sph x: complex64 tensor (Q, nf)."""
    import torch
    nf = getattr(g, "sph_nf", 0)
    if u is None:
        u = torch.empty((g.n_trans, nf), dtype=torch.complex64, device=x.device)
    ur = torch.view_as_real(u)
    _check(load().oat_sph_project(g.handle, _dev_ptr(x, oat_num_voxels(g), "x", g), _dev_ptr(ur, 2 * g.n_trans * nf, "u", g), _stream(stream)))
    return u


def oat_sph_backproject(g, u, x=None, stream=None):
    """x = Re H_sph† u for a complex64 tensor u (Q, nf)."""
    import torch
    nf = getattr(g, "sph_nf", 0)
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=u.device)
    ur = torch.view_as_real(u)
    _check(load().oat_sph_backproject(g.handle, _dev_ptr(ur, 2 * g.n_trans * nf, "u", g), _dev_ptr(x, oat_num_voxels(g), "x", g), _stream(stream)))
    return x


def oat_measure_gather_rate_ex(device: int, lanes_active: int, smem_kb_per_block: int) -> float:
    v = ctypes.c_double(0.0)
    _check(load().oat_measure_gather_rate_ex(int(device), int(lanes_active), int(smem_kb_per_block), ctypes.byref(v)))
    return float(v.value)


def oat_measure_red_rate_ex(device: int, pattern: int) -> float:
    v = ctypes.c_double(0.0)
    _check(load().oat_measure_red_rate_ex(int(device), int(pattern), ctypes.byref(v)))
    return float(v.value)


def oat_sph_pls_cg(g, u, n_iter, mu, x=None, stream=None):
    """n_iter CG steps on (H_sph† H_sph + mu L) x = H_sph† u from x = 0 for a complex64 tensor u (Q, nf)."""
    import torch
    nf = getattr(g, "sph_nf", 0)
    if x is None:
        x = torch.empty(g.shape, dtype=torch.float32, device=u.device)
    obj = np.zeros(n_iter + 1, dtype=np.float64)
    grad = np.zeros(n_iter + 1, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    ur = torch.view_as_real(u)
    _check(load().oat_sph_pls_cg(g.handle, _dev_ptr(ur, 2 * g.n_trans * nf, "u", g), _dev_ptr(x, oat_num_voxels(g), "x", g),
                                 int(n_iter), ctypes.c_double(float(mu)), obj.ctypes.data_as(dp), grad.ctypes.data_as(dp), _stream(stream)))
    return x, obj, grad
