"""oat_penalty_value_noalloc: the penalty R(x) = x^T L x (Eq. 34) for programs that cannot allocate.

Some users of liboat.so may not call cudaMalloc while they run: the application has already given all GPU memory to its
own pool, or it sits in an acquisition loop where the device-wide stall of an allocation is not acceptable.  The regular
oat_penalty_value needs a geometry handle and a lazily allocated scratch volume; the no-alloc entry point keeps its
scratch in a fixed array inside the library (8 MiB, at most OAT_NOALLOC_MAX_VOXELS = 2^21 voxels) and takes only the
volume and its dimensions.

What is checked here: on a GPU, two calls in a row (a large volume first, then a smaller, different one, so that stale
scratch contents from the first call would show in the second) return what the existing path returns, at the 1e-5
relative tolerance tests/test_gpu_pls.py uses for the penalty value; volumes over the limit are refused with a message
that names it.  The file name sorts last on purpose: pytest -x stops at the first failure, and a failure of this
add-on must not hide the parity tests.  It makes no assumption about earlier tests (it runs alone in a fresh process
as well as at the end of the whole suite).
"""
import ctypes

import numpy as np
import pytest


def test_noalloc_refuses_volumes_over_its_limit_without_a_gpu():
    """The size check comes before any CUDA call, so it can be exercised on a box without a GPU."""
    from paper_1304_2017_b200 import binding, build
    build.build()
    lib = binding.load()
    out = ctypes.c_double(-1.0)
    dummy = ctypes.c_void_p(256)                      # never dereferenced: the call is refused on its sizes alone
    rc = lib.oat_penalty_value_noalloc(129, 128, 128, dummy, ctypes.byref(out), None)
    assert rc == binding.OAT_ERR_INVALID
    msg = binding.oat_last_error()
    assert "OAT_NOALLOC_MAX_VOXELS" in msg and str(binding.OAT_NOALLOC_MAX_VOXELS) in msg
    assert out.value == -1.0                          # nothing was written
    assert lib.oat_penalty_value_noalloc(0, 4, 4, dummy, ctypes.byref(out), None) == binding.OAT_ERR_INVALID
    assert lib.oat_penalty_value_noalloc(4, 4, 4, None, ctypes.byref(out), None) == binding.OAT_ERR_INVALID
    assert lib.oat_penalty_value_noalloc(4, 4, 4, dummy, None, None) == binding.OAT_ERR_INVALID
    header = open(build.CSRC.parent.parent / "include" / "oat.h").read()
    assert f"#define OAT_NOALLOC_MAX_VOXELS (1 << {binding.OAT_NOALLOC_MAX_VOXELS.bit_length() - 1})" in header


@pytest.mark.gpu
def test_noalloc_penalty_matches_the_allocating_path_on_two_calls_in_a_row():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1304_2017_b200 import binding as oat, build, workloads as wl
    build.build()

    def existing_path(x):
        """oat_penalty_value on a handle whose grid has x's shape (one far transducer; the penalty ignores it)."""
        nz, ny, nx = x.shape
        w = wl.Workload("pen", nx, ny, nz, 0.5, (-1.0, -1.0, -1.0), np.array([[100.0, 1.0, 2.0]]), c=1.5, t0=1.0, dt=0.1,
                        nt=8, surf_step=0.5, kband=8)
        g = oat.oat_geometry_create(w)
        try:
            return oat.oat_penalty_value(g, x)
        finally:
            g.close()

    rng = np.random.default_rng(20171304)
    # first call: the largest volume the entry point takes (128^3 fills the whole scratch array);
    # second call: a smaller, ragged, different volume -- leftovers of the first call lie beyond and inside its range
    shapes = [(128, 128, 128), (37, 61, 45)]
    volumes = [torch.from_numpy(rng.standard_normal(s).astype(np.float32)).cuda() for s in shapes]
    expected = [existing_path(x) for x in volumes]
    got = [oat.oat_penalty_value_noalloc(x) for x in volumes]             # two calls in a row, nothing in between
    for s, r, e in zip(shapes, got, expected):
        assert e > 0 and abs(r - e) <= 1e-5 * e, (s, r, e)
    # the same volume again gives the same value: the accumulator really is cleared per call
    again = oat.oat_penalty_value_noalloc(volumes[1])
    assert abs(again - expected[1]) <= 1e-5 * expected[1]
    # a constant volume has no differences at all: R = 0 exactly, whatever the array held before
    assert oat.oat_penalty_value_noalloc(torch.full((16, 16, 16), 3.0, device="cuda")) == 0.0

    too_big = torch.zeros((129, 128, 128), dtype=torch.float32, device="cuda")
    with pytest.raises(oat.OatError) as ei:
        oat.oat_penalty_value_noalloc(too_big)
    assert ei.value.code == oat.OAT_ERR_INVALID and "OAT_NOALLOC_MAX_VOXELS" in str(ei.value)
    with pytest.raises(oat.OatError):                                     # host memory is refused, not dereferenced
        out = ctypes.c_double()
        host = np.zeros(64, dtype=np.float32)
        oat._check(oat.load().oat_penalty_value_noalloc(4, 4, 4, ctypes.c_void_p(host.ctypes.data), ctypes.byref(out), None))

