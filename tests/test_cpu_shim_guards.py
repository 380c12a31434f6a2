"""The "cannot hang, cannot fault" guards of the TMA kernels (csrc/tma_common.cuh), exercised on the host (`-m "not gpu"`).

The host-side test build of the kernel sources (tests/cpu_shim, compiled with -DCBCT_TEST_FAULTS) can inject deliberate
protocol mistakes; the product build cannot (the macro is never defined there and the injection points are the constant 0).
Each mistake must end as an ERROR STATUS of the handle -- not as a deadlock (which on a B200 is a hung SM, Xid 43) and not
as an out-of-range shared-memory access (an SM exception, Xid 13):

  1  the mbarrier is told to expect 16 bytes more than the TMA box delivers -> the bounded wait expires,
     CBCT_STATUS_WAIT_TIMEOUT, the kernel leaves through its normal exit path;
  2  the forward kernel's box does not cover its samples -> the per-chunk range check skips them, CBCT_STATUS_FORWARD_RANGE;
  4  the same for the scatter kernel -> CBCT_STATUS_BACKPROJECT_RANGE.

After the word is raised every hot call on the handle returns CBCT_E_DEVICE without launching; after a clear the handle
works again and matches the oracle.
"""
import ctypes as C
import math

import numpy as np
import pytest

from cpu_shim import shimlib as sl
from oracle import projector as op
from paper_1008_2042_b200 import binding as cb
from paper_1008_2042_b200 import synthetic as syn

G = syn.Geometry(44, 36, 12, 2.0, 2.5, 4.0, 53, 27, 2.1, 2.9, 1000.0, 1500.0,
                 (0.0, 0.3, math.pi / 4, 1.2, math.pi / 2, 2.2, 3.9, 5.0), ox=-3.0, oy=5.0, oz=1.5, u0=-2.2, v0=3.3, step_mm=0.9)


def fault_word():
    return C.c_int.in_dll(sl.lib(), "cbct_test_fault")


@pytest.fixture(autouse=True)
def _no_fault_left_behind():
    fault_word().value = 0
    sl.kernel_log()
    yield
    fault_word().value = 0
    sl.check(0, "end of test")


def rel_l2(a, ref):
    return float(np.linalg.norm(a.astype(np.float64).ravel() - ref.ravel()) / np.linalg.norm(ref.ravel()))


def _raw(h, name, src, out_shape):
    a, out = sl.dev(src), sl.Buf(out_shape)
    return getattr(sl.lib(), name)(h.handle, a.ptr, out.ptr, None), out


@pytest.mark.parametrize("tma_mode", ["eager", "lazy"])
def test_wrong_transaction_count_times_out_instead_of_hanging(monkeypatch, tma_mode):
    monkeypatch.setenv("SHIM_TMA", tma_mode)
    monkeypatch.setenv("SHIM_ALLOW_TX_MISMATCH", "1")      # otherwise the shim rejects the mismatch statically
    monkeypatch.setenv("CBCT_FORWARD_IMPL", "tma")
    h = sl.Geometry(G)
    x = syn.uniform_volume(G, 7)
    fault_word().value = 1
    status, _ = _raw(h, "cbct_forward", x, h.proj_shape)
    assert status == cb.CBCT_OK                              # launches are asynchronous: the launch itself succeeded
    sl.check(0, "forward with a wrong expect_tx")            # no deadlock, no rule violation reported by the shim
    assert any(k.startswith("cbct::forward_tma_kernel<") for k in sl.kernel_log())
    fault_word().value = 0
    # the next hot call refuses to launch: the mapped error word is already visible to the host
    status, _ = _raw(h, "cbct_forward", x, h.proj_shape)
    assert status == cb.CBCT_E_DEVICE
    assert sl.kernel_log() == []
    code, flags = h.status(clear=True)
    assert code == cb.CBCT_E_DEVICE and flags & 1
    assert h.status() == (cb.CBCT_OK, 0)
    g = h.forward(x)                                         # a cleared handle works again
    assert rel_l2(g, op.forward(G, x.astype(np.float64))) <= 1e-5


def test_forward_box_that_misses_its_samples_is_reported_not_read(monkeypatch):
    monkeypatch.setenv("CBCT_FORWARD_IMPL", "tma")
    for packed in ("0", "1"):
        monkeypatch.setenv("CBCT_FW_PACKED", packed)
        h = sl.Geometry(G)
        x = syn.uniform_volume(G, 8)
        fault_word().value = 2
        status, _ = _raw(h, "cbct_forward", x, h.proj_shape)
        fault_word().value = 0
        assert status == cb.CBCT_OK
        sl.check(0, "forward with a shifted box")            # in particular: no out-of-range shared-memory address
        code, flags = h.status(clear=True)
        assert code == cb.CBCT_E_DEVICE and flags == 2, (packed, flags)
        assert rel_l2(h.forward(x), op.forward(G, x.astype(np.float64))) <= 1e-5


@pytest.mark.parametrize("lanes", ["0", "1"])
@pytest.mark.parametrize("packed", ["0", "1"])
def test_scatter_box_that_misses_its_samples_is_reported_not_written(monkeypatch, lanes, packed):
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", "scatter")
    monkeypatch.setenv("CBCT_BT_LANES", lanes)
    monkeypatch.setenv("CBCT_BT_PACKED", packed)
    h = sl.Geometry(G)
    y = syn.uniform_projections(G, 9) - 0.4
    fault_word().value = 4
    status, _ = _raw(h, "cbct_backproject", y, h.vol_shape)
    fault_word().value = 0
    assert status == cb.CBCT_OK
    sl.check(0, "backproject with a shifted box")
    status, _ = _raw(h, "cbct_backproject", y, h.vol_shape)
    assert status == cb.CBCT_E_DEVICE
    code, flags = h.status(clear=True)
    assert code == cb.CBCT_E_DEVICE and flags == 4
    assert rel_l2(h.backproject(y), op.back_scatter(G, y.astype(np.float64))) <= 1e-5


def test_exhausted_fixed_point_headroom_is_reported(monkeypatch):
    """cbct_backproject plans its int32 accumulators for half their range; the conversion pass reports any sum that
    reaches 2^30.  Fault 8 makes the launcher ignore the plan (all 40 views of cfg 2 in one group instead of 13 at a
    time): P^T of all-ones then peaks above 2^30 but still below 2^31, so the volume is still right, and the word is raised."""
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", "scatter")
    Gt = syn.workload(2).geometry
    qb, group, _w = cb.backproject_fixed_point_plan(Gt)
    assert group < Gt.n_views
    h = sl.Geometry(Gt)
    ones = np.ones(Gt.proj_shape, np.float32)
    ref = op.back_scatter(Gt, ones.astype(np.float64))
    assert rel_l2(h.backproject(ones), ref) <= 1e-5
    assert h.status() == (cb.CBCT_OK, 0)                       # the plan holds: nothing reported
    fault_word().value = 8
    status, out = _raw(h, "cbct_backproject", ones, h.vol_shape)
    fault_word().value = 0
    assert status == cb.CBCT_OK
    code, flags = h.status(clear=True)
    assert code == cb.CBCT_E_DEVICE and flags == 8
    assert 2.0 ** 30 <= ref.max() / Gt.step * 2.0 ** qb < 2.0 ** 31            # the case is what the docstring says
    assert rel_l2(out.numpy(), ref) <= 1e-5


def test_fast_variants_are_default_only_after_the_create_time_self_check():
    """Unforced handles use the packed instruction streams and the skewed lane layout only if, once per process, they
    reproduce the plain variants on a built-in problem (P bit for bit, P^T to 2e-6).  A packed stream that computes
    something else (fault 16) is rejected: handles fall back to the plain variants and say so."""
    L = sl.lib()
    L.cbct_test_reset_selfcheck()
    h = sl.Geometry(G)
    d = h.describe()
    assert "forward_tma_kernel<" in d and ",packed>" in d and "LM0,packed>" in d and "rejected" not in d, d
    x = syn.uniform_volume(G, 12)
    assert rel_l2(h.forward(x), op.forward(G, x.astype(np.float64))) <= 1e-5
    sl.kernel_log()
    L.cbct_test_reset_selfcheck()
    fault_word().value = 16
    h = sl.Geometry(G)                                        # the self-check runs here, with the broken packed stream
    fault_word().value = 0
    d = h.describe()
    assert ",scalar>" in d and "LM1,scalar>" in d and "rejected by the create-time self-check" in d, d
    assert rel_l2(h.forward(x), op.forward(G, x.astype(np.float64))) <= 1e-5
    L.cbct_test_reset_selfcheck()                             # leave the process in its normal state
    assert "rejected" not in sl.Geometry(G).describe()


def test_describe_names_the_kernels_and_forced_implementations_fail_loudly(monkeypatch):
    d = sl.Geometry(G).describe()
    assert "forward_tma_kernel<" in d and "backproject_scatter_kernel<" in d
    ODD = syn.Geometry(37, 29, 11, 2.0, 3.0, 5.0, 45, 19, 2.3, 3.1, 1000.0, 1500.0, (0.0, 0.4, 2.0), step_mm=0.7)
    d = sl.Geometry(ODD).describe()                           # nx, ny not multiples of 4: planned fall-backs, named
    assert "forward_tiled_kernel" in d and "backproject_cell_kernel" in d
    monkeypatch.setenv("CBCT_FORWARD_IMPL", "tma")            # forcing what the geometry cannot use: create fails
    desc, _keep = cb.make_desc(ODD)
    out = C.c_void_p()
    assert sl.lib().cbct_geometry_create(C.byref(desc), C.byref(out)) == cb.CBCT_E_UNSUPPORTED
    monkeypatch.delenv("CBCT_FORWARD_IMPL")
    monkeypatch.setenv("CBCT_BACKPROJECT_IMPL", "scatter")
    assert sl.lib().cbct_geometry_create(C.byref(desc), C.byref(out)) == cb.CBCT_E_UNSUPPORTED


def test_misaligned_pointers_take_the_scalar_paths():
    """float4 accesses are used only from 16-byte aligned bases (a misaligned vector access is an SM exception on the
    device; the shim checks the alignment of every vector access it emulates)."""
    h = sl.Geometry(G)
    cg = sl.Cgls(h)
    nv, nr = int(np.prod(h.vol_shape)), int(np.prod(h.proj_shape))
    # carve volume / projection vectors out of larger buffers at a 4-byte offset
    big = {k: sl.Buf((n + 4,)) for k, n in (("g", nr), ("x", nv), ("r", nr), ("p", nv))}
    y = syn.uniform_projections(G, 10).ravel()
    C.memmove(big["g"].ptr + 4, y.ctypes.data, y.nbytes)
    C.memset(big["x"].ptr, 0, (nv + 4) * 4)

    class View:
        def __init__(self, buf):
            self.ptr = buf.ptr + 4
    v = {k: View(b) for k, b in big.items()}
    # the forward TMA map needs an aligned volume: the library must say so instead of faulting
    assert sl.lib().cbct_cgls_init(cg.handle, v["g"].ptr, v["x"].ptr, v["r"].ptr, v["p"].ptr, None) == cb.CBCT_E_INVALID
    # aligned volumes, misaligned projections: vector kernels fall back to scalar accesses
    xa, pa = sl.Buf((nv,)), sl.Buf((nv,))
    C.memset(xa.ptr, 0, nv * 4)
    sl.check(sl.lib().cbct_cgls_init(cg.handle, v["g"].ptr, xa.ptr, v["r"].ptr, pa.ptr, None), "cgls_init")
    sl.check(sl.lib().cbct_cgls_step(cg.handle, xa.ptr, v["r"].ptr, pa.ptr, None), "cgls_step")
    out = (C.c_double * 5)()
    sl.check(sl.lib().cbct_cgls_scalars(cg.handle, None, out, None), "cgls_scalars")
    s0 = op.back_scatter(G, y.reshape(h.proj_shape).astype(np.float64))          # first step from x0 = 0: s = P^T g
    q0 = op.forward(G, s0)
    assert abs(out[2] - np.sum(s0 * s0) / np.sum(q0 * q0)) <= 1e-5 * out[2]       # alpha = gamma / ||q||^2
