"""TEST INFRASTRUCTURE.  Loads tests/cpu_shim/build/libcbct_cpu_shim.so (the library's kernel sources compiled for the
host, README.md) and offers the few calls the shim tests need.  Buffers handed to the library are guarded
allocations of the shim (a read or write past the end is a segmentation fault, not a silent pass)."""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
import build as shim_build  # noqa: E402

from paper_1008_2042_b200 import binding as cb  # noqa: E402  (GeometryDesc marshalling and the argtypes table only)

_L = None


def lib():
    global _L
    if _L is None:
        L = cb._declare(C.CDLL(shim_build.build()))
        L.shim_malloc.restype = C.c_void_p
        L.shim_malloc.argtypes = [C.c_size_t]
        L.shim_free.argtypes = [C.c_void_p]
        L.shim_last_error.restype = C.c_char_p
        L.shim_last_error.argtypes = []
        L.shim_clear_error.argtypes = []
        L.shim_bank_stats_enable.argtypes = [C.c_int, C.c_longlong]
        L.shim_bank_stats.argtypes = [C.POINTER(C.c_double)]
        L.shim_kernel_log.restype = C.c_char_p
        L.shim_kernel_log.argtypes = [C.c_int]
        _L = L
    return _L


def kernel_log(clear: bool = True):
    """names (with template arguments) of the kernels launched since the last call"""
    return [ln.split(" grid=")[0] for ln in lib().shim_kernel_log(int(clear)).decode().splitlines()]


class bank_stats:
    """with bank_stats(block_stride) as st: ... ; st.ld / st.red = shared-memory wavefronts per warp instruction.
    block_stride > 1 executes only every n-th block of each launch: statistics only, the outputs are incomplete."""

    def __init__(self, block_stride: int = 1):
        self.stride = block_stride

    def __enter__(self):
        lib().shim_bank_stats_enable(1, self.stride)
        return self

    def __exit__(self, *exc):
        out = (C.c_double * 4)()
        lib().shim_bank_stats(out)
        lib().shim_bank_stats_enable(0, 1)
        self.ld_instr, self.ld_wavefronts, self.red_instr, self.red_wavefronts = out[0], out[1], out[2], out[3]
        self.ld = out[1] / out[0] if out[0] else float("nan")
        self.red = out[3] / out[2] if out[2] else float("nan")
        return False


class ShimViolation(AssertionError):
    pass


def check(status: int = 0, where: str = ""):
    err = lib().shim_last_error().decode()
    if err:
        lib().shim_clear_error()
        raise ShimViolation(f"{where}: {err}")
    if status not in (0, 1):
        raise RuntimeError(f"{where}: status {status} ({lib().cbct_status_string(status).decode()})")
    return status


class Buf:
    """a guarded 'device' buffer"""

    def __init__(self, shape, dtype=np.float32, init=None):
        self.shape, self.dtype = tuple(shape), np.dtype(dtype)
        self.nbytes = int(np.prod(self.shape)) * self.dtype.itemsize
        self.ptr = lib().shim_malloc(max(self.nbytes, 1))
        if init is not None:
            a = np.ascontiguousarray(init, dtype=self.dtype)
            assert a.shape == self.shape
            C.memmove(self.ptr, a.ctypes.data, self.nbytes)

    def numpy(self):
        out = np.empty(self.shape, self.dtype)
        C.memmove(out.ctypes.data, self.ptr, self.nbytes)
        return out

    def __del__(self):
        if getattr(self, "ptr", None) and _L is not None:
            _L.shim_free(self.ptr)
            self.ptr = None


def dev(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return Buf(a.shape, np.float32, a)


class Geometry:
    def __init__(self, geom):
        self.spec = geom
        d, self._keep = cb.make_desc(geom)
        h = C.c_void_p()
        check(lib().cbct_geometry_create(C.byref(d), C.byref(h)), "cbct_geometry_create")
        self.handle = h
        self.vol_shape = (geom.nz, geom.ny, geom.nx)
        self.proj_shape = (len(tuple(geom.angles)), geom.nv, geom.nu)

    def info(self):
        nv, nr, K = C.c_int64(), C.c_int64(), C.c_int32()
        t0, st, ns, ws = C.c_double(), C.c_double(), C.c_int64(), C.c_size_t()
        check(lib().cbct_geometry_info(self.handle, C.byref(nv), C.byref(nr), C.byref(K), C.byref(t0), C.byref(st), C.byref(ns),
                                       C.byref(ws)), "cbct_geometry_info")
        return dict(n_vox=nv.value, n_rays=nr.value, K=K.value, t_min=t0.value, step=st.value, n_samples=ns.value)

    def close(self):
        if self.handle:
            lib().cbct_geometry_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _call(self, name, src, out_shape):
        a, out = dev(src), Buf(out_shape)
        check(getattr(lib(), name)(self.handle, a.ptr, out.ptr, None), name)
        return out.numpy()

    def forward(self, f):
        return self._call("cbct_forward", f, self.proj_shape)

    def backproject(self, g):
        return self._call("cbct_backproject", g, self.vol_shape)

    def backproject_eq3(self, g):
        return self._call("cbct_backproject_eq3", g, self.vol_shape)

    def siddon_forward(self, f):
        check(lib().cbct_siddon_prepare(self.handle), "cbct_siddon_prepare")
        return self._call("cbct_siddon_forward", f, self.proj_shape)

    def siddon_backproject(self, g):
        check(lib().cbct_siddon_prepare(self.handle), "cbct_siddon_prepare")
        return self._call("cbct_siddon_backproject", g, self.vol_shape)

    def describe(self):
        buf = C.create_string_buffer(512)
        check(lib().cbct_geometry_describe(self.handle, buf, len(buf)), "cbct_geometry_describe")
        return buf.value.decode()

    def status(self, clear=False):
        """(status code, flags) of cbct_geometry_status"""
        flags = C.c_int(0)
        s = lib().cbct_geometry_status(self.handle, None, C.byref(flags), int(clear))
        return s, flags.value


class Cgls:
    def __init__(self, geometry: Geometry):
        self.geometry = geometry
        h = C.c_void_p()
        check(lib().cbct_cgls_create(geometry.handle, C.byref(h)), "cbct_cgls_create")
        self.handle = h

    def __del__(self):
        if getattr(self, "handle", None) and _L is not None:
            _L.cbct_cgls_destroy(self.handle)
            self.handle = None

    def init(self, g, x, r, p):
        check(lib().cbct_cgls_init(self.handle, g.ptr, x.ptr, r.ptr, p.ptr, None), "cbct_cgls_init")

    def step(self, x, r, p):
        check(lib().cbct_cgls_step(self.handle, x.ptr, r.ptr, p.ptr, None), "cbct_cgls_step")

    def scalars(self, r=None):
        out = (C.c_double * 5)()
        s = check(lib().cbct_cgls_scalars(self.handle, r.ptr if r is not None else None, out, None), "cbct_cgls_scalars")
        return dict(gamma=out[0], qq=out[1], alpha=out[2], beta=out[3], rr=out[4], breakdown=(s == 1))


def _dims(shape):
    nz, ny, nx = shape
    return int(nx), int(ny), int(nz)


def tf_decompose(f):
    out = Buf((27,) + f.shape)
    check(lib().tf_decompose(f.ptr, out.ptr, *_dims(f.shape), None), "tf_decompose")
    return out


def tf_shrink(alpha, mu):
    check(lib().tf_shrink(alpha.ptr, float(mu), *_dims(alpha.shape[1:]), None), "tf_shrink")
    return alpha


def tf_reconstruct(alpha, direct=False):
    out = Buf(alpha.shape[1:])
    fn = lib().tf_reconstruct_direct if direct else lib().tf_reconstruct
    check(fn(alpha.ptr, out.ptr, *_dims(out.shape), None), "tf_reconstruct")
    return out


def tf_apply_fused(f, mu, clamp, impl=None):
    out = Buf(f.shape)
    fn = {None: lib().tf_apply_fused, "tile": lib().tf_apply_fused_tile, "march": lib().tf_apply_fused_march}[impl]
    check(fn(f.ptr, out.ptr, float(mu), int(bool(clamp)), *_dims(f.shape), None), "tf_apply_fused")
    return out


def mg_restrict(fine, fx=2, fy=2, fz=1):
    nz, ny, nx = fine.shape
    out = Buf((nz // fz, ny // fy, nx // fx))
    check(lib().mg_restrict(fine.ptr, out.ptr, nx, ny, nz, fx, fy, fz, None), "mg_restrict")
    return out


def mg_prolong(coarse, fine_shape, fx=2, fy=2, fz=1):
    nz, ny, nx = fine_shape
    out = Buf(fine_shape)
    check(lib().mg_prolong(coarse.ptr, out.ptr, nx, ny, nz, fx, fy, fz, None), "mg_prolong")
    return out


def a2_extrapolate(cur, prev, coef):
    out = Buf(cur.shape)
    check(lib().cbct_a2_extrapolate(cur.ptr, prev.ptr, out.ptr, float(coef), int(np.prod(cur.shape)), None), "cbct_a2_extrapolate")
    return out


def tf_reconstruct_volume(geom, g, n_levels, n_outer, n_cgls=3, mu=5e-4, momentum=True):
    d, keep = cb.make_desc(geom)
    arr = (C.c_int * n_levels)(*[int(v) for v in n_outer])
    out = Buf((geom.nz, geom.ny, geom.nx))
    check(lib().cbct_tf_reconstruct(C.byref(d), g.ptr, out.ptr, int(n_levels), arr, int(n_cgls), float(mu), int(bool(momentum)), None),
          "cbct_tf_reconstruct")
    return out


def recon_run(geom, g, n_levels, n_outer, n_cgls=3, mu=5e-4, momentum=True, bin_detector=False):
    """cbct_recon_create_ex + cbct_recon_run + cbct_recon_status + destroy"""
    d, keep = cb.make_desc(geom)
    h = C.c_void_p()
    check(lib().cbct_recon_create_ex(C.byref(d), int(n_levels), 1 if bin_detector else 0, C.byref(h)), "cbct_recon_create_ex")
    arr = (C.c_int * n_levels)(*[int(v) for v in n_outer])
    out = Buf((geom.nz, geom.ny, geom.nx))
    try:
        check(lib().cbct_recon_run(h, g.ptr, out.ptr, arr, int(n_cgls), float(mu), int(bool(momentum)), None), "cbct_recon_run")
        flags = C.c_int(0)
        check(lib().cbct_recon_status(h, None, C.byref(flags), 0), "cbct_recon_status")
    finally:
        lib().cbct_recon_destroy(h)
    return out


def tv_rof(u, mu_tv, eps, max_iter=30, rel_tol=1e-3, clamp=False):
    """(f, trials, accepted, energy) of tv_rof / tv_rof_result"""
    nx, ny, nz = _dims(u.shape)
    out = Buf(u.shape)
    work = Buf((int(lib().tv_rof_workspace_bytes(nx, ny, nz)),), np.uint8)
    check(lib().tv_rof(u.ptr, out.ptr, work.ptr, float(mu_tv), float(eps), int(max_iter), float(rel_tol), int(bool(clamp)), nx, ny, nz,
                       None), "tv_rof")
    tr, ac, en = C.c_int(), C.c_int(), C.c_double()
    check(lib().tv_rof_result(work.ptr, nx, ny, nz, C.byref(tr), C.byref(ac), C.byref(en), None), "tv_rof_result")
    return out, tr.value, ac.value, en.value


def recon_run_tv(geom, g, n_levels, n_outer, n_cgls, mu_tv, eps, max_rof_iter, rel_tol, momentum=True):
    d, keep = cb.make_desc(geom)
    h = C.c_void_p()
    check(lib().cbct_recon_create_ex(C.byref(d), int(n_levels), 2, C.byref(h)), "cbct_recon_create_ex")
    arr = (C.c_int * n_levels)(*[int(v) for v in n_outer])
    out = Buf((geom.nz, geom.ny, geom.nx))
    try:
        check(lib().cbct_recon_run_tv(h, g.ptr, out.ptr, arr, int(n_cgls), float(mu_tv), float(eps), int(max_rof_iter), float(rel_tol),
                                      int(bool(momentum)), None), "cbct_recon_run_tv")
        flags = C.c_int(0)
        check(lib().cbct_recon_status(h, None, C.byref(flags), 0), "cbct_recon_status")
    finally:
        lib().cbct_recon_destroy(h)
    return out
