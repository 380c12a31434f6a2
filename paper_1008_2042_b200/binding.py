"""Thin ctypes binding of libcbct_b200.so (include/cbct.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing, or a call returns
an error status, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcbct_b200.so")

CBCT_OK, CBCT_E_INVALID, CBCT_E_UNSUPPORTED, CBCT_E_CUDA, CBCT_E_DEVICE, CBCT_BREAKDOWN = 0, -1, -2, -3, -4, 1
STATUS_BITS = {1: "wait_timeout", 2: "forward_range", 4: "backproject_range", 8: "fixed_point_range"}

# every symbol include/cbct.h and include/cbct_debug.h declare (tests check the library exports all of them)
EXPORTS = [
    "cbct_status_string", "cbct_last_cuda_error", "cbct_version", "cbct_launch_count",
    "cbct_profile_begin", "cbct_profile_end",
    "cbct_geometry_create", "cbct_geometry_destroy", "cbct_geometry_info", "cbct_geometry_describe", "cbct_geometry_status",
    "cbct_forward", "cbct_backproject", "cbct_forward_host", "cbct_backproject_host",
    "cbct_backproject_fixed_point_plan", "cbct_backproject_eq3", "cbct_siddon_prepare", "cbct_siddon_forward", "cbct_siddon_backproject",
    "cbct_siddon_fixed_point_plan", "cbct_microbench", "tf_reconstruct_direct",
    "tf_apply_fused_tile", "tf_apply_fused_march", "tf_apply_fused_describe",
    "cbct_cgls_create", "cbct_cgls_destroy", "cbct_cgls_init", "cbct_cgls_step", "cbct_cgls_scalars",
    "tf_decompose", "tf_shrink", "tf_reconstruct", "tf_apply_fused",
    "mg_restrict", "mg_prolong", "cbct_a2_extrapolate", "tv_rof_workspace_bytes", "tv_rof", "tv_rof_result", "cbct_recon_run_tv",
    "cbct_recon_create", "cbct_recon_create_ex", "cbct_recon_destroy", "cbct_recon_run", "cbct_recon_run_host", "cbct_recon_status", "cbct_recon_describe",
    "cbct_tf_reconstruct", "cbct_tf_reconstruct_host",
]


class CbctError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().cbct_status_string(status).decode()
        extra = f" (cudaError {lib().cbct_last_cuda_error()})" if status == CBCT_E_CUDA else ""
        super().__init__(f"{where}: {msg}{extra}")


class GeometryDesc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("ox", C.c_double), ("oy", C.c_double), ("oz", C.c_double),
                ("nu", C.c_int32), ("nv", C.c_int32),
                ("du", C.c_double), ("dv", C.c_double), ("u0", C.c_double), ("v0", C.c_double),
                ("sad", C.c_double), ("sdd", C.c_double),
                ("n_views", C.c_int32), ("angles", C.POINTER(C.c_double)),
                ("step_mm", C.c_double)]


_lib = None


def lib():
    """Load the CUDA library (once).  Fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1008_2042_b200.build` "
                          "(there is no CPU fallback)")
    _lib = _declare(C.CDLL(LIB_PATH))
    return _lib


def _declare(L):
    """argument / result types of every entry point of include/cbct.h on a loaded library"""
    vp, fp, ip = C.c_void_p, C.c_void_p, C.c_int
    L.cbct_status_string.restype = C.c_char_p
    L.cbct_status_string.argtypes = [ip]
    L.cbct_last_cuda_error.argtypes = []
    L.cbct_version.argtypes = []
    L.cbct_launch_count.argtypes = []
    L.cbct_profile_begin.argtypes = []
    L.cbct_profile_end.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.cbct_geometry_create.argtypes = [C.POINTER(GeometryDesc), C.POINTER(vp)]
    L.cbct_geometry_destroy.argtypes = [vp]
    L.cbct_geometry_info.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int32),
                                     C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int64),
                                     C.POINTER(C.c_size_t)]
    L.cbct_geometry_describe.argtypes = [vp, C.c_char_p, C.c_size_t]
    L.cbct_geometry_status.argtypes = [vp, vp, C.POINTER(C.c_int), ip]
    L.cbct_siddon_prepare.argtypes = [vp]
    for name in ("cbct_forward", "cbct_backproject", "cbct_forward_host", "cbct_backproject_host", "cbct_backproject_eq3",
                 "cbct_siddon_forward", "cbct_siddon_backproject"):
        getattr(L, name).argtypes = [vp, fp, fp, vp]
    L.cbct_siddon_fixed_point_plan.argtypes = [C.POINTER(GeometryDesc), C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                               C.POINTER(C.c_double)]
    L.cbct_microbench.argtypes = [ip, ip, C.POINTER(C.c_double), vp]
    L.cbct_backproject_fixed_point_plan.argtypes = [C.POINTER(GeometryDesc), C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                                    C.POINTER(C.c_double)]
    L.cbct_cgls_create.argtypes = [vp, C.POINTER(vp)]
    L.cbct_cgls_destroy.argtypes = [vp]
    L.cbct_cgls_init.argtypes = [vp, fp, fp, fp, fp, vp]
    L.cbct_cgls_step.argtypes = [vp, fp, fp, fp, vp]
    L.cbct_cgls_scalars.argtypes = [vp, fp, C.POINTER(C.c_double), vp]
    L.tf_decompose.argtypes = [fp, fp, ip, ip, ip, vp]
    L.tf_shrink.argtypes = [fp, C.c_float, ip, ip, ip, vp]
    L.tf_reconstruct.argtypes = [fp, fp, ip, ip, ip, vp]
    L.tf_reconstruct_direct.argtypes = [fp, fp, ip, ip, ip, vp]
    L.tf_apply_fused.argtypes = [fp, fp, C.c_float, ip, ip, ip, ip, vp]
    L.tf_apply_fused_tile.argtypes = [fp, fp, C.c_float, ip, ip, ip, ip, vp]
    L.tf_apply_fused_march.argtypes = [fp, fp, C.c_float, ip, ip, ip, ip, vp]
    L.tf_apply_fused_describe.restype = C.c_char_p
    L.tf_apply_fused_describe.argtypes = []
    L.mg_restrict.argtypes = [fp, fp, ip, ip, ip, ip, ip, ip, vp]
    L.mg_prolong.argtypes = [fp, fp, ip, ip, ip, ip, ip, ip, vp]
    L.cbct_a2_extrapolate.argtypes = [fp, fp, fp, C.c_float, C.c_int64, vp]
    L.tv_rof_workspace_bytes.argtypes = [ip, ip, ip]
    L.tv_rof.argtypes = [fp, fp, vp, C.c_float, C.c_float, ip, C.c_float, ip, ip, ip, ip, vp]
    L.tv_rof_result.argtypes = [vp, ip, ip, ip, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_double), vp]
    L.cbct_recon_run_tv.argtypes = [vp, fp, fp, C.POINTER(C.c_int), ip, C.c_float, C.c_float, ip, C.c_float, ip, vp]
    L.cbct_recon_create.argtypes = [C.POINTER(GeometryDesc), ip, C.POINTER(vp)]
    L.cbct_recon_create_ex.argtypes = [C.POINTER(GeometryDesc), ip, C.c_uint, C.POINTER(vp)]
    L.cbct_recon_destroy.argtypes = [vp]
    L.cbct_recon_run.argtypes = [vp, fp, fp, C.POINTER(C.c_int), ip, C.c_float, ip, vp]
    L.cbct_recon_run_host.argtypes = [vp, fp, fp, C.POINTER(C.c_int), ip, C.c_float, ip, vp]
    L.cbct_recon_status.argtypes = [vp, vp, C.POINTER(C.c_int), ip]
    L.cbct_recon_describe.argtypes = [vp, C.c_char_p, C.c_size_t]
    L.cbct_tf_reconstruct.argtypes = [C.POINTER(GeometryDesc), fp, fp, ip, C.POINTER(C.c_int), ip, C.c_float, ip, vp]
    L.cbct_tf_reconstruct_host.argtypes = [C.POINTER(GeometryDesc), fp, fp, ip, C.POINTER(C.c_int), ip, C.c_float, ip, vp]
    for name in EXPORTS:
        if name not in ("cbct_status_string", "tf_apply_fused_describe"):
            getattr(L, name).restype = C.c_int
    L.cbct_launch_count.restype = C.c_longlong
    L.tv_rof_workspace_bytes.restype = C.c_size_t
    return L


def _check(status: int, where: str, allow_breakdown: bool = False) -> int:
    if status == CBCT_OK or (allow_breakdown and status == CBCT_BREAKDOWN):
        return status
    raise CbctError(status, where)


def launch_count() -> int:
    return int(lib().cbct_launch_count())


def profile_begin() -> None:
    _check(lib().cbct_profile_begin(), "cbct_profile_begin")


def profile_end():
    """{'forward': (ms, launches), 'backproject': (ms, launches)} since profile_begin()."""
    ms, cnt = (C.c_double * 2)(), (C.c_int * 2)()
    _check(lib().cbct_profile_end(ms, cnt), "cbct_profile_end")
    return {"forward": (ms[0], cnt[0]), "backproject": (ms[1], cnt[1])}


def _stream(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dptr(t, n: Optional[int] = None) -> int:
    """Device pointer of a contiguous fp32 CUDA tensor (marshalling only)."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CUDA tensor")
    if n is not None and t.numel() != n:
        raise ValueError(f"expected {n} elements, got {t.numel()}")
    return t.data_ptr()


def _hptr(t, n: Optional[int] = None) -> int:
    """Host pointer of a contiguous fp32 CPU tensor / numpy array."""
    if isinstance(t, np.ndarray):
        if t.dtype != np.float32 or not t.flags.c_contiguous:
            raise TypeError("expected a C-contiguous float32 array")
        if n is not None and t.size != n:
            raise ValueError(f"expected {n} elements, got {t.size}")
        return t.ctypes.data
    import torch
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("expected a contiguous float32 CPU tensor")
    if n is not None and t.numel() != n:
        raise ValueError(f"expected {n} elements, got {t.numel()}")
    return t.data_ptr()


def make_desc(geom):
    """GeometryDesc (+ the angle array that must outlive it) from any object with the fields of
    synthetic.Geometry."""
    ang = np.ascontiguousarray(np.asarray(list(geom.angles), dtype=np.float64))
    d = GeometryDesc(geom.nx, geom.ny, geom.nz, geom.dx, geom.dy, geom.dz, geom.ox, geom.oy, geom.oz,
                     geom.nu, geom.nv, geom.du, geom.dv, geom.u0, geom.v0, geom.sad, geom.sdd,
                     len(ang), ang.ctypes.data_as(C.POINTER(C.c_double)), float(getattr(geom, "step_mm", 0.0)))
    return d, ang


MICROBENCH_KINDS = {0: ("ffma", "warp-instr/clk/SM"), 1: ("ffma2", "warp-instr/clk/SM"), 2: ("lds32", "warp-instr/clk/SM"),
                    3: ("atoms_add_s32", "warp-instr/clk/SM"), 4: ("ldg32_l1_hit", "warp-instr/clk/SM"),
                    5: ("l2_read_64MB", "GB/s"), 6: ("l2_red_add_s32", "Gred/s"), 7: ("atoms_add_u64", "warp-instr/clk/SM")}


def microbench(stream=None, iters: int = 0):
    """{name: (rate, unit)} of cbct_microbench for every kind; iters <= 0: the default loop length."""
    res = {}
    for kind, (name, unit) in MICROBENCH_KINDS.items():
        out = (C.c_double * 3)()
        _check(lib().cbct_microbench(kind, int(iters), out, _stream(stream)), "cbct_microbench")
        res[name] = (out[0], unit)
    return res


def backproject_fixed_point_plan(geom):
    """(qb, views_per_group, max_weight_sum_per_view) of cbct_backproject for this geometry; host only."""
    d, keep = make_desc(geom)
    qb, grp, w = C.c_int32(), C.c_int32(), C.c_double()
    _check(lib().cbct_backproject_fixed_point_plan(C.byref(d), C.byref(qb), C.byref(grp), C.byref(w)),
           "cbct_backproject_fixed_point_plan")
    return qb.value, grp.value, w.value


def siddon_fixed_point_plan(geom):
    """(qb, views_per_group, max_path_sum_per_view) of cbct_siddon_backproject for this geometry; host only."""
    d, keep = make_desc(geom)
    qb, grp, w = C.c_int32(), C.c_int32(), C.c_double()
    _check(lib().cbct_siddon_fixed_point_plan(C.byref(d), C.byref(qb), C.byref(grp), C.byref(w)), "cbct_siddon_fixed_point_plan")
    return qb.value, grp.value, w.value


class Geometry:
    """cbct_geometry handle."""

    def __init__(self, geom):
        self.spec = geom
        d, keep = make_desc(geom)
        h = C.c_void_p()
        _check(lib().cbct_geometry_create(C.byref(d), C.byref(h)), "cbct_geometry_create")
        self.handle = h
        nv, nr, K = C.c_int64(), C.c_int64(), C.c_int32()
        t0, st, ns, ws = C.c_double(), C.c_double(), C.c_int64(), C.c_size_t()
        _check(lib().cbct_geometry_info(h, C.byref(nv), C.byref(nr), C.byref(K), C.byref(t0), C.byref(st),
                                        C.byref(ns), C.byref(ws)), "cbct_geometry_info")
        self.n_vox, self.n_rays, self.K = nv.value, nr.value, K.value
        self.t_min, self.step_mm, self.n_samples, self.workspace_bytes = t0.value, st.value, ns.value, ws.value
        self.vol_shape = (geom.nz, geom.ny, geom.nx)
        self.proj_shape = (len(tuple(geom.angles)), geom.nv, geom.nu)
        self._siddon_ready = False

    def close(self):
        if getattr(self, "handle", None):
            lib().cbct_geometry_destroy(self.handle)
            self.handle = None

    def describe(self) -> str:
        """which kernels serve this handle (cbct_geometry_describe)"""
        buf = C.create_string_buffer(512)
        _check(lib().cbct_geometry_describe(self.handle, buf, len(buf)), "cbct_geometry_describe")
        return buf.value.decode()

    def status(self, clear: bool = False, stream=None):
        """(ok, [names of the raised CBCT_STATUS_* bits]); synchronises the stream (cbct_geometry_status)"""
        flags = C.c_int(0)
        s = lib().cbct_geometry_status(self.handle, _stream(stream), C.byref(flags), int(clear))
        if s not in (CBCT_OK, CBCT_E_DEVICE):
            raise CbctError(s, "cbct_geometry_status")
        return s == CBCT_OK, [n for b, n in STATUS_BITS.items() if flags.value & b]

    def siddon_prepare(self):
        if not self._siddon_ready:
            _check(lib().cbct_siddon_prepare(self.handle), "cbct_siddon_prepare")
            self._siddon_ready = True

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    def forward(self, d_vol, d_proj, stream=None):
        _check(lib().cbct_forward(self.handle, _dptr(d_vol, self.n_vox), _dptr(d_proj, self.n_rays), _stream(stream)),
               "cbct_forward")
        return d_proj

    def backproject(self, d_proj, d_vol, stream=None):
        _check(lib().cbct_backproject(self.handle, _dptr(d_proj, self.n_rays), _dptr(d_vol, self.n_vox),
                                      _stream(stream)), "cbct_backproject")
        return d_vol

    def backproject_eq3(self, d_proj, d_vol, stream=None):
        """The paper's approximate adjoint, Eq. 3 (not the transpose of forward)."""
        _check(lib().cbct_backproject_eq3(self.handle, _dptr(d_proj, self.n_rays), _dptr(d_vol, self.n_vox),
                                          _stream(stream)), "cbct_backproject_eq3")
        return d_vol

    def siddon_forward(self, d_vol, d_proj, stream=None):
        """g = P_siddon f: the paper's own projector, exact path lengths through piecewise-constant voxels."""
        self.siddon_prepare()
        _check(lib().cbct_siddon_forward(self.handle, _dptr(d_vol, self.n_vox), _dptr(d_proj, self.n_rays), _stream(stream)),
               "cbct_siddon_forward")
        return d_proj

    def siddon_backproject(self, d_proj, d_vol, stream=None):
        """f = P_siddon^T g, the exact transpose of siddon_forward."""
        self.siddon_prepare()
        _check(lib().cbct_siddon_backproject(self.handle, _dptr(d_proj, self.n_rays), _dptr(d_vol, self.n_vox), _stream(stream)),
               "cbct_siddon_backproject")
        return d_vol

    def forward_host(self, h_vol, h_proj, stream=None):
        _check(lib().cbct_forward_host(self.handle, _hptr(h_vol, self.n_vox), _hptr(h_proj, self.n_rays),
                                       _stream(stream)), "cbct_forward_host")
        return h_proj

    def backproject_host(self, h_proj, h_vol, stream=None):
        _check(lib().cbct_backproject_host(self.handle, _hptr(h_proj, self.n_rays), _hptr(h_vol, self.n_vox),
                                           _stream(stream)), "cbct_backproject_host")
        return h_vol


class Cgls:
    """cbct_cgls handle."""

    def __init__(self, geometry: Geometry):
        self.geometry = geometry
        h = C.c_void_p()
        _check(lib().cbct_cgls_create(geometry.handle, C.byref(h)), "cbct_cgls_create")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib().cbct_cgls_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    def init(self, d_g, d_x, d_r, d_p, stream=None):
        G = self.geometry
        _check(lib().cbct_cgls_init(self.handle, _dptr(d_g, G.n_rays), _dptr(d_x, G.n_vox), _dptr(d_r, G.n_rays),
                                    _dptr(d_p, G.n_vox), _stream(stream)), "cbct_cgls_init")

    def step(self, d_x, d_r, d_p, stream=None):
        G = self.geometry
        _check(lib().cbct_cgls_step(self.handle, _dptr(d_x, G.n_vox), _dptr(d_r, G.n_rays), _dptr(d_p, G.n_vox),
                                    _stream(stream)), "cbct_cgls_step")

    def scalars(self, d_r=None, stream=None):
        """dict(gamma, qq, alpha, beta, rr, breakdown); synchronises the stream."""
        out = (C.c_double * 5)()
        s = _check(lib().cbct_cgls_scalars(self.handle, _dptr(d_r, self.geometry.n_rays) if d_r is not None else None,
                                           out, _stream(stream)), "cbct_cgls_scalars", allow_breakdown=True)
        return dict(gamma=out[0], qq=out[1], alpha=out[2], beta=out[3], rr=out[4], breakdown=(s == CBCT_BREAKDOWN))


def _dims(shape):
    nz, ny, nx = shape
    return int(nx), int(ny), int(nz)


def tf_decompose(d_f, d_alpha, stream=None):
    nx, ny, nz = _dims(d_f.shape)
    _check(lib().tf_decompose(_dptr(d_f), _dptr(d_alpha, 27 * nx * ny * nz), nx, ny, nz, _stream(stream)), "tf_decompose")
    return d_alpha


def tf_shrink(d_alpha, mu: float, stream=None):
    nx, ny, nz = _dims(d_alpha.shape[1:])
    _check(lib().tf_shrink(_dptr(d_alpha, 27 * nx * ny * nz), float(mu), nx, ny, nz, _stream(stream)), "tf_shrink")
    return d_alpha


def tf_reconstruct(d_alpha, d_f, stream=None):
    nx, ny, nz = _dims(d_f.shape)
    _check(lib().tf_reconstruct(_dptr(d_alpha, 27 * nx * ny * nz), _dptr(d_f), nx, ny, nz, _stream(stream)),
           "tf_reconstruct")
    return d_f


def tf_reconstruct_direct(d_alpha, d_f, stream=None):
    """cbct_debug.h: the 27 x 27-tap cross-check of tf_reconstruct"""
    nx, ny, nz = _dims(d_f.shape)
    _check(lib().tf_reconstruct_direct(_dptr(d_alpha, 27 * nx * ny * nz), _dptr(d_f), nx, ny, nz, _stream(stream)),
           "tf_reconstruct_direct")
    return d_f


def tf_apply_fused(d_in, d_out, mu: float, clamp_nonneg: bool = False, stream=None, impl: str | None = None):
    """impl None: the library's choice (tf_apply_fused); "tile" / "march": that kernel on its own (cbct_debug.h)"""
    nx, ny, nz = _dims(d_in.shape)
    fn = {None: lib().tf_apply_fused, "tile": lib().tf_apply_fused_tile, "march": lib().tf_apply_fused_march}[impl]
    _check(fn(_dptr(d_in), _dptr(d_out, nx * ny * nz), float(mu), int(bool(clamp_nonneg)), nx, ny, nz, _stream(stream)),
           "tf_apply_fused")
    return d_out


def tf_apply_fused_describe() -> str:
    """cbct_debug.h: the kernel tf_apply_fused uses in this process"""
    return lib().tf_apply_fused_describe().decode()


def tv_rof(d_u, d_f, mu_tv: float, eps: float, max_iter: int = 30, rel_tol: float = 1e-3, clamp_nonneg: bool = False, stream=None):
    """PAPER.md:236 ROF sub-problem (tv_rof); returns (d_f, trials, accepted, energy) -- reading them back synchronises."""
    import torch
    nx, ny, nz = _dims(d_u.shape)
    work = torch.empty(int(lib().tv_rof_workspace_bytes(nx, ny, nz)), dtype=torch.uint8, device=d_u.device)
    _check(lib().tv_rof(_dptr(d_u), _dptr(d_f, nx * ny * nz), work.data_ptr(), float(mu_tv), float(eps), int(max_iter), float(rel_tol),
                        int(bool(clamp_nonneg)), nx, ny, nz, _stream(stream)), "tv_rof")
    tr, ac, en = C.c_int(), C.c_int(), C.c_double()
    _check(lib().tv_rof_result(work.data_ptr(), nx, ny, nz, C.byref(tr), C.byref(ac), C.byref(en), _stream(stream)), "tv_rof_result")
    return d_f, tr.value, ac.value, en.value


def mg_restrict(d_fine, d_coarse, fx=2, fy=2, fz=1, stream=None):
    nx, ny, nz = _dims(d_fine.shape)
    _check(lib().mg_restrict(_dptr(d_fine), _dptr(d_coarse, (nx // fx) * (ny // fy) * (nz // fz)), nx, ny, nz, fx, fy, fz,
                             _stream(stream)), "mg_restrict")
    return d_coarse


def mg_prolong(d_coarse, d_fine, fx=2, fy=2, fz=1, stream=None):
    nx, ny, nz = _dims(d_fine.shape)
    _check(lib().mg_prolong(_dptr(d_coarse, (nx // fx) * (ny // fy) * (nz // fz)), _dptr(d_fine), nx, ny, nz, fx, fy, fz,
                            _stream(stream)), "mg_prolong")
    return d_fine


def a2_extrapolate(d_f_cur, d_f_prev, d_v, coef: float, stream=None):
    n = d_f_cur.numel()
    _check(lib().cbct_a2_extrapolate(_dptr(d_f_cur), _dptr(d_f_prev, n), _dptr(d_v, n), float(coef), n, _stream(stream)),
           "cbct_a2_extrapolate")
    return d_v


class Recon:
    """cbct_recon handle: A2 inside the multigrid cascade."""

    def __init__(self, geom, n_levels: int, bin_detector: bool = False, tv: bool = False):
        d, keep = make_desc(geom)
        h = C.c_void_p()
        _check(lib().cbct_recon_create_ex(C.byref(d), int(n_levels), (1 if bin_detector else 0) | (2 if tv else 0), C.byref(h)),
               "cbct_recon_create_ex")
        self.handle, self.n_levels, self.spec = h, int(n_levels), geom
        self.n_vox = geom.nx * geom.ny * geom.nz
        self.n_rays = len(tuple(geom.angles)) * geom.nv * geom.nu

    def close(self):
        if getattr(self, "handle", None):
            lib().cbct_recon_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    def status(self, clear: bool = False, stream=None):
        """(ok, [raised CBCT_STATUS_* bits]) over all levels; synchronises the stream (cbct_recon_status)"""
        flags = C.c_int(0)
        s = lib().cbct_recon_status(self.handle, _stream(stream), C.byref(flags), int(clear))
        if s not in (CBCT_OK, CBCT_E_DEVICE):
            raise CbctError(s, "cbct_recon_status")
        return s == CBCT_OK, [n for b, n in STATUS_BITS.items() if flags.value & b]

    def describe(self) -> str:
        buf = C.create_string_buffer(512)
        _check(lib().cbct_recon_describe(self.handle, buf, len(buf)), "cbct_recon_describe")
        return buf.value.decode()

    def _outer(self, n_outer: Sequence[int]):
        assert len(n_outer) == self.n_levels
        return (C.c_int * self.n_levels)(*[int(v) for v in n_outer])

    def run(self, d_g, d_f, n_outer, n_cgls=3, mu=5e-4, momentum=True, stream=None):
        _check(lib().cbct_recon_run(self.handle, _dptr(d_g, self.n_rays), _dptr(d_f, self.n_vox), self._outer(n_outer),
                                    int(n_cgls), float(mu), int(bool(momentum)), _stream(stream)), "cbct_recon_run")
        return d_f

    def run_tv(self, d_g, d_f, n_outer, n_cgls=3, mu_tv=1e-3, eps=1e-4, max_rof_iter=30, rel_tol=1e-3, momentum=True, stream=None):
        """the TV comparison algorithm on the same cascade; the handle needs tv=True"""
        _check(lib().cbct_recon_run_tv(self.handle, _dptr(d_g, self.n_rays), _dptr(d_f, self.n_vox), self._outer(n_outer), int(n_cgls),
                                       float(mu_tv), float(eps), int(max_rof_iter), float(rel_tol), int(bool(momentum)),
                                       _stream(stream)), "cbct_recon_run_tv")
        return d_f

    def run_host(self, h_g, h_f, n_outer, n_cgls=3, mu=5e-4, momentum=True, stream=None):
        _check(lib().cbct_recon_run_host(self.handle, _hptr(h_g, self.n_rays), _hptr(h_f, self.n_vox),
                                         self._outer(n_outer), int(n_cgls), float(mu), int(bool(momentum)),
                                         _stream(stream)), "cbct_recon_run_host")
        return h_f


def tf_reconstruct_volume(geom, d_g, d_f, n_levels, n_outer, n_cgls=3, mu=5e-4, momentum=True, stream=None):
    """One-shot cbct_tf_reconstruct."""
    d, keep = make_desc(geom)
    arr = (C.c_int * n_levels)(*[int(v) for v in n_outer])
    _check(lib().cbct_tf_reconstruct(C.byref(d), _dptr(d_g), _dptr(d_f), int(n_levels), arr, int(n_cgls), float(mu),
                                     int(bool(momentum)), _stream(stream)), "cbct_tf_reconstruct")
    return d_f
