"""Thin ctypes binding over the C ABI of libcbct.so (include/cbct.h).

Argument marshalling only: every step of the hot path runs in the CUDA
kernels behind `cbct_fp`, `cbct_bp_adjoint`, `cbct_bp_fdk`.  There is no CPU
fallback: if libcbct.so is missing, or no CUDA device is present, calls raise.
Tensors may be torch CUDA tensors, torch CPU tensors (pinned or not) or numpy
arrays, fp32 and C-contiguous; PyTorch is used for memory and streams only.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcbct.so")

EXPORTS = (
    "cbct_geom_create", "cbct_geom_destroy", "cbct_fp", "cbct_bp_adjoint", "cbct_bp_fdk",
    "cbct_geom_count_samples", "cbct_geom_num_slabs", "cbct_geom_launch_count",
    "cbct_geom_symmetry", "cbct_geom_workspace_bytes", "cbct_geom_reserve", "cbct_bp_adjoint_slab", "cbct_bp_fdk_slab",
    "cbct_geom_profile", "cbct_geom_profile_read",
    "cbct_fdk_filter", "cbct_redundancy_weight", "cbct_geom_redundancy_weights",
    "cbct_fp_residual", "cbct_bp_adjoint_weighted",
    "cbct_fov", "cbct_downsample", "cbct_upsample", "cbct_proj_down",
    "cbct_water_bone", "cbct_polychromatic_primary",
    "cbct_static_scratch_setup", "cbct_bp_fdk_static",
    "cbct_status_string", "cbct_last_cuda_error",
)


STATIC_SCRATCH_BYTES = 32 << 20   # CBCT_STATIC_SCRATCH_BYTES (include/cbct.h)


class CbctError(RuntimeError):
    pass


class GeomDesc(ctypes.Structure):
    """struct cbct_geom_desc (include/cbct.h)."""
    _fields_ = [
        ("sid_mm", ctypes.c_double), ("sdd_mm", ctypes.c_double),
        ("n_views", ctypes.c_int32),
        ("angles_rad", ctypes.POINTER(ctypes.c_double)),
        ("det_nu", ctypes.c_int32), ("det_nv", ctypes.c_int32),
        ("det_du_mm", ctypes.c_double), ("det_dv_mm", ctypes.c_double),
        ("det_off_u_mm", ctypes.c_double), ("det_off_v_mm", ctypes.c_double),
        ("vol_nx", ctypes.c_int32), ("vol_ny", ctypes.c_int32), ("vol_nz", ctypes.c_int32),
        ("vox_mm", ctypes.c_double),
        ("vol_cx_mm", ctypes.c_double), ("vol_cy_mm", ctypes.c_double), ("vol_cz_mm", ctypes.c_double),
        ("step_vox", ctypes.c_double),
        ("max_workset_bytes", ctypes.c_uint64),
    ]


_lib = None


def load_library() -> ctypes.CDLL:
    """Load libcbct.so (built in-tree by paper_2512_21180_b200/build.py).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise CbctError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2512_21180_b200.build` "
            "(or __graft_entry__.build()); there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i32 = ctypes.c_void_p, ctypes.c_int32
    L.cbct_geom_create.argtypes = [ctypes.POINTER(GeomDesc), ctypes.POINTER(vp)]
    L.cbct_geom_destroy.argtypes = [vp]
    for name in ("cbct_fp", "cbct_bp_adjoint", "cbct_bp_fdk"):
        getattr(L, name).argtypes = [vp, vp, vp, i32, vp]
    L.cbct_geom_count_samples.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64)]
    L.cbct_geom_num_slabs.argtypes = [vp, i32, ctypes.POINTER(i32)]
    L.cbct_geom_launch_count.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64)]
    L.cbct_geom_workspace_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64)]
    L.cbct_geom_reserve.argtypes = [vp, i32]
    L.cbct_geom_symmetry.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i32)]
    for name in ("cbct_bp_adjoint_slab", "cbct_bp_fdk_slab"):
        getattr(L, name).argtypes = [vp, vp, vp, i32, i32, i32, i32, vp]
    L.cbct_geom_profile.argtypes = [vp, ctypes.c_int]
    L.cbct_geom_profile_read.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                         ctypes.POINTER(ctypes.c_uint64)]
    L.cbct_fdk_filter.argtypes = [vp, vp, vp, i32, i32, vp]
    L.cbct_redundancy_weight.argtypes = [vp, vp, vp, i32, vp]
    L.cbct_geom_redundancy_weights.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    L.cbct_fp_residual.argtypes = [vp, vp, vp, vp, i32, vp]
    L.cbct_bp_adjoint_weighted.argtypes = [vp, vp, vp, i32, vp]
    L.cbct_fov.argtypes = [vp, vp, vp]
    i64 = ctypes.c_int64
    L.cbct_downsample.argtypes = [vp, vp, i64, i32, i32, i32, i32, vp]
    L.cbct_upsample.argtypes = [vp, vp, i64, i32, i32, i32, i32, vp]
    L.cbct_proj_down.argtypes = [vp, vp, i64, i32, i32, i32, i32, vp]
    f64 = ctypes.c_double
    L.cbct_water_bone.argtypes = [vp, vp, vp, i64, f64, f64, f64, f64, vp]
    dp = ctypes.POINTER(ctypes.c_double)
    L.cbct_polychromatic_primary.argtypes = [vp, vp, vp, dp, dp, dp, i32, i64, i64, vp, vp]
    L.cbct_static_scratch_setup.argtypes = []
    L.cbct_bp_fdk_static.argtypes = [vp, vp, vp, i32, vp]
    L.cbct_status_string.argtypes = [ctypes.c_int]
    L.cbct_status_string.restype = ctypes.c_char_p
    L.cbct_last_cuda_error.restype = ctypes.c_char_p
    _lib = L
    return L


def _check(rc: int):
    if rc != 0:
        L = load_library()
        msg = L.cbct_status_string(rc).decode()
        cuda = L.cbct_last_cuda_error().decode()
        raise CbctError(f"{msg}" + (f" [{cuda}]" if cuda and rc == -3 else ""))


def _ptr_and_keep(t, n_expected: int):
    """Raw address of an fp32 contiguous torch tensor / numpy array."""
    if isinstance(t, np.ndarray):
        if t.dtype != np.float32 or not t.flags["C_CONTIGUOUS"]:
            raise CbctError("numpy buffers must be float32 and C-contiguous")
        if t.size != n_expected:
            raise CbctError(f"buffer has {t.size} elements, expected {n_expected}")
        return t.ctypes.data
    import torch
    if not isinstance(t, torch.Tensor):
        raise CbctError("expected a torch.Tensor or numpy.ndarray")
    if t.dtype != torch.float32 or not t.is_contiguous():
        raise CbctError("tensors must be float32 and contiguous")
    if t.numel() != n_expected:
        raise CbctError(f"tensor has {t.numel()} elements, expected {n_expected}")
    return t.data_ptr()


def _stream_handle(stream, device=None) -> int:
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return int(torch.cuda.current_stream(device).cuda_stream)
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


class _on_device_of:
    """Context for one C-ABI call: all CUDA tensors among `tensors` must live on ONE device; that device is made
    current for the call (the library launches on the current device) and `self.stream` is the handle of `stream`,
    or of torch's current stream ON THAT DEVICE.  Host tensors / numpy arrays place no constraint."""

    def __init__(self, tensors, stream):
        self.dev, self._ctx = None, None
        for t in tensors:
            d = getattr(t, "device", None)
            if d is not None and getattr(d, "type", "cpu") == "cuda":
                if self.dev is not None and d != self.dev:
                    raise CbctError(f"tensors on different CUDA devices ({self.dev} and {d}) in one call")
                self.dev = d
        self._stream = stream

    def __enter__(self):
        if self.dev is not None:
            import torch
            self._ctx = torch.cuda.device(self.dev)
            self._ctx.__enter__()
        self.stream = _stream_handle(self._stream, self.dev)
        return self

    def __exit__(self, *exc):
        if self._ctx is not None:
            self._ctx.__exit__(*exc)
        return False


class Geometry:
    """Owns one `cbct_geom*` handle (A1, `cbct_geom_create`)."""

    def __init__(self, *, sid_mm=1000.0, sdd_mm=1536.0, n_views, det_nu, det_nv, det_du_mm, det_dv_mm,
                 det_off_u_mm=0.0, det_off_v_mm=0.0, vol_nx, vol_ny, vol_nz, vox_mm,
                 vol_cx_mm=0.0, vol_cy_mm=0.0, vol_cz_mm=0.0, step_vox=0.5,
                 angles_rad: Optional[Sequence[float]] = None, max_workset_bytes: int = 0):
        L = load_library()
        d = GeomDesc()
        d.sid_mm, d.sdd_mm, d.n_views = sid_mm, sdd_mm, n_views
        d.det_nu, d.det_nv, d.det_du_mm, d.det_dv_mm = det_nu, det_nv, det_du_mm, det_dv_mm
        d.det_off_u_mm, d.det_off_v_mm = det_off_u_mm, det_off_v_mm
        d.vol_nx, d.vol_ny, d.vol_nz, d.vox_mm = vol_nx, vol_ny, vol_nz, vox_mm
        d.vol_cx_mm, d.vol_cy_mm, d.vol_cz_mm = vol_cx_mm, vol_cy_mm, vol_cz_mm
        d.step_vox, d.max_workset_bytes = step_vox, int(max_workset_bytes)
        if angles_rad is not None:
            a = np.ascontiguousarray(np.asarray(angles_rad, dtype=np.float64))
            if a.shape != (n_views,):
                raise CbctError("angles_rad must have n_views entries")
            d.angles_rad = a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        self.desc = d
        self._h = ctypes.c_void_p()
        _check(L.cbct_geom_create(ctypes.byref(d), ctypes.byref(self._h)))
        self.n_vol = vol_nx * vol_ny * vol_nz
        self.n_sino = n_views * det_nv * det_nu
        self.vol_shape = (vol_nz, vol_ny, vol_nx)
        self.sino_shape = (n_views, det_nv, det_nu)

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            load_library().cbct_geom_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- the hot path -------------------------------------------------------
    def fp(self, vol, sino, channels: int = 1, stream=None):
        """cbct_fp: vol[C,nz,ny,nx] -> sino[C,n_views,nv,nu] (overwritten)."""
        pv, ps = _ptr_and_keep(vol, channels * self.n_vol), _ptr_and_keep(sino, channels * self.n_sino)
        with _on_device_of((vol, sino), stream) as cx:
            _check(load_library().cbct_fp(self._h, pv, ps, channels, cx.stream))
        return sino

    def bp_adjoint(self, sino, vol, channels: int = 1, stream=None):
        """cbct_bp_adjoint: sino -> vol (overwritten), exact transpose of fp."""
        ps, pv = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(vol, channels * self.n_vol)
        with _on_device_of((vol, sino), stream) as cx:
            _check(load_library().cbct_bp_adjoint(self._h, ps, pv, channels, cx.stream))
        return vol

    def bp_fdk(self, sino, vol, channels: int = 1, stream=None):
        """cbct_bp_fdk: FDK-weighted voxel-driven backprojection stage."""
        ps, pv = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(vol, channels * self.n_vol)
        with _on_device_of((vol, sino), stream) as cx:
            _check(load_library().cbct_bp_fdk(self._h, ps, pv, channels, cx.stream))
        return vol

    def bp_fdk_static(self, sino, vol, channels: int = 1, stream=None):
        """cbct_bp_fdk_static: bp_fdk on device tensors without any allocation (scratch in the library's static
        device array of STATIC_SCRATCH_BYTES; calls that overlap on the GPU race on it)."""
        ps, pv = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(vol, channels * self.n_vol)
        with _on_device_of((vol, sino), stream) as cx:
            L = load_library()
            rc = L.cbct_bp_fdk_static(self._h, ps, pv, channels, cx.stream)
            if rc == -2:
                raise CbctError(f"{L.cbct_status_string(rc).decode()} [{L.cbct_last_cuda_error().decode()}]")
            _check(rc)
        return vol

    def slab_planes(self, z0: int, z1: int, mirror_pair: bool = False) -> int:
        """Planes per channel that bp_adjoint_slab / bp_fdk_slab write for the range [z0, z1)."""
        n = z1 - z0
        if not mirror_pair:
            return n
        nz = self.vol_shape[0]
        return 2 * n - (1 if nz - z1 < z1 else 0)

    def bp_adjoint_slab(self, sino, out, z0: int, z1: int, channels: int = 1, mirror_pair: bool = False, stream=None):
        """cbct_bp_adjoint_slab: planes [z0, z1) (+ their z-mirror images) of bp_adjoint, device tensors."""
        n_out = channels * self.slab_planes(z0, z1, mirror_pair) * self.vol_shape[1] * self.vol_shape[2]
        ps, po = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(out, n_out)
        with _on_device_of((sino, out), stream) as cx:
            _check(load_library().cbct_bp_adjoint_slab(self._h, ps, po, channels, z0, z1, 1 if mirror_pair else 0, cx.stream))
        return out

    def bp_fdk_slab(self, sino, out, z0: int, z1: int, channels: int = 1, mirror_pair: bool = False, stream=None):
        """cbct_bp_fdk_slab: planes [z0, z1) (+ their z-mirror images) of bp_fdk, device tensors."""
        n_out = channels * self.slab_planes(z0, z1, mirror_pair) * self.vol_shape[1] * self.vol_shape[2]
        ps, po = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(out, n_out)
        with _on_device_of((sino, out), stream) as cx:
            _check(load_library().cbct_bp_fdk_slab(self._h, ps, po, channels, z0, z1, 1 if mirror_pair else 0, cx.stream))
        return out

    # --- NEXT-1: FDK front end ------------------------------------------------
    def fdk_filter(self, sino_in, sino_out, channels: int = 1, redundancy: bool = True, stream=None):
        """cbct_fdk_filter: weighted + ramp-filtered projections q such that bp_fdk(q) = FDK_w."""
        pi, po = _ptr_and_keep(sino_in, channels * self.n_sino), _ptr_and_keep(sino_out, channels * self.n_sino)
        with _on_device_of((sino_in, sino_out), stream) as cx:
            _check(load_library().cbct_fdk_filter(self._h, pi, po, channels, 1 if redundancy else 0, cx.stream))
        return sino_out

    def redundancy_weight(self, sino_in, sino_out, channels: int = 1, stream=None):
        """cbct_redundancy_weight: sino_out = w(u) * sino_in (in place allowed)."""
        pi, po = _ptr_and_keep(sino_in, channels * self.n_sino), _ptr_and_keep(sino_out, channels * self.n_sino)
        with _on_device_of((sino_in, sino_out), stream) as cx:
            _check(load_library().cbct_redundancy_weight(self._h, pi, po, channels, cx.stream))
        return sino_out

    def redundancy_weights(self) -> np.ndarray:
        w = np.empty(self.desc.det_nu, dtype=np.float64)
        _check(load_library().cbct_geom_redundancy_weights(
            self._h, w.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
        return w

    # --- NEXT-3: fused variants ------------------------------------------------
    def fp_residual(self, vol, y, sino, channels: int = 1, stream=None):
        """cbct_fp_residual: sino = P vol - y (y: device sinogram)."""
        pv, py = _ptr_and_keep(vol, channels * self.n_vol), _ptr_and_keep(y, channels * self.n_sino)
        ps = _ptr_and_keep(sino, channels * self.n_sino)
        with _on_device_of((vol, y, sino), stream) as cx:
            _check(load_library().cbct_fp_residual(self._h, pv, py, ps, channels, cx.stream))
        return sino

    def bp_adjoint_weighted(self, sino, vol, channels: int = 1, stream=None):
        """cbct_bp_adjoint_weighted: vol = P^T (w(u) * sino)."""
        ps, pv = _ptr_and_keep(sino, channels * self.n_sino), _ptr_and_keep(vol, channels * self.n_vol)
        with _on_device_of((sino, vol), stream) as cx:
            _check(load_library().cbct_bp_adjoint_weighted(self._h, ps, pv, channels, cx.stream))
        return vol

    # --- NEXT-2: field-of-view tensor -----------------------------------------
    def fov(self, vol_out, stream=None):
        """cbct_fov: V[nz,ny,nx] = fraction of views in which each voxel is visible."""
        po = _ptr_and_keep(vol_out, self.n_vol)
        with _on_device_of((vol_out,), stream) as cx:
            _check(load_library().cbct_fov(self._h, po, cx.stream))
        return vol_out

    # --- host-side queries --------------------------------------------------
    def count_samples(self) -> int:
        out = ctypes.c_uint64()
        _check(load_library().cbct_geom_count_samples(self._h, ctypes.byref(out)))
        return int(out.value)

    def num_slabs(self, channels: int = 1) -> int:
        out = ctypes.c_int32()
        _check(load_library().cbct_geom_num_slabs(self._h, channels, ctypes.byref(out)))
        return int(out.value)

    def symmetry(self):
        """cbct_geom_symmetry: (rotations in {4, 2, 1}, z-mirror flag) of the geometry."""
        r, m = ctypes.c_int32(), ctypes.c_int32()
        _check(load_library().cbct_geom_symmetry(self._h, ctypes.byref(r), ctypes.byref(m)))
        return int(r.value), bool(m.value)

    def workspace_bytes(self) -> int:
        """cbct_geom_workspace_bytes: device bytes of workspace the handle owns right now."""
        out = ctypes.c_uint64()
        _check(load_library().cbct_geom_workspace_bytes(self._h, ctypes.byref(out)))
        return int(out.value)

    def reserve(self, channels: int = 1):
        """cbct_geom_reserve: allocate all workspace for device-pointer calls with up to `channels` channels."""
        _check(load_library().cbct_geom_reserve(self._h, channels))

    def profile(self, enable: bool = True):
        """cbct_geom_profile: record a CUDA-event pair around every main-kernel launch."""
        _check(load_library().cbct_geom_profile(self._h, 1 if enable else 0))

    def profile_read(self, kernel: int):
        """cbct_geom_profile_read: (summed launch ms, launches) of kernel 0 fp / 1 adjoint / 2 fdk."""
        ms, n = ctypes.c_double(), ctypes.c_uint64()
        _check(load_library().cbct_geom_profile_read(self._h, kernel, ctypes.byref(ms), ctypes.byref(n)))
        return float(ms.value), int(n.value)

    def launch_count(self) -> int:
        out = ctypes.c_uint64()
        _check(load_library().cbct_geom_launch_count(self._h, ctypes.byref(out)))
        return int(out.value)


# --- NEXT-2: resampling operators of the multiscale scheme (plain arrays, no geometry) ---
def _shape4(t):
    shp = tuple(t.shape)
    if len(shp) < 3:
        raise CbctError("expected at least 3 dimensions")
    outer = int(np.prod(shp[:-3])) if len(shp) > 3 else 1
    return outer, shp[-3], shp[-2], shp[-1]


def downsample(vol_in, vol_out, factor: int, stream=None):
    """cbct_downsample: average pooling of the last three axes by `factor`."""
    o, nz, ny, nx = _shape4(vol_in)
    pi = _ptr_and_keep(vol_in, o * nz * ny * nx)
    po = _ptr_and_keep(vol_out, o * (nz // factor) * (ny // factor) * (nx // factor))
    with _on_device_of((vol_in, vol_out), stream) as cx:
        _check(load_library().cbct_downsample(pi, po, o, nz, ny, nx, factor, cx.stream))
    return vol_out


def upsample(vol_in, vol_out, factor: int, stream=None):
    """cbct_upsample: nearest upsampling of the last three axes by `factor`."""
    o, nz, ny, nx = _shape4(vol_in)
    pi = _ptr_and_keep(vol_in, o * nz * ny * nx)
    po = _ptr_and_keep(vol_out, o * nz * ny * nx * factor ** 3)
    with _on_device_of((vol_in, vol_out), stream) as cx:
        _check(load_library().cbct_upsample(pi, po, o, nz, ny, nx, factor, cx.stream))
    return vol_out


def proj_down(sino_in, sino_out, factor: int, stream=None):
    """cbct_proj_down: keep every `factor`-th view, average-pool the detector by `factor`."""
    o, nviews, nv, nu = _shape4(sino_in)
    pi = _ptr_and_keep(sino_in, o * nviews * nv * nu)
    po = _ptr_and_keep(sino_out, o * (-(-nviews // factor)) * (nv // factor) * (nu // factor))
    with _on_device_of((sino_in, sino_out), stream) as cx:
        _check(load_library().cbct_proj_down(pi, po, o, nviews, nv, nu, factor, cx.stream))
    return sino_out


def water_bone(rho_hat, rho_w, rho_b, tau0: float = 0.0, tau1: float = 1.2, tau2: float = 1.6,
               kappa_b: float = 0.409, stream=None):
    """cbct_water_bone: Eq. (3)-(4) water / bone densities of a modified-CT-number array (any shape)."""
    n = int(np.prod(rho_hat.shape))
    pr, pw, pb = (_ptr_and_keep(t, n) for t in (rho_hat, rho_w, rho_b))
    with _on_device_of((rho_hat, rho_w, rho_b), stream) as cx:
        _check(load_library().cbct_water_bone(pr, pw, pb, n, tau0, tau1, tau2, kappa_b, cx.stream))
    return rho_w, rho_b


def polychromatic_primary(pw, pb, i0, mu_w, mu_b, resp, out, stream=None):
    """cbct_polychromatic_primary: noise-free Eq. (6); pw, pb, out [n_views, nv, nu], i0 [n_bins, nv, nu]."""
    n_bins = len(resp)
    if len(mu_w) != n_bins or len(mu_b) != n_bins or i0.shape[0] != n_bins:
        raise CbctError("mu_w, mu_b, resp and i0 must agree on the number of energy bins")
    n_views = int(pw.shape[0])
    n_pix = int(np.prod(pw.shape[1:]))
    pa, pb_, po = (_ptr_and_keep(t, n_views * n_pix) for t in (pw, pb, out))
    pi = _ptr_and_keep(i0, n_bins * n_pix)
    arr = [(ctypes.c_double * n_bins)(*[float(x) for x in t]) for t in (mu_w, mu_b, resp)]
    with _on_device_of((pw, pb, i0, out), stream) as cx:
        _check(load_library().cbct_polychromatic_primary(pa, pb_, pi, arr[0], arr[1], arr[2], n_bins, n_views, n_pix,
                                                         po, cx.stream))
    return out
