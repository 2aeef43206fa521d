"""fp64 CPU oracle for the cone-beam operators -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around ``oracle/cbct_oracle.c`` (plain C, fp64, OpenMP).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It
imports nothing from ``paper_2512_21180_b200`` and shares no code with the
CUDA path.  Definitions: PAPER.md:85-89 (Eq. 5), PAPER.md:61 (geometry),
PAPER.md:157/181/397 (FDK); discretisation readings R1-R11 in DESIGN.md s.3.
The NEXT rows of SURVEY.md s.8(f) (FDK front end, FoV tensor, resampling, water-bone /
polychromatic mean) are plain numpy below, each citing its passage; pins P13-P17.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cbct_oracle.c")
_LIB = os.path.join(_HERE, "libcbct_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp).  Returns the .so path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-D_GNU_SOURCE",
           "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


class _CGeom(ctypes.Structure):
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
    ]


@dataclass
class Geom:
    """Geometry descriptor of the oracle (its own type; mirrors PAPER.md:61)."""
    sid_mm: float = 1000.0
    sdd_mm: float = 1536.0
    n_views: int = 36
    det_nu: int = 48
    det_nv: int = 48
    det_du_mm: float = 3.2
    det_dv_mm: float = 3.2
    det_off_u_mm: float = 0.0
    det_off_v_mm: float = 0.0
    vol_nx: int = 32
    vol_ny: int = 32
    vol_nz: int = 32
    vox_mm: float = 4.0
    vol_cx_mm: float = 0.0
    vol_cy_mm: float = 0.0
    vol_cz_mm: float = 0.0
    step_vox: float = 0.5
    angles_rad: Optional[Sequence[float]] = None
    _keep: list = field(default_factory=list, repr=False, compare=False)

    def vol_shape(self, channels: int = 1):
        return (channels, self.vol_nz, self.vol_ny, self.vol_nx)

    def sino_shape(self, channels: int = 1):
        return (channels, self.n_views, self.det_nv, self.det_nu)

    def _c(self) -> _CGeom:
        c = _CGeom()
        for name, _ in _CGeom._fields_:
            if name == "angles_rad":
                continue
            setattr(c, name, getattr(self, name))
        if self.angles_rad is not None:
            a = np.ascontiguousarray(np.asarray(self.angles_rad, dtype=np.float64))
            assert a.shape == (self.n_views,)
            self._keep.append(a)
            c.angles_rad = a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        else:
            c.angles_rad = ctypes.POINTER(ctypes.c_double)()
        return c


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        gp = ctypes.POINTER(_CGeom)
        L.oracle_max_threads.restype = ctypes.c_int
        L.oracle_fp.argtypes = [gp, dp, dp, ctypes.c_int, ctypes.c_int]
        L.oracle_fp_rays.argtypes = [gp, dp, ctypes.c_int, ip, ctypes.c_int64, dp]
        L.oracle_count_samples.argtypes = [gp, ctypes.c_int]
        L.oracle_count_samples.restype = ctypes.c_int64
        L.oracle_bp_adjoint.argtypes = [gp, dp, dp, ctypes.c_int, ctypes.c_int]
        L.oracle_bp_adjoint_voxels.argtypes = [gp, dp, ctypes.c_int, ip, ctypes.c_int64, dp]
        L.oracle_bp_fdk.argtypes = [gp, dp, dp, ctypes.c_int]
        L.oracle_bp_fdk_voxels.argtypes = [gp, dp, ctypes.c_int, ip, ctypes.c_int64, dp]
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _iptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def _as_f64(a, shape_tail):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if a.ndim == len(shape_tail):
        a = a[None]
    assert a.shape[1:] == tuple(shape_tail), (a.shape, shape_tail)
    return a


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def fp(g: Geom, vol, clip: bool = True) -> np.ndarray:
    """A2: vol[C,nz,ny,nx] -> sino[C,n_views,nv,nu] (fp64)."""
    vol = _as_f64(vol, g.vol_shape()[1:])
    out = np.empty(g.sino_shape(vol.shape[0]), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_fp(ctypes.byref(cg), _dptr(vol), _dptr(out), vol.shape[0], int(clip))
    assert rc == 0
    return out


def fp_rays(g: Geom, vol, ray_idx) -> np.ndarray:
    """A2 at selected flat ray indices ((i*nv+iv)*nu+iu) -> out[C, n_rays]."""
    vol = _as_f64(vol, g.vol_shape()[1:])
    idx = np.ascontiguousarray(np.asarray(ray_idx, dtype=np.int64))
    out = np.empty((vol.shape[0], idx.size), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_fp_rays(ctypes.byref(cg), _dptr(vol), vol.shape[0], _iptr(idx), idx.size, _dptr(out))
    assert rc == 0
    return out


def count_samples(g: Geom, clip: bool = True) -> int:
    """Number of (ray, k) samples with -1 < q < N on every axis (one channel)."""
    cg = g._c()
    return int(lib().oracle_count_samples(ctypes.byref(cg), int(clip)))


def bp_adjoint(g: Geom, sino, clip: bool = True) -> np.ndarray:
    """A3: sino[C,n_views,nv,nu] -> vol[C,nz,ny,nx] (fp64), exact transpose of fp."""
    sino = _as_f64(sino, g.sino_shape()[1:])
    out = np.empty(g.vol_shape(sino.shape[0]), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_bp_adjoint(ctypes.byref(cg), _dptr(sino), _dptr(out), sino.shape[0], int(clip))
    assert rc == 0
    return out


def bp_adjoint_voxels(g: Geom, sino, vox_idx) -> np.ndarray:
    """A3 at selected flat voxel indices ((iz*ny+iy)*nx+ix) -> out[C, n_vox]."""
    sino = _as_f64(sino, g.sino_shape()[1:])
    idx = np.ascontiguousarray(np.asarray(vox_idx, dtype=np.int64))
    out = np.empty((sino.shape[0], idx.size), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_bp_adjoint_voxels(ctypes.byref(cg), _dptr(sino), sino.shape[0], _iptr(idx),
                                        idx.size, _dptr(out))
    assert rc == 0
    return out


def bp_fdk(g: Geom, sino) -> np.ndarray:
    """A4: FDK-weighted voxel-driven backprojection (backprojection stage only)."""
    sino = _as_f64(sino, g.sino_shape()[1:])
    out = np.empty(g.vol_shape(sino.shape[0]), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_bp_fdk(ctypes.byref(cg), _dptr(sino), _dptr(out), sino.shape[0])
    assert rc == 0
    return out


def bp_fdk_voxels(g: Geom, sino, vox_idx) -> np.ndarray:
    """A4 at selected flat voxel indices -> out[C, n_vox]."""
    sino = _as_f64(sino, g.sino_shape()[1:])
    idx = np.ascontiguousarray(np.asarray(vox_idx, dtype=np.int64))
    out = np.empty((sino.shape[0], idx.size), dtype=np.float64)
    cg = g._c()
    rc = lib().oracle_bp_fdk_voxels(ctypes.byref(cg), _dptr(sino), sino.shape[0], _iptr(idx),
                                    idx.size, _dptr(out))
    assert rc == 0
    return out


def fdk_frontend(g: Geom, proj) -> np.ndarray:
    """Caller-side FDK steps (reading R11; textbook Feldkamp, ref [9] PAPER.md:397;
    ramp taps as in Kak & Slaney eq. 61 for equispaced flat detectors):
      p~ = p * SDD / sqrt(SDD^2 + u^2 + v^2)         (cosine weight)
      q  = a * (h * p~) along u,  a = du*SID/SDD,     (ramp filter, virtual
           h[0] = 1/(4 a^2), h[odd n] = -1/(pi^2 n^2 a^2), h[even] = 0   detector at isocentre)
    and the reconstruction is (dphi/2) * bp_fdk(q).  proj[n_views,nv,nu] fp64."""
    proj = np.asarray(proj, dtype=np.float64)
    nu, nv = g.det_nu, g.det_nv
    u = (np.arange(nu) - 0.5 * (nu - 1)) * g.det_du_mm + g.det_off_u_mm
    v = (np.arange(nv) - 0.5 * (nv - 1)) * g.det_dv_mm + g.det_off_v_mm
    cosw = g.sdd_mm / np.sqrt(g.sdd_mm ** 2 + u[None, :] ** 2 + v[:, None] ** 2)
    pt = proj * cosw[None]
    a = g.det_du_mm * g.sid_mm / g.sdd_mm
    n = np.arange(-(nu - 1), nu)
    h = np.zeros(n.shape, dtype=np.float64)
    h[n == 0] = 1.0 / (4.0 * a * a)
    odd = (n % 2) != 0
    h[odd] = -1.0 / (np.pi ** 2 * n[odd].astype(np.float64) ** 2 * a * a)
    out = np.empty_like(pt)
    for i in range(pt.shape[0]):
        for r in range(nv):
            out[i, r] = a * np.convolve(pt[i, r], h)[nu - 1:2 * nu - 1]
    return out


def redundancy_weight(g: Geom) -> np.ndarray:
    """Projection-domain redundancy weight w(u) for a laterally displaced detector ("FDK_w",
    "P*(w y)": PAPER.md:167, :181, :186 name the weighting but give no formula -- reading R12,
    DESIGN.md s.3: the smooth sine weighting of displaced-detector FDK, G. Wang, Med. Phys. 29 (2002)).
    With the detector covering [u_min, u_max] (pixel CENTRES, mm, offset included) and
    tau = min(|u_min|, |u_max|) the half-width of the band measured twice over a full turn:
        w(u) = 1/2 (sin(pi atan(u/SDD) / (2 atan(tau/SDD))) + 1)   for |u| <= tau,
        w(u) = 1 beyond tau on the long side (0 on the other side, which holds no pixels),
    mirrored if the long side is the negative one; a centred detector (u_min = -u_max) gets
    w = 1/2 everywhere.  Conjugate rays u and -u then always weigh w(u) + w(-u) = 1.  Returns w[nu]."""
    nu = g.det_nu
    u = (np.arange(nu) - 0.5 * (nu - 1)) * g.det_du_mm + g.det_off_u_mm
    umin, umax = u[0], u[-1]
    if abs(umin + umax) <= 1e-9 * max(abs(umin), abs(umax), 1.0) or umin * umax >= 0.0:
        # centred detector: every ray is measured twice; a detector entirely on one side of the
        # central ray has no doubly-measured band at all -- uniform weights in both cases
        return np.full(nu, 0.5 if umin * umax < 0.0 or nu == 1 else 1.0)
    sgn = 1.0 if umax > -umin else -1.0          # long side
    tau = min(-umin, umax)
    us = sgn * u
    w = np.where(us > tau, 1.0, 0.0)
    band = np.abs(us) <= tau
    w[band] = 0.5 * (np.sin(np.pi * np.arctan(us[band] / g.sdd_mm) / (2.0 * np.arctan(tau / g.sdd_mm))) + 1.0)
    return w


def fdk_filter(g: Geom, proj, redundancy: bool = True) -> np.ndarray:
    """Complete FDK front end (NEXT-1): q = dphi * fdk_frontend(w(u) * proj), dphi = 2 pi / n_views, so that
    bp_fdk(q) IS the FDK_w reconstruction.  With redundancy=False, w = 1/2 (the textbook
    dphi/2 of a centred detector, reading R11).  proj[C?, n_views, nv, nu]."""
    proj = np.asarray(proj, dtype=np.float64)
    w = redundancy_weight(g) if redundancy else np.full(g.det_nu, 0.5)
    dphi = 2.0 * np.pi / g.n_views
    if proj.ndim == 4:
        return np.stack([dphi * fdk_frontend(g, p * w) for p in proj])
    return dphi * fdk_frontend(g, proj * w)


# ---------------------------------------------------------------------------
# NEXT-2: field-of-view tensor and the resampling operators of the multiscale scheme
# ---------------------------------------------------------------------------
def fov(g: Geom) -> np.ndarray:
    """V(p) = (number of projections where voxel p is visible) / (total projection count).
    Reading R21 (DESIGN.md s.3): voxel p is visible in view i when its CENTRE projects onto the panel's
    active area, -1/2 <= fu < nu - 1/2 and -1/2 <= fv < nv - 1/2 in pixel-index coordinates (the union of the
    pixel footprints), with (fu, fv) as in the FDK backprojection (R9).  Returns V[nz, ny, nx] fp64."""
    x = g.vol_cx_mm + (np.arange(g.vol_nx) - 0.5 * (g.vol_nx - 1)) * g.vox_mm
    y = g.vol_cy_mm + (np.arange(g.vol_ny) - 0.5 * (g.vol_ny - 1)) * g.vox_mm
    z = g.vol_cz_mm + (np.arange(g.vol_nz) - 0.5 * (g.vol_nz - 1)) * g.vox_mm
    X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
    count = np.zeros((g.vol_nz, g.vol_ny, g.vol_nx), dtype=np.int64)
    angles = g.angles_rad if g.angles_rad is not None else [2.0 * np.pi * i / g.n_views for i in range(g.n_views)]
    for phi in angles:
        c, s = np.cos(phi), np.sin(phi)
        U = g.sid_mm - (X * c + Y * s)
        ustar = g.sdd_mm * (-X * s + Y * c) / U
        vstar = g.sdd_mm * Z / U
        fu = (ustar - g.det_off_u_mm) / g.det_du_mm + 0.5 * (g.det_nu - 1)
        fv = (vstar - g.det_off_v_mm) / g.det_dv_mm + 0.5 * (g.det_nv - 1)
        count += ((fu >= -0.5) & (fu < g.det_nu - 0.5) & (fv >= -0.5) & (fv < g.det_nv - 0.5))
    return count / float(g.n_views)


def downsample(z, factor: int) -> np.ndarray:
    """Downsample_alpha: average pooling of the last three axes by `factor` = 1/alpha
    (sizes must be multiples of factor).  z[..., nz, ny, nx] -> [..., nz/f, ny/f, nx/f]."""
    z = np.asarray(z, dtype=np.float64)
    f = factor
    nz, ny, nx = z.shape[-3:]
    assert nz % f == 0 and ny % f == 0 and nx % f == 0
    return z.reshape(z.shape[:-3] + (nz // f, f, ny // f, f, nx // f, f)).mean(axis=(-5, -3, -1))


def upsample(z, factor: int) -> np.ndarray:
    """Upsample ("nearest upsampling"): every voxel repeated `factor` times along the last
    three axes."""
    z = np.asarray(z, dtype=np.float64)
    for ax in (-3, -2, -1):
        z = np.repeat(z, factor, axis=ax)
    return z


def proj_down(p, factor: int) -> np.ndarray:
    """ProjDown_alpha: keeps every `factor`-th projection (views 0, f, 2f, ...; reading R14) and
    average-pools each kept projection by `factor` along both detector axes.  p[..., n_views, nv, nu]."""
    p = np.asarray(p, dtype=np.float64)[..., ::factor, :, :]
    f = factor
    nv, nu = p.shape[-2:]
    assert nv % f == 0 and nu % f == 0
    return p.reshape(p.shape[:-2] + (nv // f, f, nu // f, f)).mean(axis=(-3, -1))


# ---------------------------------------------------------------------------
# NEXT-4: water-bone decomposition (Eq. 3-4) and the noise-free polychromatic primary (Eq. 6)
# ---------------------------------------------------------------------------
def detector_response(energy_kev) -> np.ndarray:
    """resp(e): piecewise linear through r_20 = 5, r_60 = 20, r_120 = 10 (keV)."""
    return np.interp(np.asarray(energy_kev, dtype=np.float64), [20.0, 60.0, 120.0], [5.0, 20.0, 10.0])


def water_bone(rho_hat, tau0: float = 0.0, tau1: float = 1.2, tau2: float = 1.6, kappa_b: float = 0.409):
    """Eq. (3)-(4): relative water / bone densities as functions of the modified CT number
    rho_hat = 0.001 HU + 1.  tau_1, tau_2, kappa_b are the paper's constants; tau_0 (the lower cut of the water
    branch) is named but not given a value in the paper -- reading R23: a caller parameter, default 0."""
    r = np.asarray(rho_hat, dtype=np.float64)
    rw = np.where(r < tau0, 0.0, np.where(r < tau1, r, np.where(r < tau2, tau1 * (tau2 - r) / (tau2 - tau1), 0.0)))
    rb = np.where(r < tau1, 0.0, np.where(r < tau2, kappa_b * tau2 * (r - tau1) / (tau2 - tau1), kappa_b * r))
    return rw, rb


def polychromatic_primary(pw, pb, i0, mu_w, mu_b, resp) -> np.ndarray:
    """Noise-free mean of Eq. (6): sum_e resp(e) I_{0,e}(sigma) exp(-(mu_w(e) P rho_w + mu_b(e) P rho_b))
    (the projector is linear, so P(mu~_e^w + mu~_e^b) = mu_w(e) P(rho_w) + mu_b(e) P(rho_b)).
    pw, pb: [n_views, nv, nu] line integrals of rho_w, rho_b (mm); i0: [n_bins, nv, nu] unattenuated counts per bin
    and detector element; mu_w, mu_b: [n_bins] attenuation per unit relative density (1/mm); resp: [n_bins]."""
    pw, pb, i0 = (np.asarray(a, dtype=np.float64) for a in (pw, pb, i0))
    out = np.zeros_like(pw)
    for e in range(len(resp)):
        out += resp[e] * i0[e][None] * np.exp(-(mu_w[e] * pw + mu_b[e] * pb))
    return out
