"""Seeded synthetic inputs and the BASELINE.json workload table.

This module serves BOTH the CUDA path's tests/bench and the fp64 oracle's
tests.  It holds none of the method's arithmetic (no projector, no geometry
maths): only plain numbers describing the workloads (BASELINE.json `configs`,
shaped like PAPER.md:61, :137, :139) and seeded random phantoms / sinograms.
The paper's clinical CTs are private; these phantoms stand in
for them (recipe: SURVEY.md s.8(d), DESIGN.md s.4).
"""
from __future__ import annotations

import numpy as np

# Elekta-like geometry: SID 1000 mm, isocentre-detector 536 mm,
# 115 mm lateral detector offset, 409.6 mm panel with 256x256 pixels.
_COMMON = dict(sid_mm=1000.0, sdd_mm=1536.0, det_off_v_mm=0.0,
               vol_cx_mm=0.0, vol_cy_mm=0.0, vol_cz_mm=0.0, step_vox=0.5)


def _cfg(name, n, vox, nu, du, nviews, off_u, channels, seed, n_ell, cylinder):
    d = dict(_COMMON)
    d.update(name=name, vol_nx=n, vol_ny=n, vol_nz=n, vox_mm=float(vox),
             det_nu=nu, det_nv=nu, det_du_mm=float(du), det_dv_mm=float(du),
             det_off_u_mm=float(off_u), n_views=nviews, channels=channels,
             seed=seed, n_ellipsoids=n_ell, cylinder=cylinder)
    return d


CONFIGS = {
    # BASELINE.json configs[0..4]
    "tiny": _cfg("tiny", 32, 4.0, 48, 3.2, 36, 0.0, 1, 1001, 6, False),
    "small_halffan": _cfg("small_halffan", 64, 4.0, 128, 1.6, 90, 115.0, 1, 1002, 20, True),
    "pyramid_64": _cfg("pyramid_64", 64, 8.0, 256, 1.6, 400, 115.0, 1, 1003, 100, True),
    "pyramid_128": _cfg("pyramid_128", 128, 4.0, 256, 1.6, 400, 115.0, 1, 1003, 100, True),
    "pyramid_256": _cfg("pyramid_256", 256, 2.0, 256, 1.6, 400, 115.0, 1, 1003, 100, True),
    "multichannel_256": _cfg("multichannel_256", 256, 2.0, 256, 1.6, 400, 115.0, 8, 1004, 100, True),
    "large_512": _cfg("large_512", 512, 1.0, 512, 0.8, 720, 115.0, 4, 1005, 300, True),
}

# Variants of config 4 / config 3 whose view angles are what a real scanner delivers (432-944
# projections per scan "to approximate actual variability ... in real data"; gantry angle read-outs are not
# equispaced): `angle_jitter_deg` = half-width of a seeded uniform jitter added to the equispaced angles (sorted),
# and a view count that is no multiple of 4.  Neither has the quarter-turn symmetry between views.
CONFIGS["multichannel_256_jitter"] = dict(CONFIGS["multichannel_256"], name="multichannel_256_jitter",
                                          angle_jitter_deg=0.2)
CONFIGS["pyramid_256_jitter"] = dict(CONFIGS["pyramid_256"], name="pyramid_256_jitter", angle_jitter_deg=0.2)
CONFIGS["multichannel_256_v402"] = dict(CONFIGS["multichannel_256"], name="multichannel_256_v402", n_views=402)
CONFIGS["pyramid_256_v402"] = dict(CONFIGS["pyramid_256"], name="pyramid_256_v402", n_views=402)


def view_angles(cfg: dict):
    """Per-view angles in radians, or None for the equispaced default 2 pi i / n.  Jittered lists are seeded
    (default_rng(seed + 7)), uniform in +-angle_jitter_deg about the equispaced angles, sorted."""
    jit = float(cfg.get("angle_jitter_deg", 0.0))
    if jit == 0.0:
        return None
    n = cfg["n_views"]
    rng = np.random.default_rng(cfg["seed"] + 7)
    a = 2.0 * np.pi * np.arange(n) / n + np.deg2rad(rng.uniform(-jit, jit, size=n))
    return [float(x) for x in np.sort(a)]


GEOM_KEYS = ("sid_mm", "sdd_mm", "n_views", "det_nu", "det_nv", "det_du_mm", "det_dv_mm",
             "det_off_u_mm", "det_off_v_mm", "vol_nx", "vol_ny", "vol_nz", "vox_mm",
             "vol_cx_mm", "vol_cy_mm", "vol_cz_mm", "step_vox")


def geom_kwargs(cfg: dict) -> dict:
    """The plain geometry numbers of a config (keys shared by both descriptors), plus `angles_rad` when the
    config's view angles are not the equispaced default."""
    kw = {k: cfg[k] for k in GEOM_KEYS}
    ang = view_angles(cfg)
    if ang is not None:
        kw["angles_rad"] = ang
    return kw


def _quat_to_rot(q):
    w, x, y, z = q / np.linalg.norm(q)
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def draw_ellipsoids(seed: int, count: int, extent_mm: float, axis_unit_mm: float):
    """Seeded ellipsoids: centre ~ U(-0.3, 0.3)*extent per axis, semi-axes ~
    U(2, 10)*axis_unit, rotation = normalised 4 normals as a quaternion,
    density ~ U(0.01, 0.03) /mm.  Returns a list of (centre[3], semi[3], R[3,3], rho)."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(count):
        c = rng.uniform(-0.3, 0.3, size=3) * extent_mm
        a = rng.uniform(2.0, 10.0, size=3) * axis_unit_mm
        R = _quat_to_rot(rng.normal(size=4))
        rho = rng.uniform(0.01, 0.03)
        out.append((c, a, R, float(rho)))
    return out


def rasterise(ellipsoids, n: int, vox_mm: float, cylinder: bool = False,
              cyl_radius_mm: float = 110.0, cyl_rho: float = 0.02) -> np.ndarray:
    """Centre-sampled rasterisation (R18): voxel += rho if its centre is inside;
    overlaps add.  Returns fp32 [n, n, n] (z, y, x), volume centred on isocentre."""
    ax = (np.arange(n, dtype=np.float64) - 0.5 * (n - 1)) * vox_mm
    vol = np.zeros((n, n, n), dtype=np.float64)
    if cylinder:
        rr = ax[None, :] ** 2 + ax[:, None] ** 2  # [y, x]
        vol += np.where(rr <= cyl_radius_mm ** 2, cyl_rho, 0.0)[None, :, :]
    for c, a, R, rho in ellipsoids:
        rad = float(np.max(a))
        lo = [int(np.clip(np.searchsorted(ax, c[k] - rad) - 1, 0, n)) for k in range(3)]
        hi = [int(np.clip(np.searchsorted(ax, c[k] + rad) + 1, 0, n)) for k in range(3)]
        if any(h <= l for l, h in zip(lo, hi)):
            continue
        X = ax[lo[0]:hi[0]][None, None, :] - c[0]
        Y = ax[lo[1]:hi[1]][None, :, None] - c[1]
        Z = ax[lo[2]:hi[2]][:, None, None] - c[2]
        # body coordinates: R^T (x - c), scaled by the semi-axes
        s = 0.0
        for k in range(3):
            s = s + ((R[0, k] * X + R[1, k] * Y + R[2, k] * Z) / a[k]) ** 2
        vol[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] += np.where(s <= 1.0, rho, 0.0)
    return vol.astype(np.float32)


def config_ellipsoids(cfg: dict):
    n, h = cfg["vol_nx"], cfg["vox_mm"]
    name = cfg["name"]
    if name.startswith("pyramid") or name.startswith("multichannel_256"):
        # one phantom defined once in mm on the finest (256^3 / 2 mm) grid
        return draw_ellipsoids(cfg["seed"], cfg["n_ellipsoids"], 512.0, 2.0)
    return draw_ellipsoids(cfg["seed"], cfg["n_ellipsoids"], n * h, h)


def smoothed_noise(seed: int, n: int, sigma: float = 0.01) -> np.ndarray:
    """N(0, sigma) field smoothed by a 3^3 box mean with zero padding (R17)."""
    rng = np.random.default_rng(seed)
    x = rng.normal(0.0, sigma, size=(n, n, n))
    for axis in range(3):
        p = np.pad(x, [(1, 1) if a == axis else (0, 0) for a in range(3)])
        sl = [slice(None)] * 3
        acc = 0.0
        for o in range(3):
            sl[axis] = slice(o, o + n)
            acc = acc + p[tuple(sl)]
        x = acc / 3.0
    return x.astype(np.float32)


def make_volume(cfg: dict, channels: int | None = None) -> np.ndarray:
    """fp32 [C, nz, ny, nx]: channel 0 = ellipsoid (+cylinder) phantom; further
    channels = smoothed noise fields (BASELINE.json config 4)."""
    C = cfg["channels"] if channels is None else channels
    n = cfg["vol_nx"]
    vol = np.empty((C, n, n, n), dtype=np.float32)
    vol[0] = rasterise(config_ellipsoids(cfg), n, cfg["vox_mm"], cfg["cylinder"])
    for c in range(1, C):
        vol[c] = smoothed_noise(cfg["seed"] * 100 + c, n)
    return vol


def make_sinogram(cfg: dict, channels: int | None = None) -> np.ndarray:
    """fp32 U(0,1) sinogram [C, n_views, nv, nu] from default_rng(seed+1)."""
    C = cfg["channels"] if channels is None else channels
    rng = np.random.default_rng(cfg["seed"] + 1)
    return rng.random((C, cfg["n_views"], cfg["det_nv"], cfg["det_nu"]), dtype=np.float32)


def sample_indices(seed: int, total: int, count: int) -> np.ndarray:
    """Seeded sorted unique flat indices for sampled parity at full sizes."""
    rng = np.random.default_rng(seed)
    return np.unique(rng.integers(0, total, size=count, dtype=np.int64))


def spectrum_tables(nv: int, nu: int, n_bins: int = 10, seed: int = 5):
    """Made-up inputs for the polychromatic primary (NEXT-4): bin centres 25, 35, ... keV (PAPER.md:61 names ten
    bins centred 25..115 keV), attenuation per unit relative density and mm for "water" and "bone" as smooth
    decreasing power laws of the energy (NOT xraylib's tables, which are not in this container), and per-bin
    unattenuated counts i0[e, v, u] = spectrum weight x a smooth bow-tie-like beam profile x (1 + 2% seeded ripple).
    Returns (energies_kev, mu_w, mu_b, i0 fp32)."""
    e = 25.0 + 10.0 * np.arange(n_bins)
    mu_w = 0.016 + 0.011 * (60.0 / e) ** 2.7
    mu_b = 0.025 + 0.040 * (60.0 / e) ** 3.0
    spec = np.exp(-0.5 * ((e - 60.0) / 28.0) ** 2)
    spec *= 2.0e4 / spec.sum()
    u = (np.arange(nu) + 0.5) / nu - 0.5
    v = (np.arange(nv) + 0.5) / nv - 0.5
    profile = (0.35 + 0.65 * np.cos(np.pi * u) ** 2)[None, :] * (1.0 - 0.2 * v[:, None] ** 2)
    rng = np.random.default_rng(seed)
    ripple = 1.0 + 0.02 * rng.standard_normal((n_bins, nv, nu))
    i0 = (spec[:, None, None] * profile[None] * ripple).astype(np.float32)
    return e, mu_w, mu_b, i0
