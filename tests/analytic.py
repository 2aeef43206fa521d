"""Closed-form line integrals used to pin the oracle (tests only).

Rays follow PAPER.md:85-89 (Eq. 5) with the circular-orbit geometry of
PAPER.md:61: source s = SID (cos phi, sin phi, 0), detector pixel centre
p = -(SDD-SID)(cos phi, sin phi, 0) + u (-sin phi, cos phi, 0) + v (0,0,1).
"""
import numpy as np


def rays(geom, views=None):
    """Source positions [V,1,1,3] and unit directions [V,nv,nu,3] in world mm."""
    nviews = geom["n_views"]
    phi = 2.0 * np.pi * np.arange(nviews) / nviews
    if views is not None:
        phi = phi[np.asarray(views)]
    c, s = np.cos(phi), np.sin(phi)
    nu, nv = geom["det_nu"], geom["det_nv"]
    u = (np.arange(nu) - 0.5 * (nu - 1)) * geom["det_du_mm"] + geom["det_off_u_mm"]
    v = (np.arange(nv) - 0.5 * (nv - 1)) * geom["det_dv_mm"] + geom["det_off_v_mm"]
    sid, idd = geom["sid_mm"], geom["sdd_mm"] - geom["sid_mm"]
    src = np.stack([sid * c, sid * s, np.zeros_like(c)], -1)[:, None, None, :]
    px = (-idd * c)[:, None, None] - u[None, None, :] * s[:, None, None] + 0 * v[None, :, None]
    py = (-idd * s)[:, None, None] + u[None, None, :] * c[:, None, None] + 0 * v[None, :, None]
    pz = np.broadcast_to(v[None, :, None], px.shape)
    p = np.stack([px, py, pz], -1)
    d = p - src
    d = d / np.linalg.norm(d, axis=-1, keepdims=True)
    return src, d


def ellipsoid_sinogram(geom, ellipsoids, views=None):
    """sum_e rho_e * chord_e.  With o' = D^-1 R^T (o - c), d' = D^-1 R^T d the
    chord through the unit sphere is 2 sqrt(B^2 - A C) / A, A = |d'|^2,
    B = o'.d', C = |o'|^2 - 1 (|d| = 1 so the parameter is arc length)."""
    src, d = rays(geom, views)
    out = np.zeros(d.shape[:-1])
    for c, a, R, rho in ellipsoids:
        o1 = ((src - c) @ R) / a
        d1 = (d @ R) / a
        A = np.sum(d1 * d1, -1)
        B = np.sum(o1 * d1, -1)
        C = np.sum(o1 * o1, -1) - 1.0
        disc = B * B - A * C
        out += rho * np.where(disc > 0, 2.0 * np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)
    return out


def gaussian_sinogram(geom, centre, sigma, rho, views=None):
    """Line integral of rho*exp(-|x-c|^2 / 2 sigma^2) = rho sigma sqrt(2 pi) exp(-dist^2 / 2 sigma^2)."""
    src, d = rays(geom, views)
    w = np.asarray(centre) - src
    along = np.sum(w * d, -1)
    dist2 = np.sum(w * w, -1) - along ** 2
    return rho * sigma * np.sqrt(2 * np.pi) * np.exp(-dist2 / (2 * sigma ** 2))


def gaussian_volume(n, vox_mm, centre, sigma, rho, shift_vox=0.0):
    ax = (np.arange(n) - 0.5 * (n - 1) + shift_vox) * vox_mm
    X, Y, Z = ax[None, None, :], ax[None, :, None], ax[:, None, None]
    r2 = (X - centre[0]) ** 2 + (Y - centre[1]) ** 2 + (Z - centre[2]) ** 2
    return rho * np.exp(-r2 / (2 * sigma ** 2))


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
