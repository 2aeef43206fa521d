"""The operator calls of one LIRE++ inference, RECONSTRUCT of Algorithm 1, through the C ABI.

Row A6 of SURVEY.md s.8 (multi-channel / multi-scale driver): one geometry handle per scale alpha in {25 %, 50 %,
100 %} -- the volume at alpha of the full resolution, the detector average-pooled to alpha and "only every
1/alpha-th projection" -- and, per scale, the calls Alg. 1 makes:

    l.10-13  Downsample_alpha(x), ProjDown_alpha(y), ProjDown_alpha(y_raw), Downsample_alpha(V)
    l.16     P_alpha([p_2, x])          5 channels  (cbct_fp)
    l.18     P*_alpha(w d_2)            4 channels  (cbct_bp_adjoint_weighted)
    l.19     P*_alpha(P_alpha(x) - y)   1 channel   (cbct_bp_adjoint; P_alpha(x) is channel 4 of l.16)
    l.23     Upsample_{1/alpha}(.)      1 channel
    l.28     Upsample_200%(f), Upsample_200%(h)   8 channels each, i < 3

preceded by l.3 x = FDK_w(y) (cbct_fdk_filter + cbct_bp_fdk), l.5 P*(w y) and the FoV tensor V.
The learned blocks (GC-UNet, Gamma, Lambda, the 1x1x1 output convolution, Perm) are out of scope
and need trained weights: here their outputs are stand-ins (the dual block returns its d_2 input plus the mean of
p_op, and so on), so the *operator* sequence, shapes and channel counts are those of the paper and the values are
not a reconstruction.  Every array stays on the device; every step above runs in the library's kernels.

    python -m paper_2512_21180_b200.lire_ops [--views 400] [--n 256] [--reps 3]

prints one JSON line with the time of each group of calls (CUDA events), the operator share of one inference.
"""
from __future__ import annotations

import argparse
import json

import torch

from . import cbct

SCALES = (4, 2, 1)          # 1 / alpha for alpha = 25 %, 50 %, 100 %
PANEL_MM, OFFSET_MM = 409.6, 115.0
FOV_MM = 512.0              # 256^3 at 2 mm


class LireOperators:
    """Geometry handles and work buffers of the three scales (full grid n^3, detector n x n, n_views views)."""

    def __init__(self, n: int = 256, n_views: int = 400, latent_channels: int = 8, device="cuda",
                 fov_mm: float = FOV_MM, panel_mm: float = PANEL_MM, offset_mm: float = OFFSET_MM, angles_rad=None):
        """Any view count (the scanner delivers 432-944 projections) and, with `angles_rad`, any angle
        list: scale 1/f keeps views 0, f, 2f, ... of the full list (reading R14), ceil(n_views / f) of them."""
        if n % 4:
            raise cbct.CbctError("n must be divisible by 4 (three scales of average pooling)")
        self.n, self.n_views, self.C = n, n_views, latent_channels
        self.half = latent_channels // 2
        self.dev = torch.device(device)
        self.geoms = {}
        for f in SCALES:
            m = n // f
            self.geoms[f] = cbct.Geometry(
                **self.geom_kwargs(n, n_views, f, fov_mm, panel_mm, offset_mm, angles_rad))
        g = self.geoms[1]
        self.V = g.fov(torch.empty(g.vol_shape, device=self.dev))   # PAPER.md:169, once per geometry

    @staticmethod
    def geom_kwargs(n, n_views, f, fov_mm=FOV_MM, panel_mm=PANEL_MM, offset_mm=OFFSET_MM, angles_rad=None) -> dict:
        """Geometry of the scale alpha = 1 / f (plain numbers; the tests hand the same ones to the oracle)."""
        import math
        m = n // f
        kw = dict(n_views=-(-n_views // f), det_nu=m, det_nv=m, det_du_mm=panel_mm / m, det_dv_mm=panel_mm / m,
                  det_off_u_mm=offset_mm, vol_nx=m, vol_ny=m, vol_nz=m, vox_mm=fov_mm / m)
        if angles_rad is not None or n_views % f:
            full = list(angles_rad) if angles_rad is not None else [2.0 * math.pi * i / n_views for i in range(n_views)]
            kw["angles_rad"] = full[::f]
        return kw

    def _new(self, *shape):
        return torch.empty(shape, device=self.dev, dtype=torch.float32)

    def reconstruct_operators(self, y_raw: torch.Tensor, timings: dict | None = None):
        """The operator calls of RECONSTRUCT on projections y_raw[n_views, n, n]; returns the list I of l.24
        (stand-in values, see the module docstring).  `timings`: group name -> list of CUDA-event pairs."""
        g1, C, h = self.geoms[1], self.C, self.half

        class _Timer:
            def __init__(s, name):
                s.name = name
            def __enter__(s):
                if timings is not None:
                    s.a = torch.cuda.Event(enable_timing=True)
                    s.a.record()
            def __exit__(s, *exc):
                if timings is not None:
                    b = torch.cuda.Event(enable_timing=True)
                    b.record()
                    timings.setdefault(s.name, []).append((s.a, b))

        y = y_raw                                                # l.2: GC-UNet stand-in (identity)
        with _Timer("init_fdk_w"):                               # l.3
            q = g1.fdk_filter(y, self._new(*g1.sino_shape), 1, redundancy=True)
            x = g1.bp_fdk(q, self._new(*g1.vol_shape), 1)
        with _Timer("init_adjoint"):                             # l.5
            bp_full = g1.bp_adjoint_weighted(y, self._new(*g1.vol_shape), 1)
        with _Timer("resample"):                                 # l.4-6
            f0 = SCALES[0]
            m0 = self.n // f0
            xbar = cbct.downsample(x, self._new(m0, m0, m0), f0)
            x_bp = cbct.downsample(bp_full, self._new(m0, m0, m0), f0)
            ybar = cbct.proj_down(y, self._new(*self.geoms[f0].sino_shape), f0)
        f = torch.stack([xbar, x_bp] * (C // 2))                 # l.8
        hdual = ybar.unsqueeze(0).repeat(C, 1, 1, 1)             # l.9
        outputs = []
        for i, fac in enumerate(SCALES):
            g = self.geoms[fac]
            m = self.n // fac
            with _Timer("resample"):                             # l.10-13
                if fac > 1:
                    xbar = cbct.downsample(x, self._new(m, m, m), fac)
                    ybar = cbct.proj_down(y, self._new(*g.sino_shape), fac)
                    yraw_bar = cbct.proj_down(y_raw, self._new(*g.sino_shape), fac)
                    Vbar = cbct.downsample(self.V, self._new(m, m, m), fac)
                else:
                    xbar, ybar, yraw_bar, Vbar = x, y, y_raw, self.V
            d1, d2 = hdual[:h], hdual[h:]                        # l.14
            p1, p2 = f[:h], f[h:]                                # l.15
            with _Timer(f"fp_{m}"):                              # l.16
                p_in = torch.cat([p2, xbar.unsqueeze(0)]).contiguous()
                p_op = g.fp(p_in, self._new(h + 1, *g.sino_shape), h + 1)
            # l.17: Gamma stand-in
            d2 = (d2 + 1e-3 * (p_op.mean(0, keepdim=True) + d1.mean(0, keepdim=True) + ybar + yraw_bar)).contiguous()
            with _Timer(f"adjoint_{m}"):                         # l.18, l.19
                b_op = g.bp_adjoint_weighted(d2, self._new(h, *g.vol_shape), h)
                resid = (p_op[h] - ybar).contiguous()
                lw = g.bp_adjoint(resid, self._new(*g.vol_shape), 1)
            # l.20: Lambda stand-in
            p2 = p2 + 1e-3 * (b_op + p1.mean(0, keepdim=True) + xbar + lw + Vbar)
            hdual = torch.cat([d1, d2])                          # l.21
            f = torch.cat([p1, p2])                              # l.22
            with _Timer("resample"):                             # l.23
                upd = f.mean(0).contiguous()                     # Conv3d(f; theta_o) stand-in
                if fac > 1:
                    upd = cbct.upsample(upd, self._new(*g1.vol_shape), fac)
            x = x + 1e-3 * upd
            outputs.append(x)                                    # l.24
            hdual, f = hdual.roll(1, 0), f.roll(1, 0)            # l.26: Perm stand-in
            if i < len(SCALES) - 1:                              # l.28
                with _Timer("resample"):
                    m2 = 2 * m
                    f = cbct.upsample(f.contiguous(), self._new(C, m2, m2, m2), 2)
                    nxt = self.geoms[SCALES[i + 1]]
                    nv_c, nv_f = g.sino_shape[0], nxt.sino_shape[0]
                    hdual = cbct.upsample(hdual.contiguous(), self._new(C, 2 * nv_c, *nxt.sino_shape[1:]), 2)
                    if nv_f != 2 * nv_c:      # view counts that are no multiple of 4: fine view k <- coarse view k // 2
                        hdual = hdual[:, :nv_f].contiguous()
        return outputs


def measure(n: int = 256, views: int = 400, reps: int = 3) -> dict:
    """One warm-up pass, then `reps` timed passes of the operator sequence on seeded uniform(0,1) projections;
    CUDA-event time of each group of calls, averaged over the passes."""
    if not torch.cuda.is_available():
        raise cbct.CbctError("needs a CUDA device: there is no CPU fallback")
    ops = LireOperators(n, views)
    gen = torch.Generator(device="cuda").manual_seed(1234)
    y_raw = torch.rand((views, n, n), device="cuda", generator=gen)
    ops.reconstruct_operators(y_raw)                 # warm-up
    torch.cuda.synchronize()
    timings: dict = {}
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(reps):
        ops.reconstruct_operators(y_raw, timings)
    b.record()
    torch.cuda.synchronize()
    groups = {k: sum(s.elapsed_time(e) for s, e in v) / reps for k, v in timings.items()}
    return {"what": "operator calls of one LIRE++ RECONSTRUCT (Alg. 1), learned blocks replaced by stand-ins",
            "grid": n, "views": views, "reps": reps,
            "ms_by_group": {k: round(v, 3) for k, v in groups.items()},
            "ms_operators": round(sum(groups.values()), 3),
            "ms_wall_incl_standins": round(a.elapsed_time(b) / reps, 3)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=256)
    ap.add_argument("--views", type=int, default=400, help="the paper evaluates at 720 (PAPER.md:139)")
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    print(json.dumps(measure(args.n, args.views, args.reps)))


if __name__ == "__main__":
    main()
