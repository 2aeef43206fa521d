#!/usr/bin/env python
"""bench.py -- throughput of the cone-beam hot path on B200 (contract: see DESIGN.md s.8).

One "step" = one pass of the whole hot path over one batch of synthetic input:
cbct_fp + cbct_bp_adjoint + cbct_bp_fdk over all channels of the workload
(default: BASELINE.json configs[3], the 8-channel 256^3 / 400-view primal-dual
step).  `value` is the forward projector's Gsamples/s (in-support samples,
counted analytically in fp64 by cbct_geom_count_samples); the backprojectors'
Gvoxel-views/s are reported in `backprojection`.  All timing is CUDA events on
the launching stream; inputs (1.3 GB) are larger than L2.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "forward Gsamples/s at 256^3 (backprojection Gvoxel-views/s in `backprojection`)"
UNIT = "Gsamples/s"


# dram__bytes_read.sum + dram__bytes_write.sum per launch of each kernel at the default workload,
# from the ncu --set full captures summarised in profiles/r1_final.md (multichannel_256; fp and adjoint launches
# carry 4 channels, fdk launches 1).  Reported only for that workload.
NCU_DRAM_BYTES_PER_LAUNCH = {"fp4_pair_kernel": 0.579e9, "adjoint_gather_kernel": 7.39e9, "fdk_kernel": 0.209e9}


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                if out.returncode == 0 and out.stdout.strip():
                    self.rows.append([x.strip() for x in out.stdout.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        reasons = []
        for k, name in ((3, "hw_slowdown"), (4, "hw_thermal_slowdown"), (5, "sw_thermal_slowdown"),
                        (6, "sw_power_cap")):
            if any(r[k].lower().startswith("active") for r in self.rows):
                reasons.append(name)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(float(r[2]) for r in self.rows), "samples": len(self.rows), "reasons": reasons}


def oracle_sample(cfg, steps, warmup):
    """The fp64 oracle, as it stands, on a bounded sample of the workload:
    channel 0, every 16th view, forward projection (Gsamples/s)."""
    import numpy as np
    import oracle
    from paper_2512_21180_b200 import synth
    kw = synth.geom_kwargs(cfg)
    stride = 16 if cfg["n_views"] >= 64 else 1
    views = list(range(0, cfg["n_views"], stride))
    sub = dict(kw, n_views=len(views))
    og = oracle.Geom(**sub, angles_rad=[2 * np.pi * i / cfg["n_views"] for i in views])
    vol = synth.make_volume(cfg, channels=1).astype(np.float64)
    nsamp = oracle.count_samples(og)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.fp(og, vol)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    dt = sum(times) / len(times)
    return {"value": nsamp / dt / 1e9, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
            "sample": f"cbct_fp of channel 0, {len(views)} of {cfg['n_views']} views (every {stride}th), "
                      f"{nsamp:.3e} samples, {dt:.2f} s per pass"}, dt


def run_reference(args, cfg):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cb, dt = oracle_sample(cfg, max(1, min(args.steps, 3)), min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "note": "oracle on host cores, bounded sample"},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="multichannel_256")
    ap.add_argument("--channels", type=int, default=0, help="override the workload's channel count")
    ap.add_argument("--cap-gib", type=float, default=-1.0,
                    help="max_workset_bytes in GiB (0 = none); default: 1 for large_512 (BASELINE.json config 5), else 0. "
                         "With a cap the volumes live in pinned HOST memory and stream through z-slabs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-lire", action="store_true", help="skip the Alg. 1 operator-sequence timing (context)")
    args = ap.parse_args()

    from paper_2512_21180_b200 import synth
    cfg = dict(synth.CONFIGS[args.workload])
    if args.channels:
        cfg["channels"] = args.channels
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2512_21180_b200 import cbct
    from paper_2512_21180_b200 import dist as cdist

    rank, local, world = cdist.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    C = cfg["channels"]
    kw = synth.geom_kwargs(cfg)
    cap_gib = args.cap_gib if args.cap_gib >= 0 else (1.0 if cfg["name"] == "large_512" else 0.0)
    streamed = cap_gib > 0
    g = cbct.Geometry(**kw, max_workset_bytes=int(cap_gib * (1 << 30)))
    n_samples = g.count_samples()                    # per channel, analytic fp64 (host)
    n_vv = g.n_vol * cfg["n_views"]                  # voxel-views per channel
    # every rank works on its own batch of C channels (weak scaling, no data-path collective)
    vol_h = synth.make_volume(cfg)
    sino_h = synth.make_sinogram(cfg)
    # resident case: everything in HBM; streamed case: volumes in pinned host memory (A5)
    vol = torch.from_numpy(vol_h).pin_memory() if streamed else torch.from_numpy(vol_h).cuda()
    sino_in = torch.from_numpy(sino_h).cuda()
    sino_out = torch.empty_like(sino_in)
    vol_out = torch.empty_like(vol).pin_memory() if streamed else torch.empty_like(vol)

    def step(ev=None):
        if ev:
            ev[0].record()
        g.fp(vol, sino_out, C)
        if ev:
            ev[1].record()
        g.bp_adjoint(sino_in, vol_out, C)
        if ev:
            ev[2].record()
        g.bp_fdk(sino_in, vol_out, C)
        if ev:
            ev[3].record()

    for _ in range(args.warmup):
        step()
    cdist.barrier(cuda=True)
    l0 = g.launch_count()
    g.profile(True)   # CUDA-event pair around every fp / adjoint / fdk kernel launch, on their stream
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        for k in range(args.steps):
            step(evs[k])
        cdist.barrier(cuda=True)
    g.profile(False)
    launches = g.launch_count() - l0
    # groups of 4 channels go through fp4_pair_kernel; so do the remaining channels (as their four quarter-turn
    # images) when the geometry is symmetric under quarter turns, as every bench workload is: equispaced views,
    # n_views % 4 == 0, centred square grid.  Otherwise they take the quad-packed fp_kernel (one timing slot).
    quarter_turns = (cfg["n_views"] % 4 == 0 and cfg["vol_nx"] == cfg["vol_ny"]
                     and cfg.get("vol_cx_mm", 0.0) == 0.0 and cfg.get("vol_cy_mm", 0.0) == 0.0
                     and cfg.get("angles_rad") is None)
    fp_name = ("fp4_pair_kernel" if (C % 4 == 0 or quarter_turns)
               else ("fp_kernel" if C < 4 else "fp4_pair_kernel+fp_kernel"))
    kern = {name: g.profile_read(i) for i, name in enumerate((fp_name, "adjoint_gather_kernel", "fdk_kernel"))}
    t_fp = sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps
    t_adj = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps
    t_fdk = sum(e[2].elapsed_time(e[3]) for e in evs) / args.steps
    t_total = evs[0][0].elapsed_time(evs[-1][3]) / args.steps
    t_fp, t_adj, t_fdk, t_total = cdist.max_over_ranks([t_fp, t_adj, t_fdk, t_total], device="cuda")

    # NEXT-1 kernels (not part of the step): FDK front end and redundancy weighting over all channels
    next1 = None
    if not streamed:
        evn = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        g.fdk_filter(sino_in, sino_out, C)
        cdist.barrier(cuda=True)
        evn[0].record()
        for _ in range(3):
            g.fdk_filter(sino_in, sino_out, C)
        evn[1].record()
        for _ in range(3):
            g.redundancy_weight(sino_in, sino_out, C)
        evn[2].record()
        cdist.barrier(cuda=True)
        t_flt, t_w = evn[0].elapsed_time(evn[1]) / 3, evn[1].elapsed_time(evn[2]) / 3
        next1 = {"fdk_filter_ms": t_flt, "redundancy_weight_ms": t_w,
                 "redundancy_weight_hbm_gbs": 2 * sino_h.nbytes / (t_w * 1e-3) / 1e9,
                 "fdk_filter_gmacs": C * cfg["n_views"] * cfg["det_nv"] * cfg["det_nu"] * (cfg["det_nu"] // 2 + 1)
                 / (t_flt * 1e-3) / 1e9}
        # NEXT-2: FoV tensor and the resampling operators (streaming kernels: bytes moved / time)
        def timed(fn, reps=3):
            fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        n = cfg["vol_nx"]
        half = torch.empty((C, n // 2, n // 2, n // 2), device="cuda")
        pd = torch.empty((C, cfg["n_views"] // 2, cfg["det_nv"] // 2, cfg["det_nu"] // 2), device="cuda")
        t_fov = timed(lambda: g.fov(vol_out[0]))
        t_dn = timed(lambda: cbct.downsample(vol, half, 2))
        t_up = timed(lambda: cbct.upsample(half, vol_out, 2))
        t_pd = timed(lambda: cbct.proj_down(sino_in, pd, 2))
        next1.update({"fov_ms": t_fov, "fov_gvoxel_views_per_s": n_vv / (t_fov * 1e-3) / 1e9,
                      "downsample2_ms": t_dn, "downsample2_hbm_gbs": (vol_h.nbytes * 1.125) / (t_dn * 1e-3) / 1e9,
                      "upsample2_ms": t_up, "upsample2_hbm_gbs": (vol_h.nbytes * 1.125) / (t_up * 1e-3) / 1e9,
                      "proj_down2_ms": t_pd, "proj_down2_hbm_gbs": (sino_h.nbytes * 0.5 * 1.25) / (t_pd * 1e-3) / 1e9})

        if C >= 2:
            # NEXT-4: water-bone decomposition of one volume; noise-free polychromatic signal of one sinogram pair
            _, mu_w, mu_b, i0 = synth.spectrum_tables(cfg["det_nv"], cfg["det_nu"])
            d_i0 = torch.from_numpy(i0).cuda()
            resp = [5.0 + 0.375 * (e - 20.0) if e <= 60.0 else 20.0 - (e - 60.0) / 6.0 for e in (25.0 + 10.0 * np.arange(10))]
            t_wb = timed(lambda: cbct.water_bone(vol[0], vol_out[0], vol_out[1]))
            t_poly = timed(lambda: cbct.polychromatic_primary(sino_in[0], sino_in[1], d_i0, mu_w, mu_b, resp, sino_out[0]))
            next1.update({"water_bone_ms": t_wb, "water_bone_hbm_gbs": 3 * vol_h[0].nbytes / (t_wb * 1e-3) / 1e9,
                          "polychromatic_primary_ms": t_poly,
                          "polychromatic_primary_hbm_gbs": 3 * sino_h[0].nbytes / (t_poly * 1e-3) / 1e9})

    # end to end through the C ABI with HOST (pinned) buffers: copies inside the timed region
    e2e = None
    if not args.no_e2e and not streamed:
        hv, hs = torch.from_numpy(vol_h).pin_memory(), torch.from_numpy(sino_h).pin_memory()
        hso, hvo = torch.empty_like(hs).pin_memory(), torch.empty_like(hv).pin_memory()

        def e2e_step(ev=None):
            if ev:
                ev[0].record()
            g.fp(hv, hso, C)
            if ev:
                ev[1].record()
            g.bp_adjoint(hs, hvo, C)
            g.bp_fdk(hs, hvo, C)
            if ev:
                ev[2].record()
        e2e_step()
        cdist.barrier(cuda=True)
        ev2 = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
        for k in range(args.steps):
            e2e_step(ev2[k])
        cdist.barrier(cuda=True)
        te_fp, te_step = cdist.max_over_ranks([sum(e[0].elapsed_time(e[1]) for e in ev2) / args.steps,
                                               ev2[0][0].elapsed_time(ev2[-1][2]) / args.steps], device="cuda")
        e2e = {"value": world * C * n_samples / (te_fp * 1e-3) / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(vol_h.nbytes + 2 * sino_h.nbytes),
               "d2h_bytes_per_step": int(sino_h.nbytes + 2 * vol_h.nbytes),
               "ms_per_step": te_step, "fp_ms": te_fp,
               "note": "cbct_fp/bp_adjoint/bp_fdk called with pinned HOST buffers; value = forward Gsamples/s incl. copies"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk, pk_src = peaks()
    clocks = clk.summary()
    sm_hz = (clocks["sm_mhz"] or pk.get("sm_max_mhz", 1965.0)) * 1e6
    fwd = world * C * n_samples / (t_fp * 1e-3) / 1e9
    adj_vv = world * C * n_vv / (t_adj * 1e-3) / 1e9
    fdk_vv = world * C * n_vv / (t_fdk * 1e-3) / 1e9
    if streamed and not args.no_e2e:
        # the timed region already copies the volumes host <-> device inside every call
        e2e = {"value": fwd, "unit": UNIT, "h2d_bytes_per_step": int(vol_h.nbytes),
               "d2h_bytes_per_step": int(2 * vol_h.nbytes), "ms_per_step": t_total, "fp_ms": t_fp,
               "note": "streamed workload: volumes are pinned HOST buffers in the main timed region; "
                       "sinograms stay in HBM"}
    # Roofline of the dominant kernel (DESIGN.md s.7).  Algorithmic on-SM bytes per unit:
    # forward 32 B per sample (8 taps x 4 B through L1), adjoint 64 B per sample (the scatter form's
    # 8 tap read-modify-writes; the gather does less), FDK 16 B per voxel-view; peak =
    # 148 SMs x 128 B/clk x the SM clock sampled during the timed region.  Launch durations are the
    # library's own CUDA-event pairs around each kernel launch, on the launching stream.
    l1_peak = 148 * 128 * sm_hz / 1e9
    work = {fp_name: 32.0 * C * n_samples, "adjoint_gather_kernel": 64.0 * C * n_samples,
            "fdk_kernel": 16.0 * C * n_vv}     # algorithmic bytes per step
    per_kernel = {}
    for name, (ms, n) in kern.items():
        if n == 0:
            continue
        avg = ms / n
        per_launch = work[name] * args.steps / n
        per_kernel[name] = {"launches": n, "avg_launch_ms": avg, "achieved_gbs": per_launch / (avg * 1e-3) / 1e9,
                            "frac": per_launch / (avg * 1e-3) / 1e9 / l1_peak,
                            "share_of_step": ms / args.steps / t_total}
    dom = max(per_kernel, key=lambda k: kern[k][0])
    hbm_alg = C * 4.0 * (g.n_vol + g.n_sino) * args.steps / kern[dom][1]
    roofline = {"kernel": dom, "bound": "l1", "achieved": per_kernel[dom]["achieved_gbs"], "peak": l1_peak,
                "unit": "GB/s", "frac": per_kernel[dom]["frac"], "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(dom) if (cfg["name"] == "multichannel_256" and C == 8) else None,
                "peak_source": f"derived: 148 SM x 128 B/clk x {sm_hz / 1e6:.0f} MHz (L1 data path; MEASURED_PEAKS.json "
                               "has no L1 figure; HBM is not the bound, see hbm_frac)",
                "traffic_source": "profiles/r1_final.md (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum)",
                "hbm_frac": hbm_alg / (per_kernel[dom]["avg_launch_ms"] * 1e-3) / 1e9 / pk["hbm_gbs"],
                "hbm_peak_gbs": pk["hbm_gbs"], "hbm_peak_source": pk_src,
                "per_kernel": per_kernel,
                "note": "adjoint frac is against the scatter-form 64 B/sample figure; the gather shares weights "
                        "across rotated views / mirrored voxels / channels and can read above 1"}
    line = {"metric": METRIC, "value": fwd, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_total, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg["name"], "volume": [cfg["vol_nz"], cfg["vol_ny"], cfg["vol_nx"]],
                       "vox_mm": cfg["vox_mm"], "views": cfg["n_views"], "detector": [cfg["det_nv"], cfg["det_nu"]],
                       "channels": C, "step_vox": cfg["step_vox"], "l2": "inputs larger than L2 (no flush)",
                       "max_workset_gib": cap_gib, "slabs": g.num_slabs(C),
                       "volumes": "pinned host memory, streamed by z-slabs" if streamed else "HBM-resident",
                       "step": "cbct_fp + cbct_bp_adjoint + cbct_bp_fdk over all channels",
                       "sharding": "each rank runs its own C-channel batch; no data-path collective"},
            "backprojection": {"adjoint_gvoxel_views_per_s": adj_vv, "adjoint_gsamples_per_s":
                               world * C * n_samples / (t_adj * 1e-3) / 1e9,
                               "fdk_gvoxel_views_per_s": fdk_vv, "unit": "Gvoxel-views/s"},
            "call_ms": {"cbct_fp": t_fp, "cbct_bp_adjoint": t_adj, "cbct_bp_fdk": t_fdk},
            "samples_per_channel": n_samples, "voxel_views_per_channel": n_vv,
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}
    if next1:
        line["next"] = next1
    if e2e:
        line["e2e"] = e2e
    if not args.no_lire and world == 1 and cfg["name"] == "multichannel_256" and not streamed:
        # context, outside the step: the operator calls of one LIRE++ inference (Alg. 1) at this grid and view count
        from paper_2512_21180_b200 import lire_ops
        line["lire_ops"] = lire_ops.measure(cfg["vol_nx"], cfg["n_views"], reps=2)
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"], _ = oracle_sample(cfg, 1, 0)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
