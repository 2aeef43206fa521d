#!/usr/bin/env python
"""bench.py -- throughput of the cone-beam hot path on B200 (contract: see DESIGN.md s.7-8).

One "step" = one pass of the whole hot path over one batch of synthetic input:
cbct_fp + cbct_bp_adjoint + cbct_bp_fdk over all channels of the workload
(default: BASELINE.json configs[3], the 8-channel 256^3 / 400-view primal-dual
step).  `value` is the forward projector's Gsamples/s (in-support samples,
counted analytically in fp64 by cbct_geom_count_samples); the backprojectors'
Gvoxel-views/s are reported in `backprojection`.  All timing is CUDA events on
the launching stream; inputs (1.3 GB) are larger than L2.

  --workload NAME     a key of paper_2512_21180_b200.synth.CONFIGS (multichannel_256, pyramid_256, large_512,
                      multichannel_256_jitter / pyramid_256_jitter: +-0.2 degree jittered view angles,
                      multichannel_256_v402 / pyramid_256_v402: 402 views -- no quarter-turn symmetry, ...)
  --scaling strong    under torchrun: ONE batch split over the ranks (paper_2512_21180_b200/sharded.py: view-sharded
                      forward, one all-gather of the sinogram, plane-sharded backprojection) instead of one batch
                      per rank (weak, the default)
  --impl reference    the fp64 oracle on the host cores, on a bounded sample of the same workload
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

# Measured on-chip peaks of this pool's B200s (profiles/r1_l1_microbench.md, profiles/r2_microbench.md):
L1_BYTES_PER_CLK_SM = 512.0 / 4.05     # one 512-B LDG.128 request per 4.05 cycles per SM = 126.4 B/clk/SM
L2_READ_PEAK_GBS = 9170.0              # L2-resident 64 MB buffer read by all SMs with ld.global.cg
ISSUE_LANES_PER_CLK_SM = 128.0         # FP32 lanes: 4 warp-instructions per clock per SM (measured 3.89)
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_traffic.json")


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel: str, workload: str, channels: int):
    """dram / L2 bytes per launch of `kernel` from the ncu --set full capture summarised in profiles/r2_traffic.json
    (written beside the capture; keyed by kernel, workload and channel count).  None when there is no capture of
    this kernel for this workload: a stale figure is worse than none."""
    try:
        with open(TRAFFIC_FILE) as f:
            for rec in json.load(f)["captures"]:
                if rec["kernel"] == kernel and rec["workload"] == workload and rec["channels"] == channels:
                    return rec
    except Exception:
        pass
    return None


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


# ---------------------------------------------------------------------------------------------------------------
# The fp64 oracle, as it stands, on a BOUNDED sample of the workload: channel 0, every `stride`-th view.  All three
# operators are sums over views, so the sub-sinogram of those views is a legitimate sample for the backprojectors
# too.  Only this section (cpu_baseline legs, --impl reference) touches oracle/.
# ---------------------------------------------------------------------------------------------------------------
class OracleSample:
    def __init__(self, cfg, stride=None):
        import numpy as np
        import oracle
        from paper_2512_21180_b200 import synth
        self.np, self.oracle, self.cfg = np, oracle, cfg
        kw = synth.geom_kwargs(cfg)
        n = cfg["n_views"]
        if stride is None:
            stride = 16 if n >= 64 else 1
        self.stride = stride
        self.views = list(range(0, n, stride))
        ang = kw.pop("angles_rad", None) or [2 * np.pi * i / n for i in range(n)]
        self.og = oracle.Geom(**dict(kw, n_views=len(self.views)), angles_rad=[ang[i] for i in self.views])
        self.vol = synth.make_volume(cfg, channels=1).astype(np.float64)
        self.sino = synth.make_sinogram(cfg, channels=1)[:, self.views].astype(np.float64)
        self.n_samples = oracle.count_samples(self.og)
        self.n_vv = cfg["vol_nx"] * cfg["vol_ny"] * cfg["vol_nz"] * len(self.views)
        self.cores = oracle.max_threads()

    def what(self):
        return f"channel 0, {len(self.views)} of {self.cfg['n_views']} views (every {self.stride}th)"

    def time_op(self, op: str, passes: int = 1, warmup: int = 1):
        fn = {"fp": lambda: self.oracle.fp(self.og, self.vol),
              "adjoint": lambda: self.oracle.bp_adjoint(self.og, self.sino),
              "fdk": lambda: self.oracle.bp_fdk(self.og, self.sino)}[op]
        for _ in range(warmup):
            fn()
        t0 = time.perf_counter()
        for _ in range(passes):
            fn()
        return (time.perf_counter() - t0) / passes

    def baseline(self, op: str, passes: int = 1, warmup: int = 1):
        dt = self.time_op(op, passes, warmup)
        units, unit = (self.n_samples, UNIT) if op == "fp" else (self.n_vv, "Gvoxel-views/s")
        name = {"fp": "cbct_fp", "adjoint": "cbct_bp_adjoint", "fdk": "cbct_bp_fdk"}[op]
        return {"value": units / dt / 1e9, "unit": unit, "cores": self.cores, "kind": "oracle",
                "sample": f"{name} of {self.what()}: {units:.3e} {'samples' if op == 'fp' else 'voxel-views'}, "
                          f"{dt:.2f} s per pass, {warmup} warm-up + {passes} timed pass(es)"}


def run_reference(args, cfg):
    """--impl reference: the oracle times the same step (fp + adjoint + fdk) on its bounded sample, exactly
    args.warmup + args.steps times; the sample is thinned further if that would not finish within a few minutes."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    budget_s = 240.0
    smp = OracleSample(cfg)
    t_probe = sum(smp.time_op(op, 1, 0) for op in ("fp", "adjoint", "fdk"))      # one untimed step: also the page-in
    n_total = args.steps + args.warmup
    if t_probe * n_total > budget_s and len(smp.views) > 1:
        factor = int(t_probe * n_total / budget_s) + 1
        smp = OracleSample(cfg, stride=smp.stride * factor)
    for _ in range(args.warmup):
        for op in ("fp", "adjoint", "fdk"):
            smp.time_op(op, 1, 0)
    t = {"fp": 0.0, "adjoint": 0.0, "fdk": 0.0}
    for _ in range(args.steps):
        for op in t:
            t[op] += smp.time_op(op, 1, 0)
    for op in t:
        t[op] /= args.steps
    value = smp.n_samples / t["fp"] / 1e9
    cb = {"value": value, "unit": UNIT, "cores": smp.cores, "kind": "oracle",
          "sample": f"one step = cbct_fp + cbct_bp_adjoint + cbct_bp_fdk of {smp.what()}; "
                    f"{smp.n_samples:.3e} samples, {smp.n_vv:.3e} voxel-views per step"}
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sum(t.values()) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "note": "fp64 oracle on the host cores, bounded sample: " + smp.what()},
            "call_ms": {"cbct_fp": t["fp"] * 1e3, "cbct_bp_adjoint": t["adjoint"] * 1e3, "cbct_bp_fdk": t["fdk"] * 1e3},
            "backprojection": {"adjoint_gvoxel_views_per_s": smp.n_vv / t["adjoint"] / 1e9,
                               "fdk_gvoxel_views_per_s": smp.n_vv / t["fdk"] / 1e9, "unit": "Gvoxel-views/s"},
            "cpu_baseline": cb,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def work_models(C, n_samples, n_vv, rotations, mirror):
    """Algorithmic work per STEP of the three main kernels (DESIGN.md s.7), what the method itself must do:
    forward   8 taps x 4 B = 32 B through the L1 data path per in-support sample;
    FDK       4 taps x 4 B = 16 B through the L1 data path per voxel-view;
    adjoint   its sum has 8 non-zero terms per in-support sample and channel (the transposed taps).  A gather
              (no read-modify-write traffic at all) must, per term, add weight x pixel into an accumulator
              (1 FP32 instruction) and evaluate the weight -- 3 position updates, 3 tent functions, 2 products = 8
              FP32 instructions -- once per group of terms that legitimately share it: the weight depends on the
              geometry only, so it is shared by all C channels and by the `rotations` x (2 if mirror) symmetric
              images of the voxel.  Bound: FP32 issue (thread-instructions), not bytes."""
    share = rotations * (2 if mirror else 1) * C
    return {"fp": {"bound": "l1", "unit": "GB/s", "work": 32.0 * C * n_samples, "per_unit": "32 B per sample"},
            "fdk": {"bound": "l1", "unit": "GB/s", "work": 16.0 * C * n_vv, "per_unit": "16 B per voxel-view"},
            "adjoint": {"bound": "alu", "unit": "Ginstr/s", "work": 8.0 * C * n_samples * (1.0 + 8.0 / share),
                        "per_unit": f"8 terms per sample x (1 + 8 / {share}) FP32 instructions",
                        "sharing": share}}


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
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="under torchrun: weak = one batch per rank (default); strong = one batch split over the ranks")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-lire", action="store_true", help="skip the Alg. 1 operator-sequence timing (context)")
    ap.add_argument("--no-next", action="store_true", help="skip the timings of the NEXT-row kernels (context)")
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
    strong = args.scaling == "strong" and world > 1
    g = cbct.Geometry(**kw, max_workset_bytes=int(cap_gib * (1 << 30)))
    n_samples = g.count_samples()                    # per channel, analytic fp64 (host)
    n_vv = g.n_vol * cfg["n_views"]                  # voxel-views per channel
    rotations, mirror = g.symmetry()
    vol_h = synth.make_volume(cfg)
    sino_h = synth.make_sinogram(cfg)
    # resident case: everything in HBM; streamed case: volumes in pinned host memory (A5)
    vol = torch.from_numpy(vol_h).pin_memory() if streamed else torch.from_numpy(vol_h).cuda()
    sino_in = torch.from_numpy(sino_h).cuda()
    sino_out = torch.empty_like(sino_in)
    vol_out = torch.empty_like(vol).pin_memory() if streamed else torch.empty_like(vol)

    sharding = "each rank runs its own C-channel batch; no data-path collective"
    if strong:
        from paper_2512_21180_b200 import sharded
        if streamed:
            raise SystemExit("--scaling strong runs on HBM-resident batches")
        if C >= world:
            sharding = f"strong: the {C} channels split over {world} ranks (dist.channel_shard); no collective"

            def step(ev=None):
                if ev:
                    ev[0].record()
                sharded.channel_split(g, "fp", vol, sino_out, C, rank, world)
                if ev:
                    ev[1].record()
                sharded.channel_split(g, "bp_adjoint", sino_in, vol_out, C, rank, world)
                if ev:
                    ev[2].record()
                sharded.channel_split(g, "bp_fdk", sino_in, vol_out, C, rank, world)
                if ev:
                    ev[3].record()
        else:
            sg = sharded.ShardedGeometry(kw, rank, world)
            sharding = (f"strong: {C} channel(s) over {world} ranks: view-sharded cbct_fp + ONE all-gather of the "
                        "sinogram rows, plane-sharded cbct_bp_adjoint_slab / cbct_bp_fdk_slab")
            shard_out = torch.empty((C, len(sg.planes)) + tuple(g.vol_shape[1:]), device="cuda")

            def step(ev=None):
                if ev:
                    ev[0].record()
                sg.fp(vol, C)
                if ev:
                    ev[1].record()
                sg.bp_adjoint_local(sino_in, C, out=shard_out)
                if ev:
                    ev[2].record()
                sg.bp_fdk_local(sino_in, C, out=shard_out)
                if ev:
                    ev[3].record()
    else:
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

    prof_handles = [g] if not (strong and C < world) else [sg.part, sg.full]
    prof_handles = [h for h in prof_handles if h is not None]
    for _ in range(args.warmup):
        step()
    cdist.barrier(cuda=True)
    l0 = sum(h.launch_count() for h in prof_handles)
    for h in prof_handles:
        h.profile(True)   # CUDA-event pair around every fp / adjoint / fdk kernel launch, on their stream
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        for k in range(args.steps):
            step(evs[k])
        cdist.barrier(cuda=True)
    for h in prof_handles:
        h.profile(False)
    launches = sum(h.launch_count() for h in prof_handles) - l0
    kern = {}
    for i, key in enumerate(("fp", "adjoint", "fdk")):
        reads = [h.profile_read(i) for h in prof_handles]
        kern[key] = (sum(r[0] for r in reads), sum(r[1] for r in reads))
    t_fp = sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps
    t_adj = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps
    t_fdk = sum(e[2].elapsed_time(e[3]) for e in evs) / args.steps
    t_total = evs[0][0].elapsed_time(evs[-1][3]) / args.steps
    t_fp, t_adj, t_fdk, t_total = cdist.max_over_ranks([t_fp, t_adj, t_fdk, t_total], device="cuda")
    jobs = 1 if strong else world          # batches the whole job processed per step

    # context, outside the step: NEXT-row kernels over all channels (streaming kernels: bytes moved / time)
    next1 = None
    if not streamed and not args.no_next and not strong:
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
        t_flt = timed(lambda: g.fdk_filter(sino_in, sino_out, C))
        t_w = timed(lambda: g.redundancy_weight(sino_in, sino_out, C))
        n = cfg["vol_nx"]
        half = torch.empty((C, n // 2, n // 2, n // 2), device="cuda")
        pd = torch.empty((C, -(-cfg["n_views"] // 2), cfg["det_nv"] // 2, cfg["det_nu"] // 2), device="cuda")
        t_fov = timed(lambda: g.fov(vol_out[0]))
        t_dn = timed(lambda: cbct.downsample(vol, half, 2))
        t_up = timed(lambda: cbct.upsample(half, vol_out, 2))
        t_pd = timed(lambda: cbct.proj_down(sino_in, pd, 2))
        next1 = {"fdk_filter_ms": t_flt, "redundancy_weight_ms": t_w,
                 "redundancy_weight_hbm_gbs": 2 * sino_h.nbytes / (t_w * 1e-3) / 1e9,
                 "fdk_filter_gmacs": C * cfg["n_views"] * cfg["det_nv"] * cfg["det_nu"] * (cfg["det_nu"] // 2 + 1)
                 / (t_flt * 1e-3) / 1e9,
                 "fov_ms": t_fov, "fov_gvoxel_views_per_s": n_vv / (t_fov * 1e-3) / 1e9,
                 "downsample2_ms": t_dn, "downsample2_hbm_gbs": (vol_h.nbytes * 1.125) / (t_dn * 1e-3) / 1e9,
                 "upsample2_ms": t_up, "upsample2_hbm_gbs": (vol_h.nbytes * 1.125) / (t_up * 1e-3) / 1e9,
                 "proj_down2_ms": t_pd, "proj_down2_hbm_gbs": (sino_h.nbytes * 0.5 * 1.25) / (t_pd * 1e-3) / 1e9}
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
    if not args.no_e2e and not streamed and not strong:
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
    fwd = jobs * C * n_samples / (t_fp * 1e-3) / 1e9
    adj_vv = jobs * C * n_vv / (t_adj * 1e-3) / 1e9
    fdk_vv = jobs * C * n_vv / (t_fdk * 1e-3) / 1e9
    if streamed and not args.no_e2e:
        # the timed region already copies the volumes host <-> device inside every call
        e2e = {"value": fwd, "unit": UNIT, "h2d_bytes_per_step": int(vol_h.nbytes),
               "d2h_bytes_per_step": int(2 * vol_h.nbytes), "ms_per_step": t_total, "fp_ms": t_fp,
               "note": "streamed workload: volumes are pinned HOST buffers in the main timed region; "
                       "sinograms stay in HBM"}

    # ---- rooflines (DESIGN.md s.7).  Launch durations are the library's own CUDA-event pairs around each kernel
    # launch, on the launching stream; peaks: L1 data path 148 SMs x 126.4 B/clk (MEASURED: one LDG.128 request per
    # 4.05 cycles, profiles/r1_l1_microbench.md) x the SM clock sampled during the timed region; FP32 issue 148 SMs x
    # 128 lanes x that clock (measured 3.89 of 4 warp-instructions per clock per SM, profiles/r2_microbench.md)
    quarter_turns = rotations == 4 and cfg["vol_nx"] == cfg["vol_ny"]
    # channels outside a group of 4: their quarter-turn images (fp4_pair_kernel), else mirror-paired cells (fpm_kernel)
    # on z-symmetric geometries held resident, else quad-packed cells (fp_kernel)
    tail_kernel = "fpm_kernel" if (mirror and not streamed) else "fp_kernel"
    names = {"fp": ("fp4_pair_kernel" if (C % 4 == 0 or quarter_turns)
                    else (tail_kernel if C < 4 else "fp4_pair_kernel+" + tail_kernel)),
             "adjoint": None, "fdk": "fdk_kernel"}
    # adjoint (cbct_adjoint.cu: launch_gather_channels), on grids of 200 000 base voxels or more: with rotation
    # symmetry, blocks of 4 (or 8) channels take the voxel kernel and the remaining 1-3 channels the column-walk kernel;
    # without it (irregular angle lists) the column-walk kernel takes every block
    images = rotations * (2 if mirror else 1)
    large = g.n_vol // images >= 200000
    tail = C % 4 if images == 8 else (C % 8) % 4
    if large and images <= 2:
        names["adjoint"] = "adjoint_column_kernel"
    else:
        names["adjoint"] = ("adjoint_gather_kernel" if not (large and tail) else
                            ("adjoint_column_kernel" if C < 4 else "adjoint_gather_kernel+adjoint_column_kernel"))
    l1_peak = 148 * L1_BYTES_PER_CLK_SM * sm_hz / 1e9
    issue_peak = 148 * ISSUE_LANES_PER_CLK_SM * sm_hz / 1e9
    models = work_models(C, n_samples, n_vv, rotations, mirror)
    shard_frac = (1.0 / world) if strong else 1.0        # rank 0's share of the batch under --scaling strong
    per_kernel = {}
    for key, (ms, n) in kern.items():
        if n == 0:
            continue
        m = models[key]
        avg = ms / n
        per_launch = m["work"] * shard_frac * args.steps / n
        peak = l1_peak if m["bound"] == "l1" else issue_peak
        rec = {"launches": n, "avg_launch_ms": avg, "bound": m["bound"], "unit": m["unit"],
               "achieved": per_launch / (avg * 1e-3) / 1e9, "peak": peak,
               "frac": per_launch / (avg * 1e-3) / 1e9 / peak, "work_per_unit": m["per_unit"],
               "share_of_step": ms / args.steps / t_total}
        if key == "adjoint":
            # context only: the scatter-form figure of SURVEY.md s.8(d) (8 read-modify-writes = 64 B per sample); the
            # gather performs no such traffic, so this is NOT a roofline fraction of this kernel
            rec["scatter_form_64B_per_sample_over_l1_peak"] = \
                64.0 * C * n_samples * shard_frac * args.steps / n / (avg * 1e-3) / 1e9 / l1_peak
        tr = ncu_traffic(names[key], cfg["name"], C)
        if tr:
            rec["dram_bytes_per_launch"] = tr.get("dram_bytes")
            rec["l2_bytes_per_launch"] = tr.get("lts_bytes")
            if tr.get("lts_bytes"):
                rec["l2_frac"] = tr["lts_bytes"] / (avg * 1e-3) / 1e9 / L2_READ_PEAK_GBS
        per_kernel[names[key]] = rec
    dom_key = max((k for k in kern if kern[k][1]), key=lambda k: kern[k][0])
    dom = names[dom_key]
    hbm_alg = C * 4.0 * (g.n_vol + g.n_sino) * shard_frac * args.steps / kern[dom_key][1]
    roofline = {"kernel": dom, "bound": per_kernel[dom]["bound"], "achieved": per_kernel[dom]["achieved"],
                "peak": per_kernel[dom]["peak"], "unit": per_kernel[dom]["unit"], "frac": per_kernel[dom]["frac"],
                "traffic": per_kernel[dom].get("dram_bytes_per_launch"),
                "peak_source": (f"measured: 148 SM x 126.4 B/clk (4.05 cycles per 512-B LDG.128 request, "
                                f"profiles/r1_l1_microbench.md) x {sm_hz / 1e6:.0f} MHz sampled in the timed region"
                                if per_kernel[dom]["bound"] == "l1" else
                                f"148 SM x 128 FP32 lanes x {sm_hz / 1e6:.0f} MHz (measured 3.89 of 4 warp-instr/clk/SM, "
                                "profiles/r2_microbench.md)"),
                "traffic_source": "profiles/r2_traffic.json (ncu --set full: dram__bytes_read.sum + dram__bytes_write.sum, "
                                  "lts__t_bytes.sum per launch); null = no capture of this kernel on this workload",
                "hbm_frac": hbm_alg / (per_kernel[dom]["avg_launch_ms"] * 1e-3) / 1e9 / pk["hbm_gbs"],
                "hbm_peak_gbs": pk["hbm_gbs"], "hbm_peak_source": pk_src,
                "l2_read_peak_gbs": L2_READ_PEAK_GBS, "l2_peak_source": "measured, profiles/r2_microbench.md",
                "per_kernel": per_kernel}
    config = {"workload": cfg["name"], "volume": [cfg["vol_nz"], cfg["vol_ny"], cfg["vol_nx"]],
              "vox_mm": cfg["vox_mm"], "views": cfg["n_views"],
              "view_angles": ("equispaced" if "angles_rad" not in kw
                              else f"equispaced + seeded uniform jitter of +-{cfg['angle_jitter_deg']} deg, sorted"),
              "symmetry": {"view_rotations": rotations, "z_mirror": mirror},
              "detector": [cfg["det_nv"], cfg["det_nu"]], "channels": C, "step_vox": cfg["step_vox"],
              "l2": "inputs larger than L2 (no flush)", "max_workset_gib": cap_gib, "slabs": g.num_slabs(C),
              "volumes": "pinned host memory, streamed by z-slabs" if streamed else "HBM-resident",
              "step": "cbct_fp + cbct_bp_adjoint + cbct_bp_fdk over all channels", "sharding": sharding}
    if streamed:
        config["resident_beside_the_cap_bytes"] = int(2 * sino_h.nbytes)
        config["resident_note"] = ("max_workset_bytes caps the VOLUME bytes on the device; the sinogram of all channels "
                                   "and one re-laid-out copy of it stay resident beside the slabs")
        config["workspace_bytes"] = g.workspace_bytes()
    line = {"metric": METRIC, "value": fwd, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_total, "higher_is_better": True,
            "scaling": "strong" if strong else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config,
            "backprojection": {"adjoint_gvoxel_views_per_s": adj_vv, "adjoint_gsamples_per_s":
                               jobs * C * n_samples / (t_adj * 1e-3) / 1e9,
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
        smp = OracleSample(cfg)
        line["cpu_baseline"] = smp.baseline("fp", passes=1, warmup=1)
        line["cpu_baseline_adjoint"] = smp.baseline("adjoint", passes=1, warmup=1)
        line["cpu_baseline_fdk"] = smp.baseline("fdk", passes=1, warmup=1)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
