"""GPU parity: CUDA path (through the C ABI) vs the fp64 oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's:
forward / FDK rel-L2 <= 1e-5 and max-rel <= 1e-4, adjoint rel-L2 <= 1e-4,
fp32 adjoint identity <= 1e-5 (norm definitions: reading R16, DESIGN.md s.3).
"""
import numpy as np
import pytest

from paper_2512_21180_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def cbct():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct as m
    m.load_library()
    return m


def rel_l2(g, r):
    return float(np.linalg.norm((g - r).ravel()) / np.linalg.norm(r.ravel()))


def max_rel(g, r):
    """max |g-r| / max(|r|, 1e-3 * max|r|)  (R16)."""
    floor = 1e-3 * float(np.max(np.abs(r)))
    return float(np.max(np.abs(g - r) / np.maximum(np.abs(r), floor)))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_fp(m, kw, vol, **extra):
    g = m.Geometry(**kw, **extra)
    C = vol.shape[0]
    out = torch.full((C,) + g.sino_shape, float("nan"), device="cuda", dtype=torch.float32)
    g.fp(dev(vol), out, C)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def run_adj(m, kw, sino, **extra):
    g = m.Geometry(**kw, **extra)
    C = sino.shape[0]
    out = torch.full((C,) + g.vol_shape, float("nan"), device="cuda", dtype=torch.float32)
    g.bp_adjoint(dev(sino), out, C)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def run_fdk(m, kw, sino, **extra):
    g = m.Geometry(**kw, **extra)
    C = sino.shape[0]
    out = torch.full((C,) + g.vol_shape, float("nan"), device="cuda", dtype=torch.float32)
    g.bp_fdk(dev(sino), out, C)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def check_all_three(m, o, kw, vol, sino, tag=""):
    og = o.Geom(**kw)
    r = o.fp(og, vol.astype(np.float64))
    g = run_fp(m, kw, vol)
    assert rel_l2(g, r) <= 1e-5, (tag, "fp rel-L2", rel_l2(g, r))
    assert max_rel(g, r) <= 1e-4, (tag, "fp max-rel", max_rel(g, r))
    r = o.bp_adjoint(og, sino.astype(np.float64))
    g = run_adj(m, kw, sino)
    assert rel_l2(g, r) <= 1e-4, (tag, "adjoint rel-L2", rel_l2(g, r))
    r = o.bp_fdk(og, sino.astype(np.float64))
    g = run_fdk(m, kw, sino)
    assert rel_l2(g, r) <= 1e-5, (tag, "fdk rel-L2", rel_l2(g, r))
    assert max_rel(g, r) <= 1e-4, (tag, "fdk max-rel", max_rel(g, r))


def test_config1_tiny(cbct, oracle_mod):
    cfg = synth.CONFIGS["tiny"]
    check_all_three(cbct, oracle_mod, synth.geom_kwargs(cfg), synth.make_volume(cfg), synth.make_sinogram(cfg), "tiny")


def test_config2_small_halffan(cbct, oracle_mod):
    cfg = synth.CONFIGS["small_halffan"]
    check_all_three(cbct, oracle_mod, synth.geom_kwargs(cfg), synth.make_volume(cfg), synth.make_sinogram(cfg),
                    "small")


def test_ragged_sizes_offcentre_multichannel(cbct, oracle_mod):
    """Sizes that are no multiple of any tile, anisotropic grid, off-centre
    volume, both detector offsets, 3 channels (phantom + 2 noise fields)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(vol_nx=37, vol_ny=29, vol_nz=21, det_nu=50, det_nv=35, det_du_mm=3.0, det_dv_mm=2.7,
              det_off_u_mm=23.0, det_off_v_mm=-4.0, vol_cx_mm=5.0, vol_cy_mm=-3.0, vol_cz_mm=2.5, n_views=11)
    rng = np.random.default_rng(77)
    vol = rng.random((3, 21, 29, 37), dtype=np.float32)
    sino = rng.random((3, 11, 35, 50), dtype=np.float32)
    check_all_three(cbct, oracle_mod, kw, vol, sino, "ragged")


def test_noise_channels(cbct, oracle_mod):
    """Smoothed-noise channels of config 4 (signed values, no flat regions)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["small_halffan"]))
    kw.update(n_views=24)
    vol = np.stack([synth.smoothed_noise(5, 64), synth.smoothed_noise(6, 64)])
    og = oracle_mod.Geom(**kw)
    r = oracle_mod.fp(og, vol.astype(np.float64))
    g = run_fp(cbct, kw, vol)
    assert rel_l2(g, r) <= 1e-5
    # R16b (DESIGN.md s.3): these rays are ill-conditioned sums (|P f| << P|f|), and fp32
    # rounding scales with P|f|; the max-rel denominator is max(|r|, 0.1 P|f|, 1e-3 |r|_inf).
    ra = oracle_mod.fp(og, np.abs(vol).astype(np.float64))
    den = np.maximum(np.maximum(np.abs(r), 0.1 * ra), 1e-3 * float(np.max(np.abs(r))))
    # plain R16 is reported beside R16b (it is what a reader of BASELINE.json would compute first)
    record("noise_channels_fp", rel_l2=rel_l2(g, r), max_rel_R16=max_rel(g, r),
           max_rel_R16b=float(np.max(np.abs(g - r) / den)), peak=peak_err(g, r))
    assert float(np.max(np.abs(g - r) / den)) <= 1e-4
    assert peak_err(g, r) <= 1e-5


@pytest.mark.parametrize("case", [
    dict(n_views=12),                                  # 4 rotations + z mirror
    dict(n_views=12, vol_nz=27),                       # ... odd nz: the middle plane is its own mirror image
    dict(n_views=12, det_off_v_mm=3.0),                # 4 rotations, no mirror (detector not centred in z)
    dict(n_views=10, vol_nx=30, det_off_u_mm=20.0),    # 2 rotations (nx != ny, n % 4 != 0) + mirror
    dict(n_views=10, vol_cz_mm=6.0),                   # 2 rotations, no mirror
    dict(n_views=7),                                   # no rotation (odd view count) + mirror
    dict(n_views=8, vol_cx_mm=4.0),                    # off-centre grid: no rotation
    dict(n_views=8, vol_ny=31, vol_nx=31),             # odd grid: no rotation
    dict(n_views=8, irregular=True),                   # non-equispaced angles: no rotation
])
def test_backprojector_symmetry_paths(cbct, oracle_mod, case):
    """Both backprojectors share geometry between views related by a grid rotation and
    between z-mirrored voxels when the geometry allows; every combination must equal
    the oracle (adjoint: its plain transpose), 3 channels (odd count: both channel-block sizes)."""
    case = dict(case)
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    irregular = case.pop("irregular", False)
    kw.update(case)
    extra = {}
    if irregular:
        rng = np.random.default_rng(3)
        extra["angles_rad"] = list(np.sort(rng.uniform(0, 2 * np.pi, kw["n_views"])))
    rng = np.random.default_rng(21)
    sino = rng.random((3, kw["n_views"], kw["det_nv"], kw["det_nu"]), dtype=np.float32)
    og = oracle_mod.Geom(**kw, **extra)
    r = oracle_mod.bp_adjoint(og, sino.astype(np.float64))
    g = run_adj(cbct, kw, sino, **extra)
    assert rel_l2(g, r) <= 1e-4, rel_l2(g, r)
    assert max_rel(g, r) <= 1e-3, max_rel(g, r)
    r = oracle_mod.bp_fdk(og, sino.astype(np.float64))
    g = run_fdk(cbct, kw, sino, **extra)
    assert rel_l2(g, r) <= 1e-5, rel_l2(g, r)
    assert max_rel(g, r) <= 1e-4, max_rel(g, r)


def peak_err(g, r):
    """max |g - r| / max |r|: a per-element bound that does not depend on where the reference is small."""
    return float(np.max(np.abs(g - r)) / np.max(np.abs(r)))


SYMMETRY_CASES = [
    dict(n_views=12),                                  # 4 rotations + z mirror
    dict(n_views=12, vol_nz=27),                       # ... odd nz
    dict(n_views=12, det_off_v_mm=3.0),                # 4 rotations, no mirror
    dict(n_views=10, vol_nx=30, det_off_u_mm=20.0),    # 2 rotations + mirror
    dict(n_views=10, vol_cz_mm=6.0),                   # 2 rotations, no mirror
    dict(n_views=7),                                   # no rotation + mirror
    dict(n_views=8, vol_cx_mm=4.0),                    # off-centre grid: no rotation, mirror
    dict(n_views=8, vol_ny=31, vol_nx=31, det_off_v_mm=-2.0),   # odd grid, detector rows off-centre: no symmetry at all
    dict(n_views=8, irregular=True),                   # non-equispaced angles: no rotation, mirror
]


def _symmetry_case(case):
    case = dict(case)
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    irregular = case.pop("irregular", False)
    kw.update(case)
    extra = {}
    if irregular:
        rng = np.random.default_rng(3)
        extra["angles_rad"] = list(np.sort(rng.uniform(0, 2 * np.pi, kw["n_views"])))
    return kw, extra


@pytest.mark.parametrize("C", [1, 2, 4, 8, 9])
@pytest.mark.parametrize("case", SYMMETRY_CASES)
def test_adjoint_every_instance_meets_the_oracle(cbct, oracle_mod, case, C):
    """Every compiled instance of the adjoint: each symmetry class (NR in {4, 2, 1} x NM in {2, 1}) with 1, 2, 4, 8
    and 9 channels, so that the launcher's channel blocks of 8, 4, 2 and 1 (and their remainders: 9 = 8 + 1) are
    all reached on geometries with reduced symmetry.  Whole array against the oracle's plain transpose: rel-L2 <=
    1e-4 (BASELINE.json) and a per-element bound, max error <= 1e-5 of the peak (pins P4 / P5)."""
    kw, extra = _symmetry_case(case)
    rng = np.random.default_rng(100 + C)
    sino = rng.random((C, kw["n_views"], kw["det_nv"], kw["det_nu"]), dtype=np.float32)
    sino[C // 2] -= 0.5          # one signed channel
    r = oracle_mod.bp_adjoint(oracle_mod.Geom(**kw, **extra), sino.astype(np.float64))
    g = run_adj(cbct, kw, sino, **extra)
    for c in range(C):
        assert rel_l2(g[c], r[c]) <= 1e-4, (c, rel_l2(g[c], r[c]))
    assert peak_err(g, r) <= 1e-5, peak_err(g, r)


@pytest.mark.parametrize("C", [3, 4, 9])
@pytest.mark.parametrize("case", [SYMMETRY_CASES[0], SYMMETRY_CASES[3], SYMMETRY_CASES[7], SYMMETRY_CASES[8]])
@pytest.mark.parametrize("step", [0.37, 0.2])
def test_adjoint_fine_step_instances(cbct, oracle_mod, case, C, step):
    """The FINE twins of the adjoint instances (steps below 1/2 voxel walk a longer sample window)."""
    kw, extra = _symmetry_case(case)
    kw["step_vox"] = step
    rng = np.random.default_rng(200 + C)
    sino = rng.random((C, kw["n_views"], kw["det_nv"], kw["det_nu"]), dtype=np.float32)
    r = oracle_mod.bp_adjoint(oracle_mod.Geom(**kw, **extra), sino.astype(np.float64))
    g = run_adj(cbct, kw, sino, **extra)
    assert rel_l2(g, r) <= 1e-4, rel_l2(g, r)
    assert peak_err(g, r) <= 1e-5, peak_err(g, r)


@pytest.mark.parametrize("C", [1, 4, 5])
@pytest.mark.parametrize("case", [dict(n_views=40), dict(n_views=40, irregular=True),
                                  dict(n_views=42, vol_cz_mm=6.0)])
def test_adjoint_view_splits_instances(cbct, oracle_mod, case, C):
    """Small grids split the views of a launch over groups of CTAs (partial outputs + fixed-order reduction): needs
    enough views for more than one group; all channel blocks, three symmetry classes."""
    kw, extra = _symmetry_case(case)
    if "angles_rad" in extra:
        extra["angles_rad"] = list(np.sort(np.random.default_rng(5).uniform(0, 2 * np.pi, kw["n_views"])))
    rng = np.random.default_rng(300 + C)
    sino = rng.random((C, kw["n_views"], kw["det_nv"], kw["det_nu"]), dtype=np.float32)
    r = oracle_mod.bp_adjoint(oracle_mod.Geom(**kw, **extra), sino.astype(np.float64))
    g = run_adj(cbct, kw, sino, **extra)
    assert rel_l2(g, r) <= 1e-4, rel_l2(g, r)
    assert peak_err(g, r) <= 1e-5, peak_err(g, r)


_HALFFAN_128 = dict(det_nu=128, det_nv=128, det_du_mm=3.2, det_dv_mm=3.2, det_off_u_mm=115.0)   # PAPER.md:61 panel, binned


@pytest.mark.parametrize("over,C", [
    (dict(_HALFFAN_128, vol_nx=256, vol_ny=256, vol_nz=256, vox_mm=2.0, n_views=64), 1),                  # NR 4, NM 2
    (dict(_HALFFAN_128, vol_nx=256, vol_ny=256, vol_nz=256, vox_mm=2.0, n_views=64), 3),                  # ... blocks of 2 + 1
    (dict(_HALFFAN_128, vol_nx=256, vol_ny=256, vol_nz=128, vox_mm=2.0, n_views=66), 2),                  # NR 2, NM 2
    (dict(_HALFFAN_128, vol_nx=160, vol_ny=160, vol_nz=161, vox_mm=3.0, n_views=64, irregular=True), 1),  # NR 1, NM 2, odd nz
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=130, vol_cz_mm=6.0, vol_cx_mm=-4.0), 2),  # none
    (dict(_HALFFAN_128, vol_nx=160, vol_ny=160, vol_nz=160, vox_mm=3.0, n_views=64, irregular=True), 5),  # NR 1, NM 2: blocks of 4 + 1
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64, vol_cz_mm=6.0, irregular=True), 9),  # none: 8 + 1
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64, det_off_v_mm=4.0, irregular=True), 6),  # none: 4 + 2
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64), 1),   # 262 144 base voxels: column kernel
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64), 5),   # ... 4 (voxel kernel, its own view groups) + 1
    (dict(_HALFFAN_128, vol_nx=96, vol_ny=96, vol_nz=96, vox_mm=5.0, n_views=70, irregular=True), 6),   # 442 368: groups of 4 + 2
    (dict(det_nu=48, det_nv=48, det_du_mm=8.0, det_dv_mm=8.0, det_off_u_mm=100.0, vol_nx=256, vol_ny=256, vol_nz=256,
          vox_mm=2.0, n_views=1040), 1),   # more views than one launch chunk: the groups accumulate over the chunks
])
def test_adjoint_column_kernel_with_view_groups(cbct, oracle_mod, over, C):
    """Calls of fewer than 4 channels (and all calls without rotation symmetry) on grids of 200 000 base voxels or more take the column-walk kernel
    (cbct_adjoint_column.cu), and with 64 views or more its CTAs split the views into groups whose partial outputs
    are reduced afterwards.  Whole array against the oracle, every symmetry class, channel blocks of 2 and 1."""
    kw, extra = _symmetry_case(over)
    if "angles_rad" in extra:
        extra["angles_rad"] = list(np.sort(np.random.default_rng(6).uniform(0, 2 * np.pi, kw["n_views"])))
    rng = np.random.default_rng(400 + C)
    sino = rng.random((C, kw["n_views"], kw["det_nv"], kw["det_nu"]), dtype=np.float32)
    r = oracle_mod.bp_adjoint(oracle_mod.Geom(**kw, **extra), sino.astype(np.float64))
    g = run_adj(cbct, kw, sino, **extra)
    assert np.abs(r).max() > 0
    for c in range(C):
        assert rel_l2(g[c], r[c]) <= 1e-4, (c, rel_l2(g[c], r[c]))
    assert peak_err(g, r) <= 1e-5, peak_err(g, r)
    record("column_view_groups", rel_l2=rel_l2(g, r), peak=peak_err(g, r), C=C, n=g.size)


def test_adjoint_tall_detector_window(cbct, oracle_mod):
    """A tall detector (|v| / sdd up to 0.42, cone half-angle 23 degrees) at step 1/2: the sample window of a
    (voxel, ray) pair is up to 2 sqrt(2) sqrt(1 + v^2/H^2) / step samples long, which passes 6 beyond |v|/H =
    0.354; the launcher must then walk the longer window.  Whole array against the oracle, and the adjoint
    identity <P x, y> = <x, P^T y> in fp32."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(n_views=8, vol_nx=24, vol_ny=24, vol_nz=48, vox_mm=8.0, det_nu=40, det_nv=72, det_du_mm=8.0,
              det_dv_mm=18.0, sid_mm=600.0, sdd_mm=1500.0)
    rng = np.random.default_rng(17)
    sino = rng.random((2, 8, 72, 40), dtype=np.float32)
    vol = rng.random((2, 48, 24, 24), dtype=np.float32)
    og = oracle_mod.Geom(**kw)
    r = oracle_mod.bp_adjoint(og, sino.astype(np.float64))
    g = run_adj(cbct, kw, sino)
    assert np.abs(r[:, 0]).max() > 0 and np.abs(r[:, -1]).max() > 0     # the outer planes are reached
    assert rel_l2(g, r) <= 1e-4, rel_l2(g, r)
    assert peak_err(g, r) <= 1e-5, peak_err(g, r)
    Ax = run_fp(cbct, kw, vol)
    lhs, rhs = float(np.sum(Ax * sino)), float(np.sum(vol.astype(np.float64) * g))
    assert abs(lhs - rhs) / abs(lhs) <= 1e-5


def test_adjoint_identity_fp32(cbct):
    cfg = synth.CONFIGS["small_halffan"]
    kw = synth.geom_kwargs(cfg)
    rng = np.random.default_rng(9)
    x = rng.random((1, 64, 64, 64), dtype=np.float32)
    y = rng.random((1, 90, 128, 128), dtype=np.float32)
    Ax = run_fp(cbct, kw, x)
    Aty = run_adj(cbct, kw, y)
    lhs, rhs = float(np.sum(Ax * y)), float(np.sum(x * Aty))
    assert abs(lhs - rhs) / abs(lhs) <= 1e-5


def test_slab_streaming_matches_resident(cbct, oracle_mod):
    """A5: a work-set cap forces z-slabs; results equal the resident path
    (forward: sum over slabs; adjoint / FDK: slab by slab) and the oracle."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(vol_nz=40, n_views=12, det_off_u_mm=15.0)
    rng = np.random.default_rng(4)
    vol = rng.random((2, 40, 32, 32), dtype=np.float32)
    sino = rng.random((2, 12, 48, 48), dtype=np.float32)
    packed, raw = 48 * 36 * 16 * 2, 32 * 32 * 4 * 2   # bytes per plane, 2 channels (16-B cells at row pitch 40 + 8, raw voxels)
    cap = 2 * (9 * (packed + raw) + 4 * packed) + 16   # two slab buffers of 9 planes (+ 4 border planes)
    g = cbct.Geometry(**kw, max_workset_bytes=cap)
    assert g.num_slabs(2) == 5
    og = oracle_mod.Geom(**kw)
    for host in (False, True):
        def put(a):
            return torch.from_numpy(a.copy()).pin_memory() if host else dev(a)
        out_s = torch.zeros((2,) + g.sino_shape, device="cuda")
        g.fp(put(vol), out_s, 2)
        torch.cuda.synchronize()
        r = oracle_mod.fp(og, vol.astype(np.float64))
        assert rel_l2(out_s.cpu().numpy().astype(np.float64), r) <= 1e-5
        out_v = torch.empty((2,) + g.vol_shape).pin_memory() if host else torch.zeros((2,) + g.vol_shape, device="cuda")
        g.bp_adjoint(dev(sino), out_v, 2)
        torch.cuda.synchronize()
        r = oracle_mod.bp_adjoint(og, sino.astype(np.float64))
        assert rel_l2(out_v.cpu().numpy().astype(np.float64), r) <= 1e-4
        g.bp_fdk(dev(sino), out_v, 2)
        torch.cuda.synchronize()
        r = oracle_mod.bp_fdk(og, sino.astype(np.float64))
        assert rel_l2(out_v.cpu().numpy().astype(np.float64), r) <= 1e-5


def test_host_buffers_numpy(cbct, oracle_mod):
    """Pageable host buffers through the C ABI (the e2e path of bench.py)."""
    cfg = synth.CONFIGS["tiny"]
    kw = synth.geom_kwargs(cfg)
    vol, sino = synth.make_volume(cfg), synth.make_sinogram(cfg)
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    out = np.empty((1,) + g.sino_shape, dtype=np.float32)
    g.fp(vol, out, 1)
    assert rel_l2(out.astype(np.float64), oracle_mod.fp(og, vol.astype(np.float64))) <= 1e-5
    outv = np.empty((1,) + g.vol_shape, dtype=np.float32)
    g.bp_adjoint(sino, outv, 1)
    assert rel_l2(outv.astype(np.float64), oracle_mod.bp_adjoint(og, sino.astype(np.float64))) <= 1e-4
    g.bp_fdk(sino, outv, 1)
    assert rel_l2(outv.astype(np.float64), oracle_mod.bp_fdk(og, sino.astype(np.float64))) <= 1e-5


def test_strided_views_subgeometry(cbct):
    """R14 / PAPER.md:270: a handle with a strided subset of the angles gives the corresponding rows.  Every 3rd of
    36 views keeps the quarter-turn symmetry, so both handles take the same kernel and the rows have the same
    bits; every 4th (9 views) loses it, the other kernel rounds differently: equal to 1e-6 of the scale."""
    cfg = synth.CONFIGS["tiny"]
    kw = dict(synth.geom_kwargs(cfg))
    vol = synth.make_volume(cfg)
    full = run_fp(cbct, kw, vol)
    sub3 = run_fp(cbct, dict(kw, n_views=12), vol, angles_rad=[2 * np.pi * i / 36 for i in range(0, 36, 3)])
    assert np.array_equal(full[:, ::3], sub3)
    sub4 = run_fp(cbct, dict(kw, n_views=9), vol, angles_rad=[2 * np.pi * i / 36 for i in range(0, 36, 4)])
    assert np.max(np.abs(full[:, ::4] - sub4)) <= 1e-6 * np.max(np.abs(full))


def test_degenerate_inputs(cbct):
    """Zero volume / zero sinogram give exact zeros; a detector that misses the
    volume entirely gives an exactly-zero sinogram and adjoint; outputs are overwritten."""
    cfg = synth.CONFIGS["tiny"]
    kw = dict(synth.geom_kwargs(cfg))
    z = run_fp(cbct, kw, np.zeros((1, 32, 32, 32), np.float32))
    assert np.all(z == 0.0)
    assert np.all(run_adj(cbct, kw, np.zeros((1, 36, 48, 48), np.float32)) == 0.0)
    assert np.all(run_fdk(cbct, kw, np.zeros((1, 36, 48, 48), np.float32)) == 0.0)
    far = dict(kw, det_off_u_mm=900.0)
    assert np.all(run_fp(cbct, far, synth.make_volume(cfg)) == 0.0)
    assert np.all(run_adj(cbct, far, synth.make_sinogram(cfg)) == 0.0)
    assert np.all(run_fdk(cbct, far, synth.make_sinogram(cfg)) == 0.0)
    # single view, single-row detector, 1-voxel-thick volume
    thin = dict(kw, n_views=1, det_nv=1, vol_nz=1)
    out = run_fp(cbct, thin, np.ones((1, 1, 32, 32), np.float32))
    assert out.shape == (1, 1, 1, 48) and np.all(np.isfinite(out)) and out.max() > 0


def test_errors_are_loud(cbct):
    with pytest.raises(cbct.CbctError):
        cbct.Geometry(**dict(synth.geom_kwargs(synth.CONFIGS["tiny"]), step_vox=0.0))
    g = cbct.Geometry(**synth.geom_kwargs(synth.CONFIGS["tiny"]))
    with pytest.raises(cbct.CbctError):
        g.fp(torch.zeros(5, device="cuda"), torch.zeros(g.n_sino, device="cuda"))
    with pytest.raises(cbct.CbctError):
        cbct.Geometry(**synth.geom_kwargs(synth.CONFIGS["tiny"]), max_workset_bytes=1000).num_slabs(1)


@pytest.mark.parametrize("name", ["pyramid_64", "pyramid_128", "pyramid_256"])
def test_config3_pyramid_sampled(cbct, oracle_mod, name):
    """Config 3 at full size, in the launch configuration bench.py times:
    2000 sampled rays, 256 sampled adjoint voxels, 2000 sampled FDK voxels, each
    computed one by one by the oracle; plus the fp32 adjoint identity."""
    cfg = synth.CONFIGS[name]
    kw = synth.geom_kwargs(cfg)
    og = oracle_mod.Geom(**kw)
    vol, sino = synth.make_volume(cfg), synth.make_sinogram(cfg)
    Ax = run_fp(cbct, kw, vol)
    ridx = synth.sample_indices(11, Ax[0].size, 2000)
    r = oracle_mod.fp_rays(og, vol.astype(np.float64), ridx)
    gsel = Ax.reshape(1, -1)[:, ridx]
    assert rel_l2(gsel, r) <= 1e-5, rel_l2(gsel, r)
    floor = 1e-3 * float(np.max(np.abs(r)))
    assert np.max(np.abs(gsel - r) / np.maximum(np.abs(r), floor)) <= 1e-4
    Aty = run_adj(cbct, kw, sino)
    vidx = np.union1d(synth.sample_indices(12, vol[0].size, 256), seam_voxels(vol[0].shape, 12))
    r = oracle_mod.bp_adjoint_voxels(og, sino.astype(np.float64), vidx)
    gsel = Aty.reshape(1, -1)[:, vidx]
    record("sampled_adjoint_" + name, rel_l2=rel_l2(gsel, r), peak=peak_err(gsel, r), n=vidx.size)
    assert rel_l2(gsel, r) <= 1e-4
    assert peak_err(gsel, r) <= 1e-5, peak_err(gsel, r)
    lhs, rhs = float(np.sum(Ax * sino)), float(np.sum(vol.astype(np.float64) * Aty))
    assert abs(lhs - rhs) / abs(lhs) <= 1e-5, (lhs, rhs)
    F = run_fdk(cbct, kw, sino)
    vidx = np.union1d(synth.sample_indices(13, vol[0].size, 2000), seam_voxels(vol[0].shape, 13))
    r = oracle_mod.bp_fdk_voxels(og, sino.astype(np.float64), vidx)
    gsel = F.reshape(1, -1)[:, vidx]
    assert rel_l2(gsel, r) <= 1e-5, rel_l2(gsel, r)
    floor = 1e-3 * float(np.max(np.abs(r)))
    assert np.max(np.abs(gsel - r) / np.maximum(np.abs(r), floor)) <= 1e-4


def seam_voxels(shape, seed, extras=4):
    """Structured sample of flat voxel indices for the symmetry-sharing backprojectors: the quadrant seams
    (x, y in {0, N/2-1, N/2, N-1}), the z-mirror seam and the grid faces (z in {0, N/2-1, N/2, N-1}), where the
    rotated / mirrored stores of a base voxel meet.  On each such plane: every seam row at the seam columns and
    at `extras` seeded columns, and every seam column at `extras` seeded rows."""
    nz, ny, nx = shape
    rng = np.random.default_rng(seed)
    seam = lambda n: sorted({0, max(n // 2 - 1, 0), n // 2, n - 1})
    out = set()
    for z in seam(nz):
        xs = sorted(set(seam(nx)) | set(int(v) for v in rng.integers(0, nx, extras)))
        ys = [int(v) for v in rng.integers(0, ny, extras)]
        for y in seam(ny):
            out.update((z * ny + y) * nx + x for x in xs)
        for x in seam(nx):
            out.update((z * ny + y) * nx + x for y in ys)
    return np.array(sorted(out), dtype=np.int64)


def record(name, **vals):
    """Measured error figures, printed (pytest -s / -rA) and, when CBCT_PARITY_LOG names a file, appended to it
    as JSON lines (the numbers quoted in DESIGN.md s.3 / s.5 come from such a log of the B200 run)."""
    import json
    import os
    line = json.dumps(dict(test=name, **{k: float(v) for k, v in vals.items()}))
    print(line)
    path = os.environ.get("CBCT_PARITY_LOG")
    if path:
        with open(path, "a") as f:
            f.write(line + "\n")


def _sampled_checks(oracle_mod, og, vol_c, sino_c, Ax_c, Aty_c, F_c, seeds, n_rays=2000, n_adj=48, n_fdk=2000, tag=""):
    """One channel: sampled forward rays, adjoint voxels and FDK voxels against the oracle.  The backprojectors are
    checked on a seeded random sample AND on the structured seam sample (seam_voxels), each with rel-L2 and a
    per-element bound (max error relative to the largest reference value of the sample)."""
    v64, s64 = vol_c[None].astype(np.float64), sino_c[None].astype(np.float64)
    ridx = synth.sample_indices(seeds[0], Ax_c.size, n_rays)
    r = oracle_mod.fp_rays(og, v64, ridx)[0]
    gsel = Ax_c.reshape(-1)[ridx]
    ra = oracle_mod.fp_rays(og, np.abs(v64), ridx)[0]
    floor = 1e-3 * float(np.max(np.abs(r)))
    den = np.maximum(np.maximum(np.abs(r), 0.1 * ra), floor)   # R16 / R16b
    r16 = float(np.max(np.abs(gsel - r) / np.maximum(np.abs(r), floor)))   # plain R16, reported
    r16b = float(np.max(np.abs(gsel - r) / den))
    record("sampled_fp" + tag, rel_l2=rel_l2(gsel, r), max_rel_R16=r16, max_rel_R16b=r16b, peak=peak_err(gsel, r))
    assert rel_l2(gsel, r) <= 1e-5, rel_l2(gsel, r)
    assert r16b <= 1e-4
    vidx = np.union1d(synth.sample_indices(seeds[1], vol_c.size, n_adj), seam_voxels(vol_c.shape, seeds[1]))
    r = oracle_mod.bp_adjoint_voxels(og, s64, vidx)[0]
    gsel = Aty_c.reshape(-1)[vidx]
    record("sampled_adjoint" + tag, rel_l2=rel_l2(gsel, r), peak=peak_err(gsel, r), n=vidx.size)
    assert rel_l2(gsel, r) <= 1e-4
    assert peak_err(gsel, r) <= 1e-5, peak_err(gsel, r)
    vidx = np.union1d(synth.sample_indices(seeds[2], vol_c.size, n_fdk), seam_voxels(vol_c.shape, seeds[2]))
    r = oracle_mod.bp_fdk_voxels(og, s64, vidx)[0]
    gsel = F_c.reshape(-1)[vidx]
    record("sampled_fdk" + tag, rel_l2=rel_l2(gsel, r), max_rel_R16=max_rel(gsel, r), n=vidx.size)
    assert rel_l2(gsel, r) <= 1e-5, rel_l2(gsel, r)
    assert max_rel(gsel, r) <= 1e-4


def test_config4_multichannel_sampled(cbct, oracle_mod):
    """Config 4 as bench.py launches it: 256^3, 8 channels (phantom + 7 signed noise fields), 400 views,
    one call per operator over all channels.  Channels 0, 1 and 7 are checked on sampled outputs."""
    cfg = synth.CONFIGS["multichannel_256"]
    kw = synth.geom_kwargs(cfg)
    og = oracle_mod.Geom(**kw)
    vol, sino = synth.make_volume(cfg), synth.make_sinogram(cfg)
    Ax, Aty, F = run_fp(cbct, kw, vol), run_adj(cbct, kw, sino), run_fdk(cbct, kw, sino)
    for c in (0, 1, 7):
        _sampled_checks(oracle_mod, og, vol[c], sino[c], Ax[c], Aty[c], F[c], (41 + c, 51 + c, 61 + c),
                        n_rays=800, n_adj=64, n_fdk=800, tag="_config4_c%d" % c)
    # fp32 adjoint identity <P x, y> = <x, P^T y> on every channel of the benchmarked 8-channel launches
    # (dot products accumulated in fp64 over the fp32 outputs; BASELINE.json: <= 1e-5)
    for c in range(cfg["channels"]):
        lhs = float(np.sum(Ax[c] * sino[c]))
        rhs = float(np.sum(vol[c].astype(np.float64) * Aty[c]))
        record("identity_config4_c%d" % c, rel=abs(lhs - rhs) / abs(lhs))
        assert abs(lhs - rhs) / abs(lhs) <= 1e-5, (c, lhs, rhs)
    # channel independence at full size: the batch in reversed channel order (every channel in another group of 4
    # and another component of its cells) gives the same bits.  One channel alone is projected through its four
    # quarter-turn images: the first quarter of the views has the same bits, the rest sees the rays in rotated
    # coordinates, which round differently -- on this signed noise channel (cancellation, R16b) up to 1e-5 of the
    # sinogram's scale, the size of either path's own error against the oracle
    rev = run_fp(cbct, kw, vol[::-1])
    assert np.array_equal(rev[::-1], Ax)
    one = run_fp(cbct, kw, vol[3:4])
    assert np.array_equal(one[0][:cfg["n_views"] // 4], Ax[3][:cfg["n_views"] // 4])
    assert np.max(np.abs(one[0] - Ax[3])) <= 1e-5 * np.max(np.abs(Ax[3]))
    ref = oracle_mod.fp_rays(og, vol[3].astype(np.float64), synth.sample_indices(77, Ax[3].size, 2000))[0]
    got = one[0].ravel()[synth.sample_indices(77, Ax[3].size, 2000)]
    assert rel_l2(got, ref) <= 1e-5


@pytest.mark.parametrize("name", ["pyramid_256_jitter", "pyramid_256_v402"])
def test_scanner_angle_lists_single_channel_sampled(cbct, oracle_mod, name):
    """The single-channel bench workloads without the quarter-turn symmetry between views (a seeded +-0.2 degree
    jitter on 400 angles: z-mirror only; 402 equispaced views: two-fold rotation + z-mirror), at full size and in
    the launch configuration bench.py times: mirror-paired forward cells, column-walk adjoint with view groups, FDK
    quad / pair records.  Sampled rays and voxels (random + seams) one by one against the oracle, and the fp32
    adjoint identity."""
    cfg = synth.CONFIGS[name]
    kw = synth.geom_kwargs(cfg)
    og = oracle_mod.Geom(**kw)
    vol, sino = synth.make_volume(cfg), synth.make_sinogram(cfg)
    Ax, Aty, F = run_fp(cbct, kw, vol), run_adj(cbct, kw, sino), run_fdk(cbct, kw, sino)
    _sampled_checks(oracle_mod, og, vol[0], sino[0], Ax[0], Aty[0], F[0], (101, 102, 103),
                    n_rays=1500, n_adj=128, n_fdk=1500, tag="_" + name)
    lhs, rhs = float(np.sum(Ax * sino)), float(np.sum(vol.astype(np.float64) * Aty))
    record("identity_" + name, rel=abs(lhs - rhs) / abs(lhs))
    assert abs(lhs - rhs) / abs(lhs) <= 1e-5, (lhs, rhs)


@pytest.mark.parametrize("name", ["multichannel_256_jitter", "multichannel_256_v402"])
def test_scanner_angle_lists_multichannel_sampled(cbct, oracle_mod, name):
    """The 8-channel bench workloads without the quarter-turn symmetry, as bench.py launches them (jittered angles:
    column-walk adjoint on channel-interleaved groups of 4, two FDK channels per thread; 402 views: 8-channel voxel
    kernel): channels 0 (phantom), 2 and 7 (signed noise) on sampled outputs, the adjoint identity on every channel."""
    cfg = synth.CONFIGS[name]
    kw = synth.geom_kwargs(cfg)
    og = oracle_mod.Geom(**kw)
    vol, sino = synth.make_volume(cfg), synth.make_sinogram(cfg)
    Ax, Aty, F = run_fp(cbct, kw, vol), run_adj(cbct, kw, sino), run_fdk(cbct, kw, sino)
    for c in (0, 2, 7):
        _sampled_checks(oracle_mod, og, vol[c], sino[c], Ax[c], Aty[c], F[c], (111 + c, 121 + c, 131 + c),
                        n_rays=600, n_adj=48, n_fdk=600, tag="_%s_c%d" % (name, c))
    for c in range(cfg["channels"]):
        lhs = float(np.sum(Ax[c] * sino[c]))
        rhs = float(np.sum(vol[c].astype(np.float64) * Aty[c]))
        record("identity_%s_c%d" % (name, c), rel=abs(lhs - rhs) / abs(lhs))
        assert abs(lhs - rhs) / abs(lhs) <= 1e-5, (c, lhs, rhs)


def test_config5_large_streamed_sampled(cbct, oracle_mod):
    """Config 5: 512^3 at 1 mm, 4 channels, 720 views, 512^2 offset detector, volume in pinned HOST memory
    under a 1 GiB work-set cap (forces the z-slab streaming path, A5).  Channel 0 (phantom) and channel 1
    (noise) are checked on sampled outputs; the fp32 adjoint identity is checked on channel 0."""
    cfg = synth.CONFIGS["large_512"]
    kw = synth.geom_kwargs(cfg)
    C = cfg["channels"]
    g = cbct.Geometry(**kw, max_workset_bytes=1 << 30)
    assert g.num_slabs(C) > 8
    og = oracle_mod.Geom(**kw)
    vol = torch.from_numpy(synth.make_volume(cfg)).pin_memory()
    sino = torch.from_numpy(synth.make_sinogram(cfg)).cuda()
    Ax = torch.empty((C,) + g.sino_shape, device="cuda")
    g.fp(vol, Ax, C)
    out = torch.empty((C,) + g.vol_shape).pin_memory()
    g.bp_adjoint(sino, out, C)
    torch.cuda.synchronize()
    Aty = out.numpy().copy()
    g.bp_fdk(sino, out, C)
    torch.cuda.synchronize()
    F = out.numpy()
    Ax_h, sino_h, vol_h = Ax.cpu().numpy(), sino.cpu().numpy(), vol.numpy()
    for c in (0, 1):
        _sampled_checks(oracle_mod, og, vol_h[c], sino_h[c], Ax_h[c], Aty[c], F[c], (71 + c, 81 + c, 91 + c),
                        n_rays=1000, n_adj=48, n_fdk=1000, tag="_config5_c%d" % c)
    lhs = float(np.sum(Ax_h[0].astype(np.float64) * sino_h[0]))
    rhs = float(np.sum(vol_h[0].astype(np.float64) * Aty[0]))
    assert abs(lhs - rhs) / abs(lhs) <= 1e-5, (lhs, rhs)


@pytest.mark.parametrize("n_views", [1040, 1037, 2056])
def test_more_views_than_one_launch_chunk(cbct, oracle_mod, n_views):
    """> 512 views: the kernels take the views in chunks of 512 and accumulate (with 1040 views the
    rotation-shared backprojectors cross two quarter-turn blocks inside a chunk; 1037 has no rotation; with 2056
    the forward projector's quarter-turn path, which walks n/4 = 514 base views, needs two chunks itself)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(n_views=n_views, vol_nx=16, vol_ny=16, vol_nz=12, det_nu=20, det_nv=18, det_du_mm=6.0, det_dv_mm=6.0,
              det_off_u_mm=9.0)
    rng = np.random.default_rng(5)
    vol = rng.random((2, 12, 16, 16), dtype=np.float32)
    sino = rng.random((2, n_views, 18, 20), dtype=np.float32)
    check_all_three(cbct, oracle_mod, kw, vol, sino, "chunks")


def test_outputs_stay_inside_their_buffers(cbct):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are looked for directly:
    every output lives between two guard regions that must come back untouched (ragged sizes, every
    symmetry class of the backprojectors, resident and z-slab paths)."""
    G = 4096
    for over in (dict(), dict(vol_nx=37, vol_ny=29, vol_nz=21, det_nu=50, det_nv=35, n_views=11, vol_cx_mm=5.0),
                 dict(n_views=10, vol_nx=30, vol_nz=27), dict(n_views=7, det_off_v_mm=3.0)):
        kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
        kw.update(over)
        for cap in (0, 2500000):
            g = cbct.Geometry(**kw, max_workset_bytes=cap)
            C = 3
            rng = np.random.default_rng(8)
            vol = dev(rng.random((C,) + g.vol_shape, dtype=np.float32))
            sino = dev(rng.random((C,) + g.sino_shape, dtype=np.float32))
            for fn, src, n_out in ((g.fp, vol, C * g.n_sino), (g.bp_adjoint, sino, C * g.n_vol), (g.bp_fdk, sino, C * g.n_vol)):
                buf = torch.full((n_out + 2 * G,), -7.25, device="cuda", dtype=torch.float32)
                fn(src, buf[G:G + n_out], C)
                torch.cuda.synchronize()
                assert bool((buf[:G] == -7.25).all()) and bool((buf[G + n_out:] == -7.25).all())
                assert bool(torch.isfinite(buf[G:G + n_out]).all())


@pytest.mark.parametrize("name,over", [("tiny", dict()), ("small_halffan", dict(n_views=12)),
                                       ("tiny", dict(det_nu=77, det_nv=5, det_off_u_mm=-31.0, n_views=3))])
def test_next1_fdk_filter_and_weight(cbct, oracle_mod, name, over):
    """NEXT-1: cbct_fdk_filter (redundancy weight, cosine weight, ramp filter, dphi) and
    cbct_redundancy_weight against the oracle, 2 channels, with and without redundancy weighting."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS[name]))
    kw.update(over)
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(17)
    p = rng.random((2,) + g.sino_shape, dtype=np.float32)
    dp = dev(p)
    for red in (True, False):
        out = torch.full_like(dp, float("nan"))
        g.fdk_filter(dp, out, 2, redundancy=red)
        torch.cuda.synchronize()
        r = oracle_mod.fdk_filter(og, p.astype(np.float64), redundancy=red)
        q = out.cpu().numpy().astype(np.float64)
        assert rel_l2(q, r) <= 1e-5, (red, rel_l2(q, r))
        assert float(np.max(np.abs(q - r))) <= 1e-5 * float(np.max(np.abs(r)))   # signed data: peak-normalised
    out = torch.empty_like(dp)
    g.redundancy_weight(dp, out, 2)
    g.redundancy_weight(dp, dp, 2)   # in place
    torch.cuda.synchronize()
    want = p.astype(np.float64) * oracle_mod.redundancy_weight(og)
    assert np.max(np.abs(out.cpu().numpy() - want)) <= 1e-6 and torch.equal(out, dp)
    with pytest.raises(cbct.CbctError):
        g.fdk_filter(dp, dp, 2)      # in place is refused


def test_next1_fdk_w_end_to_end(cbct, oracle_mod):
    """NEXT-1: FDK_w = cbct_bp_fdk(cbct_fdk_filter(p)) of an analytic ball on a displaced detector that
    truncates its projection (the P14 set-up): equal to the oracle pipeline and to the ball's density."""
    from tests import analytic as an
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(n_views=180, det_nu=96, det_nv=48, det_du_mm=2.0, det_dv_mm=2.0, det_off_u_mm=50.0,
              vol_nx=24, vol_ny=24, vol_nz=4)
    ball = [(np.zeros(3), np.full(3, 40.0), np.eye(3), 0.02)]
    proj = an.ellipsoid_sinogram(kw, ball).astype(np.float32)[None]
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    q = torch.empty((1,) + g.sino_shape, device="cuda")
    rec = torch.empty((1,) + g.vol_shape, device="cuda")
    g.fdk_filter(dev(proj), q, 1, redundancy=True)
    g.bp_fdk(q, rec, 1)
    torch.cuda.synchronize()
    rec = rec.cpu().numpy().astype(np.float64)[0]
    ref = oracle_mod.bp_fdk(og, oracle_mod.fdk_filter(og, proj[0].astype(np.float64)))[0]
    assert rel_l2(rec, ref) <= 2e-5, rel_l2(rec, ref)
    ax = (np.arange(24) - 11.5) * 4.0
    r = np.sqrt(ax[None, :] ** 2 + ax[:, None] ** 2)
    mid = 0.5 * (rec[1] + rec[2])
    assert abs(np.mean(mid[r < 30.0]) - 0.02) < 1e-4


@pytest.mark.parametrize("over", [dict(), dict(det_off_u_mm=40.0, det_nu=40, det_nv=30, n_views=50),
                                  dict(vol_nx=37, vol_ny=29, vol_nz=21, vol_cx_mm=5.0, det_off_v_mm=-7.0, n_views=11),
                                  dict(n_views=1040, vol_nx=16, vol_ny=16, vol_nz=6, det_nu=24, det_nv=12, det_off_u_mm=20.0)])
def test_next2_fov(cbct, oracle_mod, over):
    """NEXT-2: the field-of-view tensor V equals the oracle's view counts exactly (integer decision in fp64)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(over)
    g = cbct.Geometry(**kw)
    out = torch.full(g.vol_shape, float("nan"), device="cuda")
    g.fov(out)
    torch.cuda.synchronize()
    want = oracle_mod.fov(oracle_mod.Geom(**kw))
    got = out.cpu().numpy().astype(np.float64)
    assert np.array_equal(np.rint(got * kw["n_views"]), np.rint(want * kw["n_views"]))
    assert np.max(np.abs(got - want)) <= 1e-6


def test_next2_resampling(cbct, oracle_mod):
    """NEXT-2: Downsample (average pooling), Upsample (nearest), ProjDown against the oracle."""
    rng = np.random.default_rng(23)
    z = rng.standard_normal((3, 8, 12, 20)).astype(np.float32)
    for f in (2, 4):
        out = torch.empty((3, 8 // f, 12 // f, 20 // f), device="cuda")
        cbct.downsample(dev(z), out, f)
        want = oracle_mod.downsample(z.astype(np.float64), f)
        assert np.max(np.abs(out.cpu().numpy() - want)) <= 1e-6
        up = torch.empty((3, 8 * f, 12 * f, 20 * f), device="cuda")
        cbct.upsample(dev(z), up, f)
        assert np.array_equal(up.cpu().numpy(), oracle_mod.upsample(z, f).astype(np.float32))
    p = rng.random((2, 9, 8, 12)).astype(np.float32)
    for f in (2, 4):
        out = torch.empty((2, -(-9 // f), 8 // f, 12 // f), device="cuda")
        cbct.proj_down(dev(p), out, f)
        assert np.max(np.abs(out.cpu().numpy() - oracle_mod.proj_down(p.astype(np.float64), f))) <= 1e-6
    with pytest.raises(cbct.CbctError):
        cbct.downsample(dev(z), torch.empty((3, 2, 4, 6), device="cuda"), 3)


def test_next4_water_bone(cbct, oracle_mod):
    """NEXT-4: Eq. 3-4 against the oracle, with the paper's constants and a tau_0 that fp32 holds exactly; ragged
    length, an unaligned view (scalar path) and the empty input.  fp32 arithmetic on O(1) values: 1e-6 absolute."""
    rng = np.random.default_rng(41)
    r = (rng.random(4099) * 2.6 - 0.1).astype(np.float32)
    r[:6] = np.float32([1.2, 1.6, 0.125, 0.0, 1.4, 2.0])
    for lo, tau0 in ((0, 0.0), (0, 0.125), (1, 0.125)):
        src = dev(r)[lo:]
        w, b = torch.full_like(src, float("nan")), torch.full_like(src, float("nan"))
        cbct.water_bone(src, w, b, tau0=tau0)
        ww, wb = oracle_mod.water_bone(r[lo:].astype(np.float64), tau0=tau0)
        assert np.max(np.abs(w.cpu().numpy() - ww)) <= 1e-6 and np.max(np.abs(b.cpu().numpy() - wb)) <= 1e-6
    e = torch.empty(0, device="cuda")
    cbct.water_bone(e, e.clone(), e.clone())
    with pytest.raises(cbct.CbctError):
        cbct.water_bone(dev(r), dev(r), dev(r), tau1=1.7)


@pytest.mark.parametrize("shape", [(7, 12, 20), (3, 5, 7), (70, 16, 24)])
def test_next4_polychromatic_primary(cbct, oracle_mod, shape):
    """NEXT-4: noise-free Eq. 6 on given line integrals.  Exponents reach ~20; their fp32 rounding (coefficient,
    product, sum: ~3 x 2^-24 x 20) and exp2f's 2 ulp bound the relative error by ~5e-6 per term: 1e-5."""
    nq, nv, nu = shape
    rng = np.random.default_rng(43)
    pw = (rng.random(shape) * 420.0).astype(np.float32)
    pb = (rng.random(shape) * 60.0).astype(np.float32)
    en, mu_w, mu_b, i0 = synth.spectrum_tables(nv, nu)
    resp = oracle_mod.detector_response(en)
    out = torch.full(shape, float("nan"), device="cuda")
    cbct.polychromatic_primary(dev(pw), dev(pb), dev(i0), mu_w, mu_b, resp, out)
    want = oracle_mod.polychromatic_primary(pw, pb, i0, mu_w, mu_b, resp)
    assert np.max(np.abs(out.cpu().numpy() - want) / want) <= 1e-5
    one = torch.empty(shape, device="cuda")
    cbct.polychromatic_primary(dev(pw), dev(pb), dev(i0[3:4]), mu_w[3:4], mu_b[3:4], resp[3:4], one)
    beer = resp[3] * i0[3].astype(np.float64) * np.exp(-(mu_w[3] * pw.astype(np.float64) + mu_b[3] * pb.astype(np.float64)))
    assert np.max(np.abs(one.cpu().numpy() - beer) / beer) <= 1e-5
    with pytest.raises(cbct.CbctError):
        cbct.polychromatic_primary(dev(pw), dev(pb), dev(i0), mu_w[:4], mu_b, resp, out)


def test_next4_chain(cbct, oracle_mod):
    """NEXT-4 end to end: CT numbers -> (rho_w, rho_b) -> two-channel cbct_fp -> detector signal, each step in the
    CUDA library, against the same chain in the oracle.  The projector's error (R16: <= 1e-5 of the line integral
    scale, ~130 mm here) enters the exponent times mu <= 0.2 / mm: relative 3e-4 at most, 1e-4 expected."""
    cfg = synth.CONFIGS["tiny"]
    kw = synth.geom_kwargs(cfg)
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    ph = synth.make_volume(cfg, 1)[0]
    rho = np.where(ph > 0, 1.0 + 0.9 * ph / ph.max(), 0.0).astype(np.float32)  # tissue 1..1.9 in air
    d_rho = dev(rho)
    wb = torch.empty((2,) + tuple(rho.shape), device="cuda")
    cbct.water_bone(d_rho, wb[0], wb[1])
    sino = torch.empty((2,) + tuple(g.sino_shape), device="cuda")
    g.fp(wb, sino, channels=2)
    en, mu_w, mu_b, i0 = synth.spectrum_tables(kw["det_nv"], kw["det_nu"])
    resp = oracle_mod.detector_response(en)
    out = torch.empty(g.sino_shape, device="cuda")
    cbct.polychromatic_primary(sino[0], sino[1], dev(i0), mu_w, mu_b, resp, out)
    ow, ob = oracle_mod.water_bone(rho.astype(np.float64))
    assert ob.max() > 0 and ow.max() > 0
    want = oracle_mod.polychromatic_primary(oracle_mod.fp(og, ow)[0], oracle_mod.fp(og, ob)[0], i0, mu_w, mu_b, resp)
    rel = np.abs(out.cpu().numpy() - want) / want
    assert rel.max() <= 3e-4 and np.sqrt(np.mean(rel ** 2)) <= 3e-5


@pytest.mark.parametrize("over,cap", [(dict(), 0), (dict(n_views=10, vol_nx=30, det_off_u_mm=20.0), 0),
                                      (dict(n_views=7, det_off_u_mm=-15.0), 0), (dict(vol_nz=40, n_views=12, det_off_u_mm=15.0), 2500000)])
def test_next3_fused_residual_and_weighted_adjoint(cbct, oracle_mod, over, cap):
    """NEXT-3: cbct_fp_residual = P x - y and cbct_bp_adjoint_weighted = P^T (w y), against the oracle's
    compositions (resident and z-slab paths; rotation-interleaved and plain sinogram layouts)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(over)
    g = cbct.Geometry(**kw, max_workset_bytes=cap)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(31)
    x = rng.random((3,) + g.vol_shape, dtype=np.float32)
    y = rng.random((3,) + g.sino_shape, dtype=np.float32)
    out = torch.full((3,) + g.sino_shape, float("nan"), device="cuda")
    g.fp_residual(dev(x), dev(y), out, 3)
    Ax = oracle_mod.fp(og, x.astype(np.float64))
    res = out.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(res - (Ax - y)) <= 1e-5 * np.linalg.norm(Ax)   # error relative to the size of P x
    vol = torch.full((3,) + g.vol_shape, float("nan"), device="cuda")
    g.bp_adjoint_weighted(dev(y), vol, 3)
    torch.cuda.synchronize()
    want = oracle_mod.bp_adjoint(og, y.astype(np.float64) * oracle_mod.redundancy_weight(og))
    assert rel_l2(vol.cpu().numpy().astype(np.float64), want) <= 1e-4


@pytest.mark.parametrize("over,C", [
    (dict(_HALFFAN_128, vol_nx=96, vol_ny=96, vol_nz=96, vox_mm=5.0, n_views=70, irregular=True), 6),   # groups of 4 (w fused into the channel interleave) + 2 (weighted planar copy)
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64, vol_cz_mm=6.0, irregular=True), 9),  # no symmetry: 8 + 1
    (dict(_HALFFAN_128, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64), 3),   # full symmetry: w fused into the view interleave, column kernel 2 + 1
])
def test_next3_weighted_adjoint_on_the_column_kernel_paths(cbct, oracle_mod, over, C):
    """cbct_bp_adjoint_weighted = P^T (w y) on grids large enough for the column-walk kernel: without rotation
    symmetry w(u) is applied inside the channel-interleaving pass (groups of 4) AND in a weighted planar copy (the
    channels left over), with it inside the view-interleaving pass.  Whole array against the oracle's composition."""
    kw, extra = _symmetry_case(over)
    g = cbct.Geometry(**kw, **extra)
    og = oracle_mod.Geom(**kw, **extra)
    rng = np.random.default_rng(500 + C)
    y = rng.random((C,) + g.sino_shape, dtype=np.float32)
    y[C // 2] -= 0.5
    vol = torch.full((C,) + g.vol_shape, float("nan"), device="cuda")
    g.bp_adjoint_weighted(dev(y), vol, C)
    torch.cuda.synchronize()
    got = vol.cpu().numpy().astype(np.float64)
    want = oracle_mod.bp_adjoint(og, y.astype(np.float64) * oracle_mod.redundancy_weight(og))
    for c in range(C):
        assert rel_l2(got[c], want[c]) <= 1e-4, (c, rel_l2(got[c], want[c]))
    assert peak_err(got, want) <= 1e-5, peak_err(got, want)
    record("weighted_adjoint_column", rel_l2=rel_l2(got, want), peak=peak_err(got, want), C=C)


@pytest.mark.parametrize("step", [0.2, 0.37, 0.75, 1.0])
def test_other_ray_steps(cbct, oracle_mod, step):
    """step_vox other than 1/2 (the gather adjoint's sample window holds 2 sqrt 2 / step lattice points)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(step_vox=step, n_views=12, det_off_u_mm=18.0)
    rng = np.random.default_rng(41)
    vol = rng.random((2, 32, 32, 32), dtype=np.float32)
    sino = rng.random((2, 12, 48, 48), dtype=np.float32)
    check_all_three(cbct, oracle_mod, kw, vol, sino, "step %g" % step)


@pytest.mark.parametrize("pinned", [True, False])
def test_host_buffers_channel_pipeline(cbct, oracle_mod, pinned):
    """HOST buffers, 9 channels: the calls run as a 3-stage pipeline over blocks of channels (H2D copy, device
    implementation, D2H copy; two buffers per side), so 3 or more blocks exercise the buffer hand-over.
    Results must equal the oracle and the same calls on device buffers: bit for bit where both take the same kernels
    (adjoint, FDK); the forward pipeline sends single channels through the quarter-turn kernel where the device call
    takes groups of 4, which rounds differently (1e-6 of the scale, as in test_strided_views_subgeometry)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(n_views=12, det_off_u_mm=15.0)
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(51)
    vol = rng.random((9,) + g.vol_shape, dtype=np.float32)
    sino = rng.random((9,) + g.sino_shape, dtype=np.float32)

    def host(a):
        t = torch.from_numpy(a.copy())
        return t.pin_memory() if pinned else t
    for name, fn, src, shape, ref, tol in (
            ("fp", g.fp, vol, g.sino_shape, oracle_mod.fp(og, vol.astype(np.float64)), 1e-5),
            ("adjoint", g.bp_adjoint, sino, g.vol_shape, oracle_mod.bp_adjoint(og, sino.astype(np.float64)), 1e-4),
            ("fdk", g.bp_fdk, sino, g.vol_shape, oracle_mod.bp_fdk(og, sino.astype(np.float64)), 1e-5)):
        out_h = host(np.full((9,) + shape, np.nan, dtype=np.float32))
        fn(host(src), out_h, 9)
        torch.cuda.synchronize()
        out_d = torch.empty((9,) + shape, device="cuda")
        fn(dev(src), out_d, 9)
        torch.cuda.synchronize()
        assert rel_l2(out_h.numpy().astype(np.float64), ref) <= tol, name
        scale = float(out_d.abs().max())

        def same(a, b):
            if name == "fp":
                return float((a - b).abs().max()) <= 2e-6 * scale
            return torch.equal(a, b)
        assert same(out_h, out_d.cpu()), name
        # mixed: host input, device output
        out_m = torch.empty((9,) + shape, device="cuda")
        fn(host(src), out_m, 9)
        torch.cuda.synchronize()
        assert same(out_m, out_d), name
        assert torch.equal(out_m.cpu(), out_h), name   # the same blocks whatever side the output is on


def test_host_pipeline_block_schedule_full_size(cbct):
    """Config 4 through pinned HOST buffers: the forward pipeline runs 8 single-channel blocks, the adjoint 2 blocks
    of 4 channels, the FDK backprojection 8 single blocks.  Each channel must agree with the device-buffer call
    (checked against the oracle at this size in test_config4_multichannel_sampled): bit for bit where the same kernel
    runs, else (the forward's single channels) to the rounding of two different fp32 summation orders."""
    cfg = synth.CONFIGS["multichannel_256"]
    g = cbct.Geometry(**synth.geom_kwargs(cfg))
    C = 8
    gen = torch.Generator().manual_seed(77)
    vol_h = torch.rand((C,) + g.vol_shape, generator=gen).pin_memory()
    sino_h = torch.rand((C,) + g.sino_shape, generator=gen).pin_memory()
    for name, fn, src, shape, tol in (("fp", g.fp, vol_h, g.sino_shape, 5e-6), ("adjoint", g.bp_adjoint, sino_h, g.vol_shape, 1e-5),
                                      ("fdk", g.bp_fdk, sino_h, g.vol_shape, 0.0)):
        out_h = torch.full((C,) + shape, float("nan")).pin_memory()
        fn(src, out_h, C)
        out_d = torch.full((C,) + shape, float("nan"), device="cuda")
        fn(src.cuda(), out_d, C)
        torch.cuda.synchronize()
        ref = out_d.cpu()
        for c in range(C):
            err = float((out_h[c] - ref[c]).abs().max()) / float(ref[c].abs().max())
            record("host_pipeline_" + name, channel=c, max_err_over_peak=err)
            assert err <= tol, (name, c, err)
        del out_d, ref, out_h


@pytest.mark.parametrize("C,cap,over", [(4, 0, dict()), (7, 0, dict(vol_nx=37, vol_ny=29, vol_nz=21, vol_cx_mm=5.0, det_off_v_mm=-4.0)),
                                        (9, 0, dict(n_views=7)), (6, 2000000, dict(vol_nz=40, n_views=12, det_off_u_mm=15.0))])
def test_fp_channel_groups(cbct, oracle_mod, C, cap, over):
    """Forward projector with 4 or more channels: groups of 4 go through the channel-interleaved layout
    (fp4_kernel), the remainder through the quad-packed one; resident and z-slab paths, with and without the
    fused residual, against the oracle channel by channel."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(over)
    g = cbct.Geometry(**kw, max_workset_bytes=cap)
    if cap:
        assert g.num_slabs(C) > 2
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(61 + C)
    vol = rng.random((C,) + g.vol_shape, dtype=np.float32)
    vol[1] -= 0.5   # one signed channel
    y = rng.random((C,) + g.sino_shape, dtype=np.float32) * 50.0
    ref = oracle_mod.fp(og, vol.astype(np.float64))
    out = torch.full((C,) + g.sino_shape, float("nan"), device="cuda")
    g.fp(dev(vol), out, C)
    got = out.cpu().numpy().astype(np.float64)
    for c in range(C):
        if c != 1:
            assert rel_l2(got[c], ref[c]) <= 1e-5 and max_rel(got[c], ref[c]) <= 1e-4, c
    scale = float(np.max(np.abs(ref[0])))
    assert np.max(np.abs(got[1] - ref[1])) <= 1e-5 * scale
    g.fp_residual(dev(vol), dev(y), out, C)
    got = out.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got - (ref - y))) <= 2e-5 * scale


@pytest.mark.parametrize("over,C", [
    (dict(n_views=7), 1),                                                   # odd view count: no rotation, z-mirror
    (dict(n_views=9, irregular=True, det_off_u_mm=20.0), 3),                # irregular angles, half-fan, 3 channels
    (dict(n_views=8, irregular=True, det_nv=47, vol_nz=27), 2),             # odd detector rows (a row is its own image), odd nz
    (dict(n_views=10, vol_nx=30, det_nu=50), 5),                            # two-fold rotation only: group of 4 + 1
    (dict(n_views=530, irregular=True, vol_nx=16, vol_ny=16, vol_nz=12, det_nu=20, det_nv=18, det_du_mm=6.0,
          det_dv_mm=6.0), 1),                                               # more views than one launch chunk
])
def test_fp_mirror_paired_cells(cbct, oracle_mod, over, C):
    """Channels outside a group of 4 on z-symmetric geometries without the quarter-turn symmetry go through the
    mirror-paired cells (fpm_kernel: a thread walks the ray of a lower detector row together with its mirror image).
    Whole sinogram against the oracle, with and without the fused residual (R3, R4)."""
    kw, extra = _symmetry_case(over)
    if "angles_rad" in extra:
        extra["angles_rad"] = list(np.sort(np.random.default_rng(8).uniform(0, 2 * np.pi, kw["n_views"])))
    g = cbct.Geometry(**kw, **extra)
    assert g.symmetry()[0] != 4 and g.symmetry()[1]
    rng = np.random.default_rng(500 + C)
    vol = rng.random((C,) + g.vol_shape, dtype=np.float32)
    y = rng.random((C,) + g.sino_shape, dtype=np.float32) * 20.0
    ref = oracle_mod.fp(oracle_mod.Geom(**kw, **extra), vol.astype(np.float64))
    out = torch.full((C,) + g.sino_shape, float("nan"), device="cuda")
    g.fp(dev(vol), out, C)
    got = out.cpu().numpy().astype(np.float64)
    assert rel_l2(got, ref) <= 1e-5, rel_l2(got, ref)
    assert max_rel(got, ref) <= 1e-4, max_rel(got, ref)
    g.fp_residual(dev(vol), dev(y), out, C)
    got = out.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got - (ref - y))) <= 2e-5 * float(np.max(np.abs(ref)))


@pytest.mark.parametrize("nz,C", [(21, 1), (40, 5), (7, 2)])
def test_streamed_backprojectors_mirror_pairs(cbct, oracle_mod, nz, C):
    """A5 + z-mirror: with a work-set cap and a HOST volume the adjoint and the FDK backprojector fill each slab of the lower half together
    with its mirror image (same weights); odd nz has a middle plane that is its own image.  Against the oracle
    and, bit for bit, the resident path."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(vol_nz=nz, n_views=12, det_off_u_mm=15.0)
    plane = 32 * 32 * 4 * C
    g = cbct.Geometry(**kw, max_workset_bytes=2 * 6 * plane + 8)   # two staging buffers of 6 planes
    g0 = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(70 + nz)
    sino = rng.random((C,) + g.sino_shape, dtype=np.float32)
    out_h = torch.full((C,) + g.vol_shape, float("nan")).pin_memory()
    g.bp_adjoint(dev(sino), out_h, C)
    out_d = torch.empty((C,) + g.vol_shape, device="cuda")
    g0.bp_adjoint(dev(sino), out_d, C)
    torch.cuda.synchronize()
    ref = oracle_mod.bp_adjoint(og, sino.astype(np.float64))
    assert rel_l2(out_h.numpy().astype(np.float64), ref) <= 1e-4
    # the same terms on both paths, summed in another order (plane chunks start at the slab's first plane; the
    # resident call may share weights over more channels): equal to fp32 rounding of the sums
    assert rel_l2(out_h.numpy().astype(np.float64), out_d.cpu().numpy().astype(np.float64)) <= 1e-6
    out_h.fill_(float("nan"))
    g.bp_fdk(dev(sino), out_h, C)
    g0.bp_fdk(dev(sino), out_d, C)
    torch.cuda.synchronize()
    assert rel_l2(out_h.numpy().astype(np.float64), oracle_mod.bp_fdk(og, sino.astype(np.float64))) <= 1e-5
    assert np.array_equal(out_h.numpy(), out_d.cpu().numpy())


@pytest.mark.parametrize("C,nz", [(1, 128), (3, 129)])
def test_adjoint_two_planes_per_thread(cbct, oracle_mod, C, nz):
    """Grids of 2^23 voxels or more with fewer than 4 channels take the adjoint variant in which a thread owns two
    consecutive planes (shared horizontal weights).  256 x 256 x nz voxels of 0.5 mm under the tiny detector: the
    whole volume against the oracle (odd nz: the last thread of a column owns one plane and the middle plane is
    its own mirror image)."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(vol_nx=256, vol_ny=256, vol_nz=nz, vox_mm=0.5, n_views=8)
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(90 + C)
    sino = rng.random((C,) + g.sino_shape, dtype=np.float32)
    got = run_adj(cbct, kw, sino)
    ref = oracle_mod.bp_adjoint(og, sino.astype(np.float64))
    assert np.abs(ref).max() > 0
    assert rel_l2(got, ref) <= 1e-4
    # the same sinogram as 4 equal channels takes the one-plane-per-thread kernel: the two variants evaluate the
    # same weights (this geometry is 3072 voxels deep, where the fp32 weights themselves are good to 5e-5)
    four = run_adj(cbct, kw, np.repeat(sino[:1], 4, axis=0))
    assert np.max(np.abs(got[0] - four[0])) <= 2e-6 * np.max(np.abs(ref))
