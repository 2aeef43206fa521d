"""cbct_bp_fdk_static (include/cbct.h): the FDK backprojection with its scratch in the library's static device
array instead of a cudaMalloc'ed workspace.  Its output is compared with cbct_bp_fdk's (the existing path, itself
checked against the oracle in test_gpu_parity.py) on two calls in a row that share the array, within the FDK
tolerance of the other GPU tests (rel-L2 <= 1e-5, max-rel <= 1e-4) -- and, the kernels and launch parameters being
the same, bit for bit.  Collected last on purpose (pytest -x)."""
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
    floor = 1e-3 * float(np.max(np.abs(r)))
    return float(np.max(np.abs(g - r) / np.maximum(np.abs(r), floor)))


def _sino(cfg, channels, seed):
    rng = np.random.default_rng(seed)
    base = synth.make_sinogram(cfg)
    return np.stack([base[0] * (1.0 + 0.25 * c) + 0.1 * rng.standard_normal(base[0].shape).astype(np.float32)
                     for c in range(channels)]).astype(np.float32)


_STATIC_CALLS_BEFORE = 0

# two calls in a row on the one static array: different symmetry classes (records of 16 B / 8 B / 16 B quads),
# different sizes (the second call of each pair is SMALLER or LARGER than what the first left behind)
CASES = [
    ("tiny", 1, {}, "small_halffan", 2, {}),
    ("small_halffan", 1, {}, "tiny", 3, {}),
    ("tiny", 2, {"angle_jitter_deg": 0.3}, "tiny", 2, {}),
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"{c[0]}x{c[1]}-then-{c[3]}x{c[4]}")
def test_static_scratch_matches_existing_path_twice(cbct, case):
    name_a, ch_a, over_a, name_b, ch_b, over_b = case
    calls = []
    for name, ch, over, seed in ((name_a, ch_a, over_a, 11), (name_b, ch_b, over_b, 12)):
        cfg = dict(synth.CONFIGS[name], **over)
        g = cbct.Geometry(**synth.geom_kwargs(cfg))
        sino = torch.from_numpy(_sino(cfg, ch, seed)).cuda()
        ref = torch.full((ch,) + g.vol_shape, float("nan"), device="cuda")
        g.bp_fdk(sino, ref, ch)                      # existing path (allocates its workspace)
        calls.append((g, sino, ch, ref))
    torch.cuda.synchronize()
    outs = [torch.full_like(ref, float("nan")) for (_, _, _, ref) in calls]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (g, sino, ch, _), out in zip(calls, outs):   # back to back on one stream, no synchronisation between them
        g.bp_fdk_static(sino, out, ch)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    for i, ((g, sino, ch, ref), out) in enumerate(zip(calls, outs)):
        a, r = out.cpu().numpy().astype(np.float64), ref.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all(), i
        assert rel_l2(a, r) <= 1e-5, (i, rel_l2(a, r))
        assert max_rel(a, r) <= 1e-4, (i, max_rel(a, r))
        assert torch.equal(out, ref), (i, "same kernels, same launch parameters: expected the same bits")
    global _STATIC_CALLS_BEFORE
    if _STATIC_CALLS_BEFORE:   # (the first use in a process may load the module that holds the array)
        assert free1 >= free0, ("device memory shrank across the static-scratch calls", free0, free1)
    _STATIC_CALLS_BEFORE += 2


def test_static_scratch_rejects_oversize(cbct):
    cfg = synth.CONFIGS["pyramid_64"]               # 400 views of 256 x 256: 108 MB of padded records
    g = cbct.Geometry(**synth.geom_kwargs(cfg))
    sino = torch.zeros((1,) + g.sino_shape, device="cuda")
    vol = torch.full((1,) + g.vol_shape, 7.0, device="cuda")
    with pytest.raises(cbct.CbctError, match=r"UNSUPPORTED.*static array holds %d" % cbct.STATIC_SCRATCH_BYTES):
        g.bp_fdk_static(sino, vol, 1)
    torch.cuda.synchronize()
    assert bool((vol == 7.0).all())                  # nothing was enqueued
    # the largest channel count that fits is accepted, one more is refused
    cfg = synth.CONFIGS["small_halffan"]
    g = cbct.Geometry(**synth.geom_kwargs(cfg))
    per_channel = 45 * 132 * 132 * 2 * 4             # 45 base views, (128 + 4)^2 padded pixels, 8-byte records
    fit = cbct.STATIC_SCRATCH_BYTES // per_channel
    sino = torch.from_numpy(_sino(cfg, fit + 1, 5)).cuda()
    out = torch.empty((fit + 1,) + g.vol_shape, device="cuda")
    ref = torch.empty_like(out)
    g.bp_fdk_static(sino[:fit], out[:fit], fit)
    g.bp_fdk(sino[:fit], ref[:fit], fit)
    torch.cuda.synchronize()
    assert torch.equal(out[:fit], ref[:fit])
    with pytest.raises(cbct.CbctError, match="UNSUPPORTED"):
        g.bp_fdk_static(sino, out, fit + 1)


def test_static_scratch_rejects_host_pointers(cbct):
    cfg = synth.CONFIGS["tiny"]
    g = cbct.Geometry(**synth.geom_kwargs(cfg))
    sino = synth.make_sinogram(cfg)
    vol = torch.empty((1,) + g.vol_shape, device="cuda")
    with pytest.raises(cbct.CbctError, match="INVALID_ARG"):
        g.bp_fdk_static(sino, vol, 1)
