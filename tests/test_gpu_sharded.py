"""sharded.py on ONE GPU: the ranks' calls run one after the other (no process waits on another) and their results
are reassembled with the same functions the collectives feed; the result must equal the unsharded calls and the
oracle.  The collectives themselves are covered under gloo in tests/test_dist_cpu.py."""
import numpy as np
import pytest

from paper_2512_21180_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def rel_l2(g, r):
    return float(np.linalg.norm((g - r).ravel()) / np.linalg.norm(r.ravel()))


@pytest.mark.parametrize("over,world,C", [(dict(n_views=24), 2, 1), (dict(n_views=24), 2, 5), (dict(n_views=9), 2, 2),
                                          (dict(n_views=24, vol_nz=27), 3, 1), (dict(n_views=10, det_off_v_mm=3.0), 4, 3),
                                          (dict(n_views=24, irregular=True), 2, 1)])
def test_view_sharded_forward_and_plane_sharded_backprojection(oracle_mod, over, world, C):
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct, sharded
    over = dict(over)
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    irregular = over.pop("irregular", False)
    kw.update(over)
    if irregular:
        kw["angles_rad"] = [float(a) for a in np.sort(np.random.default_rng(3).uniform(0, 2 * np.pi, kw["n_views"]))]
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    rng = np.random.default_rng(44)
    vol_h = rng.random((C,) + g.vol_shape, dtype=np.float32)
    sino_h = rng.random((C,) + g.sino_shape, dtype=np.float32)
    vol, sino = torch.from_numpy(vol_h).cuda(), torch.from_numpy(sino_h).cuda()
    ranks = [sharded.ShardedGeometry(kw, r, world) for r in range(world)]

    # forward: every rank's rows, then the reassembly the all-gather feeds
    blocks = [sg.fp_local(vol, C) for sg in ranks]
    got = sharded.assemble_views(blocks, kw["n_views"])
    ref = g.fp(vol, torch.empty((C,) + g.sino_shape, device="cuda"), C)
    torch.cuda.synchronize()
    a = got.cpu().numpy().astype(np.float64)
    assert rel_l2(a, oracle_mod.fp(og, vol_h.astype(np.float64))) <= 1e-5
    if not irregular and (kw["n_views"] // world) % 4 == 0 and kw["n_views"] % world == 0:
        assert torch.equal(got, ref)          # same kernels, same rays: the same bits
    else:
        assert float((got - ref).abs().max()) <= 2e-6 * float(ref.abs().max())

    # backprojections: every rank's planes, scattered back into the volume
    nz = g.vol_shape[0]
    for local_fn, whole, oref, tol in (("bp_adjoint_local", g.bp_adjoint, oracle_mod.bp_adjoint, 1e-4),
                                       ("bp_fdk_local", g.bp_fdk, oracle_mod.bp_fdk, 1e-5)):
        shards = [getattr(sg, local_fn)(sino, C) for sg in ranks]
        got = sharded.scatter_planes(shards, nz, world, ranks[0].mirror)
        ref = whole(sino, torch.empty((C,) + g.vol_shape, device="cuda"), C)
        torch.cuda.synchronize()
        a = got.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert rel_l2(a, oref(og, sino_h.astype(np.float64))) <= tol
        assert float((got - ref).abs().max()) <= 2e-6 * float(ref.abs().max())   # same terms, other summation order


def test_channel_split_covers_the_batch():
    """Strong split by channels: the ranks' calls together write every channel once, with the bits of one call."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct, sharded
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]), n_views=12)
    g = cbct.Geometry(**kw)
    C, world = 8, 2
    gen = torch.Generator(device="cuda").manual_seed(1)
    vol = torch.rand((C,) + g.vol_shape, device="cuda", generator=gen)
    out = torch.full((C,) + g.sino_shape, float("nan"), device="cuda")
    seen = []
    for r in range(world):
        first, count = sharded.channel_split(g, "fp", vol, out, C, r, world)
        seen += list(range(first, first + count))
    ref = g.fp(vol, torch.empty_like(out), C)
    torch.cuda.synchronize()
    assert seen == list(range(C)) and torch.equal(out, ref)
