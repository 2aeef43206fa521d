"""How the library sits in a PyTorch program: autograd, CUDA-graph capture, several handles on several streams.

The autograd wrappers hand gradients to the matched pair: d<P x, y>/dx must be cbct_bp_adjoint(y) bit for bit,
d<P^T y, x>/dy must be cbct_fp(x), and a Landweber-type loss 1/2 |P x - y|^2 must have the gradient P^T (P x - y)
the oracle computes (Alg. 1 l.19)."""
import numpy as np
import pytest

from paper_2512_21180_b200 import synth

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def test_gradients_are_the_matched_operators(oracle_mod):
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import autograd, cbct
    cfg = synth.CONFIGS["tiny"]
    kw = synth.geom_kwargs(cfg)
    g = cbct.Geometry(**kw)
    rng = np.random.default_rng(9)
    x_h = rng.random((2, 3) + g.vol_shape, dtype=np.float32)       # batch 2 x 3 channels -> one 6-channel call
    y_h = rng.random((2, 3) + g.sino_shape, dtype=np.float32)
    x = torch.from_numpy(x_h).cuda().requires_grad_(True)
    y = torch.from_numpy(y_h).cuda().requires_grad_(True)

    px = autograd.project(g, x)
    assert px.shape == (2, 3) + g.sino_shape
    (gx,) = torch.autograd.grad((px * y.detach()).sum(), x)
    direct = g.bp_adjoint(y.detach().reshape((6,) + g.sino_shape), torch.empty((6,) + g.vol_shape, device="cuda"), 6)
    assert torch.equal(gx.reshape(direct.shape), direct)

    bty = autograd.backproject(g, y)
    (gy,) = torch.autograd.grad((bty * x.detach()).sum(), y)
    direct = g.fp(x.detach().reshape((6,) + g.vol_shape), torch.empty((6,) + g.sino_shape, device="cuda"), 6)
    assert torch.equal(gy.reshape(direct.shape), direct)

    # Landweber gradient against the oracle, one channel
    og = oracle_mod.Geom(**kw)
    x1 = torch.from_numpy(x_h[0, 0]).cuda().requires_grad_(True)
    loss = 0.5 * ((autograd.project(g, x1) - torch.from_numpy(y_h[0, 0]).cuda()) ** 2).sum()
    loss.backward()
    r = oracle_mod.fp(og, x_h[0, 0].astype(np.float64))[0] - y_h[0, 0]
    ref = oracle_mod.bp_adjoint(og, r)[0]
    got = x1.grad.cpu().numpy().astype(np.float64)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-4

    with pytest.raises(cbct.CbctError):
        autograd.project(g, torch.zeros((4, 4, 4), device="cuda"))


def test_calls_capture_into_a_cuda_graph():
    """After one warm-up call per entry point (workspaces allocated), device-buffer calls only enqueue work on the
    caller's stream, so a chain of them can be captured in a CUDA graph and replayed (launch-bound small scales of
    the multiscale scheme); the replay must reproduce the eager results bit for bit."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct
    g = cbct.Geometry(**synth.geom_kwargs(synth.CONFIGS["tiny"]))
    C = 5
    gen = torch.Generator(device="cuda").manual_seed(3)
    x = torch.rand((C,) + g.vol_shape, device="cuda", generator=gen)
    y = torch.empty((C,) + g.sino_shape, device="cuda")
    q, x2, x3 = torch.empty_like(y), torch.empty_like(x), torch.empty_like(x)

    def chain():
        g.fp(x, y, C)
        g.bp_adjoint(y, x2, C)
        g.fdk_filter(y, q, C)
        g.bp_fdk(q, x3, C)

    chain()
    torch.cuda.synchronize()
    ref = (y.clone(), x2.clone(), x3.clone())
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        chain()
    torch.cuda.current_stream().wait_stream(side)
    for t in (y, x2, x3):
        t.fill_(float("nan"))
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        chain()
    graph.replay()
    torch.cuda.synchronize()
    for a, b in zip(ref, (y, x2, x3)):
        assert torch.equal(a, b)
    x.mul_(2.0)                      # new input values in the same buffers
    graph.replay()
    torch.cuda.synchronize()
    assert torch.allclose(y, 2.0 * ref[0], rtol=1e-6, atol=0.0)


def test_two_handles_on_two_streams():
    """The library keeps no mutable global state: two handles (different geometries) driven concurrently on two
    streams give the results of running them one after the other."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct
    kws = [synth.geom_kwargs(synth.CONFIGS["tiny"]),
           dict(synth.geom_kwargs(synth.CONFIGS["small_halffan"]), n_views=20)]
    gs = [cbct.Geometry(**kw) for kw in kws]
    gen = torch.Generator(device="cuda").manual_seed(5)
    C = 3
    xs = [torch.rand((C,) + g.vol_shape, device="cuda", generator=gen) for g in gs]

    def run(g, x, stream=None):
        y = torch.empty((C,) + g.sino_shape, device="cuda")
        b = torch.empty_like(x)
        f = torch.empty_like(x)
        g.fp(x, y, C, stream=stream)
        g.bp_adjoint(y, b, C, stream=stream)
        g.bp_fdk(y, f, C, stream=stream)
        return y, b, f

    ref = [run(g, x) for g, x in zip(gs, xs)]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [None, None]
    for rep in range(3):
        for i in (0, 1):
            with torch.cuda.stream(streams[i]):
                outs[i] = run(gs[i], xs[i], stream=streams[i])
    torch.cuda.synchronize()
    for r, o in zip(ref, outs):
        for a, b in zip(r, o):
            assert torch.equal(a, b)


def test_workspace_growth_during_capture_is_refused_and_reserve_avoids_it():
    """A captured graph bakes in workspace addresses, so a call that would have to GROW the workspace while its
    stream is capturing must fail loudly (and enqueue nothing) instead of re-allocating; cbct_geom_reserve sizes
    everything up front, after which more channels than any earlier call capture fine and memory stays flat."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]), n_views=6)   # few views: the adjoint needs no partial-sum workspace
    g = cbct.Geometry(**kw)
    gen = torch.Generator(device="cuda").manual_seed(7)
    x = torch.rand((6,) + g.vol_shape, device="cuda", generator=gen)
    y = torch.empty((6,) + g.sino_shape, device="cuda")
    x2 = torch.empty_like(x)
    g.fp(x[:1], y[:1], 1)            # warm-up with ONE channel only
    g.bp_adjoint(y[:1], x2[:1], 1)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with pytest.raises(cbct.CbctError):
        with torch.cuda.graph(graph, stream=side):
            g.fp(x, y, 6)            # needs a larger packed-volume workspace
    torch.cuda.synchronize()
    g.reserve(6)
    before = g.workspace_bytes()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        g.fp(x, y, 6)
        g.bp_adjoint(y, x2, 6)
        g.bp_fdk(y, x2, 6)
    graph.replay()
    torch.cuda.synchronize()
    assert g.workspace_bytes() == before
    ref = torch.empty_like(y)
    g.fp(x, ref, 6)
    torch.cuda.synchronize()
    assert torch.equal(ref, y)


def test_capped_handle_does_not_thrash_its_workspace():
    """Alternating cbct_fp / cbct_bp_adjoint / cbct_bp_fdk on ONE handle under a work-set cap (host volumes,
    z-slab streaming): the workspace is shared by forward slabs, output staging and sinogram copies; it may grow
    during the first round and must stay flat afterwards (no re-allocation per call)."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(vol_nz=40, n_views=12, det_off_u_mm=15.0)
    g = cbct.Geometry(**kw, max_workset_bytes=2500000)
    C = 3
    assert g.num_slabs(C) > 2
    rng = np.random.default_rng(12)
    vol = torch.from_numpy(rng.random((C,) + g.vol_shape, dtype=np.float32)).pin_memory()
    sino = torch.from_numpy(rng.random((C,) + g.sino_shape, dtype=np.float32)).cuda()
    out_s = torch.empty_like(sino)
    out_v = torch.empty_like(vol).pin_memory()
    sizes = []
    for rnd in range(3):
        g.fp(vol, out_s, C)
        g.bp_adjoint(sino, out_v, C)
        g.bp_fdk(sino, out_v, C)
        g.fp(vol[:2].contiguous().pin_memory(), out_s[:2], 2)      # a smaller call in between
        torch.cuda.synchronize()
        sizes.append((g.workspace_bytes(), torch.cuda.memory_allocated()))
    assert sizes[0][0] > 0
    assert sizes[1] == sizes[0] and sizes[2] == sizes[0], sizes


_BINNED_PANEL = dict(det_nu=128, det_nv=128, det_du_mm=3.2, det_dv_mm=3.2, det_off_u_mm=115.0)   # PAPER.md:61, binned


@pytest.mark.parametrize("over", [dict(n_views=12), dict(n_views=12, vol_nz=27), dict(n_views=7, det_off_v_mm=3.0),
                                  dict(n_views=10, vol_nx=30, det_off_u_mm=20.0),
                                  # grids on which the shard of a real call takes the column-walk adjoint kernel
                                  dict(_BINNED_PANEL, vol_nx=128, vol_ny=128, vol_nz=128, vox_mm=4.0, n_views=64),
                                  dict(_BINNED_PANEL, vol_nx=96, vol_ny=96, vol_nz=97, vox_mm=5.0, n_views=70,
                                       angles_rad="seeded")])
def test_plane_range_exports_tile_the_whole_volume_calls(oracle_mod, over):
    """cbct_bp_adjoint_slab / cbct_bp_fdk_slab (the shard of a plane-sharded multi-GPU backprojection): ranges that
    tile [0, nz), plain and as z-mirror pairs, reassemble the whole-volume result (FDK bit for bit; the adjoint to
    fp32 summation order) and equal the oracle."""
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import cbct
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(over)
    if kw.get("angles_rad") == "seeded":
        kw["angles_rad"] = list(np.sort(np.random.default_rng(8).uniform(0, 2 * np.pi, kw["n_views"])))
    g = cbct.Geometry(**kw)
    og = oracle_mod.Geom(**kw)
    C = 3
    nz, ny, nx = g.vol_shape
    rng = np.random.default_rng(33)
    sino_h = rng.random((C,) + g.sino_shape, dtype=np.float32)
    sino = torch.from_numpy(sino_h).cuda()
    mirror_ok = kw.get("det_off_v_mm", 0.0) == 0.0
    for whole, slab, ref, tol in ((g.bp_adjoint, g.bp_adjoint_slab, oracle_mod.bp_adjoint(og, sino_h.astype(np.float64)), 1e-4),
                                  (g.bp_fdk, g.bp_fdk_slab, oracle_mod.bp_fdk(og, sino_h.astype(np.float64)), 1e-5)):
        full = whole(sino, torch.empty((C,) + g.vol_shape, device="cuda"), C)
        # plain ranges of ragged sizes
        got = torch.full_like(full, float("nan"))
        for z0, z1 in ((0, 5), (5, 6), (6, 19), (19, nz)):
            buf = torch.full((C, z1 - z0, ny, nx), float("nan"), device="cuda")
            slab(sino, buf, z0, z1, C)
            got[:, z0:z1] = buf
        torch.cuda.synchronize()
        a, b = got.cpu().numpy().astype(np.float64), full.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(a - ref) / np.linalg.norm(ref) <= tol
        assert np.max(np.abs(a - b)) <= 2e-6 * np.max(np.abs(b))
        if not mirror_ok:
            with pytest.raises(cbct.CbctError):
                slab(sino, torch.empty((C, 4, ny, nx), device="cuda"), 0, 2, C, mirror_pair=True)
            continue
        # mirror pairs: ranges of the lower half, each with its image
        nh = (nz + 1) // 2
        got = torch.full_like(full, float("nan"))
        for z0, z1 in ((0, 3), (3, 10), (10, nh)):
            n = g.slab_planes(z0, z1, True)
            buf = torch.full((C, n, ny, nx), float("nan"), device="cuda")
            slab(sino, buf, z0, z1, C, mirror_pair=True)
            k = z1 - z0
            got[:, z0:z1] = buf[:, :k]
            got[:, nz - z0 - (n - k):nz - z0] = buf[:, k:]
        torch.cuda.synchronize()
        a = got.cpu().numpy().astype(np.float64)
        assert np.isfinite(a).all()
        assert np.linalg.norm(a - ref) / np.linalg.norm(ref) <= tol
        assert np.max(np.abs(a - b)) <= 2e-6 * np.max(np.abs(b))
        with pytest.raises(cbct.CbctError):
            slab(sino, torch.empty((C, 2 * nh, ny, nx), device="cuda"), 1, nh + 1, C, mirror_pair=True)
