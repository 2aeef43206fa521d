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
