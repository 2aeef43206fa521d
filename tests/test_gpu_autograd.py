"""The autograd wrappers hand gradients to the matched pair: d<P x, y>/dx must be cbct_bp_adjoint(y) bit for bit,
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
