"""GPU parity of the multi-scale driver: the operator calls of Algorithm 1
 as `paper_2512_21180_b200.lire_ops` issues them through the C ABI, against the same
sequence written with the fp64 oracle's functions.  The learned blocks are stand-ins on both sides (the same
pointwise formulas, restated here in numpy), so what is compared is the chain of projector / backprojector /
FDK / resampling calls over three scales and its channel bookkeeping.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

N, C = 32, 8
GEO = dict(fov_mm=256.0, panel_mm=240.0, offset_mm=40.0)


def oracle_sequence(o, y_raw, VIEWS):
    """Alg. 1 with the oracle's operators; mirrors lire_ops.LireOperators.reconstruct_operators line by line."""
    from paper_2512_21180_b200.lire_ops import SCALES, LireOperators
    h = C // 2
    G = {f: o.Geom(**LireOperators.geom_kwargs(N, VIEWS, f, **GEO)) for f in SCALES}
    g1 = G[1]
    w1 = o.redundancy_weight(g1)
    V = o.fov(g1)
    y = y_raw
    x = o.bp_fdk(g1, o.fdk_filter(g1, y, redundancy=True))[0]                      # l.3
    bp_full = o.bp_adjoint(g1, y * w1)[0]                                          # l.5
    f0 = SCALES[0]
    xbar, x_bp, ybar = o.downsample(x, f0), o.downsample(bp_full, f0), o.proj_down(y, f0)
    f = np.stack([xbar, x_bp] * (C // 2))                                          # l.8
    hd = np.repeat(ybar[None], C, axis=0)                                          # l.9
    outs = []
    for i, fac in enumerate(SCALES):
        g = G[fac]
        if fac > 1:
            xbar, ybar, yraw_bar, Vbar = (o.downsample(x, fac), o.proj_down(y, fac), o.proj_down(y_raw, fac),
                                          o.downsample(V, fac))
        else:
            xbar, ybar, yraw_bar, Vbar = x, y, y_raw, V
        d1, d2 = hd[:h], hd[h:]
        p1, p2 = f[:h], f[h:]
        p_op = o.fp(g, np.concatenate([p2, xbar[None]]))                           # l.16
        d2 = d2 + 1e-3 * (p_op.mean(0, keepdims=True) + d1.mean(0, keepdims=True) + ybar + yraw_bar)
        b_op = o.bp_adjoint(g, d2 * o.redundancy_weight(g))                        # l.18
        lw = o.bp_adjoint(g, p_op[h] - ybar)[0]                                    # l.19
        p2 = p2 + 1e-3 * (b_op + p1.mean(0, keepdims=True) + xbar + lw + Vbar)
        hd, f = np.concatenate([d1, d2]), np.concatenate([p1, p2])
        upd = f.mean(0)
        if fac > 1:
            upd = o.upsample(upd, fac)
        x = x + 1e-3 * upd
        outs.append(x)
        hd, f = np.roll(hd, 1, axis=0), np.roll(f, 1, axis=0)
        if i < len(SCALES) - 1:
            f, hd = o.upsample(f, 2), o.upsample(hd, 2)[:, :G[SCALES[i + 1]].n_views]
    return outs


@pytest.mark.parametrize("VIEWS", [16, 18, 21])
def test_lire_operator_sequence_matches_oracle(oracle_mod, VIEWS):
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2512_21180_b200 import lire_ops
    rng = np.random.default_rng(2024)
    y_raw = rng.random((VIEWS, N, N), dtype=np.float32)
    ops = lire_ops.LireOperators(N, VIEWS, C, **GEO)
    timings = {}
    got = ops.reconstruct_operators(torch.from_numpy(y_raw).cuda(), timings)
    torch.cuda.synchronize()
    ref = oracle_sequence(oracle_mod, y_raw.astype(np.float64), VIEWS)
    assert len(got) == len(ref) == 3
    for k, (a, r) in enumerate(zip(got, ref)):
        a = a.cpu().numpy().astype(np.float64)
        assert a.shape == r.shape == (N, N, N)
        err = float(np.linalg.norm((a - r).ravel()) / np.linalg.norm(r.ravel()))
        assert err <= 1e-5, (k, err)
    # every group of calls was issued: 3 forward, 3 adjoint groups, both initialisations, resampling
    assert {f"fp_{N // f}" for f in (4, 2, 1)} | {f"adjoint_{N // f}" for f in (4, 2, 1)} | \
           {"init_fdk_w", "init_adjoint", "resample"} == set(timings)


def test_lire_ops_rejects_sizes_without_three_scales():
    from paper_2512_21180_b200 import cbct, lire_ops
    with pytest.raises(cbct.CbctError):
        lire_ops.LireOperators(30, 16)
