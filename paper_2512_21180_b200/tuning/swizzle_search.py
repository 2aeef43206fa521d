"""Bank-swizzle search for the quad-packed volume of the forward projector (cbct_fp.cu).

Simulates, for the geometry of BASELINE.json configs 3/4 (256^3 at 2 mm, 256^2 offset detector), which packed
cells the 8 lanes of a quarter-warp read at one sample step, and scores a swizzle g(jx, jy, jz) by the cost model
measured with l1_ldg128_patterns.cu on B200 (profiles/r1_l1_microbench.md): one L1 data-stage cycle per
quarter-warp if lanes reading different cells read different 16-byte positions of their 128-byte lines; equal
positions serialise; more than 4 distinct lines cost a second cycle.  Tuning tool: not imported by the library.
Run: python -m paper_2512_21180_b200.tuning.swizzle_search
"""
import numpy as np
# geometry of config 3/4 (voxel units)
sid, sdd = 500.0, 768.0; du = dv = 0.8; nu = nv = 256; u0 = (-0.5*255*1.6+115)/2; v0 = -0.5*255*0.8; n=256; step=0.5
rng = np.random.default_rng(0)
def samples(TU, nq=4000):
    """random quarter-warps: 8 lanes = TU x (8/TU) pixels; returns cells [nq, 8, 3] and slope class"""
    TV = 8 // TU
    out = []; phis = []
    while len(out) < nq:
        phi = rng.uniform(0, 2*np.pi); c, s = np.cos(phi), np.sin(phi)
        iu0 = rng.integers(0, nu - TU); iv0 = rng.integers(0, nv - TV)
        lane = np.arange(8); iu = iu0 + lane % TU; iv = iv0 + lane // TU
        u = u0 + iu*du; v = v0 + iv*dv
        D = np.stack([-sdd*c - u*s, -sdd*s + u*c, v], 1); L = np.linalg.norm(D, axis=1); d = D / L[:, None]
        S = np.array([sid*c, sid*s, 0.0])
        k = rng.integers(500, 1500)
        t = (k + 0.5)*step
        p = S + t*d + (n-1)/2 + 2
        if p.min() < 1 or p.max() > n+2: continue
        out.append(np.floor(p - 0.0).astype(int)); phis.append(phi)
    return np.array(out), np.array(phis)
def cost(cells, g):
    """cells [nq,8,3]; g [nq,8] bank group; cost = max over groups of #distinct cells (+ lines>4 penalty)"""
    tot = 0
    for q in range(cells.shape[0]):
        uniq = {}
        lines = set()
        for l in range(8):
            cx, cy, cz = cells[q, l]
            uniq.setdefault(g[q, l], set()).add((cx, cy, cz))
            lines.add((cx >> 3, cy, cz))
        m = max(len(v) for v in uniq.values())
        tot += max(m, -(-len(lines)//4))
    return tot / cells.shape[0]
def prep(TU, nq=20000):
    cells, phis = samples(TU, nq)
    U = np.zeros((nq, 8, 3), int); M = np.zeros((nq, 8), bool); NL = np.zeros(nq, int)
    for q in range(nq):
        u = sorted({tuple(c) for c in cells[q]})
        U[q, :len(u)] = u; M[q, :len(u)] = True
        NL[q] = len({(c[0] >> 3, c[1], c[2]) for c in u})
    return U, M, NL, phis
def cost_tab(U, M, NL, f):   # f[y&7, z&3]
    g = (U[..., 0] + f[U[..., 1] & 7, U[..., 2] & 3]) & 7
    oh = (g[..., None] == np.arange(8)) & M[..., None]
    mult = oh.sum(1).max(1)
    return np.maximum(mult, -(-NL // 4)).mean()
rng2 = np.random.default_rng(1)
for TU in (4, 8):
    U, M, NL, phis = prep(TU)
    lin = lambda m, n: (m*np.arange(8)[:, None] + n*np.arange(4)[None, :]) & 7
    print('TU', TU, 'current m5n0 %.3f' % cost_tab(U, M, NL, lin(5, 0)), ' m6n4 %.3f' % cost_tab(U, M, NL, lin(6, 4)), ' lower bound (mult=1) %.3f' % np.maximum(1, -(-NL//4)).mean())
    best_overall = None
    for restart in range(6):
        f = rng2.integers(0, 8, (8, 4)) if restart else lin(6, 4).copy()
        best = cost_tab(U, M, NL, f)
        for it in range(1500):
            i, j = rng2.integers(0, 8), rng2.integers(0, 4); old = f[i, j]
            f[i, j] = rng2.integers(0, 8)
            c = cost_tab(U, M, NL, f)
            if c <= best: best = c
            else: f[i, j] = old
        print('  restart', restart, 'best %.4f' % best, f.T.tolist())
        if best_overall is None or best < best_overall[0]: best_overall = (best, f.copy())
