// cbct_adjoint.cu -- A3, the matched adjoint P^T ("the Hermitian
// adjoint" of Eq. 5; reading R8: plain transpose of the matrix cbct_fp applies):
//     vol_c[j] = Delta * sum_{i,iv,iu,k} w(j; i,iv,iu,k) sino_c[i,iv,iu],
//     w = prod_axis max(0, 1 - |q_axis(s_i + t_k d) - j_axis|),  t_k = (k + 1/2) Delta.
//
// Design (DESIGN.md s.6; evidence profiles/r1_v0.md).  The v0 kernel scattered
// 8 RED.ADD.F32 per sample and ran at the per-SM global-atomic limit (about one
// lane-RED per clock per SM, 370 ms per channel at 256^3 / 400 views).  v1 is an
// exact GATHER: one thread per voxel enumerates the rays (iu, iv) whose line
// crosses the voxel's tent support and, per ray, the lattice samples inside it:
// the same terms as the scatter, summed in a fixed order, no atomics, no
// zero-fill, plain coalesced stores, deterministic.
//
// Per (voxel, view) in the rotated frame (e1 = source direction, e2 = e_u,
// e3 = z): the point of ray (u, v) at depth fraction lambda = t / L is
// (sid - lambda sdd, lambda u, lambda v).  With lambda_U = U / sdd (the depth of
// the voxel) and mu = lambda - lambda_U the offset sample - voxel is, exactly,
//     e_x = A_x + mu N_x,  e_y = A_y + mu N_y,  e_z = a_v + mu v,
//     a_u = lambda_U (u - u*),  a_v = lambda_U (v - v*),  (A_x, A_y) = a_u (-s, c),
//     (N_x, N_y) = (-(c sdd + s u), -s sdd + c u),
// all SMALL numbers (|e| < 2), so fp32 is enough after an fp64 set-up of
// U, u*, v* per (voxel, view).  Sample k of the ray has mu_k = g (k - kU),
// g = step / L, kU = lambda_U L / step - 1/2.
//
// The weights depend only on geometry, so they are shared by everything that
// sees the same geometry: CB channels; NR voxels related by a rotation of the
// (centred, square) grid about z -- the pair (view i, voxel j) has the weights
// of (view i + r n/NR, voxel j rotated by r 360/NR degrees), so a thread walks
// ALL views for its base voxel j (one quadrant of the grid) and adds
// W(j, i) y[i + r n/NR] into the accumulator of the r-th rotated voxel -- and
// NM = 2 voxels mirrored in z (ray iv <-> nv-1-iv).  One weight evaluation
// then feeds NR * NM * CB accumulators.
#include <atomic>

#include "cbct_device.cuh"
#include "cbct_adjoint.cuh"


// out[c][iq][iv][iu][p] = in[c][iq + p nq][iv][iu], iq < nq = n_views / NR
// (the NR views related by a grid rotation side by side, one vector load)
template <int NR>
__global__ void __launch_bounds__(256)
interleave_views_kernel(const float *__restrict__ in, float *__restrict__ out, int nq, size_t img, int channels,
                        const float *__restrict__ weights, int nu)
{
    const size_t n = (size_t)channels * nq * img;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        size_t pix = e % img, t = e / img;
        size_t iq = t % nq, c = t / nq;
        const float *src = in + (c * NR * nq + iq) * img + pix;
        float vals[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) vals[r] = __ldg(src + (size_t)r * nq * img);
        if (weights) {  // w(u) of P*(w y), fused into the re-layout (NEXT-3)
            const float w = __ldg(weights + pix % nu);
#pragma unroll
            for (int r = 0; r < NR; ++r) vals[r] *= w;
        }
        if (NR == 4) reinterpret_cast<float4 *>(out)[e] = make_float4(vals[0], vals[1], vals[2], vals[NR - 1]);
        else if (NR == 2) reinterpret_cast<float2 *>(out)[e] = make_float2(vals[0], vals[NR - 1]);
        else out[e] = vals[0];
    }
}

// A warp covers 8 (x) x 4 (y) voxels of one plane: compact on the detector, so the lanes walk similar
// (iu, iv) ranges (measured 32.0 -> 29.5 ms per channel against 32 x 1; 4 x 8 and 8 x 2 x 2: 29.8, 29.7).

// ADJ_BZ threads along z per CTA; MINB = CTAs per SM the register allocation aims for (0: the compiler's choice);
// ZT = consecutive planes per thread.  Voxels (x, y, z + t) see the same e_x, e_y on a ray and e_z shifted by
// exactly -t (a_v = lambda_U (v - v*) and v* moves by sdd / U per plane), so the horizontal part of every tap
// weight and all the per-pixel set-up are shared by the ZT voxels, as is the pixel load: the way to fill the
// accumulator budget when the call has too few channels.
#ifndef ADJ_BATCH_LOADS
#define ADJ_BATCH_LOADS (CB >= 4)
#endif
#ifndef ADJ_QW_4X2
#define ADJ_QW_4X2 true
#endif
#ifndef ADJ_DEFER
#define ADJ_DEFER (CB == 4)
#endif
template <int NR, int NM, int CB, bool FINE, int ADJ_BZ, int MINB, int ZT>
__global__ void __launch_bounds__(ADJ_BX *ADJ_BY *ADJ_BZ, MINB)
adjoint_gather_kernel(const float *__restrict__ sinoI, float *__restrict__ vol, const __grid_constant__ AdjGeom G,
                      const __grid_constant__ ViewChunk V, int q0, int accumulate, size_t sino_cstride,
                      size_t vol_cstride, int vol_z_origin)
{
    // Lanes of a warp (8 x 4 voxels of one plane): a quarter-warp -- the unit the L1 data stage serves per cycle for
    // LDG.128 -- covers 4 (x) x 2 (y) voxels, not 8 x 1: its pixels then span at most 1.92 (3 |sin| + |cos|) < 7
    // detector columns, so no two of them share a 16-byte position in different lines (profiles/r1_l1_microbench.md).
    // Simulated data-stage wavefronts per LDG.128 on config 4: 6.1 -> 4.6 (measured before: 6.4).
    int lx = threadIdx.x, ly = threadIdx.y;
    if (ADJ_QW_4X2) {
        const int l = threadIdx.x + ADJ_BX * (threadIdx.y & 3), qw = l >> 3, i = l & 7;
        lx = (i & 3) + 4 * (qw & 1);
        ly = (threadIdx.y & ~3) + (i >> 2) + 2 * (qw >> 1);
    }
    const int ix = blockIdx.x * ADJ_BX + lx;
    const int iy = blockIdx.y * ADJ_BY + ly;
    const int nzb = (G.bz1 - G.bz0 + ADJ_BZ * ZT - 1) / (ADJ_BZ * ZT);
    const int split = blockIdx.z / nzb;
    // plane blocks are launched from the top of the range downwards: with the z-mirror the base planes are the
    // lower half, whose top planes lie in the cone for every view (the heaviest CTAs): started last, they would
    // leave most SMs idle at the end of the launch
    const int iz = G.bz0 + ((nzb - 1 - (blockIdx.z - split * nzb)) * ADJ_BZ + threadIdx.z) * ZT;  // first of the ZT planes
    const bool valid = ix < G.bx && iy < G.by && iz < G.bz1;
    vol += split * G.split_stride;
    const int q_begin = split * G.views_per_split, q_end = min(G.nq, q_begin + G.views_per_split);
    const double X = G.x0 + ix, Y = G.y0 + iy, Z = G.z0 + iz;
    // Sums over views: registers up to 16 per thread, beyond that a private column of shared memory (touched
    // once per view, so its traffic is nothing; it keeps 4 channels x 8 symmetric voxels at the register count
    // of 2 channels).  Flat index ((m CB + c) ZT + t) NR + r.
    constexpr int NACC = NM * CB * ZT * NR;
    constexpr bool SACC = NACC > 16;
    constexpr int NT = ADJ_BX * ADJ_BY * ADJ_BZ;
    __shared__ float sacc[SACC ? NACC : 1][SACC ? NT : 1];
    const int tid = threadIdx.x + ADJ_BX * (threadIdx.y + ADJ_BY * threadIdx.z);
    float acc[SACC ? 1 : NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) {
        if (SACC) sacc[SACC ? i : 0][SACC ? tid : 0] = 0.f;
        else acc[SACC ? 0 : i] = 0.f;
    }
    const float u0f = (float)G.u0, duf = (float)G.du, v0f = (float)G.v0, dvf = (float)G.dv;
    const float sddf = (float)G.sdd, sdd2f = (float)(G.sdd * G.sdd), inv_stepf = (float)G.inv_step;
    const float zcull = 1.4143f * (float)G.inv_sdd;
    const size_t img = (size_t)G.nv * G.nu;

    for (int q = q_begin; q < q_end; ++q) {
        if (!valid) continue;
        // ---- fp64 set-up of the voxel's projection (once per voxel column and view) ----
        const double c = V.cs[q].x, s = V.cs[q].y;
        const double U = G.sid - (X * c + Y * s), w = Y * c - X * s;
        const double rU = 1.0 / U;
        const double ustar = G.sdd * w * rU, vstar = G.sdd * Z * rU;
        const double fu = (ustar - G.u0) * G.inv_du, fv = (vstar - G.v0) * G.inv_dv;
        const double lamU = U * G.inv_sdd;
        // rays whose xy-line can cross the open square |e_x|, |e_y| < 1:
        // |a_u| sdd < |N_x| + |N_y|  (support function of the square), N Lipschitz in u
        const double Bu = (fabs(c * G.sdd + s * ustar) + fabs(c * ustar - s * G.sdd)) / ((U - 1.5) * G.du);
        // rays that can have |e_z| < 1 while inside the square (|mu| sdd <= sqrt 2); plane t projects
        // t / (lambda_U dv) detector rows above plane 0
        const double rows_per_plane = 1.0 / (lamU * G.dv);
        const double Bv = (1.0 + 1.45 * (double)G.tz) * rows_per_plane;
        const int iu_lo = max(0, (int)ceil(fu - Bu)), iu_hi = min(G.nu - 1, (int)floor(fu + Bu));
        const int iv_lo = max(0, (int)ceil(fv - Bv));
        const int iv_hi = min(G.nv - 1, (int)floor(fv + (double)(ZT - 1) * rows_per_plane + Bv));
        if (iu_lo > iu_hi || iv_lo > iv_hi) continue;
        const float cf = (float)c, sf = (float)s, lamUf = (float)lamU;
        const float lu = (float)(lamU * G.du), lv = (float)(lamU * G.dv);
        const float dfu0 = (float)((double)iu_lo - fu), dfv0 = (float)((double)iv_lo - fv);
        // view i = ib + a nbase: component p of the interleaved pixel is view ib + p nbase,
        // and the r-th rotated voxel takes view i + r nbase = component (a + r) mod NR
        const int a = (q0 + q) / G.nbase, ib = (q0 + q) - a * G.nbase;
        const float *sq = sinoI + (size_t)ib * img * NR;
        // this view's sums, by stored component (added into acc, rotated by a, after the view:
        // two-level summation keeps the fp32 error at sqrt(#views) ulp, not sqrt(#terms) ulp)
        float accv[NM * CB * ZT][NR];
#pragma unroll
        for (int i = 0; i < NM * CB * ZT; ++i)
#pragma unroll
            for (int r = 0; r < NR; ++r) accv[i][r] = 0.f;

        // DEFER (instances that batch their loads): the pixels of a ray are requested when its weight is known and
        // consumed only after the NEXT ray's weight arithmetic, which covers their latency (before: 35 % of the stall
        // samples on the first FMAs behind the loads)
        constexpr bool DEFER = ADJ_BATCH_LOADS && ADJ_DEFER && ZT == 1;
        float pya[DEFER ? CB : 1][NR], pyb[DEFER && NM == 2 ? CB : 1][NR], pW = 0.f;
        bool pending = false;
        auto consume = [&]() {
#pragma unroll
            for (int cc = 0; cc < CB; ++cc)
#pragma unroll
                for (int r = 0; r < NR; ++r) {
                    accv[cc][r] = fmaf(pW, pya[DEFER ? cc : 0][r], accv[cc][r]);
                    if (NM == 2) accv[(NM - 1) * CB + cc][r] = fmaf(pW, pyb[DEFER && NM == 2 ? cc : 0][r], accv[(NM - 1) * CB + cc][r]);
                }
        };
        for (int iu = iu_lo; iu <= iu_hi; ++iu) {
            const float u = fmaf((float)iu, duf, u0f);
            const float au = lu * (dfu0 + (float)(iu - iu_lo));
            const float Nx = -fmaf(sf, u, cf * sddf), Ny = fmaf(cf, u, -sf * sddf);
            const float Ax = -sf * au, Ay = cf * au;
            // window of mu from the dominant horizontal axis: |A_d + mu N_d| < 1
            const bool domx = fabsf(Nx) >= fabsf(Ny);
            const float invNd = rcp_approx(domx ? Nx : Ny);
            const float muc = -(domx ? Ax : Ay) * invNd, hw = fabsf(invNd);
            const float lam_lo = lamUf + (muc - hw), lam_hi = lamUf + (muc + hw);
            const float H2 = fmaf(u, u, sdd2f);
            int i0 = (iv_lo * G.nu + iu) * NR, i1 = ((G.nv - 1 - iv_lo) * G.nu + iu) * NR;
            float v = fmaf((float)iv_lo, dvf, v0f), av = lv * dfv0;

            for (int iv = iv_lo; iv <= iv_hi; ++iv, i0 += G.nu * NR, i1 -= G.nu * NR, v += dvf, av += lv) {
                const float L2 = fmaf(v, v, H2);
                float invL = rsqrt_approx(L2);
                invL = fmaf(fmaf(-0.5f * L2 * invL, invL, 0.5f), invL, invL);  // one Newton step
                // inside the square |mu| sdd <= sqrt 2, so |e_z - a_v| = |mu v| <= sqrt 2 |v| / sdd; plane t has
                // a_v - t in place of a_v
                const float zb = fmaf(fabsf(v), zcull, 1.0f);
                const bool zout = ZT == 1 ? fabsf(av) >= zb : (av <= -zb || av >= (float)(ZT - 1) + zb);
                // DEFER: no divergent branch between a ray's loads and their use one ray later (ptxas makes a warp
                // wait for its outstanding loads at such a branch: 21 % of the stall samples sat on this one), so the
                // rows outside the z-window go through the weight arithmetic and are dropped with the zero weights
                if (!(ADJ_BATCH_LOADS && ADJ_DEFER && ZT == 1) && zout) continue;
                const float L = L2 * invL;
                const float invg = L * inv_stepf;  // samples per unit lambda
                const float g = G.step * invL;     // lambda per sample
                // first sample with (k + 1/2) g > lam_lo: k = rn(lam_lo invg); a tie (weight 0) may go either way
                const float klo = (fmaf(lam_lo, invg, CBCT_MAGIC)) - CBCT_MAGIC;
                const float gNx = g * Nx, gNy = g * Ny, gv = g * v;
                const float d0 = klo - fmaf(lamUf, invg, -0.5f);  // k - kU
                float ex = fmaf(d0, gNx, Ax), ey = fmaf(d0, gNy, Ay), ez = fmaf(d0, gv, av);
                float W[ZT];
#pragma unroll
                for (int t = 0; t < ZT; ++t) W[t] = 0.f;
                // the window is 2 sqrt 2 / step samples wide at most: < 6 for step >= 1/2 (5 always evaluated,
                // the 6th only when the window reaches it); samples past the window have weight 0 (clamps)
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    const float wx = __saturatef(1.0f - fabsf(ex));
                    const float wy = __saturatef(1.0f - fabsf(ey));
                    if (ZT == 1) {
                        W[0] = fmaf(wx * wy, __saturatef(1.0f - fabsf(ez)), W[0]);
                    } else {
                        const float wxy = wx * wy;
#pragma unroll
                        for (int t = 0; t < ZT; ++t) W[t] = fmaf(wxy, __saturatef(1.0f - fabsf(ez - (float)t)), W[t]);
                    }
                    if (j == 4 && fmaf(lam_hi, invg, -5.5f) <= klo) break;  // k = klo + 5 is past the window
                    ex += gNx; ey += gNy; ez += gv;
                }
                if (FINE) {  // steps finer than 1/2 voxel: walk the rest of the window
                    const float kend = fmaf(lam_hi, invg, -0.5f);  // samples with k < kend are inside
                    for (float kf = klo + 6.0f; kf < kend; kf += 1.0f) {
                        const float wxy = __saturatef(1.0f - fabsf(ex)) * __saturatef(1.0f - fabsf(ey));
#pragma unroll
                        for (int t = 0; t < ZT; ++t) W[t] = fmaf(wxy, __saturatef(1.0f - fabsf(ez - (float)t)), W[t]);
                        ex += gNx; ey += gNy; ez += gv;
                    }
                }
                bool any = false;
#pragma unroll
                for (int t = 0; t < ZT; ++t) any = any || W[t] != 0.f;
                if (!any || ((ADJ_BATCH_LOADS && ADJ_DEFER && ZT == 1) && zout)) continue;
                // All pixel loads of the ray are issued together, once its weight is known to be non-zero (24 % of the
                // enumerated rays have none), then the 32 FMAs.  Measured on the 32-accumulator instance at 256^3 / 400
                // views, per 4-channel launch: loads placed by the compiler right before their first use 49.5 ms;
                // channel 0's requested before the weight arithmetic and the others pipelined behind it 47.5 ms (ptxas
                // sinks them below the test anyway and keeps the staging registers); this form 45.3 ms.  The 8-channel
                // instances gain as much (402 views, 8 channels: 114.6 -> 101.9 ms); with 1 or 2 channels it changes nothing.
                constexpr bool BATCH = ADJ_BATCH_LOADS;
                if constexpr (DEFER) {
                    if (pending) consume();
#pragma unroll
                    for (int cc = 0; cc < CB; ++cc) {
                        load_views<NR>(sq + cc * sino_cstride + i0, pya[DEFER ? cc : 0]);
                        if (NM == 2) load_views<NR>(sq + cc * sino_cstride + i1, pyb[DEFER && NM == 2 ? cc : 0]);
                    }
                    pW = W[0];
                    pending = true;
                } else if constexpr (BATCH) {
                    float ya[CB][NR], yb[NM == 2 ? CB : 1][NR];
#pragma unroll
                    for (int cc = 0; cc < CB; ++cc) {
                        load_views<NR>(sq + cc * sino_cstride + i0, ya[cc]);
                        if (NM == 2) load_views<NR>(sq + cc * sino_cstride + i1, yb[NM == 2 ? cc : 0]);
                    }
#pragma unroll
                    for (int cc = 0; cc < CB; ++cc)
#pragma unroll
                        for (int t = 0; t < ZT; ++t)
#pragma unroll
                            for (int r = 0; r < NR; ++r) {
                                accv[cc * ZT + t][r] = fmaf(W[t], ya[cc][r], accv[cc * ZT + t][r]);
                                if (NM == 2) accv[(NM - 1) * CB * ZT + cc * ZT + t][r] = fmaf(W[t], yb[NM == 2 ? cc : 0][r], accv[(NM - 1) * CB * ZT + cc * ZT + t][r]);
                            }
                } else {
#pragma unroll
                    for (int cc = 0; cc < CB; ++cc) {
                        float y[NR];
                        load_views<NR>(sq + cc * sino_cstride + i0, y);
#pragma unroll
                        for (int t = 0; t < ZT; ++t)
#pragma unroll
                            for (int r = 0; r < NR; ++r) accv[cc * ZT + t][r] = fmaf(W[t], y[r], accv[cc * ZT + t][r]);
                        if (NM == 2) {
                            load_views<NR>(sq + cc * sino_cstride + i1, y);
#pragma unroll
                            for (int t = 0; t < ZT; ++t)
#pragma unroll
                                for (int r = 0; r < NR; ++r)
                                    accv[(NM - 1) * CB * ZT + cc * ZT + t][r] = fmaf(W[t], y[r], accv[(NM - 1) * CB * ZT + cc * ZT + t][r]);
                        }
                    }
                }
            }
        }
        if (DEFER && pending) consume();
#pragma unroll
        for (int i = 0; i < NM * CB * ZT; ++i) {
            rotate_views<NR>(accv[i], a);
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                if (SACC) sacc[SACC ? i * NR + r : 0][SACC ? tid : 0] += accv[i][r];
                else acc[SACC ? 0 : i * NR + r] += accv[i][r];
            }
        }
    }

    if (!valid) return;
    // ---- stores: rotation r maps (ix, iy) -> r quarter (NR = 4) or half (NR = 2) turns ----
#pragma unroll
    for (int m = 0; m < NM; ++m) {
#pragma unroll
        for (int t = 0; t < ZT; ++t) {
            const int izt = iz + t;
            if (izt >= G.bz1) continue;
            const int z = m == 0 ? izt : G.nz - 1 - izt;
            if (m == 1 && z == izt) continue;  // middle plane of an odd nz is its own mirror image
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                int x = ix, y = iy;
                if (NR == 4) {
                    if (r == 1) { x = G.nx - 1 - iy; y = ix; }
                    if (r == 2) { x = G.nx - 1 - ix; y = G.ny - 1 - iy; }
                    if (r == 3) { x = iy; y = G.ny - 1 - ix; }
                } else if (NR == 2 && r == 1) {
                    x = G.nx - 1 - ix; y = G.ny - 1 - iy;
                }
                const size_t o = ((size_t)(z - (m == 0 ? vol_z_origin : G.mz_origin)) * G.ny + y) * G.nx + x;
#pragma unroll
                for (int cc = 0; cc < CB; ++cc) {
                    const int i = ((m * CB + cc) * ZT + t) * NR + r;
                    float val = (SACC ? sacc[SACC ? i : 0][SACC ? tid : 0] : acc[SACC ? 0 : i]) * G.scale;
                    float *dst = vol + cc * vol_cstride + o;
                    *dst = accumulate ? *dst + val : val;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
int cbct_launch_interleave_views(cbct_geom *g, const float *sino, float *out, int channels, const float *weights,
                                 cudaStream_t st)
{
    const int NR = g->sym_rot;
    const int nq = g->d.n_views / NR;
    const size_t img = (size_t)g->d.det_nv * g->d.det_nu;
    const size_t n = (size_t)channels * nq * img;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    if (NR == 4) interleave_views_kernel<4><<<(unsigned)blocks, 256, 0, st>>>(sino, out, nq, img, channels, weights, g->d.det_nu);
    else if (NR == 2) interleave_views_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(sino, out, nq, img, channels, weights, g->d.det_nu);
    else return CBCT_ERR_INVALID_ARG;
    return cbct_check_launch(g, "interleave_views_kernel");
}

// out[c][e] (+)= sum_s partial[s][c][e], fixed order (deterministic)
__global__ void __launch_bounds__(256)
reduce_splits_kernel(const float *__restrict__ partial, float *__restrict__ out, size_t n, int cb, int nsplit,
                     size_t out_cstride)
{
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n * cb; e += (size_t)gridDim.x * blockDim.x) {
        const size_t c = e / n, v = e - c * n;
        float acc = 0.f;
        for (int s = 0; s < nsplit; ++s) acc += __ldg(partial + ((size_t)s * cb + c) * n + v);
        out[c * out_cstride + v] = acc;
    }
}

int cbct_launch_reduce_splits(cbct_geom *g, const float *partial, float *out, size_t nvox, int cb, int nsplit,
                              size_t out_cstride, cudaStream_t st)
{
    size_t blocks = (nvox * cb + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    reduce_splits_kernel<<<(unsigned)blocks, 256, 0, st>>>(partial, out, nvox, cb, nsplit, out_cstride);
    return cbct_check_launch(g, "reduce_splits_kernel");
}

template <int NR, int NM, int CB, int ADJ_BZ = 1, int MINB = 0, int ZT = 1>
static int launch_gather(cbct_geom *g, AdjGeom &G, const float *sinoI, float *vol, int accumulate_first,
                         size_t sstride, size_t vstride, int vol_z_origin, float *partial, int nsplit, cudaStream_t st)
{
    const int nq_total = g->d.n_views;
    G.nbase = g->d.n_views / NR;
    ViewChunk vc;
    dim3 block(ADJ_BX, ADJ_BY, ADJ_BZ);
    const int nzb = (G.bz1 - G.bz0 + ADJ_BZ * ZT - 1) / (ADJ_BZ * ZT);
    dim3 grid((G.bx + ADJ_BX - 1) / ADJ_BX, (G.by + ADJ_BY - 1) / ADJ_BY, nzb);
    G.nsplit = 1; G.views_per_split = CBCT_VIEWS_PER_LAUNCH; G.split_stride = 0;
    // Kernels that keep their sums in shared memory: ask for exactly the carve-out MINB CTAs need, so that the rest
    // of the 256 KB stays L1 (the driver's default rounds 2 x 33 KB up to 100 KB; the gather lives on its L1 hit
    // rate: 50.5 -> 49.5 ms per 4-channel launch at 256^3 / 400 views).  A preference, set once per instance.
    constexpr int NACC = NM * CB * ZT * NR;
    if constexpr (NACC > 16 && MINB > 0) {
        // the attribute is per device and per function: one bit per device ordinal, set once (thread-safe)
        static std::atomic<uint64_t> carved{0};
        int devid = 0;
        cudaGetDevice(&devid);
        const uint64_t bit = (uint64_t)1 << (devid & 63);
        if (!(carved.fetch_or(bit) & bit)) {
            constexpr size_t per_cta = (size_t)NACC * ADJ_BX * ADJ_BY * ADJ_BZ * sizeof(float) + 1024;
            constexpr int pct = (int)((MINB * per_cta * 100 + 228 * 1024 - 1) / (228 * 1024));
            cudaFuncSetAttribute(adjoint_gather_kernel<NR, NM, CB, false, ADJ_BZ, MINB, ZT>,
                                 cudaFuncAttributePreferredSharedMemoryCarveout, pct);
            cudaFuncSetAttribute(adjoint_gather_kernel<NR, NM, CB, true, ADJ_BZ, MINB, ZT>,
                                 cudaFuncAttributePreferredSharedMemoryCarveout, pct);
        }
    }
    if (partial && nsplit > 1 && nq_total <= CBCT_VIEWS_PER_LAUNCH) {
        // one launch, views split over groups of CTAs into partial outputs of the whole grid, then reduced
        const size_t nvox = (size_t)G.nx * G.ny * G.nz;
        for (int i = 0; i < nq_total; ++i) vc.cs[i] = make_double2(g->cosphi[i], g->sinphi[i]);
        G.nq = nq_total;
        G.nsplit = nsplit;
        G.views_per_split = (nq_total + nsplit - 1) / nsplit;
        G.split_stride = (size_t)CB * nvox;
        grid.z = nzb * nsplit;
        cbct_prof_begin(g, CBCT_KERNEL_ADJOINT, st);
        if (G.fine) adjoint_gather_kernel<NR, NM, CB, true, ADJ_BZ, MINB, ZT><<<grid, block, 0, st>>>(sinoI, partial, G, vc, 0, 0, sstride, nvox, 0);
        else adjoint_gather_kernel<NR, NM, CB, false, ADJ_BZ, MINB, ZT><<<grid, block, 0, st>>>(sinoI, partial, G, vc, 0, 0, sstride, nvox, 0);
        cbct_prof_end(g, CBCT_KERNEL_ADJOINT, st);
        int rc = cbct_check_launch(g, "adjoint_gather_kernel");
        if (rc) return rc;
        return cbct_launch_reduce_splits(g, partial, vol, nvox, CB, nsplit, vstride, st);
    }
    for (int q0 = 0; q0 < nq_total; q0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = nq_total - q0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
        G.nq = n;
        cbct_prof_begin(g, CBCT_KERNEL_ADJOINT, st);
        if (G.fine)
            adjoint_gather_kernel<NR, NM, CB, true, ADJ_BZ, MINB, ZT><<<grid, block, 0, st>>>(sinoI, vol, G, vc, q0, accumulate_first || q0 > 0,
                                                                            sstride, vstride, vol_z_origin);
        else
            adjoint_gather_kernel<NR, NM, CB, false, ADJ_BZ, MINB, ZT><<<grid, block, 0, st>>>(sinoI, vol, G, vc, q0, accumulate_first || q0 > 0,
                                                                             sstride, vstride, vol_z_origin);
        cbct_prof_end(g, CBCT_KERNEL_ADJOINT, st);
        int rc = cbct_check_launch(g, "adjoint_gather_kernel");
        if (rc) return rc;
    }
    return CBCT_OK;
}

static bool adjoint_uses_column(const cbct_geom *g, bool partial_ok);

template <int NR, int NM>
static int launch_gather_channels(cbct_geom *g, AdjGeom &G, const float *sinoI, float *vol, int channels,
                                  size_t sstride, size_t vstride, int vol_z_origin, float *partial, int nsplit,
                                  cudaStream_t st, const float *sino_ci, int ci_groups)
{
    int c = 0;
    // the partial-output workspace is sized for the regime of the grid (cbct_adjoint_partial_floats): 8 channels of
    // the voxel kernel on small grids, 2 channels of the column kernel on large ones
    // (`nsplit` != 1 only says that partial outputs may be used: the group counts are the regimes' own)
    const bool partial_ok = partial != nullptr && nsplit > 1;
    const int nsplit_voxel = partial_ok ? cbct_adjoint_view_splits(g) : 1;
    float *const partial_voxel = nsplit_voxel > 1 ? partial : nullptr;
    const int nsplit_column = partial_ok ? cbct_adjoint_column_splits(g) : 1;
    float *const partial_column = nsplit_column > 1 ? partial : nullptr;
    const bool small = !adjoint_uses_column(g, partial_ok);
    while (c < channels) {
        int left = channels - c, rc;
        const float *s = sinoI + c * sstride;
        float *v = vol + c * vstride;
        // column-walk kernel (cbct_adjoint_column.cu): blocks of 1 or 2 channels on grids large enough to fill the
        // GPU with one thread per column chunk (small grids keep the view-split path of the voxel kernel)
        // (with 4 or more channels the voxel kernel's 32 accumulators per weight win: 12.2 against 13.0 ms per channel)
        // Without rotation symmetry (NR * NM <= 2: irregular angle lists) the column kernel also takes the wide
        // blocks, 8 / (NR * NM) channels per thread: its window then holds the same 8 accumulators per plane as the
        // single-channel instance of a fully symmetric geometry.
        // (measured at 256^3 / 400 views, 8 channels, full symmetry: column kernel on blocks of 2: 98.2 ms, voxel
        // kernel on blocks of 4: 95.3 ms)
        if (!small && (left < 4 || NR * NM <= 2)) {
            int cb = left >= 2 ? 2 : 1;
            if (NR * NM <= 2 && left >= 4) cb = 4;
            if (NR * NM == 1 && left >= 8) cb = 8;
            // NR = 1: the caller may have interleaved the channels in groups of 4 (one LDG.128 per pixel and group
            // instead of 4 scalar loads); groups cover channels [0, 4 ci_groups)
            int ci = 1;
            if (NR == 1 && cb >= 4 && sino_ci && c % 4 == 0 && c + cb <= 4 * ci_groups) { ci = 4; s = sino_ci + c * sstride; }
            rc = cbct_launch_adjoint_column(g, G, NR, NM, cb, ci, s, v, sstride, vstride, vol_z_origin, partial_column, nsplit_column, st);
            if (rc == CBCT_OK) { c += cb; continue; }
            if (rc != 1) return rc;
        }
        // One weight evaluation feeds NR * NM * CB accumulators: 16 in registers; geometries with fewer
        // symmetries (irregular view angles, off-centre grids) make it up with more channels per thread.
        // 32 accumulators per weight evaluation when the channels are there; the sums over views then live in
        // shared memory and the CTA is 8 x 16 x 2 voxels, 2 CTAs = 16 warps per SM (measured at 256^3 / 400 views,
        // 8 channels: 17.5 -> 12.8 ms per channel; with 128-thread CTAs the 20 resident warps drift apart by
        // several views and evict each other's pixels from L1: hit rate 56 %, no gain)
        if constexpr (NR * NM == 8) {
            if (left >= 4) { rc = launch_gather<NR, NM, 4, 2, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 4; if (rc) return rc; continue; }
        }
        if constexpr (NR * NM == 4) {
            if (left >= 8) { rc = launch_gather<NR, NM, 8, 2, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 8; if (rc) return rc; continue; }
        }
        if constexpr (NR * NM <= 2) {
            // 16 accumulators in registers; the 256-thread CTA pays with two symmetric voxels (24.0 -> 22.0 ms
            // per channel with irregular view angles), not with one (31.0 -> 34.6)
            if (NR * NM == 2 && left >= 8) { rc = launch_gather<NR, NM, 8, 2, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 8; if (rc) return rc; continue; }
            if (left >= 8) { rc = launch_gather<NR, NM, 8>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 8; if (rc) return rc; continue; }
        }
        if constexpr (NR * NM <= 4) {
            if (left >= 4) { rc = launch_gather<NR, NM, 4>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 4; if (rc) return rc; continue; }
        }
        // fewer than 4 channels at full symmetry: two planes per thread share the horizontal tap weights, the
        // per-pixel set-up and the pixel loads (256^3 / 400 views: 28.5 -> 26.9 ms at 1 channel, 35.0 -> 31.4 ms at
        // 2); it does not pay on small grids (128^3 and below), where the longer pixel loops cost more
        if constexpr (NR * NM == 8) {
            if ((size_t)G.nx * G.ny * G.nz >= ((size_t)1 << 23)) {
                if (left >= 2) { rc = launch_gather<NR, NM, 2, 1, 0, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 2; }
                else { rc = launch_gather<NR, NM, 1, 1, 0, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 1; }
                if (rc) return rc;
                continue;
            }
        }
        if (left >= 2) { rc = launch_gather<NR, NM, 2>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 2; }
        else { rc = launch_gather<NR, NM, 1>(g, G, s, v, 0, sstride, vstride, vol_z_origin, partial_voxel, nsplit_voxel, st); c += 1; }
        if (rc) return rc;
    }
    return CBCT_OK;
}

// sino_src: the sinogram as the caller laid it out if sym_rot == 1, else the
// view-interleaved copy made by cbct_launch_interleave_views.  Writes planes
// [zs0, zs1) of vol (whose first stored plane is vol_z_origin).  The z-mirror
// is used only when the launch covers the whole grid.
// Number of view groups the adjoint uses for this geometry (1 = no splitting): enough to give the GPU
// about a million threads when one thread per base voxel would not.
static size_t adjoint_base_threads(const cbct_geom *g)
{
    const cbct_geom_desc &d = g->d;
    size_t threads = (size_t)d.vol_nx * d.vol_ny * d.vol_nz / ((size_t)g->sym_rot * (g->sym_mirror_z ? 2 : 1));
    return threads ? threads : 1;
}

// Two regimes of view groups.  VOXEL kernel: grids of fewer than 2 million base voxels do not fill the GPU with one
// thread per base voxel, so the views of a launch are split over up to 32 groups of CTAs.  COLUMN kernel: grids of
// ADJ_COLUMN_GRID base voxels or more give it enough CTAs (tiles x chunks x 8 view groups; measured at 128^3 / 400
// views: 10.0 against 11.7 ms at full symmetry, 33 against 40 ms (1 channel) and 33 against 56 ms (4 channels) with
// jittered angles; at 64^3 the voxel kernel wins, 7.5 against 28 ms); its 8 groups are there to even out the load.
#ifndef ADJ_COLUMN_GRID
#define ADJ_COLUMN_GRID 200000
#endif
bool cbct_adjoint_small_grid(const cbct_geom *g) { return adjoint_base_threads(g) < 2000000; }
static bool column_grid(const cbct_geom *g) { return adjoint_base_threads(g) >= ADJ_COLUMN_GRID; }

int cbct_adjoint_view_splits(const cbct_geom *g)   // voxel kernel
{
    const cbct_geom_desc &d = g->d;
    if (d.n_views > CBCT_VIEWS_PER_LAUNCH || !cbct_adjoint_small_grid(g)) return 1;
    size_t s = (2000000 + adjoint_base_threads(g) - 1) / adjoint_base_threads(g);
    if (s > 32) s = 32;
    if (s > (size_t)d.n_views / 8) s = (size_t)d.n_views / 8;
    return s < 1 ? 1 : (int)s;
}

int cbct_adjoint_column_splits(const cbct_geom *g)   // column kernel
{
    const cbct_geom_desc &d = g->d;
    // not under a work-set cap (the partial outputs are whole volumes) and not for a handful of views
    if (!column_grid(g) || d.max_workset_bytes != 0 || d.n_views < 64) return 1;
    return d.n_views >= 128 ? 8 : 4;   // measured at 256^3 / 400 views, 1 channel: 21.1 (none), 18.6, 16.7, 16.0 ms
}

// Does a launch that may use partial outputs (`partial_ok`: device volume, whole plane range) route its small channel
// blocks (and, without rotation symmetry, all blocks) to the column kernel?  Otherwise the voxel kernel's view groups.
static bool adjoint_uses_column(const cbct_geom *g, bool partial_ok)
{
    return column_grid(g) || !(partial_ok && cbct_adjoint_view_splits(g) > 1);
}

// The column kernel's preconditions (cbct_adjoint_column.cu) from the geometry alone: the 6-sample window and the
// three-plane identity hold on every detector row.
static bool column_kernel_serves(const cbct_geom *g)
{
    const cbct_geom_desc &d = g->d;
    const double v0 = -0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm;
    const double tz = fmax(fabs(v0), fabs(v0 + (d.det_nv - 1) * d.det_dv_mm)) / d.sdd_mm;
    return 2.0 * M_SQRT2 * sqrt(1.0 + tz * tz) / d.step_vox < 6.0 && (float)tz < 0.35f;
}

// Channels of a call that the adjoint wants interleaved in groups of 4 (NR = 1 geometries on grids the column
// kernel serves): 4 * (channels / 4), or 0.
int cbct_adjoint_channel_groups(const cbct_geom *g, int channels, bool device_volume)
{
    if (g->sym_rot != 1 || channels < 4 || !column_kernel_serves(g)) return 0;
    if (!adjoint_uses_column(g, device_volume)) return 0;  // voxel kernel's view groups
    return channels / 4;
}

// out[gq][view][pix][k] = in[4 gq + k][view][pix]: the rotation-interleaving kernel with "views per rotation block"
// = all views and "channels" = groups (weights != nullptr: times w(u), the fused P*(w y))
int cbct_launch_interleave_channels(cbct_geom *g, const float *sino, float *out, int groups, const float *weights,
                                    cudaStream_t st)
{
    const int nq = g->d.n_views;
    const size_t img = (size_t)g->d.det_nv * g->d.det_nu;
    const size_t n = (size_t)groups * nq * img;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    interleave_views_kernel<4><<<(unsigned)blocks, 256, 0, st>>>(sino, out, nq, img, groups, weights, g->d.det_nu);
    return cbct_check_launch(g, "interleave_views_kernel");
}

// floats of workspace the partial outputs of the view groups need (both regimes; 0 = none)
size_t cbct_adjoint_partial_floats(const cbct_geom *g)
{
    const size_t nvol = (size_t)g->d.vol_nx * g->d.vol_ny * g->d.vol_nz;
    const int nv = cbct_adjoint_view_splits(g), nc = cbct_adjoint_column_splits(g);
    size_t vols = 0;
    if (nv > 1) vols = (size_t)nv * 8;           // voxel kernel: up to 8 channels per launch
    if (nc > 1 && vols < 16) vols = 16;          // column kernel: nsplit * CB <= 16
    return vols * nvol;
}

// `partial` (nsplit > 1 only): workspace of nsplit * 8 * nx * ny * nz floats; used when the launch covers the
// whole grid (zs0 = 0, zs1 = nz, vol_z_origin = 0).
// mirror_z_origin != CBCT_NO_MIRROR_PAIR (z-slab streaming of a z-symmetric geometry): planes [zs0, zs1) lie in
// the lower half of the grid and the launch also fills their mirror images [nz - zs1, nz - zs0), stored from
// plane index mirror_z_origin of the same buffer.
int cbct_launch_adjoint(cbct_geom *g, const float *sino_src, float *vol, int channels, int zs0, int zs1,
                        size_t vol_channel_stride, int vol_z_origin, float *partial, int nsplit, cudaStream_t st,
                        int mirror_z_origin, const float *sino_ci, int ci_groups)
{
    const bool pair = mirror_z_origin != CBCT_NO_MIRROR_PAIR;
    if (pair && (!g->sym_mirror_z || zs1 > (g->d.vol_nz + 1) / 2)) return CBCT_ERR_INVALID_ARG;
    if (zs0 != 0 || zs1 != g->d.vol_nz || vol_z_origin != 0) { partial = nullptr; nsplit = 1; }
    const cbct_geom_desc &d = g->d;
    const double h = d.vox_mm;
    AdjGeom G;
    G.sid = d.sid_mm / h; G.sdd = d.sdd_mm / h; G.inv_sdd = 1.0 / G.sdd;
    G.du = d.det_du_mm / h; G.dv = d.det_dv_mm / h; G.inv_du = 1.0 / G.du; G.inv_dv = 1.0 / G.dv;
    G.u0 = (-0.5 * (d.det_nu - 1) * d.det_du_mm + d.det_off_u_mm) / h;
    G.v0 = (-0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm) / h;
    G.x0 = d.vol_cx_mm / h - 0.5 * (d.vol_nx - 1);
    G.y0 = d.vol_cy_mm / h - 0.5 * (d.vol_ny - 1);
    G.z0 = d.vol_cz_mm / h - 0.5 * (d.vol_nz - 1);
    G.step = (float)d.step_vox; G.inv_step = 1.0 / d.step_vox;
    G.scale = (float)(d.step_vox * d.vox_mm);
    double vmax = fmax(fabs(G.v0), fabs(G.v0 + (d.det_nv - 1) * G.dv));
    G.tz = (float)(vmax / G.sdd);
    // Window of a (voxel, ray) pair: |mu| <= 1 / |N_d| <= sqrt 2 / H with H = sqrt(sdd^2 + u^2), at L / step samples per
    // unit mu, i.e. fewer than 2 sqrt 2 (L / H) / step lattice points, L / H = sqrt(1 + v^2 / H^2) <= sqrt(1 + tz^2).
    // The unrolled loop covers 6; anything that can be longer (steps below 1/2 voxel, or a tall detector: at step 1/2
    // from |v| / sdd = 0.354, a cone half-angle of 19.5 degrees) takes the variant that walks the rest of the window.
    G.fine = !(2.0 * M_SQRT2 * sqrt(1.0 + (vmax / G.sdd) * (vmax / G.sdd)) / d.step_vox < 6.0);
    G.nu = d.det_nu; G.nv = d.det_nv; G.nx = d.vol_nx; G.ny = d.vol_ny; G.nz = d.vol_nz;
    const int NR = g->sym_rot;
    const bool mirror = pair || (g->sym_mirror_z && zs0 == 0 && zs1 == d.vol_nz && d.vol_nz > 1);
    G.bx = NR == 4 ? d.vol_nx / 2 : d.vol_nx;
    G.by = NR >= 2 ? d.vol_ny / 2 : d.vol_ny;
    G.bz0 = zs0; G.bz1 = pair ? zs1 : (mirror ? (d.vol_nz + 1) / 2 : zs1);
    G.mz_origin = pair ? mirror_z_origin : vol_z_origin;
    G.nq = 0;
    const size_t sstride = (size_t)d.n_views * d.det_nv * d.det_nu;
    if (NR == 4) {
        return mirror ? launch_gather_channels<4, 2>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups)
                      : launch_gather_channels<4, 1>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups);
    } else if (NR == 2) {
        return mirror ? launch_gather_channels<2, 2>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups)
                      : launch_gather_channels<2, 1>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups);
    }
    return mirror ? launch_gather_channels<1, 2>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups)
                  : launch_gather_channels<1, 1>(g, G, sino_src, vol, channels, sstride, vol_channel_stride, vol_z_origin, partial, nsplit, st, sino_ci, ci_groups);
}
