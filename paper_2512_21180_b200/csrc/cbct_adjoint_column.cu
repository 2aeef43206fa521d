// cbct_adjoint_column.cu -- A3, the matched adjoint P^T (reading R8), "column-walk" gather.
//
// Same sum, same enumeration of (ray, sample) terms as cbct_adjoint.cu (see its header for the exact geometry of the
// gather: offsets e = A + mu N in the view's frame, window of mu from the dominant horizontal axis, clamped tent
// weights), organised so that the HORIZONTAL part of a weight is evaluated once for all the planes a ray touches.
//
// A thread owns ZC consecutive planes of one voxel column (x, y).  Voxels (x, y, z + t) see, on one ray, the same
// horizontal offsets e_x, e_y and a vertical offset shifted by exactly -t, and along the <= 2 sqrt 2 / step samples
// of the ray's window the vertical offset moves by less than 2 zb = 2 sqrt 2 |v| / sdd < 1.  With t0 the plane
// below the window's lowest point, f_k = e_z,k(plane t0) lies in [0, 1 + 2 zb) c [0, 2) for every sample k, so the
// tent weights of the only three planes the ray can touch are, EXACTLY,
//     plane t0     : max(0, 1 - f)     = 1 - f + r
//     plane t0 + 1 : 1 - |f - 1|       = f - 2 r            r = max(0, f - 1)
//     plane t0 + 2 : max(0, f - 1)     = r
// and the three sums over the samples follow from three moments of the horizontal weight w_xy,k:
//     S0 = sum w_xy,  S1 = sum w_xy f,  S2 = sum w_xy r   =>   W(t0) = S0 - S1 + S2, W(t0+1) = S1 - 2 S2, W(t0+2) = S2.
// Per sample that is 2 tents + 1 product + 3 accumulations + 1 clamp, whatever the number of planes; the voxel
// kernel pays 3 tents + 2 products per sample AND per plane.  A thread walks the detector rows of its column from
// the bottom plane to the top one; t0 never decreases along that walk, so the planes form a sliding window of three
// register accumulators (per symmetric image and channel) whose lowest plane is flushed into the thread's private
// column of shared memory when the window moves on.  Rows are shared by the planes they touch: about
// 1 / (lambda_U dv) rows per plane instead of 2 (1 + zb) / (lambda_U dv) per voxel.
// The sums over views stay two-level as in the voxel kernel (per-view window in registers, totals in shared memory).
#include <atomic>

#include "cbct_device.cuh"
#include "cbct_adjoint.cuh"

#ifndef ADJC_BY
#define ADJC_BY ADJ_BY     // voxel columns per CTA in y (x: ADJ_BX = 8)
#endif
#define ADJC_NT (ADJ_BX * ADJC_BY)

// CI = 4 (only with NR = 1): the channels come interleaved in groups of 4 -- record (view, iv, iu) of group gq holds
// the pixel of channels 4 gq .. 4 gq + 3, one LDG.128 (cbct_launch_interleave_channels) -- instead of CB scalar loads
// from CB planar sinograms; `sino_cstride` stays the planar channel stride, a group spans 4 of them.
template <int NR, int NM, int CB, int ZC, int MINB, int CI = 1>
__global__ void __launch_bounds__(ADJC_NT, MINB)
adjoint_column_kernel(const float *__restrict__ sinoI, float *__restrict__ vol, const __grid_constant__ AdjGeom G,
                      const __grid_constant__ ViewChunk V, int q0, int accumulate, size_t sino_cstride,
                      size_t vol_cstride, int vol_z_origin)
{
    constexpr int NA = NM * CB;        // accumulators per plane and rotation: index m * CB + c
    constexpr int NACC = NA * NR;
    extern __shared__ float sacc_flat[];                      // [ZC * NACC][ADJC_NT], dynamic: may pass 48 KB
    float (*sacc)[ADJC_NT] = reinterpret_cast<float (*)[ADJC_NT]>(sacc_flat);
    const int tid = threadIdx.x + ADJ_BX * threadIdx.y;
    const int ix = blockIdx.x * ADJ_BX + threadIdx.x;
    const int iy = blockIdx.y * ADJC_BY + threadIdx.y;
    // blockIdx.z = (chunk counted from the top of the range) * nsplit + split.  Chunks are launched from the top
    // downwards: with the z-mirror the base planes are the lower half, whose top chunks lie in the cone for every
    // view (the heaviest CTAs); started last they would leave most SMs idle at the end of the launch.  For the same
    // reason the views of a launch are split over `nsplit` CTAs per tile (partial outputs, reduced in a fixed
    // order afterwards): a tile's CTA over all views runs for most of the launch, and SMs that drew five heavy
    // ones finish long after the rest (measured: SMs active 77 % of the elapsed cycles without the split).
    const int nch = gridDim.z / G.nsplit;
    const int split = blockIdx.z % G.nsplit;
    const int zc0 = G.bz0 + (nch - 1 - blockIdx.z / G.nsplit) * ZC;   // first plane of this thread's chunk
    vol += split * G.split_stride;
    const int q_begin = split * G.views_per_split, q_end = min(G.nq, q_begin + G.views_per_split);
    const int nzc = min(ZC, G.bz1 - zc0);                  // planes of the chunk inside the launch's range
    const bool valid = ix < G.bx && iy < G.by;
#pragma unroll
    for (int i = 0; i < ZC * NACC; ++i) sacc[i][tid] = 0.f;
    const double X = G.x0 + ix, Y = G.y0 + iy, Z0 = G.z0 + zc0;
    const float u0f = (float)G.u0, duf = (float)G.du, v0f = (float)G.v0, dvf = (float)G.dv;
    const float sddf = (float)G.sdd, sdd2f = (float)(G.sdd * G.sdd), inv_stepf = (float)G.inv_step;
    const float zcull = 1.4143f * (float)G.inv_sdd;
    const size_t img = (size_t)G.nv * G.nu;

    for (int q = q_begin; q < q_end; ++q) {
        if (!valid) continue;
        // ---- fp64 set-up of the column's projection (once per column, chunk and view) ----
        const double c = V.cs[q].x, s = V.cs[q].y;
        const double U = G.sid - (X * c + Y * s), w = Y * c - X * s;
        const double rU = 1.0 / U;
        const double ustar = G.sdd * w * rU;
        const double fu = (ustar - G.u0) * G.inv_du;
        const double lamU = U * G.inv_sdd;
        const double Bu = (fabs(c * G.sdd + s * ustar) + fabs(c * ustar - s * G.sdd)) / ((U - 1.5) * G.du);
        const int iu_lo = max(0, (int)ceil(fu - Bu)), iu_hi = min(G.nu - 1, (int)floor(fu + Bu));
        if (iu_lo > iu_hi) continue;
        const double fv0 = (G.sdd * Z0 * rU - G.v0) * G.inv_dv;    // detector row coordinate of plane zc0
        const double rows_per_plane = 1.0 / (lamU * G.dv);
        const double Bv = (1.0 + 1.45 * (double)G.tz) * rows_per_plane;
        const int iv_lo = max(0, (int)ceil(fv0 - Bv));
        const int iv_hi = min(G.nv - 1, (int)floor(fv0 + (double)(nzc - 1) * rows_per_plane + Bv));
        if (iv_lo > iv_hi) continue;
        const float cf = (float)c, sf = (float)s, lamUf = (float)lamU;
        const float lu = (float)(lamU * G.du), lv = (float)(lamU * G.dv);
        const float dfv0 = (float)((double)iv_lo - fv0);
        // per-ray quantities that are linear in iu: value at iu_lo and increment
        const float u_lo = fmaf((float)iu_lo, duf, u0f);
        const float au_lo = lu * (float)((double)iu_lo - fu);
        const float Nx_lo = -fmaf(sf, u_lo, cf * sddf), Ny_lo = fmaf(cf, u_lo, -sf * sddf);
        const float dNx = -sf * duf, dNy = cf * duf;
        const float Ax_lo = -sf * au_lo, Ay_lo = cf * au_lo, dAx = -sf * lu, dAy = cf * lu;
        const int a = (q0 + q) / G.nbase, ib = (q0 + q) - a * G.nbase;
        const float *sq = sinoI + (size_t)ib * img * (NR * CI);

        // sliding window: R[j] = this view's sums of plane tw + j (relative to zc0), by stored component
        float R[3][NA][NR];
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < NA; ++i)
#pragma unroll
                for (int r = 0; r < NR; ++r) R[j][i][r] = 0.f;
        int tw = 0;
        bool have = false;
        // add the finished plane `t` of the window (component order rotated by a) into the totals
        auto flush = [&](int t, float (&P)[NA][NR]) {
            if (t < 0 || t >= nzc) return;
            float *dst = &sacc[t * NACC][tid];
#pragma unroll
            for (int i = 0; i < NA; ++i) {
                float tmp[NR];
#pragma unroll
                for (int r = 0; r < NR; ++r) tmp[r] = P[i][r];
                rotate_views<NR>(tmp, a);
#pragma unroll
                for (int r = 0; r < NR; ++r) dst[(i * NR + r) * ADJC_NT] += tmp[r];
            }
        };

        // one pass beyond the last row flushes what is left in the window (same code as a window move)
        for (int iv = iv_lo;; ++iv) {
            bool last = iv > iv_hi;
            const float v = fmaf((float)iv, dvf, v0f);
            const float av0 = lv * (dfv0 + (float)(iv - iv_lo));   // e_z of plane zc0 at mu = 0
            const float zb = fabsf(v) * zcull;                      // |mu v| <= zb inside the window
            const float t0f = floorf(av0 - zb);
            int t0 = (int)t0f;
            if (!last && t0 + 2 < 0) continue;  // the row lies below the chunk
            if (t0 >= nzc) last = true;         // ... above it (rows ascend, t0 never decreases)
            if (!have) {
                if (last) break;
                have = true;
                tw = t0;
            }
            if (last) t0 = tw + 3;
            if (t0 > tw) {
                const int nflush = min(t0 - tw, 3);   // after three moves the window is empty
                for (int k = 0; k < nflush; ++k) {
                    flush(tw + k, R[0]);
#pragma unroll
                    for (int i = 0; i < NA; ++i)
#pragma unroll
                        for (int r = 0; r < NR; ++r) { R[0][i][r] = R[1][i][r]; R[1][i][r] = R[2][i][r]; R[2][i][r] = 0.f; }
                }
                tw = t0;
            }
            if (last) break;
            const float fb = av0 - t0f;    // f at mu = 0, in [zb, 1 + zb)
            const float L2row = fmaf(v, v, sdd2f);
            const float *row0 = sq + iv * G.nu * (NR * CI), *row1 = sq + (G.nv - 1 - iv) * G.nu * (NR * CI);
            float u = u_lo, Nx = Nx_lo, Ny = Ny_lo, Ax = Ax_lo, Ay = Ay_lo;

            for (int iu = iu_lo; iu <= iu_hi; ++iu, u += duf, Nx += dNx, Ny += dNy, Ax += dAx, Ay += dAy) {
                // the pixel loads go first: the weight arithmetic below covers their latency
                float y0[CB][NR], y1[NM == 2 ? CB : 1][NR];
                if constexpr (CI == 4) {
#pragma unroll
                    for (int gq = 0; gq < CB / 4; ++gq) {
                        float t[4];
                        load_views<4>(row0 + gq * 4 * sino_cstride + iu * 4, t);
#pragma unroll
                        for (int k = 0; k < 4; ++k) y0[gq * 4 + k][0] = t[k];
                        if (NM == 2) {
                            load_views<4>(row1 + gq * 4 * sino_cstride + iu * 4, t);
#pragma unroll
                            for (int k = 0; k < 4; ++k) y1[NM == 2 ? gq * 4 + k : 0][0] = t[k];
                        }
                    }
                } else {
#pragma unroll
                    for (int cc = 0; cc < CB; ++cc) {
                        load_views<NR>(row0 + cc * sino_cstride + iu * NR, y0[cc]);
                        if (NM == 2) load_views<NR>(row1 + cc * sino_cstride + iu * NR, y1[cc]);
                    }
                }
                // window of mu from the dominant horizontal axis: |A_d + mu N_d| < 1
                const bool domx = fabsf(Nx) >= fabsf(Ny);
                const float invNd = rcp_approx(domx ? Nx : Ny);
                const float muc = -(domx ? Ax : Ay) * invNd, hw = fabsf(invNd);
                const float lam_lo = lamUf + (muc - hw), lam_hi = lamUf + (muc + hw);
                const float L2 = fmaf(u, u, L2row);
                float invL = rsqrt_approx(L2);
                invL = fmaf(fmaf(-0.5f * L2 * invL, invL, 0.5f), invL, invL);  // one Newton step
                const float L = L2 * invL;
                const float invg = L * inv_stepf;  // samples per unit lambda
                const float g = G.step * invL;     // lambda per sample
                // first sample with (k + 1/2) g > lam_lo: k = rn(lam_lo invg); a tie (weight 0) may go either way
                const float klo = (fmaf(lam_lo, invg, CBCT_MAGIC)) - CBCT_MAGIC;
                const float gNx = g * Nx, gNy = g * Ny, gv = g * v;
                const float d0 = klo - fmaf(lamUf, invg, -0.5f);  // k - kU
                float ex = fmaf(d0, gNx, Ax), ey = fmaf(d0, gNy, Ay), f = fmaf(d0, gv, fb);
                float S0 = 0.f, S1 = 0.f, S2 = 0.f;
                // the window holds fewer than 6 lattice points (the launcher checks): 5 always evaluated, the 6th
                // only when the window reaches it; samples past the window have w_xy = 0 (clamps)
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    const float wxy = __saturatef(1.0f - fabsf(ex)) * __saturatef(1.0f - fabsf(ey));
                    S0 += wxy;
                    S1 = fmaf(wxy, f, S1);
                    S2 = fmaf(wxy, __saturatef(f - 1.0f), S2);
                    if (j == 4 && fmaf(lam_hi, invg, -5.5f) <= klo) break;  // k = klo + 5 is past the window
                    ex += gNx; ey += gNy; f += gv;
                }
                const float W2 = S2, W1 = fmaf(-2.0f, S2, S1), W0 = (S0 - S1) + S2;
#pragma unroll
                for (int cc = 0; cc < CB; ++cc) {
#pragma unroll
                    for (int r = 0; r < NR; ++r) {
                        R[0][cc][r] = fmaf(W0, y0[cc][r], R[0][cc][r]);
                        R[1][cc][r] = fmaf(W1, y0[cc][r], R[1][cc][r]);
                        R[2][cc][r] = fmaf(W2, y0[cc][r], R[2][cc][r]);
                    }
                    if (NM == 2) {
#pragma unroll
                        for (int r = 0; r < NR; ++r) {
                            R[0][(NM - 1) * CB + cc][r] = fmaf(W0, y1[cc][r], R[0][(NM - 1) * CB + cc][r]);
                            R[1][(NM - 1) * CB + cc][r] = fmaf(W1, y1[cc][r], R[1][(NM - 1) * CB + cc][r]);
                            R[2][(NM - 1) * CB + cc][r] = fmaf(W2, y1[cc][r], R[2][(NM - 1) * CB + cc][r]);
                        }
                    }
                }
            }
        }
    }

    if (!valid) return;
    // ---- stores: rotation r maps (ix, iy) -> r quarter (NR = 4) or half (NR = 2) turns ----
    for (int t = 0; t < nzc; ++t) {
        const int izt = zc0 + t;
#pragma unroll
        for (int m = 0; m < NM; ++m) {
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
                    const float val = sacc[t * NACC + (m * CB + cc) * NR + r][tid] * G.scale;
                    float *dst = vol + cc * vol_cstride + o;
                    *dst = accumulate ? *dst + val : val;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------
// launcher
// ---------------------------------------------------------------------------
// planes per thread: the totals of a column take ZC * NR * NM * CB floats of shared memory per thread
#ifndef ADJC_FLOATS
#define ADJC_FLOATS 64
#endif

template <int NR, int NM, int CB, int CI = 1>
static int launch_column(cbct_geom *g, AdjGeom &G, const float *sinoI, float *vol, size_t sstride, size_t vstride,
                         int vol_z_origin, float *partial, int nsplit, cudaStream_t st)
{
    constexpr int NACC = NR * NM * CB;
    // (16 accumulators per plane -- 2 channels at full symmetry -- measured best with 6 planes: 24.5 against 26.0 ms)
    constexpr int ZC = NACC == 16 ? 6 : (ADJC_FLOATS / NACC < 4 ? 4 : (ADJC_FLOATS / NACC > 32 ? 32 : ADJC_FLOATS / NACC));
#ifndef ADJC_MINB
#define ADJC_MINB 0
#endif
    constexpr int MINB = ADJC_MINB;
    auto kernel = adjoint_column_kernel<NR, NM, CB, ZC, MINB, CI>;
    const size_t smem = (size_t)ZC * NACC * ADJC_NT * sizeof(float);
    const int nq_total = g->d.n_views;
    G.nbase = g->d.n_views / NR;
    {   // leave the rest of the 256 KB to L1 (the gather lives on its L1 hit rate); once per device and instance
        static std::atomic<uint64_t> carved{0};
        int devid = 0;
        cudaGetDevice(&devid);
        const uint64_t bit = (uint64_t)1 << (devid & 63);
        if (!(carved.fetch_or(bit) & bit)) {
            int max_ctas = 0;
            cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&max_ctas, kernel, ADJC_NT, smem);
            if (max_ctas < 1) max_ctas = 1;
            const size_t per_cta = smem + 1024;
            int pct = (int)((max_ctas * per_cta * 100 + 228 * 1024 - 1) / (228 * 1024));
            if (pct > 100) pct = 100;
            cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pct);
        }
    }
    ViewChunk vc;
    dim3 block(ADJ_BX, ADJC_BY, 1);
    const int nch = (G.bz1 - G.bz0 + ZC - 1) / ZC;
    dim3 grid((G.bx + ADJ_BX - 1) / ADJ_BX, (G.by + ADJC_BY - 1) / ADJC_BY, nch);
    if (partial && nsplit > 1) {
        // the views of every launch (chunks of 512) split over nsplit CTAs per tile into partial outputs of the whole
        // grid -- group s of every chunk adds into partial volume s -- then reduced in a fixed order
        const size_t nvox = (size_t)G.nx * G.ny * G.nz;
        G.nsplit = nsplit;
        G.split_stride = (size_t)CB * nvox;
        grid.z = nch * nsplit;
        for (int q0 = 0; q0 < nq_total; q0 += CBCT_VIEWS_PER_LAUNCH) {
            int n = nq_total - q0;
            if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
            for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
            G.nq = n;
            G.views_per_split = (n + nsplit - 1) / nsplit;
            cbct_prof_begin(g, CBCT_KERNEL_ADJOINT, st);
            kernel<<<grid, block, smem, st>>>(sinoI, partial, G, vc, q0, q0 > 0, sstride, nvox, 0);
            cbct_prof_end(g, CBCT_KERNEL_ADJOINT, st);
            int rc = cbct_check_launch(g, "adjoint_column_kernel");
            if (rc) return rc;
        }
        return cbct_launch_reduce_splits(g, partial, vol, nvox, CB, nsplit, vstride, st);
    }
    G.nsplit = 1; G.views_per_split = CBCT_VIEWS_PER_LAUNCH; G.split_stride = 0;
    for (int q0 = 0; q0 < nq_total; q0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = nq_total - q0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
        G.nq = n;
        cbct_prof_begin(g, CBCT_KERNEL_ADJOINT, st);
        kernel<<<grid, block, smem, st>>>(sinoI, vol, G, vc, q0, q0 > 0, sstride, vstride, vol_z_origin);
        cbct_prof_end(g, CBCT_KERNEL_ADJOINT, st);
        int rc = cbct_check_launch(g, "adjoint_column_kernel");
        if (rc) return rc;
    }
    return CBCT_OK;
}

template <int NR, int NM>
static int launch_column_cb(cbct_geom *g, AdjGeom &G, int CB, int CI, const float *sinoI, float *vol, size_t sstride,
                            size_t vstride, int vol_z_origin, float *partial, int nsplit, cudaStream_t st)
{
    if (CI != 1 && !(CI == 4 && NR == 1 && (CB == 4 || (CB == 8 && NM == 1)))) return CBCT_ERR_INVALID_ARG;
    // the partial outputs of the view groups take nsplit * CB volumes: at most 16 (cbct_adjoint_partial_floats)
    if (nsplit * CB > 16) nsplit = 16 / CB;
    if (CB == 1) return launch_column<NR, NM, 1>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    if (CB == 2) return launch_column<NR, NM, 2>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    // geometries with few symmetric images fill the window's 8 accumulators per plane with channels instead
    if constexpr (NR == 1) {
        if (CB == 4 && CI == 4) return launch_column<NR, NM, 4, 4>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
        if (CB == 8 && CI == 4 && NM == 1) return launch_column<NR, 1, 8, 4>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    }
    if constexpr (NR * NM <= 2) {
        if (CB == 4) return launch_column<NR, NM, 4>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    }
    if constexpr (NR * NM == 1) {
        if (CB == 8) return launch_column<NR, NM, 8>(g, G, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    }
    return 1;
}

int cbct_launch_adjoint_column(cbct_geom *g, AdjGeom &G, int NR, int NM, int CB, int CI, const float *sinoI, float *vol,
                               size_t sstride, size_t vstride, int vol_z_origin, float *partial, int nsplit,
                               cudaStream_t st)
{
    // preconditions of the three-plane identity and of the 6-sample window (see the header): f < 2 needs
    // 2 zb = 2 sqrt 2 |v| / sdd < 1 on every detector row; longer windows take the voxel kernel's walking variant
    if (G.fine || !(G.tz < 0.35f)) return 1;
    if (NR == 4) return NM == 2 ? launch_column_cb<4, 2>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st)
                                : launch_column_cb<4, 1>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    if (NR == 2) return NM == 2 ? launch_column_cb<2, 2>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st)
                                : launch_column_cb<2, 1>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
    return NM == 2 ? launch_column_cb<1, 2>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st)
                   : launch_column_cb<1, 1>(g, G, CB, CI, sinoI, vol, sstride, vstride, vol_z_origin, partial, nsplit, st);
}
