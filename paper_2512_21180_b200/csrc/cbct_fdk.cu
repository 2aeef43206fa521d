// cbct_fdk.cu -- A4, the voxel-driven FDK-weighted backprojection (PAPER.md:157,
// :181 Alg. 1 l.3, ref [9] :397; readings R9-R11 in DESIGN.md s.3):
//     vol_c[z,y,x] = sum_i (SID/U_i)^2 * B[sino_c,i](fv, fu),
//     U_i = SID - (x cos phi_i + y sin phi_i),  u* = SDD (-x sin phi_i + y cos phi_i) / U_i,
//     v* = SDD z / U_i,  B = zero-extended bilinear interpolation on the detector.
//
// Design (DESIGN.md s.6).  One thread per (x, y) column with ZB consecutive z in
// registers: per (x, y, view) one fp64 set-up (U, 1/U, u*, weight); along z, u*
// and the weight are constant and v* is affine.  As in the gather adjoint the
// geometry of (view i, voxel j) equals that of (view i + r n/NR, voxel j rotated
// by r 360/NR degrees) and of the z-mirrored voxel with detector row nv-1-iv, so
// a thread owns a base column in one quadrant / the lower half and accumulates
// NR * NM voxels from one coordinate computation.  The sinogram is re-laid out
// once per call with a zero border (no bounds tests; boundary rule R10) and with
// the NR rotation-related views side by side (one LDG.128 per tap for 4 views).
#include "cbct_device.cuh"

int cbct_check_launch(cbct_geom *g, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cbct_set_cuda_error(e, what); return CBCT_ERR_CUDA; }
    g->launches++;
    return CBCT_OK;
}

// out[c][ib][pv][pu][p] = in[c][ib + p nb][v][u] inside the detector, 0 on the border
template <int NR>
__global__ void __launch_bounds__(256)
pad_sino_kernel(const float *__restrict__ in, float *__restrict__ out, int nu, int nv, int pu, int pv, int nb,
                int channels)
{
    const size_t pimg = (size_t)pu * pv, img = (size_t)nu * nv;
    const size_t n = (size_t)channels * nb * pimg;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int u = (int)(e % pu) - CBCT_PAD;
        size_t t = e / pu;
        const int v = (int)(t % pv) - CBCT_PAD;
        t /= pv;
        const size_t ib = t % nb, c = t / nb;
        float vals[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) vals[r] = 0.f;
        if (u >= 0 && u < nu && v >= 0 && v < nv) {
            const float *src = in + (c * NR * nb + ib) * img + (size_t)v * nu + u;
#pragma unroll
            for (int r = 0; r < NR; ++r) vals[r] = __ldg(src + (size_t)r * nb * img);
        }
        if (NR == 4) reinterpret_cast<float4 *>(out)[e] = make_float4(vals[0], vals[1], vals[2], vals[NR - 1]);
        else if (NR == 2) reinterpret_cast<float2 *>(out)[e] = make_float2(vals[0], vals[NR - 1]);
        else out[e] = vals[0];
    }
}

// ---------------------------------------------------------------------------
// backprojection kernel
// ---------------------------------------------------------------------------
// A warp covers 4 (x) x 8 (y) columns, so a quarter-warp (the unit the L1 data stage serves per
// cycle for LDG.128) is a compact 4 x 2 patch: its 8 taps fall on ~5.7 distinct pixels within
// ~8 detector columns instead of ~7.2 pixels over ~11 columns for 8 columns in a row, which
// halves the 16-byte-position conflicts (profiles/r1_l1_microbench.md; simulated 1.76 -> 1.29
// cycles per quarter-warp; measured 5.85 -> 5.18 ms).  A row-dependent swizzle of the sinogram
// (simulated 1.22) cost more address arithmetic than it saved (6.2 ms) and was dropped.
#define FDK_BX 4
#define FDK_BY 32

struct FdkViews {
    double2 cs[CBCT_VIEWS_PER_LAUNCH];
};

// Per (x, y, view) the detector coordinates are set up in fp64 and split into
// an integer cell and an fp32 fraction, so the fp32 work along z only ever
// sees small magnitudes (|t| < ~32): coordinate error ~1e-6 px instead of the
// 1.5e-5 px ulp of a raw fp32 coordinate near 256 (DESIGN.md s.6).
template <int NR, int NM, int ZB>
__global__ void __launch_bounds__(FDK_BX *FDK_BY)
fdk_kernel(const float *__restrict__ sinoP, float *__restrict__ vol, const __grid_constant__ FdkGeom G,
           const __grid_constant__ FdkViews V, int q0, int accumulate, int vol_z_origin)
{
    const int ix = blockIdx.x * FDK_BX + threadIdx.x;
    const int iy = blockIdx.y * FDK_BY + threadIdx.y;
    const int izb = G.bz0 + blockIdx.z * ZB;
    if (ix >= G.bx || iy >= G.by) return;
    const double X = G.x0 + (double)ix, Y = G.y0 + (double)iy, Z0 = G.z0 + (double)izb;
    float acc[NM][ZB][NR];
#pragma unroll
    for (int m = 0; m < NM; ++m)
#pragma unroll
        for (int k = 0; k < ZB; ++k)
#pragma unroll
            for (int r = 0; r < NR; ++r) acc[m][k][r] = 0.f;
    const size_t pimg = (size_t)G.pu * G.pv;
    const int rowstride = G.pu * NR;
    int a_prev = q0 / G.nbase;

    for (int q = 0; q < G.n_views; ++q) {
        // during the views of block a the accumulator of the r-th rotated voxel is
        // component (r + a) mod NR, matching the stored component of view i + r nbase
        const int a = (q0 + q) / G.nbase, ib = (q0 + q) - a * G.nbase;
        if (NR > 1 && a != a_prev) {
#pragma unroll
            for (int m = 0; m < NM; ++m)
#pragma unroll
                for (int k = 0; k < ZB; ++k) rotate_views<NR>(acc[m][k], NR - (a - a_prev));
            a_prev = a;
        }
        const double c = V.cs[q].x, s = V.cs[q].y;
        const double U = G.sid - (X * c + Y * s);
        double r = (double)__frcp_rn((float)U);
        r = r * (2.0 - U * r);  // one Newton step: relative error ~1e-14
        const double fu = fmin(fmax(G.au * (Y * c - X * s) * r + G.bu, 1.0), G.fu_max);
        const double fuf = floor(fu);
        const int ju = (int)fuf;
        const float au = (float)(fu - fuf);
        float w = (float)(G.sid * r);
        w *= w;
        const double dfv_d = G.av * r;
        const double fv0 = Z0 * dfv_d + G.bv;
        // keep the integer part of fv0 out of the fp32 arithmetic (clamped so the
        // relative coordinate stays small even for voxels projecting far outside)
        const double base = floor(fmin(fmax(fv0, -64.0), G.fv_max + 64.0));
        const int jv0 = (int)base;
        const float f0 = (float)(fv0 - base), dfv = (float)dfv_d;
        const float lo = 1.0f - (float)jv0, hi = (float)(G.fv_max - base);
        const float *p = sinoP + ((size_t)ib * pimg + ju) * NR;
#pragma unroll
        for (int k = 0; k < ZB; ++k) {
            const float t = fminf(fmaxf(fmaf((float)k, dfv, f0), lo), hi);
            int jr;
            float av;
            cbct_cell_frac(t - 0.5f, jr, av);
            const int row = jv0 + jr;
            {
                const float *q00 = p + row * rowstride;
                float y00[NR], y01[NR], y10[NR], y11[NR];
                load_views<NR>(q00, y00);
                load_views<NR>(q00 + NR, y01);
                load_views<NR>(q00 + rowstride, y10);
                load_views<NR>(q00 + rowstride + NR, y11);
#pragma unroll
                for (int rr = 0; rr < NR; ++rr) {
                    const float b0 = fmaf(au, y01[rr] - y00[rr], y00[rr]), b1 = fmaf(au, y11[rr] - y10[rr], y10[rr]);
                    acc[0][k][rr] = fmaf(w, fmaf(av, b1 - b0, b0), acc[0][k][rr]);
                }
            }
            if (NM == 2) {  // voxel mirrored in z: rows pv-2-row and pv-1-row, fraction 1 - av
                const float *q00 = p + (G.pv - 2 - row) * rowstride;
                float y00[NR], y01[NR], y10[NR], y11[NR];
                load_views<NR>(q00, y00);
                load_views<NR>(q00 + NR, y01);
                load_views<NR>(q00 + rowstride, y10);
                load_views<NR>(q00 + rowstride + NR, y11);
#pragma unroll
                for (int rr = 0; rr < NR; ++rr) {
                    const float b0 = fmaf(au, y01[rr] - y00[rr], y00[rr]), b1 = fmaf(au, y11[rr] - y10[rr], y10[rr]);
                    acc[NM - 1][k][rr] = fmaf(w, fmaf(av, b0 - b1, b1), acc[NM - 1][k][rr]);
                }
            }
        }
    }

    // ---- stores ----
#pragma unroll
    for (int m = 0; m < NM; ++m)
#pragma unroll
        for (int k = 0; k < ZB; ++k) {
            const int izk = izb + k;
            if (izk >= G.bz1) continue;
            const int z = m == 0 ? izk : G.nz - 1 - izk;
            if (m == 1 && z == izk) continue;  // middle plane of an odd nz is its own mirror image
            rotate_views<NR>(acc[m][k], a_prev);
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
                float *dst = vol + ((size_t)(z - (m == 0 ? vol_z_origin : G.mz_origin)) * G.ny + y) * G.nx + x;
                *dst = accumulate ? *dst + acc[m][k][r] : acc[m][k][r];
            }
        }
}

// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
int cbct_launch_pad_sino(cbct_geom *g, const float *src, float *dst, int channels, cudaStream_t st)
{
    const int NR = g->sym_rot, nb = g->d.n_views / NR;
    const int pu = cbct_padded_sino_pitch(g), pv = cbct_padded_sino_rows(g);
    const size_t n = (size_t)channels * nb * pu * pv;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    if (NR == 4) pad_sino_kernel<4><<<(unsigned)blocks, 256, 0, st>>>(src, dst, g->d.det_nu, g->d.det_nv, pu, pv, nb, channels);
    else if (NR == 2) pad_sino_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(src, dst, g->d.det_nu, g->d.det_nv, pu, pv, nb, channels);
    else pad_sino_kernel<1><<<(unsigned)blocks, 256, 0, st>>>(src, dst, g->d.det_nu, g->d.det_nv, pu, pv, nb, channels);
    return cbct_check_launch(g, "pad_sino_kernel");
}

template <int NR, int NM, int ZB>
static int launch_fdk(cbct_geom *g, FdkGeom &G, const float *padded, float *vol, int channels, size_t vstride,
                      int vol_z_origin, cudaStream_t st)
{
    const cbct_geom_desc &d = g->d;
    const size_t sstride = (size_t)d.n_views * G.pu * G.pv;  // floats per channel of the re-laid-out sinogram
    G.nbase = d.n_views / NR;
    FdkViews fv;
    dim3 block(FDK_BX, FDK_BY);
    dim3 grid((G.bx + FDK_BX - 1) / FDK_BX, (G.by + FDK_BY - 1) / FDK_BY, (G.bz1 - G.bz0 + ZB - 1) / ZB);
    for (int q0 = 0; q0 < d.n_views; q0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = d.n_views - q0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) fv.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
        G.n_views = n;
        for (int c = 0; c < channels; ++c) {
            cbct_prof_begin(g, CBCT_KERNEL_FDK, st);
            fdk_kernel<NR, NM, ZB><<<grid, block, 0, st>>>(padded + c * sstride, vol + c * vstride, G, fv, q0, q0 > 0,
                                                           vol_z_origin);
            cbct_prof_end(g, CBCT_KERNEL_FDK, st);
            int rc = cbct_check_launch(g, "fdk_kernel");
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}

// `padded_sino` is the output of cbct_launch_pad_sino.  Writes planes [zs0, zs1) of vol
// (whose first stored plane is vol_z_origin); the z-mirror is used only when the
// launch covers the whole grid.
// mirror_z_origin != CBCT_NO_MIRROR_PAIR: as for cbct_launch_adjoint (a slab of the lower half plus its image).
int cbct_launch_fdk(cbct_geom *g, const float *padded_sino, float *vol, int channels, int zs0, int zs1,
                    size_t vol_channel_stride, int vol_z_origin, cudaStream_t st, int mirror_z_origin)
{
    const cbct_geom_desc &d = g->d;
    const bool pair = mirror_z_origin != CBCT_NO_MIRROR_PAIR;
    if (pair && (!g->sym_mirror_z || zs1 > (d.vol_nz + 1) / 2)) return CBCT_ERR_INVALID_ARG;
    const double h = d.vox_mm;
    FdkGeom G;
    G.sid = d.sid_mm / h;
    G.au = d.sdd_mm / d.det_du_mm;  // (SDD/h) / (du/h)
    G.av = d.sdd_mm / d.det_dv_mm;
    G.bu = (-(-0.5 * (d.det_nu - 1) * d.det_du_mm + d.det_off_u_mm) / d.det_du_mm + CBCT_PAD);
    G.bv = (-(-0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm) / d.det_dv_mm + CBCT_PAD);
    G.x0 = d.vol_cx_mm / h - 0.5 * (d.vol_nx - 1);
    G.y0 = d.vol_cy_mm / h - 0.5 * (d.vol_ny - 1);
    G.z0 = d.vol_cz_mm / h - 0.5 * (d.vol_nz - 1);
    G.fu_max = (double)(d.det_nu + CBCT_PAD);
    G.fv_max = (double)(d.det_nv + CBCT_PAD);
    G.nx = d.vol_nx; G.ny = d.vol_ny; G.nz = d.vol_nz;
    G.pu = cbct_padded_sino_pitch(g);
    G.pv = cbct_padded_sino_rows(g);
    const int NR = g->sym_rot;
    const bool mirror = pair || (g->sym_mirror_z && zs0 == 0 && zs1 == d.vol_nz && d.vol_nz > 1);
    G.bx = NR == 4 ? d.vol_nx / 2 : d.vol_nx;
    G.by = NR >= 2 ? d.vol_ny / 2 : d.vol_ny;
    G.bz0 = zs0; G.bz1 = pair ? zs1 : (mirror ? (d.vol_nz + 1) / 2 : zs1);
    G.mz_origin = pair ? mirror_z_origin : vol_z_origin;
    G.n_views = 0; G.nbase = 0;
    const size_t vs = vol_channel_stride;
    // z per thread: 3 measured best for the 8-voxel variant (1: 6.3 ms, 2: 4.8, 3: 4.6, 4: 5.2, 8: 5.3 per channel)
    if (NR == 4) return mirror ? launch_fdk<4, 2, 3>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                               : launch_fdk<4, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
    if (NR == 2) return mirror ? launch_fdk<2, 2, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                               : launch_fdk<2, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
    return mirror ? launch_fdk<1, 2, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                  : launch_fdk<1, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
}
