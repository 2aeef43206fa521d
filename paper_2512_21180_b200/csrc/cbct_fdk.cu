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

// Re-layout of the sinogram for the backprojection kernel: one RECORD per padded pixel (pv, pu) of base view ib, zero
// outside the detector (boundary rule R10 without bounds tests), so that one vector load serves
//   NR = 4 (16 B): the pixel in the 4 views ib + p nb related by quarter turns   (4 LDG.128 = 4 taps of 4 voxels)
//   NR = 2 ( 8 B): the pixel in the 2 views ib, ib + nb                          (4 LDG.64  = 4 taps of 2 voxels)
//   NR = 1 (16 B): the 2 x 2 taps (v, u), (v, u + 1), (v + 1, u), (v + 1, u + 1)  (1 LDG.128 = 4 taps of 1 voxel)
// i.e. 16 B through L1 per voxel-view whatever the symmetry of the view angles (scalar taps made geometries without
// rotation symmetry twice as slow: 8.6 against 4.6 ms per channel at 256^3 / 400 views; the quad records: 6.7 ms --
// they cost L1 capacity, every pixel being stored four times; for NR = 2 the same trick -- records (u, u + 1) x
// 2 views, 2 LDG.128 -- measured slower than the plain pair of views, 6.7 against 5.8 ms, and was dropped).
#define FDK_RECF(NR) ((NR) == 2 ? 2 : 4)   // floats per record

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
        const float *src = in + (c * NR * nb + ib) * img;
        auto px = [&](int r, int vv, int uu) -> float {
            return (uu >= 0 && uu < nu && vv >= 0 && vv < nv) ? __ldg(src + (size_t)r * nb * img + (size_t)vv * nu + uu) : 0.f;
        };
        if (NR == 4) reinterpret_cast<float4 *>(out)[e] = make_float4(px(0, v, u), px(1, v, u), px(2, v, u), px(NR - 1, v, u));
        else if (NR == 2) reinterpret_cast<float2 *>(out)[e] = make_float2(px(0, v, u), px(NR - 1, v, u));
        else reinterpret_cast<float4 *>(out)[e] = make_float4(px(0, v, u), px(0, v, u + 1), px(0, v + 1, u), px(0, v + 1, u + 1));
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
// CB channels per thread share the whole per-(x, y, view) set-up (the fp64 coordinates, the weight) and the
// per-voxel row arithmetic; their records lie `sino_cstride` float4 apart.
// MB = CTAs per SM the register allocation aims for (0: the compiler's choice).  Not for occupancy's sake: the bound
// decides how many of a view's loads ptxas keeps in flight ahead of their use, and the kernel waits on its loads.
template <int NR, int NM, int ZB, int CB, int MB>
__global__ void __launch_bounds__(FDK_BX *FDK_BY, MB)
fdk_kernel(const float *__restrict__ sinoP, float *__restrict__ vol, const __grid_constant__ FdkGeom G,
           const __grid_constant__ FdkViews V, int q0, int accumulate, int vol_z_origin, size_t sino_cstride,
           size_t vol_cstride)
{
    const int ix = blockIdx.x * FDK_BX + threadIdx.x;
    const int iy = blockIdx.y * FDK_BY + threadIdx.y;
    const int izb = G.bz0 + blockIdx.z * ZB;
    if (ix >= G.bx || iy >= G.by) return;
    const double X = G.x0 + (double)ix, Y = G.y0 + (double)iy, Z0 = G.z0 + (double)izb;
    float acc[CB][NM][ZB][NR];
#pragma unroll
    for (int c = 0; c < CB; ++c)
#pragma unroll
        for (int m = 0; m < NM; ++m)
#pragma unroll
            for (int k = 0; k < ZB; ++k)
#pragma unroll
                for (int r = 0; r < NR; ++r) acc[c][m][k][r] = 0.f;
    const size_t pimg = (size_t)G.pu * G.pv;
    int a_prev = q0 / G.nbase;

    // bilinear interpolation of the NR views from the records of rows `row`, `row + 1` at column ju (rec points at
    // the record (row, ju)): fraction au along u, fv along v; adds w * value into dst[0 .. NR)
    constexpr int RECF = FDK_RECF(NR);
    const int rowstride = G.pu * RECF;
    auto taps = [&](const float *__restrict__ rec, float au, float fv, float w, float (&dst)[NR]) {
        if (NR == 1) {
            const float4 t = __ldg(reinterpret_cast<const float4 *>(rec));   // (v u, v u+1, v+1 u, v+1 u+1)
            const float b0 = fmaf(au, t.y - t.x, t.x), b1 = fmaf(au, t.w - t.z, t.z);
            dst[0] = fmaf(w, fmaf(fv, b1 - b0, b0), dst[0]);
        } else {
            float y00[NR], y01[NR], y10[NR], y11[NR];
            load_views<NR>(rec, y00);
            load_views<NR>(rec + NR, y01);
            load_views<NR>(rec + rowstride, y10);
            load_views<NR>(rec + rowstride + NR, y11);
#pragma unroll
            for (int rr = 0; rr < NR; ++rr) {
                const float b0 = fmaf(au, y01[rr] - y00[rr], y00[rr]), b1 = fmaf(au, y11[rr] - y10[rr], y10[rr]);
                dst[rr] = fmaf(w, fmaf(fv, b1 - b0, b0), dst[rr]);
            }
        }
    };

    for (int q = 0; q < G.n_views; ++q) {
        // during the views of block a the accumulator of the r-th rotated voxel is
        // component (r + a) mod NR, matching the stored component of view i + r nbase
        const int a = (q0 + q) / G.nbase, ib = (q0 + q) - a * G.nbase;
        if (NR > 1 && a != a_prev) {
#pragma unroll
            for (int c = 0; c < CB; ++c)
#pragma unroll
                for (int m = 0; m < NM; ++m)
#pragma unroll
                    for (int k = 0; k < ZB; ++k) rotate_views<NR>(acc[c][m][k], NR - (a - a_prev));
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
        const float *p = sinoP + ((size_t)ib * pimg + ju) * RECF;
#pragma unroll
        for (int k = 0; k < ZB; ++k) {
            const float t = fminf(fmaxf(fmaf((float)k, dfv, f0), lo), hi);
            int jr;
            float av;
            cbct_cell_frac(t - 0.5f, jr, av);
            const int row = jv0 + jr;
#pragma unroll
            for (int cc = 0; cc < CB; ++cc) {
                taps(p + cc * sino_cstride + row * rowstride, au, av, w, acc[cc][0][k]);
                // voxel mirrored in z: rows pv-2-row and pv-1-row, fraction 1 - av
                if (NM == 2) taps(p + cc * sino_cstride + (G.pv - 2 - row) * rowstride, au, 1.0f - av, w, acc[cc][NM - 1][k]);
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
#pragma unroll
            for (int cc = 0; cc < CB; ++cc) rotate_views<NR>(acc[cc][m][k], a_prev);
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
#pragma unroll
                for (int cc = 0; cc < CB; ++cc) {
                    float *d = dst + cc * vol_cstride;
                    *d = accumulate ? *d + acc[cc][m][k][r] : acc[cc][m][k][r];
                }
            }
        }
}

// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
// floats per channel of the re-laid-out sinogram: one 16-byte record per padded pixel of every base view
size_t cbct_padded_sino_floats(const cbct_geom *g)
{
    return (size_t)(g->d.n_views / g->sym_rot) * cbct_padded_sino_pitch(g) * cbct_padded_sino_rows(g) * FDK_RECF(g->sym_rot);
}

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

// Two channels per thread share the fp64 set-up of a (column, view) pair.  It pays only without rotation symmetry
// (8 channels with jittered angles: 6.0 against 6.7 ms per channel); with NR = 4 the 125 registers of the
// two-channel instance cut the resident warps from 24 to 16 per SM and the kernel, which waits on its loads, slows
// from 4.7 to 5.3 ms per channel.
#ifndef FDK_CB
#define FDK_CB 2
#endif

template <int NR, int NM, int ZB, int MB = 0, int MB2 = MB>
static int launch_fdk(cbct_geom *g, FdkGeom &G, const float *padded, float *vol, int channels, size_t vstride,
                      int vol_z_origin, cudaStream_t st)
{
    const cbct_geom_desc &d = g->d;
    const size_t sstride = cbct_padded_sino_floats(g);  // floats per channel of the re-laid-out sinogram
    const float *rec = padded;
    G.nbase = d.n_views / NR;
    FdkViews fv;
    dim3 block(FDK_BX, FDK_BY);
    dim3 grid((G.bx + FDK_BX - 1) / FDK_BX, (G.by + FDK_BY - 1) / FDK_BY, (G.bz1 - G.bz0 + ZB - 1) / ZB);
    for (int q0 = 0; q0 < d.n_views; q0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = d.n_views - q0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) fv.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
        G.n_views = n;
        int c = 0;
        while (c < channels) {
            cbct_prof_begin(g, CBCT_KERNEL_FDK, st);
            if (FDK_CB >= 2 && NR == 1 && channels - c >= 2) {
                fdk_kernel<NR, NM, ZB, 2, MB2><<<grid, block, 0, st>>>(rec + c * sstride, vol + c * vstride, G, fv, q0, q0 > 0,
                                                                  vol_z_origin, sstride, vstride);
                c += 2;
            } else {
                fdk_kernel<NR, NM, ZB, 1, MB><<<grid, block, 0, st>>>(rec + c * sstride, vol + c * vstride, G, fv, q0, q0 > 0,
                                                                  vol_z_origin, sstride, vstride);
                c += 1;
            }
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
    // planes per thread and register bound per instance, measured at 256^3 / 400 views (ms per channel; the bound
    // steers how many loads ptxas keeps in flight, see fdk_kernel): NR 4 / NM 2: 3 planes, bound 7: 4.48 (no bound
    // 4.62; 2 planes 4.75, 4: 4.51, 8: 5.6);  NR 2 / NM 2: 8 planes, bound 4: 4.95 (no bound 6.11);  NR 1 / NM 2:
    // 8 planes, bound 7: 5.60 (no bound 6.80), two channels per thread with bound 4: 4.64 per channel.
    if (NR == 4) return mirror ? launch_fdk<4, 2, 3, 7>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                               : launch_fdk<4, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
    if (NR == 2) return mirror ? launch_fdk<2, 2, 8, 4>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                               : launch_fdk<2, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
    return mirror ? launch_fdk<1, 2, 8, 7, 4>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st)
                  : launch_fdk<1, 1, 8>(g, G, padded_sino, vol, channels, vs, vol_z_origin, st);
}
