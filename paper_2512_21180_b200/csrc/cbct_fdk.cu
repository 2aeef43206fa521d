// cbct_fdk.cu -- A4, the voxel-driven FDK-weighted backprojection (PAPER.md:157,
// :181 Alg. 1 l.3, ref [9] :397; readings R9-R11 in DESIGN.md s.3):
//     vol_c[z,y,x] = sum_i (SID/U_i)^2 * B[sino_c,i](fv, fu).
#include "cbct_device.cuh"

int cbct_check_launch(cbct_geom *g, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cbct_set_cuda_error(e, what); return CBCT_ERR_CUDA; }
    g->launches++;
    return CBCT_OK;
}

static unsigned grid_for(size_t n, int block)
{
    size_t b = (n + block - 1) / block;
    size_t cap = 148u * 32u;
    return (unsigned)(b < cap ? (b ? b : 1) : cap);
}

// zero-bordered copy of the sinogram: rows = channels * views * pv padded rows
__global__ void pad_sino_kernel(const float *__restrict__ src, float *__restrict__ dst, int nu, int nv, int pu,
                                int pv, size_t n_rows_total)
{
    // rows = channels * views * pv padded rows
    size_t n = n_rows_total * pu;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        int u = (int)(e % pu) - CBCT_PAD;
        size_t row = e / pu;
        int v = (int)(row % pv) - CBCT_PAD;
        size_t img = row / pv;
        float val = 0.f;
        if (u >= 0 && u < nu && v >= 0 && v < nv) val = src[(img * nv + v) * nu + u];
        dst[e] = val;
    }
}

// ---------------------------------------------------------------------------
// A4 FDK backprojection, v0: thread per (x, y) with FDK_ZB consecutive z in
// registers; per (x, y, view): one reciprocal, u* and the weight are constant
// along z and v* is affine in z.  Taps come from the zero-padded sinogram.
// ---------------------------------------------------------------------------
#define FDK_ZB 8
#define FDK_BX 32
#define FDK_BY 4

struct FdkViews {
    double2 cs[CBCT_VIEWS_PER_LAUNCH];
};

// Per (x, y, view) the detector coordinates are set up in fp64 and split into
// an integer cell and an fp32 fraction, so the fp32 work along z only ever
// sees small magnitudes (|t| < ~32): coordinate error ~1e-6 px instead of the
// 1.5e-5 px ulp of a raw fp32 coordinate near 256 (DESIGN.md s.6).
__global__ void __launch_bounds__(FDK_BX *FDK_BY)
fdk_kernel_v0(const float *__restrict__ sino, float *__restrict__ vol, const __grid_constant__ FdkGeom G,
              const __grid_constant__ FdkViews V, int view0, int accumulate, size_t vol_plane_origin)
{
    int ix = blockIdx.x * FDK_BX + threadIdx.x;
    int iy = blockIdx.y * FDK_BY + threadIdx.y;
    int izb = G.zs0 + blockIdx.z * FDK_ZB;
    if (ix >= G.nx || iy >= G.ny) return;
    const double X = G.x0 + (double)ix, Y = G.y0 + (double)iy, Z0 = G.z0 + (double)izb;
    float acc[FDK_ZB];
#pragma unroll
    for (int k = 0; k < FDK_ZB; ++k) acc[k] = 0.f;
    const size_t img = (size_t)G.pu * G.pv;
    for (int i = 0; i < G.n_views; ++i) {
        double c = V.cs[i].x, s = V.cs[i].y;
        double U = G.sid - (X * c + Y * s);
        double r = (double)__frcp_rn((float)U);
        r = r * (2.0 - U * r);  // one Newton step: relative error ~1e-14
        double fu = fmin(fmax(G.au * (Y * c - X * s) * r + G.bu, 1.0), G.fu_max);
        double fuf = floor(fu);
        int ju = (int)fuf;
        float au = (float)(fu - fuf);
        float w = (float)(G.sid * r);
        w *= w;
        double dfv_d = G.av * r;
        double fv0 = Z0 * dfv_d + G.bv;
        // keep the integer part of fv0 out of the fp32 arithmetic (clamped so the
        // relative coordinate stays small even for voxels projecting far outside)
        double base = floor(fmin(fmax(fv0, -64.0), G.fv_max + 64.0));
        int jv0 = (int)base;
        float f0 = (float)(fv0 - base), dfv = (float)dfv_d;
        float lo = 1.0f - (float)jv0, hi = (float)(G.fv_max - base);
        const float *p = sino + (size_t)(view0 + i) * img + ju;
#pragma unroll
        for (int k = 0; k < FDK_ZB; ++k) {
            float t = fminf(fmaxf(fmaf((float)k, dfv, f0), lo), hi);
            int jr;
            float av;
            cbct_cell_frac(t - 0.5f, jr, av);
            const float *q = p + (size_t)(jv0 + jr) * G.pu;
            float p00 = __ldg(q), p01 = __ldg(q + 1), p10 = __ldg(q + G.pu), p11 = __ldg(q + G.pu + 1);
            float b0 = fmaf(au, p01 - p00, p00), b1 = fmaf(au, p11 - p10, p10);
            acc[k] = fmaf(w, fmaf(av, b1 - b0, b0), acc[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < FDK_ZB; ++k) {
        int iz = izb + k;
        if (iz < G.zs1) {
            size_t o = ((size_t)iz * G.ny + iy) * G.nx + ix - vol_plane_origin;
            vol[o] = accumulate ? vol[o] + acc[k] : acc[k];
        }
    }
}

// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
int cbct_launch_pad_sino(cbct_geom *g, const float *src, float *dst, int channels, cudaStream_t st)
{
    int pu = cbct_padded_sino_pitch(g), pv = cbct_padded_sino_rows(g);
    size_t rows = (size_t)channels * g->d.n_views * pv;
    pad_sino_kernel<<<grid_for(rows * pu, 256), 256, 0, st>>>(src, dst, g->d.det_nu, g->d.det_nv, pu, pv, rows);
    return cbct_check_launch(g, "pad_sino_kernel");
}

int cbct_launch_fdk(cbct_geom *g, const float *padded_sino, float *vol, int channels, int zs0, int zs1,
                    size_t vol_channel_stride, int vol_z_origin, cudaStream_t st)
{
    const cbct_geom_desc &d = g->d;
    double h = d.vox_mm;
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
    G.zs0 = zs0; G.zs1 = zs1;
    G.pu = cbct_padded_sino_pitch(g);
    G.pv = cbct_padded_sino_rows(g);
    size_t sstride = (size_t)d.n_views * G.pu * G.pv;
    size_t origin = (size_t)vol_z_origin * d.vol_ny * d.vol_nx;
    FdkViews fv;
    dim3 block(FDK_BX, FDK_BY);
    dim3 grid((d.vol_nx + FDK_BX - 1) / FDK_BX, (d.vol_ny + FDK_BY - 1) / FDK_BY, (zs1 - zs0 + FDK_ZB - 1) / FDK_ZB);
    for (int view0 = 0; view0 < d.n_views; view0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = d.n_views - view0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) fv.cs[i] = make_double2(g->cosphi[view0 + i], g->sinphi[view0 + i]);
        G.n_views = n;
        for (int c = 0; c < channels; ++c) {
            fdk_kernel_v0<<<grid, block, 0, st>>>(padded_sino + c * sstride, vol + c * vol_channel_stride, G, fv,
                                                  view0, view0 > 0, origin);
            int rc = cbct_check_launch(g, "fdk_kernel_v0");
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}
