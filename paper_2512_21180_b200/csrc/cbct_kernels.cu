// cbct_kernels.cu -- sm_100a kernels of libcbct.so (forward projector A2, matched
// adjoint A3, FDK backprojection A4, pad/unpad layout passes).
//
// Definitions: Eq. (5) (P = line integral source -> detector
// element), PAPER.md:89 (P* = adjoint), PAPER.md:157/181/397 (FDK), geometry
// PAPER.md:61; discretisation readings R1-R11 in DESIGN.md s.3.
//
// Precision plan (DESIGN.md s.6): every ray is set up in fp64 (direction,
// box clip, anchor sample in the middle of its in-support range) and rounded
// once to fp32; the sample loop evaluates p_k = fma(k - k_mid, dstep, anchor)
// so no error accumulates along the ray.  floor() is replaced by
// round-to-nearest of (p - 1/2) with the 1.5*2^23 trick: any integer j with
// p - j in [0,1] yields the same trilinear value, so ties are harmless.
#include <math.h>

#include "cbct_internal.h"

#define MAGIC 12582912.0f           // 1.5 * 2^23
#define MAGIC_BITS 0x4B400000

// ---------------------------------------------------------------------------
// layout passes
// ---------------------------------------------------------------------------
__global__ void pad_volume_kernel(const float *__restrict__ src, float *__restrict__ dst, RayGeom G,
                                  size_t src_cstride, int src_z_origin, size_t dst_cstride)
{
    // one thread per padded element of (channel = blockIdx.z)
    size_t n = (size_t)G.px * G.py * G.pz;
    const float *s = src + (size_t)blockIdx.z * src_cstride;
    float *d = dst + (size_t)blockIdx.z * dst_cstride;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        int x = (int)(e % G.px) - CBCT_PAD;
        size_t t = e / G.px;
        int y = (int)(t % G.py) - CBCT_PAD;
        int z = (int)(t / G.py) - CBCT_PAD + G.z0;
        float v = 0.f;
        if (x >= 0 && x < G.nx && y >= 0 && y < G.ny && z >= G.z0 && z < G.z1)
            v = s[((size_t)(z - src_z_origin) * G.ny + y) * G.nx + x];
        d[e] = v;
    }
}

__global__ void unpad_volume_kernel(const float *__restrict__ padded, float *__restrict__ dst, RayGeom G,
                                    size_t pad_cstride, size_t dst_cstride, int dst_z_origin)
{
    size_t n = (size_t)G.nx * G.ny * (G.z1 - G.z0);
    const float *s = padded + (size_t)blockIdx.z * pad_cstride;
    float *d = dst + (size_t)blockIdx.z * dst_cstride;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        int x = (int)(e % G.nx);
        size_t t = e / G.nx;
        int y = (int)(t % G.ny);
        int z = (int)(t / G.ny);  // relative to z0
        d[((size_t)(z + G.z0 - dst_z_origin) * G.ny + y) * G.nx + x] =
            s[((size_t)(z + CBCT_PAD) * G.py + (y + CBCT_PAD)) * G.px + (x + CBCT_PAD)];
    }
}

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
// per-ray setup (fp64), shared by the forward projector and its adjoint
// ---------------------------------------------------------------------------
struct Ray {
    float ax, ay, az;   // anchor sample position minus 1/2, padded index coordinates
    float dx, dy, dz;   // position increment per sample
    float kf0;          // first sample index relative to the anchor
    int n;              // number of samples to visit
};

__device__ __forceinline__ void clip_axis(double o, double d, double lo, double hi, double &tmin, double &tmax,
                                          bool &hit)
{
    if (d == 0.0) {
        hit = hit && (o > lo && o < hi);
    } else {
        double inv = 1.0 / d;
        double t0 = (lo - o) * inv, t1 = (hi - o) * inv;
        tmin = fmax(tmin, fmin(t0, t1));
        tmax = fmin(tmax, fmax(t0, t1));
    }
}

__device__ __forceinline__ Ray ray_setup(const RayGeom &G, double c, double s, int iu, int iv)
{
    Ray r;
    double u = G.u0 + iu * G.du, v = G.v0 + iv * G.dv;
    // D = pixel - source = -(SID+IDD)(c,s,0) + u(-s,c,0) + v(0,0,1)
    double sdd = G.sid + G.idd;
    double Dx = -sdd * c - u * s, Dy = -sdd * s + u * c, Dz = v;
    double L = sqrt(Dx * Dx + Dy * Dy + Dz * Dz);
    double invL = 1.0 / L;
    double dx = Dx * invL, dy = Dy * invL, dz = Dz * invL;
    // source in padded index coordinates
    double ox = G.sid * c - G.cx + 0.5 * (G.nx - 1) + CBCT_PAD;
    double oy = G.sid * s - G.cy + 0.5 * (G.ny - 1) + CBCT_PAD;
    double oz = -G.cz + 0.5 * (G.nz - 1) + CBCT_PAD - G.z0;
    double tmin = 0.0, tmax = L;
    bool hit = true;
    clip_axis(ox, dx, CBCT_PAD - 1.0, CBCT_PAD + (double)G.nx, tmin, tmax, hit);
    clip_axis(oy, dy, CBCT_PAD - 1.0, CBCT_PAD + (double)G.ny, tmin, tmax, hit);
    clip_axis(oz, dz, CBCT_PAD - 1.0, CBCT_PAD + (double)(G.z1 - G.z0), tmin, tmax, hit);
    r.n = 0;
    r.ax = r.ay = r.az = 1.f; r.dx = r.dy = r.dz = 0.f; r.kf0 = 0.f;
    if (!hit || !(tmin < tmax)) return r;
    double inv_step = 1.0 / G.step;
    long k0 = (long)ceil(tmin * inv_step - 0.5);    // first k with t_k >= tmin
    long k1 = (long)floor(tmax * inv_step - 0.5);   // last  k with t_k <= tmax
    if (k0 < 0) k0 = 0;
    if (k1 < k0) return r;
    long km = k0 + ((k1 - k0) >> 1);
    double tm = ((double)km + 0.5) * G.step;
    r.ax = (float)(ox + tm * dx - 0.5);
    r.ay = (float)(oy + tm * dy - 0.5);
    r.az = (float)(oz + tm * dz - 0.5);
    r.dx = (float)(G.step * dx);
    r.dy = (float)(G.step * dy);
    r.dz = (float)(G.step * dz);
    r.kf0 = (float)(k0 - km);
    r.n = (int)(k1 - k0 + 1);
    return r;
}

// Cell index and fractional offset from p - 1/2 (round-to-nearest trick).
__device__ __forceinline__ void cell_frac(float pm, int &j, float &a)
{
    float y = pm + MAGIC;
    j = __float_as_int(y) - MAGIC_BITS;
    a = (pm - (y - MAGIC)) + 0.5f;
}

// ---------------------------------------------------------------------------
// A2 forward projector, v0: one thread per ray, 8x4-pixel warp tiles, taps
// fetched with ld.global.nc from the padded volume (L1/L2 resident).
// ---------------------------------------------------------------------------
#define FP_TU 16
#define FP_TV 16

__device__ __forceinline__ void tile_pixel(int &iu, int &iv)
{
    // warp = 8(u) x 4(v) pixels; CTA = 2 x 4 warps = 16 x 16 pixels
    int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    iu = blockIdx.x * FP_TU + (warp & 1) * 8 + (lane & 7);
    iv = blockIdx.y * FP_TV + (warp >> 1) * 4 + (lane >> 3);
}

__device__ __forceinline__ float trilerp(const float *__restrict__ p, int sy, int sz, float fx, float fy, float fz)
{
    float v000 = __ldg(p), v001 = __ldg(p + 1);
    float v010 = __ldg(p + sy), v011 = __ldg(p + sy + 1);
    float v100 = __ldg(p + sz), v101 = __ldg(p + sz + 1);
    float v110 = __ldg(p + sz + sy), v111 = __ldg(p + sz + sy + 1);
    float a00 = fmaf(fx, v001 - v000, v000);
    float a01 = fmaf(fx, v011 - v010, v010);
    float a10 = fmaf(fx, v101 - v100, v100);
    float a11 = fmaf(fx, v111 - v110, v110);
    float b0 = fmaf(fy, a01 - a00, a00);
    float b1 = fmaf(fy, a11 - a10, a10);
    return fmaf(fz, b1 - b0, b0);
}

__global__ void __launch_bounds__(FP_TU *FP_TV)
fp_kernel_v0(const float *__restrict__ vol, float *__restrict__ sino, const __grid_constant__ RayGeom G,
             const __grid_constant__ ViewChunk V, int view0, int accumulate)
{
    int iu, iv;
    tile_pixel(iu, iv);
    if (iu >= G.nu || iv >= G.nv) return;
    int view = blockIdx.z;
    Ray r = ray_setup(G, V.cs[view].x, V.cs[view].y, iu, iv);
    const int sy = G.px, sz = G.px * G.py;
    float acc0 = 0.f, acc1 = 0.f;
    float kf = r.kf0;
    int it = 0;
    for (; it + 1 < r.n; it += 2, kf += 2.0f) {
        int jx, jy, jz, kx, ky, kz;
        float fx, fy, fz, gx, gy, gz;
        cell_frac(fmaf(kf, r.dx, r.ax), jx, fx);
        cell_frac(fmaf(kf, r.dy, r.ay), jy, fy);
        cell_frac(fmaf(kf, r.dz, r.az), jz, fz);
        float kg = kf + 1.0f;
        cell_frac(fmaf(kg, r.dx, r.ax), kx, gx);
        cell_frac(fmaf(kg, r.dy, r.ay), ky, gy);
        cell_frac(fmaf(kg, r.dz, r.az), kz, gz);
        acc0 += trilerp(vol + ((size_t)jz * G.py + jy) * G.px + jx, sy, sz, fx, fy, fz);
        acc1 += trilerp(vol + ((size_t)kz * G.py + ky) * G.px + kx, sy, sz, gx, gy, gz);
    }
    if (it < r.n) {
        int jx, jy, jz;
        float fx, fy, fz;
        cell_frac(fmaf(kf, r.dx, r.ax), jx, fx);
        cell_frac(fmaf(kf, r.dy, r.ay), jy, fy);
        cell_frac(fmaf(kf, r.dz, r.az), jz, fz);
        acc0 += trilerp(vol + ((size_t)jz * G.py + jy) * G.px + jx, sy, sz, fx, fy, fz);
    }
    float val = (acc0 + acc1) * (float)G.delta;
    size_t o = ((size_t)(view0 + view) * G.nv + iv) * G.nu + iu;
    sino[o] = accumulate ? sino[o] + val : val;
}

// ---------------------------------------------------------------------------
// A3 matched adjoint, v0: same traversal, 8 RED.ADD.F32 per sample into the
// zeroed padded volume.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(FP_TU *FP_TV)
adjoint_kernel_v0(const float *__restrict__ sino, float *__restrict__ vol, const __grid_constant__ RayGeom G,
                  const __grid_constant__ ViewChunk V, int view0, float scale)
{
    int iu, iv;
    tile_pixel(iu, iv);
    if (iu >= G.nu || iv >= G.nv) return;
    int view = blockIdx.z;
    float yv = sino[((size_t)(view0 + view) * G.nv + iv) * G.nu + iu] * scale;
    if (yv == 0.f) return;
    Ray r = ray_setup(G, V.cs[view].x, V.cs[view].y, iu, iv);
    const int sy = G.px, sz = G.px * G.py;
    float kf = r.kf0;
    for (int it = 0; it < r.n; ++it, kf += 1.0f) {
        int jx, jy, jz;
        float fx, fy, fz;
        cell_frac(fmaf(kf, r.dx, r.ax), jx, fx);
        cell_frac(fmaf(kf, r.dy, r.ay), jy, fy);
        cell_frac(fmaf(kf, r.dz, r.az), jz, fz);
        float *p = vol + ((size_t)jz * G.py + jy) * G.px + jx;
        float wz0 = (1.f - fz) * yv, wz1 = fz * yv;
        float w00 = wz0 * (1.f - fy), w01 = wz0 * fy, w10 = wz1 * (1.f - fy), w11 = wz1 * fy;
        float gx = 1.f - fx;
        atomicAdd(p, w00 * gx);
        atomicAdd(p + 1, w00 * fx);
        atomicAdd(p + sy, w01 * gx);
        atomicAdd(p + sy + 1, w01 * fx);
        atomicAdd(p + sz, w10 * gx);
        atomicAdd(p + sz + 1, w10 * fx);
        atomicAdd(p + sz + sy, w11 * gx);
        atomicAdd(p + sz + sy + 1, w11 * fx);
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
            cell_frac(t - 0.5f, jr, av);
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
static int check_launch(cbct_geom *g, const char *what)
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

int cbct_launch_pad_volume(cbct_geom *g, const RayGeom &r, const float *src, float *dst, int channels,
                           size_t src_channel_stride, int src_z_origin, cudaStream_t st)
{
    size_t n = cbct_padded_volume_elems(r);
    dim3 grid(grid_for(n, 256), 1, channels);
    pad_volume_kernel<<<grid, 256, 0, st>>>(src, dst, r, src_channel_stride, src_z_origin, n);
    return check_launch(g, "pad_volume_kernel");
}

int cbct_launch_unpad_volume(cbct_geom *g, const RayGeom &r, const float *padded, float *dst, int channels,
                             size_t dst_channel_stride, int dst_z_origin, cudaStream_t st)
{
    size_t n = (size_t)r.nx * r.ny * (r.z1 - r.z0);
    dim3 grid(grid_for(n, 256), 1, channels);
    unpad_volume_kernel<<<grid, 256, 0, st>>>(padded, dst, r, cbct_padded_volume_elems(r), dst_channel_stride,
                                              dst_z_origin);
    return check_launch(g, "unpad_volume_kernel");
}

int cbct_launch_pad_sino(cbct_geom *g, const float *src, float *dst, int channels, cudaStream_t st)
{
    int pu = cbct_padded_sino_pitch(g), pv = cbct_padded_sino_rows(g);
    size_t rows = (size_t)channels * g->d.n_views * pv;
    pad_sino_kernel<<<grid_for(rows * pu, 256), 256, 0, st>>>(src, dst, g->d.det_nu, g->d.det_nv, pu, pv, rows);
    return check_launch(g, "pad_sino_kernel");
}

static void fill_chunk(const cbct_geom *g, int view0, int n, ViewChunk &vc)
{
    for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[view0 + i], g->sinphi[view0 + i]);
}

int cbct_launch_fp(cbct_geom *g, const RayGeom &r, const float *padded, float *sino, int channels,
                   int accumulate, cudaStream_t st)
{
    size_t vstride = cbct_padded_volume_elems(r);
    size_t sstride = (size_t)g->d.n_views * r.nv * r.nu;
    ViewChunk vc;  // 8 KB; copied into the launch's parameter buffer at launch time
    for (int view0 = 0; view0 < g->d.n_views; view0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = g->d.n_views - view0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        fill_chunk(g, view0, n, vc);
        dim3 grid((r.nu + FP_TU - 1) / FP_TU, (r.nv + FP_TV - 1) / FP_TV, n);
        for (int c = 0; c < channels; ++c) {
            fp_kernel_v0<<<grid, FP_TU * FP_TV, 0, st>>>(padded + c * vstride, sino + c * sstride, r, vc, view0,
                                                         accumulate);
            int rc = check_launch(g, "fp_kernel_v0");
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}

int cbct_launch_adjoint(cbct_geom *g, const RayGeom &r, const float *sino, float *padded, int channels,
                        cudaStream_t st)
{
    size_t vstride = cbct_padded_volume_elems(r);
    size_t sstride = (size_t)g->d.n_views * r.nv * r.nu;
    ViewChunk vc;
    for (int view0 = 0; view0 < g->d.n_views; view0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = g->d.n_views - view0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        fill_chunk(g, view0, n, vc);
        dim3 grid((r.nu + FP_TU - 1) / FP_TU, (r.nv + FP_TV - 1) / FP_TV, n);
        for (int c = 0; c < channels; ++c) {
            adjoint_kernel_v0<<<grid, FP_TU * FP_TV, 0, st>>>(sino + c * sstride, padded + c * vstride, r, vc,
                                                              view0, (float)r.delta);
            int rc = check_launch(g, "adjoint_kernel_v0");
            if (rc) return rc;
        }
    }
    return CBCT_OK;
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
            int rc = check_launch(g, "fdk_kernel_v0");
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}
