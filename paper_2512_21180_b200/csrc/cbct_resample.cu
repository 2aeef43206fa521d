// cbct_resample.cu -- NEXT-2: the field-of-view tensor V and the
// resampling operators of the multiscale scheme, Downsample_alpha (average pooling), Upsample (nearest)
// and ProjDown_alpha (drop all but every 1/alpha-th projection + average pooling).
// All are streaming kernels (HBM-bound) except V, which is pure arithmetic (no input array).
#include <math.h>

#include "cbct_internal.h"

// V(p) = #views in which the centre of voxel p projects onto the panel's active area / #views
// (reading R21): -1/2 <= fu < nu - 1/2 and -1/2 <= fv < nv - 1/2, decided in fp64 like the oracle.
struct FovGeom {
    double sid, sdd, x0, y0, z0;       // voxel units; world coordinate of voxel index 0
    double ulo, uhi, vlo, vhi;         // panel edges in detector coordinates (voxel units)
    int nx, ny, nz, n_views;
    float inv_total;
};

__global__ void __launch_bounds__(256)
fov_kernel(float *__restrict__ out, const __grid_constant__ FovGeom G, const __grid_constant__ ViewChunk V, int first,
           int last)
{
    const int ix = blockIdx.x * 32 + (threadIdx.x & 31), iy = blockIdx.y * 8 + (threadIdx.x >> 5), iz = blockIdx.z;
    if (ix >= G.nx || iy >= G.ny) return;
    const double X = G.x0 + ix, Y = G.y0 + iy, Z = G.z0 + iz;
    int count = 0;
    for (int q = 0; q < G.n_views; ++q) {
        const double c = V.cs[q].x, s = V.cs[q].y;
        const double U = G.sid - (X * c + Y * s);
        // u* = sdd w / U within [ulo, uhi)  <=>  sdd w within [ulo U, uhi U)   (U > 0 by validation)
        const double wu = G.sdd * (Y * c - X * s), wv = G.sdd * Z;
        count += (wu >= G.ulo * U) & (wu < G.uhi * U) & (wv >= G.vlo * U) & (wv < G.vhi * U);
    }
    float *dst = out + ((size_t)iz * G.ny + iy) * G.nx + ix;
    float v = (float)count + (first ? 0.f : *dst);
    *dst = last ? v * G.inv_total : v;
}

extern "C" int cbct_fov(const cbct_geom *gc, float *vol_out, void *stream)
{
    if (!gc || !vol_out) return CBCT_ERR_INVALID_ARG;
    cbct_geom *g = const_cast<cbct_geom *>(gc);
    const cbct_geom_desc &d = g->d;
    const double h = d.vox_mm;
    FovGeom G;
    G.sid = d.sid_mm / h; G.sdd = d.sdd_mm / h;
    G.x0 = d.vol_cx_mm / h - 0.5 * (d.vol_nx - 1);
    G.y0 = d.vol_cy_mm / h - 0.5 * (d.vol_ny - 1);
    G.z0 = d.vol_cz_mm / h - 0.5 * (d.vol_nz - 1);
    G.ulo = (-0.5 * d.det_nu * d.det_du_mm + d.det_off_u_mm) / h;
    G.uhi = (0.5 * d.det_nu * d.det_du_mm + d.det_off_u_mm) / h;
    G.vlo = (-0.5 * d.det_nv * d.det_dv_mm + d.det_off_v_mm) / h;
    G.vhi = (0.5 * d.det_nv * d.det_dv_mm + d.det_off_v_mm) / h;
    G.nx = d.vol_nx; G.ny = d.vol_ny; G.nz = d.vol_nz;
    G.inv_total = (float)(1.0 / d.n_views);
    ViewChunk vc;
    dim3 grid((d.vol_nx + 31) / 32, (d.vol_ny + 7) / 8, d.vol_nz);
    for (int q0 = 0; q0 < d.n_views; q0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = d.n_views - q0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[q0 + i], g->sinphi[q0 + i]);
        G.n_views = n;
        fov_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(vol_out, G, vc, q0 == 0, q0 + n == d.n_views);
        int rc = cbct_check_launch(g, "fov_kernel");
        if (rc) return rc;
    }
    return CBCT_OK;
}

// ---------------------------------------------------------------------------
// resampling (no geometry handle: plain array operators)
// ---------------------------------------------------------------------------
// out[o][z][y][x] = mean of the f^3 block of in[o] (in dims: nz f, ny f, nx f)
__global__ void __launch_bounds__(256)
downsample_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_out, int nz, int ny, int nx, int f)
{
    const float inv = 1.0f / (float)(f * f * f);
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_out; e += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(e % nx);
        size_t t = e / nx;
        const int y = (int)(t % ny);
        t /= ny;
        const int z = (int)(t % nz);
        const size_t o = t / nz;
        const float *p = in + (((o * nz + z) * f) * (size_t)(ny * f) + (size_t)y * f) * (size_t)(nx * f) + (size_t)x * f;
        float acc = 0.f;
        for (int k = 0; k < f; ++k)
            for (int j = 0; j < f; ++j)
                for (int i = 0; i < f; ++i) acc += __ldg(p + ((size_t)k * (ny * f) + j) * (size_t)(nx * f) + i);
        out[e] = acc * inv;
    }
}

// out[o][z][y][x] = in[o][z / f][y / f][x / f]   (out dims: nz f, ny f, nx f)
__global__ void __launch_bounds__(256)
upsample_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_out, int nz, int ny, int nx, int f)
{
    const int NX = nx * f, NY = ny * f, NZ = nz * f;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_out; e += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(e % NX);
        size_t t = e / NX;
        const int y = (int)(t % NY);
        t /= NY;
        const int z = (int)(t % NZ);
        const size_t o = t / NZ;
        out[e] = __ldg(in + ((o * nz + z / f) * ny + y / f) * (size_t)nx + x / f);
    }
}

// out[o][i][v][u] = mean of the f^2 block of in[o][i f] (in dims: n_views f', nv f, nu f; views i f kept)
__global__ void __launch_bounds__(256)
proj_down_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_out, int n_views_in, int n_views_out,
                 int nv, int nu, int f)
{
    const float inv = 1.0f / (float)(f * f);
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_out; e += (size_t)gridDim.x * blockDim.x) {
        const int u = (int)(e % nu);
        size_t t = e / nu;
        const int v = (int)(t % nv);
        t /= nv;
        const int i = (int)(t % n_views_out);
        const size_t o = t / n_views_out;
        const float *p = in + ((o * n_views_in + (size_t)i * f) * (size_t)(nv * f) + (size_t)v * f) * (size_t)(nu * f) +
                         (size_t)u * f;
        float acc = 0.f;
        for (int j = 0; j < f; ++j)
            for (int k = 0; k < f; ++k) acc += __ldg(p + (size_t)j * (nu * f) + k);
        out[e] = acc * inv;
    }
}

static unsigned blocks_for(size_t n)
{
    size_t b = (n + 255) / 256;
    return (unsigned)(b < 148u * 16u ? (b ? b : 1) : 148u * 16u);
}

static int finish(const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cbct_set_cuda_error(e, what); return CBCT_ERR_CUDA; }
    return CBCT_OK;
}

extern "C" int cbct_downsample(const float *in, float *out, int64_t n_outer, int32_t nz_in, int32_t ny_in, int32_t nx_in,
                               int32_t factor, void *stream)
{
    if (!in || !out || n_outer < 1 || factor < 1 || nz_in < 1 || ny_in < 1 || nx_in < 1) return CBCT_ERR_INVALID_ARG;
    if (nz_in % factor || ny_in % factor || nx_in % factor) return CBCT_ERR_INVALID_ARG;
    const int nz = nz_in / factor, ny = ny_in / factor, nx = nx_in / factor;
    const size_t n = (size_t)n_outer * nz * ny * nx;
    downsample_kernel<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(in, out, n, nz, ny, nx, factor);
    return finish("downsample_kernel");
}

extern "C" int cbct_upsample(const float *in, float *out, int64_t n_outer, int32_t nz_in, int32_t ny_in, int32_t nx_in,
                             int32_t factor, void *stream)
{
    if (!in || !out || n_outer < 1 || factor < 1 || nz_in < 1 || ny_in < 1 || nx_in < 1) return CBCT_ERR_INVALID_ARG;
    const size_t n = (size_t)n_outer * nz_in * ny_in * nx_in * factor * factor * factor;
    upsample_kernel<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(in, out, n, nz_in, ny_in, nx_in, factor);
    return finish("upsample_kernel");
}

extern "C" int cbct_proj_down(const float *in, float *out, int64_t n_outer, int32_t n_views_in, int32_t nv_in,
                              int32_t nu_in, int32_t factor, void *stream)
{
    if (!in || !out || n_outer < 1 || factor < 1 || n_views_in < 1 || nv_in < 1 || nu_in < 1) return CBCT_ERR_INVALID_ARG;
    if (nv_in % factor || nu_in % factor) return CBCT_ERR_INVALID_ARG;
    const int n_views_out = (n_views_in + factor - 1) / factor, nv = nv_in / factor, nu = nu_in / factor;
    const size_t n = (size_t)n_outer * n_views_out * nv * nu;
    proj_down_kernel<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(in, out, n, n_views_in, n_views_out, nv, nu, factor);
    return finish("proj_down_kernel");
}
