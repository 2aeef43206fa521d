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
// Row-oriented streaming kernels: a CTA of 64 x 4 threads takes 4 output rows at a time (grid-stride over
// rows, so the only integer divisions are per row), threads run along x with vector loads / stores so that
// every 32-byte sector moved is fully used.  F = pooling factor (2 and 4 vectorised; 0 = any factor, scalar).
template <int F> struct VecOf { typedef float type; };
template <> struct VecOf<2> { typedef float2 type; };
template <> struct VecOf<4> { typedef float4 type; };
__device__ __forceinline__ float hsum(float v) { return v; }
__device__ __forceinline__ float hsum(float2 v) { return v.x + v.y; }
__device__ __forceinline__ float hsum(float4 v) { return (v.x + v.y) + (v.z + v.w); }

// sum over an F-wide run of `rows` input rows spaced `pitch` floats apart, starting at p
template <int F>
__device__ __forceinline__ float pool_rows(const float *__restrict__ p, int f, size_t pitch, int rows)
{
    float acc = 0.f;
    if (F == 0) {
        for (int j = 0; j < rows; ++j)
            for (int i = 0; i < f; ++i) acc += __ldg(p + j * pitch + i);
    } else {
        typedef typename VecOf<F>::type V;
#pragma unroll
        for (int j = 0; j < F; ++j) acc += hsum(__ldg(reinterpret_cast<const V *>(p + j * pitch)));
    }
    return acc;
}

// out[o][z][y][x] = mean of the f^3 block of in[o] (in dims: nz f, ny f, nx f)
template <int F>
__global__ void __launch_bounds__(256)
downsample_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_rows, int nz, int ny, int nx, int f)
{
    const float inv = 1.0f / (float)(f * f * f);
    const size_t in_pitch = (size_t)nx * f, in_plane = in_pitch * ny * f;
    for (size_t r = (size_t)blockIdx.x * blockDim.y + threadIdx.y; r < n_rows; r += (size_t)gridDim.x * blockDim.y) {
        const int y = (int)(r % ny);
        const size_t oz = r / ny;  // o * nz + z
        const float *src = in + (oz * f) * in_plane + (size_t)y * f * in_pitch;
        for (int x = threadIdx.x; x < nx; x += blockDim.x) {
            float acc = 0.f;
            for (int k = 0; k < f; ++k) acc += pool_rows<F>(src + k * in_plane + (size_t)x * f, f, in_pitch, f);
            out[r * nx + x] = acc * inv;
        }
    }
}

// out[o][z][y][x] = in[o][z / f][y / f][x / f]   (out dims: nz f, ny f, nx f).  A thread expands its piece of one
// INPUT row into the f x f output rows it feeds (4 outputs per store when the row length allows).
__global__ void __launch_bounds__(256)
upsample_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_rows, int nz, int ny, int nx, int f,
                int vec4)
{
    const int NX = nx * f;
    const size_t out_pitch = (size_t)NX, out_plane = out_pitch * ny * f;
    for (size_t r = (size_t)blockIdx.x * blockDim.y + threadIdx.y; r < n_rows; r += (size_t)gridDim.x * blockDim.y) {
        const int y = (int)(r % ny);
        const size_t oz = r / ny;  // o * nz + z
        const float *src = in + r * nx;
        float *dst = out + (oz * f) * out_plane + (size_t)y * f * out_pitch;
        if (vec4) {
            for (int x = threadIdx.x * 4; x < NX; x += blockDim.x * 4) {
                const float4 v = make_float4(__ldg(src + x / f), __ldg(src + (x + 1) / f), __ldg(src + (x + 2) / f),
                                             __ldg(src + (x + 3) / f));
                for (int k = 0; k < f; ++k)
                    for (int j = 0; j < f; ++j) *reinterpret_cast<float4 *>(dst + k * out_plane + j * out_pitch + x) = v;
            }
        } else {
            for (int x = threadIdx.x; x < NX; x += blockDim.x) {
                const float v = __ldg(src + x / f);
                for (int k = 0; k < f; ++k)
                    for (int j = 0; j < f; ++j) dst[k * out_plane + j * out_pitch + x] = v;
            }
        }
    }
}

// out[o][i][v][u] = mean of the f^2 block of in[o][i f] (in dims: n_views_in, nv f, nu f; views i f kept)
template <int F>
__global__ void __launch_bounds__(256)
proj_down_kernel(const float *__restrict__ in, float *__restrict__ out, size_t n_rows, int n_views_in, int n_views_out,
                 int nv, int nu, int f)
{
    const float inv = 1.0f / (float)(f * f);
    const size_t in_pitch = (size_t)nu * f, in_img = in_pitch * nv * f;
    for (size_t r = (size_t)blockIdx.x * blockDim.y + threadIdx.y; r < n_rows; r += (size_t)gridDim.x * blockDim.y) {
        const int v = (int)(r % nv);
        const size_t oi = r / nv;
        const int i = (int)(oi % n_views_out);
        const size_t o = oi / n_views_out;
        const float *src = in + (o * n_views_in + (size_t)i * f) * in_img + (size_t)v * f * in_pitch;
        for (int u = threadIdx.x; u < nu; u += blockDim.x)
            out[r * nu + u] = pool_rows<F>(src + (size_t)u * f, f, in_pitch, f) * inv;
    }
}

static unsigned row_blocks(size_t rows)
{
    size_t b = (rows + 3) / 4;
    return (unsigned)(b < 148u * 32u ? (b ? b : 1) : 148u * 32u);
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
    const size_t rows = (size_t)n_outer * nz * ny;
    const bool al = ((uintptr_t)in % 16 == 0);
    const dim3 block(64, 4);
    if (factor == 2 && al) downsample_kernel<2><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, nz, ny, nx, 2);
    else if (factor == 4 && al) downsample_kernel<4><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, nz, ny, nx, 4);
    else downsample_kernel<0><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, nz, ny, nx, factor);
    return finish("downsample_kernel");
}

extern "C" int cbct_upsample(const float *in, float *out, int64_t n_outer, int32_t nz_in, int32_t ny_in, int32_t nx_in,
                             int32_t factor, void *stream)
{
    if (!in || !out || n_outer < 1 || factor < 1 || nz_in < 1 || ny_in < 1 || nx_in < 1) return CBCT_ERR_INVALID_ARG;
    const size_t rows = (size_t)n_outer * nz_in * ny_in;
    const int vec4 = ((nx_in * factor) % 4 == 0) && ((uintptr_t)out % 16 == 0);
    upsample_kernel<<<row_blocks(rows), dim3(64, 4), 0, (cudaStream_t)stream>>>(in, out, rows, nz_in, ny_in, nx_in, factor, vec4);
    return finish("upsample_kernel");
}

extern "C" int cbct_proj_down(const float *in, float *out, int64_t n_outer, int32_t n_views_in, int32_t nv_in,
                              int32_t nu_in, int32_t factor, void *stream)
{
    if (!in || !out || n_outer < 1 || factor < 1 || n_views_in < 1 || nv_in < 1 || nu_in < 1) return CBCT_ERR_INVALID_ARG;
    if (nv_in % factor || nu_in % factor) return CBCT_ERR_INVALID_ARG;
    const int n_views_out = (n_views_in + factor - 1) / factor, nv = nv_in / factor, nu = nu_in / factor;
    const size_t rows = (size_t)n_outer * n_views_out * nv;
    const bool al = ((uintptr_t)in % 16 == 0);
    const dim3 block(64, 4);
    if (factor == 2 && al) proj_down_kernel<2><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, n_views_in, n_views_out, nv, nu, 2);
    else if (factor == 4 && al) proj_down_kernel<4><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, n_views_in, n_views_out, nv, nu, 4);
    else proj_down_kernel<0><<<row_blocks(rows), block, 0, (cudaStream_t)stream>>>(in, out, rows, n_views_in, n_views_out, nv, nu, factor);
    return finish("proj_down_kernel");
}
