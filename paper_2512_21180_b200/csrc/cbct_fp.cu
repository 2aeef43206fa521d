// cbct_fp.cu -- A2, the forward projector P (Eq. 5; readings
// R1-R7 in DESIGN.md s.3):
//     sino[c,i,iv,iu] = Delta * sum_k T[vol_c](q(s_i + t_k d)),  t_k = (k + 1/2) Delta.
//
// Design (DESIGN.md s.6; evidence profiles/r1_v0.md): one thread per ray, a warp
// covers a TU x TV patch of detector pixels so that its 32 samples at one k sit
// on a ~4 x 2 voxel patch of the sphere |x - s_i| = t_k.  The v0 kernel (one
// scalar LDG per tap) ran at 92 % of the L1 tag-stage wavefront peak, so the
// volume is first re-laid out ("quad-packed"): cell (jz, jy, jx) holds
//     float4( v[jz][jy][jx], v[jz][jy][jx+1], v[jz][jy+1][jx], v[jz][jy+1][jx+1] )
// and one trilinear sample is two LDG.128 (planes jz and jz+1) instead of eight
// LDG.32.  The packed buffer carries a zero border of CBCT_PAD cells, which
// implements the zero-extension boundary rule R4 with no bounds test in the
// loop.  CB channels share the position / weight arithmetic of a sample.
#include <stdlib.h>

#include "cbct_device.cuh"

// Position of cell jx inside its row: the cell keeps its 128-byte line (8 cells) but
// rotates inside it by a (jy, jz)-dependent amount, so that neighbouring rows and
// planes put the same jx on different L1 data banks (a quarter-warp's LDG.128 reads
// ~5 distinct cells of a 2-D patch; un-swizzled, equal jx in different rows collide).
__device__ __forceinline__ int cbct_swizzle(int jx, int jy, int jz, int swy, int swz)
{
    return (jx & ~7) | ((jx + swy * jy + swz * jz) & 7);
}

// ---------------------------------------------------------------------------
// quad-pack pass: src[C][nz_src][ny][nx] planes [z0, z1) -> packed[C][pz][py][px] float4
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
pack_volume_kernel(const float *__restrict__ src, float4 *__restrict__ dst, const __grid_constant__ RayGeom G,
                   size_t src_cstride, int src_z_origin, size_t dst_cstride)
{
    const float *s = src + (size_t)blockIdx.z * src_cstride;
    float4 *d = dst + (size_t)blockIdx.z * dst_cstride;
    int jx = blockIdx.x * blockDim.x + threadIdx.x;
    if (jx >= G.px) return;
    int x0 = jx - CBCT_PAD, x1 = x0 + 1;
    bool okx0 = x0 >= 0 && x0 < G.nx, okx1 = x1 >= 0 && x1 < G.nx;
    for (int row = blockIdx.y; row < G.py * G.pz; row += gridDim.y) {
        int jy = row % G.py, jz = row / G.py;
        int y0 = jy - CBCT_PAD, y1 = y0 + 1, z = jz - CBCT_PAD + G.z0;
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
        if (z >= G.z0 && z < G.z1) {
            const float *pl = s + (size_t)(z - src_z_origin) * G.ny * G.nx;
            if (y0 >= 0 && y0 < G.ny) {
                const float *r = pl + (size_t)y0 * G.nx;
                if (okx0) q.x = __ldg(r + x0);
                if (okx1) q.y = __ldg(r + x1);
            }
            if (y1 >= 0 && y1 < G.ny) {
                const float *r = pl + (size_t)y1 * G.nx;
                if (okx0) q.z = __ldg(r + x0);
                if (okx1) q.w = __ldg(r + x1);
            }
        }
        d[(size_t)row * G.px + cbct_swizzle(jx, jy, jz, G.swy, G.swz)] = q;
    }
}

// ---------------------------------------------------------------------------
// forward kernel
// ---------------------------------------------------------------------------
#define FP_CTA_U 16
#define FP_CTA_V 16

__device__ __forceinline__ float lerpf(float a, float b, float t) { return fmaf(t, b - a, a); }

__device__ __forceinline__ float quad_sample(const float4 *__restrict__ p0, const float4 *__restrict__ p1, float fx,
                                             float fy, float fz)
{
    float4 q0 = __ldg(p0), q1 = __ldg(p1);
    float b0 = lerpf(lerpf(q0.x, q0.y, fx), lerpf(q0.z, q0.w, fx), fy);
    float b1 = lerpf(lerpf(q1.x, q1.y, fx), lerpf(q1.z, q1.w, fx), fy);
    return lerpf(b0, b1, fz);
}

// Addresses of the cells (jx, jy, jz) and (jx, jy, jz + 1) of the packed slab.
__device__ __forceinline__ void cell_pointers(const float4 *__restrict__ packed, const RayGeom &G, int jx, int jy, int jz,
                                              const float4 *&p0, const float4 *&p1)
{
    const int row = (jz * G.py + jy) * G.px + (jx & ~7);
    const int t = jx + G.swy * jy + G.swz * jz;
    p0 = packed + (row + (t & 7));
    p1 = packed + (row + G.px * G.py + ((t + G.swz) & 7));
}

// CB channels per thread; a warp covers TU x (32 / TU) pixels; CTA = 16 x 16 pixels.
template <int CB, int TU>
__global__ void __launch_bounds__(FP_CTA_U *FP_CTA_V)
fp_kernel(const float4 *__restrict__ packed, float *__restrict__ sino, const __grid_constant__ RayGeom G,
          const __grid_constant__ ViewChunk V, int view0, int accumulate, size_t packed_cstride,
          size_t sino_cstride)
{
    constexpr int TV = 32 / TU, WU = FP_CTA_U / TU;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int iu = blockIdx.x * FP_CTA_U + (warp % WU) * TU + (lane % TU);
    // grid = (u tiles, views, v bands): CTAs in flight share a band of detector rows, i.e. a thin
    // z-slab of the volume, which then stays L2-resident across all views
    const int iv = blockIdx.z * FP_CTA_V + (warp / WU) * TV + (lane / TU);
    if (iu >= G.nu || iv >= G.nv) return;
    const int view = blockIdx.y;
    const Ray r = cbct_ray_setup(G, V.cs[view].x, V.cs[view].y, iu, iv);
    float acc[CB], acc2[CB];
#pragma unroll
    for (int c = 0; c < CB; ++c) acc[c] = acc2[c] = 0.f;
    float kf = r.kf0;
    int it = 0;
    for (; it + 1 < r.n; it += 2, kf += 2.0f) {
        int jx, jy, jz, kx, ky, kz;
        float fx, fy, fz, gx, gy, gz;
        cbct_cell_frac(fmaf(kf, r.dx, r.ax), jx, fx);
        cbct_cell_frac(fmaf(kf, r.dy, r.ay), jy, fy);
        cbct_cell_frac(fmaf(kf, r.dz, r.az), jz, fz);
        const float kg = kf + 1.0f;
        cbct_cell_frac(fmaf(kg, r.dx, r.ax), kx, gx);
        cbct_cell_frac(fmaf(kg, r.dy, r.ay), ky, gy);
        cbct_cell_frac(fmaf(kg, r.dz, r.az), kz, gz);
        const float4 *p0, *p1, *q0, *q1;
        cell_pointers(packed, G, jx, jy, jz, p0, p1);
        cell_pointers(packed, G, kx, ky, kz, q0, q1);
#pragma unroll
        for (int c = 0; c < CB; ++c) {
            acc[c] += quad_sample(p0 + c * packed_cstride, p1 + c * packed_cstride, fx, fy, fz);
            acc2[c] += quad_sample(q0 + c * packed_cstride, q1 + c * packed_cstride, gx, gy, gz);
        }
    }
    if (it < r.n) {
        int jx, jy, jz;
        float fx, fy, fz;
        cbct_cell_frac(fmaf(kf, r.dx, r.ax), jx, fx);
        cbct_cell_frac(fmaf(kf, r.dy, r.ay), jy, fy);
        cbct_cell_frac(fmaf(kf, r.dz, r.az), jz, fz);
        const float4 *p0, *p1;
        cell_pointers(packed, G, jx, jy, jz, p0, p1);
#pragma unroll
        for (int c = 0; c < CB; ++c)
            acc[c] += quad_sample(p0 + c * packed_cstride, p1 + c * packed_cstride, fx, fy, fz);
    }
    const float delta = (float)G.delta;
    const size_t o = ((size_t)(view0 + view) * G.nv + iv) * G.nu + iu;
#pragma unroll
    for (int c = 0; c < CB; ++c) {
        float val = (acc[c] + acc2[c]) * delta;
        float *dst = sino + c * sino_cstride + o;
        *dst = accumulate ? *dst + val : val;
    }
}


// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
size_t cbct_packed_volume_cells(const RayGeom &r) { return (size_t)r.px * r.py * r.pz; }

int cbct_launch_pack_volume(cbct_geom *g, const RayGeom &r, const float *src, float4 *dst, int channels,
                            size_t src_channel_stride, int src_z_origin, cudaStream_t st)
{
    int rows = r.py * r.pz;
    dim3 block(256), grid((r.px + 255) / 256, rows < 148 * 8 ? rows : 148 * 8, channels);
    pack_volume_kernel<<<grid, block, 0, st>>>(src, dst, r, src_channel_stride, src_z_origin,
                                               cbct_packed_volume_cells(r));
    return cbct_check_launch(g, "pack_volume_kernel");
}

template <int CB>
static int launch_fp_cb(cbct_geom *g, const RayGeom &r, const ViewChunk &vc, int nviews, int view0,
                        const float4 *packed, float *sino, int accumulate, size_t pstride, size_t sstride,
                        cudaStream_t st)
{
    dim3 grid((r.nu + FP_CTA_U - 1) / FP_CTA_U, nviews, (r.nv + FP_CTA_V - 1) / FP_CTA_V);
    cbct_prof_begin(g, CBCT_KERNEL_FP, st);
    static const int tu = getenv("CBCT_FP_TU") ? atoi(getenv("CBCT_FP_TU")) : 8;  // TODO(tuning): remove
    if (tu == 4) fp_kernel<CB, 4><<<grid, FP_CTA_U * FP_CTA_V, 0, st>>>(packed, sino, r, vc, view0, accumulate, pstride, sstride);
    else if (tu == 16) fp_kernel<CB, 16><<<grid, FP_CTA_U * FP_CTA_V, 0, st>>>(packed, sino, r, vc, view0, accumulate, pstride, sstride);
    else fp_kernel<CB, 8><<<grid, FP_CTA_U * FP_CTA_V, 0, st>>>(packed, sino, r, vc, view0, accumulate, pstride, sstride);
    cbct_prof_end(g, CBCT_KERNEL_FP, st);
    return cbct_check_launch(g, "fp_kernel");
}

int cbct_launch_fp(cbct_geom *g, const RayGeom &r, const float4 *packed, float *sino, int channels, int accumulate,
                   cudaStream_t st)
{
    const size_t pstride = cbct_packed_volume_cells(r);
    const size_t sstride = (size_t)g->d.n_views * r.nv * r.nu;
    static const int cbmax = getenv("CBCT_FP_CB") ? atoi(getenv("CBCT_FP_CB")) : 4;  // TODO(tuning): remove
    ViewChunk vc;  // 8 KB; copied into the launch's parameter buffer at launch time
    for (int view0 = 0; view0 < g->d.n_views; view0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = g->d.n_views - view0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[view0 + i], g->sinphi[view0 + i]);
        int c = 0;
        while (c < channels) {
            int left = channels - c, rc;
            const float4 *p = packed + c * pstride;
            float *s = sino + c * sstride;
            if (left >= 4 && cbmax >= 4) { rc = launch_fp_cb<4>(g, r, vc, n, view0, p, s, accumulate, pstride, sstride, st); c += 4; }
            else if (left >= 2 && cbmax >= 2) { rc = launch_fp_cb<2>(g, r, vc, n, view0, p, s, accumulate, pstride, sstride, st); c += 2; }
            else { rc = launch_fp_cb<1>(g, r, vc, n, view0, p, s, accumulate, pstride, sstride, st); c += 1; }
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}
