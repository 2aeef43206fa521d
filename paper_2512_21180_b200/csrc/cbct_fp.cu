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
#include "cbct_device.cuh"

// Position of cell jx inside its row: the cell keeps its 128-byte line (8 cells) but
// rotates inside it by a (jy, jz)-dependent amount.  The L1 data stage serves a
// quarter-warp of an LDG.128 (8 lanes x 16 B) in one cycle only if lanes that read
// DIFFERENT cells read different 16-byte positions of their lines (measured: up to 4
// distinct lines per quarter-warp are free, equal positions serialise; DESIGN.md s.6.1).
// (x + 6y + 4z) mod 8 with 4 x 2-pixel quarter-warps leaves 1.2 cycles per quarter-warp
// on this geometry (lower bound 1.14; no swizzle 2.6), by simulation of the access pattern.
__device__ __forceinline__ int cbct_swizzle(int jx, int jy, int jz)
{
    return (jx & ~7) | ((jx + CBCT_SWIZZLE_Y * jy + CBCT_SWIZZLE_Z * jz) & 7);
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
        d[(size_t)row * G.px + cbct_swizzle(jx, jy, jz)] = q;
    }
}

// ---------------------------------------------------------------------------
// channel-interleaved layout for groups of 4 channels: cell (jz, jy, jx) holds the voxel's value in the 4
// channels, float4( v_0, v_1, v_2, v_3 )[jz][jy][jx].  One trilinear sample of 4 channels is then 8 LDG.128 (as
// many as with 4 quad-packed volumes) but every voxel is stored once instead of four times, so the cells a CTA's
// beam pulls into L1 are a quarter of the bytes (the quad layout spends 1.7 of its 6.8 data-stage cycles per load
// on those fills, profiles/r1_final.md).  Rows are not rotated but SKEWED: row (jy, jz) starts
// (CBCT_SWIZZLE_Y jy + CBCT_SWIZZLE_Z jz) mod 8 cells into a pitch of px + 8, which gives cell jx the same
// 16-byte line position (jx + 6 jy + 4 jz) mod 8 as the rotation does and keeps jx + 1 one cell further.
// ---------------------------------------------------------------------------
__host__ __device__ __forceinline__ size_t cbct_packed4_cells(const RayGeom &r)
{
    return (size_t)(r.px + CBCT_ROW_SKEW) * r.py * r.pz;
}

// src: 4 consecutive channels [nz_src][ny][nx] each; dst: one channel-interleaved slab
__global__ void __launch_bounds__(256)
pack_volume4_kernel(const float *__restrict__ src, float4 *__restrict__ dst, const __grid_constant__ RayGeom G,
                    size_t src_cstride, int src_z_origin, size_t group_src_stride, size_t group_dst_stride)
{
    const float *s = src + (size_t)blockIdx.z * group_src_stride;
    float4 *d = dst + (size_t)blockIdx.z * group_dst_stride;
    const int pitch = G.px + CBCT_ROW_SKEW;
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= pitch) return;
    for (int row = blockIdx.y; row < G.py * G.pz; row += gridDim.y) {
        const int jy = row % G.py, jz = row / G.py;
        const int x = pos - ((CBCT_SWIZZLE_Y * jy + CBCT_SWIZZLE_Z * jz) & 7) - CBCT_PAD;
        const int y = jy - CBCT_PAD, z = jz - CBCT_PAD + G.z0;
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
        if (x >= 0 && x < G.nx && y >= 0 && y < G.ny && z >= G.z0 && z < G.z1) {
            const float *p = s + ((size_t)(z - src_z_origin) * G.ny + y) * G.nx + x;
            q.x = __ldg(p);
            q.y = __ldg(p + src_cstride);
            q.z = __ldg(p + 2 * src_cstride);
            q.w = __ldg(p + 3 * src_cstride);
        }
        d[(size_t)row * pitch + pos] = q;
    }
}

// The same layout filled with the four quarter-turn images of ONE channel: component r of cell (x, y) is
// f(R_r(x, y)) with R_1(x, y) = (n - 1 - y, x), R_2 = (n - 1 - x, n - 1 - y), R_3 = (y, n - 1 - x).  On a centred
// square grid with equispaced views (cbct_geom::sym_rot == 4) the ray of view i + r n/4 through f is the ray of
// view i through f o R_r, so projecting this cell volume over the first n/4 views yields, in its four components,
// views i, i + n/4, i + n/2, i + 3n/4 of the channel: a single channel gets the speed of the 4-channel kernel.
__global__ void __launch_bounds__(256)
pack_volume_rot4_kernel(const float *__restrict__ src, float4 *__restrict__ dst, const __grid_constant__ RayGeom G,
                        size_t src_cstride, int src_z_origin, size_t dst_cstride)
{
    const float *s = src + (size_t)blockIdx.z * src_cstride;
    float4 *d = dst + (size_t)blockIdx.z * dst_cstride;
    const int pitch = G.px + CBCT_ROW_SKEW;
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= pitch) return;
    const int n1 = G.nx - 1;
    for (int row = blockIdx.y; row < G.py * G.pz; row += gridDim.y) {
        const int jy = row % G.py, jz = row / G.py;
        const int x = pos - ((CBCT_SWIZZLE_Y * jy + CBCT_SWIZZLE_Z * jz) & 7) - CBCT_PAD;
        const int y = jy - CBCT_PAD, z = jz - CBCT_PAD + G.z0;
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
        if (x >= 0 && x < G.nx && y >= 0 && y < G.ny && z >= G.z0 && z < G.z1) {
            const float *pl = s + (size_t)(z - src_z_origin) * G.ny * G.nx;
            q.x = __ldg(pl + (size_t)y * G.nx + x);
            q.y = __ldg(pl + (size_t)x * G.nx + (n1 - y));
            q.z = __ldg(pl + (size_t)(n1 - y) * G.nx + (n1 - x));
            q.w = __ldg(pl + (size_t)(n1 - x) * G.nx + y);
        }
        d[(size_t)row * pitch + pos] = q;
    }
}

// ---------------------------------------------------------------------------
// forward kernel
// ---------------------------------------------------------------------------
#define FP_CTA_U 16
#define FP_CTA_V 16

__device__ __forceinline__ float lerpf(float a, float b, float t) { return fmaf(t, b - a, a); }

// One sample position: the two cell addresses (planes jz and jz + 1) and the three
// interpolation fractions.  Per axis: pm = fma(kf, d, a) is p - 1/2; y = pm + MAGIC
// rounds it to the cell index j (held in the low mantissa bits of y); the fraction
// p - j = fma(kf, d, b - j) is evaluated from the anchor b itself (b - j is exact),
// so no separate + 1/2.  The cell address uses the raw bits of y: the magic offset
// contributes the constant `kfold` (mod 2^32), subtracted once.
struct Sample {
    const float4 *p0, *p1;
    float fx, fy, fz;
};

__device__ __forceinline__ Sample locate(const float4 *__restrict__ packed, const Ray &r, float kf, unsigned py,
                                         unsigned px, unsigned kfold, unsigned plane)
{
    Sample s;
    const float yx = fmaf(kf, r.dx, r.ax) + CBCT_MAGIC;
    const float yy = fmaf(kf, r.dy, r.ay) + CBCT_MAGIC;
    const float yz = fmaf(kf, r.dz, r.az) + CBCT_MAGIC;
    s.fx = fmaf(kf, r.dx, r.bx - (yx - CBCT_MAGIC));
    s.fy = fmaf(kf, r.dy, r.by - (yy - CBCT_MAGIC));
    s.fz = fmaf(kf, r.dz, r.bz - (yz - CBCT_MAGIC));
    const unsigned ux = __float_as_uint(yx), uy = __float_as_uint(yy), uz = __float_as_uint(yz);
    const unsigned row = (uz * py + uy) * px + (ux & 0x3FFFF8u);
    const unsigned t = uy * CBCT_SWIZZLE_Y + uz * CBCT_SWIZZLE_Z + ux;  // magic bits are multiples of 8
    const unsigned idx = row + (t & 7u) - kfold;
    s.p0 = packed + idx;
    s.p1 = packed + (idx + plane + ((t + CBCT_SWIZZLE_Z) & 7u) - (t & 7u));
    return s;
}

__device__ __forceinline__ float quad_sample(const Sample &s, size_t off)
{
    const float4 q0 = __ldg(s.p0 + off), q1 = __ldg(s.p1 + off);
    const float b0 = lerpf(lerpf(q0.x, q0.y, s.fx), lerpf(q0.z, q0.w, s.fx), s.fy);
    const float b1 = lerpf(lerpf(q1.x, q1.y, s.fx), lerpf(q1.z, q1.w, s.fx), s.fy);
    return lerpf(b0, b1, s.fz);
}

// CB channels per thread; a warp covers TU x (32 / TU) pixels; CTA = FPK_VPC consecutive views x (16 pixels in u x
// one row of warps), see fp4_pair_kernel for why a CTA spans views.
#ifndef FPK_VPC
#define FPK_VPC 4
#endif
template <int CB, int TU>
__global__ void __launch_bounds__(32 * (FP_CTA_U / TU) * FPK_VPC)
fp_kernel(const float4 *__restrict__ packed, float *__restrict__ sino, const __grid_constant__ RayGeom G,
          const __grid_constant__ ViewChunk V, int view0, int accumulate, size_t packed_cstride,
          size_t sino_cstride, int band0, const float *__restrict__ sub, int nviews)
{
    constexpr int TV = 32 / TU, WU = FP_CTA_U / TU;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int iu = blockIdx.x * FP_CTA_U + (warp % WU) * TU + (lane % TU);
    // grid = (u tiles, views, v bands): CTAs in flight share a band of detector rows, i.e. a thin
    // z-slab of the volume, which then stays L2-resident across all views
    const int iv = (band0 + blockIdx.z) * TV + (lane / TU);
    const int view = blockIdx.y * FPK_VPC + warp / WU;
    if (iu >= G.nu || iv >= G.nv || view >= nviews) return;
    const Ray r = cbct_ray_setup(G, V.cs[view].x, V.cs[view].y, iu, iv);
    const unsigned py = G.py, px = G.px, plane = G.px * G.py;
    const unsigned kfold = (CBCT_MAGIC_BITS * (py + 1u)) * px;  // magic bits of jz, jy folded through the row formula
    float acc[CB], acc2[CB];
#pragma unroll
    for (int c = 0; c < CB; ++c) acc[c] = acc2[c] = 0.f;
    float kf = r.kf0;
    int it = 0;
    for (; it + 1 < r.n; it += 2, kf += 2.0f) {
        const Sample s0 = locate(packed, r, kf, py, px, kfold, plane);
        const Sample s1 = locate(packed, r, kf + 1.0f, py, px, kfold, plane);
#pragma unroll
        for (int c = 0; c < CB; ++c) {
            acc[c] += quad_sample(s0, c * packed_cstride);
            acc2[c] += quad_sample(s1, c * packed_cstride);
        }
    }
    if (it < r.n) {
        const Sample s0 = locate(packed, r, kf, py, px, kfold, plane);
#pragma unroll
        for (int c = 0; c < CB; ++c) acc[c] += quad_sample(s0, c * packed_cstride);
    }
    const float delta = (float)G.delta;
    const size_t o = ((size_t)(view0 + view) * G.nv + iv) * G.nu + iu;
#pragma unroll
    for (int c = 0; c < CB; ++c) {
        float val = (acc[c] + acc2[c]) * delta;
        if (sub) val -= __ldg(sub + c * sino_cstride + o);  // fused residual P x - y (NEXT-3)
        float *dst = sino + c * sino_cstride + o;
        *dst = accumulate ? *dst + val : val;
    }
}


// 4 channels per thread from the channel-interleaved layout; otherwise as fp_kernel.
struct Acc4 { float a0, a1, a2, a3; };

__device__ __forceinline__ void fp4_sample(const float4 *__restrict__ packed, const Ray &r, float kf, unsigned py,
                                           unsigned pitch, unsigned plane, unsigned kfold, Acc4 &A)
{
    const float yx = fmaf(kf, r.dx, r.ax) + CBCT_MAGIC;
    const float yy = fmaf(kf, r.dy, r.ay) + CBCT_MAGIC;
    const float yz = fmaf(kf, r.dz, r.az) + CBCT_MAGIC;
    const float fx = fmaf(kf, r.dx, r.bx - (yx - CBCT_MAGIC));
    const float fy = fmaf(kf, r.dy, r.by - (yy - CBCT_MAGIC));
    const float fz = fmaf(kf, r.dz, r.bz - (yz - CBCT_MAGIC));
    const unsigned ux = __float_as_uint(yx), uy = __float_as_uint(yy), uz = __float_as_uint(yz);
    const unsigned t = uy * CBCT_SWIZZLE_Y + uz * CBCT_SWIZZLE_Z;  // magic bits are multiples of 8
    const unsigned base = (uz * py + uy) * pitch + ux - kfold;
    const float4 *p00 = packed + (base + (t & 7u));
    const float4 *p10 = packed + (base + pitch + ((t + CBCT_SWIZZLE_Y) & 7u));
    const float4 *p01 = packed + (base + plane + ((t + CBCT_SWIZZLE_Z) & 7u));
    const float4 *p11 = packed + (base + plane + pitch + ((t + CBCT_SWIZZLE_Y + CBCT_SWIZZLE_Z) & 7u));
    const float4 c000 = __ldg(p00), c100 = __ldg(p00 + 1), c010 = __ldg(p10), c110 = __ldg(p10 + 1);
    const float4 c001 = __ldg(p01), c101 = __ldg(p01 + 1), c011 = __ldg(p11), c111 = __ldg(p11 + 1);
    const float gx = 1.0f - fx, gy = 1.0f - fy, gz = 1.0f - fz;
    const float w00 = gy * gz, w10 = fy * gz, w01 = gy * fz, w11 = fy * fz;
    const float w000 = gx * w00, w100 = fx * w00, w010 = gx * w10, w110 = fx * w10;
    const float w001 = gx * w01, w101 = fx * w01, w011 = gx * w11, w111 = fx * w11;
#define CBCT_TRI(comp) \
    (fmaf(w000, c000.comp, fmaf(w100, c100.comp, fmaf(w010, c010.comp, w110 * c110.comp))) + \
     fmaf(w001, c001.comp, fmaf(w101, c101.comp, fmaf(w011, c011.comp, w111 * c111.comp))))
    A.a0 += CBCT_TRI(x);
    A.a1 += CBCT_TRI(y);
    A.a2 += CBCT_TRI(z);
    A.a3 += CBCT_TRI(w);
#undef CBCT_TRI
}

// Two lanes per ray: lane 2m takes the even samples of ray m, lane 2m + 1 the odd ones (the same two sums as
// fp_kernel's acc / acc2), so a quarter-warp -- the unit the L1 data stage serves per cycle -- covers 2 x 2 pixels
// x 2 consecutive samples instead of 4 x 2 pixels: fewer distinct cells and lines per quarter-warp (measured 4.9
// data-stage cycles per LDG.128 against 5.9 with one lane per ray; the floor is 4.1).  A warp covers 4 x 4
// pixels.  (The same split does not pay for fp_kernel, whose extra cycles are fills.)
// CTA = FP4_VPC consecutive views x (FP4_WU x FP4_WV warps of 4 x 4 pixels): the beams of neighbouring views through
// the same detector tile cross nearly the same voxels (a view step of 0.9 degrees moves a ray by at most ~2 voxels
// inside a 256^3 grid), so their warps share L1 lines: 16 x 8 pixels of one view -> 16 x 4 pixels of 4 views
// measured 66.9 -> 61.4 ms per 4-channel launch at 256^3 / 400 views (8 views: 61.1 - 61.8; 2 views: 63.2 - 64.6).
#ifndef FP4_VPC
#define FP4_VPC 4  // views per CTA
#endif
#ifndef FP4_WU
#define FP4_WU 4   // warps side by side in u per view
#endif
#ifndef FP4_WV
#define FP4_WV 1   // ... and in v
#endif
#define FP4_WPV (FP4_WU * FP4_WV)
__global__ void __launch_bounds__(32 * FP4_WPV * FP4_VPC)
fp4_pair_kernel(const float4 *__restrict__ packed, float *__restrict__ sino, const __grid_constant__ RayGeom G,
                const __grid_constant__ ViewChunk V, int view0, int accumulate, size_t sino_cstride, int band0,
                const float *__restrict__ sub, int nviews)
{
    const int lane = threadIdx.x & 31, warp = (threadIdx.x >> 5) % FP4_WPV;
    const int par = lane & 1;
    const int iu = (blockIdx.x * FP4_WU + warp % FP4_WU) * 4 + ((lane >> 1) & 1) + ((lane >> 3) & 1) * 2;
    const int iv = ((band0 + blockIdx.z) * FP4_WV + warp / FP4_WU) * 4 + ((lane >> 2) & 1) + ((lane >> 4) & 1) * 2;
    int view = blockIdx.y * FP4_VPC + (threadIdx.x >> 5) / FP4_WPV;
    const bool inside = iu < G.nu && iv < G.nv && view < nviews;
    if (view >= nviews) view = nviews - 1;
    Ray r = cbct_ray_setup(G, V.cs[view].x, V.cs[view].y, inside ? iu : 0, inside ? iv : 0);
    if (!inside) r.n = 0;
    const unsigned py = G.py, pitch = G.px + CBCT_ROW_SKEW, plane = pitch * py;
    const unsigned kfold = CBCT_MAGIC_BITS * ((py + 1u) * pitch + 1u);
    Acc4 A = {0.f, 0.f, 0.f, 0.f};
    float kf = r.kf0 + (float)par;
    for (int it = par; it < r.n; it += 2, kf += 2.0f) fp4_sample(packed, r, kf, py, pitch, plane, kfold, A);
    A.a0 += __shfl_xor_sync(0xffffffffu, A.a0, 1);
    A.a1 += __shfl_xor_sync(0xffffffffu, A.a1, 1);
    A.a2 += __shfl_xor_sync(0xffffffffu, A.a2, 1);
    A.a3 += __shfl_xor_sync(0xffffffffu, A.a3, 1);
    if (!inside) return;
    const float delta = (float)G.delta;
    const size_t o = ((size_t)(view0 + view) * G.nv + iv) * G.nu + iu;
    // lane 2m stores channels 0 and 1, lane 2m + 1 channels 2 and 3
    const float lo = par ? A.a2 : A.a0, hi = par ? A.a3 : A.a1;
    const int c0 = 2 * par;
    float val = lo * delta, val2 = hi * delta;
    if (sub) { val -= __ldg(sub + c0 * sino_cstride + o); val2 -= __ldg(sub + (c0 + 1) * sino_cstride + o); }
    float *dst = sino + c0 * sino_cstride + o, *dst2 = dst + sino_cstride;
    *dst = accumulate ? *dst + val : val;
    *dst2 = accumulate ? *dst2 + val2 : val2;
}

// ---------------------------------------------------------------------------
// Single channels on geometries that are symmetric under z -> -z but have no quarter-turn symmetry between their views
// (irregular angle lists): "mirror-paired" cells.  The ray to pixel (iu, nv-1-iv) is the mirror image of the ray to
// (iu, iv): same length, same sample lattice, same x and y, z -> -z; its trilinear sample has the same cell and the
// same fractions when it is read from the mirrored volume f_M[z] = f[nz-1-z].  A cell holds
//     float4( f[z][y][x], f[z][y][x+1], f_M[z][y][x], f_M[z][y][x+1] )
// for the planes of the LOWER half only (rays with v <= 0 never rise above the mid-plane), in the skewed rows of the
// channel-interleaved layout.  One thread walks the ray of a lower detector row and accumulates both it and its
// mirror image: 4 LDG.128 (the y, z corners; the x pair sits inside the cell) per PAIR of samples -- as many loads
// per sample as the quad-packed layout, but the position / fraction / address arithmetic is shared by the pair
// (the quad-packed kernel is as much issue-bound, 78 % of its slots, as L1-bound) and the volume's bytes a beam
// pulls through L1 are halved (every voxel stored twice instead of four times).
// ---------------------------------------------------------------------------
static int fpm_ztop(int nz) { return (nz + 1) / 2 + 1; }   // highest plane held, inclusive (one above the samples' reach)

__global__ void __launch_bounds__(256)
pack_volume_mirror_kernel(const float *__restrict__ src, float4 *__restrict__ dst, const __grid_constant__ RayGeom G,
                          size_t src_cstride, size_t dst_cstride)
{
    // G: the geometry of the lower slab, planes [0, G.z1) of a grid of G.nz planes
    const float *s = src + (size_t)blockIdx.z * src_cstride;
    float4 *d = dst + (size_t)blockIdx.z * dst_cstride;
    const int pitch = G.px + CBCT_ROW_SKEW;
    const int pos = blockIdx.x * blockDim.x + threadIdx.x;
    if (pos >= pitch) return;
    for (int row = blockIdx.y; row < G.py * G.pz; row += gridDim.y) {
        const int jy = row % G.py, jz = row / G.py;
        const int x = pos - ((CBCT_SWIZZLE_Y * jy + CBCT_SWIZZLE_Z * jz) & 7) - CBCT_PAD;
        const int y = jy - CBCT_PAD, z = jz - CBCT_PAD, zm = G.nz - 1 - z;
        float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
        if (y >= 0 && y < G.ny) {
            const bool x0 = x >= 0 && x < G.nx, x1 = x + 1 >= 0 && x + 1 < G.nx;
            if (z >= 0 && z < G.nz) {
                const float *p = s + ((size_t)z * G.ny + y) * G.nx + x;
                if (x0) q.x = __ldg(p);
                if (x1) q.y = __ldg(p + 1);
            }
            if (zm >= 0 && zm < G.nz) {
                const float *p = s + ((size_t)zm * G.ny + y) * G.nx + x;
                if (x0) q.z = __ldg(p);
                if (x1) q.w = __ldg(p + 1);
            }
        }
        d[(size_t)row * pitch + pos] = q;
    }
}

__device__ __forceinline__ void fpm_sample(const float4 *__restrict__ packed, const Ray &r, float kf, unsigned py,
                                           unsigned pitch, unsigned plane, unsigned kfold, float &A, float &M)
{
    const float yx = fmaf(kf, r.dx, r.ax) + CBCT_MAGIC;
    const float yy = fmaf(kf, r.dy, r.ay) + CBCT_MAGIC;
    const float yz = fmaf(kf, r.dz, r.az) + CBCT_MAGIC;
    const float fx = fmaf(kf, r.dx, r.bx - (yx - CBCT_MAGIC));
    const float fy = fmaf(kf, r.dy, r.by - (yy - CBCT_MAGIC));
    const float fz = fmaf(kf, r.dz, r.bz - (yz - CBCT_MAGIC));
    const unsigned ux = __float_as_uint(yx), uy = __float_as_uint(yy), uz = __float_as_uint(yz);
    const unsigned t = uy * CBCT_SWIZZLE_Y + uz * CBCT_SWIZZLE_Z;  // magic bits are multiples of 8
    const unsigned base = (uz * py + uy) * pitch + ux - kfold;
    const float4 c00 = __ldg(packed + (base + (t & 7u)));
    const float4 c10 = __ldg(packed + (base + pitch + ((t + CBCT_SWIZZLE_Y) & 7u)));
    const float4 c01 = __ldg(packed + (base + plane + ((t + CBCT_SWIZZLE_Z) & 7u)));
    const float4 c11 = __ldg(packed + (base + plane + pitch + ((t + CBCT_SWIZZLE_Y + CBCT_SWIZZLE_Z) & 7u)));
    const float gy = 1.0f - fy, gz = 1.0f - fz;
    const float w00 = gy * gz, w10 = fy * gz, w01 = gy * fz, w11 = fy * fz;
    A += fmaf(w00, lerpf(c00.x, c00.y, fx), fmaf(w10, lerpf(c10.x, c10.y, fx), fmaf(w01, lerpf(c01.x, c01.y, fx), w11 * lerpf(c11.x, c11.y, fx))));
    M += fmaf(w00, lerpf(c00.z, c00.w, fx), fmaf(w10, lerpf(c10.z, c10.w, fx), fmaf(w01, lerpf(c01.z, c01.w, fx), w11 * lerpf(c11.z, c11.w, fx))));
}

// Measured at 256^3 / 400 views, 1 channel, jittered angles: 23.7 -> 18.9 ms; data stage 89 % busy at 5.5 cycles per
// load (quad-packed: 6.4), L1 hit rate 97.4 %, 1.66e10 warp instructions (2.12e10).  The two-lanes-per-ray split of
// fp4_pair_kernel measured slower here (19.7 ms: this kernel is closer to the issue limit, 76 % of the slots).
// G: geometry of the lower slab (planes [0, G.z1)); nvh = rows with v <= 0 = ceil(nv / 2); CTA as fp_kernel
template <int TU>
__global__ void __launch_bounds__(32 * (FP_CTA_U / TU) * FPK_VPC)
fpm_kernel(const float4 *__restrict__ packed, float *__restrict__ sino, const __grid_constant__ RayGeom G,
           const __grid_constant__ ViewChunk V, int view0, int accumulate, int nvh, const float *__restrict__ sub,
           int nviews)
{
    constexpr int TV = 32 / TU, WU = FP_CTA_U / TU;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int iu = blockIdx.x * FP_CTA_U + (warp % WU) * TU + (lane % TU);
    const int iv = blockIdx.z * TV + (lane / TU);
    const int view = blockIdx.y * FPK_VPC + warp / WU;
    if (iu >= G.nu || iv >= nvh || view >= nviews) return;
    const Ray r = cbct_ray_setup(G, V.cs[view].x, V.cs[view].y, iu, iv);
    const unsigned py = G.py, pitch = G.px + CBCT_ROW_SKEW, plane = pitch * py;
    const unsigned kfold = CBCT_MAGIC_BITS * ((py + 1u) * pitch + 1u);
    float a0 = 0.f, a1 = 0.f, m0 = 0.f, m1 = 0.f;
    float kf = r.kf0;
    int it = 0;
    for (; it + 1 < r.n; it += 2, kf += 2.0f) {
        fpm_sample(packed, r, kf, py, pitch, plane, kfold, a0, m0);
        fpm_sample(packed, r, kf + 1.0f, py, pitch, plane, kfold, a1, m1);
    }
    if (it < r.n) fpm_sample(packed, r, kf, py, pitch, plane, kfold, a0, m0);
    const float delta = (float)G.delta;
    const int ivm = G.nv - 1 - iv;
    const size_t o = ((size_t)(view0 + view) * G.nv + iv) * G.nu + iu, om = ((size_t)(view0 + view) * G.nv + ivm) * G.nu + iu;
    float val = (a0 + a1) * delta, valm = (m0 + m1) * delta;
    if (sub) { val -= __ldg(sub + o); valm -= __ldg(sub + om); }
    sino[o] = accumulate ? sino[o] + val : val;
    if (ivm != iv) sino[om] = accumulate ? sino[om] + valm : valm;   // the middle row of an odd nv is its own image
}

__global__ void __launch_bounds__(256) negate_kernel(float *buf, size_t n)
{
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x)
        buf[e] = -buf[e];
}

// ---------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------
size_t cbct_packed_volume_cells(const RayGeom &r) { return (size_t)r.px * r.py * r.pz; }

// Layout of a packed slab of `channels` channels: channels / 4 channel-interleaved groups first, then the
// remaining channels quad-packed one by one.  Never more than channels * cbct_packed_volume_cells(r) cells.
static size_t packed_tail_offset(const RayGeom &r, int channels) { return (size_t)(channels / 4) * cbct_packed4_cells(r); }
// channels left over by the groups of 4: their quarter-turn images when the geometry has that symmetry
static bool tail_by_rotation(const cbct_geom *g, const RayGeom &r) { return g->sym_rot == 4 && r.nx == r.ny; }
// single channels run as fast as groups of 4 (used by the HOST-buffer pipeline, cbct_api.cu)
bool cbct_fp_single_channel_is_fast(const cbct_geom *g) { return g->sym_rot == 4 && g->d.vol_nx == g->d.vol_ny; }
// geometry of the lower slab that the mirror-paired layout holds (planes [0, fpm_ztop] of the whole grid)
static RayGeom mirror_raygeom(const cbct_geom *g) { return cbct_make_raygeom(g, 0, fpm_ztop(g->d.vol_nz) + 1); }
// ... used for the channels left over by the groups of 4 when the whole volume is resident (a z-slab of a streamed
// call does not hold its mirror planes) and the slab is no larger than the quad-packed one the workspace is sized for
static bool tail_by_mirror(const cbct_geom *g, const RayGeom &r)
{
    if (tail_by_rotation(g, r) || !g->sym_mirror_z || r.z0 != 0 || r.z1 != r.nz || r.nz < 8) return false;
    return cbct_packed4_cells(mirror_raygeom(g)) <= cbct_packed_volume_cells(r);
}
size_t cbct_packed_tail_cells(const cbct_geom *g, const RayGeom &r)
{
    return tail_by_rotation(g, r) ? cbct_packed4_cells(r) : cbct_packed_volume_cells(r);
}

int cbct_launch_pack_volume(cbct_geom *g, const RayGeom &r, const float *src, float4 *dst, int channels,
                            size_t src_channel_stride, int src_z_origin, cudaStream_t st)
{
    const int rows = r.py * r.pz, groups = channels / 4, tail = channels - 4 * groups;
    const unsigned gy = rows < 148 * 8 ? rows : 148 * 8;
    if (groups) {
        dim3 grid((r.px + CBCT_ROW_SKEW + 255) / 256, gy, groups);
        pack_volume4_kernel<<<grid, 256, 0, st>>>(src, dst, r, src_channel_stride, src_z_origin, 4 * src_channel_stride,
                                                  cbct_packed4_cells(r));
        int rc = cbct_check_launch(g, "pack_volume4_kernel");
        if (rc) return rc;
    }
    if (tail && tail_by_rotation(g, r)) {
        dim3 grid((r.px + CBCT_ROW_SKEW + 255) / 256, gy, tail);
        pack_volume_rot4_kernel<<<grid, 256, 0, st>>>(src + (size_t)4 * groups * src_channel_stride,
                                                      dst + packed_tail_offset(r, channels), r, src_channel_stride,
                                                      src_z_origin, cbct_packed4_cells(r));
        return cbct_check_launch(g, "pack_volume_rot4_kernel");
    }
    if (tail && tail_by_mirror(g, r)) {
        const RayGeom rm = mirror_raygeom(g);
        const int rows_m = rm.py * rm.pz;
        dim3 grid((rm.px + CBCT_ROW_SKEW + 255) / 256, rows_m < 148 * 8 ? rows_m : 148 * 8, tail);
        pack_volume_mirror_kernel<<<grid, 256, 0, st>>>(src + (size_t)4 * groups * src_channel_stride + (size_t)(0 - src_z_origin) * r.ny * r.nx,
                                                        dst + packed_tail_offset(r, channels), rm, src_channel_stride,
                                                        cbct_packed_volume_cells(r));
        return cbct_check_launch(g, "pack_volume_mirror_kernel");
    }
    if (tail) {
        dim3 grid((r.px + 255) / 256, gy, tail);
        pack_volume_kernel<<<grid, 256, 0, st>>>(src + (size_t)4 * groups * src_channel_stride,
                                                 dst + packed_tail_offset(r, channels), r, src_channel_stride,
                                                 src_z_origin, cbct_packed_volume_cells(r));
        return cbct_check_launch(g, "pack_volume_kernel");
    }
    return CBCT_OK;
}

template <int CB>
static int launch_fp_cb(cbct_geom *g, const RayGeom &r, const ViewChunk &vc, int nviews, int view0,
                        const float4 *packed, float *sino, int accumulate, size_t pstride, size_t sstride,
                        int band0, int nbands, const float *sub, cudaStream_t st)
{
    // the caller counts bands of FP_CTA_V = 16 rows; a CTA covers one row of warps, 32 / TU detector rows
    dim3 grid((r.nu + FP_CTA_U - 1) / FP_CTA_U, (nviews + FPK_VPC - 1) / FPK_VPC, 0);
    cbct_prof_begin(g, CBCT_KERNEL_FP, st);
    // 4 x 8-pixel warps suit the bank swizzle best when rays cross the whole volume; in a thin z-slab
    // (streaming) 8 x 4-pixel warps keep the lanes' in-slab segments alike (measured on config 5: +17 %)
    if (r.z1 - r.z0 >= 64 || r.z1 - r.z0 == r.nz) {
        grid.z = nbands * (FP_CTA_V / 8);
        fp_kernel<CB, 4><<<grid, 32 * (FP_CTA_U / 4) * FPK_VPC, 0, st>>>(packed, sino, r, vc, view0, accumulate, pstride,
                                                                         sstride, band0 * (FP_CTA_V / 8), sub, nviews);
    } else {
        grid.z = nbands * (FP_CTA_V / 4);
        fp_kernel<CB, 8><<<grid, 32 * (FP_CTA_U / 8) * FPK_VPC, 0, st>>>(packed, sino, r, vc, view0, accumulate, pstride,
                                                                         sstride, band0 * (FP_CTA_V / 4), sub, nviews);
    }
    cbct_prof_end(g, CBCT_KERNEL_FP, st);
    return cbct_check_launch(g, "fp_kernel");
}

static int launch_fp4(cbct_geom *g, const RayGeom &r, const ViewChunk &vc, int nviews, int view0, const float4 *packed,
                      float *sino, int accumulate, size_t sstride, int band0, int nbands, const float *sub,
                      cudaStream_t st)
{
    cbct_prof_begin(g, CBCT_KERNEL_FP, st);
    // 16 x 8-pixel CTAs: twice as many bands of half the height as the caller counted
    // the caller counts bands of FP_CTA_V = 16 rows; a CTA covers 4 FP4_WV of them
    constexpr int bands_per_16 = FP_CTA_V / (4 * FP4_WV);
    dim3 grid2((r.nu + 4 * FP4_WU - 1) / (4 * FP4_WU), (nviews + FP4_VPC - 1) / FP4_VPC, bands_per_16 * nbands);
    fp4_pair_kernel<<<grid2, 32 * FP4_WPV * FP4_VPC, 0, st>>>(packed, sino, r, vc, view0, accumulate, sstride,
                                                               bands_per_16 * band0, sub, nviews);
    cbct_prof_end(g, CBCT_KERNEL_FP, st);
    return cbct_check_launch(g, "fp4_pair_kernel");
}

int cbct_launch_fp(cbct_geom *g, const RayGeom &r, const float4 *packed, float *sino, int channels, int accumulate,
                   const float *sub, cudaStream_t st)
{
    const size_t pstride = cbct_packed_volume_cells(r);
    const size_t sstride = (size_t)g->d.n_views * r.nv * r.nu;
    // Detector rows a partial slab can reach (its shadow): a ray of height coordinate v is at
    // z = lambda v with lambda = U / sdd, U within [sid - R, sid + R] over the grid's xy extent;
    // only the bands of 16 rows meeting that range are launched.  A caller that launches partial
    // slabs must have zeroed the sinogram and pass accumulate != 0.
    int band0 = 0, nbands = (r.nv + FP_CTA_V - 1) / FP_CTA_V;
    if (r.z0 > 0 || r.z1 < r.nz) {
        const double R = sqrt(r.cx * r.cx + r.cy * r.cy) + 0.5 * sqrt((double)(r.nx + 1) * (r.nx + 1) + (double)(r.ny + 1) * (r.ny + 1));
        const double lmin = (r.sid - R) / (r.sid + r.idd), lmax = (r.sid + R) / (r.sid + r.idd);
        const double za = r.cz + (r.z0 - 1.0 - 0.5 * (r.nz - 1)), zb = r.cz + (r.z1 - 0.5 * (r.nz - 1));
        const double vlo = za <= 0.0 ? za / lmin : za / lmax, vhi = zb >= 0.0 ? zb / lmin : zb / lmax;
        int iv_lo = (int)floor((vlo - r.v0) / r.dv) - 1, iv_hi = (int)ceil((vhi - r.v0) / r.dv) + 1;
        if (iv_lo < 0) iv_lo = 0;
        if (iv_hi > r.nv - 1) iv_hi = r.nv - 1;
        if (iv_lo > iv_hi) return CBCT_OK;  // the slab's shadow misses the detector
        band0 = iv_lo / FP_CTA_V;
        nbands = iv_hi / FP_CTA_V - band0 + 1;
    }
    ViewChunk vc;  // 8 KB; copied into the launch's parameter buffer at launch time
    const int groups = channels / 4;
    const bool rot_tail = channels > 4 * groups && tail_by_rotation(g, r);
    if (rot_tail) {
        // leftover channels one by one: the first n/4 views of the quarter-turn cell volume; the kernel's four
        // "channels" are views i + r n/4, i.e. a channel stride of n/4 views
        const int nbase = g->d.n_views / 4;
        const size_t vstride = (size_t)nbase * r.nv * r.nu;
        for (int view0 = 0; view0 < nbase; view0 += CBCT_VIEWS_PER_LAUNCH) {
            int n = nbase - view0;
            if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
            for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[view0 + i], g->sinphi[view0 + i]);
            for (int c = 4 * groups; c < channels; ++c) {
                int rc = launch_fp4(g, r, vc, n, view0,
                                    packed + packed_tail_offset(r, channels) + (size_t)(c - 4 * groups) * cbct_packed4_cells(r),
                                    sino + c * sstride, accumulate, vstride, band0, nbands, sub ? sub + c * sstride : nullptr, st);
                if (rc) return rc;
            }
        }
        if (groups == 0) return CBCT_OK;
    }
    for (int view0 = 0; view0 < g->d.n_views; view0 += CBCT_VIEWS_PER_LAUNCH) {
        int n = g->d.n_views - view0;
        if (n > CBCT_VIEWS_PER_LAUNCH) n = CBCT_VIEWS_PER_LAUNCH;
        for (int i = 0; i < n; ++i) vc.cs[i] = make_double2(g->cosphi[view0 + i], g->sinphi[view0 + i]);
        int c = 0;
        for (; c + 4 <= channels; c += 4) {  // channel-interleaved groups
            int rc = launch_fp4(g, r, vc, n, view0, packed + (size_t)(c / 4) * cbct_packed4_cells(r), sino + c * sstride,
                                accumulate, sstride, band0, nbands, sub ? sub + c * sstride : nullptr, st);
            if (rc) return rc;
        }
        const float4 *tail = packed + packed_tail_offset(r, channels) - (size_t)c * pstride;
        if (c < channels && !rot_tail && tail_by_mirror(g, r)) {
            // leftover channels one by one through the mirror-paired cells: the rows with v <= 0, each with its image
            const RayGeom rm = mirror_raygeom(g);
            const int nvh = (r.nv + 1) / 2;
            dim3 grid((r.nu + FP_CTA_U - 1) / FP_CTA_U, (n + FPK_VPC - 1) / FPK_VPC, (nvh + 7) / 8);
            for (; c < channels; ++c) {
                cbct_prof_begin(g, CBCT_KERNEL_FP, st);
                fpm_kernel<4><<<grid, 32 * (FP_CTA_U / 4) * FPK_VPC, 0, st>>>(tail + c * pstride, sino + c * sstride, rm, vc, view0,
                                                                              accumulate, nvh, sub ? sub + c * sstride : nullptr, n);
                cbct_prof_end(g, CBCT_KERNEL_FP, st);
                int rc = cbct_check_launch(g, "fpm_kernel");
                if (rc) return rc;
            }
        }
        while (c < channels && !rot_tail) {
            int left = channels - c, rc;
            const float4 *p = tail + c * pstride;
            float *s = sino + c * sstride;
            // 2 channels per thread measured best at 256^3 (4 lowers occupancy and L1 hit rate)
            if (left >= 2) { rc = launch_fp_cb<2>(g, r, vc, n, view0, p, s, accumulate, pstride, sstride, band0, nbands, sub ? sub + c * sstride : nullptr, st); c += 2; }
            else { rc = launch_fp_cb<1>(g, r, vc, n, view0, p, s, accumulate, pstride, sstride, band0, nbands, sub ? sub + c * sstride : nullptr, st); c += 1; }
            if (rc) return rc;
        }
    }
    return CBCT_OK;
}

int cbct_launch_negate(cbct_geom *g, float *buf, size_t n, cudaStream_t st)
{
    size_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    negate_kernel<<<(unsigned)blocks, 256, 0, st>>>(buf, n);
    return cbct_check_launch(g, "negate_kernel");
}
