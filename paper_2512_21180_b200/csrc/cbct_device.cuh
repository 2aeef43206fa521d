// cbct_device.cuh -- device helpers shared by the forward projector (A2) and
// the kernels that must reproduce its sample lattice (product code only).
//
// Sample lattice (reading R3, DESIGN.md s.3): t_k = (k + 1/2) * step measured
// from the SOURCE along the unit direction source -> pixel centre
// (Eq. 5 discretised as BASELINE.json states).
#pragma once
#include <math.h>

#include "cbct_internal.h"

#define CBCT_MAGIC 12582912.0f  // 1.5 * 2^23: x + MAGIC rounds x to the nearest integer
#define CBCT_MAGIC_BITS 0x4B400000

// Per-ray state of the forward traversal: every quantity is computed in fp64
// and rounded once to fp32; the sample loop evaluates
//     p_k - 1/2 = fma(kf, d, a),  kf = kf0, kf0 + 1, ...
// about an anchor in the MIDDLE of the in-support range, so |kf * d| <= ~N/2
// and no error accumulates along the ray (DESIGN.md s.6, precision plan).
struct Ray {
    float ax, ay, az;  // anchor sample position minus 1/2, padded index coordinates
    float bx, by, bz;  // anchor sample position itself (rounded separately from fp64)
    float dx, dy, dz;  // position increment per sample
    float kf0;         // first sample index relative to the anchor
    int n;             // number of samples to visit (0 = ray misses the slab)
};

__device__ __forceinline__ void cbct_clip_axis(double o, double d, double lo, double hi, double &tmin,
                                               double &tmax, bool &hit)
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

// (c, s) = (cos phi, sin phi) of the view; (iu, iv) the detector pixel.
__device__ __forceinline__ Ray cbct_ray_setup(const RayGeom &G, double c, double s, int iu, int iv)
{
    Ray r;
    double u = G.u0 + iu * G.du, v = G.v0 + iv * G.dv;
    // D = pixel - source = -(SID + IDD)(c, s, 0) + u (-s, c, 0) + v (0, 0, 1)
    double sdd = G.sid + G.idd;
    double Dx = -sdd * c - u * s, Dy = -sdd * s + u * c, Dz = v;
    double L = sqrt(Dx * Dx + Dy * Dy + Dz * Dz);
    double invL = 1.0 / L;
    double dx = Dx * invL, dy = Dy * invL, dz = Dz * invL;
    // source in padded index coordinates of the slab
    double ox = G.sid * c - G.cx + 0.5 * (G.nx - 1) + CBCT_PAD;
    double oy = G.sid * s - G.cy + 0.5 * (G.ny - 1) + CBCT_PAD;
    double oz = -G.cz + 0.5 * (G.nz - 1) + CBCT_PAD - G.z0;
    double tmin = 0.0, tmax = L;
    bool hit = true;
    cbct_clip_axis(ox, dx, CBCT_PAD - 1.0, CBCT_PAD + (double)G.nx, tmin, tmax, hit);
    cbct_clip_axis(oy, dy, CBCT_PAD - 1.0, CBCT_PAD + (double)G.ny, tmin, tmax, hit);
    cbct_clip_axis(oz, dz, CBCT_PAD - 1.0, CBCT_PAD + (double)(G.z1 - G.z0), tmin, tmax, hit);
    r.n = 0;
    r.ax = r.ay = r.az = 1.f;
    r.bx = r.by = r.bz = 1.5f;
    r.dx = r.dy = r.dz = 0.f;
    r.kf0 = 0.f;
    if (!hit || !(tmin < tmax)) return r;
    double inv_step = 1.0 / G.step;
    long k0 = (long)ceil(tmin * inv_step - 0.5);   // first k with t_k >= tmin
    long k1 = (long)floor(tmax * inv_step - 0.5);  // last  k with t_k <= tmax
    if (k0 < 0) k0 = 0;
    if (k1 < k0) return r;
    long km = k0 + ((k1 - k0) >> 1);
    double tm = ((double)km + 0.5) * G.step;
    r.ax = (float)(ox + tm * dx - 0.5);
    r.ay = (float)(oy + tm * dy - 0.5);
    r.az = (float)(oz + tm * dz - 0.5);
    r.bx = (float)(ox + tm * dx);
    r.by = (float)(oy + tm * dy);
    r.bz = (float)(oz + tm * dz);
    r.dx = (float)(G.step * dx);
    r.dy = (float)(G.step * dy);
    r.dz = (float)(G.step * dz);
    r.kf0 = (float)(k0 - km);
    r.n = (int)(k1 - k0 + 1);
    return r;
}

// Cell index and fractional offset from pm = p - 1/2 (round-to-nearest trick):
// any integer j with p - j in [0, 1] gives the same trilinear value, so ties
// and the last-ulp rounding of pm are harmless.
__device__ __forceinline__ void cbct_cell_frac(float pm, int &j, float &a)
{
    float y = pm + CBCT_MAGIC;
    j = __float_as_int(y) - CBCT_MAGIC_BITS;
    a = (pm - (y - CBCT_MAGIC)) + 0.5f;
}

// ---------------------------------------------------------------------------
// Views related by a rotation of the grid (cbct_geom::sym_rot = NR) are stored
// side by side by the backprojectors' re-layout passes: component p of a pixel
// of "base view" ib < n/NR is view ib + p n/NR, so one vector load fetches the
// pixel for all NR rotated copies of a voxel.
// ---------------------------------------------------------------------------
template <int NR>
__device__ __forceinline__ void load_views(const float *__restrict__ p, float (&y)[NR])
{
    if (NR == 4) {
        float4 t = __ldg(reinterpret_cast<const float4 *>(p));
        y[0] = t.x; y[1] = t.y; y[2] = t.z; y[NR - 1] = t.w;
    } else if (NR == 2) {
        float2 t = __ldg(reinterpret_cast<const float2 *>(p));
        y[0] = t.x; y[NR - 1] = t.y;
    } else {
        y[0] = __ldg(p);
    }
}

__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ float rsqrt_approx(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// y[r] <- y[(a + r) mod NR]  (a is uniform over the CTA: no divergence)
template <int NR>
__device__ __forceinline__ void rotate_views(float (&y)[NR], int a)
{
    if (NR == 2) {
        if (a & 1) { float t = y[0]; y[0] = y[NR - 1]; y[NR - 1] = t; }
    } else if (NR == 4) {
        if (a & 1) { float t = y[0]; y[0] = y[1]; y[1] = y[2]; y[2] = y[NR - 1]; y[NR - 1] = t; }
        if (a & 2) { float t = y[0]; y[0] = y[2]; y[2] = t; t = y[1]; y[1] = y[NR - 1]; y[NR - 1] = t; }
    }
}

