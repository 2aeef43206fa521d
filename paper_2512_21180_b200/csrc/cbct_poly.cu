// cbct_poly.cu -- NEXT-4: the pointwise steps of the polychromatic primary model around the
// forward projector: water-bone decomposition (Eq. 3-4) and the noise-free detector signal
// (Eq. 6).  The projector is linear, so P(mu~_e^w + mu~_e^b) = mu_w(e) P rho_w + mu_b(e) P rho_b:
// two calls of cbct_fp (rho_w, rho_b as two channels) serve every energy bin.  Both kernels are streaming
// (HBM-bound); the attenuation / spectrum tables are the caller's (the paper takes them from xraylib / measured
// beam profiles, which are not part of this library).
#include <math.h>
#include <stdint.h>

#include "cbct_internal.h"

struct WaterBone {
    float tau0, tau1, tau2, kb;
    float w_scale;  // tau1 / (tau2 - tau1)
    float b_scale;  // kb tau2 / (tau2 - tau1)
};

__device__ __forceinline__ void water_bone(float r, const WaterBone &P, float &w, float &b)
{
    // Eq. (3): rho_w;  Eq. (4): rho_b
    w = r < P.tau0 ? 0.f : (r < P.tau1 ? r : (r < P.tau2 ? P.w_scale * (P.tau2 - r) : 0.f));
    b = r < P.tau1 ? 0.f : (r < P.tau2 ? P.b_scale * (r - P.tau1) : P.kb * r);
}

template <bool VEC>
__global__ void __launch_bounds__(256)
water_bone_kernel(const float *__restrict__ rho, float *__restrict__ rw, float *__restrict__ rb, size_t n,
                  const __grid_constant__ WaterBone P)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    if (VEC) {
        const size_t n4 = n >> 2;
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
            const float4 r = __ldcs(reinterpret_cast<const float4 *>(rho) + i);
            float4 w, b;
            water_bone(r.x, P, w.x, b.x); water_bone(r.y, P, w.y, b.y);
            water_bone(r.z, P, w.z, b.z); water_bone(r.w, P, w.w, b.w);
            __stcs(reinterpret_cast<float4 *>(rw) + i, w);
            __stcs(reinterpret_cast<float4 *>(rb) + i, b);
        }
        for (size_t i = (n4 << 2) + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            water_bone(rho[i], P, rw[i], rb[i]);
    } else {
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            water_bone(rho[i], P, rw[i], rb[i]);
    }
}

#define CBCT_MAX_BINS 32
struct PolyTab {
    float aw[CBCT_MAX_BINS], ab[CBCT_MAX_BINS];  // mu_w(e) log2(e), mu_b(e) log2(e)
    float resp[CBCT_MAX_BINS];
    int n_bins;
};

// out[q][p] = sum_e resp_e i0[e][p] 2^-(aw_e pw[q][p] + ab_e pb[q][p]); one thread per 4 detector elements p,
// grid-stride over views q so that a CTA keeps re-reading the same I0 columns (L1 / L2 hits after the first view).
template <bool VEC>
__global__ void __launch_bounds__(256)
poly_primary_kernel(const float *__restrict__ pw, const float *__restrict__ pb, const float *__restrict__ i0,
                    float *__restrict__ out, size_t n_views, size_t n_pix, const __grid_constant__ PolyTab T)
{
    constexpr int W = VEC ? 4 : 1;
    const size_t p = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * W;
    if (p >= n_pix) return;
    for (size_t q = blockIdx.y; q < n_views; q += gridDim.y) {
        float a[W], b[W], acc[W];
        if (VEC) {
            const float4 ta = __ldcs(reinterpret_cast<const float4 *>(pw + q * n_pix + p));
            const float4 tb = __ldcs(reinterpret_cast<const float4 *>(pb + q * n_pix + p));
            a[0] = ta.x; a[1 % W] = ta.y; a[2 % W] = ta.z; a[3 % W] = ta.w;
            b[0] = tb.x; b[1 % W] = tb.y; b[2 % W] = tb.z; b[3 % W] = tb.w;
        } else {
            a[0] = pw[q * n_pix + p];
            b[0] = pb[q * n_pix + p];
        }
#pragma unroll
        for (int j = 0; j < W; ++j) acc[j] = 0.f;
        for (int e = 0; e < T.n_bins; ++e) {
            float w[W];
            if (VEC) {
                const float4 t = __ldg(reinterpret_cast<const float4 *>(i0 + (size_t)e * n_pix + p));
                w[0] = t.x; w[1 % W] = t.y; w[2 % W] = t.z; w[3 % W] = t.w;
            } else {
                w[0] = __ldg(i0 + (size_t)e * n_pix + p);
            }
            const float re = T.resp[e], aw = T.aw[e], ab = T.ab[e];
#pragma unroll
            for (int j = 0; j < W; ++j) acc[j] = fmaf(re * w[j], exp2f(-fmaf(aw, a[j], ab * b[j])), acc[j]);
        }
        if (VEC) __stcs(reinterpret_cast<float4 *>(out + q * n_pix + p), make_float4(acc[0], acc[1 % W], acc[2 % W], acc[3 % W]));
        else out[q * n_pix + p] = acc[0];
    }
}

static int finish(const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cbct_set_cuda_error(e, what); return CBCT_ERR_CUDA; }
    return CBCT_OK;
}

static bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

extern "C" int cbct_water_bone(const float *rho_hat, float *rho_w, float *rho_b, int64_t n, double tau0, double tau1,
                               double tau2, double kappa_b, void *stream)
{
    if (n < 0 || !(tau0 <= tau1) || !(tau1 < tau2)) return CBCT_ERR_INVALID_ARG;
    if (n == 0) return CBCT_OK;
    if (!rho_hat || !rho_w || !rho_b) return CBCT_ERR_INVALID_ARG;
    WaterBone P;
    P.tau0 = (float)tau0; P.tau1 = (float)tau1; P.tau2 = (float)tau2; P.kb = (float)kappa_b;
    P.w_scale = (float)(tau1 / (tau2 - tau1));
    P.b_scale = (float)(kappa_b * tau2 / (tau2 - tau1));
    const bool vec = aligned16(rho_hat) && aligned16(rho_w) && aligned16(rho_b);
    size_t blocks = ((size_t)n / (vec ? 4 : 1) + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    if (blocks < 1) blocks = 1;
    if (vec) water_bone_kernel<true><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(rho_hat, rho_w, rho_b, (size_t)n, P);
    else water_bone_kernel<false><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(rho_hat, rho_w, rho_b, (size_t)n, P);
    return finish("water_bone_kernel");
}

extern "C" int cbct_polychromatic_primary(const float *pw, const float *pb, const float *i0, const double *mu_w,
                                          const double *mu_b, const double *resp, int32_t n_bins, int64_t n_views,
                                          int64_t n_pix, float *out, void *stream)
{
    if (!pw || !pb || !i0 || !mu_w || !mu_b || !resp || !out) return CBCT_ERR_INVALID_ARG;
    if (n_bins < 1 || n_bins > CBCT_MAX_BINS || n_views < 0 || n_pix < 1) return CBCT_ERR_INVALID_ARG;
    if (n_views == 0) return CBCT_OK;
    PolyTab T;
    const double log2e = 1.4426950408889634074;
    for (int e = 0; e < n_bins; ++e) {
        T.aw[e] = (float)(mu_w[e] * log2e);
        T.ab[e] = (float)(mu_b[e] * log2e);
        T.resp[e] = (float)resp[e];
    }
    T.n_bins = n_bins;
    const bool vec = (n_pix % 4 == 0) && aligned16(pw) && aligned16(pb) && aligned16(i0) && aligned16(out);
    const size_t threads = (size_t)n_pix / (vec ? 4 : 1);
    const unsigned gx = (unsigned)((threads + 255) / 256);
    // enough CTAs to fill the GPU several times over while each thread still reuses its I0 column over views
    size_t gy = (148u * 16u + gx - 1) / gx;
    if (gy > (size_t)n_views) gy = (size_t)n_views;
    if (gy > 65535) gy = 65535;
    dim3 grid(gx, (unsigned)gy);
    if (vec) poly_primary_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>(pw, pb, i0, out, (size_t)n_views, (size_t)n_pix, T);
    else poly_primary_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>(pw, pb, i0, out, (size_t)n_views, (size_t)n_pix, T);
    return finish("poly_primary_kernel");
}
