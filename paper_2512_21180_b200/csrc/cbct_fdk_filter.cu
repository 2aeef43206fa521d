// cbct_fdk_filter.cu -- NEXT-1: the projection-domain front end of FDK_w
// (Alg. 1 l.3 "x <- FDK_w(y)"; "projection-domain redundancy weighting
// for offset detector"; "P*(w y)"; Feldkamp ref [9] PAPER.md:397).  Readings R11, R12
// (DESIGN.md s.3):
//     q[c,i,iv,iu] = dphi * a * sum_j h[iu - j] * ( w(u_j) * SDD / sqrt(SDD^2 + u_j^2 + v^2) * p[c,i,iv,j] ),
//     a = du SID / SDD,  h[0] = 1/(4 a^2),  h[odd n] = -1/(pi^2 n^2 a^2),  h[even n] = 0,  dphi = 2 pi / n_views,
// so that cbct_bp_fdk(q) is the FDK_w reconstruction.  w(u) is the smooth sine weighting of a
// laterally displaced detector (1/2 everywhere for a centred one); conjugate rays weigh 1 in total.
//
// One CTA filters one detector row: the weighted row is staged in shared memory between two zero
// aprons (so the convolution needs no bounds test), and every thread accumulates its outputs over
// the odd offsets only.  Tables w[nu] and H[n] = dphi a h[n] are built in fp64 on the host.
#include <math.h>

#include <vector>

#include "cbct_internal.h"

__global__ void __launch_bounds__(256)
fdk_filter_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ tab_w,
                  const float *__restrict__ tab_h, int nu, int nv, size_t n_rows, float u0, float du, float v0,
                  float dv, float sdd)
{
    extern __shared__ float smem[];
    float *row = smem;            // [3 nu]: zeros | weighted row | zeros
    float *taps = smem + 3 * nu;  // [nu]
    for (int j = threadIdx.x; j < nu; j += blockDim.x) {
        row[j] = 0.f;
        row[2 * nu + j] = 0.f;
        taps[j] = tab_h[j];
    }
    for (size_t r = blockIdx.x; r < n_rows; r += gridDim.x) {
        const float v = fmaf((float)(r % nv), dv, v0);
        const float s2 = fmaf(v, v, sdd * sdd);
        __syncthreads();  // previous row fully consumed (and the aprons / taps written)
        for (int j = threadIdx.x; j < nu; j += blockDim.x) {
            const float u = fmaf((float)j, du, u0);
            row[nu + j] = in[r * nu + j] * (tab_w[j] * sdd * rsqrtf(fmaf(u, u, s2)));
        }
        __syncthreads();
        for (int j = threadIdx.x; j < nu; j += blockDim.x) {
            const float *c = row + nu + j;
            float acc0 = taps[0] * c[0], acc1 = 0.f;
            int n = 1;
            for (; n + 2 < nu; n += 4) {
                acc0 = fmaf(taps[n], c[-n] + c[n], acc0);
                acc1 = fmaf(taps[n + 2], c[-n - 2] + c[n + 2], acc1);
            }
            for (; n < nu; n += 2) acc0 = fmaf(taps[n], c[-n] + c[n], acc0);
            out[r * nu + j] = acc0 + acc1;
        }
    }
}

// Register-tiled variant for nu % 8 == 0: a thread owns 8 consecutive outputs, as two interleaved sets of 4
// (even / odd columns).  For a set with outputs j0 + 2i the inputs of tap n+2 are those of tap n shifted by one
// output (c[j0+2i-(n+2)] = c[j0+2(i-1)-n]), so each step loads only one new value on each side and reuses the
// other three from registers: 2 LDS + 1 broadcast tap per 8 multiply-adds instead of 3 per 2.
__global__ void __launch_bounds__(256)
fdk_filter8_kernel(const float *__restrict__ in, float *__restrict__ out, const float *__restrict__ tab_w,
                   const float *__restrict__ tab_h, int nu, int nv, size_t n_rows, float u0, float du, float v0,
                   float dv, float sdd)
{
    extern __shared__ float smem[];
    const int tpr = blockDim.x, rpc = blockDim.y;      // threads per row, rows per CTA
    // zeros | row | zeros; one pad word per 32 (element J sits at J + J/32): a thread's columns are 8 apart,
    // and without the padding lanes t and t + 4 would hit the same bank
    const int span = 3 * nu + 16, base = nu + 8, pitch = span + span / 32 + 1;
    float *taps = smem;                                 // [nu]
    float *rowbuf = smem + nu + (size_t)threadIdx.y * pitch;
#define PADIDX(J) ((J) + ((J) >> 5))
    for (int j = threadIdx.y * tpr + threadIdx.x; j < nu; j += tpr * rpc) taps[j] = tab_h[j];
    for (int j = threadIdx.x; j < pitch; j += tpr) rowbuf[j] = 0.f;
    const float h0 = tab_h[0];
    for (size_t r0 = (size_t)blockIdx.x * rpc; r0 < n_rows; r0 += (size_t)gridDim.x * rpc) {
        const size_t r = r0 + threadIdx.y;
        __syncthreads();  // previous rows consumed; aprons / taps written
        if (r < n_rows) {
            const float v = fmaf((float)(r % nv), dv, v0);
            const float s2 = fmaf(v, v, sdd * sdd);
            for (int j = threadIdx.x; j < nu; j += tpr) {
                const float u = fmaf((float)j, du, u0);
                rowbuf[PADIDX(base + j)] = in[r * nu + j] * (tab_w[j] * sdd * rsqrtf(fmaf(u, u, s2)));
            }
        }
        __syncthreads();
        if (r >= n_rows) continue;
        float res[8];
#pragma unroll
        for (int set = 0; set < 2; ++set) {
            const int c0 = base + 8 * threadIdx.x + set;  // outputs at columns c0, c0 + 2, c0 + 4, c0 + 6
            float acc[4], L[4], R[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                acc[i] = h0 * rowbuf[PADIDX(c0 + 2 * i)];
                L[i] = rowbuf[PADIDX(c0 + 2 * i - 1)];
                R[i] = rowbuf[PADIDX(c0 + 2 * i + 1)];
            }
            for (int n = 1; n < nu; n += 8) {
#pragma unroll
                for (int u4 = 0; u4 < 4; ++u4) {  // tap n + 2 u4; logical L[i] lives in L[(i - u4) & 3], R[i] in R[(i + u4) & 3]
                    const float h = taps[n + 2 * u4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) acc[i] = fmaf(h, L[(i - u4) & 3] + R[(i + u4) & 3], acc[i]);
                    const int jl = c0 - (n + 2 * u4) - 2, jr = c0 + 6 + (n + 2 * u4) + 2;
                    L[(3 - u4) & 3] = rowbuf[PADIDX(jl)];          // new logical L[0] of the next tap
                    R[u4 & 3] = rowbuf[PADIDX(jr)];                // new logical R[3] of the next tap
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) res[2 * i + set] = acc[i];
        }
        float4 *dst = reinterpret_cast<float4 *>(out + r * nu + 8 * threadIdx.x);
        dst[0] = make_float4(res[0], res[1], res[2], res[3]);
        dst[1] = make_float4(res[4], res[5], res[6], res[7]);
    }
#undef PADIDX
}

// out = w(u) * in   (P*(w y); in place allowed)
__global__ void __launch_bounds__(256)
redundancy_weight_kernel(const float *in, float *out, const float *__restrict__ tab_w, int nu,
                         size_t n)
{
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x)
        out[e] = in[e] * tab_w[e % nu];
}

// same, 4 pixels per thread (nu % 4 == 0, 16-byte aligned buffers): the HBM-bound common case
__global__ void __launch_bounds__(256)
redundancy_weight4_kernel(const float4 *in, float4 *out, const float4 *__restrict__ tab_w4, unsigned nu4, size_t n4)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned col = (unsigned)(e % nu4);
    const unsigned dcol = (unsigned)(stride % nu4);
    for (; e < n4; e += stride) {
        float4 v = in[e];
        const float4 w = __ldg(tab_w4 + col);
        v.x *= w.x; v.y *= w.y; v.z *= w.z; v.w *= w.w;
        out[e] = v;
        col += dcol;
        if (col >= nu4) col -= nu4;
    }
}

// ---------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------
// w(u) of reading R12: with the pixel centres covering [u_min, u_max] and tau = min(|u_min|, |u_max|),
// w = 1/2 (sin(pi atan(u/SDD) / (2 atan(tau/SDD))) + 1) inside |u| <= tau, 1 beyond tau on the long
// side; mirrored when the long side is the negative one; 1/2 for a centred detector; 1 when the
// detector lies entirely on one side of the central ray (nothing is measured twice).
static void redundancy_weights(const cbct_geom_desc &d, std::vector<double> &w)
{
    const int nu = d.det_nu;
    w.assign(nu, 0.5);
    const double umin = -0.5 * (nu - 1) * d.det_du_mm + d.det_off_u_mm;
    const double umax = 0.5 * (nu - 1) * d.det_du_mm + d.det_off_u_mm;
    const double big = fmax(fmax(fabs(umin), fabs(umax)), 1.0);
    if (fabs(umin + umax) <= 1e-9 * big) return;                    // centred
    if (umin * umax >= 0.0) { w.assign(nu, nu == 1 ? 0.5 : 1.0); return; }  // one-sided
    const double sgn = umax > -umin ? 1.0 : -1.0;
    const double tau = fmin(-umin, umax);
    const double denom = 2.0 * atan(tau / d.sdd_mm);
    for (int j = 0; j < nu; ++j) {
        const double us = sgn * (umin + j * d.det_du_mm);
        if (us > tau) w[j] = 1.0;
        else if (us < -tau) w[j] = 0.0;
        else w[j] = 0.5 * (sin(M_PI * atan(us / d.sdd_mm) / denom) + 1.0);
    }
}

extern "C" int cbct_geom_redundancy_weights(const cbct_geom *g, double *w_out)
{
    if (!g || !w_out) return CBCT_ERR_INVALID_ARG;
    std::vector<double> w;
    redundancy_weights(g->d, w);
    for (int j = 0; j < g->d.det_nu; ++j) w_out[j] = w[j];
    return CBCT_OK;
}

// device tables: [0, nu) redundancy weights, [nu, 2nu) uniform 1/2, [2nu, 3nu) H[n] = dphi a h[n]
int cbct_ensure_filter_tables(cbct_geom *g)
{
    if (g->d_filter_tab) return CBCT_OK;
    const cbct_geom_desc &d = g->d;
    const int nu = d.det_nu;
    std::vector<double> w;
    redundancy_weights(d, w);
    std::vector<float> tab(3 * (size_t)nu);
    const double a = d.det_du_mm * d.sid_mm / d.sdd_mm, dphi = 2.0 * M_PI / d.n_views;
    for (int j = 0; j < nu; ++j) {
        tab[j] = (float)w[j];
        tab[nu + j] = 0.5f;
        double h = 0.0;
        if (j == 0) h = 1.0 / (4.0 * a * a);
        else if (j & 1) h = -1.0 / (M_PI * M_PI * (double)j * (double)j * a * a);
        tab[2 * (size_t)nu + j] = (float)(dphi * a * h);
    }
    CBCT_CUDA_TRY(cudaMalloc((void **)&g->d_filter_tab, tab.size() * sizeof(float)));
    // synchronous copy from a stack-lifetime vector; happens once per handle
    CBCT_CUDA_TRY(cudaMemcpy(g->d_filter_tab, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice));
    return CBCT_OK;
}

static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

extern "C" int cbct_fdk_filter(const cbct_geom *gc, const float *sino_in, float *sino_out, int32_t channels,
                               int32_t flags, void *stream)
{
    if (!gc || !sino_in || !sino_out || channels < 1 || sino_in == sino_out) return CBCT_ERR_INVALID_ARG;
    cbct_geom *g = const_cast<cbct_geom *>(gc);
    const cbct_geom_desc &d = g->d;
    if (d.det_nu > 2048) return CBCT_ERR_UNSUPPORTED;  // 4 nu floats of shared memory per CTA
    if (!is_device_ptr(sino_in) || !is_device_ptr(sino_out)) return CBCT_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = cbct_ensure_filter_tables(g);
    if (rc) return rc;
    const int nu = d.det_nu;
    const size_t n_rows = (size_t)channels * d.n_views * d.det_nv;
    const float *tw = g->d_filter_tab + ((flags & CBCT_FILTER_REDUNDANCY) ? 0 : nu);
    const size_t smem = 4 * (size_t)nu * sizeof(float);
    const unsigned grid = (unsigned)(n_rows < 148u * 8u ? n_rows : 148u * 8u);
    // coordinates in mm here (the weights only need ratios)
    const float fu0 = (float)(-0.5 * (nu - 1) * d.det_du_mm + d.det_off_u_mm);
    const float fv0 = (float)(-0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm);
    if (nu % 8 == 0 && (uintptr_t)sino_out % 16 == 0) {
        const int tpr = nu / 8, rpc = 256 / tpr < 1 ? 1 : 256 / tpr;
        const int span = 3 * nu + 16;
        const size_t smem8 = ((size_t)nu + (size_t)rpc * (span + span / 32 + 1)) * sizeof(float);
        const size_t want = (n_rows + rpc - 1) / rpc;
        const unsigned grid8 = (unsigned)(want < 148u * 8u ? want : 148u * 8u);
        fdk_filter8_kernel<<<grid8, dim3(tpr, rpc), smem8, st>>>(sino_in, sino_out, tw, g->d_filter_tab + 2 * (size_t)nu, nu,
                                                               d.det_nv, n_rows, fu0, (float)d.det_du_mm, fv0,
                                                                  (float)d.det_dv_mm, (float)d.sdd_mm);
        return cbct_check_launch(g, "fdk_filter8_kernel");
    }
    fdk_filter_kernel<<<grid, 256, smem, st>>>(sino_in, sino_out, tw, g->d_filter_tab + 2 * (size_t)nu, nu, d.det_nv, n_rows,
                                               (float)(-0.5 * (nu - 1) * d.det_du_mm + d.det_off_u_mm),
                                               (float)d.det_du_mm,
                                               (float)(-0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm),
                                               (float)d.det_dv_mm, (float)d.sdd_mm);
    return cbct_check_launch(g, "fdk_filter_kernel");
}

int cbct_launch_redundancy_weight(cbct_geom *g, const float *sino_in, float *sino_out, int channels, cudaStream_t st)
{
    int rc = cbct_ensure_filter_tables(g);
    if (rc) return rc;
    const size_t n = (size_t)channels * g->d.n_views * g->d.det_nv * g->d.det_nu;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148u * 16u) blocks = 148u * 16u;
    if (g->d.det_nu % 4 == 0 && ((uintptr_t)sino_in | (uintptr_t)sino_out) % 16 == 0) {
        blocks = (n / 4 + 255) / 256;
        if (blocks > 148u * 16u) blocks = 148u * 16u;
        redundancy_weight4_kernel<<<(unsigned)blocks, 256, 0, st>>>(
            reinterpret_cast<const float4 *>(sino_in), reinterpret_cast<float4 *>(sino_out),
            reinterpret_cast<const float4 *>(g->d_filter_tab), (unsigned)(g->d.det_nu / 4), n / 4);
    } else {
        redundancy_weight_kernel<<<(unsigned)blocks, 256, 0, st>>>(sino_in, sino_out, g->d_filter_tab, g->d.det_nu, n);
    }
    return cbct_check_launch(g, "redundancy_weight_kernel");
}

extern "C" int cbct_redundancy_weight(const cbct_geom *gc, const float *sino_in, float *sino_out, int32_t channels,
                                      void *stream)
{
    if (!gc || !sino_in || !sino_out || channels < 1) return CBCT_ERR_INVALID_ARG;
    if (!is_device_ptr(sino_in) || !is_device_ptr(sino_out)) return CBCT_ERR_INVALID_ARG;
    return cbct_launch_redundancy_weight(const_cast<cbct_geom *>(gc), sino_in, sino_out, channels, (cudaStream_t)stream);
}
