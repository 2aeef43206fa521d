// cbct_api.cu -- C ABI entry points of libcbct.so (include/cbct.h): pointer
// classification, device workspace, host staging and the z-slab streaming
// driver (A5; exact by linearity: P f = sum_s P(f 1_slab_s), and (P^T y)|slab,
// FDK|slab are independent per slab because the sample lattice is anchored at
// the source, reading R3).  PAPER.md:165, :292 motivate the streaming.
#include <string.h>

#include "cbct_internal.h"

enum MemKind { MEM_DEVICE = 0, MEM_HOST_PINNED = 1, MEM_HOST_PAGEABLE = 2 };

static MemKind classify(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return MEM_HOST_PAGEABLE; }
    switch (a.type) {
        case cudaMemoryTypeDevice:
        case cudaMemoryTypeManaged: return MEM_DEVICE;
        case cudaMemoryTypeHost: return MEM_HOST_PINNED;
        default: return MEM_HOST_PAGEABLE;
    }
}

static int ensure(float **p, size_t *have, size_t need)
{
    if (*have >= need) return CBCT_OK;
    if (*p) { cudaDeviceSynchronize(); cudaFree(*p); *p = nullptr; *have = 0; }
    cudaError_t e = cudaMalloc((void **)p, need);
    if (e != cudaSuccess) { cbct_set_cuda_error(e, "cudaMalloc(workspace)"); *p = nullptr; return CBCT_ERR_NOMEM; }
    *have = need;
    return CBCT_OK;
}

static int ensure_streams(cbct_geom *g)
{
    if (!g->copy_stream) CBCT_CUDA_TRY(cudaStreamCreateWithFlags(&g->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 4; ++i)
        if (!g->ev[i]) CBCT_CUDA_TRY(cudaEventCreateWithFlags(&g->ev[i], cudaEventDisableTiming));
    return CBCT_OK;
}

static int have_device(void)
{
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n < 1) {
        cbct_set_cuda_error(e != cudaSuccess ? e : cudaErrorNoDevice, "cudaGetDeviceCount");
        return CBCT_ERR_CUDA;
    }
    return CBCT_OK;
}

// Copy planes [z0,z1) of a HOST volume (all channels) into the interior of a
// zeroed padded device buffer: one pitched 3-D copy per channel.
static int h2d_slab(const RayGeom &r, const float *host, float *padded, int channels, size_t host_cstride,
                    cudaStream_t st)
{
    size_t pelems = cbct_padded_volume_elems(r);
    CBCT_CUDA_TRY(cudaMemsetAsync(padded, 0, pelems * channels * sizeof(float), st));
    for (int c = 0; c < channels; ++c) {
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof(p));
        p.srcPtr = make_cudaPitchedPtr((void *)(host + c * host_cstride + (size_t)r.z0 * r.ny * r.nx),
                                       r.nx * sizeof(float), r.nx, r.ny);
        p.dstPtr = make_cudaPitchedPtr((void *)(padded + c * pelems), r.px * sizeof(float), r.px, r.py);
        p.dstPos = make_cudaPos(CBCT_PAD * sizeof(float), CBCT_PAD, CBCT_PAD);
        p.extent = make_cudaExtent(r.nx * sizeof(float), r.ny, r.z1 - r.z0);
        p.kind = cudaMemcpyHostToDevice;
        CBCT_CUDA_TRY(cudaMemcpy3DAsync(&p, st));
    }
    return CBCT_OK;
}

// Copy the interior of a padded device slab to planes [z0,z1) of a HOST volume.
static int d2h_slab(const RayGeom &r, const float *padded, float *host, int channels, size_t host_cstride,
                    cudaStream_t st)
{
    size_t pelems = cbct_padded_volume_elems(r);
    for (int c = 0; c < channels; ++c) {
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof(p));
        p.srcPtr = make_cudaPitchedPtr((void *)(padded + c * pelems), r.px * sizeof(float), r.px, r.py);
        p.srcPos = make_cudaPos(CBCT_PAD * sizeof(float), CBCT_PAD, CBCT_PAD);
        p.dstPtr = make_cudaPitchedPtr((void *)(host + c * host_cstride + (size_t)r.z0 * r.ny * r.nx),
                                       r.nx * sizeof(float), r.nx, r.ny);
        p.extent = make_cudaExtent(r.nx * sizeof(float), r.ny, r.z1 - r.z0);
        p.kind = cudaMemcpyDeviceToHost;
        CBCT_CUDA_TRY(cudaMemcpy3DAsync(&p, st));
    }
    return CBCT_OK;
}

struct CallCtx {
    cbct_geom *g;
    cudaStream_t st;
    int channels;
    size_t nvol, nsino;   // elements per channel
    int planes, n_slabs;
    bool pageable;
};

static int begin_call(const cbct_geom *gc, const void *a, const void *b, int32_t channels, void *stream,
                      CallCtx &cx)
{
    if (!gc || !a || !b || channels < 1) return CBCT_ERR_INVALID_ARG;
    int rc = have_device();
    if (rc) return rc;
    cx.g = const_cast<cbct_geom *>(gc);
    cx.st = (cudaStream_t)stream;
    cx.channels = channels;
    cx.nvol = (size_t)gc->d.vol_nx * gc->d.vol_ny * gc->d.vol_nz;
    cx.nsino = (size_t)gc->d.n_views * gc->d.det_nv * gc->d.det_nu;
    cx.planes = cbct_plan_slab_planes(gc, channels);
    if (cx.planes < 1) return CBCT_ERR_NOMEM;
    cx.n_slabs = (gc->d.vol_nz + cx.planes - 1) / cx.planes;
    cx.pageable = false;
    return ensure_streams(cx.g);
}

// ---------------------------------------------------------------------------
extern "C" int cbct_fp(const cbct_geom *gc, const float *vol, float *sino, int32_t channels, void *stream)
{
    CallCtx cx;
    int rc = begin_call(gc, vol, sino, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    MemKind kv = classify(vol), ks = classify(sino);
    cx.pageable = (kv == MEM_HOST_PAGEABLE) || (ks == MEM_HOST_PAGEABLE);

    float *d_sino = sino;
    if (ks != MEM_DEVICE) {
        rc = ensure(&g->ws_sino, &g->ws_sino_bytes, cx.nsino * channels * sizeof(float));
        if (rc) return rc;
        d_sino = g->ws_sino;
    }
    RayGeom rmax = cbct_make_raygeom(g, 0, cx.planes);
    size_t slab_elems = cbct_padded_volume_elems(rmax) * channels;
    int nbuf = cx.n_slabs > 1 ? 2 : 1;
    rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_elems * nbuf * sizeof(float));
    if (rc) return rc;

    if (cx.n_slabs == 1) {
        RayGeom r = cbct_make_raygeom(g, 0, g->d.vol_nz);
        if (kv == MEM_DEVICE) rc = cbct_launch_pad_volume(g, r, vol, g->ws_vol, channels, cx.nvol, 0, st);
        else rc = h2d_slab(r, vol, g->ws_vol, channels, cx.nvol, st);
        if (rc) return rc;
        rc = cbct_launch_fp(g, r, g->ws_vol, d_sino, channels, 0, st);
        if (rc) return rc;
    } else {
        // double-buffered slabs: copy stream fills buffer b while `st` projects the other
        CBCT_CUDA_TRY(cudaEventRecord(g->ev[0], st));
        CBCT_CUDA_TRY(cudaStreamWaitEvent(g->copy_stream, g->ev[0], 0));
        for (int s = 0; s < cx.n_slabs; ++s) {
            int b = s & 1;
            int z0 = s * cx.planes, z1 = z0 + cx.planes < g->d.vol_nz ? z0 + cx.planes : g->d.vol_nz;
            RayGeom r = cbct_make_raygeom(g, z0, z1);
            float *buf = g->ws_vol + (size_t)b * slab_elems;
            if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(g->copy_stream, g->ev[2 + b], 0));
            if (kv == MEM_DEVICE) rc = cbct_launch_pad_volume(g, r, vol, buf, channels, cx.nvol, 0, g->copy_stream);
            else rc = h2d_slab(r, vol, buf, channels, cx.nvol, g->copy_stream);
            if (rc) return rc;
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], g->copy_stream));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));
            rc = cbct_launch_fp(g, r, buf, d_sino, channels, s > 0, st);
            if (rc) return rc;
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
        }
    }
    if (ks != MEM_DEVICE)
        CBCT_CUDA_TRY(cudaMemcpyAsync(sino, d_sino, cx.nsino * channels * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

// ---------------------------------------------------------------------------
extern "C" int cbct_bp_adjoint(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream)
{
    CallCtx cx;
    int rc = begin_call(gc, sino, vol, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    MemKind kv = classify(vol), ks = classify(sino);
    cx.pageable = (kv == MEM_HOST_PAGEABLE) || (ks == MEM_HOST_PAGEABLE);

    const float *d_sino = sino;
    if (ks != MEM_DEVICE) {
        rc = ensure(&g->ws_sino, &g->ws_sino_bytes, cx.nsino * channels * sizeof(float));
        if (rc) return rc;
        CBCT_CUDA_TRY(cudaMemcpyAsync(g->ws_sino, sino, cx.nsino * channels * sizeof(float), cudaMemcpyHostToDevice, st));
        d_sino = g->ws_sino;
    }
    RayGeom rmax = cbct_make_raygeom(g, 0, cx.planes);
    size_t slab_elems = cbct_padded_volume_elems(rmax) * channels;
    int nbuf = cx.n_slabs > 1 ? 2 : 1;
    rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_elems * nbuf * sizeof(float));
    if (rc) return rc;

    for (int s = 0; s < cx.n_slabs; ++s) {
        int b = s & 1;
        int z0 = s * cx.planes, z1 = z0 + cx.planes < g->d.vol_nz ? z0 + cx.planes : g->d.vol_nz;
        RayGeom r = cbct_make_raygeom(g, z0, z1);
        float *buf = g->ws_vol + (size_t)b * slab_elems;
        if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));  // buffer drained by its copy
        CBCT_CUDA_TRY(cudaMemsetAsync(buf, 0, cbct_padded_volume_elems(r) * channels * sizeof(float), st));
        rc = cbct_launch_adjoint(g, r, d_sino, buf, channels, st);
        if (rc) return rc;
        if (cx.n_slabs == 1) {
            if (kv == MEM_DEVICE) rc = cbct_launch_unpad_volume(g, r, buf, vol, channels, cx.nvol, 0, st);
            else rc = d2h_slab(r, buf, vol, channels, cx.nvol, st);
            if (rc) return rc;
        } else {
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(g->copy_stream, g->ev[2 + b], 0));
            if (kv == MEM_DEVICE) rc = cbct_launch_unpad_volume(g, r, buf, vol, channels, cx.nvol, 0, g->copy_stream);
            else rc = d2h_slab(r, buf, vol, channels, cx.nvol, g->copy_stream);
            if (rc) return rc;
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], g->copy_stream));
        }
    }
    if (cx.n_slabs > 1) {  // join the copy stream back into `st`
        CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[0], 0));
        CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[1], 0));
    }
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

// ---------------------------------------------------------------------------
extern "C" int cbct_bp_fdk(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream)
{
    CallCtx cx;
    int rc = begin_call(gc, sino, vol, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    MemKind kv = classify(vol), ks = classify(sino);
    cx.pageable = (kv == MEM_HOST_PAGEABLE) || (ks == MEM_HOST_PAGEABLE);

    int pu = cbct_padded_sino_pitch(g), pv = cbct_padded_sino_rows(g);
    size_t psino = (size_t)g->d.n_views * pu * pv * channels;
    rc = ensure(&g->ws_sino, &g->ws_sino_bytes, psino * sizeof(float));
    if (rc) return rc;
    if (ks == MEM_DEVICE) {
        rc = cbct_launch_pad_sino(g, sino, g->ws_sino, channels, st);
        if (rc) return rc;
    } else {
        CBCT_CUDA_TRY(cudaMemsetAsync(g->ws_sino, 0, psino * sizeof(float), st));
        cudaMemcpy3DParms p;
        memset(&p, 0, sizeof(p));
        p.srcPtr = make_cudaPitchedPtr((void *)sino, g->d.det_nu * sizeof(float), g->d.det_nu, g->d.det_nv);
        p.dstPtr = make_cudaPitchedPtr((void *)g->ws_sino, pu * sizeof(float), pu, pv);
        p.dstPos = make_cudaPos(CBCT_PAD * sizeof(float), CBCT_PAD, 0);
        p.extent = make_cudaExtent(g->d.det_nu * sizeof(float), g->d.det_nv, (size_t)g->d.n_views * channels);
        p.kind = cudaMemcpyHostToDevice;
        CBCT_CUDA_TRY(cudaMemcpy3DAsync(&p, st));
    }
    if (kv == MEM_DEVICE && cx.n_slabs == 1) {
        rc = cbct_launch_fdk(g, g->ws_sino, vol, channels, 0, g->d.vol_nz, cx.nvol, 0, st);
        if (rc) return rc;
    } else {
        // output slabs staged through device workspace (unpadded), double-buffered
        size_t plane = (size_t)g->d.vol_nx * g->d.vol_ny;
        size_t slab_elems = plane * cx.planes * channels;
        int nbuf = cx.n_slabs > 1 ? 2 : 1;
        rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_elems * nbuf * sizeof(float));
        if (rc) return rc;
        for (int s = 0; s < cx.n_slabs; ++s) {
            int b = s & 1;
            int z0 = s * cx.planes, z1 = z0 + cx.planes < g->d.vol_nz ? z0 + cx.planes : g->d.vol_nz;
            float *buf = g->ws_vol + (size_t)b * slab_elems;
            size_t bstride = plane * (z1 - z0);
            if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));
            rc = cbct_launch_fdk(g, g->ws_sino, buf, channels, z0, z1, bstride, z0, st);
            if (rc) return rc;
            cudaStream_t cs = cx.n_slabs > 1 ? g->copy_stream : st;
            if (cx.n_slabs > 1) {
                CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
                CBCT_CUDA_TRY(cudaStreamWaitEvent(cs, g->ev[2 + b], 0));
            }
            for (int c = 0; c < channels; ++c)
                CBCT_CUDA_TRY(cudaMemcpyAsync(vol + c * cx.nvol + (size_t)z0 * plane, buf + c * bstride,
                                              bstride * sizeof(float),
                                              kv == MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, cs));
            if (cx.n_slabs > 1) CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], cs));
        }
        if (cx.n_slabs > 1) {
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[0], 0));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[1], 0));
        }
    }
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}
