// cbct_api.cu -- C ABI entry points of libcbct.so (include/cbct.h): pointer
// classification, device workspace, host staging and the z-slab streaming
// driver (A5; exact by linearity: P f = sum_s P(f 1_slab_s), and (P^T y)|slab,
// FDK|slab are independent per slab because the sample lattice is anchored at
// the source, reading R3).  PAPER.md:165, :292 motivate the streaming.
//
// Forward: the volume is quad-packed slab by slab (cbct_fp.cu) into device
// workspace capped by max_workset_bytes; a copy stream fills one slab buffer
// (H2D copy of the raw planes if the volume is in host memory, then the pack
// kernel) while the caller's stream projects the other.  Backprojectors write
// disjoint output planes: straight into a device volume, or slab by slab
// through a double-buffered device staging buffer into a host volume.
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

// Set by begin_call: the caller's stream is being captured into a CUDA graph.  A captured graph bakes in the
// workspace addresses, and cudaMalloc / cudaFree / cudaDeviceSynchronize are not allowed during capture, so a call
// that would have to GROW the workspace then fails loudly (CBCT_ERR_UNSUPPORTED) instead: warm the handle up with
// one uncaptured call of the same shape, or cbct_geom_reserve, first.
static thread_local bool g_capturing = false;

static int ensure(float **p, size_t *have, size_t need)
{
    if (*have >= need) return CBCT_OK;
    if (g_capturing) {
        cbct_set_cuda_error(cudaErrorStreamCaptureUnsupported, "workspace growth while the stream is capturing "
                            "(warm up or cbct_geom_reserve first)");
        return CBCT_ERR_UNSUPPORTED;
    }
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


struct CallCtx {
    cbct_geom *g;
    cudaStream_t st;
    int channels;
    size_t nvol, nsino, plane;  // elements per channel; elements per z-plane
    MemKind kv, ks;
    bool pageable;
};

static int begin_call(const cbct_geom *gc, const void *vol, const void *sino, int32_t channels, void *stream,
                      CallCtx &cx)
{
    if (!gc || !vol || !sino || channels < 1) return CBCT_ERR_INVALID_ARG;
    int rc = have_device();
    if (rc) return rc;
    cx.g = const_cast<cbct_geom *>(gc);
    cx.st = (cudaStream_t)stream;
    cx.channels = channels;
    cx.plane = (size_t)gc->d.vol_nx * gc->d.vol_ny;
    cx.nvol = cx.plane * gc->d.vol_nz;
    cx.nsino = (size_t)gc->d.n_views * gc->d.det_nv * gc->d.det_nu;
    cx.kv = classify(vol);
    cx.ks = classify(sino);
    cx.pageable = (cx.kv == MEM_HOST_PAGEABLE) || (cx.ks == MEM_HOST_PAGEABLE);
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(cx.st, &cap) != cudaSuccess) { (void)cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
    g_capturing = cap != cudaStreamCaptureStatusNone;
    if (g_capturing && (cx.kv != MEM_DEVICE || cx.ks != MEM_DEVICE)) return CBCT_ERR_UNSUPPORTED;  // host staging uses side streams
    if (g_capturing && (!cx.g->copy_stream || !cx.g->ev[3])) return CBCT_ERR_UNSUPPORTED;           // never warmed up
    return ensure_streams(cx.g);
}

// ---------------------------------------------------------------------------
// A2 + A5
// ---------------------------------------------------------------------------
// ---------------------------------------------------------------------------
// HOST buffers without a work-set cap: the call is cut into blocks of 2 channels (4 for the forward projector and the adjoint) that flow through a
// three-stage pipeline -- H2D copy of block b+1 (one stream), the device implementation on block b (the
// caller's stream), D2H copy of block b-1 (another stream) -- with two device buffers per side, so the
// PCIe copies in both directions hide behind the kernels.  `inner(din, dout, c0, nc)` enqueues the
// device implementation for channels [c0, c0 + nc) on the caller's stream.
// ---------------------------------------------------------------------------
// `sched(c0, left)` = channels of the block that starts at channel c0 (clamped to [1, min(BK, left)]): the first
// block's H2D copy and the last block's D2H copy are the only transfers no kernel hides, so a call whose kernels run
// as fast on narrower blocks starts and ends with those (measured on config 4 through pinned buffers, 8 channels:
// cbct_fp 135.5 -> see DESIGN.md s.6.4).
template <class Inner, class Sched>
static int blocked_call(CallCtx &cx, const float *in, size_t n_in, MemKind kin, float *out, size_t n_out, MemKind kout,
                        Inner inner, int BK, Sched sched)
{
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    const int channels = cx.channels;
    if (!g->h2d_stream) CBCT_CUDA_TRY(cudaStreamCreateWithFlags(&g->h2d_stream, cudaStreamNonBlocking));
    if (!g->d2h_stream) CBCT_CUDA_TRY(cudaStreamCreateWithFlags(&g->d2h_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 7; ++i)
        if (!g->ev_blk[i]) CBCT_CUDA_TRY(cudaEventCreateWithFlags(&g->ev_blk[i], cudaEventDisableTiming));
    cudaEvent_t *evH = g->ev_blk, *evC = g->ev_blk + 2, *evD = g->ev_blk + 4, ev0 = g->ev_blk[6];
    int rc;
    if (kin != MEM_DEVICE) {
        rc = ensure(&g->ws_blk_in, &g->ws_blk_in_bytes, 2 * BK * n_in * sizeof(float));
        if (rc) return rc;
    }
    if (kout != MEM_DEVICE) {
        rc = ensure(&g->ws_blk_out, &g->ws_blk_out_bytes, 2 * BK * n_out * sizeof(float));
        if (rc) return rc;
    }
    // the copy streams start after everything already queued on `st`
    CBCT_CUDA_TRY(cudaEventRecord(ev0, st));
    CBCT_CUDA_TRY(cudaStreamWaitEvent(g->h2d_stream, ev0, 0));
    CBCT_CUDA_TRY(cudaStreamWaitEvent(g->d2h_stream, ev0, 0));
    int nb = 0;
    for (int b = 0, c0 = 0, nc = 0; c0 < channels; ++b, c0 += nc, nb = b) {
        const int i = b & 1, left = channels - c0;
        nc = sched(c0, left);
        if (nc > BK) nc = BK;
        if (nc > left) nc = left;
        if (nc < 1) nc = 1;
        const float *din = in + (size_t)c0 * n_in;
        float *dout = out + (size_t)c0 * n_out;
        if (kin != MEM_DEVICE) {
            float *buf = g->ws_blk_in + (size_t)i * BK * n_in;
            if (b >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(g->h2d_stream, evC[i], 0));  // block b-2 consumed
            CBCT_CUDA_TRY(cudaMemcpyAsync(buf, din, (size_t)nc * n_in * sizeof(float), cudaMemcpyHostToDevice, g->h2d_stream));
            CBCT_CUDA_TRY(cudaEventRecord(evH[i], g->h2d_stream));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, evH[i], 0));
            din = buf;
        }
        if (kout != MEM_DEVICE) {
            if (b >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, evD[i], 0));  // block b-2 copied out
            dout = g->ws_blk_out + (size_t)i * BK * n_out;
        }
        rc = inner(din, dout, c0, nc);
        if (rc) return rc;
        CBCT_CUDA_TRY(cudaEventRecord(evC[i], st));
        if (kout != MEM_DEVICE) {
            CBCT_CUDA_TRY(cudaStreamWaitEvent(g->d2h_stream, evC[i], 0));
            CBCT_CUDA_TRY(cudaMemcpyAsync(out + (size_t)c0 * n_out, dout, (size_t)nc * n_out * sizeof(float),
                                          cudaMemcpyDeviceToHost, g->d2h_stream));
            CBCT_CUDA_TRY(cudaEventRecord(evD[i], g->d2h_stream));
        }
    }
    if (kout != MEM_DEVICE) {  // join the D2H stream back into `st`
        CBCT_CUDA_TRY(cudaStreamWaitEvent(st, evD[0], 0));
        if (nb > 1) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, evD[1], 0));
    }
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

// y != nullptr: sino = P vol - y (the residual of the Landweber term, fused into the epilogue; y is a
// DEVICE sinogram).  In the slab path the sinogram starts as -y instead of zero.
static int fp_impl(const cbct_geom *gc, const float *vol, const float *y, float *sino, int32_t channels, void *stream)
{
    CallCtx cx;
    int rc = begin_call(gc, vol, sino, channels, stream, cx);
    if (rc) return rc;
    if (y && (classify(y) != MEM_DEVICE || y == sino)) return CBCT_ERR_INVALID_ARG;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    const int nz = g->d.vol_nz;
    const int planes = cbct_plan_slab_planes(g, channels);
    if (planes < 1) return CBCT_ERR_NOMEM;
    const int n_slabs = (nz + planes - 1) / planes;
    const int nbuf = n_slabs > 1 ? 2 : 1;
    const bool host_vol = cx.kv != MEM_DEVICE;
    if ((host_vol || cx.ks != MEM_DEVICE) && g->d.max_workset_bytes == 0)
        return blocked_call(cx, vol, cx.nvol, cx.kv, sino, cx.nsino, cx.ks,
                            [&](const float *dv, float *ds, int c0, int nc) {
                                return fp_impl(gc, dv, y ? y + (size_t)c0 * cx.nsino : nullptr, ds, nc, stream);
                            },
                            channels >= 4 ? 4 : 2,  // blocks of 4 channels take the channel-interleaved kernel ...
                            // ... unless single channels run as fast (through their quarter-turn images)
                            [&](int, int) { return cbct_fp_single_channel_is_fast(g) ? 1 : 4; });

    float *d_sino = sino;
    if (cx.ks != MEM_DEVICE) {
        rc = ensure(&g->ws_sino, &g->ws_sino_bytes, cx.nsino * channels * sizeof(float));
        if (rc) return rc;
        d_sino = g->ws_sino;
    }
    const RayGeom rmax = cbct_make_raygeom(g, 0, planes);
    // float4 cells per buffer: channel-interleaved groups of 4, then quad-packed channels (cbct_fp.cu)
    const size_t slab_cells = (size_t)(channels / 4) * (size_t)(rmax.px + CBCT_ROW_SKEW) * rmax.py * rmax.pz
                              + (size_t)(channels % 4) * cbct_packed_tail_cells(g, rmax);
    rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_cells * nbuf * sizeof(float4));
    if (rc) return rc;
    const size_t stage_elems = cx.plane * planes * channels;
    if (host_vol) {
        rc = ensure(&g->ws_stage, &g->ws_stage_bytes, stage_elems * nbuf * sizeof(float));
        if (rc) return rc;
    }
    if (n_slabs > 1) {
        // every slab adds its part (only into the detector rows its shadow covers) to a zeroed sinogram
        if (y) {
            CBCT_CUDA_TRY(cudaMemcpyAsync(d_sino, y, cx.nsino * channels * sizeof(float), cudaMemcpyDeviceToDevice, st));
            rc = cbct_launch_negate(g, d_sino, cx.nsino * channels, st);
            if (rc) return rc;
        } else {
            CBCT_CUDA_TRY(cudaMemsetAsync(d_sino, 0, cx.nsino * channels * sizeof(float), st));
        }
        // the copy stream starts after everything already queued on `st`
        CBCT_CUDA_TRY(cudaEventRecord(g->ev[0], st));
        CBCT_CUDA_TRY(cudaStreamWaitEvent(g->copy_stream, g->ev[0], 0));
    }
    for (int s = 0; s < n_slabs; ++s) {
        const int b = s & 1;
        const int z0 = s * planes, z1 = z0 + planes < nz ? z0 + planes : nz;
        const RayGeom r = cbct_make_raygeom(g, z0, z1);
        float4 *buf = reinterpret_cast<float4 *>(g->ws_vol) + (size_t)b * slab_cells;
        cudaStream_t cs = n_slabs > 1 ? g->copy_stream : st;
        // buffer b is free once the projection of slab s-2 has finished
        if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(cs, g->ev[2 + b], 0));
        if (host_vol) {
            float *stage = g->ws_stage + (size_t)b * stage_elems;
            const size_t n = cx.plane * (z1 - z0);
            for (int c = 0; c < channels; ++c)
                CBCT_CUDA_TRY(cudaMemcpyAsync(stage + c * n, vol + c * cx.nvol + (size_t)z0 * cx.plane,
                                              n * sizeof(float), cudaMemcpyHostToDevice, cs));
            rc = cbct_launch_pack_volume(g, r, stage, buf, channels, n, z0, cs);
        } else {
            rc = cbct_launch_pack_volume(g, r, vol, buf, channels, cx.nvol, 0, cs);
        }
        if (rc) return rc;
        if (n_slabs > 1) {
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], cs));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));
        }
        rc = cbct_launch_fp(g, r, buf, d_sino, channels, n_slabs > 1, n_slabs > 1 ? nullptr : y, st);
        if (rc) return rc;
        if (n_slabs > 1) CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
    }
    if (cx.ks != MEM_DEVICE)
        CBCT_CUDA_TRY(cudaMemcpyAsync(sino, d_sino, cx.nsino * channels * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" int cbct_fp(const cbct_geom *gc, const float *vol, float *sino, int32_t channels, void *stream)
{
    return fp_impl(gc, vol, nullptr, sino, channels, stream);
}

extern "C" int cbct_fp_residual(const cbct_geom *gc, const float *vol, const float *y, float *sino, int32_t channels,
                                void *stream)
{
    if (!y) return CBCT_ERR_INVALID_ARG;
    return fp_impl(gc, vol, y, sino, channels, stream);
}

// ---------------------------------------------------------------------------
// Output side of A3 / A4: `launch(dst, zs0, zs1, channel_stride, z_origin)`
// fills planes [zs0, zs1).  A device volume is written in place in one pass; a
// host volume is produced slab by slab through double-buffered device staging
// (two buffers of all channels under max_workset_bytes; D2H copies on the copy
// stream overlap the next slab's kernel).
// ---------------------------------------------------------------------------
// `pairs` (the launch can fill a slab of the lower half of the grid together with its mirror image, which shares
// all its weights): slabs then cover [z0, z1) below the middle plane plus [nz - z1, nz - z0), staged back to back.
template <class Launch>
static int produce_volume(CallCtx &cx, float *vol, bool pairs, Launch launch)
{
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    const int nz = g->d.vol_nz;
    if (cx.kv == MEM_DEVICE) return launch(vol, 0, nz, cx.nvol, 0, CBCT_NO_MIRROR_PAIR);
    const uint64_t cap = g->d.max_workset_bytes;
    const uint64_t plane_bytes = (uint64_t)cx.plane * sizeof(float) * (uint64_t)cx.channels;
    int planes = nz;
    if (cap != 0 && plane_bytes * (uint64_t)nz > cap) planes = (int)(cap / (2 * plane_bytes));
    if (planes < 1) return CBCT_ERR_NOMEM;
    if (pairs && planes >= 2 && nz > 1) {
        const int nh = (nz + 1) / 2;
        const int hp = planes >= nz ? nh : planes / 2;  // planes of the lower half per slab
        const int n_slabs = (nh + hp - 1) / hp;
        const int nbuf = n_slabs > 1 ? 2 : 1;
        const size_t slab_elems = cx.plane * 2 * hp * cx.channels;
        int rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_elems * nbuf * sizeof(float));
        if (rc) return rc;
        for (int s = 0; s < n_slabs; ++s) {
            const int b = s & 1;
            const int z0 = s * hp, z1 = z0 + hp < nh ? z0 + hp : nh, n = z1 - z0;
            const int mlo = nz - z1;                    // mirror images: planes [mlo, nz - z0)
            const int skip = mlo < z1 ? z1 - mlo : 0;   // odd nz: the middle plane is its own image
            float *buf = g->ws_vol + (size_t)b * slab_elems;
            const size_t bstride = cx.plane * 2 * n;
            if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));  // buffer drained by its copies
            rc = launch(buf, z0, z1, bstride, z0, mlo - n);
            if (rc) return rc;
            cudaStream_t cs = n_slabs > 1 ? g->copy_stream : st;
            if (n_slabs > 1) {
                CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
                CBCT_CUDA_TRY(cudaStreamWaitEvent(cs, g->ev[2 + b], 0));
            }
            for (int c = 0; c < cx.channels; ++c) {
                CBCT_CUDA_TRY(cudaMemcpyAsync(vol + c * cx.nvol + (size_t)z0 * cx.plane, buf + c * bstride,
                                              cx.plane * n * sizeof(float), cudaMemcpyDeviceToHost, cs));
                if (n > skip)
                    CBCT_CUDA_TRY(cudaMemcpyAsync(vol + c * cx.nvol + (size_t)(mlo + skip) * cx.plane,
                                                  buf + c * bstride + cx.plane * (n + skip),
                                                  cx.plane * (n - skip) * sizeof(float), cudaMemcpyDeviceToHost, cs));
            }
            if (n_slabs > 1) CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], cs));
        }
        if (n_slabs > 1) {  // join the copy stream back into `st`
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[0], 0));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[1], 0));
        }
        return CBCT_OK;
    }
    const int n_slabs = (nz + planes - 1) / planes;
    const int nbuf = n_slabs > 1 ? 2 : 1;
    const size_t slab_elems = cx.plane * planes * cx.channels;
    int rc = ensure(&g->ws_vol, &g->ws_vol_bytes, slab_elems * nbuf * sizeof(float));
    if (rc) return rc;
    for (int s = 0; s < n_slabs; ++s) {
        const int b = s & 1;
        const int z0 = s * planes, z1 = z0 + planes < nz ? z0 + planes : nz;
        float *buf = g->ws_vol + (size_t)b * slab_elems;
        const size_t bstride = cx.plane * (z1 - z0);
        if (s >= 2) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[b], 0));  // buffer drained by its copy
        rc = launch(buf, z0, z1, bstride, z0, CBCT_NO_MIRROR_PAIR);
        if (rc) return rc;
        cudaStream_t cs = n_slabs > 1 ? g->copy_stream : st;
        if (n_slabs > 1) {
            CBCT_CUDA_TRY(cudaEventRecord(g->ev[2 + b], st));
            CBCT_CUDA_TRY(cudaStreamWaitEvent(cs, g->ev[2 + b], 0));
        }
        for (int c = 0; c < cx.channels; ++c)
            CBCT_CUDA_TRY(cudaMemcpyAsync(vol + c * cx.nvol + (size_t)z0 * cx.plane, buf + c * bstride,
                                          bstride * sizeof(float), cudaMemcpyDeviceToHost, cs));
        if (n_slabs > 1) CBCT_CUDA_TRY(cudaEventRecord(g->ev[b], cs));
    }
    if (n_slabs > 1) {  // join the copy stream back into `st`
        CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[0], 0));
        if (n_slabs > 1) CBCT_CUDA_TRY(cudaStreamWaitEvent(st, g->ev[1], 0));
    }
    return CBCT_OK;
}

// ---------------------------------------------------------------------------
// A3
// ---------------------------------------------------------------------------
static int adjoint_impl(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream, bool weighted)
{
    CallCtx cx;
    int rc = begin_call(gc, vol, sino, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    const size_t sino_bytes = cx.nsino * channels * sizeof(float);
    if ((cx.kv != MEM_DEVICE || cx.ks != MEM_DEVICE) && g->d.max_workset_bytes == 0)
        return blocked_call(cx, sino, cx.nsino, cx.ks, vol, cx.nvol, cx.kv,
                            [&](const float *ds, float *dv, int, int nc) {
                                return adjoint_impl(gc, ds, dv, nc, stream, weighted);
                            },
                            channels >= 4 ? 4 : 2,  // blocks of 4 channels take the 32-accumulator kernel
                            // (pairs at both ends of the call -- the column-walk kernel, 12.3 ms per channel -- paid
                            // while blocks of 4 ran at 11.9 ms per channel; at 10.1 they no longer do: 8 channels
                            // through pinned buffers 95.6 ms as 2 + 4 + 2, 93.5 ms as 4 + 4)
                            [&](int, int) { return 4; });

    const float *d_sino = sino;
    if (cx.ks != MEM_DEVICE) {
        rc = ensure(&g->ws_sino, &g->ws_sino_bytes, sino_bytes);
        if (rc) return rc;
        CBCT_CUDA_TRY(cudaMemcpyAsync(g->ws_sino, sino, sino_bytes, cudaMemcpyHostToDevice, st));
        d_sino = g->ws_sino;
    }
    if (weighted) {
        rc = cbct_ensure_filter_tables(g);
        if (rc) return rc;
    }
    if (g->sym_rot > 1) {  // views related by a grid rotation, interleaved for vector loads (+ w(u) if asked)
        rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, sino_bytes);
        if (rc) return rc;
        rc = cbct_launch_interleave_views(g, d_sino, g->ws_sino2, channels, weighted ? g->d_filter_tab : nullptr, st);
        if (rc) return rc;
        d_sino = g->ws_sino2;
    }
    // no rotation symmetry: channels interleaved in groups of 4 for the column kernel's vector loads (w(u) fused into
    // that pass), and, if weighted, one weighting pass for the channels and kernels that read the planar layout
    const float *sino_ci = nullptr;
    const int ci_groups = g->sym_rot == 1 ? cbct_adjoint_channel_groups(g, channels, cx.kv == MEM_DEVICE) : 0;
    if (g->sym_rot == 1 && (weighted || ci_groups)) {
        const size_t plain = weighted ? cx.nsino * channels : 0, grouped = (size_t)ci_groups * 4 * cx.nsino;
        rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, (plain + grouped) * sizeof(float));
        if (rc) return rc;
        if (ci_groups) {
            rc = cbct_launch_interleave_channels(g, d_sino, g->ws_sino2 + plain, ci_groups, weighted ? g->d_filter_tab : nullptr, st);
            if (rc) return rc;
            sino_ci = g->ws_sino2 + plain;
        }
        if (weighted) {
            rc = cbct_launch_redundancy_weight(g, d_sino, g->ws_sino2, channels, st);
            if (rc) return rc;
            d_sino = g->ws_sino2;
        }
    }
    // the views of a launch split over groups of CTAs (partial outputs in workspace, then reduced)
    const size_t partial_floats = cx.kv == MEM_DEVICE ? cbct_adjoint_partial_floats(g) : 0;
    const int nsplit = partial_floats ? 2 : 1;   // "partial outputs may be used": the launcher picks the group counts
    float *partial = nullptr;
    if (partial_floats) {
        rc = ensure(&g->ws_vol, &g->ws_vol_bytes, partial_floats * sizeof(float));
        if (rc) return rc;
        partial = g->ws_vol;
    }
    rc = produce_volume(cx, vol, g->sym_mirror_z != 0, [&](float *dst, int zs0, int zs1, size_t cstride, int z_origin, int mirror_origin) {
        return cbct_launch_adjoint(g, d_sino, dst, channels, zs0, zs1, cstride, z_origin, partial, nsplit, st, mirror_origin,
                                   sino_ci, ci_groups);
    });
    if (rc) return rc;
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" int cbct_bp_adjoint(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream)
{
    return adjoint_impl(gc, sino, vol, channels, stream, false);
}

extern "C" int cbct_bp_adjoint_weighted(const cbct_geom *gc, const float *sino, float *vol, int32_t channels,
                                        void *stream)
{
    return adjoint_impl(gc, sino, vol, channels, stream, true);
}

// ---------------------------------------------------------------------------
// A4
// ---------------------------------------------------------------------------
extern "C" int cbct_bp_fdk(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream)
{
    CallCtx cx;
    int rc = begin_call(gc, vol, sino, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    if ((cx.kv != MEM_DEVICE || cx.ks != MEM_DEVICE) && g->d.max_workset_bytes == 0)
        return blocked_call(cx, sino, cx.nsino, cx.ks, vol, cx.nvol, cx.kv,
                            [&](const float *ds, float *dv, int, int nc) { return cbct_bp_fdk(gc, ds, dv, nc, stream); },
                            2, [&](int, int) { return g->sym_rot == 1 ? 2 : 1; });  // the kernel takes 1 channel per launch (2 without rotation symmetry)

    // zero-bordered, rotation-interleaved copy of the sinogram (cbct_fdk.cu)
    const size_t psino = cbct_padded_sino_floats(g) * channels;
    const size_t sino_bytes = cx.nsino * channels * sizeof(float);
    const float *d_sino = sino;
    if (cx.ks != MEM_DEVICE) {
        rc = ensure(&g->ws_sino, &g->ws_sino_bytes, sino_bytes);
        if (rc) return rc;
        CBCT_CUDA_TRY(cudaMemcpyAsync(g->ws_sino, sino, sino_bytes, cudaMemcpyHostToDevice, st));
        d_sino = g->ws_sino;
    }
    rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, psino * sizeof(float));
    if (rc) return rc;
    rc = cbct_launch_pad_sino(g, d_sino, g->ws_sino2, channels, st);
    if (rc) return rc;
    const float *padded = g->ws_sino2;
    rc = produce_volume(cx, vol, g->sym_mirror_z != 0, [&](float *dst, int zs0, int zs1, size_t cstride, int z_origin, int mirror_origin) {
        return cbct_launch_fdk(g, padded, dst, channels, zs0, zs1, cstride, z_origin, st, mirror_origin);
    });
    if (rc) return rc;
    if (cx.pageable) CBCT_CUDA_TRY(cudaStreamSynchronize(st));
    return CBCT_OK;
}

// ---------------------------------------------------------------------------
// Plane ranges of the backprojectors (the unit a multi-GPU caller shards by; also the
// unit of the streaming path above).  DEVICE pointers.  out[c] holds planes [z0, z1) of channel c; with
// mirror_pair != 0 (geometry symmetric under z -> -z, z1 <= ceil(nz / 2)) it holds 2 (z1 - z0) - skip planes per
// channel: [z0, z1) followed by their mirror images [nz - z1 + skip, nz - z0) in ascending order, skip = 1 when
// the range contains the middle plane of an odd nz (its own image), else 0.  The pair shares every weight.
// ---------------------------------------------------------------------------
static int slab_impl(const cbct_geom *gc, const float *sino, float *out, int32_t channels, int32_t z0, int32_t z1,
                     int32_t mirror_pair, void *stream, int which)
{
    CallCtx cx;
    int rc = begin_call(gc, out, sino, channels, stream, cx);
    if (rc) return rc;
    cbct_geom *g = cx.g;
    cudaStream_t st = cx.st;
    const int nz = g->d.vol_nz;
    if (cx.kv != MEM_DEVICE || cx.ks != MEM_DEVICE) return CBCT_ERR_INVALID_ARG;
    if (z0 < 0 || z1 > nz || z0 >= z1) return CBCT_ERR_INVALID_ARG;
    if (mirror_pair && (!g->sym_mirror_z || z1 > (nz + 1) / 2)) return CBCT_ERR_INVALID_ARG;
    const int n = z1 - z0;
    const int mlo = nz - z1;
    const int skip = mirror_pair && mlo < z1 ? z1 - mlo : 0;
    const size_t cstride = cx.plane * (size_t)(mirror_pair ? 2 * n - skip : n);
    const int morigin = mirror_pair ? mlo + skip - n : CBCT_NO_MIRROR_PAIR;  // plane index stored at out[c] + 0
    const size_t sino_bytes = cx.nsino * channels * sizeof(float);
    if (which == 0) {
        const float *d_sino = sino;
        if (g->sym_rot > 1) {
            rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, sino_bytes);
            if (rc) return rc;
            rc = cbct_launch_interleave_views(g, sino, g->ws_sino2, channels, nullptr, st);
            if (rc) return rc;
            d_sino = g->ws_sino2;
        }
        return cbct_launch_adjoint(g, d_sino, out, channels, z0, z1, cstride, z0, nullptr, 1, st, morigin);
    }
    rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, cbct_padded_sino_floats(g) * channels * sizeof(float));
    if (rc) return rc;
    rc = cbct_launch_pad_sino(g, sino, g->ws_sino2, channels, st);
    if (rc) return rc;
    return cbct_launch_fdk(g, g->ws_sino2, out, channels, z0, z1, cstride, z0, st, morigin);
}

extern "C" int cbct_bp_adjoint_slab(const cbct_geom *g, const float *sino, float *out, int32_t channels, int32_t z0,
                                    int32_t z1, int32_t mirror_pair, void *stream)
{
    return slab_impl(g, sino, out, channels, z0, z1, mirror_pair, stream, 0);
}

extern "C" int cbct_bp_fdk_slab(const cbct_geom *g, const float *sino, float *out, int32_t channels, int32_t z0,
                                int32_t z1, int32_t mirror_pair, void *stream)
{
    return slab_impl(g, sino, out, channels, z0, z1, mirror_pair, stream, 1);
}

// ---------------------------------------------------------------------------
// Workspace queries / up-front allocation (so that later calls neither allocate nor synchronise: CUDA graphs)
// ---------------------------------------------------------------------------
extern "C" int cbct_geom_workspace_bytes(const cbct_geom *g, uint64_t *out)
{
    if (!g || !out) return CBCT_ERR_INVALID_ARG;
    *out = (uint64_t)g->ws_vol_bytes + g->ws_sino_bytes + g->ws_sino2_bytes + g->ws_stage_bytes + g->ws_blk_in_bytes +
           g->ws_blk_out_bytes + (g->d_filter_tab ? 3u * (uint64_t)g->d.det_nu * sizeof(float) : 0u);
    return CBCT_OK;
}

extern "C" int cbct_geom_reserve(cbct_geom *g, int32_t channels)
{
    if (!g || channels < 1) return CBCT_ERR_INVALID_ARG;
    int rc = have_device();
    if (rc) return rc;
    g_capturing = false;
    rc = ensure_streams(g);
    if (rc) return rc;
    const size_t nsino = (size_t)g->d.n_views * g->d.det_nv * g->d.det_nu;
    // forward: packed slab buffer(s)
    const int planes = cbct_plan_slab_planes(g, channels);
    if (planes < 1) return CBCT_ERR_NOMEM;
    const int n_slabs = (g->d.vol_nz + planes - 1) / planes;
    const RayGeom rmax = cbct_make_raygeom(g, 0, planes);
    size_t vol_bytes = ((size_t)(channels / 4) * (size_t)(rmax.px + CBCT_ROW_SKEW) * rmax.py * rmax.pz +
                        (size_t)(channels % 4) * cbct_packed_tail_cells(g, rmax)) * (n_slabs > 1 ? 2 : 1) * sizeof(float4);
    // adjoint on small grids: partial outputs of the view groups
    if (cbct_adjoint_partial_floats(g) * sizeof(float) > vol_bytes) vol_bytes = cbct_adjoint_partial_floats(g) * sizeof(float);
    rc = ensure(&g->ws_vol, &g->ws_vol_bytes, vol_bytes);
    if (rc) return rc;
    // backprojectors: re-laid-out sinogram (view-interleaved / zero-bordered)
    const size_t psino = cbct_padded_sino_floats(g);
    // (sym_rot == 1: the weighted adjoint keeps a weighted planar copy beside the channel groups)
    const size_t adj_sino = g->sym_rot == 1 ? 2 * nsino : nsino;
    rc = ensure(&g->ws_sino2, &g->ws_sino2_bytes, (psino > adj_sino ? psino : adj_sino) * channels * sizeof(float));
    if (rc) return rc;
    return cbct_ensure_filter_tables(g);
}
