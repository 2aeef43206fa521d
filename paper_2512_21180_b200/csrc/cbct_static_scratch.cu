// cbct_static_scratch.cu -- cbct_bp_fdk_static: the FDK-weighted backprojection (A4, include/cbct.h)
// for callers that may not allocate: code under CUDA-graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  cbct_bp_fdk keeps the kernel's scratch -- the zero-bordered, record-interleaved copy of the
// sinogram that fdk_kernel gathers from (cbct_fdk.cu) -- in a workspace it grows with cudaMalloc; here the same
// scratch lives in a file-scope device array of CBCT_STATIC_SCRATCH_BYTES, which every GPU that loads the library
// holds until the process exits.  The two kernels (pad_sino_kernel, fdk_kernel) and their launch parameters are
// those of the device-pointer path of cbct_bp_fdk, so the output is the same bit for bit.
//
// This entry point calls no cudaMalloc / cudaFree, creates no stream or event, and never synchronises.
//
// Sharing: there is ONE array per device.  Every call on that device overwrites it, and two calls that overlap on
// the GPU (different streams, or two host threads) race on it: the caller serialises them.  The array keeps the
// last call's contents; nothing in it has to start at zero, because pad_sino_kernel writes every record of the
// region a call uses, the zero border included, before fdk_kernel reads it on the same stream.
#include <stdio.h>

#include "cbct_internal.h"

static __device__ __align__(256) float g_static_scratch[CBCT_STATIC_SCRATCH_BYTES / sizeof(float)];

// In host code `g_static_scratch` is only a handle of the symbol, not a device address: the address is asked for
// once per device, with that device current, and kept here.
#define CBCT_STATIC_MAX_DEVICES 64
static float *g_scratch_addr[CBCT_STATIC_MAX_DEVICES];  // written once per device; a racing second writer stores the same value

static int static_scratch(float **out)
{
    int dev = -1;
    CBCT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= CBCT_STATIC_MAX_DEVICES) return CBCT_ERR_UNSUPPORTED;
    float *p = g_scratch_addr[dev];
    if (!p) {
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            cbct_set_cuda_error(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_scratch)");
            return CBCT_ERR_CUDA;
        }
        g_scratch_addr[dev] = p;
    }
    *out = p;
    return CBCT_OK;
}

static bool is_device_pointer(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

extern "C" int cbct_static_scratch_setup(void)
{
    float *p = nullptr;
    return static_scratch(&p);
}

extern "C" int cbct_bp_fdk_static(const cbct_geom *gc, const float *sino, float *vol, int32_t channels, void *stream)
{
    if (!gc || !sino || !vol || channels < 1) return CBCT_ERR_INVALID_ARG;
    cbct_geom *g = const_cast<cbct_geom *>(gc);
    if (!is_device_pointer(sino) || !is_device_pointer(vol)) return CBCT_ERR_INVALID_ARG;
    if (g->profiling) return CBCT_ERR_UNSUPPORTED;  // the per-launch event pairs of cbct_geom_profile are created on the fly
    const unsigned long long need = (unsigned long long)cbct_padded_sino_floats(g) * (unsigned)channels * sizeof(float);
    if (need > CBCT_STATIC_SCRATCH_BYTES) {
        char msg[200];
        snprintf(msg, sizeof msg, "cbct_bp_fdk_static: this geometry with %d channel(s) needs %llu bytes of scratch, the "
                 "static array holds %llu (use cbct_bp_fdk)", (int)channels, need, (unsigned long long)CBCT_STATIC_SCRATCH_BYTES);
        cbct_set_cuda_error(cudaErrorInvalidValue, msg);
        return CBCT_ERR_UNSUPPORTED;
    }
    float *scratch = nullptr;
    int rc = static_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = cbct_launch_pad_sino(g, sino, scratch, channels, st);
    if (rc) return rc;
    const size_t nvol = (size_t)g->d.vol_nx * g->d.vol_ny * g->d.vol_nz;
    return cbct_launch_fdk(g, scratch, vol, channels, 0, g->d.vol_nz, nvol, 0, st, CBCT_NO_MIRROR_PAIR);
}
