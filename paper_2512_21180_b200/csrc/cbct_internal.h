// cbct_internal.h -- shared declarations of libcbct.so (product code; no oracle code).
//
// Coordinates used by every kernel: "voxel units" = world mm / vox_mm, world
// origin at the isocentre.  A device volume buffer ("padded
// volume") holds planes [z0, z1) of the grid with a zero border of CBCT_PAD
// voxels on every side, so the zero-extended trilinear interpolant (reading
// R4, DESIGN.md s.3) needs no bounds test in the sample loop:
//     padded index p = q + CBCT_PAD  (z: q - z0 + CBCT_PAD).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <utility>
#include <vector>

#include "../../include/cbct.h"

#define CBCT_PAD 2              // zero border (voxels / pixels) of padded buffers
#define CBCT_VIEWS_PER_LAUNCH 512
// bank swizzle of the packed cells: cell (jx, jy, jz) sits at position
// (jx & ~7) | ((jx + CBCT_SWIZZLE_Y jy + CBCT_SWIZZLE_Z jz) & 7) of its row (cbct_fp.cu)
#define CBCT_SWIZZLE_Y 6
#define CBCT_SWIZZLE_Z 4
#define CBCT_NO_MIRROR_PAIR (-2147483647 - 1)
#define CBCT_ROW_SKEW 8          // extra cells per row of the channel-interleaved (skewed) layout (cbct_fp.cu)

// View-independent geometry in voxel units (fp64), passed by value to kernels.
struct RayGeom {
    double sid, idd;        // source-isocentre, isocentre-detector distance
    double u0, du, v0, dv;  // detector coordinate of pixel 0 and pixel pitch
    double cx, cy, cz;      // volume centre
    double step;            // ray step (voxel units)
    double delta;           // ray step in mm = step * vox_mm (scale of the line integral)
    int nu, nv;             // detector size
    int nx, ny, nz;         // full grid size
    int z0, z1;             // planes [z0, z1) held by the padded buffer
    int px, py, pz;         // padded buffer dims (x pitch, rows, planes)
};

struct ViewChunk {
    double2 cs[CBCT_VIEWS_PER_LAUNCH];  // (cos phi, sin phi)
};

// per-launch parameters of the FDK backprojection kernel (fp64 setup, fp32 inner loop).
struct FdkGeom {
    double sid;             // voxel units
    double au, bu, av, bv;  // fu_pad = au * (-X s + Y c) / U + bu ; fv_pad = av * Z / U + bv
    double x0, y0, z0;      // centred world coordinate (voxel units) of voxel index 0
    double fu_max, fv_max;  // clamp range upper bounds in padded pixel coordinates
    int nx, ny, nz;
    int bx, by;             // base columns: ix < bx, iy < by (a quadrant / half if views rotate)
    int bz0, bz1;           // base planes [bz0, bz1) (the lower half if the z-mirror is used)
    int mz_origin;          // first stored plane of the z-mirrored voxels' output (NM = 2)
    int pu, pv;             // padded sinogram pitch / rows
    int n_views;            // views in this launch
    int nbase;              // n_views_total / sym_rot
};

struct cbct_geom {
    cbct_geom_desc d;
    std::vector<double> angles, cosphi, sinphi;
    // device workspace (lazily allocated, grown on demand)
    float *ws_vol = nullptr;   size_t ws_vol_bytes = 0;    // packed volume slab(s) / output staging slabs
    float *ws_sino = nullptr;  size_t ws_sino_bytes = 0;   // device copy of a host sinogram
    float *ws_sino2 = nullptr; size_t ws_sino2_bytes = 0;  // re-laid-out sinogram (view-interleaved / zero-bordered)
    float *ws_stage = nullptr; size_t ws_stage_bytes = 0;  // raw planes of a host volume on their way to the pack kernel
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    // channel-block pipeline for HOST buffers (cbct_api.cu): H2D and D2H streams, double-buffered blocks
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    cudaEvent_t ev_blk[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    float *ws_blk_in = nullptr;  size_t ws_blk_in_bytes = 0;
    float *ws_blk_out = nullptr; size_t ws_blk_out_bytes = 0;
    uint64_t launches = 0;
    int64_t sample_count = -1;
    float *d_filter_tab = nullptr;  // FDK front-end tables (cbct_fdk_filter.cu), built on first use
    // optional per-launch event pairs of the three main kernels (cbct_geom_profile)
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof[3];
    // symmetries of the geometry the gather adjoint may exploit (cbct_geom.cu):
    int sym_rot = 1;        // 4 / 2 / 1: views i and i + n/sym_rot see the grid rotated by 360/sym_rot deg
    bool sym_mirror_z = false;  // volume and detector symmetric under z -> -z
};

void cbct_set_cuda_error(cudaError_t e, const char *what);

#define CBCT_CUDA_TRY(expr)                                 \
    do {                                                    \
        cudaError_t e__ = (expr);                           \
        if (e__ != cudaSuccess) {                           \
            cbct_set_cuda_error(e__, #expr);                \
            return CBCT_ERR_CUDA;                           \
        }                                                   \
    } while (0)

// --- geometry helpers (cbct_geom.cu) ---------------------------------------
RayGeom cbct_make_raygeom(const cbct_geom *g, int z0, int z1);
size_t cbct_packed_volume_cells(const RayGeom &r);  // float4 cells per channel of a quad-packed slab
size_t cbct_packed_tail_cells(const cbct_geom *g, const RayGeom &r);  // ... per channel left over by the groups of 4
int cbct_padded_sino_pitch(const cbct_geom *g);
int cbct_padded_sino_rows(const cbct_geom *g);
size_t cbct_padded_sino_floats(const cbct_geom *g);  // per channel of the FDK kernel's record layout (cbct_fdk.cu)
int cbct_plan_slab_planes(const cbct_geom *g, int channels);  // planes per z-slab, <1 = cap too small

// --- kernel launchers; all enqueue on `st` ----------------------------------
int cbct_check_launch(cbct_geom *g, const char *what);
// bracket a main-kernel launch with an event pair when profiling is on (cbct_geom.cu)
void cbct_prof_begin(cbct_geom *g, int kernel, cudaStream_t st);
void cbct_prof_end(cbct_geom *g, int kernel, cudaStream_t st);
// quad-pack: src[C][nz_src][ny][nx] planes [r.z0, r.z1) -> dst[C][pz][py][px] float4 cells (cbct_fp.cu)
int cbct_launch_pack_volume(cbct_geom *g, const RayGeom &r, const float *src, float4 *dst, int channels,
                            size_t src_channel_stride, int src_z_origin, cudaStream_t st);
// forward projection of the packed slab(s); accumulate != 0 adds into sino; sub != nullptr: minus sub (same layout)
int cbct_launch_fp(cbct_geom *g, const RayGeom &r, const float4 *packed, float *sino, int channels,
                   int accumulate, const float *sub, cudaStream_t st);
// view-interleaved copy of the sinogram for the gather adjoint (only if g->sym_rot > 1);
// weights != nullptr: every pixel is multiplied by weights[iu] on the way (NEXT-3)
int cbct_launch_interleave_views(cbct_geom *g, const float *sino, float *out, int channels, const float *weights,
                                 cudaStream_t st);
// device tables of the FDK front end (cbct_fdk_filter.cu): g->d_filter_tab[0, nu) = redundancy weights
int cbct_ensure_filter_tables(cbct_geom *g);
int cbct_launch_negate(cbct_geom *g, float *buf, size_t n, cudaStream_t st);  // buf = -buf (cbct_fp.cu)
int cbct_launch_redundancy_weight(cbct_geom *g, const float *in, float *out, int channels, cudaStream_t st);
// gather adjoint into vol planes [zs0, zs1)
// sino_ci / ci_groups (sym_rot == 1 only, else nullptr / 0): channels [0, 4 ci_groups) also given interleaved in
// groups of 4 (cbct_launch_interleave_channels), which the column kernel reads with one vector load per pixel
int cbct_launch_adjoint(cbct_geom *g, const float *sino_src, float *vol, int channels, int zs0, int zs1,
                        size_t vol_channel_stride, int vol_z_origin, float *partial, int nsplit, cudaStream_t st,
                        int mirror_z_origin = CBCT_NO_MIRROR_PAIR, const float *sino_ci = nullptr, int ci_groups = 0);
int cbct_adjoint_channel_groups(const cbct_geom *g, int channels, bool device_volume);
// block widths of the HOST-buffer pipeline (cbct_api.cu): is a narrower block as fast per channel as a block of 4?
bool cbct_fp_single_channel_is_fast(const cbct_geom *g);   // cbct_fp.cu
int cbct_launch_interleave_channels(cbct_geom *g, const float *sino, float *out, int groups, const float *weights,
                                    cudaStream_t st);
int cbct_adjoint_view_splits(const cbct_geom *g);   // view groups of the adjoint's voxel kernel on small grids (1 = none)
int cbct_adjoint_column_splits(const cbct_geom *g); // view groups per tile of the adjoint's column kernel (1 = none)
bool cbct_adjoint_small_grid(const cbct_geom *g);    // fewer than 2 million base voxels: the voxel kernel splits views
size_t cbct_adjoint_partial_floats(const cbct_geom *g);  // workspace floats of the view groups' partial outputs
int cbct_launch_pad_sino(cbct_geom *g, const float *src, float *dst, int channels, cudaStream_t st);
// FDK backprojection from the padded sinogram into vol planes [zs0, zs1)
int cbct_launch_fdk(cbct_geom *g, const float *padded_sino, float *vol, int channels, int zs0, int zs1,
                    size_t vol_channel_stride, int vol_z_origin, cudaStream_t st,
                    int mirror_z_origin = CBCT_NO_MIRROR_PAIR);
