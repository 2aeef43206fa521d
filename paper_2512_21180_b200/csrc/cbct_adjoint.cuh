// cbct_adjoint.cuh -- declarations shared by the two gather kernels of the matched adjoint (A3):
// cbct_adjoint.cu (a thread owns one or two voxels per symmetric image) and cbct_adjoint_column.cu (a thread walks a
// column of planes).  Product code only.
#pragma once
#include "cbct_internal.h"

struct AdjGeom {
    double sid, sdd, inv_sdd;
    double u0, du, inv_du, v0, dv, inv_dv;  // detector coordinate of pixel 0, pitch (voxel units)
    double x0, y0, z0;                      // world coordinate (voxel units) of voxel index 0
    double inv_step;
    float step, scale;                      // ray step (voxel units); Delta in mm
    float tz;                               // max |v| / sdd over the detector
    int fine;                               // the sample window of a (voxel, ray) pair can hold more than 6 lattice points
    int nu, nv, nx, ny, nz;
    int bx, by;                             // base domain: ix < bx, iy < by
    int bz0, bz1;                           // base planes [bz0, bz1)
    int mz_origin;                          // first stored plane of the z-mirrored voxels' output (NM = 2)
    int nq;                                 // views in this launch
    int nbase;                              // n_views / NR: views i and i + nbase differ by 360/NR degrees
    // small grids do not fill the GPU with one thread per base voxel: the views of a launch are then split
    // over `nsplit` groups of CTAs, each writing its partial sums to its own copy of the output
    int nsplit, views_per_split;
    size_t split_stride;                    // floats between the partial outputs of consecutive splits
};

// 8 (x) x 16 (y) voxel columns per CTA; a warp covers 8 x 4 columns of one plane: compact on the detector, so its
// lanes walk similar (iu, iv) ranges
#define ADJ_BX 8
#define ADJ_BY 16

// column-walk kernel (cbct_adjoint_column.cu): returns CBCT_OK after launching, or 1 if this geometry / channel block
// is not one it serves (the caller then takes the voxel kernel).  CB channels starting at sinoI / vol.
// `partial` (nsplit > 1): workspace of nsplit * CB * nx * ny * nz floats for the partial outputs of the view groups.
// CI = 4: sinoI points at channel-interleaved groups of 4 (NR = 1 only; CB = 4, or 8 with NM = 1), else CI = 1.
int cbct_launch_adjoint_column(cbct_geom *g, AdjGeom &G, int NR, int NM, int CB, int CI, const float *sinoI, float *vol,
                               size_t sstride, size_t vstride, int vol_z_origin, float *partial, int nsplit,
                               cudaStream_t st);
// out[c][e] = sum_s partial[s][c][e], fixed order (cbct_adjoint.cu)
int cbct_launch_reduce_splits(cbct_geom *g, const float *partial, float *out, size_t nvox, int cb, int nsplit,
                              size_t out_cstride, cudaStream_t st);
