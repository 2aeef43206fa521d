/*
 * cbct.h -- C ABI of libcbct.so: circular-orbit cone-beam CT operators for
 * NVIDIA B200 (sm_100a), the data-parallel hot path of LIRE++
 * (arxiv 2512.21180; section/line citations refer to PAPER.md).
 *
 *   P   forward projector   PAPER.md:85-89 Eq. (5): P(mu)(t,u) = int_{L_{t,u}} mu(z) dz,
 *                           L_{t,u} the line from the source to detector element u at view t
 *   P*  backprojector       PAPER.md:89 (+ footnote :101): the Hermitian adjoint of P
 *   FDK backprojection      PAPER.md:157, :181 (Alg. 1 l.3), ref [9] :397 (Feldkamp)
 *   geometry                PAPER.md:61 (SID 1000 mm, isocentre-detector 536 mm,
 *                           115 mm lateral detector offset, 409.6 mm / 256^2 panel)
 *   multi-channel use       PAPER.md:167, :221, :227, :230 (Alg. 1 l.16-19)
 *   multi-scale use         PAPER.md:270 (one handle per scale / view subset)
 *   streaming               PAPER.md:165, :292 (data kept on the host, parts sent to the GPU)
 *   beyond the four core calls (SURVEY.md s.8(f) NEXT-1..3): the FDK_w front end and redundancy
 *   weight w, the field-of-view tensor V, Downsample /
 *   Upsample / ProjDown and the fused P x - y / P^T(w y) of Alg. 1 l.18-19
 *
 * The paper defines P only as a continuous integral; the discretisation is
 * the one BASELINE.json names (ray-driven, trilinear samples at a fixed step)
 * with the readings R1-R22 listed in DESIGN.md section 3.
 *
 * Conventions
 *   - World frame (mm): isocentre at the origin, rotation axis +z.  View i has
 *     angle phi_i; source s_i = SID (cos phi_i, sin phi_i, 0); detector centre
 *     -(SDD-SID)(cos phi_i, sin phi_i, 0); e_u = (-sin phi_i, cos phi_i, 0),
 *     e_v = (0,0,1).  Pixel (iv,iu) centre: u = (iu-(nu-1)/2) du + off_u,
 *     v = (iv-(nv-1)/2) dv + off_v.
 *   - Volume: voxel (iz,iy,ix) centre at c + (i-(N-1)/2) h per axis; zero
 *     outside the grid, trilinear interpolation fades to zero over the outer
 *     voxel (support -1 < q < N in index coordinates).
 *   - Layouts (fp32, C-contiguous): vol[C][nz][ny][nx] (x fastest),
 *     sino[C][n_views][nv][nu] (u fastest).
 *   - Every data pointer may be a DEVICE pointer or a HOST pointer (pinned or
 *     pageable); the library detects which with cudaPointerGetAttributes.
 *     Host buffers are staged through library-owned device workspace inside
 *     the call: without a work-set cap, as a pipeline over blocks of 1 to 4
 *     channels (H2D copy / kernels / D2H copy on three streams, joined back
 *     into `cuda_stream` before the call's work ends; the block widths follow
 *     the kernels' channel grouping, so single channels may round differently
 *     -- by fp32 summation order -- from the same call on device buffers);
 *     with a cap, by z-slabs (A5).
 *     A call with any pageable host buffer synchronises the stream before
 *     returning.
 *   - Outputs are OVERWRITTEN, never accumulated into.
 *   - Ownership: the caller owns all data buffers; the library owns the
 *     handle and its device workspace, freed by cbct_geom_destroy.
 *   - Asynchrony: with device pointers all work is enqueued on `cuda_stream`
 *     (a cudaStream_t cast to void*, NULL = legacy default stream) and the
 *     call returns without synchronising.  A handle carries mutable
 *     workspace: calls on one handle must be ordered on one stream at a time.
 *     The workspace grows (cudaFree + cudaMalloc, with a device
 *     synchronisation) only when a call needs more than any earlier call on
 *     the handle did; after one warm-up call of the same shape -- or
 *     cbct_geom_reserve -- device-pointer calls issue nothing but kernel
 *     launches and memsets on `cuda_stream`, so they may be captured into a
 *     CUDA graph (cudaStreamBeginCapture) and replayed.  A captured graph
 *     bakes in the workspace addresses: ANY later growth of the workspace
 *     (a call with more channels, the first call of another operator)
 *     invalidates graphs captured before it -- reserve for the largest call
 *     first.  A call that would have to grow the workspace while its stream
 *     is capturing returns CBCT_ERR_UNSUPPORTED and enqueues nothing; host
 *     buffers are refused during capture (their staging uses side streams).
 *   - Devices: the library launches on the CUDA device that is current in the calling thread; a handle's
 *     workspace belongs to the device that was current at its first compute call, so use one handle per
 *     device.  All device pointers of a call must belong to that device (the Python binding checks this and
 *     makes the tensors' device current for the call).
 *   - Errors: 0 on success, a negative cbct_status otherwise; nothing throws
 *     across the ABI.  There is NO CPU fallback: without a CUDA device every
 *     compute entry point returns CBCT_ERR_CUDA.
 */
#ifndef CBCT_H
#define CBCT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum cbct_status {
    CBCT_OK = 0,
    CBCT_ERR_INVALID_ARG = -1, /* NULL pointer, non-positive size, geometry that puts samples
                                  behind the source or beyond the detector, bad step      */
    CBCT_ERR_UNSUPPORTED = -2, /* e.g. more views than CBCT_MAX_VIEWS                      */
    CBCT_ERR_CUDA = -3,        /* a CUDA runtime call failed (cbct_last_cuda_error)        */
    CBCT_ERR_NOMEM = -4        /* host or device allocation failed, or the work-set cap
                                  is too small for even one slab                           */
} cbct_status;

#define CBCT_MAX_VIEWS 4096

typedef struct cbct_geom cbct_geom; /* opaque; owns host tables + device workspace */

/* Geometry descriptor (host memory, copied at create time).  Defaults of the
 * paper's scanner in comments. */
typedef struct cbct_geom_desc {
    double sid_mm;                /* source-isocentre distance                 1000       */
    double sdd_mm;                /* source-detector distance                  1536       */
    int32_t n_views;              /* 1..CBCT_MAX_VIEWS                         400..944   */
    const double *angles_rad;     /* n_views angles, or NULL => 2*pi*i/n_views            */
    int32_t det_nu, det_nv;       /* detector columns (lateral u), rows (axial v)  256    */
    double det_du_mm, det_dv_mm;  /* pixel pitch                               1.6        */
    double det_off_u_mm;          /* lateral offset along e_u (half-fan)       +115       */
    double det_off_v_mm;          /* axial offset along e_v                    0          */
    int32_t vol_nx, vol_ny, vol_nz; /* grid size                               256^3      */
    double vox_mm;                /* isotropic voxel pitch h                   2.0        */
    double vol_cx_mm, vol_cy_mm, vol_cz_mm; /* volume centre rel. to isocentre  0,0,0     */
    double step_vox;              /* ray step in voxel units, 0 < step <= 1    0.5        */
    uint64_t max_workset_bytes;   /* 0 = no cap; else cap on device bytes holding VOLUME
                                     data at once => z-slab streaming (A5).  It does not
                                     cap the sinogram side: a call keeps the sinogram of
                                     all its channels (when given as a host buffer) and one
                                     re-laid-out copy of it (view-interleaved for the
                                     adjoint, zero-bordered for FDK) resident beside the
                                     slabs: 2 x 4 B x channels x n_views x nv x nu, e.g.
                                     3.0 + 3.0 GB for 4 channels of 720 x 512 x 512
                                     (cbct_geom_workspace_bytes reports the total).       */
} cbct_geom_desc;

/* A1.  Validates `d`, precomputes the per-view tables (fp64 on the host,
 * passed to the kernels through constant memory) and returns a handle in
 * *out.  Needs no CUDA device (device workspace is allocated lazily by the
 * first compute call).  Requires sdd > sid, the sphere bounding the
 * zero-extended volume strictly between source and detector plane (with two
 * voxels of clearance on the source side), positive sizes and pitches,
 * 0 < step_vox <= 1. */
int cbct_geom_create(const cbct_geom_desc *d, cbct_geom **out);

/* Frees the handle, its tables and its device workspace (synchronises the device). */
int cbct_geom_destroy(cbct_geom *g);

/* A2.  sino[c,i,iv,iu] = Delta * sum_k T[vol_c](q(s_i + t_k d)),  t_k = (k+1/2) Delta,
 * Delta = step_vox * vox_mm, k over all samples between source and pixel, T the
 * zero-extended trilinear interpolant, d the unit vector source -> pixel centre.
 * vol: channels*nz*ny*nx floats (read), sino: channels*n_views*nv*nu floats (written).
 * Channels are independent.  Batching pays: groups of 4 channels share one re-laid-out copy of the volume and all
 * tap weights (and the backprojectors share their weights over up to 4 channels); a channel outside such a group
 * is projected through its four quarter-turn images when the geometry has that symmetry, else together with its
 * z-mirror image when volume and detector rows are centred in z.  So a channel's bits may
 * differ between a batched and a single-channel call by fp32 rounding (1e-6 .. 1e-5 of the result's scale, the
 * error either call has against an exact evaluation), never by more. */
int cbct_fp(const cbct_geom *g, const float *vol, float *sino, int32_t channels, void *cuda_stream);

/* A3.  The exact transpose of the matrix applied by cbct_fp (plain Euclidean
 * dot products): vol_c[j] = Delta * sum_{i,iv,iu,k} w(j; i,iv,iu,k) sino_c[i,iv,iu].
 * Floating-point summation order is unspecified (fp32 accumulation). */
int cbct_bp_adjoint(const cbct_geom *g, const float *sino, float *vol, int32_t channels, void *cuda_stream);

/* A4.  Backprojection stage of FDK for a flat detector, voxel-driven:
 * vol_c[z,y,x] = sum_i (SID/U_i)^2 * B[sino_c,i](fv, fu),  U_i = SID - (x cos phi_i + y sin phi_i),
 * u* = SDD (-x sin phi_i + y cos phi_i)/U_i, v* = SDD z/U_i, (fu,fv) their detector index
 * coordinates, B the zero-extended bilinear interpolant.  `sino` is the already
 * weighted + ramp-filtered projection data; no dphi/2 factor is applied. */
int cbct_bp_fdk(const cbct_geom *g, const float *sino, float *vol, int32_t channels, void *cuda_stream);

/* NEXT-1: the projection-domain front end of FDK_w (ref [9] :397;
 * readings R11, R12 in DESIGN.md s.3).  sino_out = dphi * a * ramp_u( w(u) * cos-weight * sino_in ), row by row,
 * with a = du SID/SDD, Kak-Slaney taps h[0] = 1/(4a^2), h[odd n] = -1/(pi^2 n^2 a^2), h[even n] = 0, cos-weight
 * SDD/sqrt(SDD^2+u^2+v^2) and dphi = 2 pi / n_views, so that cbct_bp_fdk(sino_out) is the reconstruction.
 * flags & CBCT_FILTER_REDUNDANCY: w(u) = redundancy weight of a laterally displaced detector (smooth sine
 * weighting; conjugate rays weigh 1 in total; see cbct_geom_redundancy_weights); otherwise w = 1/2.
 * DEVICE pointers only, sino_out != sino_in, det_nu <= 2048; enqueued on `cuda_stream`. */
#define CBCT_FILTER_REDUNDANCY 1
int cbct_fdk_filter(const cbct_geom *g, const float *sino_in, float *sino_out, int32_t channels, int32_t flags,
                    void *cuda_stream);

/* sino_out = w(u) * sino_in, the weighting of P*(w y).  DEVICE pointers; in place allowed. */
int cbct_redundancy_weight(const cbct_geom *g, const float *sino_in, float *sino_out, int32_t channels,
                           void *cuda_stream);

/* The det_nu redundancy weights w(u) in fp64 (host; needs no CUDA device). */
int cbct_geom_redundancy_weights(const cbct_geom *g, double *w_out);

/* NEXT-3: fusions on the hot path of Alg. 1.
 * cbct_fp_residual: sino = P vol - y, the argument of the Landweber term P*(P x - y); the subtraction happens in the
 * projector's epilogue (y: DEVICE sinogram of the same layout, y != sino).
 * cbct_bp_adjoint_weighted: vol = P^T (w(u) * sino), i.e. P*(w d) / P*(w y); the weighting is
 * fused into the adjoint's sinogram re-layout pass.  Otherwise as cbct_fp / cbct_bp_adjoint. */
int cbct_fp_residual(const cbct_geom *g, const float *vol, const float *y, float *sino, int32_t channels,
                     void *cuda_stream);
int cbct_bp_adjoint_weighted(const cbct_geom *g, const float *sino, float *vol, int32_t channels, void *cuda_stream);

/* NEXT-2.  Field-of-view tensor: vol_out[z,y,x] = (number of views in which the
 * centre of voxel (z,y,x) projects onto the panel's active area, -1/2 <= fu < nu-1/2 and -1/2 <= fv < nv-1/2) /
 * n_views (reading R21).  vol_out: nz*ny*nx floats, DEVICE pointer, overwritten. */
int cbct_fov(const cbct_geom *g, float *vol_out, void *cuda_stream);

/* Resampling operators of the multiscale scheme; plain arrays, DEVICE pointers, `n_outer` leading
 * items (channels).  cbct_downsample: average pooling by `factor` of in[n_outer][nz_in][ny_in][nx_in] (sizes must be
 * multiples of factor).  cbct_upsample: nearest upsampling, out[n_outer][nz_in f][ny_in f][nx_in f].
 * cbct_proj_down: keeps views 0, f, 2f, ... of in[n_outer][n_views_in][nv_in][nu_in] and average-pools the detector
 * by f: out[n_outer][ceil(n_views_in / f)][nv_in / f][nu_in / f]. */
int cbct_downsample(const float *in, float *out, int64_t n_outer, int32_t nz_in, int32_t ny_in, int32_t nx_in,
                    int32_t factor, void *cuda_stream);
int cbct_upsample(const float *in, float *out, int64_t n_outer, int32_t nz_in, int32_t ny_in, int32_t nx_in,
                  int32_t factor, void *cuda_stream);
int cbct_proj_down(const float *in, float *out, int64_t n_outer, int32_t n_views_in, int32_t nv_in, int32_t nu_in,
                   int32_t factor, void *cuda_stream);

/* Number of in-support samples of ONE channel: pairs (ray, k) with -1 < q < N
 * on every axis, counted analytically in fp64 on the host from the geometry
 * (the unit of the forward Gsamples/s metric).  Needs no CUDA device. */
int cbct_geom_count_samples(const cbct_geom *g, uint64_t *out);

/* Number of z-slabs the streaming path (A5) uses for `channels` channels
 * (1 = everything resident).  Needs no CUDA device. */
int cbct_geom_num_slabs(const cbct_geom *g, int32_t channels, int32_t *out);

/* Symmetries of the geometry that the kernels exploit (weights of symmetric voxel / view pairs are equal):
 * *rotations = 4, 2 or 1 -- views i and i + n_views / rotations see the (centred, for 4: square) grid rotated by
 * 360 / rotations degrees; *mirror_z = 1 if volume and detector rows are centred in z.  Needs no CUDA device. */
int cbct_geom_symmetry(const cbct_geom *g, int32_t *rotations, int32_t *mirror_z);

/* Device bytes of workspace the handle owns right now (packed slabs / staging, sinogram copies, tables). */
int cbct_geom_workspace_bytes(const cbct_geom *g, uint64_t *out);

/* Allocates, up front, all the workspace that device-pointer calls of cbct_fp / cbct_bp_adjoint(_weighted) /
 * cbct_bp_fdk / cbct_fdk_filter with up to `channels` channels need, so that they neither allocate nor
 * synchronise afterwards (CUDA-graph capture; flat memory).  Synchronises the device if it has to grow. */
int cbct_geom_reserve(cbct_geom *g, int32_t channels);

/* Plane ranges of the backprojectors: the shard a rank owns when one volume is split over GPUs (SURVEY.md
 * s.8(e) item 2: view-sharded cbct_fp, one all-gather of the sinogram, plane-sharded backprojection).
 * DEVICE pointers.  out[c] receives planes [z0, z1) of channel c of what cbct_bp_adjoint / cbct_bp_fdk would
 * write (the same terms; fp32 summation order, hence the last bits, may differ from the whole-volume call, which
 * pairs planes and splits views differently on some grids).  mirror_pair != 0 (only for geometries symmetric under z -> -z: vol_cz_mm = 0,
 * det_off_v_mm = 0; needs z1 <= ceil(nz / 2)): out[c] holds [z0, z1) followed by the mirror images
 * [nz - z1 + skip, nz - z0) in ascending order, skip = 1 if the range contains the middle plane of an odd nz
 * (its own image), else 0 -- 2 (z1 - z0) - skip planes per channel; the pair shares every weight, as in the
 * whole-volume call. */
int cbct_bp_adjoint_slab(const cbct_geom *g, const float *sino, float *out, int32_t channels, int32_t z0, int32_t z1,
                         int32_t mirror_pair, void *cuda_stream);
int cbct_bp_fdk_slab(const cbct_geom *g, const float *sino, float *out, int32_t channels, int32_t z0, int32_t z1,
                     int32_t mirror_pair, void *cuda_stream);

/* cbct_bp_fdk for callers that may not allocate (code under CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same two kernels as cbct_bp_fdk with DEVICE pointers (the result is
 * the same bit for bit), but the kernel's scratch -- the zero-bordered, record-interleaved copy of the sinogram --
 * lives in a file-scope device array of CBCT_STATIC_SCRATCH_BYTES that every GPU which loads the library holds
 * until the process exits.  The call makes no cudaMalloc / cudaFree, creates no stream or event and does not
 * synchronise; it enqueues on `cuda_stream` of the current device.  sino: [channels][n_views][det_nv][det_nu],
 * vol: [channels][nz][ny][nx], both DEVICE pointers owned by the caller (host pointers: CBCT_ERR_INVALID_ARG).
 * A geometry / channel count whose padded sinogram (about 4 x, with two-fold view symmetry 1 x, the sinogram's
 * bytes) exceeds the array returns CBCT_ERR_UNSUPPORTED, with the two sizes in cbct_last_cuda_error, and enqueues
 * nothing; so does a handle with cbct_geom_profile switched on.  max_workset_bytes is not consulted.
 * ONE array per device serves every handle and every call: it keeps the last call's contents (nothing needs
 * clearing: each call rewrites the region it reads, zero border included), and calls that overlap on the GPU
 * (two streams, two threads) RACE on it -- the caller serialises them.
 * cbct_static_scratch_setup resolves the array's device address for the CURRENT device (cbct_bp_fdk_static does
 * the same on its first call per device); call it once per device outside stream capture. */
#define CBCT_STATIC_SCRATCH_BYTES (32u << 20)
int cbct_static_scratch_setup(void);
int cbct_bp_fdk_static(const cbct_geom *g, const float *sino, float *vol, int32_t channels, void *cuda_stream);

/* Kernels launched by this handle since creation (for bench.py's gpu_launches). */
int cbct_geom_launch_count(const cbct_geom *g, uint64_t *out);

/* Per-kernel device timing for roofline reports.  cbct_geom_profile(g, 1) clears the
 * records and makes every later launch of the three main kernels record a CUDA-event
 * pair on the stream it is launched on; cbct_geom_profile(g, 0) stops recording.
 * cbct_geom_profile_read waits for the recorded events and returns, for `kernel`
 * (CBCT_KERNEL_FP / _ADJOINT / _FDK), the summed launch durations in ms and the launch count. */
#define CBCT_KERNEL_FP 0
#define CBCT_KERNEL_ADJOINT 1
#define CBCT_KERNEL_FDK 2
int cbct_geom_profile(cbct_geom *g, int enable);
int cbct_geom_profile_read(cbct_geom *g, int kernel, double *ms_total, uint64_t *launches);

/* Static description of a status code. */
/* NEXT-4: pointwise steps of the polychromatic primary model, DEVICE pointers.
 * cbct_water_bone, Eq. (3)-(4): rho_w[i], rho_b[i] from the modified CT number rho_hat[i] = 0.001 HU + 1
 *   rho_w = 0 (r < tau0), r (r < tau1), tau1 (tau2 - r)/(tau2 - tau1) (r < tau2), 0 otherwise;
 *   rho_b = 0 (r < tau1), kappa_b tau2 (r - tau1)/(tau2 - tau1) (r < tau2), kappa_b r otherwise.
 * The paper's constants are tau1 = 1.2, tau2 = 1.6, kappa_b = 0.409; it does not print tau0 (reading R23: the
 * caller's, 0 keeps all soft tissue).  n elements each; outputs overwritten; needs tau0 <= tau1 < tau2.
 * cbct_polychromatic_primary, Eq. (6) without the Poisson draw (its mean):
 *   out[q][p] = sum_e resp[e] i0[e][p] exp(-(mu_w[e] pw[q][p] + mu_b[e] pb[q][p])),
 * pw, pb = cbct_fp of rho_w, rho_b ([n_views][n_pix], mm), i0: [n_bins][n_pix] unattenuated counts per energy bin and
 * detector element, mu_w / mu_b / resp: HOST arrays of n_bins (<= 32) doubles (attenuation per unit relative
 * density in 1/mm; detector response), read before the call returns. */
int cbct_water_bone(const float *rho_hat, float *rho_w, float *rho_b, int64_t n, double tau0, double tau1, double tau2,
                    double kappa_b, void *cuda_stream);
int cbct_polychromatic_primary(const float *pw, const float *pb, const float *i0, const double *mu_w,
                               const double *mu_b, const double *resp, int32_t n_bins, int64_t n_views, int64_t n_pix,
                               float *out, void *cuda_stream);

const char *cbct_status_string(int status);

/* Text of the last CUDA error seen by the calling thread ("" if none). */
const char *cbct_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CBCT_H */
