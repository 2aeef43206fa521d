// cbct_geom.cu -- A1: geometry module (host side) of libcbct.so.
// Validates the descriptor, precomputes per-view (cos phi, sin phi) in fp64,
// converts every length to voxel units, plans z-slabs, and counts in-support
// samples analytically.  Geometry: PAPER.md:61; readings R2-R7 (DESIGN.md s.3).
#include <math.h>
#include <string.h>

#include <new>
#include <string>

#include "cbct_internal.h"

static thread_local std::string g_last_cuda_error;

void cbct_set_cuda_error(cudaError_t e, const char *what)
{
    g_last_cuda_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " in " + what;
    (void)cudaGetLastError();  // clear the sticky-less error state
}

extern "C" const char *cbct_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

extern "C" const char *cbct_status_string(int status)
{
    switch (status) {
        case CBCT_OK: return "CBCT_OK";
        case CBCT_ERR_INVALID_ARG: return "CBCT_ERR_INVALID_ARG: bad pointer, size or geometry";
        case CBCT_ERR_UNSUPPORTED: return "CBCT_ERR_UNSUPPORTED: configuration outside library limits";
        case CBCT_ERR_CUDA: return "CBCT_ERR_CUDA: a CUDA runtime call failed (see cbct_last_cuda_error)";
        case CBCT_ERR_NOMEM: return "CBCT_ERR_NOMEM: allocation failed or work-set cap too small";
        default: return "CBCT: unknown status";
    }
}

extern "C" int cbct_geom_create(const cbct_geom_desc *d, cbct_geom **out)
{
    if (!d || !out) return CBCT_ERR_INVALID_ARG;
    *out = nullptr;
    if (!(d->sid_mm > 0.0) || !(d->sdd_mm > d->sid_mm)) return CBCT_ERR_INVALID_ARG;
    if (d->n_views < 1 || d->det_nu < 1 || d->det_nv < 1) return CBCT_ERR_INVALID_ARG;
    if (d->vol_nx < 1 || d->vol_ny < 1 || d->vol_nz < 1) return CBCT_ERR_INVALID_ARG;
    if (!(d->det_du_mm > 0.0) || !(d->det_dv_mm > 0.0) || !(d->vox_mm > 0.0)) return CBCT_ERR_INVALID_ARG;
    if (!(d->step_vox > 0.0) || !(d->step_vox <= 1.0)) return CBCT_ERR_INVALID_ARG;
    if (!isfinite(d->det_off_u_mm) || !isfinite(d->det_off_v_mm) || !isfinite(d->vol_cx_mm) ||
        !isfinite(d->vol_cy_mm) || !isfinite(d->vol_cz_mm))
        return CBCT_ERR_INVALID_ARG;
    if (d->n_views > CBCT_MAX_VIEWS) return CBCT_ERR_UNSUPPORTED;
    if ((int64_t)d->vol_nx + 2 * CBCT_PAD > 4096 || (int64_t)d->vol_ny + 2 * CBCT_PAD > 4096 ||
        (int64_t)d->vol_nz + 2 * CBCT_PAD > 4096 || d->det_nu > 8192 || d->det_nv > 8192)
        return CBCT_ERR_UNSUPPORTED;
    // The sphere bounding the zero-extended volume (grid + one voxel of fade)
    // must lie strictly inside the source orbit: no sample behind the source
    // and U > 0 for every voxel of the FDK backprojection.
    double hx = 0.5 * (d->vol_nx + 1) * d->vox_mm, hy = 0.5 * (d->vol_ny + 1) * d->vox_mm,
           hz = 0.5 * (d->vol_nz + 1) * d->vox_mm;
    double rc = sqrt(d->vol_cx_mm * d->vol_cx_mm + d->vol_cy_mm * d->vol_cy_mm + d->vol_cz_mm * d->vol_cz_mm);
    double rbound = rc + sqrt(hx * hx + hy * hy + hz * hz);
    // (two voxels of clearance: the gather adjoint bounds its ray search with U - 1.5 voxels > 0)
    if (!(rbound + 2.0 * d->vox_mm < d->sid_mm)) return CBCT_ERR_INVALID_ARG;
    // ... and strictly in front of the detector plane, so every in-support
    // sample has t_k < |p - s| (the forward sum stops at the detector).
    if (!(rbound < d->sdd_mm - d->sid_mm)) return CBCT_ERR_INVALID_ARG;

    cbct_geom *g = new (std::nothrow) cbct_geom();
    if (!g) return CBCT_ERR_NOMEM;
    g->d = *d;
    g->angles.resize(d->n_views);
    g->cosphi.resize(d->n_views);
    g->sinphi.resize(d->n_views);
    for (int i = 0; i < d->n_views; ++i) {
        double phi = d->angles_rad ? d->angles_rad[i] : 2.0 * M_PI * (double)i / (double)d->n_views;
        if (!isfinite(phi)) { delete g; return CBCT_ERR_INVALID_ARG; }
        g->angles[i] = phi;
        g->cosphi[i] = cos(phi);
        g->sinphi[i] = sin(phi);
    }
    g->d.angles_rad = g->angles.data();
    // Symmetries the gather adjoint exploits (cbct_adjoint.cu): a centred grid and
    // views i, i + n/R that differ by exactly 360/R degrees see the same geometry
    // up to a rotation of the grid; a volume and detector centred in z are
    // mirror-symmetric under z -> -z.
    auto views_rotate = [&](int R) {
        if (d->n_views % R) return false;
        const int nq = d->n_views / R;
        for (int r = 1; r < R; ++r) {
            const double cr = cos(2.0 * M_PI * r / R), sr = sin(2.0 * M_PI * r / R);
            for (int i = 0; i < nq; ++i) {
                double c = g->cosphi[i] * cr - g->sinphi[i] * sr, s = g->sinphi[i] * cr + g->cosphi[i] * sr;
                if (fabs(c - g->cosphi[i + r * nq]) > 1e-13 || fabs(s - g->sinphi[i + r * nq]) > 1e-13) return false;
            }
        }
        return true;
    };
    const bool centred_xy = d->vol_cx_mm == 0.0 && d->vol_cy_mm == 0.0;
    if (centred_xy && d->vol_nx == d->vol_ny && d->vol_nx % 2 == 0 && views_rotate(4)) g->sym_rot = 4;
    else if (centred_xy && d->vol_ny % 2 == 0 && views_rotate(2)) g->sym_rot = 2;
    else g->sym_rot = 1;
    g->sym_mirror_z = d->vol_cz_mm == 0.0 && d->det_off_v_mm == 0.0;
    *out = g;
    return CBCT_OK;
}

static void prof_clear(cbct_geom *g);

extern "C" int cbct_geom_destroy(cbct_geom *g)
{
    if (!g) return CBCT_ERR_INVALID_ARG;
    if (g->ws_vol || g->ws_sino || g->ws_sino2 || g->ws_stage || g->copy_stream || g->d_filter_tab || g->h2d_stream) {
        cudaDeviceSynchronize();
        cudaFree(g->ws_vol);
        cudaFree(g->ws_sino);
        cudaFree(g->ws_sino2);
        cudaFree(g->d_filter_tab);
        cudaFree(g->ws_stage);
        for (int i = 0; i < 4; ++i)
            if (g->ev[i]) cudaEventDestroy(g->ev[i]);
        prof_clear(g);
        if (g->copy_stream) cudaStreamDestroy(g->copy_stream);
        cudaFree(g->ws_blk_in);
        cudaFree(g->ws_blk_out);
        for (int i = 0; i < 7; ++i)
            if (g->ev_blk[i]) cudaEventDestroy(g->ev_blk[i]);
        if (g->h2d_stream) cudaStreamDestroy(g->h2d_stream);
        if (g->d2h_stream) cudaStreamDestroy(g->d2h_stream);
    }
    delete g;
    return CBCT_OK;
}

RayGeom cbct_make_raygeom(const cbct_geom *g, int z0, int z1)
{
    const cbct_geom_desc &d = g->d;
    RayGeom r;
    double h = d.vox_mm;
    r.sid = d.sid_mm / h;
    r.idd = (d.sdd_mm - d.sid_mm) / h;
    r.du = d.det_du_mm / h;
    r.dv = d.det_dv_mm / h;
    r.u0 = (-0.5 * (d.det_nu - 1) * d.det_du_mm + d.det_off_u_mm) / h;
    r.v0 = (-0.5 * (d.det_nv - 1) * d.det_dv_mm + d.det_off_v_mm) / h;
    r.cx = d.vol_cx_mm / h;
    r.cy = d.vol_cy_mm / h;
    r.cz = d.vol_cz_mm / h;
    r.step = d.step_vox;
    r.delta = d.step_vox * d.vox_mm;
    r.nu = d.det_nu; r.nv = d.det_nv;
    r.nx = d.vol_nx; r.ny = d.vol_ny; r.nz = d.vol_nz;
    r.z0 = z0; r.z1 = z1;
    r.px = (d.vol_nx + 2 * CBCT_PAD + 7) & ~7;  // row pitch: whole 128-byte lines of 8 float4 cells
    r.py = d.vol_ny + 2 * CBCT_PAD;
    r.pz = (z1 - z0) + 2 * CBCT_PAD;
    return r;
}

int cbct_padded_sino_pitch(const cbct_geom *g) { return (g->d.det_nu + 2 * CBCT_PAD + 3) & ~3; }
int cbct_padded_sino_rows(const cbct_geom *g) { return g->d.det_nv + 2 * CBCT_PAD; }

// Analytic in-support sample count, fp64, host.  For each ray the open
// t-interval where -1 < q < N holds on every axis is intersected with (0, L);
// the count is the number of lattice points t_k = (k + 1/2) step inside it.
extern "C" int cbct_geom_count_samples(const cbct_geom *gc, uint64_t *out)
{
    if (!gc || !out) return CBCT_ERR_INVALID_ARG;
    cbct_geom *g = const_cast<cbct_geom *>(gc);
    if (g->sample_count >= 0) { *out = (uint64_t)g->sample_count; return CBCT_OK; }
    RayGeom r = cbct_make_raygeom(g, 0, g->d.vol_nz);
    const double lo[3] = { r.cx - 0.5 * (r.nx - 1) - 1.0, r.cy - 0.5 * (r.ny - 1) - 1.0, r.cz - 0.5 * (r.nz - 1) - 1.0 };
    const double hi[3] = { lo[0] + r.nx + 1.0, lo[1] + r.ny + 1.0, lo[2] + r.nz + 1.0 };
    uint64_t total = 0;
    for (int i = 0; i < g->d.n_views; ++i) {
        double c = g->cosphi[i], s = g->sinphi[i];
        double S[3] = { r.sid * c, r.sid * s, 0.0 };
        for (int iv = 0; iv < r.nv; ++iv) {
            double v = r.v0 + iv * r.dv;
            for (int iu = 0; iu < r.nu; ++iu) {
                double u = r.u0 + iu * r.du;
                double D[3] = { -r.idd * c - u * s - S[0], -r.idd * s + u * c - S[1], v };
                double L = sqrt(D[0] * D[0] + D[1] * D[1] + D[2] * D[2]);
                double tmin = 0.0, tmax = L;
                bool hit = true;
                for (int a = 0; a < 3 && hit; ++a) {
                    double da = D[a] / L;
                    if (da == 0.0) {
                        hit = (S[a] > lo[a] && S[a] < hi[a]);
                    } else {
                        double t0 = (lo[a] - S[a]) / da, t1 = (hi[a] - S[a]) / da;
                        if (t0 > t1) { double t = t0; t0 = t1; t1 = t; }
                        if (t0 > tmin) tmin = t0;
                        if (t1 < tmax) tmax = t1;
                    }
                }
                if (!hit || !(tmin < tmax)) continue;
                // smallest k with t_k > tmin, largest k with t_k < tmax
                long kf = (long)floor(tmin / r.step - 0.5) + 1;
                long kl = (long)ceil(tmax / r.step - 0.5) - 1;
                if (kf < 0) kf = 0;
                if (kl >= kf) total += (uint64_t)(kl - kf + 1);
            }
        }
    }
    g->sample_count = (int64_t)total;
    *out = total;
    return CBCT_OK;
}

// z-slab plan (A5) of the forward projector: planes per slab so that two slab
// buffers of all `channels` channels fit under max_workset_bytes.  A slab buffer
// holds the packed cells (16 B per padded cell: one per voxel and channel when quad-packed, one per voxel and
// group of 4 channels when channel-interleaved, cbct_fp.cu) plus the raw planes they
// are packed from when the caller's volume is in host memory (4 B per voxel;
// counted always, so the plan does not depend on where the volume lives).
// Returns planes per slab (nz when everything is resident) or <= 0 if not even
// one plane fits.
int cbct_plan_slab_planes(const cbct_geom *g, int channels)
{
    RayGeom r = cbct_make_raygeom(g, 0, g->d.vol_nz);
    uint64_t cap = g->d.max_workset_bytes;
    // groups of 4 channels share one channel-interleaved cell per voxel (row pitch px + 8); the rest are quad-packed
    // or, with the quarter-turn symmetry, stored as cells of their four rotated images (cbct_fp.cu)
    uint64_t packed_plane = (uint64_t)(channels / 4) * (uint64_t)(r.px + CBCT_ROW_SKEW) * r.py * 16u
                            + (uint64_t)(channels % 4) * (uint64_t)(g->sym_rot == 4 && r.nx == r.ny ? r.px + CBCT_ROW_SKEW : r.px) * r.py * 16u;
    uint64_t raw_plane = (uint64_t)r.nx * r.ny * 4u * (uint64_t)channels;
    if (cap == 0 || packed_plane * (uint64_t)r.pz + raw_plane * (uint64_t)r.nz <= cap) return g->d.vol_nz;
    int64_t planes = ((int64_t)(cap / 2) - (int64_t)(packed_plane * 2 * CBCT_PAD)) / (int64_t)(packed_plane + raw_plane);
    if (planes > g->d.vol_nz) planes = g->d.vol_nz;
    return (int)planes;
}

extern "C" int cbct_geom_num_slabs(const cbct_geom *g, int32_t channels, int32_t *out)
{
    if (!g || !out || channels < 1) return CBCT_ERR_INVALID_ARG;
    int planes = cbct_plan_slab_planes(g, channels);
    if (planes < 1) return CBCT_ERR_NOMEM;
    *out = (g->d.vol_nz + planes - 1) / planes;
    return CBCT_OK;
}

void cbct_prof_begin(cbct_geom *g, int kernel, cudaStream_t st)
{
    if (!g->profiling) return;
    cudaEvent_t a = nullptr, b = nullptr;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
    cudaEventRecord(a, st);
    g->prof[kernel].push_back(std::make_pair(a, b));
}

void cbct_prof_end(cbct_geom *g, int kernel, cudaStream_t st)
{
    if (!g->profiling || g->prof[kernel].empty()) return;
    cudaEventRecord(g->prof[kernel].back().second, st);
}

static void prof_clear(cbct_geom *g)
{
    for (int k = 0; k < 3; ++k) {
        for (auto &p : g->prof[k]) { cudaEventDestroy(p.first); cudaEventDestroy(p.second); }
        g->prof[k].clear();
    }
}

extern "C" int cbct_geom_profile(cbct_geom *g, int enable)
{
    if (!g) return CBCT_ERR_INVALID_ARG;
    if (enable) prof_clear(g);
    g->profiling = enable != 0;
    return CBCT_OK;
}

extern "C" int cbct_geom_profile_read(cbct_geom *g, int kernel, double *ms_total, uint64_t *launches)
{
    if (!g || kernel < 0 || kernel > 2 || !ms_total || !launches) return CBCT_ERR_INVALID_ARG;
    double total = 0.0;
    for (auto &p : g->prof[kernel]) {
        CBCT_CUDA_TRY(cudaEventSynchronize(p.second));
        float ms = 0.f;
        CBCT_CUDA_TRY(cudaEventElapsedTime(&ms, p.first, p.second));
        total += ms;
    }
    *ms_total = total;
    *launches = g->prof[kernel].size();
    return CBCT_OK;
}

extern "C" int cbct_geom_symmetry(const cbct_geom *g, int32_t *rotations, int32_t *mirror_z)
{
    if (!g || !rotations || !mirror_z) return CBCT_ERR_INVALID_ARG;
    *rotations = g->sym_rot;
    *mirror_z = g->sym_mirror_z ? 1 : 0;
    return CBCT_OK;
}

extern "C" int cbct_geom_launch_count(const cbct_geom *g, uint64_t *out)
{
    if (!g || !out) return CBCT_ERR_INVALID_ARG;
    *out = g->launches;
    return CBCT_OK;
}
