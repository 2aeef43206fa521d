/*
 * cbct_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the circular-orbit cone-beam operators of
 * LIRE++ (arxiv 2512.21180).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
 * code, header, table or helper with the CUDA path under
 * paper_2512_21180_b200/csrc/.
 *
 * What the paper fixes:
 *   - P is the line integral along the line from the source to detector
 *     element u at time (view) t              (Eq. 5)
 *   - P* is its Hermitian adjoint             (footnote :101)
 *   - geometry: circular orbit, full 2*pi, SID 1000 mm, isocentre-detector
 *     536 mm, detector laterally offset "in the direction of rotation",
 *     flat square panel
 *   - FDK = Feldkamp analytic reconstruction  (ref [9] :397)
 * What the paper leaves open (discretisation) is fixed by the readings
 * R1..R11 of SURVEY.md section 8(c), restated in DESIGN.md section 3:
 *   R1 ray-driven, one ray per pixel centre, trilinear, fixed step
 *   R2 step = step_vox * voxel pitch (0.5 voxel in every config)
 *   R3 midpoint lattice measured from the SOURCE: t_k = (k + 1/2) * Delta
 *   R4 volume is zero outside the grid; trilinear interpolation fades
 *      linearly to zero over the outer voxel (support -1 < q < N per axis)
 *   R5 cell-centred voxel grid, R6 pixel-centre formula + offset sign,
 *   R7 phi_i = 2*pi*i/n_views, R8 adjoint = plain matrix transpose,
 *   R9-R11 FDK backprojection stage = sum_i (SID/U)^2 * bilinear(q_i)(u*,v*).
 *
 * Every function follows its definition step by step, in the paper's /
 * SURVEY's notation, with no blocking, fusion or reordering.  The only
 * shortcut is the conservative k-range clip in ray_k_range(), which skips
 * samples that are provably outside the support (value exactly zero); the
 * `clip` flag turns it off so tests can pin that it changes nothing.
 *
 * Pins (tests/test_oracle_pins.py): P1 ball chords, P2 ellipsoid sinogram
 * convergence, P3 Gaussian blob, P4 adjoint identity, P5 explicit 8^3 matrix
 * transpose, P6 four-fold view symmetry, P7 all-ones cube, P8 linearity,
 * P9 slab decomposition, P10 strided views, P11 FDK weight-sum closed form,
 * P12 end-to-end FDK of an analytic ball.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct oracle_geom {
    double sid_mm, sdd_mm;          /* source-isocentre, source-detector distance   */
    int32_t n_views;                /* number of views                               */
    const double *angles_rad;       /* n_views angles, or NULL => 2*pi*i/n_views (R7) */
    int32_t det_nu, det_nv;         /* detector columns (u, lateral), rows (v, axial) */
    double det_du_mm, det_dv_mm;    /* pixel pitch                                   */
    double det_off_u_mm, det_off_v_mm; /* detector centre offset along e_u, e_v (R6) */
    int32_t vol_nx, vol_ny, vol_nz; /* grid size                                     */
    double vox_mm;                  /* isotropic voxel pitch h                       */
    double vol_cx_mm, vol_cy_mm, vol_cz_mm; /* volume centre rel. to isocentre (R5)  */
    double step_vox;                /* ray step in voxel units (R2)                  */
} oracle_geom;

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static double view_angle(const oracle_geom *g, int i)
{
    if (g->angles_rad) return g->angles_rad[i];
    return 2.0 * M_PI * (double)i / (double)g->n_views; /* R7 */
}

/* Zero-extended trilinear interpolation T[f](q) (R4).  q = (qx,qy,qz) in index
 * coordinates; f[iz][iy][ix], x fastest; f = 0 at any index outside the grid. */
static double vox_or_zero(const double *f, int nx, int ny, int nz, long ix, long iy, long iz)
{
    if (ix < 0 || iy < 0 || iz < 0 || ix >= nx || iy >= ny || iz >= nz) return 0.0;
    return f[((size_t)iz * ny + iy) * nx + ix];
}

static double trilinear(const double *f, int nx, int ny, int nz, double qx, double qy, double qz)
{
    double fx = floor(qx), fy = floor(qy), fz = floor(qz);
    long jx = (long)fx, jy = (long)fy, jz = (long)fz;
    double ax = qx - fx, ay = qy - fy, az = qz - fz;
    double acc = 0.0;
    for (int dz = 0; dz < 2; ++dz)
        for (int dy = 0; dy < 2; ++dy)
            for (int dx = 0; dx < 2; ++dx) {
                double w = (dx ? ax : 1.0 - ax) * (dy ? ay : 1.0 - ay) * (dz ? az : 1.0 - az);
                acc += w * vox_or_zero(f, nx, ny, nz, jx + dx, jy + dy, jz + dz);
            }
    return acc;
}

/* Ray of view i through the centre of pixel (iv, iu):
 * source s, unit direction d, length L = |p - s|   (world mm; R6). */
static void ray_setup(const oracle_geom *g, int i, int iv, int iu, double s[3], double d[3], double *L)
{
    double phi = view_angle(g, i);
    double c = cos(phi), sn = sin(phi);
    double u = ((double)iu - 0.5 * (g->det_nu - 1)) * g->det_du_mm + g->det_off_u_mm;
    double v = ((double)iv - 0.5 * (g->det_nv - 1)) * g->det_dv_mm + g->det_off_v_mm;
    double idd = g->sdd_mm - g->sid_mm; /* isocentre-detector distance */
    s[0] = g->sid_mm * c;
    s[1] = g->sid_mm * sn;
    s[2] = 0.0;
    /* p = c_i + u e_u + v e_v,  c_i = -idd (cos,sin,0), e_u = (-sin,cos,0), e_v = (0,0,1) */
    double p[3] = { -idd * c - u * sn, -idd * sn + u * c, v };
    double dx = p[0] - s[0], dy = p[1] - s[1], dz = p[2] - s[2];
    double len = sqrt(dx * dx + dy * dy + dz * dz);
    d[0] = dx / len; d[1] = dy / len; d[2] = dz / len;
    *L = len;
}

/* world mm -> index coordinates (R5) */
static void world_to_index(const oracle_geom *g, const double x[3], double q[3])
{
    q[0] = (x[0] - g->vol_cx_mm) / g->vox_mm + 0.5 * (g->vol_nx - 1);
    q[1] = (x[1] - g->vol_cy_mm) / g->vox_mm + 0.5 * (g->vol_ny - 1);
    q[2] = (x[2] - g->vol_cz_mm) / g->vox_mm + 0.5 * (g->vol_nz - 1);
}

/* k-range [k0, k1) to visit.  Without clip: every k with t_k < L.  With clip:
 * the slab intersection of the ray with the box q in [-1, N]^3 (the closure of
 * the support), widened by one sample on each side -- a superset of every
 * sample whose interpolated value can be non-zero. */
static void ray_k_range(const oracle_geom *g, const double s[3], const double d[3], double L,
                        int clip, long *k0, long *k1)
{
    double delta = g->step_vox * g->vox_mm;
    /* all k >= 0 with (k + 1/2) delta < L */
    long kend = (long)ceil(L / delta - 0.5);
    if (kend < 0) kend = 0;
    while ((kend + 0.5) * delta < L) ++kend;
    while (kend > 0 && (kend - 1 + 0.5) * delta >= L) --kend;
    *k0 = 0; *k1 = kend;
    if (!clip) return;
    double tmin = 0.0, tmax = L;
    const double ctr[3] = { g->vol_cx_mm, g->vol_cy_mm, g->vol_cz_mm };
    const int n[3] = { g->vol_nx, g->vol_ny, g->vol_nz };
    for (int a = 0; a < 3; ++a) {
        /* world coordinate of index -1 and index N on this axis */
        double lo = ctr[a] + (-1.0 - 0.5 * (n[a] - 1)) * g->vox_mm;
        double hi = ctr[a] + ((double)n[a] - 0.5 * (n[a] - 1)) * g->vox_mm;
        if (fabs(d[a]) < 1e-300) {
            if (s[a] <= lo || s[a] >= hi) { *k0 = 0; *k1 = 0; return; }
        } else {
            double t0 = (lo - s[a]) / d[a], t1 = (hi - s[a]) / d[a];
            if (t0 > t1) { double tt = t0; t0 = t1; t1 = tt; }
            if (t0 > tmin) tmin = t0;
            if (t1 < tmax) tmax = t1;
        }
    }
    if (tmin >= tmax) { *k0 = 0; *k1 = 0; return; }
    long a0 = (long)floor(tmin / delta - 0.5) - 1;
    long a1 = (long)ceil(tmax / delta - 0.5) + 2;
    if (a0 < 0) a0 = 0;
    if (a1 > kend) a1 = kend;
    if (a1 < a0) a1 = a0;
    *k0 = a0; *k1 = a1;
}

/* One ray of the forward projector:  Delta * sum_k T[f](q(s + t_k d)). */
static double fp_ray(const oracle_geom *g, const double *f, int i, int iv, int iu, int clip)
{
    double s[3], d[3], L;
    ray_setup(g, i, iv, iu, s, d, &L);
    long k0, k1;
    ray_k_range(g, s, d, L, clip, &k0, &k1);
    double delta = g->step_vox * g->vox_mm;
    double acc = 0.0;
    for (long k = k0; k < k1; ++k) {
        double t = ((double)k + 0.5) * delta; /* R3 */
        double x[3] = { s[0] + t * d[0], s[1] + t * d[1], s[2] + t * d[2] };
        double q[3];
        world_to_index(g, x, q);
        acc += trilinear(f, g->vol_nx, g->vol_ny, g->vol_nz, q[0], q[1], q[2]);
    }
    return delta * acc;
}

/* A2 forward projection.  vol[C][nz][ny][nx] -> sino[C][n_views][nv][nu] (overwritten). */
int oracle_fp(const oracle_geom *g, const double *vol, double *sino, int channels, int clip)
{
    size_t nvol = (size_t)g->vol_nx * g->vol_ny * g->vol_nz;
    size_t nsino = (size_t)g->n_views * g->det_nv * g->det_nu;
    for (int c = 0; c < channels; ++c) {
        const double *f = vol + c * nvol;
        double *y = sino + c * nsino;
        long nrows = (long)g->n_views * g->det_nv;
#pragma omp parallel for schedule(dynamic, 4)
        for (long row = 0; row < nrows; ++row) {
            int i = (int)(row / g->det_nv), iv = (int)(row % g->det_nv);
            for (int iu = 0; iu < g->det_nu; ++iu)
                y[(size_t)row * g->det_nu + iu] = fp_ray(g, f, i, iv, iu, clip);
        }
    }
    return 0;
}

/* Forward projection of selected rays only (sampled parity at full sizes).
 * ray_idx[r] = flat index (i * nv + iv) * nu + iu;  out[c * n_rays + r]. */
int oracle_fp_rays(const oracle_geom *g, const double *vol, int channels,
                   const int64_t *ray_idx, int64_t n_rays, double *out)
{
    size_t nvol = (size_t)g->vol_nx * g->vol_ny * g->vol_nz;
    for (int c = 0; c < channels; ++c) {
        const double *f = vol + c * nvol;
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t r = 0; r < n_rays; ++r) {
            int64_t idx = ray_idx[r];
            int iu = (int)(idx % g->det_nu);
            int iv = (int)((idx / g->det_nu) % g->det_nv);
            int i = (int)(idx / ((int64_t)g->det_nu * g->det_nv));
            out[(size_t)c * n_rays + r] = fp_ray(g, f, i, iv, iu, 1);
        }
    }
    return 0;
}

/* Number of in-support samples: (ray, k) with -1 < q < N on every axis. */
int64_t oracle_count_samples(const oracle_geom *g, int clip)
{
    int64_t total = 0;
    long nrows = (long)g->n_views * g->det_nv;
    double delta = g->step_vox * g->vox_mm;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : total)
    for (long row = 0; row < nrows; ++row) {
        int i = (int)(row / g->det_nv), iv = (int)(row % g->det_nv);
        for (int iu = 0; iu < g->det_nu; ++iu) {
            double s[3], d[3], L;
            ray_setup(g, i, iv, iu, s, d, &L);
            long k0, k1;
            ray_k_range(g, s, d, L, clip, &k0, &k1);
            for (long k = k0; k < k1; ++k) {
                double t = ((double)k + 0.5) * delta;
                double x[3] = { s[0] + t * d[0], s[1] + t * d[1], s[2] + t * d[2] };
                double q[3];
                world_to_index(g, x, q);
                if (q[0] > -1.0 && q[0] < g->vol_nx && q[1] > -1.0 && q[1] < g->vol_ny &&
                    q[2] > -1.0 && q[2] < g->vol_nz)
                    ++total;
            }
        }
    }
    return total;
}

/* ------------------------------------------------------------------------- */
/* A3 matched adjoint: the transpose of exactly the matrix applied by
 * oracle_fp (R8: plain Euclidean dot products, no L2 weights).  For every
 * (view, pixel, k) and each of the 8 taps that falls inside the grid:
 *     vol[j + delta] += Delta * weight_delta * sino[view, pixel]. */
static void adjoint_ray(const oracle_geom *g, double *f, double yval, int i, int iv, int iu, int clip)
{
    double s[3], d[3], L;
    ray_setup(g, i, iv, iu, s, d, &L);
    long k0, k1;
    ray_k_range(g, s, d, L, clip, &k0, &k1);
    double delta = g->step_vox * g->vox_mm;
    const int nx = g->vol_nx, ny = g->vol_ny, nz = g->vol_nz;
    for (long k = k0; k < k1; ++k) {
        double t = ((double)k + 0.5) * delta;
        double x[3] = { s[0] + t * d[0], s[1] + t * d[1], s[2] + t * d[2] };
        double q[3];
        world_to_index(g, x, q);
        double fx = floor(q[0]), fy = floor(q[1]), fz = floor(q[2]);
        long jx = (long)fx, jy = (long)fy, jz = (long)fz;
        double ax = q[0] - fx, ay = q[1] - fy, az = q[2] - fz;
        for (int dz = 0; dz < 2; ++dz)
            for (int dy = 0; dy < 2; ++dy)
                for (int dx = 0; dx < 2; ++dx) {
                    long ix = jx + dx, iy = jy + dy, iz = jz + dz;
                    if (ix < 0 || iy < 0 || iz < 0 || ix >= nx || iy >= ny || iz >= nz) continue;
                    double w = (dx ? ax : 1.0 - ax) * (dy ? ay : 1.0 - ay) * (dz ? az : 1.0 - az);
                    f[((size_t)iz * ny + iy) * nx + ix] += delta * w * yval;
                }
    }
}

/* sino[C][n_views][nv][nu] -> vol[C][nz][ny][nx] (overwritten).
 * Views are split statically over threads, each thread scatters into a private
 * fp64 volume, and the private volumes are summed in thread order. */
int oracle_bp_adjoint(const oracle_geom *g, const double *sino, double *vol, int channels, int clip)
{
    size_t nvol = (size_t)g->vol_nx * g->vol_ny * g->vol_nz;
    size_t nsino = (size_t)g->n_views * g->det_nv * g->det_nu;
    int nthreads = oracle_max_threads();
    size_t cap = ((size_t)4 << 30) / (nvol * sizeof(double)); /* <= 4 GiB of private volumes */
    if (cap < 1) cap = 1;
    if ((size_t)nthreads > cap) nthreads = (int)cap;
    if (nthreads > g->n_views) nthreads = g->n_views > 0 ? g->n_views : 1;
    double *priv = (double *)malloc((size_t)nthreads * nvol * sizeof(double));
    if (!priv) return -1;
    for (int c = 0; c < channels; ++c) {
        const double *y = sino + c * nsino;
        double *f = vol + c * nvol;
        memset(priv, 0, (size_t)nthreads * nvol * sizeof(double));
#pragma omp parallel num_threads(nthreads)
        {
#ifdef _OPENMP
            int tid = omp_get_thread_num(), nt = omp_get_num_threads();
#else
            int tid = 0, nt = 1;
#endif
            double *mine = priv + (size_t)tid * nvol;
            for (int i = tid; i < g->n_views; i += nt)
                for (int iv = 0; iv < g->det_nv; ++iv)
                    for (int iu = 0; iu < g->det_nu; ++iu) {
                        double yv = y[((size_t)i * g->det_nv + iv) * g->det_nu + iu];
                        if (yv != 0.0) adjoint_ray(g, mine, yv, i, iv, iu, clip);
                    }
        }
#pragma omp parallel for schedule(static)
        for (long p = 0; p < (long)nvol; ++p) {
            double acc = 0.0;
            for (int t = 0; t < nthreads; ++t) acc += priv[(size_t)t * nvol + p];
            f[p] = acc;
        }
    }
    free(priv);
    return 0;
}

/* Adjoint at selected voxels only (sampled parity at full sizes).  For voxel
 * p the rays that can touch its tent support (the cube p +- 1 voxel) lie
 * inside the detector bounding box of the cube's 8 projected corners (the
 * perspective image of a convex set is inside the hull of its projected
 * vertices); widened by one pixel each side.  Every such ray is marched and
 * only the weight landing on p is kept.  tests pin this against the full
 * oracle_bp_adjoint on small grids.
 * vox_idx[r] = flat (iz * ny + iy) * nx + ix;  out[c * n_vox + r]. */
int oracle_bp_adjoint_voxels(const oracle_geom *g, const double *sino, int channels,
                             const int64_t *vox_idx, int64_t n_vox, double *out)
{
    size_t nsino = (size_t)g->n_views * g->det_nv * g->det_nu;
    const int nx = g->vol_nx, ny = g->vol_ny, nz = g->vol_nz;
    double delta = g->step_vox * g->vox_mm;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t r = 0; r < n_vox; ++r) {
        int64_t idx = vox_idx[r];
        long px = (long)(idx % nx), py = (long)((idx / nx) % ny), pz = (long)(idx / ((int64_t)nx * ny));
        for (int c = 0; c < channels; ++c) out[(size_t)c * n_vox + r] = 0.0;
        for (int i = 0; i < g->n_views; ++i) {
            double phi = view_angle(g, i), cs = cos(phi), sn = sin(phi);
            double umin = 1e300, umax = -1e300, vmin = 1e300, vmax = -1e300;
            for (int corner = 0; corner < 8; ++corner) {
                double qx = px + ((corner & 1) ? 1.0 : -1.0);
                double qy = py + ((corner & 2) ? 1.0 : -1.0);
                double qz = pz + ((corner & 4) ? 1.0 : -1.0);
                double x = g->vol_cx_mm + (qx - 0.5 * (nx - 1)) * g->vox_mm;
                double y = g->vol_cy_mm + (qy - 0.5 * (ny - 1)) * g->vox_mm;
                double z = g->vol_cz_mm + (qz - 0.5 * (nz - 1)) * g->vox_mm;
                double U = g->sid_mm - (x * cs + y * sn);
                double us = g->sdd_mm * (-x * sn + y * cs) / U;
                double vs = g->sdd_mm * z / U;
                double fu = (us - g->det_off_u_mm) / g->det_du_mm + 0.5 * (g->det_nu - 1);
                double fv = (vs - g->det_off_v_mm) / g->det_dv_mm + 0.5 * (g->det_nv - 1);
                if (fu < umin) umin = fu;
                if (fu > umax) umax = fu;
                if (fv < vmin) vmin = fv;
                if (fv > vmax) vmax = fv;
            }
            long iu0 = (long)floor(umin) - 1, iu1 = (long)ceil(umax) + 1;
            long iv0 = (long)floor(vmin) - 1, iv1 = (long)ceil(vmax) + 1;
            if (iu0 < 0) iu0 = 0;
            if (iv0 < 0) iv0 = 0;
            if (iu1 > g->det_nu - 1) iu1 = g->det_nu - 1;
            if (iv1 > g->det_nv - 1) iv1 = g->det_nv - 1;
            for (long iv = iv0; iv <= iv1; ++iv)
                for (long iu = iu0; iu <= iu1; ++iu) {
                    double s[3], d[3], L;
                    ray_setup(g, i, (int)iv, (int)iu, s, d, &L);
                    long k0, k1;
                    ray_k_range(g, s, d, L, 1, &k0, &k1);
                    double wsum = 0.0;
                    for (long k = k0; k < k1; ++k) {
                        double t = ((double)k + 0.5) * delta;
                        double x[3] = { s[0] + t * d[0], s[1] + t * d[1], s[2] + t * d[2] };
                        double q[3];
                        world_to_index(g, x, q);
                        double fx = floor(q[0]), fy = floor(q[1]), fz = floor(q[2]);
                        long jx = (long)fx, jy = (long)fy, jz = (long)fz;
                        double ax = q[0] - fx, ay = q[1] - fy, az = q[2] - fz;
                        for (int dz = 0; dz < 2; ++dz)
                            for (int dy = 0; dy < 2; ++dy)
                                for (int dx = 0; dx < 2; ++dx)
                                    if (jx + dx == px && jy + dy == py && jz + dz == pz)
                                        wsum += (dx ? ax : 1.0 - ax) * (dy ? ay : 1.0 - ay) *
                                                (dz ? az : 1.0 - az);
                    }
                    if (wsum != 0.0)
                        for (int c = 0; c < channels; ++c)
                            out[(size_t)c * n_vox + r] +=
                                delta * wsum *
                                sino[c * nsino + ((size_t)i * g->det_nv + iv) * g->det_nu + iu];
                }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* A4 FDK-weighted voxel-driven backprojection (R9-R11): the backprojection
 * stage of Feldkamp's algorithm (ref [9] PAPER.md:397) for
 * a flat detector.  For voxel centre (x,y,z) and view i:
 *   U  = SID - (x cos phi_i + y sin phi_i)
 *   u* = SDD (-x sin phi_i + y cos phi_i) / U,   v* = SDD z / U
 *   fu = (u* - off_u)/du + (nu-1)/2,             fv = (v* - off_v)/dv + (nv-1)/2
 *   vol += (SID/U)^2 * B[sino_i](fv, fu),  B = zero-extended bilinear (R10).
 * No ramp filter, cosine weight, redundancy weight or dphi/2 in here. */
static double pix_or_zero(const double *p, int nu, int nv, long iu, long iv)
{
    if (iu < 0 || iv < 0 || iu >= nu || iv >= nv) return 0.0;
    return p[(size_t)iv * nu + iu];
}

static double fdk_voxel(const oracle_geom *g, const double *y, long ix, long iy, long iz)
{
    double x = g->vol_cx_mm + ((double)ix - 0.5 * (g->vol_nx - 1)) * g->vox_mm;
    double yy = g->vol_cy_mm + ((double)iy - 0.5 * (g->vol_ny - 1)) * g->vox_mm;
    double z = g->vol_cz_mm + ((double)iz - 0.5 * (g->vol_nz - 1)) * g->vox_mm;
    size_t npix = (size_t)g->det_nv * g->det_nu;
    double acc = 0.0;
    for (int i = 0; i < g->n_views; ++i) {
        double phi = view_angle(g, i), cs = cos(phi), sn = sin(phi);
        double U = g->sid_mm - (x * cs + yy * sn);
        double us = g->sdd_mm * (-x * sn + yy * cs) / U;
        double vs = g->sdd_mm * z / U;
        double fu = (us - g->det_off_u_mm) / g->det_du_mm + 0.5 * (g->det_nu - 1);
        double fv = (vs - g->det_off_v_mm) / g->det_dv_mm + 0.5 * (g->det_nv - 1);
        double ffu = floor(fu), ffv = floor(fv);
        long ju = (long)ffu, jv = (long)ffv;
        double au = fu - ffu, av = fv - ffv;
        const double *p = y + (size_t)i * npix;
        double b = (1.0 - av) * ((1.0 - au) * pix_or_zero(p, g->det_nu, g->det_nv, ju, jv) +
                                 au * pix_or_zero(p, g->det_nu, g->det_nv, ju + 1, jv)) +
                   av * ((1.0 - au) * pix_or_zero(p, g->det_nu, g->det_nv, ju, jv + 1) +
                         au * pix_or_zero(p, g->det_nu, g->det_nv, ju + 1, jv + 1));
        double w = g->sid_mm / U;
        acc += w * w * b;
    }
    return acc;
}

int oracle_bp_fdk(const oracle_geom *g, const double *sino, double *vol, int channels)
{
    size_t nvol = (size_t)g->vol_nx * g->vol_ny * g->vol_nz;
    size_t nsino = (size_t)g->n_views * g->det_nv * g->det_nu;
    for (int c = 0; c < channels; ++c) {
        const double *y = sino + c * nsino;
        double *f = vol + c * nvol;
        long nrows = (long)g->vol_nz * g->vol_ny;
#pragma omp parallel for schedule(dynamic, 8)
        for (long row = 0; row < nrows; ++row) {
            long iz = row / g->vol_ny, iy = row % g->vol_ny;
            for (long ix = 0; ix < g->vol_nx; ++ix)
                f[(size_t)row * g->vol_nx + ix] = fdk_voxel(g, y, ix, iy, iz);
        }
    }
    return 0;
}

/* FDK backprojection at selected voxels (sampled parity at full sizes). */
int oracle_bp_fdk_voxels(const oracle_geom *g, const double *sino, int channels,
                         const int64_t *vox_idx, int64_t n_vox, double *out)
{
    size_t nsino = (size_t)g->n_views * g->det_nv * g->det_nu;
    const int nx = g->vol_nx, ny = g->vol_ny;
    for (int c = 0; c < channels; ++c) {
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t r = 0; r < n_vox; ++r) {
            int64_t idx = vox_idx[r];
            long ix = (long)(idx % nx), iy = (long)((idx / nx) % ny), iz = (long)(idx / ((int64_t)nx * ny));
            out[(size_t)c * n_vox + r] = fdk_voxel(g, sino + c * nsino, ix, iy, iz);
        }
    }
    return 0;
}
