/*
 * cbct_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the TV-regularised cone-beam CT forward-backward
 * splitting hot path of Jia, Lou, Li, Song, Jiang (arXiv 1002.3675).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call
 * it.  It shares no code with the CUDA path (paper_1002_3675_b200/csrc) and never
 * reads anything that path produced.
 *
 * Citations: P:<n> = /root/reference/PAPER.md line n; O<n>/Q<n> = SURVEY.md §8(c)
 * readings (every place the paper is silent is listed in DESIGN.md "Readings").
 *
 *   O0 geometry        P:63 "projects f onto an x-ray imager plane in a cone beam geometry"
 *   O1 projector       P:63, P:99  exact radiological path (length of segment ∩ voxel box)
 *   O2 backprojector   P:95  "P^T denotes a matrix transpose": literal scatter of O1
 *   O3/O4 TV           P:69 E1 = (1/V)||grad f||_1, smoothed by eps (Q6); P:93 gradient descent
 *
 *   NEXT-1 eq. 2     P:97-99  the paper's voxel-driven backprojector (oracle_backproject_eq2)
 *
 * Pins (tests/test_oracle_*.py): closed-form box chord (I1), brute-force dense matrix
 * on 8^3 and 6x8x4 (I2), analytic ellipsoid chords (I3), dot-product identity (I4), eq. 2
 * weight (I5), rot90 / z-flip symmetry (I6), TV invariants + finite differences (I7),
 * descent (I8, I9), dense-matrix FBS (I10), NNLS limit (I11), transfer identities (I12);
 * eq. 2: hand-worked weights and interpolation, a library interpolation routine on a tiny case,
 * convergence to (du dv / dV) P^T under refinement (test_oracle_eq2.py).
 * Parity unpinned BY THE PAPER (fixed by DESIGN.md, identical on both sides): the choice of
 * eps, omega, u0, the coarsening rule and prolongation weights (those live in fbs.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double sad, sdd;            /* source-axis, source-detector distance (L0), mm */
    int n_angles;
    const double *angles;       /* radians */
    int nu, nv;
    double du, dv;              /* detector pixel pitch, mm */
    int nx, ny, nz;
    double hx, hy, hz;          /* voxel size, mm */
    double off_u, off_v;        /* NEXT-3: in-plane shift of the detector panel, mm (0 = centred full-fan, Q14) */
} og_geom;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* O0: source S(theta) and pixel centre D(theta, iu, iv). */
static void ray_endpoints(const og_geom *g, int ia, int iv, int iu, double S[3], double D[3])
{
    double t = g->angles[ia], c = cos(t), s = sin(t);
    double uc = ((double)iu - 0.5 * (g->nu - 1)) * g->du + g->off_u;
    double vc = ((double)iv - 0.5 * (g->nv - 1)) * g->dv + g->off_v;
    S[0] = g->sad * c;  S[1] = g->sad * s;  S[2] = 0.0;
    D[0] = -(g->sdd - g->sad) * c + uc * (-s);
    D[1] = -(g->sdd - g->sad) * s + uc * c;
    D[2] = vc;
}

/*
 * O1.  All non-zero chords of the segment S->D through the voxel grid, Siddon's way:
 * the parameters alpha in [0,1] at which the segment crosses the x-, y- and z-planes of the
 * grid are three monotone sequences; merged, every consecutive pair bounds a piece that lies
 * in ONE voxel (found from the piece's midpoint); the chord is (d alpha) * |D - S|.
 * Plane parameters are always computed directly from the plane index (no running sums).
 * Returns the number of pieces written to idx[] (linear voxel index k*ny*nx + j*nx + i)
 * and len[] (mm).  Buffers need nx+ny+nz+4 entries.
 */
static int ray_chords(const og_geom *g, const double S[3], const double D[3], long *idx, double *len)
{
    const int n[3] = { g->nx, g->ny, g->nz };
    const double h[3] = { g->hx, g->hy, g->hz };
    double lo[3], d[3], L = 0.0;
    double amin = 0.0, amax = 1.0;
    int a;
    for (a = 0; a < 3; ++a) {
        lo[a] = -0.5 * n[a] * h[a];
        d[a] = D[a] - S[a];
        L += d[a] * d[a];
    }
    L = sqrt(L);
    for (a = 0; a < 3; ++a) {
        double hi = lo[a] + n[a] * h[a];
        if (d[a] != 0.0) {
            double a0 = (lo[a] - S[a]) / d[a], a1 = (hi - S[a]) / d[a];
            double lo_a = a0 < a1 ? a0 : a1, hi_a = a0 < a1 ? a1 : a0;
            if (lo_a > amin) amin = lo_a;
            if (hi_a < amax) amax = hi_a;
        } else if (S[a] < lo[a] || S[a] > hi) {
            return 0;                    /* parallel to this axis' planes and outside the slab (Q15) */
        }
    }
    if (!(amin < amax)) return 0;         /* misses the volume (Q15) */

    /* per axis: next plane index p[a], its direction s[a], and the parameter of that plane */
    int p[3], s[3];
    double nxt[3];
    for (a = 0; a < 3; ++a) {
        if (d[a] == 0.0) { nxt[a] = HUGE_VAL; p[a] = 0; s[a] = 0; continue; }
        double pos = (S[a] + amin * d[a] - lo[a]) / h[a];     /* entry position in voxel units */
        if (d[a] > 0.0) { s[a] = 1;  p[a] = (int)floor(pos) - 1; if (p[a] < 0) p[a] = 0; }
        else            { s[a] = -1; p[a] = (int)ceil(pos) + 1;  if (p[a] > n[a]) p[a] = n[a]; }
        /* skip planes at or before the entry parameter */
        for (;;) {
            if (p[a] < 0 || p[a] > n[a]) { nxt[a] = HUGE_VAL; break; }
            nxt[a] = (lo[a] + p[a] * h[a] - S[a]) / d[a];
            if (nxt[a] > amin) break;
            p[a] += s[a];
        }
    }
    int cnt = 0;
    double cur = amin;
    for (;;) {
        double an = amax;
        for (a = 0; a < 3; ++a) if (nxt[a] < an) an = nxt[a];
        if (an > cur) {
            double mid = 0.5 * (cur + an);
            long v[3];
            for (a = 0; a < 3; ++a) {
                long q = (long)floor((S[a] + mid * d[a] - lo[a]) / h[a]);
                if (q < 0) q = 0;
                if (q > n[a] - 1) q = n[a] - 1;
                v[a] = q;
            }
            idx[cnt] = (v[2] * g->ny + v[1]) * (long)g->nx + v[0];
            len[cnt] = (an - cur) * L;
            ++cnt;
            cur = an;
        }
        if (an >= amax) break;
        for (a = 0; a < 3; ++a) {
            if (nxt[a] <= an) {
                p[a] += s[a];
                if (p[a] < 0 || p[a] > n[a]) nxt[a] = HUGE_VAL;
                else nxt[a] = (lo[a] + p[a] * h[a] - S[a]) / d[a];
            }
        }
    }
    return cnt;
}

/* O1: proj[ia][iv][iu] = sum_j a_{ray,j} vol[j]. */
void oracle_forward(const og_geom *g, const double *vol, double *proj)
{
    const long nrow = (long)g->n_angles * g->nv;
    const int nb = g->nx + g->ny + g->nz + 4;
#pragma omp parallel
    {
        long *idx = (long *)malloc(sizeof(long) * nb);
        double *len = (double *)malloc(sizeof(double) * nb);
#pragma omp for schedule(dynamic, 4)
        for (long r = 0; r < nrow; ++r) {
            int ia = (int)(r / g->nv), iv = (int)(r % g->nv);
            for (int iu = 0; iu < g->nu; ++iu) {
                double S[3], D[3], acc = 0.0;
                ray_endpoints(g, ia, iv, iu, S, D);
                int c = ray_chords(g, S, D, idx, len);
                for (int m = 0; m < c; ++m) acc += len[m] * vol[idx[m]];
                proj[r * g->nu + iu] = acc;
            }
        }
        free(idx); free(len);
    }
}

/* O1 on a list of rays (sampled outputs at full size). */
void oracle_forward_rays(const og_geom *g, const double *vol, long n,
                         const int *ia, const int *iv, const int *iu, double *out)
{
    const int nb = g->nx + g->ny + g->nz + 4;
#pragma omp parallel
    {
        long *idx = (long *)malloc(sizeof(long) * nb);
        double *len = (double *)malloc(sizeof(double) * nb);
#pragma omp for schedule(dynamic, 64)
        for (long r = 0; r < n; ++r) {
            double S[3], D[3], acc = 0.0;
            ray_endpoints(g, ia[r], iv[r], iu[r], S, D);
            int c = ray_chords(g, S, D, idx, len);
            for (int m = 0; m < c; ++m) acc += len[m] * vol[idx[m]];
            out[r] = acc;
        }
        free(idx); free(len);
    }
}

/* Number of non-zero chords of the whole system matrix (work counting). */
long oracle_count_chords(const og_geom *g)
{
    const long nrow = (long)g->n_angles * g->nv;
    const int nb = g->nx + g->ny + g->nz + 4;
    long total = 0;
#pragma omp parallel reduction(+ : total)
    {
        long *idx = (long *)malloc(sizeof(long) * nb);
        double *len = (double *)malloc(sizeof(double) * nb);
#pragma omp for schedule(dynamic, 4)
        for (long r = 0; r < nrow; ++r) {
            int ia = (int)(r / g->nv), iv = (int)(r % g->nv);
            for (int iu = 0; iu < g->nu; ++iu) {
                double S[3], D[3];
                ray_endpoints(g, ia, iv, iu, S, D);
                total += ray_chords(g, S, D, idx, len);
            }
        }
        free(idx); free(len);
    }
    return total;
}

/*
 * O2: vol[j] = sum_rays a_{ray,j} proj[ray] — the literal scatter of O1's traversal.
 * Each thread scatters a contiguous block of detector rows into its own private volume;
 * the private volumes are then added in thread order, so the result is deterministic for a
 * given thread count.  Returns 0, or 1 if memory for the private volumes could not be had.
 */
int oracle_backproject(const og_geom *g, const double *proj, double *vol)
{
    const long nvox = (long)g->nx * g->ny * g->nz;
    const long nrow = (long)g->n_angles * g->nv;
    const int nb = g->nx + g->ny + g->nz + 4;
    int nt = oracle_num_threads();
    double **priv = (double **)calloc((size_t)nt, sizeof(double *));
    int fail = 0;
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int t = omp_get_thread_num();
#else
        int t = 0;
#endif
        priv[t] = (double *)calloc((size_t)nvox, sizeof(double));
        if (!priv[t]) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
            long *idx = (long *)malloc(sizeof(long) * nb);
            double *len = (double *)malloc(sizeof(double) * nb);
            double *mine = priv[t];
#pragma omp for schedule(static)
            for (long r = 0; r < nrow; ++r) {
                int ia = (int)(r / g->nv), iv = (int)(r % g->nv);
                for (int iu = 0; iu < g->nu; ++iu) {
                    double y = proj[r * g->nu + iu];
                    if (y == 0.0) continue;
                    double S[3], D[3];
                    ray_endpoints(g, ia, iv, iu, S, D);
                    int c = ray_chords(g, S, D, idx, len);
                    for (int m = 0; m < c; ++m) mine[idx[m]] += len[m] * y;
                }
            }
            free(idx); free(len);
#pragma omp for schedule(static)
            for (long j = 0; j < nvox; ++j) {
                double acc = 0.0;
                for (int q = 0; q < nt; ++q) acc += priv[q][j];
                vol[j] = acc;
            }
        }
    }
    for (int q = 0; q < nt; ++q) free(priv[q]);
    free(priv);
    return fail;
}

/* Length of the part of segment S->D inside the box [lo,hi] (slab clipping; the plain
 * definition of one matrix entry a_{ray,voxel}, O1). */
static double clip_chord(const double S[3], const double D[3], const double lo[3], const double hi[3])
{
    double amin = 0.0, amax = 1.0, L = 0.0;
    for (int a = 0; a < 3; ++a) {
        double d = D[a] - S[a];
        L += d * d;
        if (d != 0.0) {
            double a0 = (lo[a] - S[a]) / d, a1 = (hi[a] - S[a]) / d;
            double l = a0 < a1 ? a0 : a1, u = a0 < a1 ? a1 : a0;
            if (l > amin) amin = l;
            if (u < amax) amax = u;
        } else if (S[a] < lo[a] || S[a] >= hi[a]) {
            return 0.0;   /* in-plane ray: belongs to the voxel with lo <= S < hi (same as the midpoint rule) */
        }
    }
    return amax > amin ? (amax - amin) * sqrt(L) : 0.0;
}

/*
 * O2 for a list of voxels, one matrix column at a time and WITHOUT the traversal:
 * for every angle, project the voxel's 8 corners onto the detector, take the pixel bounding
 * box padded by one, and clip each candidate ray against the voxel box.
 */
void oracle_backproject_voxels(const og_geom *g, const double *proj, long n,
                               const int *ix, const int *iy, const int *iz, double *out)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (long q = 0; q < n; ++q) {
        double lo[3], hi[3];
        lo[0] = (ix[q] - 0.5 * g->nx) * g->hx; hi[0] = lo[0] + g->hx;
        lo[1] = (iy[q] - 0.5 * g->ny) * g->hy; hi[1] = lo[1] + g->hy;
        lo[2] = (iz[q] - 0.5 * g->nz) * g->hz; hi[2] = lo[2] + g->hz;
        double acc = 0.0;
        for (int ia = 0; ia < g->n_angles; ++ia) {
            double t = g->angles[ia], c = cos(t), s = sin(t);
            double umin = HUGE_VAL, umax = -HUGE_VAL, vmin = HUGE_VAL, vmax = -HUGE_VAL;
            for (int m = 0; m < 8; ++m) {
                double P[3] = { (m & 1) ? hi[0] : lo[0], (m & 2) ? hi[1] : lo[1], (m & 4) ? hi[2] : lo[2] };
                double depth = g->sad - (P[0] * c + P[1] * s);       /* distance from the source along the central ray */
                double mag = g->sdd / depth;
                double u = (mag * (-P[0] * s + P[1] * c) - g->off_u) / g->du + 0.5 * (g->nu - 1);
                double v = (mag * P[2] - g->off_v) / g->dv + 0.5 * (g->nv - 1);
                if (u < umin) umin = u;
                if (u > umax) umax = u;
                if (v < vmin) vmin = v;
                if (v > vmax) vmax = v;
            }
            int u0 = (int)floor(umin) - 1, u1 = (int)ceil(umax) + 1;
            int v0 = (int)floor(vmin) - 1, v1 = (int)ceil(vmax) + 1;
            if (u0 < 0) u0 = 0;
            if (v0 < 0) v0 = 0;
            if (u1 > g->nu - 1) u1 = g->nu - 1;
            if (v1 > g->nv - 1) v1 = g->nv - 1;
            for (int iv = v0; iv <= v1; ++iv)
                for (int iu = u0; iu <= u1; ++iu) {
                    double S[3], D[3];
                    ray_endpoints(g, ia, iv, iu, S, D);
                    double a = clip_chord(S, D, lo, hi);
                    if (a > 0.0) acc += a * proj[((long)ia * g->nv + iv) * g->nu + iu];
                }
        }
        out[q] = acc;
    }
}

/*
 * NEXT-1: the paper's own voxel-driven backprojector, eq. 2, without the prefactor
 * 2/(N_theta A) (applied by the caller):
 *   (B r)(x) = sum_theta  L^3(u*,v*) / (L0 l^2(x)) * r^theta(u*,v*)
 * x the voxel centre; (u*,v*) where the line source -> x meets the imager; L0 the source-imager
 * distance; l = |x - S|; L = |(u*,v*) - S|.  r at (u*,v*) by bilinear interpolation between
 * pixel centres, r = 0 outside the detector (reading Q4).  Not the transpose of O1; it agrees with
 * (du dv / dV) P^T r as the grids are refined (pinned in tests/test_oracle_eq2.py).
 */
void oracle_backproject_eq2(const og_geom *g, const double *proj, double *vol)
{
    const double L0 = g->sdd;
#pragma omp parallel for schedule(static)
    for (long kj = 0; kj < (long)g->nz * g->ny; ++kj) {
        int k = (int)(kj / g->ny), j = (int)(kj % g->ny);
        for (int i = 0; i < g->nx; ++i) {
            double x[3] = {((double)i - 0.5 * (g->nx - 1)) * g->hx, ((double)j - 0.5 * (g->ny - 1)) * g->hy,
                           ((double)k - 0.5 * (g->nz - 1)) * g->hz};
            double acc = 0.0;
            for (int ia = 0; ia < g->n_angles; ++ia) {
                double t = g->angles[ia], c = cos(t), s = sin(t);
                double S[3] = {g->sad * c, g->sad * s, 0.0};
                double Cd[3] = {-(g->sdd - g->sad) * c, -(g->sdd - g->sad) * s, 0.0};   /* imager centre */
                double n[3] = {-c, -s, 0.0};                                             /* source -> imager normal */
                double uh[3] = {-s, c, 0.0}, vh[3] = {0.0, 0.0, 1.0};                    /* imager axes */
                double dxs[3] = {x[0] - S[0], x[1] - S[1], x[2] - S[2]};
                double depth = dxs[0] * n[0] + dxs[1] * n[1] + dxs[2] * n[2];
                if (depth <= 0.0) continue;
                double tau = L0 / depth;                                                 /* S + tau (x - S) lies on the imager */
                double Pt[3] = {S[0] + tau * dxs[0], S[1] + tau * dxs[1], S[2] + tau * dxs[2]};
                double ustar = (Pt[0] - Cd[0]) * uh[0] + (Pt[1] - Cd[1]) * uh[1] + (Pt[2] - Cd[2]) * uh[2];
                double vstar = (Pt[0] - Cd[0]) * vh[0] + (Pt[1] - Cd[1]) * vh[1] + (Pt[2] - Cd[2]) * vh[2];
                double l = sqrt(dxs[0] * dxs[0] + dxs[1] * dxs[1] + dxs[2] * dxs[2]);
                double L = sqrt((Pt[0] - S[0]) * (Pt[0] - S[0]) + (Pt[1] - S[1]) * (Pt[1] - S[1]) + (Pt[2] - S[2]) * (Pt[2] - S[2]));
                double pu = (ustar - g->off_u) / g->du + 0.5 * (g->nu - 1), pv = (vstar - g->off_v) / g->dv + 0.5 * (g->nv - 1);
                double fu = floor(pu), fv = floor(pv);
                int iu = (int)fu, iv = (int)fv;
                double au = pu - fu, av = pv - fv, val = 0.0;
                const double *img = proj + (size_t)ia * g->nv * g->nu;
                for (int dv_ = 0; dv_ < 2; ++dv_)
                    for (int du_ = 0; du_ < 2; ++du_) {
                        int uu = iu + du_, vv = iv + dv_;
                        if (uu < 0 || uu >= g->nu || vv < 0 || vv >= g->nv) continue;
                        val += (du_ ? au : 1.0 - au) * (dv_ ? av : 1.0 - av) * img[(size_t)vv * g->nu + uu];
                    }
                acc += L * L * L / (L0 * l * l) * val;
            }
            vol[((size_t)k * g->ny + j) * g->nx + i] = acc;
        }
    }
}

/*
 * NEXT-4: the backprojection step of the FDK algorithm (Feldkamp, Davis, Kress; ref. 1 of the paper; the paper's
 * comparison images Fig. 1(d), Fig. 2 at P:105, P:125 are FDK reconstructions):
 *   f(x) = (dtheta / 2) sum_theta  SAD^2 / U^2(x, theta)  q^theta(u*, v*),
 * q the pre-weighted, ramp-filtered projections (oracle/fdk.py), x the voxel centre, U = SAD - (x cos theta + y sin theta)
 * the distance of x from the source along the central ray, (u*,v*) = SDD (lat, z) / U the point where the line
 * source -> x meets the imager; q at (u*,v*) bilinear between pixel centres, 0 outside the detector (as Q4).
 * `scale` = dtheta / 2 is passed in (equally spaced full rotation: dtheta = 2 pi / N_theta).
 */
void oracle_fdk_backproject(const og_geom *g, const double *q, double scale, double *vol)
{
#pragma omp parallel for schedule(static)
    for (long kj = 0; kj < (long)g->nz * g->ny; ++kj) {
        int k = (int)(kj / g->ny), j = (int)(kj % g->ny);
        for (int i = 0; i < g->nx; ++i) {
            double x = ((double)i - 0.5 * (g->nx - 1)) * g->hx, y = ((double)j - 0.5 * (g->ny - 1)) * g->hy,
                   z = ((double)k - 0.5 * (g->nz - 1)) * g->hz;
            double acc = 0.0;
            for (int ia = 0; ia < g->n_angles; ++ia) {
                double t = g->angles[ia], c = cos(t), s = sin(t);
                double U = g->sad - (x * c + y * s);
                if (U <= 0.0) continue;
                double lat = -x * s + y * c;
                double ustar = g->sdd * lat / U, vstar = g->sdd * z / U;
                double pu = (ustar - g->off_u) / g->du + 0.5 * (g->nu - 1), pv = (vstar - g->off_v) / g->dv + 0.5 * (g->nv - 1);
                double fu = floor(pu), fv = floor(pv);
                int iu = (int)fu, iv = (int)fv;
                double au = pu - fu, av = pv - fv, val = 0.0;
                const double *img = q + (size_t)ia * g->nv * g->nu;
                for (int dv_ = 0; dv_ < 2; ++dv_)
                    for (int du_ = 0; du_ < 2; ++du_) {
                        int uu = iu + du_, vv = iv + dv_;
                        if (uu < 0 || uu >= g->nu || vv < 0 || vv >= g->nv) continue;
                        val += (du_ ? au : 1.0 - au) * (dv_ ? av : 1.0 - av) * img[(size_t)vv * g->nu + uu];
                    }
                acc += (g->sad * g->sad) / (U * U) * val;
            }
            vol[((size_t)k * g->ny + j) * g->nx + i] = scale * acc;
        }
    }
}

/* ------------------------------------------------------------------------------------
 * O3 / O4: smoothed isotropic total variation (P:69 E1, ROF semi-norm of ref. 5; Q5, Q6).
 *   d_x = (f[i+1]-f[i])/hx  (0 at the last index: Neumann), likewise d_y, d_z
 *   n_ijk = sqrt(d_x^2 + d_y^2 + d_z^2 + eps^2),   TV_eps(f) = sum_ijk n_ijk
 * ---------------------------------------------------------------------------------- */
#define VIDX(i, j, k) (((long)(k) * ny + (j)) * nx + (i))

static inline void fwd_diff(const double *f, int nx, int ny, int nz, double hx, double hy, double hz,
                            int i, int j, int k, double *dx, double *dy, double *dz)
{
    double c = f[VIDX(i, j, k)];
    *dx = (i + 1 < nx) ? (f[VIDX(i + 1, j, k)] - c) / hx : 0.0;
    *dy = (j + 1 < ny) ? (f[VIDX(i, j + 1, k)] - c) / hy : 0.0;
    *dz = (k + 1 < nz) ? (f[VIDX(i, j, k + 1)] - c) / hz : 0.0;
}

double oracle_tv_value(const double *f, int nx, int ny, int nz, double hx, double hy, double hz, double eps)
{
    double total = 0.0;
#pragma omp parallel for reduction(+ : total) schedule(static)
    for (int k = 0; k < nz; ++k) {
        double plane = 0.0;
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double dx, dy, dz;
                fwd_diff(f, nx, ny, nz, hx, hy, hz, i, j, k, &dx, &dy, &dz);
                plane += sqrt(dx * dx + dy * dy + dz * dz + eps * eps);
            }
        total += plane;
    }
    return total;
}

/* O4: exact gradient of TV_eps:
 *  grad[ijk] = -(dx/hx + dy/hy + dz/hz)/n |ijk + (dx/hx)/n |i-1,j,k + (dy/hy)/n |i,j-1,k + (dz/hz)/n |i,j,k-1
 * (terms with an index -1 dropped).  eps must be > 0. */
static inline double tv_grad_at(const double *f, int nx, int ny, int nz, double hx, double hy, double hz,
                                double eps, int i, int j, int k)
{
    double dx, dy, dz, n, gsum;
    fwd_diff(f, nx, ny, nz, hx, hy, hz, i, j, k, &dx, &dy, &dz);
    n = sqrt(dx * dx + dy * dy + dz * dz + eps * eps);
    gsum = -(dx / hx + dy / hy + dz / hz) / n;
    if (i > 0) {
        fwd_diff(f, nx, ny, nz, hx, hy, hz, i - 1, j, k, &dx, &dy, &dz);
        n = sqrt(dx * dx + dy * dy + dz * dz + eps * eps);
        gsum += (dx / hx) / n;
    }
    if (j > 0) {
        fwd_diff(f, nx, ny, nz, hx, hy, hz, i, j - 1, k, &dx, &dy, &dz);
        n = sqrt(dx * dx + dy * dy + dz * dz + eps * eps);
        gsum += (dy / hy) / n;
    }
    if (k > 0) {
        fwd_diff(f, nx, ny, nz, hx, hy, hz, i, j, k - 1, &dx, &dy, &dz);
        n = sqrt(dx * dx + dy * dy + dz * dz + eps * eps);
        gsum += (dz / hz) / n;
    }
    return gsum;
}

void oracle_tv_grad(const double *f, int nx, int ny, int nz, double hx, double hy, double hz,
                    double eps, double *grad)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                grad[VIDX(i, j, k)] = tv_grad_at(f, nx, ny, nz, hx, hy, hz, eps, i, j, k);
}

/* O4 inner loop (P:89 step 2, "solved by a simple gradient descent method"):
 *   u^{m+1} = u^m - dt [ beta (u^m - g) + grad TV_eps(u^m) ],
 *   dt = omega / ( beta + 4 (1/hx^2 + 1/hy^2 + 1/hz^2) / eps )          (Q7)
 * Jacobi: every voxel of u^{m+1} is computed from u^m (two buffers).  u holds the start
 * on entry and the result on exit. */
void oracle_tv_prox(const double *g, double *u, int nx, int ny, int nz, double hx, double hy, double hz,
                    double beta, double eps, double omega, int n_inner)
{
    long nvox = (long)nx * ny * nz;
    double dt = omega / (beta + 4.0 * (1.0 / (hx * hx) + 1.0 / (hy * hy) + 1.0 / (hz * hz)) / eps);
    double *a = u, *b = (double *)malloc(sizeof(double) * (size_t)nvox);
    for (int m = 0; m < n_inner; ++m) {
#pragma omp parallel for schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    long q = VIDX(i, j, k);
                    double gr = tv_grad_at(a, nx, ny, nz, hx, hy, hz, eps, i, j, k);
                    b[q] = a[q] - dt * (beta * (a[q] - g[q]) + gr);
                }
        double *t = a; a = b; b = t;
    }
    if (a != u) { memcpy(u, a, sizeof(double) * (size_t)nvox); free(a); }
    else free(b);
}
