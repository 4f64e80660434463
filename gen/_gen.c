/*
 * gen/_gen.c -- seeded synthetic workload generators (geometry only).
 *
 * TEST / BENCH INFRASTRUCTURE shared by the oracle harness and the CUDA harness.
 * This file holds NONE of the method's arithmetic (no projections, no sweeps, no
 * objectives): it only builds sparse system matrices from geometry, in canonical
 * CSR (int64 row pointers, int32 sorted distinct columns, fp32 values rounded once
 * from fp64).  Recipes: DESIGN.md "Input recipe" (BASELINE.json configs 1-4).
 *
 *   line_*   : exact line/cell intersection lengths on a regular 2-D grid
 *              (parallel-beam CT rays; crosswell source->receiver segments)
 *   imrt_*   : pencil-beam dose-influence entries on a 3-D voxel grid
 *
 * Two-pass protocol: *_count fills per-row counts, the caller prefix-sums them
 * into rowptr, *_fill writes col/val.  OpenMP over rows.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define DROP_EPS 1e-7 /* entries shorter than this (length units) are dropped */

typedef struct {
    int32_t c;
    float v;
} ent_t;

static int ent_cmp(const void* a, const void* b) {
    int32_t ca = ((const ent_t*)a)->c, cb = ((const ent_t*)b)->c;
    return (ca > cb) - (ca < cb);
}

/* Trace the parametric line P(t) = (px + t dx, py + t dy), t in [t0, t1], through the
 * grid of unit cells [X0, X0+nx) x [Y0, Y0+ny) (half-open cells: a point on a grid line
 * belongs to the cell on its + side).  Cell (iy, ix) has index iy*nx + ix.  Emits
 * (cell, length) for every crossed cell with length >= DROP_EPS, in order of t.
 * `out` may be NULL (count only).  `scratch` must hold nx + ny + 4 doubles. */
static int trace_line(double px, double py, double dx, double dy, double t0, double t1,
                      int nx, int ny, double X0, double Y0, ent_t* out, double* scratch) {
    /* clip to the closed bounding box of the grid */
    double lo = t0, hi = t1;
    if (dx != 0.0) {
        double ta = (X0 - px) / dx, tb = (X0 + nx - px) / dx;
        if (ta > tb) { double s = ta; ta = tb; tb = s; }
        if (ta > lo) lo = ta;
        if (tb < hi) hi = tb;
    } else if (px < X0 || px > X0 + nx) return 0;
    if (dy != 0.0) {
        double ta = (Y0 - py) / dy, tb = (Y0 + ny - py) / dy;
        if (ta > tb) { double s = ta; ta = tb; tb = s; }
        if (ta > lo) lo = ta;
        if (tb < hi) hi = tb;
    } else if (py < Y0 || py > Y0 + ny) return 0;
    if (!(hi > lo)) return 0;

    /* crossing parameters with the two families of grid lines, merged in increasing t */
    double* ts = scratch;
    int nt = 0;
    ts[nt++] = lo;
    /* vertical lines x = X0 + k */
    int kx0 = 0, kx1 = -1, sx = 1;
    if (dx != 0.0) {
        double xa = px + lo * dx, xb = px + hi * dx;
        double xl = xa < xb ? xa : xb, xh = xa < xb ? xb : xa;
        kx0 = (int)ceil(xl - X0 - 1e-12);
        kx1 = (int)floor(xh - X0 + 1e-12);
        if (kx0 < 0) kx0 = 0;
        if (kx1 > nx) kx1 = nx;
        sx = dx > 0 ? 1 : -1;
    }
    int ky0 = 0, ky1 = -1, sy = 1;
    if (dy != 0.0) {
        double ya = py + lo * dy, yb = py + hi * dy;
        double yl = ya < yb ? ya : yb, yh = ya < yb ? yb : ya;
        ky0 = (int)ceil(yl - Y0 - 1e-12);
        ky1 = (int)floor(yh - Y0 + 1e-12);
        if (ky0 < 0) ky0 = 0;
        if (ky1 > ny) ky1 = ny;
        sy = dy > 0 ? 1 : -1;
    }
    int ix = sx > 0 ? kx0 : kx1, nxc = kx1 - kx0 + 1;
    int iy = sy > 0 ? ky0 : ky1, nyc = ky1 - ky0 + 1;
    if (nxc < 0) nxc = 0;
    if (nyc < 0) nyc = 0;
    int ax = 0, ay = 0;
    while (ax < nxc || ay < nyc) {
        double tx = ax < nxc ? (X0 + ix - px) / dx : INFINITY;
        double ty = ay < nyc ? (Y0 + iy - py) / dy : INFINITY;
        double t;
        if (tx <= ty) { t = tx; ix += sx; ax++; } else { t = ty; iy += sy; ay++; }
        if (t > lo && t < hi) ts[nt++] = t;
    }
    ts[nt++] = hi;

    double norm = sqrt(dx * dx + dy * dy);
    int ne = 0;
    for (int s = 0; s + 1 < nt; ++s) {
        double ta = ts[s], tb = ts[s + 1];
        double len = (tb - ta) * norm;
        if (len < DROP_EPS) continue;
        double tm = 0.5 * (ta + tb);
        double cx = floor(px + tm * dx - X0), cy = floor(py + tm * dy - Y0);
        if (cx < 0 || cx >= nx || cy < 0 || cy >= ny) continue;
        int32_t cell = (int32_t)cy * nx + (int32_t)cx;
        if (out) {
            if (ne > 0 && out[ne - 1].c == cell) { /* merge a split caused by a dropped sliver */
                out[ne - 1].v = (float)((double)out[ne - 1].v + len);
                continue;
            }
            out[ne].c = cell;
            out[ne].v = (float)len;
        }
        ne++;
    }
    return ne;
}

/* The `out == NULL` count above cannot merge; to keep count == fill we always trace into
 * a scratch entry buffer in both passes. */

typedef struct {
    int nx, ny;       /* grid cells (columns of A = ny*nx) */
    double X0, Y0;    /* lower-left corner of the grid */
} grid_t;

/* ---- parallel-beam CT: row = q*n_bins + p; ray {(x,y): x cos(th)+y sin(th) = s_p}, th_q = q*pi/n_angles,
 *      s_p = (p - (n_bins-1)/2) * bin_spacing.  th = 0 and th = pi/2 use exact (1,0)/(0,1). ---- */
static void ct_ray(int q, int p, int n_angles, int n_bins, double spacing, double* px, double* py,
                   double* dx, double* dy) {
    double c, s;
    if (q == 0) { c = 1.0; s = 0.0; }
    else if (2 * q == n_angles) { c = 0.0; s = 1.0; }
    else { double th = (double)q * M_PI / (double)n_angles; c = cos(th); s = sin(th); }
    double off = ((double)p - 0.5 * (double)(n_bins - 1)) * spacing;
    *px = off * c; *py = off * s; *dx = -s; *dy = c;
}

static void rows_generic(int mode, int64_t m, const double* seg /* mode 1: [m][4] */, int n_angles, int n_bins,
                         double spacing, grid_t g, const int64_t* rowptr, int64_t* counts, int32_t* col,
                         float* val) {
    int diag = g.nx + g.ny + 8;
#pragma omp parallel
    {
        double* scratch = (double*)malloc(sizeof(double) * (size_t)(diag + 8));
        ent_t* ents = (ent_t*)malloc(sizeof(ent_t) * (size_t)(diag + 8));
#pragma omp for schedule(dynamic, 64)
        for (int64_t r = 0; r < m; ++r) {
            double px, py, dx, dy, t0, t1;
            if (mode == 0) {
                ct_ray((int)(r / n_bins), (int)(r % n_bins), n_angles, n_bins, spacing, &px, &py, &dx, &dy);
                t0 = -1e30; t1 = 1e30;
            } else {
                px = seg[4 * r + 0]; py = seg[4 * r + 1];
                dx = seg[4 * r + 2] - px; dy = seg[4 * r + 3] - py;
                t0 = 0.0; t1 = 1.0;
            }
            int ne = trace_line(px, py, dx, dy, t0, t1, g.nx, g.ny, g.X0, g.Y0, ents, scratch);
            if (counts) counts[r] = ne;
            if (col) {
                qsort(ents, (size_t)ne, sizeof(ent_t), ent_cmp);
                int64_t k = rowptr[r];
                for (int e = 0; e < ne; ++e) { col[k + e] = ents[e].c; val[k + e] = ents[e].v; }
            }
        }
        free(scratch);
        free(ents);
    }
}

void ct_count(int n_angles, int n_bins, double spacing, int nx, int ny, int64_t* counts) {
    grid_t g = {nx, ny, -0.5 * nx, -0.5 * ny};
    rows_generic(0, (int64_t)n_angles * n_bins, NULL, n_angles, n_bins, spacing, g, NULL, counts, NULL, NULL);
}
void ct_fill(int n_angles, int n_bins, double spacing, int nx, int ny, const int64_t* rowptr, int32_t* col,
             float* val) {
    grid_t g = {nx, ny, -0.5 * nx, -0.5 * ny};
    rows_generic(0, (int64_t)n_angles * n_bins, NULL, n_angles, n_bins, spacing, g, rowptr, NULL, col, val);
}

/* ---- straight segments (crosswell): seg[r] = (xs, ys, xr, yr); grid [0,nx] x [0,ny] ---- */
void seg_count(int64_t m, const double* seg, int nx, int ny, int64_t* counts) {
    grid_t g = {nx, ny, 0.0, 0.0};
    rows_generic(1, m, seg, 0, 0, 0.0, g, NULL, counts, NULL, NULL);
}
void seg_fill(int64_t m, const double* seg, int nx, int ny, const int64_t* rowptr, int32_t* col, float* val) {
    grid_t g = {nx, ny, 0.0, 0.0};
    rows_generic(1, m, seg, 0, 0, 0.0, g, rowptr, NULL, col, val);
}

/* ---- IMRT pencil-beam dose influence -------------------------------------------------
 * Voxel grid gx*gy*gz, spacing h (mm), centred at the isocentre; voxel (x,y,z) centre =
 * ((x-(gx-1)/2) h, (y-(gy-1)/2) h, (z-(gz-1)/2) h).  Beam b: direction (cos phi, sin phi, 0),
 * beam's-eye axes e_u = (-sin phi, cos phi, 0), e_v = (0,0,1).  Beamlet (u,v), u,v in [0,nb):
 * axis offset ((u-(nb-1)/2) bs, (v-(nb-1)/2) bs); column = b*nb*nb + v*nb + u.
 * Entry = exp(-mu*depth) * exp(-rho^2/(2 sigma^2)), depth = depth0 + <p, dir>.
 * Rows = the voxels listed in vox[] (body voxels, linear index (z*gy+y)*gx+x), in that order.
 * Kept iff entry >= trunc * colmax[column], colmax = max over the listed voxels. */
typedef struct {
    int gx, gy, gz; double h;
    int n_beams; const double* phi;
    int nb; double bs;
    double mu, sigma, depth0, trunc;
} imrt_t;

static inline void imrt_voxel_pos(const imrt_t* P, int64_t lin, double* p) {
    int x = (int)(lin % P->gx), y = (int)((lin / P->gx) % P->gy), z = (int)(lin / ((int64_t)P->gx * P->gy));
    p[0] = (x - 0.5 * (P->gx - 1)) * P->h;
    p[1] = (y - 0.5 * (P->gy - 1)) * P->h;
    p[2] = (z - 0.5 * (P->gz - 1)) * P->h;
}

/* visit candidate beamlets of one voxel; cb(col, value) */
#define IMRT_FOR_CANDIDATES(P, p, BODY)                                                        \
    {                                                                                          \
        double rmax = (P)->sigma * sqrt(2.0 * log(1.0 / (P)->trunc)) + 1e-9;                   \
        for (int b = 0; b < (P)->n_beams; ++b) {                                               \
            double cph = cos((P)->phi[b]), sph = sin((P)->phi[b]);                             \
            double depth = (P)->depth0 + p[0] * cph + p[1] * sph;                              \
            double pu = -p[0] * sph + p[1] * cph, pv = p[2];                                   \
            double half = 0.5 * ((P)->nb - 1);                                                 \
            int u0 = (int)ceil((pu - rmax) / (P)->bs + half), u1 = (int)floor((pu + rmax) / (P)->bs + half); \
            int v0 = (int)ceil((pv - rmax) / (P)->bs + half), v1 = (int)floor((pv + rmax) / (P)->bs + half); \
            if (u0 < 0) u0 = 0; if (v0 < 0) v0 = 0;                                            \
            if (u1 > (P)->nb - 1) u1 = (P)->nb - 1; if (v1 > (P)->nb - 1) v1 = (P)->nb - 1;    \
            for (int v = v0; v <= v1; ++v)                                                     \
                for (int u = u0; u <= u1; ++u) {                                               \
                    double lu = pu - (u - half) * (P)->bs, lv = pv - (v - half) * (P)->bs;     \
                    double rho2 = lu * lu + lv * lv;                                           \
                    if (rho2 > rmax * rmax) continue;                                          \
                    double value = exp(-(P)->mu * depth) * exp(-rho2 / (2.0 * (P)->sigma * (P)->sigma)); \
                    int32_t colidx = (int32_t)(b * (P)->nb * (P)->nb + v * (P)->nb + u);       \
                    BODY                                                                       \
                }                                                                              \
        }                                                                                      \
    }

void imrt_colmax(int gx, int gy, int gz, double h, int n_beams, const double* phi, int nb, double bs, double mu,
                 double sigma, double depth0, double trunc, int64_t n_vox, const int64_t* vox, double* colmax) {
    imrt_t P = {gx, gy, gz, h, n_beams, phi, nb, bs, mu, sigma, depth0, trunc};
    int ncol = n_beams * nb * nb;
    for (int c = 0; c < ncol; ++c) colmax[c] = 0.0;
#pragma omp parallel
    {
        double* loc = (double*)calloc((size_t)ncol, sizeof(double));
#pragma omp for schedule(static)
        for (int64_t r = 0; r < n_vox; ++r) {
            double p[3];
            imrt_voxel_pos(&P, vox[r], p);
            IMRT_FOR_CANDIDATES(&P, p, { if (value > loc[colidx]) loc[colidx] = value; })
        }
#pragma omp critical
        for (int c = 0; c < ncol; ++c) if (loc[c] > colmax[c]) colmax[c] = loc[c];
        free(loc);
    }
}

/* rowptr == NULL: count only (counts[r]); else fill col/val at rowptr[r]. Columns come out sorted. */
void imrt_rows(int gx, int gy, int gz, double h, int n_beams, const double* phi, int nb, double bs, double mu,
               double sigma, double depth0, double trunc, int64_t n_vox, const int64_t* vox, const double* colmax,
               const int64_t* rowptr, int64_t* counts, int32_t* col, float* val) {
    imrt_t P = {gx, gy, gz, h, n_beams, phi, nb, bs, mu, sigma, depth0, trunc};
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n_vox; ++r) {
        double p[3];
        imrt_voxel_pos(&P, vox[r], p);
        int64_t ne = 0, k0 = rowptr ? rowptr[r] : 0;
        IMRT_FOR_CANDIDATES(&P, p, {
            if (value >= trunc * colmax[colidx]) {
                if (rowptr) { col[k0 + ne] = colidx; val[k0 + ne] = (float)value; }
                ne++;
            }
        })
        if (counts) counts[r] = ne;
    }
}
