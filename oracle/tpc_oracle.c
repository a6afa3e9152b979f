/*
 * oracle/tpc_oracle.c -- CPU ORACLE of the TPC sector tracker.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the CUDA
 * path (paper_1709_00618_b200/csrc, include/); neither side includes the other.
 *
 * What it computes: the sector tracker of /root/reference/PAPER.md:25 (section 2, "Online
 * Tracking in ALICE"), stage by stage, in the paper's order:
 *   S1 grid (acceleration only)           -- not in the paper; BASELINE.json north_star
 *   S2 neighbour finding ("forming links of adjacent hits arranged close to a straight line")
 *   S3 neighbour cleaning (mutual links)  -- north_star
 *   S4 start hits + concatenation ("concatenating links", candidates "of usually 4 to 10 hits")
 *   S5 track following ("fits track parameters to the track candidate and extrapolates the
 *      trajectory through the TPC sector volume to pick up additional clusters and refine the
 *      fit using a simplified Kalman filter"); pure Bz
 *   S6 selection ("selection of good tracks and final assignment of clusters to tracks
 *      dissolving ambiguities")
 * The paper gives no formula for any stage; every formula below is the reading fixed in
 * SURVEY.md section 8(c) and restated in DESIGN.md ("Readings").  The method is a heuristic
 * pipeline, so the oracle is the algorithm written out step by step, in plain loops.
 *
 * Arithmetic: S2 and the S5 pick-up test are fp32 with every operation individually rounded
 * (compile with -ffp-contract=off, no -ffast-math); the Kalman filter is fp64.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): grid search == brute force; noise-free straight
 * and helical tracks link to their own neighbours and are recovered with all hits; cleaning and
 * chain invariants; Jacobian == central finite differences; forward+backward transport is the
 * identity; Bz->0 limit is the straight line; zero-smear fits reproduce the generating helix to
 * 1e-6; pulls ~ N(0,1) and chi2/ndf ~ 1; in the linear regime (Bz = 0, residuals of 1e-6 cm)
 * the sequential filter equals a one-shot weighted least-squares fit with the prior folded in
 * (numpy, state and covariance); the pick-up and stop rules of pickup() / follow_dir() on
 * hand-placed straight tracks: nearest of several clusters in the gate, lowest local index on
 * an exact tie, gate = 4 sigma capped at 3 cm, 5 empty rows bridged / 6 stop / a hit resets the
 * count, stop at the first row beyond the sector edge + margin (tests/test_oracle_follow_rules.py);
 * for the optional class-1 links of S2 (nf_bridge_rows, reading A2'): grid == brute force,
 * hand-placed lines with one / two missing rows, the cut the 2.25 factor implies, the exact tie
 * between the two kinds (tests/test_oracle_bridge.py).  Parity unpinned: the absolute values of
 * the tuning constants (window sizes, D2 cuts, gate, gap, selector threshold) -- the paper gives
 * none (readings A2',A3,A4,A9,A11).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t n_rows;
    const float *row_x;          /* [n_rows] */
    int32_t sectors_per_event;   /* 36: instance i is sector i % 36; sector >= 18 is the z<0 side */
    float half_angle_rad;
    float z_lo, z_hi;            /* z range of the z>=0 side; mirrored for the z<0 side */
    float sigma_y, sigma_z;
    float nf_win_y, nf_win_z, nf_d2_max;
    int32_t cand_min_hits, cand_max_hits;
    double kf_p0[5];
    double kf_gate_sigma, kf_win_max;
    int32_t kf_max_gap;
    double kf_max_sinphi, kf_edge_margin;
    int32_t sel_min_hits;
    float grid_cell_y, grid_cell_z;
    double bz;
    int32_t nf_bridge_rows;      /* 0: links join adjacent rows only; 1: a single missing row may be bridged (A2') */
    int32_t pad_;
} orc_config;

typedef struct {               /* one tracklet (S5 output) */
    int32_t ok;                /* 0: candidate produced no tracklet */
    int32_t nhits, first_row, last_row, ref_row;
    double p[5];
    double cov[15];            /* lower triangle, row-major: (0,0),(1,0),(1,1),(2,0),... */
    double chi2;
} orc_tracklet;

#define KAPPA_PER_TESLA 0.00299792458

static double curv_const(const orc_config *c) { return -KAPPA_PER_TESLA * c->bz; }

/* ------------------------------------------------------------------ S1: grid (acceleration) */

typedef struct {
    int ny, nz;
    float y0, z0, inv_cy, inv_cz;
    int32_t *bin_start;  /* [ny*nz+1] */
    int32_t *perm;       /* [n] local indices sorted by bin, stable */
    int n;
} orc_rowgrid;

static int grid_bin1(float v, float origin, float inv, int n) {
    int b = (int)floorf((v - origin) * inv);
    if (b < 0) b = 0;
    if (b > n - 1) b = n - 1;
    return b;
}

/* origin y0 = -y_max(r) - 1 cm, z0 = z_lo (mirrored for z<0 sectors), bin id = bz*ny + by. */
static void grid_build(orc_rowgrid *g, const orc_config *c, int inst, int row, const float *cl, int n) {
    double ymax = (double)c->row_x[row] * tan((double)c->half_angle_rad);
    int side_c = (inst % c->sectors_per_event) >= c->sectors_per_event / 2;
    float zlo = side_c ? -c->z_hi : c->z_lo, zhi = side_c ? -c->z_lo : c->z_hi;
    g->y0 = (float)(-ymax - 1.0);
    g->z0 = zlo;
    g->inv_cy = 1.0f / c->grid_cell_y;
    g->inv_cz = 1.0f / c->grid_cell_z;
    g->ny = (int)ceil((2.0 * ymax + 2.0) / c->grid_cell_y);
    g->nz = (int)ceil(((double)zhi - (double)zlo) / c->grid_cell_z);
    if (g->ny < 1) g->ny = 1;
    if (g->nz < 1) g->nz = 1;
    g->n = n;
    int nb = g->ny * g->nz;
    g->bin_start = (int32_t *)calloc((size_t)nb + 1, sizeof(int32_t));
    g->perm = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *bins = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    for (int i = 0; i < n; i++) {
        int by = grid_bin1(cl[4 * i + 1], g->y0, g->inv_cy, g->ny);
        int bz = grid_bin1(cl[4 * i + 2], g->z0, g->inv_cz, g->nz);
        bins[i] = bz * g->ny + by;
        g->bin_start[bins[i] + 1]++;
    }
    for (int b = 0; b < nb; b++) g->bin_start[b + 1] += g->bin_start[b];
    int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)nb);
    memcpy(fill, g->bin_start, sizeof(int32_t) * (size_t)nb);
    for (int i = 0; i < n; i++) g->perm[fill[bins[i]]++] = i;
    free(fill);
    free(bins);
}

static void grid_free(orc_rowgrid *g) {
    free(g->bin_start);
    free(g->perm);
    g->bin_start = NULL;
    g->perm = NULL;
}

/* ------------------------------------------------------------------ S2: neighbour finder */

/* Hits of one row inside the window [ylo,yhi] x [zlo,zhi] (pure comparisons against pre-rounded bounds), as local
 * indices (positions within the row segment of the input array).  use_grid = 0: all hits of the row are tested;
 * 1: only the bins overlapping the window.  Both apply the identical exact test, so they must agree
 * (pin: tests/test_oracle_ca.py). */
static int window_list(const float *cl, int n, const orc_rowgrid *g, int use_grid, float ylo, float yhi, float zlo,
                       float zhi, int32_t *list) {
    int cnt = 0;
    if (!use_grid) {
        for (int j = 0; j < n; j++) {
            float yj = cl[4 * j + 1], zj = cl[4 * j + 2];
            if (ylo <= yj && yj <= yhi && zlo <= zj && zj <= zhi) list[cnt++] = j;
        }
    } else if (n > 0) {
        int by0 = grid_bin1(ylo, g->y0, g->inv_cy, g->ny), by1 = grid_bin1(yhi, g->y0, g->inv_cy, g->ny);
        int bz0 = grid_bin1(zlo, g->z0, g->inv_cz, g->nz), bz1 = grid_bin1(zhi, g->z0, g->inv_cz, g->nz);
        for (int bz = bz0; bz <= bz1; bz++)
            for (int k = g->bin_start[bz * g->ny + by0]; k < g->bin_start[bz * g->ny + by1 + 1]; k++) {
                int j = g->perm[k];
                float yj = cl[4 * j + 1], zj = cl[4 * j + 2];
                if (ylo <= yj && yj <= yhi && zlo <= zj && zj <= zhi) list[cnt++] = j;
            }
    }
    return cnt;
}

/* Reading A5' (SURVEY 8(f) NEXT-2 "non-uniform pad-row pitch with the weighted second difference"): the
 * pad rows need not be equally spaced (the real TPC has three pad lengths).  For row r with steps du = x[r+1] - x[r]
 * and dd = x[r] - x[r-1], three points are collinear iff dd (u - h) - du (h - d) = 0; normalised so that equal steps
 * give the plain second difference:   e = wu (u - h) - wd (h - d),  wu = 2 dd / (du + dd),  wd = 2 du / (du + dd).
 * The search window is a slope bound (reading A3), so it scales with the step: the half-sizes towards row r+1 are
 * (WY su, WZ su), su = du / p_ref, towards row r-1 (WY sd, WZ sd), sd = dd / p_ref, p_ref = mean pitch.
 * A step within 1e-4 p_ref + 4e-5 cm of p_ref counts as p_ref (factor exactly 1; both steps such -> wu = wd = 1), so
 * every geometry that passes the uniformity test of the default reading keeps that reading's arithmetic bit for bit.
 * Computed in double from the fp32 row_x, rounded to fp32. */
static void row_step_factors(const orc_config *c, int r, float *wu, float *wd, float *su, float *sd) {
    const int R = c->n_rows;
    const double pref = ((double)c->row_x[R - 1] - (double)c->row_x[0]) / (R - 1);
    const double du = (double)c->row_x[r + 1] - (double)c->row_x[r], dd = (double)c->row_x[r] - (double)c->row_x[r - 1];
    const double tol = 1e-4 * pref + 4e-5;
    const int ureg = fabs(du - pref) <= tol, dreg = fabs(dd - pref) <= tol;
    *su = ureg ? 1.0f : (float)(du / pref);
    *sd = dreg ? 1.0f : (float)(dd / pref);
    if (ureg && dreg) {
        *wu = 1.0f;
        *wd = 1.0f;
    } else {
        *wu = (float)(2.0 * dd / (du + dd));
        *wd = (float)(2.0 * du / (du + dd));
    }
}

/* SURVEY 8(c) S2 for one sector instance (ro = its row offsets [R+1], indices of `clusters`); link_up/link_dn are
 * written at those indices and hold such indices, -1 if none.  All fp32, every operation individually rounded
 * (this file is compiled with -ffp-contract=off).
 *
 * Class 0 (the reading of BASELINE.json north_star, "adjacent pad rows"): u in row r+1, d in row r-1, both inside
 * the window of half-widths (WY, WZ) around the hit; D = (t1 - t2)^2 + (t3 - t4)^2 with t1 = y_u - y, t2 = y - y_d,
 * t3 = z_u - z, t4 = z - z_d; admissible iff D <= D2MAX; minimum over (D, u, d).
 *
 * Class 1 (nf_bridge_rows = 1, reading A2': "bridge single missing rows"; defined for
 * equally spaced rows only -- the library rejects it with a non-uniform pitch): only for
 * a hit with NO admissible class-0 pair.  One of the two partners may lie two rows away (a row without a usable
 * cluster is skipped): (du, dd) = (1, 2): u in row r+1, d in row r-2, or (2, 1): u in row r+2, d in row r-1.  The
 * partner two rows away is searched in the doubled window (2 WY, 2 WZ; exact doubling).  The deviation from a
 * straight line for unequal spacing is dd * (u - h) - du * (h - d):
 *     (1,2): ey = (t1 + t1) - t2,   (2,1): ey = t1 - (t2 + t2),   same for z;   D = ey*ey + ez*ez.
 * Its variance for cluster errors sigma is 14 sigma^2 against 6 sigma^2 for class 0, so the cut is
 * D <= 2.25 * D2MAX (2.25 is exact in binary; the same ~4 sigma).  Minimum over (D, du, u, d) lexicographically. */
static void neighbours_instance(const orc_config *c, const float *clusters, const int32_t *ro,
                                const orc_rowgrid *grids, int use_grid, int32_t *link_up, int32_t *link_dn) {
    const int R = c->n_rows;
    const float WY = c->nf_win_y, WZ = c->nf_win_z, D2MAX = c->nf_d2_max;
    const float WY2 = WY + WY, WZ2 = WZ + WZ, D2MAX1 = D2MAX * 2.25f;
    int nmax = 1;
    for (int r = 0; r < R; r++)
        if (ro[r + 1] - ro[r] > nmax) nmax = ro[r + 1] - ro[r];
    int32_t *ulist = (int32_t *)malloc(sizeof(int32_t) * (size_t)nmax);
    int32_t *dlist = (int32_t *)malloc(sizeof(int32_t) * (size_t)nmax);
    int32_t *xlist = (int32_t *)malloc(sizeof(int32_t) * (size_t)nmax);
#define ROWCL(rr) (clusters + 4 * (size_t)ro[rr])
#define ROWN(rr) (ro[(rr) + 1] - ro[rr])
#define ROWG(rr) (use_grid ? &grids[rr] : (const orc_rowgrid *)0)
    for (int r = 0; r < R; r++) {
        const int n_r = ROWN(r);
        const float *cl_r = ROWCL(r);
        float wu = 1.0f, wd = 1.0f, su = 1.0f, sd = 1.0f;
        if (r >= 1 && r <= R - 2) row_step_factors(c, r, &wu, &wd, &su, &sd);
        for (int h = 0; h < n_r; h++) {
            int32_t lu = -1, ld = -1;
            if (r >= 1 && r <= R - 2) { /* rows 0 and R-1 never own links (reading A6) */
                const float y = cl_r[4 * h + 1], z = cl_r[4 * h + 2];
                /* window towards row r+1 and towards row r-1 (reading A5': the half-sizes scale with the row step;
                 * su = sd = 1 and wu = wd = 1 for equally spaced rows, where x * 1.0f is exact) */
                const float WYu = WY * su, WZu = WZ * su, WYd = WY * sd, WZd = WZ * sd;
                const float ylo = y - WYu, yhi = y + WYu, zlo = z - WZu, zhi = z + WZu;
                const float ylo_d = y - WYd, yhi_d = y + WYd, zlo_d = z - WZd, zhi_d = z + WZd;
                const float *cl_up = ROWCL(r + 1), *cl_dn = ROWCL(r - 1);
                const int nu = window_list(cl_up, ROWN(r + 1), ROWG(r + 1), use_grid, ylo, yhi, zlo, zhi, ulist);
                const int nd = window_list(cl_dn, ROWN(r - 1), ROWG(r - 1), use_grid, ylo_d, yhi_d, zlo_d, zhi_d, dlist);
                /* class 0: minimum over (D, u, d) lexicographically: independent of the visiting order */
                int bu = -1, bd = -1, bdu = 1, bdd = 1;
                float bD = 0.0f;
                for (int a = 0; a < nu; a++)
                    for (int b = 0; b < nd; b++) {
                        int u = ulist[a], d = dlist[b];
                        float t1 = cl_up[4 * u + 1] - y, t2 = y - cl_dn[4 * d + 1];
                        float t3 = cl_up[4 * u + 2] - z, t4 = z - cl_dn[4 * d + 2];
                        float a1 = wu * t1, a2 = wd * t2, ey = a1 - a2;
                        float a3 = wu * t3, a4 = wd * t4, ez = a3 - a4;
                        float pyy = ey * ey, pzz = ez * ez;
                        float D = pyy + pzz;
                        if (!(D <= D2MAX)) continue;
                        if (bu < 0 || D < bD || (D == bD && (u < bu || (u == bu && d < bd)))) {
                            bD = D; bu = u; bd = d;
                        }
                    }
                if (bu < 0 && c->nf_bridge_rows) {
                    const float ylo2 = y - WY2, yhi2 = y + WY2, zlo2 = z - WZ2, zhi2 = z + WZ2;
                    if (r - 2 >= 0) { /* (du, dd) = (1, 2) */
                        const float *cl_d2 = ROWCL(r - 2);
                        const int nx = window_list(cl_d2, ROWN(r - 2), ROWG(r - 2), use_grid, ylo2, yhi2, zlo2, zhi2, xlist);
                        for (int a = 0; a < nu; a++)
                            for (int b = 0; b < nx; b++) {
                                int u = ulist[a], d = xlist[b];
                                float t1 = cl_up[4 * u + 1] - y, t2 = y - cl_d2[4 * d + 1], ey = (t1 + t1) - t2;
                                float t3 = cl_up[4 * u + 2] - z, t4 = z - cl_d2[4 * d + 2], ez = (t3 + t3) - t4;
                                float pyy = ey * ey, pzz = ez * ez;
                                float D = pyy + pzz;
                                if (!(D <= D2MAX1)) continue;
                                if (bu < 0 || D < bD || (D == bD && (u < bu || (u == bu && d < bd)))) {
                                    bD = D; bu = u; bd = d; bdu = 1; bdd = 2;
                                }
                            }
                    }
                    if (r + 2 <= R - 1) { /* (du, dd) = (2, 1); on an exact tie of D the (1, 2) pair found above stays */
                        const float *cl_u2 = ROWCL(r + 2);
                        const int nx = window_list(cl_u2, ROWN(r + 2), ROWG(r + 2), use_grid, ylo2, yhi2, zlo2, zhi2, xlist);
                        for (int a = 0; a < nx; a++)
                            for (int b = 0; b < nd; b++) {
                                int u = xlist[a], d = dlist[b];
                                float t1 = cl_u2[4 * u + 1] - y, t2 = y - cl_dn[4 * d + 1], ey = t1 - (t2 + t2);
                                float t3 = cl_u2[4 * u + 2] - z, t4 = z - cl_dn[4 * d + 2], ez = t3 - (t4 + t4);
                                float pyy = ey * ey, pzz = ez * ez;
                                float D = pyy + pzz;
                                if (!(D <= D2MAX1)) continue;
                                if (bu < 0 || D < bD ||
                                    (D == bD && bdu == 2 && (u < bu || (u == bu && d < bd)))) {
                                    bD = D; bu = u; bd = d; bdu = 2; bdd = 1;
                                }
                            }
                    }
                }
                if (bu >= 0) {
                    lu = ro[r + bdu] + bu;
                    ld = ro[r - bdd] + bd;
                }
            }
            link_up[ro[r] + h] = lu;
            link_dn[ro[r] + h] = ld;
        }
    }
#undef ROWCL
#undef ROWN
#undef ROWG
    free(ulist);
    free(dlist);
    free(xlist);
}

/* Raw links for all instances.  link_up/link_dn: [n_clusters] GLOBAL cluster indices or -1. */
int orc_neighbours(const orc_config *c, const float *clusters, const int32_t *row_offsets, int32_t n_inst,
                   int32_t use_grid, int32_t *link_up, int32_t *link_dn) {
    const int R = c->n_rows;
    for (int inst = 0; inst < n_inst; inst++) {
        const int32_t *ro = row_offsets + (size_t)inst * R;
        orc_rowgrid *grids = (orc_rowgrid *)calloc((size_t)R, sizeof(orc_rowgrid));
        if (use_grid)
            for (int r = 0; r < R; r++) grid_build(&grids[r], c, inst, r, clusters + 4 * (size_t)ro[r], ro[r + 1] - ro[r]);
        neighbours_instance(c, clusters, ro, grids, use_grid, link_up, link_dn);
        if (use_grid)
            for (int r = 0; r < R; r++) grid_free(&grids[r]);
        free(grids);
    }
    return 0;
}

/* ------------------------------------------------------------------ S3: cleaning */

/* keep up[h]=u iff dn[u]==h; keep dn[h]=d iff up[d]==h; from the raw arrays into new ones. */
void orc_clean(int64_t n, const int32_t *up, const int32_t *dn, int32_t *cu, int32_t *cd) {
    for (int64_t h = 0; h < n; h++) {
        cu[h] = (up[h] >= 0 && dn[up[h]] == h) ? up[h] : -1;
        cd[h] = (dn[h] >= 0 && up[dn[h]] == h) ? dn[h] : -1;
    }
}

/* ------------------------------------------------------------------ S4: start hits, candidates */

/* SURVEY 8(c) S4.  start hit: cu>=0 and cd<0; chain follows cu; candidate iff length >= cand_min; it keeps the
 * first min(L,cand_max) hits.  Order = ascending global index of the start hit.  Returns the REQUIRED counts in
 * n_out[0]=n_start, n_out[1]=n_cand even if the capacities are smaller (nothing is written beyond them). */
void orc_candidates(const orc_config *c, int64_t n, const int32_t *cu, const int32_t *cd, int32_t *start_hits,
                    int64_t start_cap, int32_t *cand_hits /*[cap][cand_max]*/, int32_t *cand_n, int64_t cand_cap,
                    int64_t *n_out) {
    int64_t ns = 0, nc = 0;
    const int M = c->cand_max_hits;
    for (int64_t h = 0; h < n; h++) {
        if (!(cu[h] >= 0 && cd[h] < 0)) continue;
        if (ns < start_cap) start_hits[ns] = (int32_t)h;
        ns++;
        int len = 0;
        for (int32_t x = (int32_t)h; x >= 0; x = cu[x]) len++;
        if (len < c->cand_min_hits) continue;
        if (nc < cand_cap) {
            int k = 0;
            for (int32_t x = (int32_t)h; x >= 0 && k < M; x = cu[x]) cand_hits[nc * M + k++] = x;
            cand_n[nc] = k;
            for (; k < M; k++) cand_hits[nc * M + k] = -1;
        }
        nc++;
    }
    n_out[0] = ns;
    n_out[1] = nc;
}

/* ------------------------------------------------------------------ S5: Kalman track following */

/* arc length over chord ratio asin(a)/a */
static double asin_over(double a) { return fabs(a) < 1e-8 ? 1.0 + a * a / 6.0 : asin(a) / a; }

/* SURVEY 8(c) S5 "Transport by dx": exact helix for constant Bz (only Bz is respected).
 * p = (y, z, sinphi, dz/ds, q/pt).  P is a full symmetric 5x5 (row-major).  F (row-major 5x5) may be NULL.
 * Returns 0 on success, 1 if |sinphi| would exceed max_sinphi (outputs untouched). */
int orc_transport(const double p[5], const double P[25], double dx, double cB, double max_sinphi, double p1[5],
                  double P1[25], double F_out[25]) {
    const double y = p[0], z = p[1], s = p[2], t = p[3], k = p[4];
    const double kap = cB * k;
    const double s1 = s + kap * dx;
    if (fabs(s) > max_sinphi || fabs(s1) > max_sinphi) return 1;
    const double c0 = sqrt(1.0 - s * s), c1 = sqrt(1.0 - s1 * s1);
    const double tg = (s + s1) / (c0 + c1);
    const double sec2 = 1.0 + tg * tg;
    const double chord = dx * sqrt(sec2);
    const double a = 0.5 * kap * chord;
    const double dS = chord * asin_over(a);
    double F[25];
    for (int i = 0; i < 25; i++) F[i] = (i % 6 == 0) ? 1.0 : 0.0;
    F[0 * 5 + 2] = dx * sec2 * 0.5 * (1.0 / c0 + 1.0 / c1);
    F[0 * 5 + 4] = cB * dx * dx * sec2 / (2.0 * c1);
    F[1 * 5 + 2] = t * dx * tg / (c0 * c1);
    F[1 * 5 + 3] = dS;
    /* d(dS)/d(kappa) = (dx/c1 - dS)/kappa exactly (dS = (asin s1 - asin s)/kappa).  For |kappa dx| < 1e-4 the
     * difference cancels; there use its Taylor series 1/2 dx^2 g(s) + 1/3 kappa dx^3 g'(s) + ..., g = s/c^3, which to
     * second order is 1/2 dx^2 g(s + 2/3 kappa dx) (relative error O((kappa dx)^2) < 1e-8). */
    if (fabs(kap * dx) > 1e-4) {
        F[1 * 5 + 4] = cB * t * (dx / c1 - dS) / kap;
    } else {
        const double se = s + (2.0 / 3.0) * kap * dx, ce = sqrt(1.0 - se * se);
        F[1 * 5 + 4] = cB * t * 0.5 * dx * dx * se / (ce * ce * ce);
    }
    F[2 * 5 + 4] = cB * dx;
    double FP[25], Pn[25];
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            double acc = 0.0;
            for (int m = 0; m < 5; m++) acc += F[i * 5 + m] * P[m * 5 + j];
            FP[i * 5 + j] = acc;
        }
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            double acc = 0.0;
            for (int m = 0; m < 5; m++) acc += FP[i * 5 + m] * F[j * 5 + m];
            Pn[i * 5 + j] = acc;
        }
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) P1[i * 5 + j] = 0.5 * (Pn[i * 5 + j] + Pn[j * 5 + i]);
    p1[0] = y + dx * tg;
    p1[1] = z + t * dS;
    p1[2] = s1;
    p1[3] = t;
    p1[4] = k;
    if (F_out) memcpy(F_out, F, sizeof(F));
    return 0;
}

/* SURVEY 8(c) S5 "Update": two sequential scalar updates (y with sigma_y^2, then z with sigma_z^2). In place.
 * Returns the chi2 increment. */
double orc_update(double p[5], double P[25], double ym, double zm, double sy2, double sz2) {
    double chi2 = 0.0;
    for (int i = 0; i < 2; i++) {
        const double m = i ? zm : ym, r = i ? sz2 : sy2;
        const double S = P[i * 5 + i] + r;
        const double res = m - p[i];
        double K[5], Pi[5];
        for (int a = 0; a < 5; a++) { K[a] = P[a * 5 + i] / S; Pi[a] = P[i * 5 + a]; }
        chi2 += res * res / S;
        for (int a = 0; a < 5; a++) p[a] += K[a] * res;
        for (int a = 0; a < 5; a++)
            for (int b = 0; b < 5; b++) P[a * 5 + b] -= K[a] * Pi[b];
        for (int a = 0; a < 5; a++)
            for (int b = a + 1; b < 5; b++) {
                double v = 0.5 * (P[a * 5 + b] + P[b * 5 + a]);
                P[a * 5 + b] = P[b * 5 + a] = v;
            }
    }
    return chi2;
}

/* SURVEY 8(c) S5 "Seed": circle through three points in (x,y), dz/ds from the end points. */
void orc_seed(const double x[3], const double y[3], const double z[3], double cB, double p[5]) {
    const double ax = x[1] - x[0], ay = y[1] - y[0], bx = x[2] - x[0], by = y[2] - y[0];
    const double cross = ax * by - ay * bx;
    const double d01 = sqrt(ax * ax + ay * ay), d02 = sqrt(bx * bx + by * by);
    const double ex = x[2] - x[1], ey = y[2] - y[1];
    const double d12 = sqrt(ex * ex + ey * ey);
    const double kap = 2.0 * cross / (d01 * d02 * d12);
    const double phi0 = atan2(ay, ax) - asin(0.5 * kap * d01);
    const double S02 = d02 * asin_over(0.5 * kap * d02);
    p[0] = y[0];
    p[1] = z[0];
    p[2] = sin(phi0);
    p[3] = (z[2] - z[0]) / S02;
    p[4] = cB != 0.0 ? kap / cB : 0.0;
}

static int row_of(const int32_t *ro, int R, int32_t h) { /* ro: this instance's row offsets [R+1] */
    int lo = 0, hi = R; /* find r with ro[r] <= h < ro[r+1] */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (ro[mid] <= h) lo = mid; else hi = mid;
    }
    return lo;
}

/* SURVEY 8(c) S5 pick-up: nearest cluster of the row inside the window; fp32 test on the fp32-rounded prediction;
 * tie -> lowest local index.  Returns the local index or -1. */
static int pickup(const float *cl, int n, const orc_rowgrid *g, double y_pred, double z_pred, double wy_d,
                  double wz_d) {
    const float yp = (float)y_pred, zp = (float)z_pred, wy = (float)wy_d, wz = (float)wz_d;
    int best = -1;
    float bd2 = 0.0f;
    if (!g) {
        for (int j = 0; j < n; j++) {
            float dy = cl[4 * j + 1] - yp, dz = cl[4 * j + 2] - zp;
            if (!(fabsf(dy) <= wy && fabsf(dz) <= wz)) continue;
            float a = dy * dy, b = dz * dz, d2 = a + b;
            if (best < 0 || d2 < bd2 || (d2 == bd2 && j < best)) { best = j; bd2 = d2; }
        }
        return best;
    }
    if (n == 0) return -1;
    const float m = 1e-3f; /* bin margin: makes the visited bins a superset of the fp32 window test */
    int by0 = grid_bin1(yp - wy - m, g->y0, g->inv_cy, g->ny), by1 = grid_bin1(yp + wy + m, g->y0, g->inv_cy, g->ny);
    int bz0 = grid_bin1(zp - wz - m, g->z0, g->inv_cz, g->nz), bz1 = grid_bin1(zp + wz + m, g->z0, g->inv_cz, g->nz);
    for (int bz = bz0; bz <= bz1; bz++)
        for (int k = g->bin_start[bz * g->ny + by0]; k < g->bin_start[bz * g->ny + by1 + 1]; k++) {
            int j = g->perm[k];
            float dy = cl[4 * j + 1] - yp, dz = cl[4 * j + 2] - zp;
            if (!(fabsf(dy) <= wy && fabsf(dz) <= wz)) continue;
            float a = dy * dy, b = dz * dz, d2 = a + b;
            if (best < 0 || d2 < bd2 || (d2 == bd2 && j < best)) { best = j; bd2 = d2; }
        }
    return best;
}

static void unpack_cov_c(const double c[15], double P[25]) {
    int k = 0;
    for (int i = 0; i < 5; i++)
        for (int j = 0; j <= i; j++) { P[i * 5 + j] = c[k]; P[j * 5 + i] = c[k]; k++; }
}

static void pack_cov(const double P[25], double c[15]) {
    int k = 0;
    for (int i = 0; i < 5; i++)
        for (int j = 0; j <= i; j++) c[k++] = P[i * 5 + j];
}

/* One direction of the pick-up loop (SURVEY 8(c) S5 phases A and B).  step = +1 / -1.  (p,P) at row *r_cur. */
static void follow_dir(const orc_config *c, const float *clusters, const int32_t *ro, const orc_rowgrid *grids,
                       int step, double p[5], double P[25], int *r_cur, double *chi2, int32_t *hits /*[R]*/,
                       int *nhits, int *last_hit_row, double p_at_hit[5], double P_at_hit[25]) {
    const int R = c->n_rows;
    const double cB = curv_const(c), sy2 = (double)c->sigma_y * c->sigma_y, sz2 = (double)c->sigma_z * c->sigma_z;
    const double tanh_ = tan((double)c->half_angle_rad);
    int gap = 0, r = *r_cur;
    for (;;) {
        int rn = r + step;
        if (rn < 0 || rn >= R) break;
        double p1[5], P1[25];
        if (orc_transport(p, P, (double)c->row_x[rn] - (double)c->row_x[r], cB, c->kf_max_sinphi, p1, P1, NULL)) break;
        memcpy(p, p1, sizeof(p1));
        memcpy(P, P1, sizeof(P1));
        r = rn;
        if (fabs(p[0]) > (double)c->row_x[r] * tanh_ + c->kf_edge_margin) break;
        double wy = c->kf_gate_sigma * sqrt(P[0] + sy2), wz = c->kf_gate_sigma * sqrt(P[6] + sz2);
        if (wy > c->kf_win_max) wy = c->kf_win_max;
        if (wz > c->kf_win_max) wz = c->kf_win_max;
        int n = ro[r + 1] - ro[r];
        int j = pickup(clusters + 4 * (size_t)ro[r], n, grids ? &grids[r] : NULL, p[0], p[1], wy, wz);
        if (j >= 0) {
            const float *h = clusters + 4 * (size_t)(ro[r] + j);
            *chi2 += orc_update(p, P, (double)h[1], (double)h[2], sy2, sz2);
            hits[r] = ro[r] + j;
            (*nhits)++;
            gap = 0;
            *last_hit_row = r;
            if (p_at_hit) { memcpy(p_at_hit, p, 5 * sizeof(double)); memcpy(P_at_hit, P, 25 * sizeof(double)); }
        } else {
            gap++;
            if (gap > c->kf_max_gap) break;
        }
    }
    *r_cur = r;
}

/* Follow one candidate (global hit indices, rows increasing).  ro = row offsets of ITS instance [R+1] (global
 * indices).  grids: per-row grids of the instance or NULL for the linear scan.  hits: [R], filled with the global
 * cluster index attached in each row or -1. */
void orc_follow_one(const orc_config *c, const float *clusters, const int32_t *ro, const orc_rowgrid *grids,
                    const int32_t *cand, int n, orc_tracklet *t, int32_t *hits) {
    const int R = c->n_rows;
    const double cB = curv_const(c), sy2 = (double)c->sigma_y * c->sigma_y, sz2 = (double)c->sigma_z * c->sigma_z;
    memset(t, 0, sizeof(*t));
    for (int r = 0; r < R; r++) hits[r] = -1;
    int rows[64];
    for (int i = 0; i < n; i++) rows[i] = row_of(ro, R, cand[i]);
    const int ii[3] = {0, n / 2, n - 1};
    double sx[3], sy[3], sz[3];
    for (int m = 0; m < 3; m++) {
        const float *h = clusters + 4 * (size_t)cand[ii[m]];
        sx[m] = (double)c->row_x[rows[ii[m]]];
        sy[m] = (double)h[1];
        sz[m] = (double)h[2];
    }
    double p[5], P[25];
    orc_seed(sx, sy, sz, cB, p);
    if (!(fabs(p[2]) <= c->kf_max_sinphi)) return;
    memset(P, 0, sizeof(P));
    for (int i = 0; i < 5; i++) P[i * 5 + i] = c->kf_p0[i];
    double chi2 = 0.0;
    int nhits = 0, r = rows[0];
    /* phase A: candidate hits, then upward pick-up */
    for (int i = 0; i < n; i++) {
        if (i > 0) {
            double p1[5], P1[25];
            if (orc_transport(p, P, (double)c->row_x[rows[i]] - (double)c->row_x[r], cB, c->kf_max_sinphi, p1, P1, NULL))
                return;
            memcpy(p, p1, sizeof(p1));
            memcpy(P, P1, sizeof(P1));
            r = rows[i];
        }
        const float *h = clusters + 4 * (size_t)cand[i];
        chi2 += orc_update(p, P, (double)h[1], (double)h[2], sy2, sz2);
        hits[r] = cand[i];
        nhits++;
    }
    int last_row = r, dummy = r;
    follow_dir(c, clusters, ro, grids, +1, p, P, &r, &chi2, hits, &nhits, &last_row, NULL, NULL);
    /* phase B: one step back to the start row, no update there, then downward pick-up */
    {
        double p1[5], P1[25];
        if (orc_transport(p, P, (double)c->row_x[rows[0]] - (double)c->row_x[r], cB, c->kf_max_sinphi, p1, P1, NULL))
            return;
        memcpy(p, p1, sizeof(p1));
        memcpy(P, P1, sizeof(P1));
        r = rows[0];
    }
    double pr[5], Pr[25];
    memcpy(pr, p, sizeof(pr));
    memcpy(Pr, P, sizeof(Pr));
    int first_row = rows[0];
    dummy = first_row;
    follow_dir(c, clusters, ro, grids, -1, p, P, &r, &chi2, hits, &nhits, &dummy, pr, Pr);
    first_row = dummy;
    t->ok = 1;
    t->nhits = nhits;
    t->first_row = first_row;
    t->last_row = last_row;
    t->ref_row = first_row;
    memcpy(t->p, pr, sizeof(pr));
    pack_cov(Pr, t->cov);
    t->chi2 = chi2;
}

/* Follow all candidates.  cand_hits [n_cand][cand_max] global indices.  tracklets [n_cand]; trk_hits [n_cand][R]. */
int orc_follow(const orc_config *c, const float *clusters, const int32_t *row_offsets, int32_t n_inst,
               const int32_t *cand_hits, const int32_t *cand_n, int64_t n_cand, int32_t use_grid,
               orc_tracklet *tracklets, int32_t *trk_hits) {
    const int R = c->n_rows, M = c->cand_max_hits;
    int64_t ci = 0;
    for (int inst = 0; inst < n_inst && ci < n_cand; inst++) {
        const int32_t *ro = row_offsets + (size_t)inst * R;
        if (!(cand_hits[ci * M] < ro[R])) continue;
        orc_rowgrid *grids = NULL;
        if (use_grid) {
            grids = (orc_rowgrid *)calloc((size_t)R, sizeof(orc_rowgrid));
            for (int r = 0; r < R; r++) grid_build(&grids[r], c, inst, r, clusters + 4 * (size_t)ro[r], ro[r + 1] - ro[r]);
        }
        for (; ci < n_cand && cand_hits[ci * M] < ro[R]; ci++)
            orc_follow_one(c, clusters, ro, grids, cand_hits + ci * M, cand_n[ci], &tracklets[ci], trk_hits + ci * R);
        if (use_grid) {
            for (int r = 0; r < R; r++) grid_free(&grids[r]);
            free(grids);
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ S6: tracklet selector */

/* SURVEY 8(c) S6.  weight = (nhits, -candidate id); every cluster goes to the claiming tracklet of maximal weight;
 * a tracklet keeps the hits it owns and becomes a final track iff kept >= sel_min_hits; final tracks in ascending
 * candidate id.  Outputs: cluster_owner [n_clusters] final track index or -1; trk_cand [n_tracks]; trk_hit_offset
 * [n_tracks+1]; trk_hit_list (kept hits, rows increasing).  Returns the number of final tracks (required count;
 * nothing is written beyond trk_cap / hits_cap).  n_out[0] = n_tracks, n_out[1] = total kept hits. */
void orc_select(const orc_config *c, int64_t n_clusters, const orc_tracklet *tracklets, const int32_t *trk_hits,
                int64_t n_cand, int32_t *cluster_owner, int32_t *trk_cand, int64_t *trk_hit_offset,
                int32_t *trk_hit_list, int64_t trk_cap, int64_t hits_cap, int64_t *n_out) {
    const int R = c->n_rows;
    int32_t *best = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_clusters > 0 ? n_clusters : 1));
    for (int64_t h = 0; h < n_clusters; h++) { best[h] = -1; cluster_owner[h] = -1; }
    for (int64_t ci = 0; ci < n_cand; ci++) {
        if (!tracklets[ci].ok) continue;
        for (int r = 0; r < R; r++) {
            int32_t h = trk_hits[ci * R + r];
            if (h < 0) continue;
            int32_t b = best[h];
            /* ascending ci: an earlier claimant wins ties, so replace only on strictly more hits */
            if (b < 0 || tracklets[ci].nhits > tracklets[b].nhits) best[h] = (int32_t)ci;
        }
    }
    int64_t nt = 0, nh = 0;
    for (int64_t ci = 0; ci < n_cand; ci++) {
        if (!tracklets[ci].ok) continue;
        int kept = 0;
        for (int r = 0; r < R; r++) {
            int32_t h = trk_hits[ci * R + r];
            if (h >= 0 && best[h] == ci) kept++;
        }
        if (kept < c->sel_min_hits) continue;
        if (nt < trk_cap) {
            trk_cand[nt] = (int32_t)ci;
            trk_hit_offset[nt] = nh;
        }
        for (int r = 0; r < R; r++) {
            int32_t h = trk_hits[ci * R + r];
            if (h >= 0 && best[h] == ci) {
                if (nt < trk_cap) cluster_owner[h] = (int32_t)nt;
                if (nh < hits_cap && nt < trk_cap) trk_hit_list[nh] = h;
                nh++;
            }
        }
        nt++;
    }
    if (nt <= trk_cap) trk_hit_offset[nt] = nh;
    n_out[0] = nt;
    n_out[1] = nh;
    free(best);
}

/* ------------------------------------------------------------------ whole chain, per instance (for timing) */

/* Runs S1-S6 on every instance independently (optionally one OpenMP thread per instance) and reports only the
 * totals: n_out = {n_start, n_cand, n_tracklets, n_tracks, n_track_hits}.  Used by bench.py's cpu_baseline leg:
 * it executes exactly the stage functions above, instance by instance. */
int orc_track_count(const orc_config *c, const float *clusters, const int32_t *row_offsets, int32_t n_inst,
                    int32_t n_threads, int64_t *n_out) {
    const int R = c->n_rows, M = c->cand_max_hits;
    int64_t tot[5] = {0, 0, 0, 0, 0};
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads > 0 ? n_threads : 1)
#endif
    for (int inst = 0; inst < n_inst; inst++) {
        const int32_t *ro = row_offsets + (size_t)inst * R;
        const int32_t base = ro[0];
        const int64_t n = ro[R] - base;
        /* re-base this instance to local indices so that the stage functions see a one-instance problem */
        int32_t *lro = (int32_t *)malloc(sizeof(int32_t) * (size_t)(R + 1));
        for (int r = 0; r <= R; r++) lro[r] = ro[r] - base;
        const float *cl = clusters + 4 * (size_t)base;
        size_t nn = (size_t)(n > 0 ? n : 1);
        int32_t *up = (int32_t *)malloc(sizeof(int32_t) * nn), *dn = (int32_t *)malloc(sizeof(int32_t) * nn);
        int32_t *cu = (int32_t *)malloc(sizeof(int32_t) * nn), *cd = (int32_t *)malloc(sizeof(int32_t) * nn);
        orc_config ci = *c;
        /* the instance's side (z>=0 / z<0) must survive the re-basing: keep inst % sectors_per_event */
        int32_t *ro1 = lro;
        /* orc_neighbours derives the side from the instance index; emulate by calling the per-row code directly */
        {
            orc_rowgrid *grids = (orc_rowgrid *)calloc((size_t)R, sizeof(orc_rowgrid));
            for (int r = 0; r < R; r++) grid_build(&grids[r], &ci, inst, r, cl + 4 * (size_t)ro1[r], ro1[r + 1] - ro1[r]);
            neighbours_instance(&ci, cl, ro1, grids, 1, up, dn);
            orc_clean(n, up, dn, cu, cd);
            int64_t cnt[2];
            orc_candidates(&ci, n, cu, cd, NULL, 0, NULL, NULL, 0, cnt);
            int64_t nc = cnt[1];
            int32_t *ch = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nc * M + 1));
            int32_t *cn = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nc + 1));
            int32_t *sh = (int32_t *)malloc(sizeof(int32_t) * (size_t)(cnt[0] + 1));
            orc_candidates(&ci, n, cu, cd, sh, cnt[0], ch, cn, nc, cnt);
            orc_tracklet *tl = (orc_tracklet *)malloc(sizeof(orc_tracklet) * (size_t)(nc + 1));
            int32_t *th = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nc * R + 1));
            int64_t ntl = 0;
            for (int64_t k = 0; k < nc; k++) {
                orc_follow_one(&ci, cl, ro1, grids, ch + k * M, cn[k], &tl[k], th + k * R);
                ntl += tl[k].ok;
            }
            int32_t *owner = (int32_t *)malloc(sizeof(int32_t) * nn);
            int32_t *tc = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nc + 1));
            int64_t *tho = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nc + 2));
            int32_t *thl = (int32_t *)malloc(sizeof(int32_t) * nn);
            int64_t so[2];
            orc_select(&ci, n, tl, th, nc, owner, tc, tho, thl, nc + 1, (int64_t)nn, so);
#ifdef _OPENMP
#pragma omp critical
#endif
            {
                tot[0] += cnt[0]; tot[1] += nc; tot[2] += ntl; tot[3] += so[0]; tot[4] += so[1];
            }
            free(owner); free(tc); free(tho); free(thl); free(tl); free(th); free(ch); free(cn); free(sh);
            for (int r = 0; r < R; r++) grid_free(&grids[r]);
            free(grids);
        }
        free(up); free(dn); free(cu); free(cd); free(lro);
    }
    for (int i = 0; i < 5; i++) n_out[i] = tot[i];
    return 0;
}

int32_t orc_sizeof_tracklet(void) { return (int32_t)sizeof(orc_tracklet); }
int32_t orc_sizeof_config(void) { return (int32_t)sizeof(orc_config); }

/* ================================================================== PHASE 2: sector merger + refit
 *
 * PAPER.md:27 "The second phase merges the track segments found in the individual sectors to final tracks and
 * performs a track refit" (PAPER.md:33 names a GPU prototype of this fit).  The paper gives
 * no rule for either step; the reading is fixed in DESIGN.md ("Phase 2", readings M1-M4):
 *  M1 refit of one segment = the S5 filter over the hits the track KEPT in S6 only, each used once: seed from the
 *     kept hits (first, middle, last in row order) at the innermost hit, transport that state in one step to the
 *     outermost hit's row, reset the covariance to the prior P0, then filter inward hit by hit (transport, update).
 *     The state after the innermost hit is reported.  Any failed transport (|sinPhi| > max) -> no refit (ok = 0).
 *  M2 frame change between neighbouring sectors = exact rotation of the helix state about the beam axis by
 *     alpha = (sector difference) * 2 * half_angle; the rotated state sits at x' = x cos(alpha) + y sin(alpha) of the
 *     new frame (no longer a pad-row plane) and is transported to a row from there.
 *  M3 matching: segment B continues segment A outward iff same event/window (instance / sectors_per_event), same z
 *     side, neighbouring sectors (cyclic), first_row(B) > last_row(A), first_row(B) - last_row(A) <= 10; B's
 *     refitted state at its innermost hit, rotated into A's frame and transported to A's outermost row, must pass
 *     |dy| <= 2 cm and |dz| <= 2 cm against A's outermost HIT; among those B the one with the smallest dy^2 + dz^2
 *     (tie: lowest track index) is A's successor candidate, likewise every B picks its best A; a link exists iff the
 *     choice is mutual.
 *  M4 merged track = maximal chain of links, ordered inside out.  Its fit: M1 on the outermost segment, then at that
 *     segment's innermost hit the state is rotated (M2) into the next segment's frame, transported to that segment's
 *     outermost hit row, and the filter continues inward; reported at the innermost hit of the innermost segment, in
 *     its frame.  chi2 and the hit count run over the whole chain.  Merged tracks are listed in ascending index of
 *     their innermost segment.
 */

/* M2.  p at plane x of the old frame -> p1 at plane *x1 of the frame rotated by +alpha about the beam axis (the new
 * frame's x axis points alpha further in azimuth).  P (5x5, row-major) -> P1 = J P J^T with the exact Jacobian of the
 * map "state on the plane x = const of the old frame -> state on the plane x' = const of the new frame":
 * a variation of y moves the point along the old plane; it is brought back to the new plane by sliding along the
 * track, which scales y by cos(phi)/cos(phi'), shifts z by the dz/ds of that slide and turns the direction by the
 * curvature over it.  J (row-major) may be NULL.  Returns 0 on success, 1 (outputs untouched) if |sinPhi| exceeds
 * max_sinphi before or after the rotation or the rotated direction points backwards (cos <= 0). */
int orc_rotate(const double p[5], const double P[25], double x, double alpha, double cB, double max_sinphi,
               double p1[5], double P1[25], double *x1, double J_out[25]) {
    const double ca = cos(alpha), sa = sin(alpha);
    const double s = p[2];
    if (fabs(s) > max_sinphi) return 1;
    const double c = sqrt(1.0 - s * s);
    /* new frame: x' = x cos(a) + y sin(a), y' = -x sin(a) + y cos(a); direction angle phi' = phi - alpha */
    const double s1 = s * ca - c * sa, c1 = c * ca + s * sa;
    if (fabs(s1) > max_sinphi || c1 <= 0.0) return 1;
    *x1 = x * ca + p[0] * sa;
    p1[0] = -x * sa + p[0] * ca;
    p1[1] = p[1];
    p1[2] = s1;
    p1[3] = p[3];
    p1[4] = p[4];
    /* Jacobian at fixed new plane x' = *x1.  A shift dy of the point along the old plane changes x' by dy sin(a);
     * sliding back along the track by path length ds = -dy sin(a) / c1 (so that x' is restored) gives
     *   dy' = dy cos(a) + ds s1 = dy (cos(a) c1 - sin(a) s1) / c1 = dy c / c1,
     *   dz' = ds t = -dy sin(a) t / c1,   d(sinPhi') = c1 kappa ds = -dy sin(a) kappa   (kappa = cB k). */
    double J[25];
    for (int i = 0; i < 25; i++) J[i] = (i % 6 == 0) ? 1.0 : 0.0;
    J[0 * 5 + 0] = c / c1;
    J[1 * 5 + 0] = -sa * p[3] / c1;
    J[2 * 5 + 0] = -sa * cB * p[4];
    J[2 * 5 + 2] = c1 / c; /* d sin(phi - a) / d sin(phi) = cos(phi - a) / cos(phi) */
    double JP[25], Pn[25];
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            double acc = 0.0;
            for (int m = 0; m < 5; m++) acc += J[i * 5 + m] * P[m * 5 + j];
            JP[i * 5 + j] = acc;
        }
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) {
            double acc = 0.0;
            for (int m = 0; m < 5; m++) acc += JP[i * 5 + m] * J[j * 5 + m];
            Pn[i * 5 + j] = acc;
        }
    for (int i = 0; i < 5; i++)
        for (int j = 0; j < 5; j++) P1[i * 5 + j] = 0.5 * (Pn[i * 5 + j] + Pn[j * 5 + i]);
    if (J_out) memcpy(J_out, J, sizeof(J));
    return 0;
}

/* One segment of a merged track for orc_refit_chain: its sector-local frame (azimuth index) and its kept hits. */
typedef struct {
    int32_t sector;   /* geometric sector 0 .. sectors_per_event-1 (frame of the hits) */
    int32_t n;        /* kept hits */
    const int32_t *rows; /* [n] pad rows, increasing */
    const float *y;   /* [n] */
    const float *z;   /* [n] */
} orc_segment;

typedef struct {
    int32_t ok, nhits, nseg, first_row; /* first_row: innermost row of the innermost segment = reference row */
    double p[5], cov[15], chi2;
} orc_fit;

static double sector_alpha(const orc_config *c, int from_sector, int to_sector) {
    /* rotation angle from the frame of from_sector to the frame of to_sector, both on the same z side */
    const int half = c->sectors_per_event / 2;
    int d = (to_sector % half) - (from_sector % half);
    if (d > half / 2) d -= half;
    if (d < -half / 2) d += half;
    return 2.0 * (double)c->half_angle_rad * d;
}

/* M1 + M4: fit of a chain of segments given inside out (seg[0] innermost).  n_seg = 1 is the plain refit of one
 * track's kept hits. */
void orc_refit_chain(const orc_config *c, const orc_segment *seg, int n_seg, orc_fit *f) {
    const double cB = curv_const(c), sy2 = (double)c->sigma_y * c->sigma_y, sz2 = (double)c->sigma_z * c->sigma_z;
    memset(f, 0, sizeof(*f));
    f->nseg = n_seg;
    const orc_segment *o = &seg[n_seg - 1]; /* outermost segment: seed and start there */
    if (o->n < 3) return;
    const int ii[3] = {0, o->n / 2, o->n - 1};
    double sx[3], sy[3], sz[3];
    for (int m = 0; m < 3; m++) {
        sx[m] = (double)c->row_x[o->rows[ii[m]]];
        sy[m] = (double)o->y[ii[m]];
        sz[m] = (double)o->z[ii[m]];
    }
    double p[5], P[25], p1[5], P1[25];
    orc_seed(sx, sy, sz, cB, p);
    if (!(fabs(p[2]) <= c->kf_max_sinphi)) return;
    memset(P, 0, sizeof(P));
    for (int i = 0; i < 5; i++) P[i * 5 + i] = c->kf_p0[i];
    /* one step from the seed's plane (innermost hit of the outermost segment) to its outermost hit; only the state
     * is kept, the covariance restarts from the prior there */
    double x = (double)c->row_x[o->rows[o->n - 1]];
    if (o->n > 1) {
        if (orc_transport(p, P, x - sx[0], cB, c->kf_max_sinphi, p1, P1, NULL)) return;
        memcpy(p, p1, sizeof(p1));
    }
    memset(P, 0, sizeof(P));
    for (int i = 0; i < 5; i++) P[i * 5 + i] = c->kf_p0[i];
    double chi2 = 0.0;
    int nhits = 0;
    for (int s = n_seg - 1; s >= 0; s--) {
        const orc_segment *g = &seg[s];
        if (s < n_seg - 1) { /* M2: into this segment's frame, then to its outermost hit's row */
            double xr;
            if (orc_rotate(p, P, x, sector_alpha(c, seg[s + 1].sector, g->sector), cB, c->kf_max_sinphi, p1, P1, &xr, NULL))
                return;
            memcpy(p, p1, sizeof(p1));
            memcpy(P, P1, sizeof(P1));
            x = xr;
        }
        for (int i = g->n - 1; i >= 0; i--) {
            const double xi = (double)c->row_x[g->rows[i]];
            if (xi != x) {
                if (orc_transport(p, P, xi - x, cB, c->kf_max_sinphi, p1, P1, NULL)) return;
                memcpy(p, p1, sizeof(p1));
                memcpy(P, P1, sizeof(P1));
                x = xi;
            }
            chi2 += orc_update(p, P, (double)g->y[i], (double)g->z[i], sy2, sz2);
            nhits++;
        }
    }
    f->ok = 1;
    f->nhits = nhits;
    f->first_row = seg[0].rows[0];
    memcpy(f->p, p, sizeof(p));
    pack_cov(P, f->cov);
    f->chi2 = chi2;
}

/* Phase 2 on the S6 output (final tracks with their kept hits as global cluster indices, rows increasing).
 * trk_inst[t] = sector instance of track t.  Outputs: seg_fit [n_tracks] (M1 of every track alone), seg_next /
 * seg_prev [n_tracks] (M3 links, -1 none), merged tracks (M4) in ascending innermost segment: m_first [<= n_tracks],
 * m_fit.  Returns the number of merged tracks. */
int64_t orc_phase2(const orc_config *c, const float *clusters, const int32_t *row_offsets, int32_t n_inst,
                   int64_t n_tracks, const int32_t *trk_inst, const int64_t *trk_hit_offset, const int32_t *trk_hits,
                   orc_fit *seg_fit, int32_t *seg_next, int32_t *seg_prev, int32_t *m_first, orc_fit *m_fit) {
    const int R = c->n_rows, spe = c->sectors_per_event, half = spe / 2;
    const double cB = curv_const(c);
    const int64_t nh_all = n_tracks > 0 ? trk_hit_offset[n_tracks] : 0;
    int32_t *rows = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nh_all + 1));
    float *hy = (float *)malloc(sizeof(float) * (size_t)(nh_all + 1));
    float *hz = (float *)malloc(sizeof(float) * (size_t)(nh_all + 1));
    orc_segment *segs = (orc_segment *)malloc(sizeof(orc_segment) * (size_t)(n_tracks + 1));
    for (int64_t t = 0; t < n_tracks; t++) {
        const int32_t *ro = row_offsets + (size_t)trk_inst[t] * R;
        for (int64_t k = trk_hit_offset[t]; k < trk_hit_offset[t + 1]; k++) {
            rows[k] = row_of(ro, R, trk_hits[k]);
            hy[k] = clusters[4 * (size_t)trk_hits[k] + 1];
            hz[k] = clusters[4 * (size_t)trk_hits[k] + 2];
        }
        segs[t].sector = trk_inst[t] % spe;
        segs[t].n = (int32_t)(trk_hit_offset[t + 1] - trk_hit_offset[t]);
        segs[t].rows = rows + trk_hit_offset[t];
        segs[t].y = hy + trk_hit_offset[t];
        segs[t].z = hz + trk_hit_offset[t];
        orc_refit_chain(c, &segs[t], 1, &seg_fit[t]); /* M1 */
        seg_next[t] = seg_prev[t] = -1;
    }
    /* M3: best successor of every A, best predecessor of every B, then mutual choices.  Tracks of one window are
     * contiguous in t (instances ascending), so the scan over B is limited to that window. */
    int32_t *best_next = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_tracks + 1));
    int32_t *best_prev = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_tracks + 1));
    double *best_prev_d2 = (double *)malloc(sizeof(double) * (size_t)(n_tracks + 1));
    for (int64_t t = 0; t < n_tracks; t++) { best_next[t] = best_prev[t] = -1; best_prev_d2[t] = 0.0; }
    int64_t w0 = 0;
    while (w0 < n_tracks) {
        int64_t w1 = w0;
        while (w1 < n_tracks && trk_inst[w1] / spe == trk_inst[w0] / spe) w1++;
        for (int64_t a = w0; a < w1; a++) {
            const orc_segment *A = &segs[a];
            const int side_a = A->sector >= half, la = A->rows[A->n - 1];
            double bd2 = 0.0;
            for (int64_t b = w0; b < w1; b++) {
                const orc_segment *B = &segs[b];
                if (b == a || !seg_fit[b].ok || (B->sector >= half) != side_a) continue;
                int ds = (B->sector % half) - (A->sector % half);
                if (ds < 0) ds += half;
                if (ds != 1 && ds != half - 1) continue; /* neighbouring sectors, cyclic */
                const int fb = B->rows[0];
                if (!(fb > la && fb - la <= 10)) continue;
                double p1[5], P1[25], p2[5], P2[25], P0[25], xr;
                unpack_cov_c(seg_fit[b].cov, P0);
                if (orc_rotate(seg_fit[b].p, P0, (double)c->row_x[fb], sector_alpha(c, B->sector, A->sector), cB,
                               c->kf_max_sinphi, p1, P1, &xr, NULL))
                    continue;
                if (orc_transport(p1, P1, (double)c->row_x[la] - xr, cB, c->kf_max_sinphi, p2, P2, NULL)) continue;
                const double dy = p2[0] - (double)A->y[A->n - 1], dz = p2[1] - (double)A->z[A->n - 1];
                if (!(fabs(dy) <= 2.0 && fabs(dz) <= 2.0)) continue;
                const double d2 = dy * dy + dz * dz;
                if (best_next[a] < 0 || d2 < bd2) { best_next[a] = (int32_t)b; bd2 = d2; } /* b ascending: ties keep the lower */
                if (best_prev[b] < 0 || d2 < best_prev_d2[b]) { best_prev[b] = (int32_t)a; best_prev_d2[b] = d2; }
            }
        }
        w0 = w1;
    }
    for (int64_t a = 0; a < n_tracks; a++)
        if (best_next[a] >= 0 && best_prev[best_next[a]] == a) {
            seg_next[a] = best_next[a];
            seg_prev[best_next[a]] = (int32_t)a;
        }
    /* M4: chains, inside out, in ascending innermost segment */
    int64_t nm = 0;
    orc_segment chain[64];
    for (int64_t t = 0; t < n_tracks; t++) {
        if (seg_prev[t] >= 0) continue; /* not an innermost segment */
        int n = 0;
        for (int32_t x = (int32_t)t; x >= 0 && n < 64; x = seg_next[x]) chain[n++] = segs[x];
        m_first[nm] = (int32_t)t;
        if (n == 1) m_fit[nm] = seg_fit[t];
        else orc_refit_chain(c, chain, n, &m_fit[nm]);
        nm++;
    }
    free(rows); free(hy); free(hz); free(segs); free(best_next); free(best_prev); free(best_prev_d2);
    return nm;
}

int32_t orc_sizeof_fit(void) { return (int32_t)sizeof(orc_fit); }
int32_t orc_sizeof_segment(void) { return (int32_t)sizeof(orc_segment); }

/* ================================================================== TIME-COORDINATE TRACKING: vertex estimate
 *
 * PAPER.md:102 (Run 3, continuous read-out): "the tracking will run in time coordinate first to estimate the vertex
 * and only then convert to spacial coordinates".  In continuous read-out the z of a cluster is
 * its drift time, i.e. the true z plus an unknown offset common to all clusters of one collision (CFG:4 generates
 * exactly that).  Phases 1 and 2 are translation invariant in z, so they run on the time-like coordinate unchanged;
 * what is added here (readings T1-T3) is the step the paper names:
 *  T1 every merged track is extrapolated along its helix to the point of closest approach to the beam line (the z
 *     axis; a rotation between sector frames does not move it): with u = x c + y s, v = -x s + y c the position along
 *     and across the direction (c = cos phi, s = sin phi) and kappa = cB q/pt,
 *         ds = atan2(-kappa u, 1 + kappa v) / kappa   (-> -u / (1 + kappa v) for kappa -> 0),
 *         z_v = z + (dz/ds) ds,   dca = (sqrt((kappa u)^2 + (1 + kappa v)^2) - 1) / kappa   (-> v).
 *  T2 per event window (sectors_per_event instances) the z_v of the vertex-like tracks (ok, >= 30 hits, |dca| <= 3 cm)
 *     are histogrammed in 0.5 cm bins over [z_lo - 50, z_hi + 50) of the geometry; a bin is a vertex seed iff the sum
 *     of it and its two neighbours is >= 10 and is the maximum over the bins within +-4 (ties: the lowest bin wins);
 *     the vertex position is the mean z_v of the vertex-like tracks within 1.5 cm of the seed bin's centre.
 *  T3 every merged track (vertex-like or not) with a successful fit is assigned to the nearest vertex of its window
 *     within 3 cm in z_v, else to none; z_v(vertex) is the offset that converts the z of the track and of its
 *     clusters from the time-like to the spatial coordinate.
 */
void orc_track_vertex_z(const double p[5], double x, double cB, double *z_v, double *dca) {
    const double s = p[2], c = sqrt(1.0 - s * s), kap = cB * p[4];
    const double u = x * c + p[0] * s, v = -x * s + p[0] * c;
    const double a = -kap * u, b = 1.0 + kap * v;
    double ds, d;
    if (fabs(kap) * (fabs(u) + fabs(v)) < 1e-9) {
        ds = -u / b;
        d = v;
    } else {
        ds = atan2(a, b) / kap;
        d = (sqrt(a * a + b * b) - 1.0) / kap;
    }
    *z_v = p[1] + p[3] * ds;
    *dca = d;
}

#define ORC_VTX_BIN 0.5
#define ORC_VTX_MARGIN 50.0
#define ORC_VTX_MAX_PER_WINDOW 64

/* T1-T3 on the merged tracks of orc_phase2.  m_inst[m] = sector instance of the innermost segment.  Outputs per
 * merged track: trk_zv, trk_dca, trk_vtx (global vertex index or -1); vertices (ascending window, then bin): vtx_z,
 * vtx_window, vtx_ntracks (assigned tracks).  Returns the number of vertices (nothing is written beyond vtx_cap). */
int64_t orc_vertices(const orc_config *c, int64_t n_merged, const orc_fit *m_fit, const int32_t *m_inst, double *trk_zv,
                     double *trk_dca, int32_t *trk_vtx, double *vtx_z, int32_t *vtx_window, int32_t *vtx_ntracks,
                     int64_t vtx_cap) {
    const double cB = curv_const(c);
    const int spe = c->sectors_per_event;
    const double h_lo = (double)c->z_lo - ORC_VTX_MARGIN, h_hi = (double)c->z_hi + ORC_VTX_MARGIN;
    /* the z < 0 side mirrors the range: use the union [-h, h] with h = max(|h_lo|, |h_hi|) */
    const double h = fabs(h_lo) > fabs(h_hi) ? fabs(h_lo) : fabs(h_hi);
    const int nb = (int)ceil(2.0 * h / ORC_VTX_BIN);
    int32_t *hist = (int32_t *)malloc(sizeof(int32_t) * (size_t)nb);
    char *like = (char *)malloc((size_t)(n_merged > 0 ? n_merged : 1));
    for (int64_t m = 0; m < n_merged; m++) {
        trk_zv[m] = trk_dca[m] = 0.0;
        trk_vtx[m] = -1;
        like[m] = 0;
        if (!m_fit[m].ok) continue;
        orc_track_vertex_z(m_fit[m].p, (double)c->row_x[m_fit[m].first_row], cB, &trk_zv[m], &trk_dca[m]);
        like[m] = m_fit[m].nhits >= 30 && fabs(trk_dca[m]) <= 3.0;
    }
    int64_t nv = 0, w0 = 0;
    while (w0 < n_merged) { /* merged tracks are in ascending innermost segment, hence in ascending window */
        int64_t w1 = w0;
        const int win = m_inst[w0] / spe;
        while (w1 < n_merged && m_inst[w1] / spe == win) w1++;
        memset(hist, 0, sizeof(int32_t) * (size_t)nb);
        for (int64_t m = w0; m < w1; m++)
            if (like[m]) {
                const int b = (int)floor((trk_zv[m] + h) / ORC_VTX_BIN);
                if (b >= 0 && b < nb) hist[b]++;
            }
        const int64_t nv0 = nv;
        int n_here = 0;
        for (int b = 0; b < nb && n_here < ORC_VTX_MAX_PER_WINDOW; b++) {
#define SUM3(q) ((q) < 0 || (q) >= nb ? 0 : hist[q] + ((q) > 0 ? hist[(q) - 1] : 0) + ((q) + 1 < nb ? hist[(q) + 1] : 0))
            const int s3 = SUM3(b);
            if (s3 < 10) continue;
            int is_max = 1;
            for (int q = b - 4; q <= b + 4 && is_max; q++) {
                if (q == b) continue;
                const int o = SUM3(q);
                if (o > s3 || (o == s3 && q < b)) is_max = 0;
            }
#undef SUM3
            if (!is_max) continue;
            const double zc = -h + (b + 0.5) * ORC_VTX_BIN;
            double sum = 0.0;
            int n = 0;
            for (int64_t m = w0; m < w1; m++)
                if (like[m] && fabs(trk_zv[m] - zc) <= 1.5) { sum += trk_zv[m]; n++; }
            if (nv < vtx_cap) {
                vtx_z[nv] = sum / n;
                vtx_window[nv] = win;
                vtx_ntracks[nv] = 0;
            }
            nv++;
            n_here++;
        }
        for (int64_t m = w0; m < w1; m++) { /* T3 */
            if (!m_fit[m].ok) continue;
            double best = 0.0;
            for (int64_t k = nv0; k < nv && k < vtx_cap; k++) {
                const double d = fabs(trk_zv[m] - vtx_z[k]);
                if (d <= 3.0 && (trk_vtx[m] < 0 || d < best)) { trk_vtx[m] = (int32_t)k; best = d; }
            }
            if (trk_vtx[m] >= 0) vtx_ntracks[trk_vtx[m]]++;
        }
        w0 = w1;
    }
    free(hist);
    free(like);
    return nv;
}
