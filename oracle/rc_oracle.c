/*
 * rc_oracle.c — fp64 CPU oracle for the radiance-cascades formal solution (flatland).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant with the CUDA path under paper_2408_14425_b200/csrc/.
 *
 * It follows the paper (Osborne & Sannikov, arxiv 2408.14425; /root/reference/PAPER.md) step by
 * step, in the paper's order, in double precision, with no blocking, tiling or early exit:
 *
 *   radiance interval  R_{a,b}(p,w) = [I, tau] along p + t w, t in [a,b]   PAPER.md:137-139 (eq. 9)
 *   per-cell update    tau += chi ds; I <- I e^{-chi ds} + (eta/chi)(1-e^{-chi ds})
 *                                                                         PAPER.md:297-300 (eq. 16)
 *   grid walk          uniform-grid DDA
 *   cascade i          probe spacing 2^i, 4^(i+1) directions, shell [t_i,t_{i+1}],
 *                      t_i = c0 (4^i-1)/3  (eq. 12-13 with alpha = 2)
 *   cascade 0 probes   at the cell centres
 *   top cascade        runs to the domain edge; boundary intensity there
 *   merge              near interval attenuates the far one (eq. 11)
 *   interpolation      bilinear over the 4 parent probes of cascade i+1,
 *                      each interval merged with its 4 children in the cone PAPER.md:199-207
 *   lattice edge       parent lookup clamped
 *   J                  mean over the 4 merged cascade-0 directions         PAPER.md:36 (eq. 1), 191
 *   2.5D  each flatland ray replaced by rays with the same projection and
 *                      different inclinations to the invariant axis: same cells, path length
 *                      ds / sin(inclination); J = sum_m w_m J_m
 *                      (rc_oracle_solve_scaled does one inclination; oracle/rc_oracle.py sums)
 *   sparsity  "we can first determine the cells of interest ... This flag then defines the
 *                      probes of cascade 0 that may be involved ... Their bilinear "parents" are recursively
 *                      flagged up to the maximum cascade, and the radiance intervals are only computed for these
 *                      flagged probes, and non-flagged cells are treated as transparent with no emission"
 *                                                                         PAPER.md:380 (rc_oracle_solve_active)
 *
 * Readings where the paper is silent or garbled are DESIGN.md §3 (G1..G19 of SURVEY.md §8(c)).
 * The only loop restructuring relative to SURVEY.md's listing: the wavelength loop is innermost
 * (the cell segments of a ray do not depend on the wavelength), which changes no arithmetic of
 * any (probe, direction, wavelength) triple.
 *
 * The per-segment update is written in the equivalent front-to-back form ("works
 * equally well"):  I += T * eta*ds*f(chi ds),  T *= exp(-chi ds),  f(x) = (1-e^{-x})/x, f(0)=1,
 * which is eq. 16 rearranged and has the chi -> 0 limit built in (reading G11).  A back-to-front
 * variant (eq. 16 literally, towards the probe) is kept beside it and tested to agree (G13).
 *
 * Pinned by tests/test_oracle_pins.py (closed forms, invariants, brute force).  Not pinned against
 * any number printed in the paper (it prints none for this path): the direction convention (G4)
 * and the probe placement for i >= 1 (G5) are "parity unpinned vs the paper" — see DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int nx, ny, L;
    const float *chi, *eta; /* [ny][nx][L], wavelength fastest, y = 0 bottom row */
    double path_scale;      /* true path length per unit length in the plane: 1 in flatland; 1/sin(inclination
                               to the invariant axis) for the inclined rays of the 2.5D scheme (PAPER.md:281:
                               "the same x-z projection and different inclinations in y") */
    /* velocity-dependent line mode ("velocity-dependent terms (spectral lines) are computed
       on the fly for each ray given its specific direction, and thus projected plasma velocity"): when
       `line` is set, chi/eta above are unused and the opacity and emissivity of cell c at wavelength l
       seen by a ray are those of cell_chi_eta() below */
    const float *line;  /* [ny][nx][6]: chi_c, S_c, chi_line, S_line, v_x, v_y (velocities in Doppler widths) */
    const double *xl;   /* [L] wavelengths as offsets from line centre, in Doppler widths */
    double vel_scale;   /* 2.5D line mode: an inclined ray with direction cosine mu to the invariant axis has the
                           in-plane direction sqrt(1-mu^2) (wx, wy); velocities are in the plane, so v.n is scaled by
                           sqrt(1-mu^2) = 1/path_scale.  1 in flatland. */
    const unsigned char *active; /* [ny][nx] or NULL: cells of interest; a cell that is not flagged
                                    is "treated as transparent with no emission" whatever chi, eta hold there */
} grid_t;

/* Opacity and emissivity of cell `cell` at wavelength l for the photons that travel along a ray traced
 * from its probe in direction (wx, wy): they move along n = -(wx, wy), so in the observer's frame the line
 * of a cell with velocity v is centred at x = v.n:
 *     a = x_l - v.n ,  phi = exp(-a^2)/sqrt(pi) ,
 *     chi = chi_c + chi_line phi ,  eta = chi_c S_c + chi_line S_line phi . */
static void cell_chi_eta(const grid_t *g, int cell, int l, double wx, double wy, double *chi, double *eta) {
    if (g->active && !g->active[cell]) { *chi = 0.0; *eta = 0.0; return; }
    if (!g->line) {
        size_t c = (size_t)cell * g->L + l;
        *chi = (double)g->chi[c];
        *eta = (double)g->eta[c];
        return;
    }
    const float *f = g->line + (size_t)cell * 6;
    double a = g->xl[l] + g->vel_scale * ((double)f[4] * wx + (double)f[5] * wy);
    double phi = exp(-a * a) / sqrt(M_PI);
    *chi = (double)f[0] + (double)f[2] * phi;
    *eta = (double)f[0] * (double)f[1] + (double)f[2] * (double)f[3] * phi;
}

typedef struct {
    int cell;  /* y*nx + x */
    double ds; /* path length inside the cell */
} seg_t;

/* Interval ends, eq. 12-13 with alpha = 2 as fixed by BASELINE.json: t_i = c0 (4^i - 1)/3. */
static double t_of(int i, double c0) { return c0 * (pow(4.0, (double)i) - 1.0) / 3.0; }

/* f(x) = (1 - exp(-x))/x, f(0) = 1 (reading G11). */
static double f_emis(double x) { return x == 0.0 ? 1.0 : -expm1(-x) / x; }

/*
 * Cell segments of {p + t w : ta <= t <= tb} inside the box [0,nx] x [0,ny]: standard 2D DDA
 * (PAPER.md:314).  Probes lie inside the box and the box is convex, so a ray whose start point
 * p + ta w is outside never re-enters (reading G10: outside is vacuum).  Each crossing parameter
 * is recomputed from the grid line it belongs to, not accumulated.  Returns the segment count.
 */
static int dda_segments(int nx, int ny, double px, double py, double wx, double wy, double ta,
                        double tb, seg_t *out) {
    double x0 = px + ta * wx, y0 = py + ta * wy;
    if (!(x0 >= 0.0 && x0 <= nx && y0 >= 0.0 && y0 <= ny)) return 0;
    int ix = (int)floor(x0), iy = (int)floor(y0);
    if ((double)ix == x0 && wx < 0.0) ix--; /* on a grid line: the cell the ray moves into */
    if ((double)iy == y0 && wy < 0.0) iy--;
    if (ix < 0 || ix >= nx || iy < 0 || iy >= ny) return 0;
    int sx = wx > 0.0 ? 1 : -1, sy = wy > 0.0 ? 1 : -1;
    int gx = wx > 0.0 ? ix + 1 : ix; /* next grid line crossed in x */
    int gy = wy > 0.0 ? iy + 1 : iy;
    double tmx = wx != 0.0 ? (gx - px) / wx : INFINITY;
    double tmy = wy != 0.0 ? (gy - py) / wy : INFINITY;
    double t = ta;
    int n = 0;
    for (;;) {
        double tn = fmin(fmin(tmx, tmy), tb);
        double ds = tn - t;
        if (ds > 0.0) {
            out[n].cell = iy * nx + ix;
            out[n].ds = ds;
            n++;
        }
        if (tn >= tb) break;
        int stepx = tmx <= tmy, stepy = tmy <= tmx; /* a tie is a corner: step both */
        if (stepx) { ix += sx; gx += sx; tmx = (gx - px) / wx; }
        if (stepy) { iy += sy; gy += sy; tmy = (gy - py) / wy; }
        if (ix < 0 || ix >= nx || iy < 0 || iy >= ny) break;
        t = tn;
    }
    return n;
}

/*
 * Cascade 0: the four directions are the diagonals (reading G4) and start at a cell centre
 * (PAPER.md:312), so they pass exactly through cell corners; the segments are written in closed
 * form (reading G12): cell m along the diagonal covers t in [sqrt2 (m - 1/2), sqrt2 (m + 1/2)].
 * quadrant q = 0..3: (+,+), (-,+), (-,-), (+,-), i.e. theta = pi/4 + q pi/2.
 */
static int diag_segments(int nx, int ny, int cx, int cy, int q, double ta, double tb, seg_t *out) {
    static const int SX[4] = {1, -1, -1, 1}, SY[4] = {1, 1, -1, -1};
    const double r2 = sqrt(2.0);
    int n = 0;
    for (int m = 0;; m++) {
        int ix = cx + m * SX[q], iy = cy + m * SY[q];
        if (ix < 0 || ix >= nx || iy < 0 || iy >= ny) break;
        double lo = m == 0 ? 0.0 : r2 * (m - 0.5), hi = r2 * (m + 0.5);
        if (lo >= tb) break;
        if (lo < ta) lo = ta;
        if (hi > tb) hi = tb;
        if (hi > lo) {
            out[n].cell = iy * nx + ix;
            out[n].ds = hi - lo;
            n++;
        }
    }
    return n;
}

/* eq. 16 along the segments, front-to-back, all wavelengths: I[l], T[l] = exp(-tau[l]). */
static void integrate_ftb(const grid_t *g, const seg_t *seg, int n, double wx, double wy, double *I, double *T) {
    for (int l = 0; l < g->L; l++) {
        double Il = 0.0, Tl = 1.0;
        for (int s = 0; s < n; s++) {
            double chi, eta;
            cell_chi_eta(g, seg[s].cell, l, wx, wy, &chi, &eta);
            double ds = seg[s].ds * g->path_scale, x = chi * ds;
            Il += Tl * eta * ds * f_emis(x);
            Tl *= exp(-x);
        }
        I[l] = Il;
        T[l] = Tl;
    }
}

/* eq. 16 literally: start at the far end with I = 0 and integrate towards the probe
 * ("back-to-front"); tau accumulated, T = exp(-tau). */
static void integrate_btf(const grid_t *g, const seg_t *seg, int n, double wx, double wy, double *I, double *T) {
    for (int l = 0; l < g->L; l++) {
        double Il = 0.0, tau = 0.0;
        for (int s = n - 1; s >= 0; s--) {
            double chi, eta;
            cell_chi_eta(g, seg[s].cell, l, wx, wy, &chi, &eta);
            double ds = seg[s].ds * g->path_scale, x = chi * ds;
            tau += x;
            Il = Il * exp(-x) + (chi > 0.0 ? (eta / chi) * (-expm1(-x)) : eta * ds);
        }
        I[l] = Il;
        T[l] = exp(-tau);
    }
}

/* Position of child probe a among the parents of the next cascade (n of them per axis):
 * a/2 - 1/4 in parent index units (reading G5), indices clamped at the lattice edge
 * (reading G6). */
static void parent_axis(int a, int n, int *q0, int *q1, double *frac) {
    int base;
    if ((a & 1) == 0) { base = a / 2 - 1; *frac = 0.75; }
    else              { base = (a - 1) / 2; *frac = 0.25; }
    int b1 = base + 1;
    *q0 = base < 0 ? 0 : (base > n - 1 ? n - 1 : base);
    *q1 = b1 < 0 ? 0 : (b1 > n - 1 ? n - 1 : b1);
}

/* ------------------------------------------------------------------------------------------ */
/* Exported entry points (host pointers throughout).                                           */
/* ------------------------------------------------------------------------------------------ */

/* Segments of one ray, for the tests that pin the DDA.  diag_q >= 0 selects the cascade-0 closed
 * form from the centre of cell (floor(px), floor(py)); otherwise direction angle theta.
 * cells[] / ds[] must hold nx + ny + 4 entries.  Returns the count. */
int rc_oracle_ray_segments(int nx, int ny, double px, double py, double theta, int diag_q,
                           double ta, double tb, int *cells, double *ds) {
    seg_t *seg = (seg_t *)malloc(sizeof(seg_t) * (size_t)(nx + ny + 4));
    int n = diag_q >= 0 ? diag_segments(nx, ny, (int)floor(px), (int)floor(py), diag_q, ta, tb, seg)
                        : dda_segments(nx, ny, px, py, cos(theta), sin(theta), ta, tb, seg);
    for (int s = 0; s < n; s++) { cells[s] = seg[s].cell; ds[s] = seg[s].ds; }
    free(seg);
    return n;
}

/* One radiance interval [I[l], T[l]] (eq. 9) of one ray; order: 0 front-to-back, 1 back-to-front. */
int rc_oracle_interval(const float *chi, const float *eta, int nx, int ny, int L, double px,
                       double py, double theta, int diag_q, double ta, double tb, int order,
                       double *I, double *T) {
    grid_t g = {nx, ny, L, chi, eta, 1.0, NULL, NULL, 1.0, NULL};
    seg_t *seg = (seg_t *)malloc(sizeof(seg_t) * (size_t)(nx + ny + 4));
    int n = diag_q >= 0 ? diag_segments(nx, ny, (int)floor(px), (int)floor(py), diag_q, ta, tb, seg)
                        : dda_segments(nx, ny, px, py, cos(theta), sin(theta), ta, tb, seg);
    if (diag_q >= 0) theta = 2.0 * M_PI * (diag_q + 0.5) / 4.0;
    if (order == 0) integrate_ftb(&g, seg, n, cos(theta), sin(theta), I, T);
    else integrate_btf(&g, seg, n, cos(theta), sin(theta), I, T);
    free(seg);
    return n;
}

/* Merge operator, eq. 11 in the physical reading G1: near = [a,b], far = [b,c]. */
void rc_oracle_merge(double I_near, double tau_near, double I_far, double tau_far, double *I_out,
                     double *tau_out) {
    *I_out = I_near + exp(-tau_near) * I_far;
    *tau_out = tau_near + tau_far;
}

typedef struct {
    int64_t intervals[16]; /* intervals computed per cascade (inside the requested window) */
    int64_t segments[16];  /* cell segments walked per cascade (per wavelength)             */
} rc_oracle_counts;

/*
 * The whole path for the cascade-0 cells x0 <= x < x1, y0 <= y < y1 (the full grid for the full
 * solve).  Cascade i is computed only on the probes the window's cells depend on through the
 * bilinear parent lookups; every computed number is the same as in the full solve.
 *
 *   J_out   [(y1-y0)][(x1-x0)][L]  double
 *   Jbar_out[(y1-y0)][(x1-x0)]     double, = sum_l w[l] J[..][l]; may be NULL
 *   I_below/I_above/w: [L] or NULL (zero / zero / ones)
 *   dump_cascade >= 0: also write that cascade's intervals before merging (dump_I, dump_T) and
 *   after merging (dump_M), each [wy][wx][N][L] over that cascade's probe window; dump_win gets
 *   {ax0, ax1, by0, by1} (inclusive probe index ranges).
 *   order: bit 0: 0 front-to-back, 1 back-to-front (G13); bit 1: the bilinear fix.
 * Returns 0, or -1 on bad arguments / -2 out of memory.
 */
static int solve_impl(const float *chi, const float *eta, const float *line, const double *xl, int nx, int ny,
                      int L, int ncasc,
                           double c0, const float *I_below, const float *I_above, const float *w,
                           int x0, int x1, int y0, int y1, double *J_out, double *Jbar_out, int nthreads,
                           int order, int dump_cascade, double *dump_I, double *dump_T, double *dump_M,
                           int *dump_win, rc_oracle_counts *counts, double path_scale,
                           const unsigned char *active) {
    if (!((chi && eta) || (line && xl)) || !J_out || nx <= 0 || ny <= 0 || L <= 0 || ncasc < 1 || ncasc > 15)
        return -1;
    int top = ncasc - 1;
    if (nx % (1 << top) || ny % (1 << top)) return -1; /* reading G19 */
    if (x0 < 0 || y0 < 0 || x1 > nx || y1 > ny || x0 >= x1 || y0 >= y1) return -1;
    grid_t g = {nx, ny, L, chi, eta, path_scale, line, xl, 1.0 / path_scale, active};
    const int fix = (order & 2) != 0; /* order: bit 0 = back-to-front (G13), bit 1 = bilinear fix */
    if (counts) memset(counts, 0, sizeof(*counts));
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    /* probe windows per cascade (inclusive), propagated through parent_axis */
    int ax0[16], ax1[16], by0[16], by1[16];
    ax0[0] = x0; ax1[0] = x1 - 1; by0[0] = y0; by1[0] = y1 - 1;
    for (int i = 0; i < top; i++) {
        int npx = nx >> (i + 1), npy = ny >> (i + 1), q0, q1; double fr;
        parent_axis(ax0[i], npx, &q0, &q1, &fr); ax0[i + 1] = q0;
        parent_axis(ax1[i], npx, &q0, &q1, &fr); ax1[i + 1] = q1;
        parent_axis(by0[i], npy, &q0, &q1, &fr); by0[i + 1] = q0;
        parent_axis(by1[i], npy, &q0, &q1, &fr); by1[i + 1] = q1;
    }
    /* Sparsity: flag[0] = the cells of interest = the cascade-0 probes that may be involved; the
     * bilinear parents of every flagged probe of cascade i are flagged in cascade i+1, up to the top.  Intervals are
     * computed for flagged probes only; everything else in a cascade's storage stays NaN, so a read of a value
     * that was never computed would poison J (the pins check it never happens).  active == NULL: all flagged. */
    unsigned char *flag[16];
    for (int i = 0; i <= top; i++) flag[i] = NULL;
    if (active) {
        for (int i = 0; i <= top; i++) {
            flag[i] = (unsigned char *)calloc((size_t)(nx >> i) * (ny >> i), 1);
            if (!flag[i]) { for (int j = 0; j < i; j++) free(flag[j]); return -2; }
        }
        for (size_t c = 0; c < (size_t)nx * ny; c++) flag[0][c] = active[c] != 0;
        for (int i = 0; i < top; i++) {
            int npx = nx >> i, npy = ny >> i, upx = npx / 2, upy = npy / 2;
            for (int b = 0; b < npy; b++)
                for (int a = 0; a < npx; a++) {
                    if (!flag[i][(size_t)b * npx + a]) continue;
                    int a0, a1, b0, b1; double fr;
                    parent_axis(a, upx, &a0, &a1, &fr);
                    parent_axis(b, upy, &b0, &b1, &fr);
                    flag[i + 1][(size_t)b0 * upx + a0] = 1; flag[i + 1][(size_t)b0 * upx + a1] = 1;
                    flag[i + 1][(size_t)b1 * upx + a0] = 1; flag[i + 1][(size_t)b1 * upx + a1] = 1;
                }
        }
    }
    double *Mup = NULL; /* merged cascade i+1: [wy][wx][N_{i+1}][L] */
    int upx0 = 0, upy0 = 0, upwx = 0;
    long upN = 0;
    int status = 0;
    for (int i = top; i >= 0; i--) {
        int s = 1 << i;
        int npx = nx / s, npy = ny / s;
        long N = 1L << (2 * (i + 1)); /* 4^(i+1) directions */
        double ta = t_of(i, c0), tb = i == top ? INFINITY : t_of(i + 1, c0); /* G8 */
        int wx = ax1[i] - ax0[i] + 1, wy = by1[i] - by0[i] + 1;
        double *M = (double *)malloc(sizeof(double) * (size_t)wx * wy * N * L);
        if (!M) { status = -2; break; }
        if (active) for (size_t q = 0; q < (size_t)wx * wy * N * L; q++) M[q] = NAN;
        int64_t nflagged = 0;
        for (int b = by0[i]; b <= by1[i]; b++)
            for (int a = ax0[i]; a <= ax1[i]; a++) nflagged += !active || flag[i][(size_t)b * npx + a];
        int dump = i == dump_cascade;
        if (dump && dump_win) { dump_win[0] = ax0[i]; dump_win[1] = ax1[i]; dump_win[2] = by0[i]; dump_win[3] = by1[i]; }
        int64_t nseg_total = 0;
#pragma omp parallel reduction(+ : nseg_total)
        {
            seg_t *seg = (seg_t *)malloc(sizeof(seg_t) * (size_t)(nx + ny + 4));
            double *I = (double *)malloc(sizeof(double) * L);
            double *T = (double *)malloc(sizeof(double) * L);
#pragma omp for collapse(3) schedule(dynamic, 16)
            for (int b = by0[i]; b <= by1[i]; b++) {
                for (int a = ax0[i]; a <= ax1[i]; a++) {
                    for (long k = 0; k < N; k++) {
                        if (active && !flag[i][(size_t)b * npx + a]) continue; /* not flagged: not computed */
                        double px = (a + 0.5) * s, py = (b + 0.5) * s; /* PAPER.md:312, reading G5 */
                        double theta = 2.0 * M_PI * (k + 0.5) / (double)N; /* reading G4 */
                        size_t o = ((((size_t)(b - by0[i])) * wx + (a - ax0[i])) * N + k) * L;
                        if (fix && i < top) {
                            /* Bilinear fix: "each radiance interval in cascade i is traced from its
                             * usual starting position to the starting position of the associated child cone on each
                             * of the four probes of cascade i+1 that are normally bilinearly interpolated ... the four
                             * distinct radiance intervals are each merged with their associated samples from cascade
                             * i+1, and then averaged using the usual bilinear weights".  Reading G24: the child cone of
                             * direction k on parent q starts at P_q + t_{i+1} w_k; its sample is the mean of the 4
                             * children 4k..4k+3 of q.  A sub-ray whose start lies outside the box is vacuum (G10). */
                            int a0, a1, b0, b1; double fa, fb;
                            parent_axis(a, npx / 2, &a0, &a1, &fa);
                            parent_axis(b, npy / 2, &b0, &b1, &fb);
                            for (int l = 0; l < L; l++) M[o + l] = 0.0;
                            double Ax = px + ta * cos(theta), Ay = py + ta * sin(theta);
                            for (int slot = 0; slot < 4; slot++) {
                                int aq = (slot & 1) ? a1 : a0, bq = (slot & 2) ? b1 : b0;
                                double wq = ((slot & 1) ? fa : 1.0 - fa) * ((slot & 2) ? fb : 1.0 - fb);
                                double Bx = (aq + 0.5) * (2 * s) + tb * cos(theta), By = (bq + 0.5) * (2 * s) + tb * sin(theta);
                                double dx = Bx - Ax, dy = By - Ay, len = sqrt(dx * dx + dy * dy);
                                int n = dda_segments(nx, ny, Ax, Ay, dx / len, dy / len, 0.0, len, seg);
                                nseg_total += n;
                                if (order & 1) integrate_btf(&g, seg, n, dx / len, dy / len, I, T);
                                else integrate_ftb(&g, seg, n, dx / len, dy / len, I, T);
                                for (int l = 0; l < L; l++) {
                                    double U = 0.0;
                                    for (int j = 0; j < 4; j++) {
                                        long kk = 4 * k + j;
                                        U += Mup[((((size_t)(bq - upy0)) * upwx + (aq - upx0)) * upN + kk) * L + l];
                                    }
                                    M[o + l] += wq * (I[l] + T[l] * U / 4.0);
                                }
                            }
                            if (dump) for (int l = 0; l < L; l++) dump_M[o + l] = M[o + l];
                            continue;
                        }
                        /* a1: the radiance interval of this probe and direction */
                        int n = i == 0 ? diag_segments(nx, ny, a, b, (int)k, ta, tb, seg)
                                       : dda_segments(nx, ny, px, py, cos(theta), sin(theta), ta, tb, seg);
                        nseg_total += n;
                        if (order & 1) integrate_btf(&g, seg, n, cos(theta), sin(theta), I, T);
                        else integrate_ftb(&g, seg, n, cos(theta), sin(theta), I, T);
                        if (dump) for (int l = 0; l < L; l++) { dump_I[o + l] = I[l]; dump_T[o + l] = T[l]; }
                        if (i == top) {
                            /* a2: boundary intensity enters on the top cascade only (G9) */
                            for (int l = 0; l < L; l++) {
                                double Ib = sin(theta) < 0.0 ? (I_below ? I_below[l] : 0.0)
                                                             : (I_above ? I_above[l] : 0.0);
                                M[o + l] = I[l] + T[l] * Ib;
                            }
                        } else {
                            /* a3: bilinear over the 4 parents, mean over the 4 children, eq. 11 */
                            int a0, a1, b0, b1; double fa, fb;
                            parent_axis(a, npx / 2, &a0, &a1, &fa);
                            parent_axis(b, npy / 2, &b0, &b1, &fb);
                            for (int l = 0; l < L; l++) {
                                double U = 0.0;
                                for (int j = 0; j < 4; j++) {
                                    long kk = 4 * k + j;
#define MUP(bb, aa) Mup[((((size_t)((bb) - upy0)) * upwx + ((aa) - upx0)) * upN + kk) * L + l]
                                    U += (1.0 - fb) * ((1.0 - fa) * MUP(b0, a0) + fa * MUP(b0, a1))
                                       +        fb  * ((1.0 - fa) * MUP(b1, a0) + fa * MUP(b1, a1));
#undef MUP
                                }
                                M[o + l] = I[l] + T[l] * U / 4.0;
                            }
                        }
                        if (dump) for (int l = 0; l < L; l++) dump_M[o + l] = M[o + l];
                    }
                }
            }
            free(seg); free(I); free(T);
        }
        if (counts) { counts->intervals[i] = nflagged * N; counts->segments[i] = nseg_total; }
        free(Mup);
        Mup = M; upx0 = ax0[i]; upy0 = by0[i]; upwx = wx; upN = N;
    }
    if (status == 0) {
        /* a4: J = mean of the 4 merged cascade-0 directions (eq. 1 in flatland, reading G14) */
        int wx = x1 - x0, wy = y1 - y0;
        for (int y = 0; y < wy; y++)
            for (int x = 0; x < wx; x++) {
                double jb = 0.0;
                int on = !active || active[(size_t)(y0 + y) * nx + (x0 + x)];
                for (int l = 0; l < L; l++) {
                    const double *m = Mup + (((size_t)y * wx + x) * 4) * L + l;
                    /* J is defined on the cells of interest; elsewhere it is not computed: 0 */
                    double J = on ? (m[0] + m[(size_t)L] + m[2 * (size_t)L] + m[3 * (size_t)L]) / 4.0 : 0.0;
                    J_out[((size_t)y * wx + x) * L + l] = J;
                    jb += (w ? (double)w[l] : 1.0) * J;
                }
                if (Jbar_out) Jbar_out[(size_t)y * wx + x] = jb;
            }
    }
    free(Mup);
    for (int i = 0; i <= top; i++) free(flag[i]);
    return status;
}

int rc_oracle_solve_scaled(const float *chi, const float *eta, int nx, int ny, int L, int ncasc,
                           double c0, const float *I_below, const float *I_above, const float *w,
                           int x0, int x1, int y0, int y1, double *J_out, double *Jbar_out, int nthreads,
                           int order, int dump_cascade, double *dump_I, double *dump_T, double *dump_M,
                           int *dump_win, rc_oracle_counts *counts, double path_scale) {
    return solve_impl(chi, eta, NULL, NULL, nx, ny, L, ncasc, c0, I_below, I_above, w, x0, x1, y0, y1, J_out,
                      Jbar_out, nthreads, order, dump_cascade, dump_I, dump_T, dump_M, dump_win, counts, path_scale, NULL);
}

/* Sparse solve: `active` [ny][nx] flags the cells of interest (non-zero = flagged).  Either mode:
 * chi, eta or line, xl (the other pair NULL). */
int rc_oracle_solve_active(const float *chi, const float *eta, const float *line, const double *xl, int nx, int ny,
                           int L, int ncasc, double c0, const float *I_below, const float *I_above, const float *w,
                           int x0, int x1, int y0, int y1, double *J_out, double *Jbar_out, int nthreads, int order,
                           rc_oracle_counts *counts, double path_scale, const unsigned char *active) {
    return solve_impl(chi, eta, line, xl, nx, ny, L, ncasc, c0, I_below, I_above, w, x0, x1, y0, y1, J_out, Jbar_out,
                      nthreads, order, -1, NULL, NULL, NULL, NULL, counts, path_scale, active);
}

/* Velocity-dependent line mode: line [ny][nx][6] and xl [L] instead of chi, eta (cell_chi_eta above). */
int rc_oracle_solve_line(const float *line, const double *xl, int nx, int ny, int L, int ncasc, double c0,
                         const float *I_below, const float *I_above, const float *w, int x0, int x1, int y0,
                         int y1, double *J_out, double *Jbar_out, int nthreads, int order,
                         rc_oracle_counts *counts, double path_scale) {
    return solve_impl(NULL, NULL, line, xl, nx, ny, L, ncasc, c0, I_below, I_above, w, x0, x1, y0, y1, J_out,
                      Jbar_out, nthreads, order, -1, NULL, NULL, NULL, NULL, counts, path_scale, NULL);
}

/* The same, also writing one cascade's intervals before and after merging (as rc_oracle_solve does): an output
 * path for the pins of the directional transmittances, no arithmetic of its own. */
int rc_oracle_solve_line_dump(const float *line, const double *xl, int nx, int ny, int L, int ncasc, double c0,
                              const float *I_below, const float *I_above, const float *w, double *J_out,
                              double *Jbar_out, int nthreads, int order, int dump_cascade, double *dump_I,
                              double *dump_T, double *dump_M, int *dump_win, double path_scale) {
    return solve_impl(NULL, NULL, line, xl, nx, ny, L, ncasc, c0, I_below, I_above, w, 0, nx, 0, ny, J_out,
                      Jbar_out, nthreads, order, dump_cascade, dump_I, dump_T, dump_M, dump_win, NULL, path_scale, NULL);
}

/* Flatland (path_scale = 1): the solve of SURVEY.md §8(c). */
int rc_oracle_solve(const float *chi, const float *eta, int nx, int ny, int L, int ncasc,
                    double c0, const float *I_below, const float *I_above, const float *w,
                    int x0, int x1, int y0, int y1, double *J_out, double *Jbar_out, int nthreads,
                    int order, int dump_cascade, double *dump_I, double *dump_T, double *dump_M,
                    int *dump_win, rc_oracle_counts *counts) {
    return rc_oracle_solve_scaled(chi, eta, nx, ny, L, ncasc, c0, I_below, I_above, w, x0, x1, y0, y1, J_out,
                                  Jbar_out, nthreads, order, dump_cascade, dump_I, dump_T, dump_M, dump_win,
                                  counts, 1.0);
}

int rc_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
