/*
 * radt_oracle.c -- TEST INFRASTRUCTURE (see radt_oracle.h).  Plain fp64 CPU oracle.
 *
 * Follows, step by step and in the paper's notation, the algorithm O1-O11 stated in DESIGN.md
 * (from SURVEY.md section 8(c)); each function cites the passage of PAPER.md it implements.
 * No blocking, fusion, skipping, windowing or early termination: every ray visits every step and
 * every channel.  OpenMP only distributes independent rays over host threads.
 *
 * Pins (tests/, all `-m "not gpu"`):
 *   orc_render        isothermal slab closed form B_nu(T)(1-exp(-tau)) with tau from the Einstein-B
 *                     form of Eq. 14 and worked values under tests/golden/; optically thin limit
 *                     int j ds (uniform and Gaussian density); line-profile normalisation;
 *                     face-on and minor-axis velocity mirror symmetries; azimuth invariance;
 *                     step-refinement convergence; independent numpy brute force on tiny scenes.
 *   orc_ray_geometry  path length through sphere/box, closest-approach identity, rotation
 *                     orthonormality, receding side of the major axis.
 *   orc_partition     asymptotic rigid-rotor expansion; source function vs Rayleigh-Jeans limit.
 *   orc_render_bwd    central finite differences of orc_render (element-wise and directional),
 *                     linearity in G, dot-product test.
 * UNPINNED: agreement with RADMC-3D / RadJAX themselves (not available offline).
 */
#include "radt_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018, CGS (SURVEY.md section 8(c) "Constants") */
#define ORC_H 6.62607015e-27
#define ORC_K 1.380649e-16
#define ORC_C 2.99792458e10
#define ORC_AU 1.495978707e13
#define ORC_PC 3.0856775814913673e18
#define ORC_PI 3.14159265358979323846

typedef struct {
    double cth, sth, ci, si, ca, sa;
    double dir[3];
} orc_orient;

typedef struct {
    double T0;       /* h nu0 / k */
    double a1, a0;   /* alpha^2 = a1 T + a0  (Eq. 16-17) */
    double Ck;       /* K = Ck n_u (e^x - 1) ds[au] / alpha */
    double Sunit;    /* S0 / intensity unit */
} orc_consts;

typedef struct {
    int inside;
    int ncorner;
    int64_t idx[8];
    double w[8];
    double r;        /* cylindrical radius, au */
    double rho;      /* spherical radius, au */
    double x, y, z;  /* disk frame, au */
} orc_sample;

typedef struct {
    int active;      /* inside the grid and r > 0 */
    int t_clamped;
    double n, T, vphi, vk, proj, vlos, alpha, x, ex, Q, F, K, S;
} orc_step;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Threads the ray loops may use from now on (timing only: the arithmetic of a ray does not depend on it). */
void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* O2 orientation: sky (X right, Y up, zeta to the observer, s = -zeta) -> disk frame.
 * Geometry parameters: Table 2 (inclination, position angle, azimuth). */
static void orc_make_orient(const orc_geom *g, orc_orient *o)
{
    double th = g->pa + 0.5 * ORC_PI;
    o->cth = cos(th); o->sth = sin(th);
    o->ci = cos(g->incl); o->si = sin(g->incl);
    o->ca = cos(g->az); o->sa = sin(g->az);
    /* before azimuth the direction of increasing s is (0, sin i, -cos i) */
    o->dir[0] = o->si * o->sa;
    o->dir[1] = o->si * o->ca;
    o->dir[2] = -o->ci;
}

/* O1 pixel centres + O2: disk-frame position of the point s = 0 of ray (ix, iy). */
static void orc_pixel_origin(const orc_geom *g, const orc_orient *o, int64_t ray, double org[3],
                             double *Xs, double *Ys)
{
    int64_t ix = ray % g->nx, iy = ray / g->nx;
    double X = g->x0 + ((double)ix + 0.5 - 0.5 * (double)g->nx) * g->fov_x / (double)g->nx;
    double Y = g->y0 + ((double)iy + 0.5 - 0.5 * (double)g->ny) * g->fov_y / (double)g->ny;
    double xp = X * o->cth + Y * o->sth;
    double yp = -X * o->sth + Y * o->cth;
    double ypp = yp * o->ci;   /* zeta = 0 */
    double zpp = yp * o->si;
    org[0] = xp * o->ca + ypp * o->sa;
    org[1] = -xp * o->sa + ypp * o->ca;
    org[2] = zpp;
    *Xs = X; *Ys = Y;
}

/* O3 clipping of the ray against the bounding sphere (axisymmetric) or the box (3-D). */
static int orc_clip(const orc_geom *g, const orc_grid *gr, const orc_orient *o, const double org[3],
                    double X, double Y, double *s0, double *s1)
{
    if (gr->kind == ORC_AXISYM) {
        double zm = fmax(fabs(gr->lo[1]), fabs(gr->hi[1]));
        double Rb = gr->hi[0] * sqrt(1.0 + zm * zm);
        double b = hypot(X, Y);
        if (!(b < Rb)) return 0;
        double sh = sqrt(Rb * Rb - b * b);
        *s0 = -sh; *s1 = sh;
        return 1;
    }
    if (gr->kind == ORC_SPH3D) {
        /* spherical (r, theta, phi) grid: bounding sphere of radius r_max */
        double Rb = gr->hi[0];
        double b = hypot(X, Y);
        if (!(b < Rb)) return 0;
        double sh = sqrt(Rb * Rb - b * b);
        *s0 = -sh; *s1 = sh;
        return 1;
    }
    double tmin = -INFINITY, tmax = INFINITY;
    for (int a = 0; a < 3; ++a) {
        double d = o->dir[a];
        if (d != 0.0) {
            double t1 = (gr->lo[a] - org[a]) / d, t2 = (gr->hi[a] - org[a]) / d;
            if (t1 > t2) { double t = t1; t1 = t2; t2 = t; }
            if (t1 > tmin) tmin = t1;
            if (t2 < tmax) tmax = t2;
        } else if (org[a] < gr->lo[a] || org[a] > gr->hi[a]) {
            return 0;
        }
    }
    (void)g;
    if (!(tmax > tmin)) return 0;
    *s0 = tmin; *s1 = tmax;
    return 1;
}

/* O5 / O6 field sampling: interpolation nodes and weights at a disk-frame point.
 * Grids: PAPER.md:296 ("regularly spaced (or log-spaced) ... grids"); bi/tri-linear in index space. */
static void orc_locate(const orc_grid *gr, double x, double y, double z, orc_sample *sp)
{
    sp->x = x; sp->y = y; sp->z = z;
    sp->r = hypot(x, y);
    sp->rho = sqrt(x * x + y * y + z * z);
    sp->inside = 0;
    sp->ncorner = 0;
    if (gr->kind == ORC_AXISYM) {
        int nr = gr->n[0], nz = gr->n[1];
        double rmin = gr->lo[0], rmax = gr->hi[0], zlo = gr->lo[1], zhi = gr->hi[1];
        if (!(sp->r > 0.0)) return;
        double zeta = (gr->mirror_z ? fabs(z) : z) / sp->r;
        if (!(sp->r >= rmin && sp->r <= rmax && zeta >= zlo && zeta <= zhi)) return;
        double u = log(sp->r / rmin) / log(rmax / rmin) * (double)(nr - 1);
        double w = (zeta - zlo) / (zhi - zlo) * (double)(nz - 1);
        if (u < 0.0) u = 0.0;
        if (u > (double)(nr - 1)) u = (double)(nr - 1);
        if (w < 0.0) w = 0.0;
        if (w > (double)(nz - 1)) w = (double)(nz - 1);
        int i = (int)floor(u); if (i > nr - 2) i = nr - 2;
        int j = (int)floor(w); if (j > nz - 2) j = nz - 2;
        double fu = u - (double)i, fw = w - (double)j;
        sp->inside = 1;
        sp->ncorner = 4;
        for (int c = 0; c < 4; ++c) {
            int di = c >> 1, dj = c & 1;
            sp->idx[c] = (int64_t)(i + di) * nz + (j + dj);
            sp->w[c] = (di ? fu : 1.0 - fu) * (dj ? fw : 1.0 - fw);
        }
        return;
    }
    if (gr->kind == ORC_SPH3D) {
        /* nodes: r_i = r_min (r_max/r_min)^(i/(nr-1)); theta_j = lo[1] + (hi[1]-lo[1]) j/(nt-1), the polar angle from
         * the +z axis of the disk frame; phi_k = 2 pi k/np, periodic (the cell after node np-1 ends at node 0).
         * Tri-linear in index space (ln r, theta, phi); outside the (r, theta) range is vacuum. */
        int nr = gr->n[0], nt = gr->n[1], np_ = gr->n[2];
        double rmin = gr->lo[0], rmax = gr->hi[0], tlo = gr->lo[1], thi = gr->hi[1];
        const double two_pi = 6.283185307179586476925286766559;
        if (!(sp->rho > 0.0)) return;
        double theta = acos(z / sp->rho);
        if (!(sp->rho >= rmin && sp->rho <= rmax && theta >= tlo && theta <= thi)) return;
        double phi = atan2(y, x);
        if (phi < 0.0) phi += two_pi;
        double u = log(sp->rho / rmin) / log(rmax / rmin) * (double)(nr - 1);
        double w = (theta - tlo) / (thi - tlo) * (double)(nt - 1);
        double q = phi / two_pi * (double)np_;
        if (u < 0.0) u = 0.0;
        if (u > (double)(nr - 1)) u = (double)(nr - 1);
        if (w < 0.0) w = 0.0;
        if (w > (double)(nt - 1)) w = (double)(nt - 1);
        if (q < 0.0) q = 0.0;
        if (q > (double)np_) q = (double)np_;
        int i = (int)floor(u); if (i > nr - 2) i = nr - 2;
        int j = (int)floor(w); if (j > nt - 2) j = nt - 2;
        int k = (int)floor(q); if (k > np_ - 1) k = np_ - 1;
        double fu = u - (double)i, fw = w - (double)j, fq = q - (double)k;
        int k1 = (k + 1) % np_;
        sp->inside = 1;
        sp->ncorner = 8;
        for (int c = 0; c < 8; ++c) {
            int di = (c >> 2) & 1, dj = (c >> 1) & 1, dk = c & 1;
            sp->idx[c] = ((int64_t)(i + di) * nt + (j + dj)) * np_ + (dk ? k1 : k);
            sp->w[c] = (di ? fu : 1.0 - fu) * (dj ? fw : 1.0 - fw) * (dk ? fq : 1.0 - fq);
        }
        return;
    }
    double p[3] = { x, y, z };
    int i0[3];
    double f[3];
    for (int a = 0; a < 3; ++a) {
        if (!(p[a] >= gr->lo[a] && p[a] <= gr->hi[a])) return;
        double t = (p[a] - gr->lo[a]) / (gr->hi[a] - gr->lo[a]) * (double)(gr->n[a] - 1);
        if (t < 0.0) t = 0.0;
        if (t > (double)(gr->n[a] - 1)) t = (double)(gr->n[a] - 1);
        int i = (int)floor(t); if (i > gr->n[a] - 2) i = gr->n[a] - 2;
        i0[a] = i; f[a] = t - (double)i;
    }
    sp->inside = 1;
    sp->ncorner = 8;
    for (int c = 0; c < 8; ++c) {
        int dx = (c >> 2) & 1, dy = (c >> 1) & 1, dz = c & 1;
        sp->idx[c] = ((int64_t)(i0[0] + dx) * gr->n[1] + (i0[1] + dy)) * gr->n[2] + (i0[2] + dz);
        sp->w[c] = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
    }
}

static double orc_interp(const float *a, const orc_sample *sp)
{
    double v = 0.0;
    for (int c = 0; c < sp->ncorner; ++c) v += sp->w[c] * (double)a[sp->idx[c]];
    return v;
}

/* Partition function Q(T) = sum_J g_J exp(-E_J / kT)  (Boltzmann statistics). */
double orc_partition(const orc_line *ln, double T)
{
    double q = 0.0;
    for (int l = 0; l < ln->nlev; ++l) q += ln->g_lev[l] * exp(-ln->e_lev_K[l] / T);
    return q;
}

static double orc_partition_dT(const orc_line *ln, double T)
{
    double q = 0.0;
    for (int l = 0; l < ln->nlev; ++l)
        q += ln->g_lev[l] * (ln->e_lev_K[l] / (T * T)) * exp(-ln->e_lev_K[l] / T);
    return q;
}

double orc_source_unit(const orc_line *ln, const orc_geom *g)
{
    double S0 = 2.0 * ORC_H * ln->nu0 * ln->nu0 * ln->nu0 / (ORC_C * ORC_C);
    if (ln->unit == ORC_UNIT_CGS) return S0;
    if (ln->unit == ORC_UNIT_JY_PIXEL) {
        double d_au = g->dist_pc * ORC_PC / ORC_AU;
        double omega = (g->fov_x / (double)g->nx) * (g->fov_y / (double)g->ny) / (d_au * d_au);
        return S0 * omega * 1.0e23;
    }
    return 1.0;
}

static void orc_make_consts(const orc_geom *g, const orc_line *ln, orc_consts *k)
{
    k->T0 = ORC_H * ln->nu0 / ORC_K;
    k->a1 = 2.0 * ORC_K / ln->m_line + ln->vturb_mach * ln->vturb_mach * 2.0 * ORC_K / ln->m_gas; /* Eq. 16-17 */
    k->a0 = ln->vturb_abs * ln->vturb_abs;
    /* beta = (c^2 / 8 pi nu0^2) A_ul n_u (e^x - 1) phi_nu, phi_nu = c / (nu0 alpha sqrt(pi)) exp(-u^2)
     * (Eq. 14 with the LTE identity, Eq. 15); times ds in cm. */
    k->Ck = ORC_C * ORC_C / (8.0 * ORC_PI * ln->nu0 * ln->nu0) * ln->a_ul * ORC_C / (ln->nu0 * sqrt(ORC_PI)) * ORC_AU;
    k->Sunit = orc_source_unit(ln, g);
}

/* O7 per-step, channel-independent quantities. */
static void orc_physics(const orc_geom *g, const orc_line *ln, const orc_grid *gr, const orc_consts *k,
                        const orc_orient *o, const orc_sample *sp, double ds, orc_step *st)
{
    memset(st, 0, sizeof(*st));
    if (!sp->inside || !(sp->r > 0.0)) return;
    st->active = 1;
    double draw = orc_interp(gr->dens, sp);
    double traw = orc_interp(gr->temp, sp);
    double vraw = orc_interp(gr->vel, sp);
    st->n = (gr->dens_mode == ORC_DENS_LN) ? exp(draw) : draw;
    st->t_clamped = !(traw >= 1.0);
    st->T = st->t_clamped ? 1.0 : traw;
    if (gr->vel_mode == ORC_VEL_KEPLER_FRAC) {
        /* Eq. 6 without the pressure term: v_K^2 / r = G M r / (r^2 + z^2)^(3/2) */
        double rc = sp->r * ORC_AU, rhoc = sp->rho * ORC_AU;
        st->vk = sqrt(g->gm_star * rc * rc / (rhoc * rhoc * rhoc));
        st->vphi = st->vk * (1.0 + vraw);
    } else {
        st->vk = 1.0;
        st->vphi = vraw;
    }
    /* v_los = omega . v, v = v_phi (-y, x, 0) / r */
    st->proj = (-sp->y * o->dir[0] + sp->x * o->dir[1]) / sp->r;
    st->vlos = st->vphi * st->proj;
    st->alpha = sqrt(k->a1 * st->T + k->a0);                 /* Eq. 16 */
    st->x = k->T0 / st->T;
    st->ex = exp(st->x);
    st->Q = orc_partition(ln, st->T);
    st->F = ln->g_u * exp(-ln->e_u_K / st->T) * (st->ex - 1.0) / st->Q;   /* n_u (e^x - 1) / n */
    st->K = k->Ck * st->n * st->F * ds / st->alpha;          /* line-centre optical depth of the step */
    st->S = k->Sunit / (st->ex - 1.0);                       /* S = j / beta = B_nu0(T) */
}

static void orc_step_at(const orc_geom *g, const orc_line *ln, const orc_grid *gr, const orc_consts *k,
                        const orc_orient *o, const double org[3], double s, double ds,
                        orc_sample *sp, orc_step *st)
{
    orc_locate(gr, org[0] + s * o->dir[0], org[1] + s * o->dir[1], org[2] + s * o->dir[2], sp);
    orc_physics(g, ln, gr, k, o, sp, ds, st);
}

int orc_ray_geometry(const orc_geom *geom, const orc_grid *grid, int64_t nrays, const int64_t *ray_idx,
                     double *out_origin, double *out_dir, double *out_s0, double *out_ds, int32_t *out_valid)
{
    orc_orient o;
    orc_make_orient(geom, &o);
    if (out_dir) memcpy(out_dir, o.dir, sizeof(o.dir));
    for (int64_t q = 0; q < nrays; ++q) {
        int64_t ray = ray_idx ? ray_idx[q] : q;
        double org[3], X, Y, s0 = 0.0, s1 = 0.0;
        orc_pixel_origin(geom, &o, ray, org, &X, &Y);
        int valid = orc_clip(geom, grid, &o, org, X, Y, &s0, &s1);
        if (out_origin) memcpy(out_origin + 3 * q, org, sizeof(org));
        if (out_s0) out_s0[q] = valid ? s0 : 0.0;
        if (out_ds) out_ds[q] = valid ? (s1 - s0) / (double)geom->nstep : 0.0;
        if (out_valid) out_valid[q] = valid;
    }
    return 0;
}

int orc_trace_ray(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t ray,
                  int32_t *inside, double *n, double *T, double *vlos, double *alpha, double *K, double *S)
{
    orc_orient o; orc_consts k;
    orc_make_orient(geom, &o);
    orc_make_consts(geom, line, &k);
    double org[3], X, Y, s0, s1;
    orc_pixel_origin(geom, &o, ray, org, &X, &Y);
    int valid = orc_clip(geom, grid, &o, org, X, Y, &s0, &s1);
    for (int kk = 0; kk < geom->nstep; ++kk) {
        orc_sample sp; orc_step st;
        memset(&st, 0, sizeof(st));
        if (valid) {
            double ds = (s1 - s0) / (double)geom->nstep;
            orc_step_at(geom, line, grid, &k, &o, org, s0 + ((double)kk + 0.5) * ds, ds, &sp, &st);
        }
        inside[kk] = st.active; n[kk] = st.n; T[kk] = st.T; vlos[kk] = st.vlos;
        alpha[kk] = st.alpha; K[kk] = st.K; S[kk] = st.S;
    }
    return valid;
}

/* O4, O8, O9, O10: march one ray front to back (k = 0 nearest the observer). */
int orc_render(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t nrays,
               const int64_t *ray_idx, double *cube_out)
{
    orc_orient o; orc_consts k;
    orc_make_orient(geom, &o);
    orc_make_consts(geom, line, &k);
    const int C = line->nchan, N = geom->nstep;
#pragma omp parallel
    {
        double *tr = (double *)malloc(sizeof(double) * (size_t)C);
#pragma omp for schedule(dynamic, 8)
        for (int64_t q = 0; q < nrays; ++q) {
            int64_t ray = ray_idx ? ray_idx[q] : q;
            double *I = cube_out + (size_t)q * (size_t)C;
            for (int c = 0; c < C; ++c) { I[c] = 0.0; tr[c] = 1.0; }
            double org[3], X, Y, s0, s1;
            orc_pixel_origin(geom, &o, ray, org, &X, &Y);
            if (!orc_clip(geom, grid, &o, org, X, Y, &s0, &s1)) continue;   /* reading 22: zeros */
            double ds = (s1 - s0) / (double)N;
            for (int kk = 0; kk < N; ++kk) {
                orc_sample sp; orc_step st;
                orc_step_at(geom, line, grid, &k, &o, org, s0 + ((double)kk + 0.5) * ds, ds, &sp, &st);
                if (!st.active) continue;   /* vacuum: contributes nothing */
                for (int c = 0; c < C; ++c) {
                    double u = (line->vchan[c] - geom->vsys - st.vlos) / st.alpha;   /* O8 */
                    double gph = exp(-u * u);
                    double dtau = st.K * gph;
                    I[c] += st.S * (-expm1(-dtau)) * tr[c];                          /* O9 */
                    tr[c] *= exp(-dtau);
                }
            }
        }
        free(tr);
    }
    return 0;
}

static void orc_atomic_add(double *p, double v)
{
#pragma omp atomic
    *p += v;
}

/* O11: exact derivative of O1-O10 with respect to the stored grid values. */
int orc_render_bwd(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t nrays,
                   const int64_t *ray_idx, const double *G, double *g_dens, double *g_temp, double *g_vel)
{
    orc_orient o; orc_consts k;
    orc_make_orient(geom, &o);
    orc_make_consts(geom, line, &k);
    const int C = line->nchan, N = geom->nstep;
#pragma omp parallel
    {
        orc_sample *sps = (orc_sample *)malloc(sizeof(orc_sample) * (size_t)N);
        orc_step *sts = (orc_step *)malloc(sizeof(orc_step) * (size_t)N);
        double *e = (double *)malloc(sizeof(double) * (size_t)N * (size_t)C);    /* exp(-dtau_k,c) */
        double *tf = (double *)malloc(sizeof(double) * (size_t)N * (size_t)C);   /* T_k,c in front of step k */
        double *B = (double *)malloc(sizeof(double) * (size_t)C);                /* intensity from behind */
        double *tr = (double *)malloc(sizeof(double) * (size_t)C);
#pragma omp for schedule(dynamic, 8)
        for (int64_t q = 0; q < nrays; ++q) {
            int64_t ray = ray_idx ? ray_idx[q] : q;
            const double *Gq = G + (size_t)q * (size_t)C;
            double org[3], X, Y, s0, s1;
            orc_pixel_origin(geom, &o, ray, org, &X, &Y);
            if (!orc_clip(geom, grid, &o, org, X, Y, &s0, &s1)) continue;
            double ds = (s1 - s0) / (double)N;
            for (int c = 0; c < C; ++c) tr[c] = 1.0;
            for (int kk = 0; kk < N; ++kk) {
                orc_step_at(geom, line, grid, &k, &o, org, s0 + ((double)kk + 0.5) * ds, ds, &sps[kk], &sts[kk]);
                for (int c = 0; c < C; ++c) {
                    double ek = 1.0;
                    if (sts[kk].active) {
                        double u = (line->vchan[c] - geom->vsys - sts[kk].vlos) / sts[kk].alpha;
                        ek = exp(-sts[kk].K * exp(-u * u));
                    }
                    e[(size_t)kk * C + c] = ek;
                    tf[(size_t)kk * C + c] = tr[c];
                    tr[c] *= ek;
                }
            }
            for (int c = 0; c < C; ++c) B[c] = 0.0;
            for (int kk = N - 1; kk >= 0; --kk) {
                const orc_step *st = &sts[kk];
                const orc_sample *sp = &sps[kk];
                if (!st->active) continue;   /* e = 1: B unchanged, no dependence on any field */
                double A0 = 0.0, A1 = 0.0, A2 = 0.0, Bs = 0.0;
                for (int c = 0; c < C; ++c) {
                    double ek = e[(size_t)kk * C + c], tk = tf[(size_t)kk * C + c];
                    double u = (line->vchan[c] - geom->vsys - st->vlos) / st->alpha;
                    double gph = exp(-u * u);
                    double dtau = st->K * gph;
                    double om = -expm1(-dtau);
                    double a = Gq[c] * tk * ek * (st->S - B[c]);   /* dL/d dtau_k,c */
                    double b = Gq[c] * om * tk;                     /* dL/dS_k through channel c */
                    A0 += a * gph;
                    A1 += a * dtau * u;
                    A2 += a * dtau * u * u;
                    Bs += b;
                    B[c] = st->S * om + ek * B[c];
                }
                /* chain rule to (n, T, v_phi) at the sample point */
                double dL_dvlos = 2.0 / st->alpha * A1;
                double dL_dalpha = 2.0 / st->alpha * A2 - A0 * st->K / st->alpha;
                double dL_dn = A0 * k.Ck * st->F * ds / st->alpha;
                double T = st->T;
                double dlnF_dT = line->e_u_K / (T * T) - (k.T0 / (T * T)) * st->ex / (st->ex - 1.0)
                               - orc_partition_dT(line, T) / st->Q;
                double dS_dT = k.Sunit * st->ex * (k.T0 / (T * T)) / ((st->ex - 1.0) * (st->ex - 1.0));
                double dalpha_dT = k.a1 / (2.0 * st->alpha);
                double dL_dT = A0 * st->K * dlnF_dT + dL_dalpha * dalpha_dT + Bs * dS_dT;
                if (st->t_clamped) dL_dT = 0.0;
                double dL_dvphi = dL_dvlos * st->proj;
                double dL_ddens = (grid->dens_mode == ORC_DENS_LN) ? dL_dn * st->n : dL_dn;
                double dL_dvel = (grid->vel_mode == ORC_VEL_KEPLER_FRAC) ? dL_dvphi * st->vk : dL_dvphi;
                for (int cc = 0; cc < sp->ncorner; ++cc) {
                    if (g_dens) orc_atomic_add(&g_dens[sp->idx[cc]], sp->w[cc] * dL_ddens);
                    if (g_temp) orc_atomic_add(&g_temp[sp->idx[cc]], sp->w[cc] * dL_dT);
                    if (g_vel) orc_atomic_add(&g_vel[sp->idx[cc]], sp->w[cc] * dL_dvel);
                }
            }
        }
        free(sps); free(sts); free(e); free(tf); free(B); free(tr);
    }
    return 0;
}
