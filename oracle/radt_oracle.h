/*
 * radt_oracle.h -- TEST INFRASTRUCTURE.  Plain, slow, fp64 CPU oracle of the line-RT render.
 *
 * This is the reference the CUDA path is checked against.  It is NOT part of the product:
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  It shares no code, header, table or constant generator with the CUDA library
 * (include/radt.h, paper_2509_03623_b200/csrc); the structs below are the oracle's own.
 *
 * What it computes: the discretised integral-form transfer equation of the paper,
 *   I_nu = int j_nu exp(-tau_nu) ds            (Eq. 11-12)
 * with the LTE line emissivity/extinction of Eq. 13-14, the Doppler-shifted
 * Gaussian profile of Eq. 15 and the line width of Eq. 16-17
 * (PAPER.md:288-294), by backward ray tracing from every image pixel on a
 * regular / log-spaced grid, plus the exact derivative of that discretisation
 * with respect to the stored grid values (Fig. 2 E PAPER.md:56).
 * The step-by-step algorithm (O1-O11) and the readings taken where the paper is silent are
 * listed in DESIGN.md ("Readings of the paper") and SURVEY.md section 8(c).
 *
 * Pins: every function here is pinned by tests/test_oracle_*.py (closed forms, invariants,
 * finite differences, brute force) -- see the header of radt_oracle.c.  Parity with RADMC-3D or
 * RadJAX themselves is UNPINNED (neither is available; the paper prints no worked numbers).
 */
#ifndef RADT_ORACLE_H
#define RADT_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_AXISYM = 0, ORC_CART3D = 1, ORC_SPH3D = 2 };
enum { ORC_DENS_LINEAR = 0, ORC_DENS_LN = 1 };
enum { ORC_VEL_VPHI = 0, ORC_VEL_KEPLER_FRAC = 1 };
enum { ORC_UNIT_S0 = 0, ORC_UNIT_CGS = 1, ORC_UNIT_JY_PIXEL = 2 };

typedef struct {
    int32_t nx, ny, nstep, pad_;
    double fov_x, fov_y;      /* au */
    double x0, y0;            /* au */
    double incl, pa, az;      /* rad */
    double dist_pc;
    double vsys;              /* cm/s */
    double gm_star;           /* cm^3 s^-2 */
} orc_geom;

typedef struct {
    double nu0, a_ul, g_u, e_u_K;
    int32_t nlev, nchan;
    const double *e_lev_K;    /* [nlev] */
    const double *g_lev;      /* [nlev] */
    double m_line, m_gas;     /* g */
    double vturb_abs;         /* cm/s */
    double vturb_mach;
    const double *vchan;      /* [nchan] cm/s */
    int32_t unit, pad_;
} orc_line;

typedef struct {
    int32_t kind;
    int32_t n[3];
    double lo[3], hi[3];
    int32_t mirror_z, dens_mode, vel_mode, pad_;
    const float *dens, *temp, *vel;   /* host, C-contiguous, last index fastest */
} orc_grid;

/* Ray table: for each listed ray the disk-frame origin (s = 0), the entry parameter s0, the step
 * ds (both au) and a validity flag.  ray_idx == NULL means all nx*ny rays in (iy, ix) order.
 * out_origin [nrays][3], out_s0 [nrays], out_ds [nrays], out_valid [nrays]; out_dir [3]. */
int orc_ray_geometry(const orc_geom *geom, const orc_grid *grid, int64_t nrays, const int64_t *ray_idx,
                     double *out_origin, double *out_dir, double *out_s0, double *out_ds, int32_t *out_valid);

/* Forward render of the listed rays: cube_out [nrays][nchan] (fp64). */
int orc_render(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t nrays,
               const int64_t *ray_idx, double *cube_out);

/* Adjoint: given G = dL/dcube [nrays][nchan] for the listed rays, ACCUMULATES (+=) dL/d(stored
 * grid values) into g_dens, g_temp, g_vel (fp64, grid-shaped; any may be NULL). */
int orc_render_bwd(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t nrays,
                   const int64_t *ray_idx, const double *G, double *g_dens, double *g_temp, double *g_vel);

/* Per-step diagnostics of ONE ray (for tests): for each of nstep steps writes
 * inside flag, n, T, v_los, alpha, K (line-centre dtau), S (in output units). */
int orc_trace_ray(const orc_geom *geom, const orc_line *line, const orc_grid *grid, int64_t ray,
                  int32_t *inside, double *n, double *T, double *vlos, double *alpha, double *K, double *S);

/* Scalar helpers exposed for the textbook pins. */
double orc_partition(const orc_line *line, double T);
double orc_source_unit(const orc_line *line, const orc_geom *geom);   /* S0 / intensity unit */
int orc_num_threads(void);
void orc_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
