// radt_dev.cuh -- device-side parameter blocks and math helpers of the B200 line-RT render.
// Product code: shares nothing with oracle/.  Algorithm statement: DESIGN.md O1-O11
// (Eq. 11-17).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#ifndef RADT_WARPS_PER_CTA
#define RADT_WARPS_PER_CTA 4          // one warp per ray; CTA = 2 x 2 pixel tile (measured against 8 warps, 4 x 2: the
#define RADT_TILE_X 2                 // finer granularity fills the SMs 2-3 % better at the same registers per thread)
#define RADT_TILE_Y 2
#endif
#define RADT_MAXB 16                  // batch items per launch (geometry travels in kernel params)
#define RADT_NQ 4096                  // partition-function table intervals over log2 T in [0, 14]
#define RADT_NQ_OCTAVES 14.0f
#define RADT_TMAX 16384.0f             // upper end of that table: temperatures above it are clamped (zero gradient)
#define RADT_MAXLEV 64
#define RADT_MAXCHAN 256
#define RADT_LOSS_SLOTS 1024           // partial sums of the fused chi^2 loss
#define RADT_CNT_USEFUL 4              // workspace counter: forward (channel, step) samples inside their line window
#define RADT_CNT_TMAX 7                // workspace counter slot holding the bits of the grid's maximum temperature

#define RADT_LOG2E 1.4426950408889634f
#define RADT_LN2 0.6931471805599453f
#define RADT_SQRT_LOG2E 1.2011224087864498f

// Per batch item viewing geometry, precomputed on the host in fp64 (O1-O2).
struct DevGeom {
    double cth, sth, ci, si, ca, sa;   // cos/sin of PA + pi/2, inclination, azimuth
    double wx, wy, wz;                 // ray direction (increasing s) in the disk frame
    double x0, y0, pix_x, pix_y;       // image centre offset and pixel pitch, au
    double gm_au_d;                    // G M / au  [(cm/s)^2 au]  (KEPLER_FRAC)
    double v0;                         // velocity of channel 0 minus v_sys, cm/s (uniform channel lattice)
    float sunit;                       // S0 / intensity unit
    float wxf, wyf, wzf;               // fp32 copy of the ray direction (prefilter of the window kernels)
};

struct DevGrid {
    int kind, mirror, dens_mode, vel_mode;
    int n0, n1, n2;
    long long cells;                   // cells per batch item
    // axisymmetric
    double rmin2, rmax2, inv_rmin, zlo, zhi;
    double wscale_d;                   // (nzeta-1)/(zeta_hi-zeta_lo)
    double lg2_ratio;                  // log2(r_max/r_min)
    float uscale;                      // (nr-1)/log2(r_max/r_min)
    float inv_cell_ln, inv_cell_lg2;   // 1/ln(rho), 1/log2(rho), rho = node ratio r_{i+1}/r_i
    int fine_r;                        // rho^2 - 1 < 0.35: log1p series for the in-cell fraction
    float zlo_f, wscale_f;             // fp32 copies for the index coordinates
    float inv_rmin2_f, half_uscale;    // u = lg2(r^2 / r_min^2) (nr-1) / (2 log2(r_max/r_min))
    // cartesian
    double lo[3], hi[3], inv_d[3];
    double rb2;                        // bounding sphere radius^2 (axisym and spherical clip)
    // spherical (kind 2): n0 = nr (log-spaced, shares rmin2/rmax2/uscale/... with the axisymmetric axis), n1 = ntheta, n2 = nphi
    double cos_tlo, cos_thi;           // cos of the theta range (decreasing in theta)
    double rho2_lo, rho2_hi;           // in range iff rho2_lo <= rho^2 <= rho2_hi, rho^2 = (x x + y y) + z z with every operation
                                       // rounded: exactly the doubles t with r_min <= sqrt(t) <= r_max (correctly rounded sqrt),
                                       // i.e. the decision of a plain fp64 evaluation, ties on the boundary included
    float th_c0, th_scale, ph_scale;   // theta index = (th_c0 - asin(z/rho)) th_scale, th_c0 = pi/2 - theta_lo; phi index = phi ph_scale
    // fp32 constants of the window kernels' prefilter (a superset test with one cell of margin, radt_march_win.cu)
    float pre_us_half, pre_uoff;       // axisym / spherical: u = lg2(r^2) pre_us_half + pre_uoff
    float pre_wscale, pre_woff;        // axisym: w = zeta pre_wscale + pre_woff
    float pre_n0f, pre_n1f, pre_n2f;   // node counts as floats
    float pre_czlo, pre_czhi;          // spherical: accepted range of z/rho = cos(theta), two theta cells of margin
    float pre_cscale;                  // spherical: occupancy bin of cos(theta) = (z/rho - pre_czlo) pre_cscale, n1 bins
    float pre_lo[3], pre_inv_d[3];     // cartesian
};

struct DevLine {
    float T0;          // h nu0 / k
    float T0l2;        // T0 * log2(e)
    float Eu;          // E_u / k
    float Eul2;        // Eu * log2(e)
    float gu;
    float a1, a0;      // alpha^2 = a1 T + a0   [(cm/s)^2]
    float Ck2;         // line-centre dtau * log2e = Ck2 * n * W * (e^x - 1) * ds[au] / alpha
    int nchan;
    int ngroups;       // ceil(nchan / 32)
    // uniform channel lattice v_c = v0 + c dv (window path)
    int uniform;       // the channel table is such a lattice
    double inv_dv;     // 1 / dv
    float dvf;         // dv sqrt(log2 e)           (u' step between channels = dvf / alpha)
    float c_hw;        // 1 / (sqrt(log2 e) |dv|)   (half-width of the line window in channels = u'_cut c_hw alpha)
};

// K1 output per ray: clipped interval and the conservative range of steps that can lie inside the grid
struct __align__(16) RayRec {
    double s0, ds;         // au; ds = 0 marks a ray that misses the volume
    int k_lo, k_hi;        // in-grid samples have k_lo <= k < k_hi
    int pad0, pad1;
};

// Workspace layout (all offsets in bytes from the workspace base, 256-byte aligned)
struct DevWs {
    RayRec *rays;          // [batch*ny*nx]
    float2 *qtab;          // [RADT_NQ + 2] {Q, dQ/dlnT}
    float2 *vcs;           // [batch][RADT_MAXCHAN] channel velocity minus v_sys, cm/s, as (hi, lo) float pair
    double2 *rnode;        // [nr] {r_i, 1/r_i^2} node radii of the log-spaced axis (axisym), fp64
    float4 *cells;         // [batch][cells] packed {dens, temp, vel, 0}
    float4 *grad;          // [batch][cells] packed gradient accumulators {dens, temp, vel, -} (bwd only)
    unsigned *occ;         // [batch][occ_words] axisym: bit (i, j): some cell within one cell of (i, j) can emit;
                           // 3-D: one bit per block of 4 x 4 x 4 cells, same dilation; spherical: bit (radial cell,
                           // bin of cos theta), any phi (radt_setup.cu)
    unsigned *nodeflag;    // spherical: [batch][nr][ceil(ntheta / 32)] bit j of row i: some phi node of (i, j) can emit
    unsigned long long *counters;   // [8 + RADT_LOSS_SLOTS] 0-3 work counters; [4] forward samples inside their line window;
                                    // [7] bits of the grid's maximum temperature; [8..] partial sums of the fused loss (double)
};

struct MarchParams {
    DevGeom geom[RADT_MAXB];
    DevGrid grid;
    DevLine line;
    DevWs ws;
    int nx, ny, nstep;
    int tiles_x, tiles_y;
    int tile_y0, launch_ty; // this launch covers tile rows [tile_y0, tile_y0 + launch_ty) (row bands of the HOST entry points);
    int banded;             // 1: tile rows in image order (a band is a contiguous row range); 0: centre-out over the whole image
    int b0;                // first batch item of this launch
    int opt_window, opt_skip_empty;
    int opt_zero_grad;     // adjoint: zero-opacity steps of LINEAR density grids are marched for their dL/dn (default)
    int chan_lo;           // some channel velocity is not exactly representable in fp32: use the lo parts
    int use_win;           // uniform-channel window kernels (radt_march_win.cu)
    int use_occ;           // candidate steps are prefiltered with the occupancy bitmap
    int occ_words, occ_wpr; // words per batch item; words per radial row (axisym) / per line of blocks along z (3-D)
    int occ_nbj;            // 3-D: blocks along y
    float *cube;           // fwd: output; bwd: saved forward output (const)
    float *cube_lo;        // low-order word of the fp32 sum behind every voxel (fwd: output, bwd: input); may be null
    const float *dl_dcube; // bwd
    // fused chi^2 data term of the forward (radt_render_loss): all null / 0 for a plain render
    const float *target;   // [batch][ny][nx][nchan]
    float *dl_out;         // dL/dcube = (cube - target) / (sigma^2 n)
    float inv_s2n;
};

struct SetupParams {
    DevGeom geom[RADT_MAXB];
    DevGrid grid;
    DevWs ws;
    int nx, ny, nstep, nbatch, b0;
    int nlev, nchan;
    int do_rays, do_tables, do_pack, do_zero_grad, do_occ;
    int occ_words, occ_wpr, occ_nbj;
    int flag_wpr;          // spherical: words per radial row of nodeflag
    float occ_thr;         // stored density value above which a node can emit
    long long batch_stride;
    const float *dens, *temp, *vel;
    double2 *rays_user;    // radt_ray_geometry output {s0, ds} (may be null)
    double vsys[RADT_MAXB];
};

struct LevelTable {
    double e[RADT_MAXLEV];
    double g[RADT_MAXLEV];
};

struct ChanTable {
    double v[RADT_MAXCHAN];
};

// ---- physics pre-pass (radt_disk.cu): per batch item constants and the launch parameter block ----
struct DiskDev {
    double gm_star, m_gas, sigma0, r_c, gamma, x_co, t_freeze, n_dissoc, f_col;
};
struct DiskParamsDev {
    DiskDev disk[RADT_MAXB];
    int nr, nz, nbatch;
    long long batch_stride;
    double rmin, lg2_ratio, dlnr, dzeta;
    const float *temp;                   // [batch][nr][nz]
    float *dens_out, *vel_out;           // forward outputs
    const float *g_dens, *g_vel;         // adjoint inputs
    float *g_temp;                       // adjoint output (+=)
    double *rt, *rho, *P, *gP, *grho;    // workspace, [batch][nr][nz]
    double *colscale, *colH;             // workspace, [batch][nr]
    unsigned char *mask;                 // workspace, [batch][nr][nz]
};

// ---- MLP temperature field (radt_mlp_tc.cu, radt_mlp_tc_bwd.cu) ----
struct MlpParamsDev {
    int nr, nz, L, nparams;
    float t_lo, t_hi;
    const float *params;                 // flat parameter vector (layout: include/radt.h radt_mlp)
    float *temp_out;                     // forward: [nr][nz]
    const float *g_temp;                 // adjoint input
    float *g_params;                     // adjoint output
};

// ---- single-instruction SFU helpers (MUFU.*) ----
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
// fp64 1/sqrt(x) to ~1e-13: the SFU's fp64 seed (MUFU.RSQ64H: relative error 2^-22, no fp32 round trip) and one Newton step
__device__ __forceinline__ double rsqrt_d(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y * fma(-0.5 * x, y * y, 1.5);
}
// (double)k for 0 <= k < 2^31 without the conversion pipe: 2^52 + k is exact in the low word of the mantissa
__device__ __forceinline__ double int_to_double(int k) { return __hiloint2double(0x43300000, k) - 4503599627370496.0; }

// Disk-frame position of the s = 0 point of pixel (ix, iy)  (O1-O2).
__device__ __forceinline__ void pixel_origin(const DevGeom &G, int nx, int ny, int ix, int iy,
                                             double &ox, double &oy, double &oz, double &X, double &Y)
{
    X = G.x0 + ((double)ix + 0.5 - 0.5 * (double)nx) * G.pix_x;
    Y = G.y0 + ((double)iy + 0.5 - 0.5 * (double)ny) * G.pix_y;
    double xp = X * G.cth + Y * G.sth;
    double yp = -X * G.sth + Y * G.cth;
    double ypp = yp * G.ci;
    oz = yp * G.si;
    ox = xp * G.ca + ypp * G.sa;
    oy = -xp * G.sa + ypp * G.ca;
}
