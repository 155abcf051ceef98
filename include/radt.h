/*
 * radt.h -- C ABI of the B200-native differentiable line radiative transfer render.
 *
 * The library renders velocity cubes of one molecular line in LTE by backward ray tracing through
 * gridded density / temperature / velocity fields, and returns the gradient of a scalar loss with
 * respect to the stored grid values.  It implements the render of
 *   "Revealing Fine Structure in Protoplanetary Disks with Physics Constrained Neural Fields"
 *   (RadJAX), section "Line Radiative Transfer with RadJAX", Eq. 11-17,
 * discretised as stated in DESIGN.md (algorithm O1-O11).
 *
 * Conventions
 *   - plain C, no torch / C++ types; every pointer is documented as HOST or DEVICE memory;
 *   - the library never allocates device memory and never synchronises in the *_device* entry
 *     points: the caller passes a workspace (size from radt_workspace_bytes) and a CUDA stream;
 *     all work is enqueued on that stream (stream-ordered, CUDA-graph capturable);
 *   - the *_host entry points take HOST buffers, allocate stream-ordered device memory internally,
 *     copy in, run the same kernels, copy out and synchronise the stream before returning;
 *   - units: lengths au, velocities cm/s, number densities cm^-3, temperatures K, angles rad,
 *     frequencies Hz, masses g;
 *   - arrays are C-contiguous, last index fastest: axisymmetric grids [b][ir][izeta], 3-D grids
 *     [b][ix][iy][iz], cubes [b][iy][ix][channel];
 *   - return value 0 on success, a negative RADT_E_* code otherwise; radt_last_error() returns a
 *     thread-local message.  Numerical conditions are not errors: the temperature is clamped to
 *     [1 K, 16384 K] (the range of the device partition-function table; zero gradient through either
 *     clamp; a NaN temperature counts as below the clamp, i.e. 1 K); NaN densities and velocities
 *     propagate into the cube.
 *   - there is no CPU fallback and no other back-end: without a CUDA device every compute entry
 *     point fails with RADT_E_CUDA.
 */
#ifndef RADT_H
#define RADT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RADT_VERSION 200          /* 0.2.0: per-call radt_options, cube_lo, packed-gradient access */
#define RADT_MAX_LEVELS 64        /* partition-function table length limit */
#define RADT_MAX_CHANNELS 256     /* channels per render call */

enum {
    RADT_OK = 0,
    RADT_E_INVALID = -1,          /* null pointer, non-positive size, bad struct_size, limits exceeded */
    RADT_E_UNSUPPORTED = -2,      /* grid kind / flag combination not implemented */
    RADT_E_WORKSPACE = -3,        /* workspace too small */
    RADT_E_CUDA = -4              /* CUDA runtime error (message in radt_last_error) */
};

enum { RADT_GRID_AXISYM = 0, RADT_GRID_CART3D = 1, RADT_GRID_SPH3D = 2 };
enum { RADT_DENS_LINEAR = 0, RADT_DENS_LN = 1 };
enum { RADT_VEL_VPHI = 0, RADT_VEL_KEPLER_FRAC = 1 };
enum { RADT_UNIT_S0 = 0, RADT_UNIT_CGS = 1, RADT_UNIT_JY_PIXEL = 2 };
enum { RADT_PASS_FWD = 0, RADT_PASS_BWD = 1 };

/* Image plane and viewing geometry of ONE batch item (Table 2 "Ray-tracing
 * Geometry": inclination, position angle, azimuth, distance, v_LSR).  Rays are orthographic, one per
 * pixel centre, X_ix = x0 + (ix + 1/2 - nx/2) fov_x / nx (O1-O3).  All batch items of a
 * call must share nx, ny and nstep. */
typedef struct radt_geom {
    uint32_t struct_size;         /* = sizeof(radt_geom) */
    int32_t nx, ny;               /* image size in pixels */
    int32_t nstep;                /* steps per ray (midpoint rule over the clipped interval) */
    double fov_x, fov_y;          /* au, full extent of the image */
    double x0, y0;                /* au, sky offset of the image centre from the star */
    double incl, pa, az;          /* rad */
    double dist_pc;               /* pc; only used by RADT_UNIT_JY_PIXEL */
    double vsys;                  /* cm/s, systemic velocity (v_LSR) */
    double gm_star;               /* cm^3 s^-2, G M_star; only used by RADT_VEL_KEPLER_FRAC */
} radt_geom;

/* One line in LTE and the channel grid (Eq. 13-17).  Level tables are HOST
 * pointers; the library copies them into kernel arguments at call time. */
typedef struct radt_line {
    uint32_t struct_size;         /* = sizeof(radt_line) */
    int32_t nlev;                 /* 1 .. RADT_MAX_LEVELS */
    int32_t nchan;                /* 1 .. RADT_MAX_CHANNELS */
    int32_t unit;                 /* RADT_UNIT_* of the output cube */
    double nu0;                   /* Hz, rest frequency */
    double a_ul;                  /* s^-1, Einstein A */
    double g_u;                   /* degeneracy of the upper level */
    double e_u_K;                 /* E_u / k [K] */
    const double *e_lev_K;        /* HOST [nlev], level energies / k for Q(T) */
    const double *g_lev;          /* HOST [nlev], level degeneracies */
    double m_line;                /* g, mass of the emitting molecule (m_CO in Eq. 16) */
    double m_gas;                 /* g, mean molecular mass (m_mol in Eq. 17) */
    double vturb_abs;             /* cm/s, absolute micro-turbulence added in quadrature */
    double vturb_mach;            /* dimensionless turbulent velocity of Eq. 16 */
    const double *vchan;          /* HOST [nchan], channel-centre velocities, cm/s, radio convention */
} radt_line;

/* Field grids of the whole batch (regular or log-spaced grids).
 *   AXISYM : n = {nr, nzeta, 1}; nodes r_i = lo[0] (hi[0]/lo[0])^(i/(nr-1)), zeta_j = lo[1] +
 *            (hi[1]-lo[1]) j/(nzeta-1), zeta = |z|/r if mirror_z else z/r (mirror_z needs lo[1] >= 0);
 *   CART3D : n = {nx, ny, nz}; nodes lo[a] + (hi[a]-lo[a]) i/(n[a]-1) in the disk frame.
 *   SPH3D  : n = {nr, ntheta, nphi}; r_i as AXISYM (spherical radius); theta_j = lo[1] + (hi[1]-lo[1]) j/(ntheta-1), the
 *            polar angle from the +z axis of the disk frame, 0 <= lo[1] < hi[1] <= pi; phi_k = 2 pi k/nphi, periodic
 *            (lo[2], hi[2] are ignored); arrays [b][ir][itheta][iphi].
 * Interpolation is bi/tri-linear in index space; outside the node range is vacuum.
 * dens/temp/vel are DEVICE pointers to float32 arrays [batch][cells]; item b starts at
 * ptr + b * batch_stride (elements).  Caller owns all memory. */
typedef struct radt_grid {
    uint32_t struct_size;         /* = sizeof(radt_grid) */
    int32_t kind;                 /* RADT_GRID_* */
    int32_t n[3];
    int32_t mirror_z;             /* AXISYM only */
    int32_t dens_mode;            /* RADT_DENS_LINEAR: n [cm^-3]; RADT_DENS_LN: ln n */
    int32_t vel_mode;             /* RADT_VEL_VPHI: v_phi [cm/s]; RADT_VEL_KEPLER_FRAC: delta, v_phi = v_K (1 + delta) */
    double lo[3], hi[3];
    int64_t batch_stride;         /* elements between batch items (>= cells), ignored for batch 1 */
    const float *dens;            /* DEVICE (HOST for the *_host entry points) */
    const float *temp;
    const float *vel;
} radt_grid;

int radt_version(void);
const char *radt_last_error(void);

/* Per-call options.  Every compute entry point takes a `const radt_options *` (HOST; NULL = the defaults that
 * radt_options_default writes).  There is no process-wide state: two threads may render with different options.
 * radt_render (or radt_render_loss) and the radt_render_bwd that differentiates its cube must be called with the same
 * window / skip_empty / win_path and the same cube_lo choice, because the adjoint re-marches the ray with the very
 * arithmetic of the forward; the library remembers, per cube pointer, the options of the last
 * forward that wrote it and radt_render_bwd fails with RADT_E_INVALID when they differ. */
typedef struct radt_options {
    uint32_t struct_size;         /* = sizeof(radt_options) */
    int32_t window;               /* 1 (default): channels outside the line window of a step (dtau < 2^-60 .. 2^-40 of its
                                     line-centre value) are skipped; 0: every channel of every step (dense) */
    int32_t skip_empty;           /* 1 (default): steps with zero opacity are skipped in the forward; 0: dense */
    int32_t win_path;             /* 1 (default): channel tables that are uniform lattices v_0 + c dv use the window kernels
                                     (one channel per lane inside the line window); 0: always the channel-table kernels */
    int32_t zero_dens_grad;       /* 1 (default): exact gradient; 0: the adjoint skips steps without opacity on LINEAR
                                     density grids.  Those steps carry only dL/dn of cells whose density is exactly zero
                                     (masked CO, Eq. 9), which a fit through radt_disk_fields_bwd discards anyway
                                     (the mask is held fixed), so g_temp, g_vel and g_dens at cells with non-zero density
                                     are unchanged.  They are 48-65 % of the adjoint's steps on the disk configs. */
    int32_t reuse_setup;          /* radt_render_bwd only.  0 (default): the call rebuilds ray table, Q(T) table, packed
                                     fields and occupancy words in the workspace.  1: the caller states that `ws` was last
                                     used by radt_render / radt_render_loss with the same geom, line, grid (same field
                                     pointers AND unchanged field values) and options; the adjoint then reuses what that
                                     call left there.  The library checks what it can (descriptors, pointers, options,
                                     remembered per workspace pointer) and fails with RADT_E_INVALID otherwise. */
} radt_options;
void radt_options_default(radt_options *opt);

/* Bytes of DEVICE workspace needed by radt_render (pass = RADT_PASS_FWD) or radt_render_bwd
 * (RADT_PASS_BWD) for `batch` items.  The size does not depend on the options; a RADT_PASS_BWD workspace also
 * serves the forward (same layout, the gradient cells come last).  HOST pointers in, size out. */
int radt_workspace_bytes(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                         int32_t pass, size_t *bytes_out);

/* K1: ray geometry (O1-O3).  Writes for every ray of every batch item
 * rays_out[(b*ny + iy)*nx + ix] = {s0, ds} (two doubles, au; ds = 0 marks a ray that misses the
 * volume).  geom: HOST [batch]; rays_out: DEVICE [batch*ny*nx*2] doubles. */
int radt_ray_geometry(const radt_geom *geom, const radt_grid *grid, int32_t batch, double *rays_out,
                      void *cuda_stream);

/* Forward render (O1-O10; Eq. 11-17).  Overwrites
 * cube [batch][ny][nx][nchan] (DEVICE float32, rays that miss write zeros).  geom: HOST [batch];
 * line, grid, opt: HOST structs; ws: DEVICE workspace of ws_bytes.  Asynchronous on cuda_stream.
 * cube_lo (DEVICE float32, same shape as cube, or NULL): the low-order word of the fp32 sum behind every voxel,
 * cube + cube_lo being that sum to about twice the precision.  Pass it on to radt_render_bwd: the adjoint forms the
 * residual intensity behind a step as (cube - P_k) + (cube_lo - P_lo,k), free of the cancellation noise that a ray
 * which is optically thick in every channel would otherwise put on its gradients.  `cube` is
 * the same bit for bit with and without it. */
int radt_render(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                const radt_options *opt, float *cube, float *cube_lo, void *ws, size_t ws_bytes, void *cuda_stream);

/* Adjoint (O11; Fig. 2 E).  Given the forward output `cube` (and `cube_lo` if the
 * forward wrote one, else NULL) and dl_dcube = dLoss/dcube (all DEVICE float32 [batch][ny][nx][nchan]) OVERWRITES
 * g_dens, g_temp, g_vel (DEVICE float32, grid-shaped incl. batch with the grid's batch_stride; any may be NULL) with
 * dLoss/d(stored grid value): d/d(ln n) for RADT_DENS_LN, d/d(delta) for RADT_VEL_KEPLER_FRAC.
 * Memory-free: no per-step activations are stored; the rays are re-marched.  Float atomics make
 * the last bits order-dependent.  With all three outputs NULL the gradient stays in the workspace as packed cells
 * (radt_grad_layout), e.g. for ONE all-reduce over ranks before radt_unpack_grad. */
int radt_render_bwd(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                    const radt_options *opt, const float *cube, const float *cube_lo, const float *dl_dcube,
                    float *g_dens, float *g_temp, float *g_vel, void *ws, size_t ws_bytes, void *cuda_stream);

/* Drops what the library remembers about a device pointer (the options of the last forward that wrote a cube there, the
 * setup a forward left in a workspace there).  The memory is keyed by raw pointer and knows nothing of cudaFree: call
 * this when a cube buffer is refilled by something other than radt_render / radt_render_loss (a copy, a collective, an
 * upload) or when the allocator may hand its address to a new tensor, so that a later radt_render_bwd is not refused on
 * the strength of a forward that no longer applies.  Unknown pointers are fine.  HOST call, no CUDA work. */
int radt_forget(const void *device_ptr);

/* Where radt_render_bwd leaves the gradient inside a RADT_PASS_BWD workspace: [batch][cells] packed float4 cells
 * {dL/d dens, dL/d temp, dL/d vel, 0}, *nfloat_out floats starting *offset_out bytes into `ws` (HOST outputs).
 * Multi-GPU image sharding sums exactly this range over the ranks with one all-reduce on the
 * adjoint's stream and then calls radt_unpack_grad. */
int radt_grad_layout(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     size_t *offset_out, size_t *nfloat_out);
/* Packed cells of `ws` -> the caller's three planes (DEVICE float32, grid's batch_stride; any may be NULL). */
int radt_unpack_grad(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     const void *ws, size_t ws_bytes, float *g_dens, float *g_temp, float *g_vel, void *cuda_stream);

/* L2 data term used by the configs (chi^2 of PAPER.md:79, 252):
 * L = 1/(2 n) sum ((cube - target)/sigma)^2, dl_dcube = (cube - target)/(sigma^2 n).
 * cube, target, dl_dcube: DEVICE float32 [n]; loss_out: DEVICE double[1] (overwritten). */
int radt_l2_loss_grad(const float *cube, const float *target, double sigma, int64_t n, float *dl_dcube,
                      double *loss_out, void *cuda_stream);

/* Forward render with the chi^2 data term fused into its epilogue (the step after the render in
 * the paper's fit, Fig. 2 D): writes cube (and cube_lo) as radt_render does and, without a
 * second pass over it, dl_dcube = (cube - target) / (sigma^2 n) and *loss_out = sum (cube - target)^2 / (2 sigma^2 n),
 * n = number of voxels of the whole batch.  Same results as radt_render followed by radt_l2_loss_grad (the loss up to
 * the order of its fp64 sum).  target, cube, cube_lo, dl_dcube: DEVICE float32 [batch][ny][nx][nchan]; loss_out:
 * DEVICE double[1]. */
int radt_render_loss(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     const radt_options *opt, const float *target, double sigma, float *cube, float *cube_lo,
                     float *dl_dcube, double *loss_out, void *ws, size_t ws_bytes, void *cuda_stream);

/* Same operations with HOST buffers (grid->dens/temp/vel, cube, cube_lo, dl_dcube, g_* are HOST pointers).
 * Device memory comes from an arena the library keeps per calling thread and device (grown on demand, never
 * returned); the work runs on stream 0 of the current device and the call returns after the results are in host
 * memory.  cube_lo may be NULL in both calls that take it. */
int radt_render_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     const radt_options *opt, float *cube, float *cube_lo);
/* Forward + chi^2 term against `target` (HOST; uploaded on a second stream under the forward march) + adjoint in one
 * call; the low-order words stay on the device; cube may be NULL.  Batched calls (radt_fit_step_host and radt_render_host)
 * whose cube exceeds 32 MB run in chunks of items of at most 32 MB of cube (at least one item), and single images of more
 * than 16 MB in bands of rows of about 16 MB (one setup; per band the forward march and, in a fit step on axisymmetric grids,
 * the adjoint march of the same rows; fit steps on 3-D grids stay in one piece), the transfers of one chunk / band under the
 * marches of another; the results are those of the one-call path (cube bit for bit).  If a call fails half-way the library
 * waits for every transfer it started before it returns, so the host buffers are the caller's again on every return. */
int radt_fit_step_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                       const radt_options *opt, const float *target, double sigma, float *cube, double *loss_out,
                       float *g_dens, float *g_temp, float *g_vel);
int radt_render_bwd_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                         const radt_options *opt, const float *cube, const float *cube_lo, const float *dl_dcube,
                         float *g_dens, float *g_temp, float *g_vel);

/* ---- Physics pre-pass (Eq. 1-2, 6-9) ---------------------------------
 * Turns a temperature grid into the render's CO density and v_phi grids, as the paper's fit does before every render:
 * hydrostatic density along z (Eq. 1, trapezoid rule), normalised to the surface density of Eq. 2 (both sides of the
 * mirror-symmetric disk), H2 column above every node (Eq. 8), CO abundance mask (Eq. 7, 9), rotation with the radial
 * pressure gradient (Eq. 6, centred differences on the (ln r, zeta) grid).  DESIGN.md section 10 states the
 * discretisation P1-P7.  One radt_disk per batch item (HOST). */
typedef struct radt_disk {
    uint32_t struct_size;         /* = sizeof(radt_disk) */
    uint32_t pad_;
    double gm_star;               /* cm^3 s^-2 */
    double m_gas;                 /* g, mean molecular mass (m_mol of Eq. 1) */
    double sigma0;                /* g cm^-2, Eq. 2 */
    double r_c;                   /* au, Eq. 2 */
    double gamma;                 /* Eq. 2 */
    double x_co;                  /* Eq. 7 (1e-4) */
    double t_freeze;              /* K, Eq. 9 */
    double n_dissoc;              /* cm^-2, Eq. 9 */
    double f_col;                 /* Eq. 9 (0.706) */
} radt_disk;

/* `grid` gives the node layout only (kind AXISYM with mirror_z = 1 and lo[1] = 0, dens_mode LINEAR, vel_mode VPHI; its
 * field pointers are ignored); item b of every array starts at b * grid->batch_stride elements.
 * radt_disk_fields: temp (DEVICE float32 [batch][nr][nzeta], K) -> dens_out = n_CO [cm^-3], vel_out = v_phi [cm/s]
 * (DEVICE float32, overwritten).
 * radt_disk_fields_bwd: ADDS to g_temp (DEVICE float32, in/out) the gradient that reaches the temperature through the
 * density and velocity fields, d L/d temp += (d n_CO/d temp)^T g_dens + (d v_phi/d temp)^T g_vel, with the CO mask held
 * fixed (it is piecewise constant); g_dens, g_vel: DEVICE float32 as returned by radt_render_bwd.  Passing the
 * render's own g_temp therefore yields the total derivative w.r.t. the temperature grid.
 * Both are asynchronous on cuda_stream, never allocate, and recompute what they need (no state between calls). */
int radt_disk_workspace_bytes(const radt_grid *grid, int32_t batch, size_t *bytes_out);
int radt_disk_fields(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp, float *dens_out,
                     float *vel_out, void *ws, size_t ws_bytes, void *cuda_stream);
int radt_disk_fields_bwd(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp,
                         const float *g_dens, const float *g_vel, float *g_temp, void *ws, size_t ws_bytes,
                         void *cuda_stream);

/* radt_disk_fields without a workspace, for callers that cannot allocate device memory.  Who that is: a plug-in or
 * solver running inside a process whose device memory was handed out in full at start-up (to the host application's
 * pool, or to fixed partitions of a control loop), where a cudaMalloc for the workspace fails or is forbidden, and loops
 * that cannot accept the device-wide synchronisation and the unbounded latency of cudaMalloc / cudaFree.  The scratch
 * that radt_disk_fields keeps in `ws` lives here in a fixed array inside the library image instead: about 8 MiB that
 * EVERY GPU which loads libradt.so holds until the process exits, used or not.  The caller still passes the inputs and
 * the outputs (DEVICE float32, as radt_disk_fields); results are those of radt_disk_fields (same kernels).
 *   - Limit: batch * nr * nzeta <= RADT_DISK_STATIC_MAX_CELLS (configs 1-3 whole, config 5 in two halves); more fails
 *     with RADT_E_INVALID before anything is launched.  Split the batch, or use radt_disk_fields.
 *   - The call itself makes no cudaMalloc / cudaFree and calls no allocating library routine.  The FIRST call on each
 *     device looks up the array's device address (cudaGetSymbolAddress, with that device current; the runtime may load
 *     the library's kernels onto the device at that moment).  Make that first call early, with the device you will use
 *     current, and before any stream capture is begun.
 *   - One array per device serves every call, and it keeps what the last call left.  Nothing needs clearing (each call
 *     overwrites all it reads), but two calls that overlap on the same GPU (different streams, different threads) race
 *     on it: order them on one stream or with events.  Calls on different devices do not interfere.
 * Asynchronous on cuda_stream; disk, grid: HOST, as radt_disk_fields. */
#define RADT_DISK_STATIC_MAX_CELLS 262144
int radt_disk_fields_static(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp,
                            float *dens_out, float *vel_out, void *cuda_stream);

/* ---- Symmetric MLP temperature field (Eq. 10) ----------------------------------------
 * T(r, |z|) = MLP_w(gamma(r, |z|)) on the nodes of an AXISYM grid (mirror symmetric, so a function of |z|):
 * p = (i/(nr-1), j/(nzeta-1)); gamma(p) = (p_0, p_1, {sin(2^k pi p_0), cos(2^k pi p_0), sin(2^k pi p_1), cos(2^k pi p_1)},
 * k = 0..L-1); `nhidden` fully connected layers of `width` units with ReLU; T = t_lo + (t_hi - t_lo) sigmoid(w . h + b).
 * Parameters: one flat DEVICE float32 vector [W_1 (width x D) | b_1 | W_2 (width x width) | b_2 | ... | w_out (width) |
 * b_out], row-major, D = 2 + 4 L; its length comes from radt_mlp_num_params.  This build supports width = 64,
 * nhidden = 4 (the paper's network) and L <= 8. */
typedef struct radt_mlp {
    uint32_t struct_size;         /* = sizeof(radt_mlp) */
    int32_t L;                    /* degree of the positional encoding (paper: 4) */
    int32_t width, nhidden;       /* 64, 4 */
    double t_lo, t_hi;            /* K (paper: 5, 400) */
} radt_mlp;

int radt_mlp_num_params(const radt_mlp *mlp, int64_t *count_out);
/* temp_out: DEVICE float32 [nr][nzeta] (overwritten).  grid: node counts only (kind AXISYM). */
int radt_mlp_temperature(const radt_mlp *mlp, const radt_grid *grid, const float *params, float *temp_out,
                         void *cuda_stream);
/* g_params (DEVICE float32 [num_params], OVERWRITTEN) = (dT/dparams)^T g_temp; g_temp: DEVICE float32 [nr][nzeta].
 * Recomputes the activations (nothing is kept from the forward); float atomics make the last bits order dependent.
 * Accuracy: every contraction of the adjoint, the recomputation of the activations included, runs as split-bf16 products with
 * fp32 accumulation, about 2^-16 relative per product, where the forward's three-product split is good to about fp32.  Away
 * from the ReLU kinks the parameter gradient of a whole grid agrees with an fp64 evaluation to ~2.5e-5 of its largest entry.
 * relu' is decided on the adjoint's own recomputed pre-activation: a unit within ~1e-4 (relative to the layer's scale) of
 * its kink may take the other branch than the forward and an fp64 evaluation do.  Both branches are valid subgradients, but
 * the result is then NOT within the 1e-3 gradient tolerance of an fp64 reference: measured 6e-3 of the largest entry (4e-3
 * in L2) on a 256 x 128 grid with a random network of three times the initialisation scale, no node masked
 * (tests/test_gpu_mlp_field.py).  A recomputation with a third bf16 term would remove this; it is not built. */
int radt_mlp_temperature_bwd(const radt_mlp *mlp, const radt_grid *grid, const float *params, const float *g_temp,
                             float *g_params, void *cuda_stream);

/* M1 micro-benchmarks of the issue peaks the roofline is quoted against.
 * Runs a full-occupancy dependent-chain loop of `kind` on the current device and returns the
 * achieved rate in lane-operations per second (HOST double).  kind: 0 MUFU.EX2, 1 FFMA, 2 DFMA,
 * 3 FFMA2 (packed f32x2, counted as 2 lane-ops). */
int radt_pipe_peak(int32_t kind, double *ops_per_s_out, double *sm_clock_mhz_out);

/* Work counters of the last render / adjoint that used workspace `ws` (DEVICE): copies 4 uint64 to
 * out4 (HOST): {forward active ray-steps, forward per-sample MUFU.EX2 warp instructions (x32 = transcendental
 * lane-operations spent on (channel, step) samples), adjoint active ray-steps, adjoint per-sample MUFU.EX2 warp
 * instructions}.  Synchronises cuda_stream. */
int radt_read_counters(const void *ws, uint64_t *out4, void *cuda_stream);
/* Lane use of the last FORWARD march on workspace `ws` (window kernels; executed work is reported beside
 * nominal work): out2 (HOST) = {(channel, step) samples inside the line window of their step, i.e. samples that can contribute;
 * samples executed = 32 lanes x emitting steps}.  The channel-table kernels leave the first figure 0.  Synchronises cuda_stream. */
int radt_read_lane_counters(const void *ws, uint64_t *out2, void *cuda_stream);

/* Counters of the last radt_render / radt_render_bwd call on this thread (HOST): number of kernel
 * launches enqueued. */
int radt_last_launch_count(void);

/* TEST HOOK of the *_host entry points, per calling thread: chunk_items >= 1 forces batched calls into chunks of that many
 * items, band_rows >= 1 forces single images into bands of that many rows (rounded up to whole tile rows; also for fit steps
 * on 3-D grids), whatever their size; 0 restores the library's own policy.  Results do not depend on it (tests/ checks that
 * on small scenes); it exists so that the chunked and banded paths can be exercised without gigabyte inputs. */
int radt_debug_host_split(int32_t chunk_items, int32_t band_rows);

#ifdef __cplusplus
}
#endif
#endif /* RADT_H */
