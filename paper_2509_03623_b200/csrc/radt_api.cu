// radt_api.cu -- the C ABI of include/radt.h: validation, host-side constants, workspace layout, launches.
// No CPU fallback: every compute entry point enqueues CUDA kernels or fails with RADT_E_CUDA.
#include "../../include/radt.h"
#include "radt_dev.cuh"
#include "radt_kernels.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

namespace {

thread_local char g_err[512] = "";
thread_local int g_launches = 0;

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                     \
    do {                                                                                   \
        cudaError_t e_ = (expr);                                                           \
        if (e_ != cudaSuccess) return fail(RADT_E_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
    } while (0)

// Resolved per-call options (include/radt.h radt_options; NULL = defaults).  No process-wide option state.
struct Opts {
    int window = 1, skip_empty = 1, win_path = 1, zero_dens_grad = 1, reuse_setup = 0;
};

int resolve_options(const radt_options *o, Opts &out)
{
    out = Opts();
    if (!o) return RADT_OK;
    if (o->struct_size != sizeof(radt_options)) return fail(RADT_E_INVALID, "radt_options.struct_size mismatch");
    out.window = o->window != 0; out.skip_empty = o->skip_empty != 0; out.win_path = o->win_path != 0;
    out.zero_dens_grad = o->zero_dens_grad != 0; out.reuse_setup = o->reuse_setup != 0;
    return RADT_OK;
}

// What the library remembers between a forward and its adjoint (HOST side, keyed by device pointer, a few entries,
// oldest replaced): per cube the options that shaped its partial sums, per workspace what the last forward left there.
struct Remembered {
    const void *key = nullptr;
    unsigned long long tag = 0;
    unsigned long long age = 0;
};
struct Registry {
    static const int N = 64;
    Remembered e[N];
    unsigned long long clock = 0;
    std::mutex mu;
    void put(const void *key, unsigned long long tag)
    {
        std::lock_guard<std::mutex> lk(mu);
        int slot = 0;
        for (int i = 0; i < N; ++i) {
            if (e[i].key == key) { slot = i; break; }
            if (e[i].age < e[slot].age) slot = i;
        }
        e[slot].key = key; e[slot].tag = tag; e[slot].age = ++clock;
    }
    bool get(const void *key, unsigned long long &tag)
    {
        std::lock_guard<std::mutex> lk(mu);
        for (int i = 0; i < N; ++i)
            if (e[i].key == key && e[i].age) { tag = e[i].tag; return true; }
        return false;
    }
    void forget(const void *key)
    {
        std::lock_guard<std::mutex> lk(mu);
        for (int i = 0; i < N; ++i)
            if (e[i].key == key) e[i] = Remembered();
    }
};
Registry g_cubes, g_workspaces;
// Set while a HOST entry point runs its passes on the arena's own buffers: those calls pair every forward with its adjoint
// themselves, so their cubes and workspaces stay out of the shared tables (a chunked call would otherwise push up to 256
// entries through the 64 slots and silently evict what the callers of the DEVICE entry points rely on).
thread_local bool g_internal_pass = false;
// Test hook of the HOST entry points (radt_debug_host_split): forced chunk / band sizes of the calling thread, 0 = the library's
// own policy.  (Until round 3 these were environment variables read on every call of the shipped library.)
thread_local int g_force_chunk_items = 0, g_force_band_rows = 0;
struct InternalPass {
    bool prev;
    InternalPass() : prev(g_internal_pass) { g_internal_pass = true; }
    ~InternalPass() { g_internal_pass = prev; }
};

unsigned long long fnv(unsigned long long h, const void *p, size_t n)
{
    const unsigned char *b = (const unsigned char *)p;
    for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    return h;
}

// CODATA 2018, CGS
const double kH = 6.62607015e-27, kK = 1.380649e-16, kC = 2.99792458e10;
const double kAU = 1.495978707e13, kPC = 3.0856775814913673e18, kPI = 3.14159265358979323846;
const double kLOG2E = 1.4426950408889634;

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int validate(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int batch)
{
    if (!geom || !grid) return fail(RADT_E_INVALID, "null descriptor");
    if (batch < 1) return fail(RADT_E_INVALID, "batch must be >= 1");
    if (grid->struct_size != sizeof(radt_grid)) return fail(RADT_E_INVALID, "radt_grid.struct_size mismatch");
    for (int b = 0; b < batch; ++b) {
        const radt_geom &g = geom[b];
        if (g.struct_size != sizeof(radt_geom)) return fail(RADT_E_INVALID, "radt_geom.struct_size mismatch");
        if (g.nx < 1 || g.ny < 1 || g.nstep < 1) return fail(RADT_E_INVALID, "nx, ny, nstep must be positive");
        if (!(g.fov_x > 0) || !(g.fov_y > 0)) return fail(RADT_E_INVALID, "fov must be positive");
        if (g.nx != geom[0].nx || g.ny != geom[0].ny || g.nstep != geom[0].nstep)
            return fail(RADT_E_INVALID, "all batch items must share nx, ny, nstep");
        if ((long long)g.nx * g.ny * (long long)batch > (1ll << 40)) return fail(RADT_E_INVALID, "too many rays");
    }
    if (line) {
        if (line->struct_size != sizeof(radt_line)) return fail(RADT_E_INVALID, "radt_line.struct_size mismatch");
        if (line->nlev < 1 || line->nlev > RADT_MAX_LEVELS) return fail(RADT_E_INVALID, "nlev out of range");
        if (line->nchan < 1 || line->nchan > RADT_MAX_CHANNELS) return fail(RADT_E_INVALID, "nchan out of range (max %d)", RADT_MAX_CHANNELS);
        if (!line->e_lev_K || !line->g_lev || !line->vchan) return fail(RADT_E_INVALID, "null line table");
        if (!(line->nu0 > 0) || !(line->a_ul > 0) || !(line->m_line > 0) || !(line->m_gas > 0))
            return fail(RADT_E_INVALID, "line constants must be positive");
        if (line->unit < 0 || line->unit > 2) return fail(RADT_E_INVALID, "unknown intensity unit");
    }
    if (grid->kind == RADT_GRID_AXISYM) {
        if (grid->n[0] < 2 || grid->n[1] < 2) return fail(RADT_E_INVALID, "axisymmetric grid needs >= 2 nodes per axis");
        if (!(grid->lo[0] > 0) || !(grid->hi[0] > grid->lo[0])) return fail(RADT_E_INVALID, "need 0 < r_min < r_max");
        if (!(grid->hi[1] > grid->lo[1])) return fail(RADT_E_INVALID, "need zeta_lo < zeta_hi");
        if (grid->mirror_z && grid->lo[1] < 0) return fail(RADT_E_INVALID, "mirror_z needs zeta_lo >= 0");
    } else if (grid->kind == RADT_GRID_CART3D) {
        for (int a = 0; a < 3; ++a) {
            if (grid->n[a] < 2) return fail(RADT_E_INVALID, "3-D grid needs >= 2 nodes per axis");
            if (!(grid->hi[a] > grid->lo[a])) return fail(RADT_E_INVALID, "need lo < hi");
        }
        if (grid->mirror_z) return fail(RADT_E_UNSUPPORTED, "mirror_z applies to axisymmetric grids only");
    } else if (grid->kind == RADT_GRID_SPH3D) {
        for (int a = 0; a < 3; ++a)
            if (grid->n[a] < 2) return fail(RADT_E_INVALID, "spherical grid needs >= 2 nodes per axis");
        if (!(grid->lo[0] > 0) || !(grid->hi[0] > grid->lo[0])) return fail(RADT_E_INVALID, "need 0 < r_min < r_max");
        if (!(grid->lo[1] >= 0) || !(grid->hi[1] > grid->lo[1]) || !(grid->hi[1] <= kPI))
            return fail(RADT_E_INVALID, "need 0 <= theta_lo < theta_hi <= pi");
        if (grid->mirror_z) return fail(RADT_E_UNSUPPORTED, "mirror_z applies to axisymmetric grids only");
    } else {
        return fail(RADT_E_UNSUPPORTED, "unknown grid kind %d", grid->kind);
    }
    if (grid->dens_mode < 0 || grid->dens_mode > 1 || grid->vel_mode < 0 || grid->vel_mode > 1)
        return fail(RADT_E_UNSUPPORTED, "unknown dens_mode / vel_mode");
    if ((grid->kind == RADT_GRID_AXISYM ? (long long)grid->n[0] * grid->n[1] : (long long)grid->n[0] * grid->n[1] * grid->n[2]) >
        (1ll << 30))
        return fail(RADT_E_INVALID, "grid too large: at most 2^30 cells per batch item");
    return RADT_OK;
}

long long grid_cells(const radt_grid *grid)
{
    return grid->kind == RADT_GRID_AXISYM ? (long long)grid->n[0] * grid->n[1]
                                          : (long long)grid->n[0] * grid->n[1] * grid->n[2];
}

void make_dev_grid(const radt_grid *grid, DevGrid &d)
{
    memset(&d, 0, sizeof(d));
    d.kind = grid->kind; d.mirror = grid->mirror_z; d.dens_mode = grid->dens_mode; d.vel_mode = grid->vel_mode;
    d.n0 = grid->n[0]; d.n1 = grid->n[1]; d.n2 = grid->kind == RADT_GRID_AXISYM ? 1 : grid->n[2];
    d.cells = grid_cells(grid);
    if (grid->kind == RADT_GRID_AXISYM || grid->kind == RADT_GRID_SPH3D) {
        double rmin = grid->lo[0], rmax = grid->hi[0];
        d.rmin2 = rmin * rmin; d.rmax2 = rmax * rmax; d.inv_rmin = 1.0 / rmin;
        {
            // smallest double t with sqrt(t) >= r_min and largest with sqrt(t) <= r_max (IEEE sqrt is correctly rounded and
            // monotone): a step whose radius equals a boundary up to rounding is then decided as a plain fp64 evaluation
            // decides it (random scenes 4841, 6865: a ray through the star with |s| = r_min exactly)
            double t = d.rmin2;
            while (t > 0.0 && std::sqrt(t) >= rmin) t = std::nextafter(t, 0.0);
            while (std::sqrt(t) < rmin) t = std::nextafter(t, INFINITY);
            d.rho2_lo = t;
            t = d.rmax2;
            while (std::sqrt(t) <= rmax) t = std::nextafter(t, INFINITY);
            while (std::sqrt(t) > rmax) t = std::nextafter(t, 0.0);
            d.rho2_hi = t;
        }
        d.zlo = grid->lo[1]; d.zhi = grid->hi[1];
        d.lg2_ratio = std::log2(rmax / rmin);
        d.uscale = (float)((double)(grid->n[0] - 1) / d.lg2_ratio);
        d.wscale_d = (double)(grid->n[1] - 1) / (grid->hi[1] - grid->lo[1]);
        double cell_lg2 = d.lg2_ratio / (double)(grid->n[0] - 1);
        d.inv_cell_lg2 = (float)(1.0 / cell_lg2);
        d.inv_cell_ln = (float)(1.0 / (cell_lg2 * std::log(2.0)));
        d.fine_r = (std::exp2(2.0 * cell_lg2) - 1.0) < 0.35;
        d.zlo_f = (float)d.zlo; d.wscale_f = (float)d.wscale_d;
        d.inv_rmin2_f = (float)(1.0 / (rmin * rmin)); d.half_uscale = (float)(0.5 * (double)(grid->n[0] - 1) / d.lg2_ratio);
        double zm = std::fmax(std::fabs(grid->lo[1]), std::fabs(grid->hi[1]));
        d.rb2 = rmax * rmax * (1.0 + zm * zm);
        if (grid->kind == RADT_GRID_SPH3D) {
            d.n2 = grid->n[2];
            d.rb2 = rmax * rmax;
            d.cos_tlo = std::cos(grid->lo[1]); d.cos_thi = std::cos(grid->hi[1]);
            d.th_c0 = (float)(0.5 * kPI - grid->lo[1]);
            d.th_scale = (float)((double)(grid->n[1] - 1) / (grid->hi[1] - grid->lo[1]));
            d.ph_scale = (float)((double)grid->n[2] / (2.0 * kPI));
        }
    } else {
        for (int a = 0; a < 3; ++a) {
            d.lo[a] = grid->lo[a]; d.hi[a] = grid->hi[a];
            d.inv_d[a] = (double)(grid->n[a] - 1) / (grid->hi[a] - grid->lo[a]);
            d.pre_lo[a] = (float)d.lo[a]; d.pre_inv_d[a] = (float)d.inv_d[a];
        }
    }
    d.pre_n0f = (float)d.n0; d.pre_n1f = (float)d.n1; d.pre_n2f = (float)d.n2;
    if (grid->kind != RADT_GRID_CART3D) {
        // u = log2(r / r_min) (nr - 1) / log2(r_max / r_min) = lg2(r^2) us_half - lg2(r_min) uscale
        d.pre_us_half = (float)(0.5 * (double)(grid->n[0] - 1) / d.lg2_ratio);
        d.pre_uoff = (float)(-std::log2(grid->lo[0]) * (double)(grid->n[0] - 1) / d.lg2_ratio);
        d.pre_wscale = (float)d.wscale_d;
        d.pre_woff = (float)(-d.zlo * d.wscale_d);
        if (grid->kind == RADT_GRID_SPH3D) {
            // margins: one radial cell (as on the axisymmetric grid), two theta cells in z/rho (|d cos| <= |d theta|)
            const double dth = 2.0 / (double)d.th_scale;
            d.pre_czlo = (float)(d.cos_thi - dth); d.pre_czhi = (float)(d.cos_tlo + dth);
            d.pre_cscale = (float)((double)grid->n[1] / ((double)d.pre_czhi - (double)d.pre_czlo) * (1.0 - 1e-6));
        }
    }
}

// The prefilter of the window kernels locates steps in fp32 (positions good to ~1e-7 of the grid's extent) and
// tolerates one cell of error: require the smallest cell to be 100 times coarser than that.
bool prefilter_safe(const radt_grid *grid)
{
    if (grid->kind == RADT_GRID_SPH3D) return true;      // its prefilter tests the (r, theta) range with wide margins only
    if (grid->kind == RADT_GRID_AXISYM) {
        double rmin = grid->lo[0], rmax = grid->hi[0];
        double zm = std::fmax(std::fabs(grid->lo[1]), std::fabs(grid->hi[1]));
        double ext = rmax * std::sqrt(1.0 + zm * zm);
        double dr = rmin * (std::pow(rmax / rmin, 1.0 / (grid->n[0] - 1)) - 1.0);
        double dz = rmin * (grid->hi[1] - grid->lo[1]) / (grid->n[1] - 1);
        return std::fmin(dr, dz) > 1.2e-5 * ext;
    }
    double ext = 0.0, dmin = 1e300;
    for (int a = 0; a < 3; ++a) {
        ext = std::fmax(ext, std::fmax(std::fabs(grid->lo[a]), std::fabs(grid->hi[a])));
        dmin = std::fmin(dmin, (grid->hi[a] - grid->lo[a]) / (grid->n[a] - 1));
    }
    return dmin > 1.2e-5 * ext;
}

double source_unit(const radt_geom &g, const radt_line *line)
{
    double S0 = 2.0 * kH * line->nu0 * line->nu0 * line->nu0 / (kC * kC);
    if (line->unit == RADT_UNIT_CGS) return S0;
    if (line->unit == RADT_UNIT_JY_PIXEL) {
        double d_au = g.dist_pc * kPC / kAU;
        return S0 * (g.fov_x / g.nx) * (g.fov_y / g.ny) / (d_au * d_au) * 1.0e23;
    }
    return 1.0;
}

void make_dev_geom(const radt_geom &g, const radt_line *line, DevGeom &d)
{
    double th = g.pa + 0.5 * kPI;
    d.cth = std::cos(th); d.sth = std::sin(th);
    d.ci = std::cos(g.incl); d.si = std::sin(g.incl);
    d.ca = std::cos(g.az); d.sa = std::sin(g.az);
    d.wx = d.si * d.sa; d.wy = d.si * d.ca; d.wz = -d.ci;
    d.x0 = g.x0; d.y0 = g.y0; d.pix_x = g.fov_x / g.nx; d.pix_y = g.fov_y / g.ny;
    d.gm_au_d = std::fmax(g.gm_star, 0.0) / kAU;
    d.sunit = line ? (float)source_unit(g, line) : 1.0f;
    d.wxf = (float)d.wx; d.wyf = (float)d.wy; d.wzf = (float)d.wz;
}

void make_dev_line(const radt_line *line, DevLine &d)
{
    double T0 = kH * line->nu0 / kK;
    d.T0 = (float)T0; d.T0l2 = (float)(T0 * kLOG2E);
    d.Eu = (float)line->e_u_K; d.Eul2 = (float)(line->e_u_K * kLOG2E);
    d.gu = (float)line->g_u;
    d.a1 = (float)(2.0 * kK / line->m_line + line->vturb_mach * line->vturb_mach * 2.0 * kK / line->m_gas);
    d.a0 = (float)(line->vturb_abs * line->vturb_abs);
    double Ck = kC * kC / (8.0 * kPI * line->nu0 * line->nu0) * line->a_ul * kC / (line->nu0 * std::sqrt(kPI)) * kAU;
    d.Ck2 = (float)(Ck * kLOG2E);
    d.nchan = line->nchan;
    d.ngroups = (line->nchan + 31) / 32;
    // uniform channel lattice v_c = v_0 + c dv (any sign of dv)?  One channel counts as a lattice of 1 km/s.
    const int n = line->nchan;
    double dv = n > 1 ? (line->vchan[n - 1] - line->vchan[0]) / (double)(n - 1) : 1.0e5;
    bool uni = dv != 0.0 && std::isfinite(dv);
    for (int c = 0; c < n && uni; ++c)
        if (!(std::fabs(line->vchan[c] - (line->vchan[0] + c * dv)) <= 1e-9 * std::fabs(dv))) uni = false;
    d.uniform = uni ? 1 : 0;
    d.inv_dv = uni ? 1.0 / dv : 0.0;
    d.dvf = uni ? (float)(dv * std::sqrt(kLOG2E)) : 0.f;
    d.c_hw = uni ? (float)(1.0 / (std::sqrt(kLOG2E) * std::fabs(dv))) : 0.f;
}

struct WsLayout {
    size_t rays, qtab, vcs, rnode, cells, occ, grad, counters, nodeflag, total;
    size_t zero_bytes;                  // counters + spherical node flags: one memset per pass
    int occ_wpr, occ_words, occ_nbj, flag_wpr;
};

WsLayout ws_layout(const radt_geom *geom, const radt_grid *grid, int batch, int pass)
{
    WsLayout w;
    size_t off = 0;
    size_t nrays = (size_t)geom[0].nx * geom[0].ny * (size_t)batch;
    w.counters = off; off = off + (8 + RADT_LOSS_SLOTS) * sizeof(unsigned long long);
    // spherical grids: (i, j) node flags of the occupancy prefilter, zeroed together with the counters
    w.nodeflag = off;
    w.flag_wpr = grid->kind == RADT_GRID_SPH3D ? (grid->n[1] + 31) / 32 : 0;
    off = off + (size_t)w.flag_wpr * (size_t)grid->n[0] * (size_t)batch * sizeof(unsigned);
    w.zero_bytes = off - w.counters;
    off = align256(off);
    w.rays = off; off = align256(off + nrays * sizeof(RayRec));
    w.qtab = off; off = align256(off + (RADT_NQ + 2) * sizeof(float2));
    w.vcs = off; off = align256(off + (size_t)batch * RADT_MAXCHAN * sizeof(float2));
    w.rnode = off; off = align256(off + (size_t)(grid->kind != RADT_GRID_CART3D ? grid->n[0] : 1) * sizeof(double2));
    size_t cells = (size_t)grid_cells(grid) * (size_t)batch;
    w.cells = off; off = align256(off + cells * sizeof(float4));
    if (grid->kind == RADT_GRID_AXISYM) {
        // bit (I, J), I = floor(u) + 1 in 0..nr, J = floor(w) + 1 in 0..nzeta (radt_setup.cu)
        w.occ_wpr = (grid->n[1] + 1 + 31) / 32;
        w.occ_words = (grid->n[0] + 1) * w.occ_wpr;
        w.occ_nbj = 1;
    } else if (grid->kind == RADT_GRID_SPH3D) {
        // bit (I, C): I = floor(u) + 1 in 0..nr, C = bin of cos(theta) in 0..ntheta-1, any phi (radt_setup.cu k_occ_sph)
        w.occ_wpr = (grid->n[1] + 31) / 32;
        w.occ_words = (grid->n[0] + 1) * w.occ_wpr;
        w.occ_nbj = 1;
    } else {
        // 3-D: one bit per block of 4 x 4 x 4 cells
        int nbi = (grid->n[0] - 1 + 3) / 4, nbj = (grid->n[1] - 1 + 3) / 4, nbl = (grid->n[2] - 1 + 3) / 4;
        w.occ_wpr = (nbl + 31) / 32;
        w.occ_nbj = nbj;
        w.occ_words = nbi * nbj * w.occ_wpr;
    }
    w.occ = off; off = align256(off + (size_t)w.occ_words * (size_t)batch * sizeof(unsigned));
    w.grad = off;
    if (pass == RADT_PASS_BWD) off = align256(off + cells * sizeof(float4));
    w.total = off;
    return w;
}

DevWs make_dev_ws(void *ws, const WsLayout &w)
{
    char *base = (char *)ws;
    DevWs d;
    d.counters = (unsigned long long *)(base + w.counters);
    d.rays = (RayRec *)(base + w.rays);
    d.qtab = (float2 *)(base + w.qtab);
    d.vcs = (float2 *)(base + w.vcs);
    d.rnode = (double2 *)(base + w.rnode);
    d.cells = (float4 *)(base + w.cells);
    d.occ = (unsigned *)(base + w.occ);
    d.nodeflag = (unsigned *)(base + w.nodeflag);
    d.grad = (float4 *)(base + w.grad);
    return d;
}

// fused chi^2 data term of a forward pass (radt_render_loss); target == nullptr: plain render
struct LossArgs {
    const float *target = nullptr;
    float *dl_out = nullptr;
    double *loss = nullptr;
    double sigma = 0.0;
    double nvox_total = 0.0;      // > 0: the call renders a chunk of a larger batch; normalise with the whole batch's voxel count
};

// A row band of the image (HOST entry points: transfers of one band under the marches of another).  nty == 0: the whole image
// in one launch.  Only the FIRST band of a pass runs the setup kernel and the zeroing, only the LAST one the loss reduction /
// the gradient unpack; the bands of one pass share workspace, ray table and (adjoint) gradient cells.
struct Band {
    int ty0 = 0, nty = 0;
    bool first = true, last = true;
};

// What shapes the partial sums of a cube (a forward and its adjoint must agree on it): the skipping and window switches, the
// kernel family, the low-order words and the channel count.  NOT the batch or the image size: the adjoint of the first items
// of a batched forward (same pointer, smaller batch) is a valid call ...
unsigned long long cube_tag(const Opts &o, bool use_win, bool comp, const radt_line *line)
{
    unsigned long long h = 1469598103934665603ull;
    const int v[5] = { o.window, o.skip_empty, use_win ? 1 : 0, comp ? 1 : 0, line->nchan };
    return fnv(h, v, sizeof(v)) | 1ull;
}
// ... and what a forward leaves in its workspace for an adjoint with reuse_setup: every input of the setup kernel.
unsigned long long setup_tag(const Opts &o, bool use_win, const radt_geom *geom, const radt_line *line, const radt_grid *grid,
                             int batch)
{
    unsigned long long h = 1469598103934665603ull;
    h = fnv(h, geom, sizeof(radt_geom) * (size_t)batch);
    h = fnv(h, grid, sizeof(radt_grid));
    radt_line l = *line;
    l.e_lev_K = nullptr; l.g_lev = nullptr; l.vchan = nullptr;
    h = fnv(h, &l, sizeof(l));
    h = fnv(h, line->e_lev_K, sizeof(double) * (size_t)line->nlev);
    h = fnv(h, line->g_lev, sizeof(double) * (size_t)line->nlev);
    h = fnv(h, line->vchan, sizeof(double) * (size_t)line->nchan);
    const int v[4] = { o.window, o.skip_empty, use_win ? 1 : 0, batch };
    return fnv(h, v, sizeof(v)) | 1ull;
}

// Enqueue setup + march for all batch chunks.  pass 0: forward into `cube`; pass 1: adjoint.
int run_pass(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int batch, const radt_options *opt_in,
             int pass, float *cube, float *cube_lo, const float *dl_dcube, float *g_dens, float *g_temp, float *g_vel,
             void *ws, size_t ws_bytes, cudaStream_t st, const LossArgs &loss = LossArgs(), const Band &band = Band())
{
    int rc = validate(geom, line, grid, batch);
    if (rc) return rc;
    Opts opt;
    if ((rc = resolve_options(opt_in, opt)) != 0) return rc;
    if (!line) return fail(RADT_E_INVALID, "null line descriptor");
    if (!ws) return fail(RADT_E_INVALID, "null workspace");
    if (!grid->dens || !grid->temp || !grid->vel) return fail(RADT_E_INVALID, "null field pointer");
    if (!cube) return fail(RADT_E_INVALID, "null cube pointer");
    if (pass == RADT_PASS_BWD && !dl_dcube) return fail(RADT_E_INVALID, "null dl_dcube pointer");
    if (pass == RADT_PASS_FWD && opt.reuse_setup) return fail(RADT_E_INVALID, "reuse_setup applies to radt_render_bwd only");
    WsLayout w = ws_layout(geom, grid, batch, pass);
    if (ws_bytes < w.total) return fail(RADT_E_WORKSPACE, "workspace too small: need %zu bytes, got %zu", w.total, ws_bytes);
    if (((uintptr_t)ws & 15) != 0) return fail(RADT_E_INVALID, "workspace must be 16-byte aligned");
    long long stride = batch > 1 ? grid->batch_stride : grid_cells(grid);
    if (batch > 1 && stride < grid_cells(grid)) return fail(RADT_E_INVALID, "batch_stride smaller than the grid");

    g_launches = 0;
    static thread_local MarchParams MP;
    static thread_local SetupParams SP;
    static thread_local LevelTable LT;
    static thread_local ChanTable CT;
    memset(&LT, 0, sizeof(LT));
    memset(&CT, 0, sizeof(CT));
    for (int l = 0; l < line->nlev; ++l) { LT.e[l] = line->e_lev_K[l]; LT.g[l] = line->g_lev[l]; }
    for (int c = 0; c < line->nchan; ++c) CT.v[c] = line->vchan[c];

    DevGrid dg;
    make_dev_grid(grid, dg);
    DevWs dws = make_dev_ws(ws, w);
    DevLine dl_probe;
    make_dev_line(line, dl_probe);
    // window kernels: uniform channel lattice, and cells no finer than the fp32 positions of the prefilter resolve
    const bool use_win = opt.win_path && dl_probe.uniform && prefilter_safe(grid);
    const bool comp = cube_lo != nullptr;

    // a forward and its adjoint must agree on what shapes the partial sums of the cube
    const unsigned long long ctag = cube_tag(opt, use_win, comp, line);
    const unsigned long long stag = setup_tag(opt, use_win, geom, line, grid, batch);
    bool reuse = false;
    if (g_internal_pass) {
        reuse = pass == RADT_PASS_BWD && opt.reuse_setup;      // the HOST entry point ran the matching forward in this very call
    } else if (pass == RADT_PASS_FWD) {
        g_cubes.put(cube, ctag);
        g_workspaces.put(ws, stag);
    } else {
        unsigned long long seen = 0;
        if (g_cubes.get(cube, seen) && seen != 0 && seen != ctag)      // (tag 0: a cube of unknown origin)
            return fail(RADT_E_INVALID, "this cube was rendered with other options (window / skip_empty / win_path / cube_lo) "
                                        "than radt_render_bwd was given: the adjoint re-marches with the forward's arithmetic "
                                        "(radt_forget(cube) if the buffer now holds a cube of another origin)");
        if (opt.reuse_setup) {
            if (!g_workspaces.get(ws, seen) || seen != stag)
                return fail(RADT_E_INVALID, "reuse_setup: this workspace was not last set up by a forward with the same "
                                            "geom, line, grid and options");
            reuse = true;
        } else {
            g_workspaces.put(ws, 0);          // the adjoint's own setup replaces the forward's (no occupancy words for LINEAR grids)
        }
    }

    // counters: 0-3 work counters, 4 forward in-window samples, 7 the grid's maximum temperature (setup), 8.. loss slots
    // (forward); an adjoint that reuses the forward's setup keeps 4.. (the forward's figures stay readable)
    if (band.first) {
        CUDA_TRY(cudaMemsetAsync(dws.counters, 0, reuse ? 4 * sizeof(unsigned long long) : w.zero_bytes, st));
        if (reuse) CUDA_TRY(cudaMemsetAsync(dws.grad, 0, (size_t)grid_cells(grid) * (size_t)batch * sizeof(float4), st));
    }
    for (int b0 = 0; b0 < batch; b0 += RADT_MAXB) {
        int nb = batch - b0 < RADT_MAXB ? batch - b0 : RADT_MAXB;
        memset(&SP, 0, sizeof(SP));
        for (int b = 0; b < nb; ++b) {
            make_dev_geom(geom[b0 + b], line, SP.geom[b]);
            SP.geom[b].v0 = line->vchan[0] - geom[b0 + b].vsys;
            SP.vsys[b] = geom[b0 + b].vsys;
        }
        SP.grid = dg; SP.ws = dws;
        SP.nx = geom[0].nx; SP.ny = geom[0].ny; SP.nstep = geom[0].nstep; SP.nbatch = nb; SP.b0 = b0;
        SP.nlev = line->nlev; SP.nchan = line->nchan;
        SP.do_rays = 1; SP.do_tables = 1; SP.do_pack = 1; SP.do_zero_grad = (pass == RADT_PASS_BWD);
        SP.batch_stride = stride;
        // Occupancy words for the window kernels' prefilter.  The forward always builds them (an adjoint with
        // reuse_setup may want them); with LINEAR densities the exact adjoint needs every in-grid step (dL/dn of
        // empty cells) and marches without them.
        const bool win = use_win;
        const bool occ_fwd = win && opt.skip_empty;
        const bool occ = occ_fwd && (pass == RADT_PASS_FWD || grid->dens_mode == RADT_DENS_LN || !opt.zero_dens_grad);
        SP.do_occ = occ; SP.occ_words = w.occ_words; SP.occ_wpr = w.occ_wpr; SP.occ_nbj = w.occ_nbj; SP.flag_wpr = w.flag_wpr;
        SP.occ_thr = grid->dens_mode == RADT_DENS_LN ? -39.1439f : 1e-17f;     // N_EMPTY of the march kernels
        SP.dens = grid->dens; SP.temp = grid->temp; SP.vel = grid->vel;
        if (!reuse && band.first) {
            CUDA_TRY(radt_launch_setup(SP, LT, CT, st));
            ++g_launches;
            if (occ && grid->kind == RADT_GRID_SPH3D) {      // the (r, theta) occupancy words need every node flag: own launch
                CUDA_TRY(radt_launch_occ_sph(SP, st));
                ++g_launches;
            }
        }

        memset(&MP, 0, sizeof(MP));
        memcpy(MP.geom, SP.geom, sizeof(MP.geom));
        MP.grid = dg; MP.ws = dws;
        make_dev_line(line, MP.line);
        MP.nx = SP.nx; MP.ny = SP.ny; MP.nstep = SP.nstep;
        MP.tiles_x = (MP.nx + RADT_TILE_X - 1) / RADT_TILE_X;
        MP.tiles_y = (MP.ny + RADT_TILE_Y - 1) / RADT_TILE_Y;
        MP.tile_y0 = band.nty ? band.ty0 : 0; MP.launch_ty = band.nty ? band.nty : MP.tiles_y; MP.banded = band.nty ? 1 : 0;
        if (MP.tile_y0 < 0 || MP.tile_y0 + MP.launch_ty > MP.tiles_y) return fail(RADT_E_INVALID, "row band outside the image");
        MP.b0 = b0;
        MP.opt_window = opt.window; MP.opt_skip_empty = opt.skip_empty;
        MP.opt_zero_grad = opt.zero_dens_grad || !opt.skip_empty;
        MP.chan_lo = 0;
        for (int b = 0; b < nb && !MP.chan_lo; ++b)
            for (int c = 0; c < line->nchan; ++c) {
                double vv = line->vchan[c] - geom[b0 + b].vsys;
                if ((double)(float)vv != vv) { MP.chan_lo = 1; break; }
            }
        MP.cube = cube; MP.cube_lo = cube_lo; MP.dl_dcube = dl_dcube;
        if (pass == RADT_PASS_FWD && loss.target) {
            const double nvox = loss.nvox_total > 0 ? loss.nvox_total : (double)batch * geom[0].nx * geom[0].ny * line->nchan;
            const double inv = 1.0 / (loss.sigma * loss.sigma * nvox);
            MP.target = loss.target; MP.dl_out = loss.dl_out;
            MP.inv_s2n = (float)inv;
        }
        MP.use_win = win; MP.use_occ = occ; MP.occ_words = w.occ_words; MP.occ_wpr = w.occ_wpr; MP.occ_nbj = w.occ_nbj;
        if (pass == RADT_PASS_FWD && win) CUDA_TRY(radt_launch_march_fwd_win(MP, nb, st));
        else if (pass == RADT_PASS_FWD) CUDA_TRY(radt_launch_march_fwd(MP, nb, st));
        else if (win) CUDA_TRY(radt_launch_march_bwd_win(MP, nb, st));
        else CUDA_TRY(radt_launch_march_bwd(MP, nb, st));
        ++g_launches;
    }
    if (pass == RADT_PASS_FWD && loss.target && band.last) {
        const double nvox = loss.nvox_total > 0 ? loss.nvox_total : (double)batch * geom[0].nx * geom[0].ny * line->nchan;
        CUDA_TRY(radt_launch_loss_finish(reinterpret_cast<double *>(dws.counters + 8),
                                         0.5 / (loss.sigma * loss.sigma * nvox), loss.loss, st));
        ++g_launches;
    }
    if (pass == RADT_PASS_BWD && (g_dens || g_temp || g_vel) && band.last) {
        CUDA_TRY(radt_launch_unpack(dws.grad, dg.cells, batch, stride, g_dens, g_temp, g_vel, st));
        ++g_launches;
    }
    return RADT_OK;
}

}  // namespace

extern "C" {

int radt_version(void) { return RADT_VERSION; }
const char *radt_last_error(void) { return g_err; }
int radt_last_launch_count(void) { return g_launches; }

int radt_debug_host_split(int32_t chunk_items, int32_t band_rows)
{
    if (chunk_items < 0 || band_rows < 0) return fail(RADT_E_INVALID, "sizes must be >= 0 (0 = library policy)");
    g_force_chunk_items = chunk_items;
    g_force_band_rows = band_rows;
    return RADT_OK;
}

int radt_forget(const void *device_ptr)
{
    if (!device_ptr) return fail(RADT_E_INVALID, "null pointer");
    g_cubes.forget(device_ptr);
    g_workspaces.forget(device_ptr);
    return RADT_OK;
}

void radt_options_default(radt_options *opt)
{
    if (!opt) return;
    opt->struct_size = sizeof(radt_options);
    opt->window = 1; opt->skip_empty = 1; opt->win_path = 1; opt->zero_dens_grad = 1; opt->reuse_setup = 0;
}

int radt_workspace_bytes(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                         int32_t pass, size_t *bytes_out)
{
    if (!bytes_out) return fail(RADT_E_INVALID, "null bytes_out");
    int rc = validate(geom, line, grid, batch);
    if (rc) return rc;
    if (pass != RADT_PASS_FWD && pass != RADT_PASS_BWD) return fail(RADT_E_INVALID, "unknown pass");
    *bytes_out = ws_layout(geom, grid, batch, pass).total;
    return RADT_OK;
}

int radt_grad_layout(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     size_t *offset_out, size_t *nfloat_out)
{
    if (!offset_out || !nfloat_out) return fail(RADT_E_INVALID, "null output pointer");
    int rc = validate(geom, line, grid, batch);
    if (rc) return rc;
    WsLayout w = ws_layout(geom, grid, batch, RADT_PASS_BWD);
    *offset_out = w.grad;
    *nfloat_out = (size_t)grid_cells(grid) * (size_t)batch * 4;
    return RADT_OK;
}

int radt_unpack_grad(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch, const void *ws,
                     size_t ws_bytes, float *g_dens, float *g_temp, float *g_vel, void *cuda_stream)
{
    int rc = validate(geom, line, grid, batch);
    if (rc) return rc;
    if (!ws) return fail(RADT_E_INVALID, "null workspace");
    WsLayout w = ws_layout(geom, grid, batch, RADT_PASS_BWD);
    if (ws_bytes < w.total) return fail(RADT_E_WORKSPACE, "workspace too small: need %zu bytes, got %zu", w.total, ws_bytes);
    long long stride = batch > 1 ? grid->batch_stride : grid_cells(grid);
    g_launches = 0;
    if (g_dens || g_temp || g_vel) {
        CUDA_TRY(radt_launch_unpack((const float4 *)((const char *)ws + w.grad), grid_cells(grid), batch, stride, g_dens, g_temp,
                                    g_vel, (cudaStream_t)cuda_stream));
        g_launches = 1;
    }
    return RADT_OK;
}

int radt_ray_geometry(const radt_geom *geom, const radt_grid *grid, int32_t batch, double *rays_out, void *cuda_stream)
{
    int rc = validate(geom, nullptr, grid, batch);
    if (rc) return rc;
    if (!rays_out) return fail(RADT_E_INVALID, "null rays_out");
    static thread_local SetupParams SP;
    static thread_local LevelTable LT;
    static thread_local ChanTable CT;
    DevGrid dg;
    make_dev_grid(grid, dg);
    g_launches = 0;
    for (int b0 = 0; b0 < batch; b0 += RADT_MAXB) {
        int nb = batch - b0 < RADT_MAXB ? batch - b0 : RADT_MAXB;
        memset(&SP, 0, sizeof(SP));
        for (int b = 0; b < nb; ++b) make_dev_geom(geom[b0 + b], nullptr, SP.geom[b]);
        SP.grid = dg;
        SP.rays_user = (double2 *)rays_out;
        SP.nx = geom[0].nx; SP.ny = geom[0].ny; SP.nstep = geom[0].nstep; SP.nbatch = nb; SP.b0 = b0;
        SP.do_rays = 1;
        CUDA_TRY(radt_launch_setup(SP, LT, CT, (cudaStream_t)cuda_stream));
        ++g_launches;
    }
    return RADT_OK;
}

int radt_render(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch, const radt_options *opt,
                float *cube, float *cube_lo, void *ws, size_t ws_bytes, void *cuda_stream)
{
    return run_pass(geom, line, grid, batch, opt, RADT_PASS_FWD, cube, cube_lo, nullptr, nullptr, nullptr, nullptr, ws,
                    ws_bytes, (cudaStream_t)cuda_stream);
}

int radt_render_loss(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     const radt_options *opt, const float *target, double sigma, float *cube, float *cube_lo,
                     float *dl_dcube, double *loss_out, void *ws, size_t ws_bytes, void *cuda_stream)
{
    if (!target || !dl_dcube || !loss_out) return fail(RADT_E_INVALID, "null target / dl_dcube / loss_out pointer");
    if (!(sigma > 0)) return fail(RADT_E_INVALID, "sigma must be positive");
    LossArgs la;
    la.target = target; la.dl_out = dl_dcube; la.loss = loss_out; la.sigma = sigma;
    return run_pass(geom, line, grid, batch, opt, RADT_PASS_FWD, cube, cube_lo, nullptr, nullptr, nullptr, nullptr, ws,
                    ws_bytes, (cudaStream_t)cuda_stream, la);
}

int radt_render_bwd(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                    const radt_options *opt, const float *cube, const float *cube_lo, const float *dl_dcube, float *g_dens,
                    float *g_temp, float *g_vel, void *ws, size_t ws_bytes, void *cuda_stream)
{
    return run_pass(geom, line, grid, batch, opt, RADT_PASS_BWD, const_cast<float *>(cube), const_cast<float *>(cube_lo),
                    dl_dcube, g_dens, g_temp, g_vel, ws, ws_bytes, (cudaStream_t)cuda_stream);
}

int radt_l2_loss_grad(const float *cube, const float *target, double sigma, int64_t n, float *dl_dcube,
                      double *loss_out, void *cuda_stream)
{
    if (!cube || !target || !dl_dcube || !loss_out) return fail(RADT_E_INVALID, "null pointer");
    if (n < 1 || !(sigma > 0)) return fail(RADT_E_INVALID, "need n >= 1 and sigma > 0");
    CUDA_TRY(radt_launch_l2(cube, target, sigma, n, dl_dcube, loss_out, (cudaStream_t)cuda_stream));
    g_launches = 1;
    return RADT_OK;
}

int radt_read_counters(const void *ws, uint64_t *out4, void *cuda_stream)
{
    if (!ws || !out4) return fail(RADT_E_INVALID, "null pointer");
    CUDA_TRY(cudaMemcpyAsync(out4, ws, 4 * sizeof(uint64_t), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    return RADT_OK;
}

int radt_read_lane_counters(const void *ws, uint64_t *out2, void *cuda_stream)
{
    if (!ws || !out2) return fail(RADT_E_INVALID, "null pointer");
    uint64_t c[5];
    CUDA_TRY(cudaMemcpyAsync(c, ws, 5 * sizeof(uint64_t), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    out2[0] = c[RADT_CNT_USEFUL];
    out2[1] = 32 * c[1] / 2;          // 2 MUFU.EX2 lane-operations per executed sample
    return RADT_OK;
}

// ------------------------------------------------------------------------------------------
// HOST-buffer entry points: stream-ordered allocation, H2D, same kernels, D2H, synchronise.
// ------------------------------------------------------------------------------------------
namespace {
// Device memory of the HOST-buffer entry points: one arena per thread and device, grown when a call needs more and kept
// between calls (a fit loop calls with the same sizes; per-call cudaMallocAsync / cudaFreeAsync of nine buffers made the
// call time vary by 0.7 ms from process to process).  Every call ends with a stream synchronisation, so the arena
// is idle when the next call starts.
struct DevArena {
    char *base = nullptr;
    size_t cap = 0;
    int dev = -1;
};
thread_local DevArena g_arena;

struct DevBufs {
    cudaStream_t st = 0;
    size_t used = 0;
    bool reserve(size_t bytes)
    {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return false;
        if (g_arena.dev == dev && g_arena.cap >= bytes) return true;
        if (g_arena.base) {
            cudaSetDevice(g_arena.dev);
            cudaFree(g_arena.base);
            cudaSetDevice(dev);
        }
        g_arena = DevArena();
        void *p = nullptr;
        if (cudaMalloc(&p, bytes) != cudaSuccess) return false;
        g_arena.base = (char *)p; g_arena.cap = bytes; g_arena.dev = dev;
        return true;
    }
    void *alloc(size_t bytes)
    {
        const size_t a = align256(bytes ? bytes : 16);
        if (used + a > g_arena.cap) return nullptr;
        void *p = g_arena.base + used;
        used += a;
        return p;
    }
};
}  // namespace

static int host_common_impl(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                            const radt_options *opt, int mode, const float *target, double sigma, float *cube, float *cube_lo,
                            const float *cube_in, const float *lo_in, const float *dl_in, double *loss_out, float *g_dens,
                            float *g_temp, float *g_vel);

static int host_common(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                       const radt_options *opt, int mode, const float *target, double sigma, float *cube, float *cube_lo,
                       const float *cube_in, const float *lo_in, const float *dl_in, double *loss_out, float *g_dens,
                       float *g_temp, float *g_vel)
{
    InternalPass guard;           // the arena's cubes and workspaces stay out of the shared forward/adjoint tables
    const int rc = host_common_impl(geom, line, grid, batch, opt, mode, target, sigma, cube, cube_lo, cube_in, lo_in, dl_in,
                                    loss_out, g_dens, g_temp, g_vel);
    // An error exit half-way through a chunk or band loop may leave copies into or out of the CALLER's host buffers in flight on
    // either stream: wait for them before handing the buffers back (error path only; the message of `rc` is kept).
    if (rc != RADT_OK) cudaDeviceSynchronize();
    return rc;
}

static int host_common_impl(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                            const radt_options *opt, int mode, const float *target, double sigma, float *cube, float *cube_lo,
                            const float *cube_in, const float *lo_in, const float *dl_in, double *loss_out, float *g_dens,
                            float *g_temp, float *g_vel)
{
    // mode 0: forward only; 1: forward + chi^2 term + adjoint; 2: adjoint from given cube and dl_dcube
    int rc = validate(geom, line, grid, batch);
    if (rc) return rc;
    Opts o;
    if ((rc = resolve_options(opt, o)) != 0) return rc;
    if (o.reuse_setup) return fail(RADT_E_INVALID, "reuse_setup is for the device entry points (the host calls manage their own workspace)");
    if (!line) return fail(RADT_E_INVALID, "null line descriptor");
    if (!grid->dens || !grid->temp || !grid->vel) return fail(RADT_E_INVALID, "null field pointer");
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) return fail(RADT_E_CUDA, "no CUDA device");
    DevBufs B;
    long long cells = grid_cells(grid);
    long long stride = batch > 1 ? grid->batch_stride : cells;
    size_t fbytes = (size_t)((batch - 1) * stride + cells) * sizeof(float);
    size_t nvox = (size_t)batch * geom[0].nx * geom[0].ny * line->nchan;
    static thread_local cudaStream_t s2 = nullptr;
    static thread_local cudaEvent_t ev_alloc = nullptr, ev_copied = nullptr;
    // an earlier call that failed half-way may still own the arena (main stream, or the target upload on s2)
    CUDA_TRY(cudaStreamSynchronize(B.st));
    if (s2) CUDA_TRY(cudaStreamSynchronize(s2));
    const size_t wsb_need = ws_layout(geom, grid, batch, mode == 0 ? RADT_PASS_FWD : RADT_PASS_BWD).total;
    if (!B.reserve(6 * align256(fbytes) + 4 * align256(nvox * sizeof(float)) + align256(wsb_need) + 4096))
        return fail(RADT_E_CUDA, "device allocation failed");
    float *d_dens = (float *)B.alloc(fbytes), *d_temp = (float *)B.alloc(fbytes), *d_vel = (float *)B.alloc(fbytes);
    float *d_cube = (float *)B.alloc(nvox * sizeof(float));
    // low-order words: kept on the device between the forward and the adjoint of a fit step; mode 0 / 2 only when the
    // caller has a host buffer for them
    const bool want_lo = mode == 1 || (mode == 0 && cube_lo) || (mode == 2 && lo_in);
    float *d_lo = want_lo ? (float *)B.alloc(nvox * sizeof(float)) : nullptr;
    if (!d_dens || !d_temp || !d_vel || !d_cube || (want_lo && !d_lo)) return fail(RADT_E_CUDA, "device allocation failed");
    CUDA_TRY(cudaMemcpyAsync(d_dens, grid->dens, fbytes, cudaMemcpyHostToDevice, B.st));
    CUDA_TRY(cudaMemcpyAsync(d_temp, grid->temp, fbytes, cudaMemcpyHostToDevice, B.st));
    CUDA_TRY(cudaMemcpyAsync(d_vel, grid->vel, fbytes, cudaMemcpyHostToDevice, B.st));
    radt_grid dgrid = *grid;
    dgrid.dens = d_dens; dgrid.temp = d_temp; dgrid.vel = d_vel;
    size_t wsb = wsb_need;
    void *ws = B.alloc(wsb);
    if (!ws) return fail(RADT_E_CUDA, "device allocation failed");
    int launches = 0;
    float *d_dl = nullptr;
    if (mode != 0 && !(d_dl = (float *)B.alloc(nvox * sizeof(float)))) return fail(RADT_E_CUDA, "device allocation failed");
    radt_options ob;
    radt_options_default(&ob);
    if (opt) ob = *opt;
    // Batched calls (config 5: 16 items, 2.1 GB of target and of cube) run item chunk by item chunk so that PCIe and the SMs
    // work at the same time: fit step = the upload of chunk c + 1's target under the forward and adjoint of chunk c (and the
    // chi^2 term FUSED into each chunk's forward, which only waits for its own chunk's upload); render = the download of chunk
    // c's cube under the march of chunk c + 1.  Results are those of the one-call path (items are independent; the loss is the
    // sum of the chunks' shares).
    const size_t item_vox = (size_t)geom[0].nx * geom[0].ny * line->nchan;
    int chunk = batch;
    if (batch > 1 && mode != 2) {
        const size_t per = item_vox * sizeof(float);
        chunk = (int)(((size_t)32 << 20) / per);
        if (chunk < 1) chunk = 1;
        if (chunk > batch) chunk = batch;
        if ((batch + chunk - 1) / chunk > 256) chunk = (batch + 255) / 256;
        // test hook (radt_debug_host_split): chunks of n items (tests/test_gpu_parity.py runs the chunked path on small scenes)
        if (g_force_chunk_items >= 1) chunk = g_force_chunk_items < batch ? g_force_chunk_items : batch;
    }
    if (chunk < batch) {
        static thread_local std::vector<cudaEvent_t> evs;
        const int nchunks = (batch + chunk - 1) / chunk;
        if (!s2) {
            CUDA_TRY(cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
            CUDA_TRY(cudaEventCreateWithFlags(&ev_alloc, cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&ev_copied, cudaEventDisableTiming));
        }
        while ((int)evs.size() < nchunks) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            evs.push_back(e);
        }
        auto chunk_grid = [&](int b0) {
            radt_grid g = dgrid;
            g.dens = d_dens + (size_t)b0 * stride; g.temp = d_temp + (size_t)b0 * stride; g.vel = d_vel + (size_t)b0 * stride;
            return g;
        };
        CUDA_TRY(cudaEventRecord(ev_alloc, B.st));          // (the arena is ours from here on; the fields are on their way)
        CUDA_TRY(cudaStreamWaitEvent(s2, ev_alloc, 0));
        if (mode == 0) {
            for (int c = 0; c < nchunks; ++c) {
                const int b0 = c * chunk, nb = batch - b0 < chunk ? batch - b0 : chunk;
                const size_t off = (size_t)b0 * item_vox, nby = (size_t)nb * item_vox * sizeof(float);
                radt_grid g = chunk_grid(b0);
                rc = radt_render(geom + b0, line, &g, nb, opt, d_cube + off, d_lo ? d_lo + off : nullptr, ws, wsb, B.st);
                if (rc) { cudaStreamSynchronize(s2); return rc; }
                launches += g_launches;
                CUDA_TRY(cudaEventRecord(evs[c], B.st));
                CUDA_TRY(cudaStreamWaitEvent(s2, evs[c], 0));
                CUDA_TRY(cudaMemcpyAsync(cube + off, d_cube + off, nby, cudaMemcpyDeviceToHost, s2));
                if (cube_lo) CUDA_TRY(cudaMemcpyAsync(cube_lo + off, d_lo + off, nby, cudaMemcpyDeviceToHost, s2));
            }
            CUDA_TRY(cudaStreamSynchronize(B.st));
            CUDA_TRY(cudaStreamSynchronize(s2));
            g_launches = launches;
            return RADT_OK;
        }
        // mode 1
        if (!target) return fail(RADT_E_INVALID, "null target");
        float *d_t = (float *)B.alloc(nvox * sizeof(float));
        double *d_loss = (double *)B.alloc(sizeof(double) * (size_t)nchunks);
        float *d_g[3] = { nullptr, nullptr, nullptr };
        float *h_g[3] = { g_dens, g_temp, g_vel };
        for (int i = 0; i < 3; ++i)
            if (h_g[i] && !(d_g[i] = (float *)B.alloc(fbytes))) return fail(RADT_E_CUDA, "device allocation failed");
        if (!d_t || !d_loss) return fail(RADT_E_CUDA, "device allocation failed");
        for (int c = 0; c < nchunks; ++c) {
            const int b0 = c * chunk, nb = batch - b0 < chunk ? batch - b0 : chunk;
            const size_t off = (size_t)b0 * item_vox;
            CUDA_TRY(cudaMemcpyAsync(d_t + off, target + off, (size_t)nb * item_vox * sizeof(float), cudaMemcpyHostToDevice, s2));
            CUDA_TRY(cudaEventRecord(evs[c], s2));
        }
        ob.reuse_setup = 1;
        for (int c = 0; c < nchunks; ++c) {
            const int b0 = c * chunk, nb = batch - b0 < chunk ? batch - b0 : chunk;
            const size_t off = (size_t)b0 * item_vox;
            radt_grid g = chunk_grid(b0);
            CUDA_TRY(cudaStreamWaitEvent(B.st, evs[c], 0));
            LossArgs la;
            la.target = d_t + off; la.dl_out = d_dl + off; la.loss = d_loss + c; la.sigma = sigma; la.nvox_total = (double)nvox;
            rc = run_pass(geom + b0, line, &g, nb, opt, RADT_PASS_FWD, d_cube + off, d_lo + off, nullptr, nullptr, nullptr, nullptr,
                          ws, wsb, B.st, la);
            if (rc) { cudaStreamSynchronize(s2); return rc; }
            launches += g_launches;
            rc = radt_render_bwd(geom + b0, line, &g, nb, &ob, d_cube + off, d_lo + off, d_dl + off,
                                 d_g[0] ? d_g[0] + (size_t)b0 * stride : nullptr, d_g[1] ? d_g[1] + (size_t)b0 * stride : nullptr,
                                 d_g[2] ? d_g[2] + (size_t)b0 * stride : nullptr, ws, wsb, B.st);
            if (rc) { cudaStreamSynchronize(s2); return rc; }
            launches += g_launches;
        }
        std::vector<double> parts((size_t)nchunks, 0.0);
        if (loss_out) CUDA_TRY(cudaMemcpyAsync(parts.data(), d_loss, sizeof(double) * (size_t)nchunks, cudaMemcpyDeviceToHost, B.st));
        if (cube) CUDA_TRY(cudaMemcpyAsync(cube, d_cube, nvox * sizeof(float), cudaMemcpyDeviceToHost, B.st));
        for (int i = 0; i < 3; ++i)
            if (h_g[i]) CUDA_TRY(cudaMemcpyAsync(h_g[i], d_g[i], fbytes, cudaMemcpyDeviceToHost, B.st));
        CUDA_TRY(cudaStreamSynchronize(B.st));
        CUDA_TRY(cudaStreamSynchronize(s2));
        if (loss_out) {
            double acc = 0.0;
            for (double v : parts) acc += v;
            *loss_out = acc;
        }
        g_launches = launches;
        return RADT_OK;
    }
    // A single large image runs in ROW BANDS the same way: ONE setup, then per band of tile rows the forward march (chi^2 term
    // fused: it only needs its own rows of the target) and, in a fit step, the adjoint march of the same rows, which adds into
    // the shared gradient cells; the target rows of band r + 1 upload / the cube rows of band r download under those marches.
    if (batch == 1 && mode != 2) {
        const int nx = geom[0].nx, ny = geom[0].ny;
        const size_t row_vox = (size_t)nx * line->nchan;
        long long rows = (long long)(((size_t)16 << 20) / (row_vox * sizeof(float)));
        if (g_force_band_rows >= 1) rows = g_force_band_rows;      // test hook (radt_debug_host_split)
        rows = (rows + RADT_TILE_Y - 1) / RADT_TILE_Y * RADT_TILE_Y;
        if (rows < RADT_TILE_Y) rows = RADT_TILE_Y;
        if ((ny + rows - 1) / rows > 256) rows = ((ny + 255) / 256 + RADT_TILE_Y - 1) / RADT_TILE_Y * RADT_TILE_Y;
        int nbands = (int)((ny + rows - 1) / rows);
        // Fit steps on 3-D grids stay in one piece: their forward march is longer than the target upload, which the plain path
        // already hides under it, and bands only add launch tails (measured on config 4: 13.0 -> 13.4 ms with bands; on the
        // axisymmetric config 3 the upload is three times the forward: 4.99 -> 3.95 ms).  The test hook overrides.
        if (mode == 1 && grid->kind != RADT_GRID_AXISYM && g_force_band_rows < 1) nbands = 1;
        if (nbands > 1) {
            static thread_local std::vector<cudaEvent_t> evs;
            if (!s2) {
                CUDA_TRY(cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
                CUDA_TRY(cudaEventCreateWithFlags(&ev_alloc, cudaEventDisableTiming));
                CUDA_TRY(cudaEventCreateWithFlags(&ev_copied, cudaEventDisableTiming));
            }
            while ((int)evs.size() < nbands) {
                cudaEvent_t e;
                CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                evs.push_back(e);
            }
            auto band_of = [&](int k) {
                Band bd;
                const long long r0 = (long long)k * rows, r1 = r0 + rows < ny ? r0 + rows : ny;
                bd.ty0 = (int)(r0 / RADT_TILE_Y); bd.nty = (int)((r1 - r0 + RADT_TILE_Y - 1) / RADT_TILE_Y);
                bd.first = k == 0; bd.last = k == nbands - 1;
                return bd;
            };
            CUDA_TRY(cudaEventRecord(ev_alloc, B.st));
            CUDA_TRY(cudaStreamWaitEvent(s2, ev_alloc, 0));
            if (mode == 0) {
                for (int k = 0; k < nbands; ++k) {
                    const long long r0 = (long long)k * rows, r1 = r0 + rows < ny ? r0 + rows : ny;
                    const size_t off = (size_t)r0 * row_vox, nby = (size_t)(r1 - r0) * row_vox * sizeof(float);
                    rc = run_pass(geom, line, &dgrid, 1, opt, RADT_PASS_FWD, d_cube, d_lo, nullptr, nullptr, nullptr, nullptr, ws, wsb,
                                  B.st, LossArgs(), band_of(k));
                    if (rc) { cudaStreamSynchronize(s2); return rc; }
                    launches += g_launches;
                    CUDA_TRY(cudaEventRecord(evs[k], B.st));
                    CUDA_TRY(cudaStreamWaitEvent(s2, evs[k], 0));
                    CUDA_TRY(cudaMemcpyAsync(cube + off, d_cube + off, nby, cudaMemcpyDeviceToHost, s2));
                    if (cube_lo) CUDA_TRY(cudaMemcpyAsync(cube_lo + off, d_lo + off, nby, cudaMemcpyDeviceToHost, s2));
                }
                CUDA_TRY(cudaStreamSynchronize(B.st));
                CUDA_TRY(cudaStreamSynchronize(s2));
                g_launches = launches;
                return RADT_OK;
            }
            if (!target) return fail(RADT_E_INVALID, "null target");
            float *d_t = (float *)B.alloc(nvox * sizeof(float));
            double *d_loss = (double *)B.alloc(sizeof(double));
            float *d_g[3] = { nullptr, nullptr, nullptr };
            float *h_g[3] = { g_dens, g_temp, g_vel };
            for (int i = 0; i < 3; ++i)
                if (h_g[i] && !(d_g[i] = (float *)B.alloc(fbytes))) return fail(RADT_E_CUDA, "device allocation failed");
            if (!d_t || !d_loss) return fail(RADT_E_CUDA, "device allocation failed");
            for (int k = 0; k < nbands; ++k) {
                const long long r0 = (long long)k * rows, r1 = r0 + rows < ny ? r0 + rows : ny;
                const size_t off = (size_t)r0 * row_vox;
                CUDA_TRY(cudaMemcpyAsync(d_t + off, target + off, (size_t)(r1 - r0) * row_vox * sizeof(float), cudaMemcpyHostToDevice, s2));
                CUDA_TRY(cudaEventRecord(evs[k], s2));
            }
            ob.reuse_setup = 1;
            LossArgs la;
            la.target = d_t; la.dl_out = d_dl; la.loss = d_loss; la.sigma = sigma;
            for (int k = 0; k < nbands; ++k) {
                const Band bd = band_of(k);
                CUDA_TRY(cudaStreamWaitEvent(B.st, evs[k], 0));
                rc = run_pass(geom, line, &dgrid, 1, opt, RADT_PASS_FWD, d_cube, d_lo, nullptr, nullptr, nullptr, nullptr, ws, wsb, B.st,
                              la, bd);
                if (rc) { cudaStreamSynchronize(s2); return rc; }
                launches += g_launches;
                rc = run_pass(geom, line, &dgrid, 1, &ob, RADT_PASS_BWD, d_cube, d_lo, d_dl, d_g[0], d_g[1], d_g[2], ws, wsb, B.st,
                              LossArgs(), bd);
                if (rc) { cudaStreamSynchronize(s2); return rc; }
                launches += g_launches;
            }
            if (loss_out) CUDA_TRY(cudaMemcpyAsync(loss_out, d_loss, sizeof(double), cudaMemcpyDeviceToHost, B.st));
            if (cube) CUDA_TRY(cudaMemcpyAsync(cube, d_cube, nvox * sizeof(float), cudaMemcpyDeviceToHost, B.st));
            for (int i = 0; i < 3; ++i)
                if (h_g[i]) CUDA_TRY(cudaMemcpyAsync(h_g[i], d_g[i], fbytes, cudaMemcpyDeviceToHost, B.st));
            CUDA_TRY(cudaStreamSynchronize(B.st));
            CUDA_TRY(cudaStreamSynchronize(s2));
            g_launches = launches;
            return RADT_OK;
        }
    }
    if (mode == 0) {
        rc = radt_render(geom, line, &dgrid, batch, opt, d_cube, d_lo, ws, wsb, B.st);
        if (rc) return rc;
        launches += g_launches;
    } else if (mode == 1) {
        // The target cube is the bulk of the input bytes (97 % on config 2) and PCIe is the long pole of this call: its
        // upload runs on a second stream UNDER the setup and the forward march, and the chi^2 term follows as its own
        // small pass (the fused radt_render_loss would have to wait for the whole upload before its first ray:
        // measured 0.15 ms slower per step on config 2, 17 ms on config 5).
        if (!target) return fail(RADT_E_INVALID, "null target");
        if (!s2) {
            CUDA_TRY(cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking));
            CUDA_TRY(cudaEventCreateWithFlags(&ev_alloc, cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&ev_copied, cudaEventDisableTiming));
        }
        float *d_t = (float *)B.alloc(nvox * sizeof(float));
        double *d_loss = (double *)B.alloc(sizeof(double));
        if (!d_t || !d_loss) return fail(RADT_E_CUDA, "device allocation failed");
        CUDA_TRY(cudaEventRecord(ev_alloc, B.st));
        CUDA_TRY(cudaStreamWaitEvent(s2, ev_alloc, 0));
        CUDA_TRY(cudaMemcpyAsync(d_t, target, nvox * sizeof(float), cudaMemcpyHostToDevice, s2));
        CUDA_TRY(cudaEventRecord(ev_copied, s2));
        rc = radt_render(geom, line, &dgrid, batch, opt, d_cube, d_lo, ws, wsb, B.st);
        if (rc) { cudaStreamSynchronize(s2); return rc; }
        launches += g_launches;
        CUDA_TRY(cudaStreamWaitEvent(B.st, ev_copied, 0));
        rc = radt_l2_loss_grad(d_cube, d_t, sigma, (int64_t)nvox, d_dl, d_loss, B.st);
        if (rc) { cudaStreamSynchronize(s2); return rc; }
        launches += g_launches;
        if (loss_out) CUDA_TRY(cudaMemcpyAsync(loss_out, d_loss, sizeof(double), cudaMemcpyDeviceToHost, B.st));
    }
    if ((mode == 0 || mode == 1) && cube)
        CUDA_TRY(cudaMemcpyAsync(cube, d_cube, nvox * sizeof(float), cudaMemcpyDeviceToHost, B.st));
    if (mode == 0 && cube_lo) CUDA_TRY(cudaMemcpyAsync(cube_lo, d_lo, nvox * sizeof(float), cudaMemcpyDeviceToHost, B.st));
    if (mode == 1 || mode == 2) {
        float *d_g[3] = { nullptr, nullptr, nullptr };
        float *h_g[3] = { g_dens, g_temp, g_vel };
        for (int i = 0; i < 3; ++i)
            if (h_g[i] && !(d_g[i] = (float *)B.alloc(fbytes))) return fail(RADT_E_CUDA, "device allocation failed");
        if (mode == 2) {
            if (!cube_in || !dl_in) return fail(RADT_E_INVALID, "null cube / dl_dcube");
            CUDA_TRY(cudaMemcpyAsync(d_cube, cube_in, nvox * sizeof(float), cudaMemcpyHostToDevice, B.st));
            if (lo_in) CUDA_TRY(cudaMemcpyAsync(d_lo, lo_in, nvox * sizeof(float), cudaMemcpyHostToDevice, B.st));
            CUDA_TRY(cudaMemcpyAsync(d_dl, dl_in, nvox * sizeof(float), cudaMemcpyHostToDevice, B.st));
        }
        ob.reuse_setup = mode == 1;          // the forward of this very call set the workspace up
        rc = radt_render_bwd(geom, line, &dgrid, batch, &ob, d_cube, d_lo, d_dl, d_g[0], d_g[1], d_g[2], ws, wsb, B.st);
        if (rc) return rc;
        launches += g_launches;
        for (int i = 0; i < 3; ++i)
            if (h_g[i]) CUDA_TRY(cudaMemcpyAsync(h_g[i], d_g[i], fbytes, cudaMemcpyDeviceToHost, B.st));
    }
    CUDA_TRY(cudaStreamSynchronize(B.st));
    g_launches = launches;
    return RADT_OK;
}

int radt_render_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                     const radt_options *opt, float *cube, float *cube_lo)
{
    if (!cube) return fail(RADT_E_INVALID, "null cube pointer");
    return host_common(geom, line, grid, batch, opt, 0, nullptr, 0.0, cube, cube_lo, nullptr, nullptr, nullptr, nullptr,
                       nullptr, nullptr, nullptr);
}

int radt_fit_step_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                       const radt_options *opt, const float *target, double sigma, float *cube, double *loss_out,
                       float *g_dens, float *g_temp, float *g_vel)
{
    if (!(sigma > 0)) return fail(RADT_E_INVALID, "sigma must be positive");
    return host_common(geom, line, grid, batch, opt, 1, target, sigma, cube, nullptr, nullptr, nullptr, nullptr, loss_out,
                       g_dens, g_temp, g_vel);
}

int radt_render_bwd_host(const radt_geom *geom, const radt_line *line, const radt_grid *grid, int32_t batch,
                         const radt_options *opt, const float *cube, const float *cube_lo, const float *dl_dcube,
                         float *g_dens, float *g_temp, float *g_vel)
{
    return host_common(geom, line, grid, batch, opt, 2, nullptr, 0.0, nullptr, nullptr, cube, cube_lo, dl_dcube, nullptr,
                       g_dens, g_temp, g_vel);
}

// ------------------------------------------------------------------------------------------
// physics pre-pass (radt_disk.cu)
// ------------------------------------------------------------------------------------------
static int disk_setup(const radt_disk *disk, const radt_grid *grid, int32_t batch, void *ws, size_t ws_bytes,
                      DiskParamsDev &Q, size_t *need_out)
{
    if (!grid) return fail(RADT_E_INVALID, "null grid descriptor");
    if (grid->struct_size != sizeof(radt_grid)) return fail(RADT_E_INVALID, "radt_grid.struct_size mismatch");
    if (batch < 1 || batch > RADT_MAXB) return fail(RADT_E_INVALID, "batch must be 1..%d", RADT_MAXB);
    if (grid->kind != RADT_GRID_AXISYM || !grid->mirror_z || grid->lo[1] != 0.0 || grid->dens_mode != RADT_DENS_LINEAR ||
        grid->vel_mode != RADT_VEL_VPHI)
        return fail(RADT_E_UNSUPPORTED, "the pre-pass needs a mirror-symmetric (r, zeta) grid from zeta = 0 with LINEAR density and VPHI velocity");
    if (grid->n[0] < 2 || grid->n[1] < 2 || !(grid->lo[0] > 0) || !(grid->hi[0] > grid->lo[0]) || !(grid->hi[1] > 0))
        return fail(RADT_E_INVALID, "bad grid extents");
    const size_t cells = (size_t)grid->n[0] * grid->n[1] * batch, cols = (size_t)grid->n[0] * batch;
    size_t off = 0, o_rt, o_rho, o_P, o_gP, o_grho, o_cs, o_cH, o_mask;
    o_rt = off; off = align256(off + cells * 8);
    o_rho = off; off = align256(off + cells * 8);
    o_P = off; off = align256(off + cells * 8);
    o_gP = off; off = align256(off + cells * 8);
    o_grho = off; off = align256(off + cells * 8);
    o_cs = off; off = align256(off + cols * 8);
    o_cH = off; off = align256(off + cols * 8);
    o_mask = off; off = align256(off + cells);
    if (need_out) { *need_out = off; return RADT_OK; }
    if (!disk) return fail(RADT_E_INVALID, "null disk descriptor");
    if (!ws) return fail(RADT_E_INVALID, "null workspace");
    if (ws_bytes < off) return fail(RADT_E_WORKSPACE, "workspace too small: need %zu bytes, got %zu", off, ws_bytes);
    if (((uintptr_t)ws & 15) != 0) return fail(RADT_E_INVALID, "workspace must be 16-byte aligned");
    memset(&Q, 0, sizeof(Q));
    for (int b = 0; b < batch; ++b) {
        const radt_disk &d = disk[b];
        if (d.struct_size != sizeof(radt_disk)) return fail(RADT_E_INVALID, "radt_disk.struct_size mismatch");
        if (!(d.gm_star > 0) || !(d.m_gas > 0) || !(d.sigma0 > 0) || !(d.r_c > 0))
            return fail(RADT_E_INVALID, "disk constants must be positive");
        Q.disk[b] = DiskDev{ d.gm_star, d.m_gas, d.sigma0, d.r_c, d.gamma, d.x_co, d.t_freeze, d.n_dissoc, d.f_col };
    }
    Q.nr = grid->n[0]; Q.nz = grid->n[1]; Q.nbatch = batch;
    Q.batch_stride = batch > 1 ? grid->batch_stride : (long long)grid->n[0] * grid->n[1];
    if (batch > 1 && Q.batch_stride < (long long)grid->n[0] * grid->n[1])
        return fail(RADT_E_INVALID, "batch_stride smaller than the grid");
    Q.rmin = grid->lo[0];
    Q.lg2_ratio = std::log2(grid->hi[0] / grid->lo[0]);
    Q.dlnr = std::log(grid->hi[0] / grid->lo[0]) / (double)(grid->n[0] - 1);
    Q.dzeta = grid->hi[1] / (double)(grid->n[1] - 1);
    char *base = (char *)ws;
    Q.rt = (double *)(base + o_rt); Q.rho = (double *)(base + o_rho); Q.P = (double *)(base + o_P);
    Q.gP = (double *)(base + o_gP); Q.grho = (double *)(base + o_grho);
    Q.colscale = (double *)(base + o_cs); Q.colH = (double *)(base + o_cH);
    Q.mask = (unsigned char *)(base + o_mask);
    return RADT_OK;
}

int radt_disk_workspace_bytes(const radt_grid *grid, int32_t batch, size_t *bytes_out)
{
    if (!bytes_out) return fail(RADT_E_INVALID, "null bytes_out");
    DiskParamsDev Q;
    return disk_setup(nullptr, grid, batch, nullptr, 0, Q, bytes_out);
}

int radt_disk_fields(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp, float *dens_out,
                     float *vel_out, void *ws, size_t ws_bytes, void *cuda_stream)
{
    if (!temp || !dens_out || !vel_out) return fail(RADT_E_INVALID, "null field pointer");
    static thread_local DiskParamsDev Q;
    int rc = disk_setup(disk, grid, batch, ws, ws_bytes, Q, nullptr);
    if (rc) return rc;
    Q.temp = temp; Q.dens_out = dens_out; Q.vel_out = vel_out;
    CUDA_TRY(radt_launch_disk_fwd(Q, (cudaStream_t)cuda_stream));
    g_launches = 2;
    return RADT_OK;
}

// The forward pre-pass for callers that cannot give it a workspace (include/radt.h).  Allocates nothing: the scratch is
// the fixed array inside radt_disk.cu, whose address radt_launch_disk_fwd_static looks up on the first call per device.
int radt_disk_fields_static(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp,
                            float *dens_out, float *vel_out, void *cuda_stream)
{
    if (!temp || !dens_out || !vel_out) return fail(RADT_E_INVALID, "null field pointer");
    static thread_local DiskParamsDev Q;
    size_t need = 0;
    int rc = disk_setup(nullptr, grid, batch, nullptr, 0, Q, &need);         // grid and batch checks only
    if (rc) return rc;
    const long long cells = (long long)grid->n[0] * grid->n[1] * batch;
    if (cells > RADT_DISK_STATIC_MAX_CELLS)
        return fail(RADT_E_INVALID, "radt_disk_fields_static: batch x nr x nzeta = %lld cells exceeds the fixed scratch of "
                    "%d cells; split the batch or use radt_disk_fields with a workspace", cells, RADT_DISK_STATIC_MAX_CELLS);
    // descriptor checks and the scalar members of Q; the placeholder workspace is never dereferenced and the launcher
    // replaces every scratch pointer derived from it
    rc = disk_setup(disk, grid, batch, (void *)(uintptr_t)256, need, Q, nullptr);
    if (rc) return rc;
    Q.rt = Q.rho = Q.P = Q.gP = Q.grho = Q.colscale = Q.colH = nullptr;
    Q.mask = nullptr;
    Q.temp = temp; Q.dens_out = dens_out; Q.vel_out = vel_out;
    CUDA_TRY(radt_launch_disk_fwd_static(Q, (cudaStream_t)cuda_stream));
    g_launches = 2;
    return RADT_OK;
}

int radt_disk_fields_bwd(const radt_disk *disk, const radt_grid *grid, int32_t batch, const float *temp,
                         const float *g_dens, const float *g_vel, float *g_temp, void *ws, size_t ws_bytes,
                         void *cuda_stream)
{
    if (!temp || !g_dens || !g_vel || !g_temp) return fail(RADT_E_INVALID, "null field pointer");
    static thread_local DiskParamsDev Q;
    int rc = disk_setup(disk, grid, batch, ws, ws_bytes, Q, nullptr);
    if (rc) return rc;
    Q.temp = temp; Q.g_dens = g_dens; Q.g_vel = g_vel; Q.g_temp = g_temp;
    CUDA_TRY(radt_launch_disk_bwd(Q, (cudaStream_t)cuda_stream));
    g_launches = 3;
    return RADT_OK;
}

// ------------------------------------------------------------------------------------------
// MLP temperature field (radt_mlp_tc.cu, radt_mlp_tc_bwd.cu)
// ------------------------------------------------------------------------------------------
static int mlp_check(const radt_mlp *mlp, const radt_grid *grid, long long *count)
{
    if (!mlp) return fail(RADT_E_INVALID, "null mlp descriptor");
    if (mlp->struct_size != sizeof(radt_mlp)) return fail(RADT_E_INVALID, "radt_mlp.struct_size mismatch");
    if (mlp->width != 64 || mlp->nhidden != 4) return fail(RADT_E_UNSUPPORTED, "this build supports width 64 and 4 hidden layers");
    if (mlp->L < 0 || mlp->L > 8) return fail(RADT_E_UNSUPPORTED, "encoding degree L must be 0..8");
    if (!(mlp->t_hi > mlp->t_lo)) return fail(RADT_E_INVALID, "need t_lo < t_hi");
    if (grid) {
        if (grid->struct_size != sizeof(radt_grid)) return fail(RADT_E_INVALID, "radt_grid.struct_size mismatch");
        if (grid->kind != RADT_GRID_AXISYM) return fail(RADT_E_UNSUPPORTED, "the MLP field lives on an axisymmetric grid");
        if (grid->n[0] < 2 || grid->n[1] < 2) return fail(RADT_E_INVALID, "grid needs >= 2 nodes per axis");
    }
    const long long D = 2 + 4 * mlp->L;
    if (count) *count = 64 * D + 64 + 3 * (64 * 64 + 64) + 64 + 1;
    return RADT_OK;
}

int radt_mlp_num_params(const radt_mlp *mlp, int64_t *count_out)
{
    if (!count_out) return fail(RADT_E_INVALID, "null count_out");
    long long c = 0;
    int rc = mlp_check(mlp, nullptr, &c);
    if (rc) return rc;
    *count_out = c;
    return RADT_OK;
}

static void mlp_fill(const radt_mlp *mlp, const radt_grid *grid, MlpParamsDev &Q)
{
    memset(&Q, 0, sizeof(Q));
    Q.nparams = 64 * (2 + 4 * mlp->L) + 64 + 3 * (64 * 64 + 64) + 64 + 1;
    Q.nr = grid->n[0]; Q.nz = grid->n[1]; Q.L = mlp->L;
    Q.t_lo = (float)mlp->t_lo; Q.t_hi = (float)mlp->t_hi;
}

int radt_mlp_temperature(const radt_mlp *mlp, const radt_grid *grid, const float *params, float *temp_out,
                         void *cuda_stream)
{
    if (!grid) return fail(RADT_E_INVALID, "null grid descriptor");
    int rc = mlp_check(mlp, grid, nullptr);
    if (rc) return rc;
    if (!params || !temp_out) return fail(RADT_E_INVALID, "null pointer");
    if (((uintptr_t)params & 15) != 0) return fail(RADT_E_INVALID, "params must be 16-byte aligned");
    MlpParamsDev Q;
    mlp_fill(mlp, grid, Q);
    Q.params = params; Q.temp_out = temp_out;
    CUDA_TRY(radt_launch_mlp_fwd(Q, (cudaStream_t)cuda_stream));
    g_launches = 1;
    return RADT_OK;
}

int radt_mlp_temperature_bwd(const radt_mlp *mlp, const radt_grid *grid, const float *params, const float *g_temp,
                             float *g_params, void *cuda_stream)
{
    if (!grid) return fail(RADT_E_INVALID, "null grid descriptor");
    long long count = 0;
    int rc = mlp_check(mlp, grid, &count);
    if (rc) return rc;
    if (!params || !g_temp || !g_params) return fail(RADT_E_INVALID, "null pointer");
    MlpParamsDev Q;
    mlp_fill(mlp, grid, Q);
    Q.params = params; Q.g_temp = g_temp; Q.g_params = g_params;
    CUDA_TRY(radt_launch_mlp_bwd(Q, (int)count, (cudaStream_t)cuda_stream));
    g_launches = 1;
    return RADT_OK;
}

int radt_pipe_peak(int32_t kind, double *ops_per_s_out, double *sm_clock_mhz_out)
{
    if (!ops_per_s_out) return fail(RADT_E_INVALID, "null output");
    if (kind < 0 || kind > 3) return fail(RADT_E_INVALID, "unknown pipe kind");
    double clk = 0.0;
    CUDA_TRY(radt_run_pipe_peak(kind, ops_per_s_out, &clk));
    if (sm_clock_mhz_out) *sm_clock_mhz_out = clk;
    return RADT_OK;
}

}  // extern "C"
