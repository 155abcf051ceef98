// radt_disk.cu -- physics pre-pass on the (r, zeta) grid: temperature grid -> CO density and v_phi
// fields of the render, and its adjoint w.r.t. the temperature.  PAPER.md:156-203 (Eq. 1-2, 6-9).
// Algorithm P1-P7 of DESIGN.md section 10: hydrostatic integration along z with the trapezoid rule, surface-density
// normalisation, column above every node, CO mask, pressure-corrected rotation.  fp64 throughout (32 k cells: the
// pass is latency bound, not throughput bound).  Shares nothing with oracle/.
#include "radt_dev.cuh"
#include "radt_kernels.h"
#include <mutex>

#define KB_CGS 1.380649e-16
#define AU_CM 1.495978707e13

__device__ __forceinline__ double disk_sigma(const DiskDev &D, double r_au)
{
    double x = r_au / D.r_c;
    return D.sigma0 * pow(x, -D.gamma) * exp(-pow(x, 2.0 - D.gamma));
}

// Warp-wide scans over the lanes' chunk totals (fp64)
__device__ __forceinline__ double warp_excl_scan_up(double v, int lane)        // sum of the lanes below
{
    double inc = v;
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, inc, m);
        if (lane >= m) inc += t;
    }
    return inc - v;
}
__device__ __forceinline__ double warp_excl_scan_down(double v, int lane)      // sum of the lanes above
{
    double inc = v;
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const double t = __shfl_down_sync(0xffffffffu, inc, m);
        if (lane + m < 32) inc += t;
    }
    return inc - v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    return v;
}

// One WARP per column (b, i); lane l owns the nodes [l C, (l+1) C), C = ceil(nz / 32): the expensive terms (sqrt, exp)
// of different nodes are independent, only the running sums of P2, P4 and P5 are scans (a thread per column was a chain
// of nz fp64 exp: 0.12 ms for 128 nodes).  Writes rt = rho~ (P3), rho (P4), P (P7) to the workspace, the column
// scale Sigma / 2H and H, and the CO density (FWD) or the mask (adjoint).
template <bool FWD>
__global__ void __launch_bounds__(128) k_disk_columns(const __grid_constant__ DiskParamsDev Q)
{
    const int col = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (col >= Q.nr * Q.nbatch) return;
    const int b = col / Q.nr, i = col - b * Q.nr;
    const DiskDev &D = Q.disk[b];
    const int nz = Q.nz, C = (nz + 31) >> 5, j0 = min(lane * C, nz), j1 = min(j0 + C, nz);
    const float *T = Q.temp + (long long)b * Q.batch_stride + (long long)i * nz;
    double *rt = Q.rt + (long long)col * nz, *rho = Q.rho + (long long)col * nz, *P = Q.P + (long long)col * nz;
    const double r_au = Q.rmin * exp2((double)i * Q.lg2_ratio / (double)(Q.nr - 1));
    const double r = r_au * AU_CM, dz = Q.dzeta * r, c = D.gm_star * D.m_gas / KB_CGS;
    const double T0 = (double)T[0];
    auto fgrav = [&](int j) {                                     // P1
        const double z = (double)j * dz, s = r * r + z * z;
        return z / ((double)T[j] * s * sqrt(s));
    };
    // P2: A_j, chunk-local running sum first (kept in rho[] as scratch), then the offset of the lanes below
    double f_prev = j0 > 0 && j0 < nz ? fgrav(j0 - 1) : 0.0, a = 0.0;
    for (int j = j0; j < j1; ++j) {
        const double f = fgrav(j);
        if (j > 0) a += 0.5 * (f_prev + f) * dz;
        rho[j] = a;
        f_prev = f;
    }
    const double a_off = warp_excl_scan_up(a, lane);
    // P3 and the integral of P4
    double first = 0.0, last = 0.0;
    for (int j = j0; j < j1; ++j) {
        const double v = T0 / (double)T[j] * exp(-c * (a_off + rho[j]));
        rt[j] = v;
        if (j == j0) first = v;
        last = v;
    }
    // the value just below / above the chunk (empty chunks sit at the top and pass nothing on)
    double below = __shfl_up_sync(0xffffffffu, last, 1), above = __shfl_down_sync(0xffffffffu, first, 1);
    double h = 0.0, prev = below;
    for (int j = j0; j < j1; ++j) {
        const double v = rt[j];
        if (j > 0) h += 0.5 * (prev + v) * dz;
        prev = v;
    }
    const double H = warp_sum(h);
    const double scale = disk_sigma(D, r_au) / (2.0 * H);
    if (lane == 0) { Q.colscale[col] = scale; Q.colH[col] = H; }
    // P5: column above every node: chunk-local from the chunk's top node down, plus everything in the lanes above
    double nloc = 0.0, next = above;
    for (int j = j1 - 1; j >= j0; --j) {
        const double v = rt[j];
        if (j < nz - 1) nloc += 0.5 * (v + next) * dz;
        next = v;
    }
    const double n_off = warp_excl_scan_down(nloc, lane);
    float *dens = FWD ? Q.dens_out + (long long)b * Q.batch_stride + (long long)i * nz : nullptr;
    const double nscale = scale / D.m_gas;
    double N = n_off;
    next = above;
    for (int j = j1 - 1; j >= j0; --j) {                         // P4-P7 (pressure)
        const double v = rt[j], Tj = (double)T[j], rj = v * scale;
        if (j < nz - 1) N += 0.5 * (v + next) * dz;
        next = v;
        rho[j] = rj;
        P[j] = rj * KB_CGS * Tj / D.m_gas;
        const bool co = Tj > D.t_freeze && D.f_col * (N * nscale) > D.n_dissoc;
        if (FWD) dens[j] = co ? (float)(D.x_co * rj / D.m_gas) : 0.0f;
        else Q.mask[(long long)col * nz + j] = co ? 1 : 0;
    }
}

// dP/dr at fixed z on the (ln r, zeta) grid: centred differences in index space, one-sided at the edges (P7)
__device__ __forceinline__ double disk_dPdr(const DiskParamsDev &Q, const double *P, int i, int j, double r)
{
    const int nz = Q.nz, im = i > 0 ? i - 1 : i, ip = i < Q.nr - 1 ? i + 1 : i, jm = j > 0 ? j - 1 : j, jp = j < nz - 1 ? j + 1 : j;
    const double d1 = (P[(long long)ip * nz + j] - P[(long long)im * nz + j]) / ((double)(ip - im) * Q.dlnr);
    const double d2 = (P[(long long)i * nz + jp] - P[(long long)i * nz + jm]) / ((double)(jp - jm) * Q.dzeta);
    return (d1 - (double)j * Q.dzeta * d2) / r;
}

// One thread per cell: v_phi (forward) or the transpose of P7 (adjoint).
template <bool FWD>
__global__ void __launch_bounds__(256) k_disk_velocity(const __grid_constant__ DiskParamsDev Q)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long per = (long long)Q.nr * Q.nz;
    if (q >= per * Q.nbatch) return;
    const int b = (int)(q / per), nz = Q.nz;
    const long long c = q - (long long)b * per;
    const int i = (int)(c / nz), j = (int)(c - (long long)i * nz);
    const DiskDev &D = Q.disk[b];
    const double *P = Q.P + (long long)b * per;
    const double r = Q.rmin * exp2((double)i * Q.lg2_ratio / (double)(Q.nr - 1)) * AU_CM, z = (double)j * Q.dzeta * r;
    const double s = r * r + z * z, kep = D.gm_star * r * r / (s * sqrt(s));
    const double rh = Q.rho[q];
    const double dPdr = disk_dPdr(Q, P, i, j, r);
    const double v2 = kep + (rh > 0.0 ? r / rh * dPdr : 0.0);
    const long long ext = (long long)b * Q.batch_stride + c;
    if (FWD) {
        Q.vel_out[ext] = (float)sqrt(fmax(v2, 0.0));
        return;
    }
    double g_rho = 0.0;
    if (v2 > 0.0 && rh > 0.0) {
        const double g_v2 = (double)Q.g_vel[ext] / (2.0 * sqrt(v2));
        const double g_dPdr = g_v2 * r / rh, gr = g_dPdr / r;
        g_rho = -g_v2 * r * dPdr / (rh * rh);
        // transpose of the two difference stencils
        double *gP = Q.gP + (long long)b * per;
        const int im = i > 0 ? i - 1 : i, ip = i < Q.nr - 1 ? i + 1 : i, jm = j > 0 ? j - 1 : j, jp = j < nz - 1 ? j + 1 : j;
        const double a1 = gr / ((double)(ip - im) * Q.dlnr);
        const double a2 = -(double)j * Q.dzeta * gr / ((double)(jp - jm) * Q.dzeta);
        atomicAdd(gP + (long long)ip * nz + j, a1);
        atomicAdd(gP + (long long)im * nz + j, -a1);
        atomicAdd(gP + (long long)i * nz + jp, a2);
        atomicAdd(gP + (long long)i * nz + jm, -a2);
    }
    Q.grho[q] = g_rho;
}

// Adjoint of the column part (reverse of P6..P1), one warp per column, lanes over chunks of nodes as above.  Uses
// rt, rho, mask, the column scale and H recomputed by k_disk_columns<false>, grho (P7's direct term) and gP from
// k_disk_velocity<false>.  ADDS dL/dT of the pre-pass to g_temp.
__global__ void __launch_bounds__(128) k_disk_columns_bwd(const __grid_constant__ DiskParamsDev Q)
{
    const int col = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (col >= Q.nr * Q.nbatch) return;
    const int b = col / Q.nr, i = col - b * Q.nr;
    const DiskDev &D = Q.disk[b];
    const int nz = Q.nz, C = (nz + 31) >> 5, j0 = min(lane * C, nz), j1 = min(j0 + C, nz);
    const long long ext0 = (long long)b * Q.batch_stride + (long long)i * nz;
    const float *T = Q.temp + ext0;
    const float *g_nco = Q.g_dens + ext0;
    float *gT = Q.g_temp + ext0;
    const double *rt = Q.rt + (long long)col * nz, *rho = Q.rho + (long long)col * nz, *gP = Q.gP + (long long)col * nz;
    double *grho = Q.grho + (long long)col * nz;
    const unsigned char *mask = Q.mask + (long long)col * nz;
    const double r = Q.rmin * exp2((double)i * Q.lg2_ratio / (double)(Q.nr - 1)) * AU_CM;
    const double dz = Q.dzeta * r, c = D.gm_star * D.m_gas / KB_CGS;
    const double scale = Q.colscale[col], H = Q.colH[col];
    // total dL/drho per node (P7's pressure, P6/P5's CO density) and dL/dH of the normalisation (P4)
    double acc = 0.0;
    for (int j = j0; j < j1; ++j) {
        double g = grho[j] + gP[j] * KB_CGS * (double)T[j] / D.m_gas;
        if (mask[j]) g += D.x_co * (double)g_nco[j] / D.m_gas;
        grho[j] = g;
        acc += g * rho[j];
    }
    const double gH = -warp_sum(acc) / H, T0 = (double)T[0];
    // t_j = dL/drt_j rt_j; gA accumulates from the top node down (P2): chunk-local sum plus the lanes above
    double tsum = 0.0, asum = 0.0;
    for (int j = j0; j < j1; ++j) {
        const double w = (j == 0 || j == nz - 1) ? 0.5 * dz : dz;
        const double t = (grho[j] * scale + gH * w) * rt[j];
        grho[j] = t;                                              // keep t_j
        tsum += t;
        if (j >= 1) asum += -c * t;
    }
    const double sumt = warp_sum(tsum);
    const double a_above = warp_excl_scan_down(asum, lane);
    // gAcum of the first node of the chunk above (= a_above when that node exists and is >= 1)
    double gAcum = a_above, half_above = (j1 < nz) ? 0.5 * dz * a_above : 0.0;
    for (int j = j1 - 1; j >= j0; --j) {
        const double Tj = (double)T[j], t = grho[j];
        double gf = half_above;
        if (j >= 1) {
            gAcum += -c * t;
            half_above = 0.5 * dz * gAcum;
            gf += half_above;
        }
        const double z = (double)j * dz, s = r * r + z * z, f = z / (Tj * s * sqrt(s));
        double g = gP[j] * rho[j] * KB_CGS / D.m_gas - t / Tj - gf * f / Tj;
        if (j == 0) g += sumt / T0;
        gT[j] += (float)g;
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
cudaError_t radt_launch_disk_fwd(const DiskParamsDev &Q, cudaStream_t st)
{
    const int ncol = Q.nr * Q.nbatch;
    const long long ncell = (long long)ncol * Q.nz;
    k_disk_columns<true><<<(ncol + 3) / 4, 128, 0, st>>>(Q);
    k_disk_velocity<true><<<(int)((ncell + 255) / 256), 256, 0, st>>>(Q);
    return cudaGetLastError();
}

cudaError_t radt_launch_disk_bwd(const DiskParamsDev &Q, cudaStream_t st)
{
    const int ncol = Q.nr * Q.nbatch;
    const long long ncell = (long long)ncol * Q.nz;
    cudaError_t e = cudaMemsetAsync(Q.gP, 0, (size_t)ncell * sizeof(double), st);
    if (e != cudaSuccess) return e;
    k_disk_columns<false><<<(ncol + 3) / 4, 128, 0, st>>>(Q);
    k_disk_velocity<false><<<(int)((ncell + 255) / 256), 256, 0, st>>>(Q);
    k_disk_columns_bwd<<<(ncol + 3) / 4, 128, 0, st>>>(Q);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// radt_disk_fields_static: the forward pre-pass on scratch that lives inside the library image
// ---------------------------------------------------------------------------------------------
// Some programs that want the pre-pass have no way to hand it a workspace: every byte of device memory was given to
// another owner when the process started (a host application's memory pool, a fixed partition for a control loop that
// must not hit cudaMalloc's device-wide synchronisation or its unbounded latency), so a cudaMalloc made on their behalf
// either fails or is forbidden.  For them the scratch of the forward pre-pass (rt, rho, P per cell; column scale and H
// per column) is this file-scope array.  It is part of the loaded module: every GPU whose context loads libradt.so
// carries these 8 MiB (+ 1.25 KiB of alignment slack) until the process exits, whether or not the entry point is used,
// which is why the limit is kept modest: DISK_STATIC_MAX_CELLS = RADT_DISK_STATIC_MAX_CELLS (include/radt.h) cells per
// call, batch included.
//
// In host code the identifier g_disk_scratch is only the host-side shadow of the symbol, not a device address: a kernel
// handed `g_disk_scratch` by the host would fault, or on a system where the GPU can reach host memory it would quietly
// work on the wrong bytes.  The device address comes from cudaGetSymbolAddress, asked once per device with that device
// current (each device has its own copy of the array) and kept in g_disk_scratch_addr.
#define DISK_STATIC_MAX_CELLS 262144ll
#define DISK_STATIC_BYTES (3 * DISK_STATIC_MAX_CELLS * 8 + 2 * (DISK_STATIC_MAX_CELLS / 2) * 8 + 5 * 256)
#define DISK_STATIC_MAX_DEVICES 64
static __device__ __align__(256) unsigned char g_disk_scratch[DISK_STATIC_BYTES];

static std::mutex g_disk_scratch_lock;
static void *g_disk_scratch_addr[DISK_STATIC_MAX_DEVICES];       // per device ordinal; nullptr = not asked yet

// Device address of the current device's copy of g_disk_scratch.  The first call on a device resolves the symbol (which
// makes the runtime load this module on that device if it has not yet); later calls read the table.
static cudaError_t disk_static_scratch(unsigned char **ptr_out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= DISK_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_disk_scratch_lock);
    if (!g_disk_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_disk_scratch);
        if (e != cudaSuccess) return e;
        if (!p || ((uintptr_t)p & 255) != 0) return cudaErrorInvalidSymbol;
        g_disk_scratch_addr[dev] = p;
    }
    *ptr_out = (unsigned char *)g_disk_scratch_addr[dev];
    return cudaSuccess;
}

// Q arrives with everything but the scratch pointers filled in (radt_api.cu checked the descriptors and the size limit).
// Same two kernels as radt_launch_disk_fwd.  Nothing has to be cleared between calls: k_disk_columns<true> writes every
// word of rt, rho, P, colscale and colH of the columns of THIS call before it or k_disk_velocity<true> reads them, and
// neither kernel reads beyond those columns, so whatever an earlier (larger or smaller) call left behind is never seen.
cudaError_t radt_launch_disk_fwd_static(DiskParamsDev Q, cudaStream_t st)
{
    const long long cells = (long long)Q.nr * Q.nz * Q.nbatch, cols = (long long)Q.nr * Q.nbatch;
    auto up256 = [](long long x) { return (x + 255) & ~255ll; };
    const long long o_rt = 0, o_rho = up256(o_rt + cells * 8), o_P = up256(o_rho + cells * 8), o_cs = up256(o_P + cells * 8),
                    o_cH = up256(o_cs + cols * 8), end = up256(o_cH + cols * 8);
    if (cells < 1 || cells > DISK_STATIC_MAX_CELLS || end > (long long)DISK_STATIC_BYTES) return cudaErrorInvalidValue;
    unsigned char *base = nullptr;
    cudaError_t e = disk_static_scratch(&base);
    if (e != cudaSuccess) return e;
    Q.rt = (double *)(base + o_rt); Q.rho = (double *)(base + o_rho); Q.P = (double *)(base + o_P);
    Q.colscale = (double *)(base + o_cs); Q.colH = (double *)(base + o_cH);
    Q.gP = nullptr; Q.grho = nullptr; Q.mask = nullptr;           // adjoint-only scratch: the forward kernels never touch it
    return radt_launch_disk_fwd(Q, st);
}
