// radt_march.cu -- forward march (K2/K3) and memory-free adjoint march (K4/K5) for sm_100a.
//
// Mapping: one warp per ray.  Every 32-step block runs in two phases:
//   phase A  lanes over STEPS   : position (fp64), grid lookup, LTE thermodynamics -> 4 scalars/step
//   phase B  lanes over CHANNELS: for each active step, broadcast the 4 scalars from shared memory,
//                                 2 x MUFU.EX2 per (channel, step) sample, accumulate in registers
//   phase C  (adjoint) lanes over STEPS again: chain rule + vector atomics into the packed gradient.
// Algorithm: DESIGN.md O4-O11; PAPER.md:262-294 (Eq. 11-17).
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define FULL 0xffffffffu
#define UWIN 7.75f          // |u'| cut (u' = u sqrt(log2 e)): exp(-u^2) < 2^-60 beyond it
#define K2_EMPTY 1e-20f     // line-centre dtau*log2e below this adds < 1e-20 S per step: treated as vacuum
#define N_EMPTY 1e-17f      // density below which a sample is empty (K2 < 1e-19 for any realistic line)

struct StepState {
    bool inside;
    float vh, A, mvlA, K2, S;           // phase-B scalars: u' = (vcs - vh)*A + mvlA ; d = K2*g ; I += S*(1-e)*T
    // adjoint extras (dead code in the forward instantiation)
    float n, T, invT, ex, em1, W, invalpha, proj, vk, dsf, qy;
    float f0, f1, f2;
    long long cell;
    bool tclamp;
};

__device__ __forceinline__ float lerp1(float a, float b, float f) { return fmaf(f, b - a, a); }

template <int KIND, bool FWD>
__device__ __forceinline__ void phase_a(const MarchParams &P, const DevGeom &G, const float4 *__restrict__ cells,
                                        double ox, double oy, double oz, double s0, double ds, int k, StepState &st)
{
    const DevGrid &g = P.grid;
    const DevLine &L = P.line;
    st.inside = false;
    st.K2 = 0.f; st.A = 0.f; st.vh = 0.f; st.mvlA = 0.f; st.S = 0.f;
    double s = s0 + ((double)k + 0.5) * ds;
    double x = fma(s, G.wx, ox), y = fma(s, G.wy, oy), z = fma(s, G.wz, oz);
    double r2 = x * x + y * y;
    float r2f = (float)r2;
    float rs = rsqrt_approx(r2f);
    float dens, temp, vel;
    float rf, irf;
    double vel_d, ir_d;
    if (KIND == 0) {
        // fp64 1/r and r by one Newton step on the SFU seed: the in/out decision matches the fp64 oracle
        double y1 = (double)rs;
        y1 = y1 * fma(-0.5 * r2, y1 * y1, 1.5);
        double r = r2 * y1;
        double az = g.mirror ? fabs(z) : z;
        bool in = (k < P.nstep) && (r2 >= g.rmin2) && (r2 <= g.rmax2) && (az >= g.zlo * r) && (az <= g.zhi * r);
        if (!in) return;
        rf = (float)r;
        irf = (float)y1;
        // index coordinate along zeta in fp64; along log r: cell from the SFU estimate, corrected against
        // the fp64 node table, in-cell fraction from t = r / r_i by a log1p series (fine grids) or lg2
        double wd = fmin(fmax((az * y1 - g.zlo) * g.wscale_d, 0.0), (double)(g.n1 - 1));
        int j = min((int)wd, g.n1 - 2);
        float fw = (float)(wd - (double)j);
        float uf = lg2_approx((float)(r * g.inv_rmin)) * g.uscale;
        int i = min(max((int)uf, 0), g.n0 - 2);
        double2 nd = __ldg(P.ws.rnode + i);
        if (r < nd.x && i > 0) nd = __ldg(P.ws.rnode + (--i));
        else if (i < g.n0 - 2) {
            double2 nu = __ldg(P.ws.rnode + i + 1);
            if (r >= nu.x) { nd = nu; ++i; }
        }
        double t = r * nd.y;
        float fu;
        if (g.fine_r) {
            float xm = (float)(t - 1.0);
            float sq = xm * rcp_approx(2.0f + xm);
            float s2 = sq * sq;
            fu = 2.0f * sq * fmaf(s2, fmaf(s2, fmaf(s2, fmaf(s2, 1.0f / 9.0f, 1.0f / 7.0f), 0.2f), 1.0f / 3.0f), 1.0f) * g.inv_cell_ln;
        } else {
            fu = lg2_approx((float)t) * g.inv_cell_lg2;
        }
        fu = fminf(fmaxf(fu, 0.f), 1.f);
        long long cell = (long long)i * g.n1 + j;
        float4 c00 = __ldg(cells + cell), c01 = __ldg(cells + cell + 1);
        float4 c10 = __ldg(cells + cell + g.n1), c11 = __ldg(cells + cell + g.n1 + 1);
        dens = lerp1(lerp1(c00.x, c01.x, fw), lerp1(c10.x, c11.x, fw), fu);
        temp = lerp1(lerp1(c00.y, c01.y, fw), lerp1(c10.y, c11.y, fw), fu);
        {
            double fwd = (double)fw, fud = (double)fu;
            double a0 = fma(fwd, (double)c01.z - (double)c00.z, (double)c00.z);
            double a1 = fma(fwd, (double)c11.z - (double)c10.z, (double)c10.z);
            vel_d = fma(fud, a1 - a0, a0);
        }
        vel = (float)vel_d;
        ir_d = y1;
        st.f0 = fu; st.f1 = fw; st.f2 = 0.f; st.cell = cell;
    } else {
        bool in = (k < P.nstep) && (r2 > 0.0) && (x >= g.lo[0]) && (x <= g.hi[0]) && (y >= g.lo[1]) && (y <= g.hi[1]) &&
                  (z >= g.lo[2]) && (z <= g.hi[2]);
        if (!in) return;
        double y1 = (double)rs;
        y1 = y1 * fma(-0.5 * r2, y1 * y1, 1.5);
        ir_d = y1;
        rf = (float)(r2 * y1);
        irf = (float)y1;
        double tx = fmin(fmax((x - g.lo[0]) * g.inv_d[0], 0.0), (double)(g.n0 - 1));
        double ty = fmin(fmax((y - g.lo[1]) * g.inv_d[1], 0.0), (double)(g.n1 - 1));
        double tz = fmin(fmax((z - g.lo[2]) * g.inv_d[2], 0.0), (double)(g.n2 - 1));
        int i = min((int)tx, g.n0 - 2), j = min((int)ty, g.n1 - 2), l = min((int)tz, g.n2 - 2);
        float fx = (float)(tx - (double)i), fy = (float)(ty - (double)j), fz = (float)(tz - (double)l);
        long long cell = ((long long)i * g.n1 + j) * g.n2 + l;
        long long sy = g.n2, sx = (long long)g.n1 * g.n2;
        float4 c000 = __ldg(cells + cell), c001 = __ldg(cells + cell + 1);
        float4 c010 = __ldg(cells + cell + sy), c011 = __ldg(cells + cell + sy + 1);
        float4 c100 = __ldg(cells + cell + sx), c101 = __ldg(cells + cell + sx + 1);
        float4 c110 = __ldg(cells + cell + sx + sy), c111 = __ldg(cells + cell + sx + sy + 1);
        dens = lerp1(lerp1(lerp1(c000.x, c001.x, fz), lerp1(c010.x, c011.x, fz), fy),
                     lerp1(lerp1(c100.x, c101.x, fz), lerp1(c110.x, c111.x, fz), fy), fx);
        temp = lerp1(lerp1(lerp1(c000.y, c001.y, fz), lerp1(c010.y, c011.y, fz), fy),
                     lerp1(lerp1(c100.y, c101.y, fz), lerp1(c110.y, c111.y, fz), fy), fx);
        {
            double fzd = (double)fz, fyd = (double)fy, fxd = (double)fx;
            double a00 = fma(fzd, (double)c001.z - (double)c000.z, (double)c000.z);
            double a01 = fma(fzd, (double)c011.z - (double)c010.z, (double)c010.z);
            double a10 = fma(fzd, (double)c101.z - (double)c100.z, (double)c100.z);
            double a11 = fma(fzd, (double)c111.z - (double)c110.z, (double)c110.z);
            double b0 = fma(fyd, a01 - a00, a00), b1 = fma(fyd, a11 - a10, a10);
            vel_d = fma(fxd, b1 - b0, b0);
        }
        vel = (float)vel_d;
        st.f0 = fx; st.f1 = fy; st.f2 = fz; st.cell = cell;
    }
    // ---- O7: channel-independent LTE quantities (Eq. 13-17) ----
    float n = (g.dens_mode == 1) ? ex2_approx(dens * RADT_LOG2E) : dens;
    // empty samples: no opacity, hence no contribution to the cube; their only gradient is dL/dn, which exists
    // when the grid stores n itself (LINEAR) and vanishes with n when it stores ln n
    if ((FWD || g.dens_mode == 1) && P.opt_skip_empty && !(n > N_EMPTY)) return;
    st.inside = true;
    bool tcl = !(temp >= 1.0f);
    float T = tcl ? 1.0f : temp;
    float invT = rcp_approx(T);
    float xx = L.T0 * invT;
    float ex = ex2_approx(L.T0l2 * invT);
    float em1 = (xx < 0.0625f)
                    ? xx * fmaf(xx, fmaf(xx, fmaf(xx, fmaf(xx, 1.0f / 120.0f, 1.0f / 24.0f), 1.0f / 6.0f), 0.5f), 1.0f)
                    : ex - 1.0f;
    float S = G.sunit * rcp_approx(em1);
    float invalpha = rsqrt_approx(fmaf(L.a1, T, L.a0));
    float tq = fminf(lg2_approx(T) * ((float)RADT_NQ / RADT_NQ_OCTAVES), (float)RADT_NQ);
    int iq = (int)tq;
    float fq = tq - (float)iq;
    float2 q0 = __ldg(P.ws.qtab + iq), q1 = __ldg(P.ws.qtab + iq + 1);
    float Q = lerp1(q0.x, q1.x, fq);
    float iQ = rcp_approx(Q);
    float W = L.gu * ex2_approx(-L.Eul2 * invT) * iQ;
    float dsf = (float)ds;
    float K2 = L.Ck2 * n * W * em1 * dsf * invalpha;
    // v_los = omega . v in fp64: the velocity gradient is an odd sum over the line
    // profile, so v_los is carried as a two-float (hi, lo) pair into phase B
    double proj_d = (x * G.wy - y * G.wx) * ir_d;
    float proj = (float)proj_d;
    float vk = 1.0f;
    double vphi_d = vel_d;
    if (g.vel_mode == 1) {
        // Keplerian speed of Eq. 6 without the pressure term: v_K^2 = (GM/au) r^2 / rho^3, lengths in au
        double rho2 = r2 + z * z;
        double yr = (double)rsqrt_approx((float)rho2);
        yr = yr * fma(-0.5 * rho2, yr * yr, 1.5);
        double vk2 = G.gm_au_d * r2 * yr * yr * yr;
        double yv = (double)rsqrt_approx(fmaxf((float)vk2, 1e-30f));
        yv = yv * fma(-0.5 * vk2, yv * yv, 1.5);
        double vk_d = vk2 * yv;
        vk = (float)vk_d;
        vphi_d = vk_d * (1.0 + vel_d);
    }
    double vlos_d = vphi_d * proj_d;
    float vh = (float)vlos_d;
    float vl = (float)(vlos_d - (double)vh);
    st.A = invalpha * RADT_SQRT_LOG2E;
    st.vh = vh;
    st.mvlA = -vl * st.A;
    st.K2 = K2;
    st.S = S;
    st.n = n; st.T = T; st.invT = invT; st.ex = ex; st.em1 = em1; st.W = W; st.invalpha = invalpha;
    st.proj = proj; st.vk = vk; st.dsf = dsf; st.tclamp = tcl;
    st.qy = lerp1(q0.y, q1.y, fq) * iQ;      // dlnQ/dlnT
}


// ---------------------------------------------------------------------------------------------
// packed f32x2 arithmetic (sm_100: FADD2 / FMUL2 / FFMA2 issue one slot for two lanes' worth of work)
// ---------------------------------------------------------------------------------------------
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f2 pk1(float v) { return pk(v, v); }
__device__ __forceinline__ void upk(f2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

#define C_LN2 0.6931471805599453f
#define C_LN2SQ_2 0.2402265069591007f
#define C_LN2CU_6 0.05550410866482158f
#define D_SERIES 0.015625f   // below this 1 - 2^-d comes from the series (else cancellation breaks 1e-4 in thin wings)

// One (step, channel pair) sample of O8-O9 in log2 units.  q = {v_hi, A, -v_lo A, K'}; outputs u, g, d, e, 1-e.
struct Pair {
    f2 u, g, d, e, om;
};
template <bool CL>
__device__ __forceinline__ f2 pair_u(f2 vcs, f2 vcl, const float4 &q)
{
    f2 u = fma2(sub2(vcs, pk1(q.x)), pk1(q.y), pk1(q.z));      // exact difference of the hi parts
    if (CL) u = fma2(vcl, pk1(q.y), u);
    return u;
}
__device__ __forceinline__ void pair_eval(f2 u, float K2, Pair &s)
{
    s.u = u;
    float t0, t1;
    upk(mul2(u, u), t0, t1);
    s.g = pk(ex2_approx(-t0), ex2_approx(-t1));
    s.d = mul2(s.g, pk1(K2));
    float d0, d1;
    upk(s.d, d0, d1);
    s.e = pk(ex2_approx(-d0), ex2_approx(-d1));
    f2 sm = mul2(s.d, fma2(s.d, fma2(s.d, pk1(C_LN2CU_6), pk1(-C_LN2SQ_2)), pk1(C_LN2)));
    f2 bg = fma2(s.e, pk1(-1.0f), pk1(1.0f));
    float s0, s1, b0, b1;
    upk(sm, s0, s1);
    upk(bg, b0, b1);
    s.om = pk(d0 < D_SERIES ? s0 : b0, d1 < D_SERIES ? s1 : b1);
}
__device__ __forceinline__ bool pair_in_window(f2 u)
{
    float u0, u1;
    upk(u, u0, u1);
    return fabsf(u0) < UWIN || fabsf(u1) < UWIN;
}

struct RayCtx {
    int ix, iy, b;
    size_t ray;
    double s0, ds, ox, oy, oz;
    int k_lo, k_hi;
};

__device__ __forceinline__ bool ray_setup(const MarchParams &P, RayCtx &rc, int warp)
{
    int tx = blockIdx.x % P.tiles_x, ty = blockIdx.x / P.tiles_x;
    rc.b = blockIdx.y;
    rc.ix = tx * RADT_TILE_X + (warp & (RADT_TILE_X - 1));
    rc.iy = ty * RADT_TILE_Y + (warp / RADT_TILE_X);
    if (rc.ix >= P.nx || rc.iy >= P.ny) return false;
    rc.ray = ((size_t)(P.b0 + rc.b) * P.ny + rc.iy) * P.nx + rc.ix;
    RayRec rr = P.ws.rays[rc.ray];
    rc.s0 = rr.s0; rc.ds = rr.ds; rc.k_lo = rr.k_lo; rc.k_hi = rr.k_hi;
    double X, Y;
    pixel_origin(P.geom[rc.b], P.nx, P.ny, rc.ix, rc.iy, rc.ox, rc.oy, rc.oz, X, Y);
    return true;
}

// Channel velocities of this lane (pairs of channels lane + 64 p, lane + 64 p + 32) and the span of all
// channels of the item: a step whose line window misses the whole span contributes nothing.
template <int NP>
__device__ __forceinline__ void load_channels(const float2 *__restrict__ vtab, int nchan, int lane, f2 (&vcs)[NP],
                                              f2 (&vcl)[NP], float &vmin, float &vmax)
{
    vmin = 3.0e38f; vmax = -3.0e38f;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        int c0 = lane + 64 * p, c1 = c0 + 32;
        float2 v0 = (c0 < nchan) ? __ldg(vtab + c0) : make_float2(0.f, 0.f);
        float2 v1 = (c1 < nchan) ? __ldg(vtab + c1) : make_float2(0.f, 0.f);
        vcs[p] = pk(v0.x, v1.x); vcl[p] = pk(v0.y, v1.y);
        if (c0 < nchan) { vmin = fminf(vmin, v0.x); vmax = fmaxf(vmax, v0.x); }
        if (c1 < nchan) { vmin = fminf(vmin, v1.x); vmax = fmaxf(vmax, v1.x); }
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) {
        vmin = fminf(vmin, __shfl_xor_sync(FULL, vmin, m));
        vmax = fmaxf(vmax, __shfl_xor_sync(FULL, vmax, m));
    }
}

__device__ __forceinline__ bool line_hits_span(const StepState &st, float vmin, float vmax)
{
    return (vmin - st.vh) * st.A < UWIN && (vmax - st.vh) * st.A > -UWIN;
}

// ---------------------------------------------------------------------------------------------
// K2 / K3 forward march.  NP = channel-group pairs per lane: lane owns channels lane + 32 g, g < 2 NP.
// ---------------------------------------------------------------------------------------------
template <int KIND, int NP, bool CL>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32) k_march_fwd(const __grid_constant__ MarchParams P)
{
    __shared__ float4 sh_p[RADT_WARPS_PER_CTA][32];
    __shared__ float sh_s[RADT_WARPS_PER_CTA][32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RayCtx rc;
    if (!ray_setup(P, rc, warp)) return;
    const DevGeom &G = P.geom[rc.b];
    const int nchan = P.line.nchan;
    float *out = P.cube + rc.ray * (size_t)nchan;
    f2 I[NP], T[NP], vcs[NP], vcl[NP];
    float vmin, vmax;
    load_channels<NP>(P.ws.vcs + (size_t)(P.b0 + rc.b) * RADT_MAXCHAN, nchan, lane, vcs, vcl, vmin, vmax);
#pragma unroll
    for (int p = 0; p < NP; ++p) { I[p] = pk(0.f, 0.f); T[p] = pk(1.f, 1.f); }
    unsigned n_steps = 0, n_mufu = 0;
    if (rc.ds != 0.0) {
        const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
        // only the 32-step blocks that can hold in-grid samples (K1's conservative step range)
        for (int kb = rc.k_lo & ~31; kb < rc.k_hi; kb += 32) {
            StepState st;
            phase_a<KIND, true>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, kb + lane, st);
            bool active = st.inside && (st.K2 > K2_EMPTY || !P.opt_skip_empty) &&
                          (!P.opt_window || line_hits_span(st, vmin, vmax));
            unsigned mask = __ballot_sync(FULL, active);
            if (mask == 0u) continue;
            // compact the active steps (in march order) so that phase B is a plain counted loop
            if (active) {
                int pos = __popc(mask & ((1u << lane) - 1u));
                sh_p[warp][pos] = make_float4(st.vh, st.A, st.mvlA, st.K2);
                sh_s[warp][pos] = st.S;
            }
            __syncwarp();
            const int cnt = __popc(mask);
            n_steps += cnt;
#pragma unroll 2
            for (int j = 0; j < cnt; ++j) {
                float4 q = sh_p[warp][j];
                f2 S2 = pk1(sh_s[warp][j]);
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    f2 u = pair_u<CL>(vcs[p], vcl[p], q);
                    if (NP > 1 && P.opt_window && !__any_sync(FULL, pair_in_window(u))) continue;
                    n_mufu += 4;
                    Pair s;
                    pair_eval(u, q.w, s);
                    // contribution c = S ((1-e) T) and partial sum I += c as ONE explicit FMA: the adjoint
                    // re-march repeats exactly this sequence and so reproduces the partial sums bit for bit
                    I[p] = fma2(S2, mul2(s.om, T[p]), I[p]);
                    T[p] = mul2(T[p], s.e);
                }
            }
            __syncwarp();
        }
    }
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        int c0 = lane + 64 * p, c1 = c0 + 32;
        float i0, i1;
        upk(I[p], i0, i1);
        if (c0 < nchan) out[c0] = i0;
        if (c1 < nchan) out[c1] = i1;
    }
    if (lane == 0 && n_steps) {
        atomicAdd(P.ws.counters + 0, (unsigned long long)n_steps);
        atomicAdd(P.ws.counters + 1, (unsigned long long)n_mufu);
    }
}

// ---------------------------------------------------------------------------------------------
// K4 / K5 adjoint march: front-to-back re-march with the saved cube
//   dL/d dtau_k,c = G_c (T_{k+1,c} S_k - R_k,c),  R_k = I - I_{<=k}        dL/dS_k = sum_c G_c (1-e_k,c) T_k,c
// Steps come in two kinds: E (emitting, K > 0) update the transmittance and the partial sums and feed all four
// channel sums; Z (zero opacity, LINEAR density grids) leave the ray state untouched and feed dL/dn only.
// Channel sums are written per lane to shared memory and reduced for RADT_NS steps at a time.
// ---------------------------------------------------------------------------------------------
#define RADT_NS 8

// Gradient cells are accumulated as packed float4 {dens, temp, vel, -} (one vector reduction per corner),
// unpacked to the caller's planes by k_unpack_grad.
__device__ __forceinline__ void red_add_cell(float4 *cell, float w, float a, float b, float c)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(cell), "f"(w * a), "f"(w * b), "f"(w * c), "f"(0.f)
                 : "memory");
}
__device__ __forceinline__ void red_add_dens(float4 *cell, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(cell), "f"(v) : "memory");
}

__device__ __forceinline__ f2 clamp_nR(f2 PmI, f2 Tn, f2 nsmax2)
{
    // -R = P - I_saved, R = T_{k+1} B_{k+1}: the truth lies in [0, T_{k+1} S_max]; clamping there makes the
    // rounding error of the subtraction decay with the transmittance
    float r0, r1, b0, b1;
    upk(PmI, r0, r1);
    upk(mul2(Tn, nsmax2), b0, b1);
    return pk(fminf(fmaxf(r0, b0), 0.f), fminf(fmaxf(r1, b1), 0.f));
}

template <int NP, bool CL>
__device__ __forceinline__ float4 bwd_estep(const float4 q, const float S, const float nsmax, const bool window,
                                            f2 (&T)[NP], f2 (&Pp)[NP], const f2 (&Isv)[NP], const f2 (&Gc)[NP],
                                            const f2 (&vcs)[NP], const f2 (&vcl)[NP], unsigned &n_mufu)
{
    const f2 S2 = pk1(S), nsm2 = pk1(nsmax);
    f2 a0 = pk(0.f, 0.f), a1 = a0, a2 = a0, a3 = a0;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        f2 u = pair_u<CL>(vcs[p], vcl[p], q);
        if (NP > 1 && window && !__any_sync(FULL, pair_in_window(u))) continue;
        n_mufu += 4;
        Pair s;
        pair_eval(u, q.w, s);
        f2 omT = mul2(s.om, T[p]);
        Pp[p] = fma2(S2, omT, Pp[p]);                 // = the forward's partial sum I_{<=k}, bit for bit
        f2 Tn = mul2(T[p], s.e);
        f2 nR = clamp_nR(sub2(Pp[p], Isv[p]), Tn, nsm2);
        f2 a = mul2(Gc[p], fma2(Tn, S2, nR));         // dL/d dtau
        f2 w = mul2(a, s.g), wu = mul2(w, s.u);
        if (NP == 1) {
            a0 = w; a1 = wu; a2 = mul2(wu, s.u); a3 = mul2(Gc[p], omT);
        } else {
            a0 = add2(a0, w); a1 = add2(a1, wu); a2 = fma2(wu, s.u, a2); a3 = fma2(Gc[p], omT, a3);
        }
        T[p] = Tn;
    }
    float x0, x1, y0, y1, z0, z1, w0, w1;
    upk(a0, x0, x1); upk(a1, y0, y1); upk(a2, z0, z1); upk(a3, w0, w1);
    return make_float4(x0 + x1, y0 + y1, z0 + z1, w0 + w1);
}

template <int NP, bool CL>
__device__ __forceinline__ float bwd_zstep(const float4 q, const float S, const bool window, const f2 (&GT)[NP],
                                           const f2 (&GnR)[NP], const f2 (&vcs)[NP], const f2 (&vcl)[NP],
                                           unsigned &n_mufu)
{
    const f2 S2 = pk1(S);
    f2 acc = pk(0.f, 0.f);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        f2 u = pair_u<CL>(vcs[p], vcl[p], q);
        if (NP > 1 && window && !__any_sync(FULL, pair_in_window(u))) continue;
        n_mufu += 2;
        float t0, t1;
        upk(mul2(u, u), t0, t1);
        f2 g = pk(ex2_approx(-t0), ex2_approx(-t1));
        f2 w = mul2(fma2(GT[p], S2, GnR[p]), g);
        acc = (NP == 1) ? w : add2(acc, w);
    }
    float x0, x1;
    upk(acc, x0, x1);
    return x0 + x1;
}

// Sum the RADT_NS x 32 per-lane partials of a batch over the lanes; lanes 0..nb-1 store the sums of steps 0..nb-1.
// Lane (s = lane & 7, h = lane >> 3) adds the 8 source lanes 8h..8h+7 of step s (skewed: conflict-free
// 16-byte reads), then the four quarters are combined with two shuffle rounds.
template <bool ZONLY>
__device__ __forceinline__ void reduce_batch(const float4 (*red)[32], int nb, float4 *out, int lane)
{
    const int s = lane & 7, h8 = lane & 24;
    float4 acc;
    if (ZONLY) {
        acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc.x += red[s][h8 + ((i + s) & 7)].x;
        acc.x += __shfl_xor_sync(FULL, acc.x, 8);
        acc.x += __shfl_xor_sync(FULL, acc.x, 16);
    } else {
        acc = red[s][h8 + s];
#pragma unroll
        for (int i = 1; i < 8; ++i) {
            float4 v = red[s][h8 + ((i + s) & 7)];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
#pragma unroll
        for (int m = 8; m <= 16; m <<= 1) {
            acc.x += __shfl_xor_sync(FULL, acc.x, m);
            acc.y += __shfl_xor_sync(FULL, acc.y, m);
            acc.z += __shfl_xor_sync(FULL, acc.z, m);
            acc.w += __shfl_xor_sync(FULL, acc.w, m);
        }
    }
    if (lane < nb) out[lane] = acc;
}

template <int KIND, int NP, bool CL>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32, 3) k_march_bwd(const __grid_constant__ MarchParams P)
{
    __shared__ float4 sh_p[RADT_WARPS_PER_CTA][32];
    __shared__ float sh_s[RADT_WARPS_PER_CTA][32];
    __shared__ float4 sh_sum[RADT_WARPS_PER_CTA][32];
    __shared__ float4 sh_red[RADT_WARPS_PER_CTA][RADT_NS][32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RayCtx rc;
    if (!ray_setup(P, rc, warp)) return;
    if (rc.ds == 0.0) return;
    const DevGeom &G = P.geom[rc.b];
    const DevLine &L = P.line;
    const int nchan = L.nchan;
    const float *Isave = P.cube + rc.ray * (size_t)nchan;
    const float *Gin = P.dl_dcube + rc.ray * (size_t)nchan;
    f2 Isv[NP], Pp[NP], T[NP], vcs[NP], vcl[NP], Gc[NP];
    float vmin, vmax;
    load_channels<NP>(P.ws.vcs + (size_t)(P.b0 + rc.b) * RADT_MAXCHAN, nchan, lane, vcs, vcl, vmin, vmax);
    bool anyg = false;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        int c0 = lane + 64 * p, c1 = c0 + 32;
        bool ok0 = c0 < nchan, ok1 = c1 < nchan;
        float g0 = ok0 ? __ldg(Gin + c0) : 0.f, g1 = ok1 ? __ldg(Gin + c1) : 0.f;
        T[p] = pk(1.f, 1.f); Pp[p] = pk(0.f, 0.f);
        Isv[p] = pk(ok0 ? __ldg(Isave + c0) : 0.f, ok1 ? __ldg(Isave + c1) : 0.f);
        Gc[p] = pk(g0, g1);
        anyg |= (g0 != 0.f) || (g1 != 0.f);
    }
    if (!__any_sync(FULL, anyg)) return;     // dL/dcube vanishes on this ray: no gradient
    const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    float4 *grad = P.ws.grad + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    // upper bound of the source function anywhere on the grid (S grows with T)
    const float tmax = fmaxf(__int_as_float(*reinterpret_cast<const int *>(P.ws.counters + 4)), 1.0f);
    const float nsmax = -G.sunit * 1.0001f / (ex2_approx(L.T0l2 / tmax) - 1.0f);
    const float kthr = P.opt_skip_empty ? K2_EMPTY : 0.f;    // the forward's own test for an emitting step
    const bool window = P.opt_window;
    unsigned n_steps = 0, n_mufu = 0;
    for (int kb = rc.k_lo & ~31; kb < rc.k_hi; kb += 32) {
        StepState st;
        phase_a<KIND, false>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, kb + lane, st);
        const bool isE = st.inside && st.K2 > kthr;
        // zero-opacity steps still carry dL/dn when the grid stores n itself (LINEAR)
        const bool active = st.inside && (isE || P.grid.dens_mode == 0) && (!window || line_hits_span(st, vmin, vmax));
        const unsigned mask = __ballot_sync(FULL, active);
        if (mask == 0u) continue;
        const int pos = __popc(mask & ((1u << lane) - 1u));
        if (active) {
            sh_p[warp][pos] = make_float4(st.vh, st.A, st.mvlA, isE ? st.K2 : 0.f);
            sh_s[warp][pos] = st.S;
        }
        __syncwarp();
        const int cnt = __popc(mask);
        n_steps += cnt;
        const unsigned emask = __ballot_sync(FULL, lane < cnt && sh_p[warp][lane].w > 0.f);   // compacted E flags
        for (int base = 0; base < cnt; base += RADT_NS) {
            const int nb = min(RADT_NS, cnt - base);
            if ((emask >> base) & ((1u << RADT_NS) - 1u)) {
#pragma unroll 2
                for (int jj = 0; jj < nb; ++jj) {
                    float4 q = sh_p[warp][base + jj];
                    float S = sh_s[warp][base + jj];
                    sh_red[warp][jj][lane] = bwd_estep<NP, CL>(q, S, nsmax, window, T, Pp, Isv, Gc, vcs, vcl, n_mufu);
                }
                __syncwarp();
                reduce_batch<false>(sh_red[warp], nb, &sh_sum[warp][base], lane);
            } else {
                // a run of zero-opacity steps: T, P and hence G T and G R stay fixed
                f2 GT[NP], GnR[NP];
                const f2 nsm2 = pk1(nsmax);
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    GT[p] = mul2(Gc[p], T[p]);
                    GnR[p] = mul2(Gc[p], clamp_nR(sub2(Pp[p], Isv[p]), T[p], nsm2));
                }
#pragma unroll 4
                for (int jj = 0; jj < nb; ++jj) {
                    float4 q = sh_p[warp][base + jj];
                    float S = sh_s[warp][base + jj];
                    sh_red[warp][jj][lane].x = bwd_zstep<NP, CL>(q, S, window, GT, GnR, vcs, vcl, n_mufu);
                }
                __syncwarp();
                reduce_batch<true>(sh_red[warp], nb, &sh_sum[warp][base], lane);
            }
            __syncwarp();
        }
        // ---- phase C: chain rule to (n, T, v_phi) at this lane's step, scatter to the grid (O11) ----
        if (active) {
            float4 sm = sh_sum[warp][pos];
            const float iL2 = RADT_LN2;                       // 1 / log2(e)
            float ia = st.invalpha;
            float A0 = sm.x;
            float dL_dn = A0 * (L.Ck2 * iL2) * st.W * st.em1 * st.dsf * ia;
            float dL_dd = (P.grid.dens_mode == 1) ? dL_dn * st.n : dL_dn;
            float4 *gp = grad + st.cell;
            if (isE) {
                // the lane sums are moments of w = a g: sum a dtau u^m = K sum w u^m
                float A1 = st.K2 * sm.y * (iL2 / RADT_SQRT_LOG2E);
                float A2 = st.K2 * sm.z * (iL2 * iL2);
                float Bs = sm.w;
                float K = st.K2 * iL2;
                float dL_dvlos = 2.0f * ia * A1;
                float dL_dalpha = ia * (2.0f * A2 - A0 * K);
                float iT2 = st.invT * st.invT;
                float iem1 = rcp_approx(st.em1);
                float exs = (st.em1 + 1.0f);                       // e^x, consistent with the series branch
                float dlnF_dT = L.Eu * iT2 - L.T0 * iT2 * exs * iem1 - st.qy * st.invT;
                float dS_dT = st.S * exs * iem1 * L.T0 * iT2;
                float dalpha_dT = 0.5f * L.a1 * ia;
                float dL_dT = A0 * K * dlnF_dT + dL_dalpha * dalpha_dT + Bs * dS_dT;
                if (st.tclamp) dL_dT = 0.f;
                float dL_dv = dL_dvlos * st.proj * st.vk;
                if (KIND == 0) {
                    float fu = st.f0, fw = st.f1;
                    long long n1 = P.grid.n1;
                    red_add_cell(gp, (1.f - fu) * (1.f - fw), dL_dd, dL_dT, dL_dv);
                    red_add_cell(gp + 1, (1.f - fu) * fw, dL_dd, dL_dT, dL_dv);
                    red_add_cell(gp + n1, fu * (1.f - fw), dL_dd, dL_dT, dL_dv);
                    red_add_cell(gp + n1 + 1, fu * fw, dL_dd, dL_dT, dL_dv);
                } else {
                    long long sy = P.grid.n2, sx = (long long)P.grid.n1 * P.grid.n2;
#pragma unroll
                    for (int cidx = 0; cidx < 8; ++cidx) {
                        int dx = (cidx >> 2) & 1, dy = (cidx >> 1) & 1, dz = cidx & 1;
                        float w = (dx ? st.f0 : 1.f - st.f0) * (dy ? st.f1 : 1.f - st.f1) * (dz ? st.f2 : 1.f - st.f2);
                        red_add_cell(gp + (dx * sx + dy * sy + dz), w, dL_dd, dL_dT, dL_dv);
                    }
                }
            } else {
                if (KIND == 0) {
                    float fu = st.f0, fw = st.f1;
                    long long n1 = P.grid.n1;
                    red_add_dens(gp, (1.f - fu) * (1.f - fw) * dL_dd);
                    red_add_dens(gp + 1, (1.f - fu) * fw * dL_dd);
                    red_add_dens(gp + n1, fu * (1.f - fw) * dL_dd);
                    red_add_dens(gp + n1 + 1, fu * fw * dL_dd);
                } else {
                    long long sy = P.grid.n2, sx = (long long)P.grid.n1 * P.grid.n2;
#pragma unroll
                    for (int cidx = 0; cidx < 8; ++cidx) {
                        int dx = (cidx >> 2) & 1, dy = (cidx >> 1) & 1, dz = cidx & 1;
                        float w = (dx ? st.f0 : 1.f - st.f0) * (dy ? st.f1 : 1.f - st.f1) * (dz ? st.f2 : 1.f - st.f2);
                        red_add_dens(gp + (dx * sx + dy * sy + dz), w * dL_dd);
                    }
                }
            }
        }
        __syncwarp();
    }
    if (lane == 0 && n_steps) {
        atomicAdd(P.ws.counters + 2, (unsigned long long)n_steps);
        atomicAdd(P.ws.counters + 3, (unsigned long long)n_mufu);
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
template <int KIND, int NP>
static cudaError_t launch_fwd_t(const MarchParams &P, int nbatch, cudaStream_t st)
{
    dim3 grid(P.tiles_x * P.tiles_y, nbatch);
    if (P.chan_lo) k_march_fwd<KIND, NP, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else k_march_fwd<KIND, NP, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    return cudaGetLastError();
}

template <int KIND, int NP>
static cudaError_t launch_bwd_t(const MarchParams &P, int nbatch, cudaStream_t st)
{
    dim3 grid(P.tiles_x * P.tiles_y, nbatch);
    if (P.chan_lo) k_march_bwd<KIND, NP, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else k_march_bwd<KIND, NP, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    return cudaGetLastError();
}

#define RADT_DISPATCH(fn)                                                        \
    int np = (P.line.ngroups + 1) / 2;                                           \
    if (P.grid.kind == 0) {                                                      \
        if (np <= 1) return fn<0, 1>(P, nbatch, st);                             \
        if (np <= 2) return fn<0, 2>(P, nbatch, st);                             \
        return fn<0, 4>(P, nbatch, st);                                          \
    }                                                                            \
    if (np <= 1) return fn<1, 1>(P, nbatch, st);                                 \
    if (np <= 2) return fn<1, 2>(P, nbatch, st);                                 \
    return fn<1, 4>(P, nbatch, st);

cudaError_t radt_launch_march_fwd(const MarchParams &P, int nbatch, cudaStream_t st) { RADT_DISPATCH(launch_fwd_t) }
cudaError_t radt_launch_march_bwd(const MarchParams &P, int nbatch, cudaStream_t st) { RADT_DISPATCH(launch_bwd_t) }
