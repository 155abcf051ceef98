// radt_march.cuh -- device code shared by the two march kernel families (radt_march.cu: channel-table path,
// radt_march_win.cu: uniform-channel window path): per-step sampling and LTE thermodynamics (phase A), packed
// f32x2 helpers, the (channel, step) sample, ray set-up.  Algorithm: DESIGN.md O4-O11.
#pragma once
#include "radt_dev.cuh"
#include "radt_kernels.h"
#define FULL 0xffffffffu
#define UWIN 7.75f          // channel-table path: |u'| cut (u' = u sqrt(log2 e)), exp(-u^2) < 2^-60 beyond it
#define UWIN2_MIN 40.0f     // window path: cut where dtau = K' 2^(-u'^2) < 2^-40 .. 2^-60, i.e. u'^2 > 40 .. 60 + log2 K'
#define UWIN2_MAX 60.0f
#define K2_EMPTY 1e-20f     // line-centre dtau*log2e below this adds < 1e-20 S per step: treated as vacuum
#define N_EMPTY 1e-17f      // density below which a sample is empty (K2 < 1e-19 for any realistic line)

struct StepState {
    bool inside;
    float vh, A, mvlA, K2, S;           // phase-B scalars: u' = (vcs - vh)*A + mvlA ; d = K2*g ; I += S*(1-e)*T
    // adjoint extras (dead code in the forward instantiation): the chain rule of phase C as coefficients of the four
    // channel sums {sum w, sum w u', sum w u'^2, sum G (1-e) T}, formed in phase A so that nothing else of the step's
    // thermodynamics has to stay in registers across phase B:
    //   dL/d(stored density) = cd sum_w;  dL/dT = cT0 sum_w + cT2 sum_wuu + cT3 sum_GcT;  dL/d(stored velocity) = cv sum_wu
    float cd, cT0, cT2, cT3, cv;
    float f0, f1, f2;                   // in-cell fractions
    int cell;                           // first corner of the cell (within the batch item)
    int dk;                             // spherical grids: offset of the next phi node (1, or 1 - nphi across the seam)
    // uniform channel lattice (window path): u'(c) = u0 + (c - cref) dvA; channels wlo..whi can lie inside the line
    float u0, dvA;
    int cref, wlo, whi;
};

__device__ __forceinline__ float lerp1(float a, float b, float f) { return fmaf(f, b - a, a); }

// round to nearest integer of |y| < 2^22 without the conversion pipe
__device__ __forceinline__ int rn_int(float y) { return __float_as_int(y + 12582912.0f) - 0x4B400000; }

template <int KIND, bool FWD, bool UNI>
__device__ __forceinline__ void phase_a(const MarchParams &P, const DevGeom &G, const float4 *__restrict__ cells,
                                        double ox, double oy, double oz, double s0, double ds, int k, StepState &st)
{
    const DevGrid &g = P.grid;
    const DevLine &L = P.line;
    st.inside = false;
    st.K2 = 0.f; st.A = 0.f; st.vh = 0.f; st.mvlA = 0.f; st.S = 0.f;
    // Sample position with every product and sum rounded separately (no FMA contraction): the in/out decisions and
    // the r = 0 rule are exact comparisons, and they agree with a plain fp64 evaluation of O4 only if the
    // position carries the same roundings (a ray through the star whose midpoint falls on it gave s = 1e-14 with
    // an FMA and s = 0, a skipped step, without: randomised parity scenes 5, 20, 21).
    const double s = __dadd_rn(s0, __dmul_rn(__hiloint2double(0x43300000, k) - 4503599627370495.5, ds));   // (k + 1/2) ds, exact k + 1/2
    const double x = __dadd_rn(ox, __dmul_rn(s, G.wx)), y = __dadd_rn(oy, __dmul_rn(s, G.wy)), z = __dadd_rn(oz, __dmul_rn(s, G.wz));
    double r2 = x * x + y * y;
    float r2f = (float)r2;
    double ir_d = rsqrt_d(r2);          // fp64 1/r: SFU seed + one Newton step
    float dens, temp;
    double vel_d;
    if (KIND == 0) {
        // the in/out decision is taken in fp64 so that it matches the fp64 oracle (reading (a))
        double r = r2 * ir_d;
        double az = g.mirror ? fabs(z) : z;
        bool in = (k < P.nstep) && (r2 >= g.rmin2) && (r2 <= g.rmax2) && (az >= g.zlo * r) && (az <= g.zhi * r);
        if (!in) return;
        // Index coordinates (O5).  The cell comes from an fp32 estimate (round to nearest without the conversion
        // pipe); the in-cell fractions are formed in the cell, so they do not carry the rounding of an index of
        // several hundred: zeta in fp64, log r from t = r^2 / r_i^2 by a log1p series (fine grids) or MUFU.LG2.
        // A fraction a few 1e-5 outside [0, 1] (estimate off by one cell next to a node) extrapolates the
        // neighbouring cell's bilinear form, which differs from the exact value by that distance times the
        // change of slope.
        double wd = (az * ir_d - g.zlo) * g.wscale_d;
        int j = min(max(rn_int((float)wd - 0.5f), 0), g.n1 - 2);
        float fw = (float)(wd - int_to_double(j));
        float uf = lg2_approx(r2f * g.inv_rmin2_f) * g.half_uscale;
        int i = min(max(rn_int(uf - 0.5f), 0), g.n0 - 2);
        double t = r2 * __ldg(P.ws.rnode + i).y;
        float fu;
        if (g.fine_r) {
            float xm = (float)(t - 1.0);
            float sq = xm * rcp_approx(2.0f + xm);
            float s2 = sq * sq;
            fu = sq * fmaf(s2, fmaf(s2, fmaf(s2, fmaf(s2, 1.0f / 9.0f, 1.0f / 7.0f), 0.2f), 1.0f / 3.0f), 1.0f) * g.inv_cell_ln;
        } else {
            fu = lg2_approx((float)t) * (0.5f * g.inv_cell_lg2);
        }
        int cell = i * g.n1 + j;
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
        if (!FWD) { st.f0 = fu; st.f1 = fw; st.f2 = 0.f; st.cell = cell; }
    } else if (KIND == 2) {
        // spherical (r, theta, phi) grid.  In/out decision in fp64 on rho^2 and cos(theta);
        // radial index as on the axisymmetric grid (cell from an fp32 estimate, in-cell fraction from rho^2/r_i^2);
        // theta through asin(z/rho), which is well conditioned around the equator where disk grids live; phi
        // through atan2 in fp32 (1e-7 rad is 4e-6 of a cell at 256 nodes).
        // rho^2 with every product and sum rounded, and thresholds that are exactly the doubles whose square root lies in
        // [r_min, r_max]: the radial in/out decision of a plain fp64 evaluation, boundary ties included (radt_dev.cuh)
        double rho2 = __dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z));
        double irho = rsqrt_d(rho2);
        double cz = z * irho;
        bool in = (k < P.nstep) && (r2 > 0.0) && (rho2 >= g.rho2_lo) && (rho2 <= g.rho2_hi) && (cz <= g.cos_tlo) && (cz >= g.cos_thi);
        if (!in) return;
        float wf = fminf(fmaxf((g.th_c0 - asinf((float)cz)) * g.th_scale, 0.f), (float)(g.n1 - 1));
        int j = min(max(rn_int(wf - 0.5f), 0), g.n1 - 2);
        float fw = wf - (float)j;
        float uf = lg2_approx((float)rho2 * g.inv_rmin2_f) * g.half_uscale;
        int i = min(max(rn_int(uf - 0.5f), 0), g.n0 - 2);
        double t = rho2 * __ldg(P.ws.rnode + i).y;
        float fu;
        if (g.fine_r) {
            float xm = (float)(t - 1.0);
            float sq = xm * rcp_approx(2.0f + xm);
            float s2 = sq * sq;
            fu = sq * fmaf(s2, fmaf(s2, fmaf(s2, fmaf(s2, 1.0f / 9.0f, 1.0f / 7.0f), 0.2f), 1.0f / 3.0f), 1.0f) * g.inv_cell_ln;
        } else {
            fu = lg2_approx((float)t) * (0.5f * g.inv_cell_lg2);
        }
        float qf = atan2f((float)y, (float)x) * g.ph_scale;
        if (qf < 0.f) qf += (float)g.n2;
        qf = fminf(fmaxf(qf, 0.f), (float)g.n2);
        int l = min(max(rn_int(qf - 0.5f), 0), g.n2 - 1);
        float fq = fminf(fmaxf(qf - (float)l, 0.f), 1.f);
        int dk = (l == g.n2 - 1) ? 1 - g.n2 : 1;
        long long cell = ((long long)i * g.n1 + j) * g.n2 + l;
        long long sy = g.n2, sx = (long long)g.n1 * g.n2;
        float4 c000 = __ldg(cells + cell), c001 = __ldg(cells + cell + dk);
        float4 c010 = __ldg(cells + cell + sy), c011 = __ldg(cells + cell + sy + dk);
        float4 c100 = __ldg(cells + cell + sx), c101 = __ldg(cells + cell + sx + dk);
        float4 c110 = __ldg(cells + cell + sx + sy), c111 = __ldg(cells + cell + sx + sy + dk);
        dens = lerp1(lerp1(lerp1(c000.x, c001.x, fq), lerp1(c010.x, c011.x, fq), fw),
                     lerp1(lerp1(c100.x, c101.x, fq), lerp1(c110.x, c111.x, fq), fw), fu);
        temp = lerp1(lerp1(lerp1(c000.y, c001.y, fq), lerp1(c010.y, c011.y, fq), fw),
                     lerp1(lerp1(c100.y, c101.y, fq), lerp1(c110.y, c111.y, fq), fw), fu);
        {
            double fzd = (double)fq, fyd = (double)fw, fxd = (double)fu;
            double a00 = fma(fzd, (double)c001.z - (double)c000.z, (double)c000.z);
            double a01 = fma(fzd, (double)c011.z - (double)c010.z, (double)c010.z);
            double a10 = fma(fzd, (double)c101.z - (double)c100.z, (double)c100.z);
            double a11 = fma(fzd, (double)c111.z - (double)c110.z, (double)c110.z);
            double b0 = fma(fyd, a01 - a00, a00), b1 = fma(fyd, a11 - a10, a10);
            vel_d = fma(fxd, b1 - b0, b0);
        }
        if (!FWD) { st.f0 = fu; st.f1 = fw; st.f2 = fq; st.cell = (int)cell; st.dk = dk; }
    } else {
        bool in = (k < P.nstep) && (r2 > 0.0) && (x >= g.lo[0]) && (x <= g.hi[0]) && (y >= g.lo[1]) && (y <= g.hi[1]) &&
                  (z >= g.lo[2]) && (z <= g.hi[2]);
        if (!in) return;
        float tx = fminf(fmaxf((float)((x - g.lo[0]) * g.inv_d[0]), 0.f), (float)(g.n0 - 1));
        float ty = fminf(fmaxf((float)((y - g.lo[1]) * g.inv_d[1]), 0.f), (float)(g.n1 - 1));
        float tz = fminf(fmaxf((float)((z - g.lo[2]) * g.inv_d[2]), 0.f), (float)(g.n2 - 1));
        int i = min(max(rn_int(tx - 0.5f), 0), g.n0 - 2), j = min(max(rn_int(ty - 0.5f), 0), g.n1 - 2);
        int l = min(max(rn_int(tz - 0.5f), 0), g.n2 - 2);
        float fx = tx - (float)i, fy = ty - (float)j, fz = tz - (float)l;
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
        if (!FWD) { st.f0 = fx; st.f1 = fy; st.f2 = fz; st.cell = (int)cell; st.dk = 1; }
    }
    // ---- O7: channel-independent LTE quantities (Eq. 13-17) ----
    float n = (g.dens_mode == 1) ? ex2_approx(dens * RADT_LOG2E) : dens;
    // empty samples: no opacity, hence no contribution to the cube; their only gradient is dL/dn, which exists
    // when the grid stores n itself (LINEAR) and vanishes with n when it stores ln n
    if ((FWD || g.dens_mode == 1 || !P.opt_zero_grad) && P.opt_skip_empty && !(n > N_EMPTY)) return;
    st.inside = true;
    // T is clamped to [1 K, RADT_TMAX] (the range of the Q(T) table, include/radt.h); no gradient through either clamp
    bool tcl = !(temp >= 1.0f) || temp > RADT_TMAX;
    float T = tcl ? (temp > RADT_TMAX ? RADT_TMAX : 1.0f) : temp;
    float invT = rcp_approx(T);
    float xx = L.T0 * invT;
    float ex = ex2_approx(L.T0l2 * invT);
    float em1 = (xx < 0.0625f)
                    ? xx * fmaf(xx, fmaf(xx, fmaf(xx, fmaf(xx, 1.0f / 120.0f, 1.0f / 24.0f), 1.0f / 6.0f), 0.5f), 1.0f)
                    : ex - 1.0f;
    float S = G.sunit * rcp_approx(em1);
    float invalpha = rsqrt_approx(fmaf(L.a1, T, L.a0));
    float tq = fminf(lg2_approx(T) * ((float)RADT_NQ / RADT_NQ_OCTAVES), (float)RADT_NQ);
    int iq = min(max(rn_int(tq - 0.5f), 0), RADT_NQ);
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
        double yr = rsqrt_d(rho2);
        double vk2 = G.gm_au_d * r2 * yr * yr * yr;
        double vk_d = vk2 * rsqrt_d(fmax(vk2, 1e-300));
        vk = (float)vk_d;
        vphi_d = vk_d * (1.0 + vel_d);
    }
    double vlos_d = vphi_d * proj_d;
    st.A = invalpha * RADT_SQRT_LOG2E;
    if (UNI) {
        // channel lattice v_c = v0 + c dv: with c_ref the channel nearest to v_los, u'(c) = u0 + (c - c_ref) dvA
        // and |u0| <= |dvA|/2, so u' carries only the relative rounding of dvA
        double xd = (vlos_d - G.v0) * L.inv_dv;
        if (!(fabs(xd) <= 1.0e6)) xd = xd > 0.0 ? 1.0e6 : -1.0e6;      // (far off the cube: any channel out of range will do)
        double xm = xd + 6755399441055744.0;             // 1.5 2^52: the rounded integer sits in the low word
        st.cref = __double2loint(xm);
        float del = (float)((xm - 6755399441055744.0) - xd);   // c_ref - x
        st.dvA = L.dvf * invalpha;
        st.u0 = del * st.dvA;
        // line window |c - x| <= hw: the channels where dtau = K' 2^(-u'^2) >= 2^-60 (K' < 2^ek from the exponent
        // bits) as long as that keeps the window within 29 channels, so that a pair of steps fits one 32-channel
        // group; otherwise as many channels as fit, but never fewer than dtau >= 2^-40 asks for
        int ek = max(((__float_as_int(K2) >> 23) & 255) - 126, 0);
        float ca = L.c_hw * (fmaf(L.a1, T, L.a0) * invalpha);          // channels per unit of u'
        float ul = 14.0f * rcp_approx(ca);
        float U2 = fmaxf(UWIN2_MIN + (float)ek, fminf(UWIN2_MAX + (float)ek, ul * ul));
        // the 2^-40 window is wider than a 32-channel group: the step runs over the fixed 32-channel blocks whatever its cut,
        // so it takes the full 2^-60 window (a scene whose whole velocity gradient came from the far wings of very wide lines,
        // 2 channels of 0.02 km/s under a 0.4 km/s line, showed the relaxed cut at 5e-3 of that - tiny - gradient: random scene
        // 764).  Windows of 30-32 channels keep the relaxed cut: they still fit one group (frequent among the optically thick steps of configs 3 and 5:
        // taking the full window there too cost 14 % of the config-5 step).
        {
            const float u16 = 15.5f * rcp_approx(ca);
            if (UWIN2_MIN + (float)ek > u16 * u16) U2 = UWIN2_MAX + (float)ek;
        }
        float hw = fminf(sqrt_approx(U2) * ca, 1.0e6f);
        if (!P.opt_window) hw = 1.0e6f;
        // channels with |c - x| <= hw, x = c_ref - del: floor(y) = rn(y - 1/2) up to ties, which sit on the cut
        st.wlo = st.cref - rn_int(del + hw - 0.5f);
        st.whi = st.cref + rn_int(hw - del - 0.5f);
    } else {
        float vh = (float)vlos_d;
        float vl = (float)(vlos_d - (double)vh);
        st.vh = vh;
        st.mvlA = -vl * st.A;
    }
    st.K2 = K2;
    st.S = S;
    if (!FWD) {
        // chain rule of O11 (SURVEY.md section 8(a) row i) as coefficients of the channel sums.  The lane sums are moments
        // of w = a g in log2 units: sum a dtau u^m = K sum w u'^m / log2(e)^(m/2), K = K2 / log2(e).
        const float iL2 = RADT_LN2;                       // 1 / log2(e)
        const float ia = invalpha;
        const float qy = lerp1(q0.y, q1.y, fq) * iQ;      // dlnQ/dlnT
        const float cdn = (L.Ck2 * iL2) * W * em1 * dsf * ia;          // dK/dn (valid at n = 0)
        st.cd = (g.dens_mode == 1) ? cdn * n : cdn;
        const float K = K2 * iL2;
        const float iT2 = invT * invT;
        const float iem1 = rcp_approx(em1);
        const float exs = em1 + 1.0f;                     // e^x, consistent with the series branch
        const float dlnF_dT = L.Eu * iT2 - L.T0 * iT2 * exs * iem1 - qy * invT;
        const float dS_dT = S * exs * iem1 * L.T0 * iT2;
        const float dalpha_dT = 0.5f * L.a1 * ia;
        // dL/dT = A0 K dlnF/dT + ia (2 A2 - A0 K) dalpha/dT + Bs dS/dT; zero through the 1 K clamp
        st.cT0 = tcl ? 0.f : K * (dlnF_dT - ia * dalpha_dT);
        st.cT2 = tcl ? 0.f : 2.0f * ia * dalpha_dT * K2 * (iL2 * iL2);
        st.cT3 = tcl ? 0.f : dS_dT;
        // dL/dv_phi = (2/alpha) A1 proj (v_K for KEPLER_FRAC), A1 = K2 sum_wu / (log2(e) sqrt(log2(e)))
        st.cv = 2.0f * ia * K2 * (iL2 / RADT_SQRT_LOG2E) * proj * vk;
    }
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
__device__ __forceinline__ void pair_eval(f2 u, f2 K2, Pair &s)
{
    s.u = u;
    float t0, t1;
    upk(mul2(u, u), t0, t1);
    s.g = pk(ex2_approx(-t0), ex2_approx(-t1));
    s.d = mul2(s.g, K2);
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
__device__ __forceinline__ void pair_eval(f2 u, float K2, Pair &s) { pair_eval(u, pk1(K2), s); }
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

// k-th index of 0..n-1 in centre-out order: c, c-1, c+1, c-2, ... with c = n/2 (a bijection for any n)
__device__ __forceinline__ int centre_out(int k, int n)
{
    const int c = n >> 1, h = (k + 1) >> 1;
    int t = (k & 1) ? c - h : c + h;
    // one side runs out first when n is even (c + h reaches n): the remaining indices continue on the other side
    if (t >= n) t = n - 1 - k;
    if (t < 0) t = k;
    return t;
}

__device__ __forceinline__ bool ray_setup(const MarchParams &P, RayCtx &rc, int warp)
{
    // Tiles are issued from the image centre outwards (rows, and tiles within a row, alternate around the centre):
    // rays through the disk centre carry the most steps, the empty corners fill the tail of the launch
    // (measured on config 2: under 1 % either way; kept because the heavy tiles no longer depend on the PA).
    const int kx = blockIdx.x, ky = blockIdx.y + P.tile_y0;     // grid = (tiles_x, tile rows of this launch, batch chunk)
    int tx = centre_out(kx, P.tiles_x), ty = P.banded ? ky : centre_out(ky, P.tiles_y);
    rc.b = blockIdx.z;
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

// Fused chi^2 data term: a warp adds the squared residuals of its ray to one
// of RADT_LOSS_SLOTS double slots with a fire-and-forget reduction; k_loss_finish (radt_setup.cu) sums the slots
// after the last march launch of the call.  The ray's target row is prefetched to L2 before the march.
__device__ __forceinline__ void loss_prefetch(const MarchParams &P, size_t row, int nchan, int lane)
{
    if (lane * 32 < nchan) asm volatile("prefetch.global.L2 [%0];" ::"l"(P.target + row + lane * 32));
}
__device__ __forceinline__ void loss_report(const MarchParams &P, double acc, int lane)
{
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) acc += __shfl_xor_sync(FULL, acc, m);
    if (lane == 0 && acc != 0.0) {
        double *part = reinterpret_cast<double *>(P.ws.counters + 8);
        const unsigned w = ((blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * RADT_WARPS_PER_CTA + (threadIdx.x >> 5);
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(part + (w & (RADT_LOSS_SLOTS - 1))), "d"(acc) : "memory");
    }
}
// residual of one voxel: writes dL/dcube, returns r^2
__device__ __forceinline__ double loss_voxel(const MarchParams &P, size_t idx, float I)
{
    const float r = I - __ldg(P.target + idx);
    P.dl_out[idx] = r * P.inv_s2n;
    return (double)r * (double)r;
}

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


// ---------------------------------------------------------------------------------------------
// phase C of the adjoint (lane = step): chain rule from the four channel sums sm = {sum w, sum w u', sum w u'^2,
// sum G (1-e) T} (w = dL/d dtau g) to (n, T, v_phi) and scatter to the packed gradient cells (O11,
// SURVEY.md section 8(a) rows i-j).  Zero-opacity steps (isE false) carry dL/dn only.
// ---------------------------------------------------------------------------------------------
template <int KIND>
__device__ __forceinline__ void phase_c(const MarchParams &P, const StepState &st, const float4 sm, const bool isE,
                                        float4 *__restrict__ grad)
{
    const float dL_dd = sm.x * st.cd;
    float4 *gp = grad + st.cell;
    if (isE) {
        const float dL_dT = fmaf(sm.x, st.cT0, fmaf(sm.z, st.cT2, sm.w * st.cT3));
        const float dL_dv = sm.y * st.cv;
        if (KIND == 0) {
            float fu = st.f0, fw = st.f1;
            int n1 = P.grid.n1;
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
                red_add_cell(gp + (dx * sx + dy * sy + dz * st.dk), w, dL_dd, dL_dT, dL_dv);
            }
        }
    } else {
        if (KIND == 0) {
            float fu = st.f0, fw = st.f1;
            int n1 = P.grid.n1;
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
                red_add_dens(gp + (dx * sx + dy * sy + dz * st.dk), w * dL_dd);
            }
        }
    }
}
