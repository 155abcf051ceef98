// radt_march_win.cu -- forward march (K2/K3) and adjoint march (K4/K5) on a UNIFORM channel lattice, sm_100a.
//
// The line profile of one ray step touches only the channels within +-6.4 alpha of its v_los (Eq. 15,
// PAPER.md:280): ~21 of 64 channels in config 2.  This path therefore gives every lane ONE channel of the
// step's 32-channel group [c_lo, c_lo + 32) instead of a fixed set of channels:
//   prefilter (lanes over steps, fp32): drop steps that cannot lie in a cell that emits (occupancy bitmap,
//       dilated by one cell), compact the candidates of several 32-step blocks;
//   phase A (lanes over candidate steps): exact fp64 in/out decision, sampling, LTE thermodynamics, the step's
//       channel window and group -> compacted step entries in shared memory, two steps per slot pair;
//   phase B (lanes over channels): per PAIR of steps one packed f32x2 evaluation (4 MUFU.EX2) and the
//       sequential accumulate of O9; the (I, T) of all channels of the ray sit in shared memory, the lane
//       keeps those of the one channel it serves in registers and swaps them when the group moves, which
//       happens only when the next pair's union window no longer fits the current group (hysteresis).
// Steps wider than 32 channels (or RADT_OPT_WINDOW = 0) run one pass per fixed 32-channel block.
// Algorithm: DESIGN.md O4-O11; PAPER.md:262-294 (Eq. 11-17).
#include "radt_march.cuh"

#define RADT_WIN_MINB_FWD 4     // CTAs per SM the kernels are compiled for (measured: 4 vs 3 gives fwd -3 %, bwd +2 %)
#define RADT_WIN_MINB_BWD 3
#define WIN_PAIRS 16         // slot pairs per batch of 32 steps
#define NO_GROUP 0x7fffffff

struct __align__(16) WinShared {          // per warp
    float4 a[WIN_PAIRS];                  // {u0_a, u0_b, dvA_a, dvA_b}
    float4 b[WIN_PAIRS];                  // {K2_a, K2_b, S_a, S_b}
    float4 c[WIN_PAIRS];                  // {c_ref_a, c_ref_b, bits of u_lo, bits of u_hi}: union window of the pair
    int cand[64];                         // candidate step indices waiting for phase A
    int2 win[32];                         // channel windows of the compacted steps
};

// fp32 copy of the ray and of the grid mapping for the prefilter
struct PreCtx {
    float ox, oy, oz, wx, wy, wz, s0, ds;
    float us_half, lrm;                   // u = lg2(r^2) us_half - lrm
    float zlo, wscale;
    float r2lo, r2hi, czlo, czhi;         // spherical: accepted ranges of rho^2 and z/rho, with margins
    float lo[3], inv_d[3];
};

template <int KIND>
__device__ __forceinline__ void pre_setup(const MarchParams &P, const DevGeom &G, const RayCtx &rc, PreCtx &pc)
{
    pc.ox = (float)rc.ox; pc.oy = (float)rc.oy; pc.oz = (float)rc.oz;
    pc.wx = (float)G.wx; pc.wy = (float)G.wy; pc.wz = (float)G.wz;
    pc.s0 = (float)rc.s0; pc.ds = (float)rc.ds;
    if (KIND == 0) {
        pc.us_half = 0.5f * P.grid.uscale;
        pc.lrm = -lg2_approx((float)P.grid.inv_rmin) * P.grid.uscale;
        pc.zlo = (float)P.grid.zlo; pc.wscale = (float)P.grid.wscale_d;
    } else if (KIND == 2) {
        // margins: one percent in radius, two theta cells in z/rho (|d cos| <= |d theta|)
        const float dth = 2.0f / P.grid.th_scale;
        pc.r2lo = (float)P.grid.rmin2 * 0.98f; pc.r2hi = (float)P.grid.rmax2 * 1.02f;
        pc.czlo = (float)P.grid.cos_thi - dth; pc.czhi = (float)P.grid.cos_tlo + dth;
    } else {
#pragma unroll
        for (int a = 0; a < 3; ++a) { pc.lo[a] = (float)P.grid.lo[a]; pc.inv_d[a] = (float)P.grid.inv_d[a]; }
    }
}

// Can step k lie in a cell that matters?  A superset test in fp32: positions are good to ~1e-4 au, the test
// accepts one cell of margin around the grid and the bitmap is dilated by one cell (radt_setup.cu).
template <int KIND>
__device__ __forceinline__ bool prefilter(const MarchParams &P, const PreCtx &pc, const unsigned *__restrict__ occ, int k)
{
    float s = fmaf((float)k + 0.5f, pc.ds, pc.s0);
    float x = fmaf(s, pc.wx, pc.ox), y = fmaf(s, pc.wy, pc.oy), z = fmaf(s, pc.wz, pc.oz);
    if (KIND == 0) {
        float r2 = fmaf(x, x, y * y);
        float ri = rsqrt_approx(fmaxf(r2, 1e-30f));
        float zeta = (P.grid.mirror ? fabsf(z) : z) * ri;
        float uf = fmaf(lg2_approx(fmaxf(r2, 1e-30f)), pc.us_half, -pc.lrm);
        float wf = (zeta - pc.zlo) * pc.wscale;
        bool in = uf > -1.0f && uf < (float)P.grid.n0 && wf > -1.0f && wf < (float)P.grid.n1;
        if (!in) return false;
        if (!P.use_occ) return true;
        int i = min(max(rn_int(uf - 0.5f), 0), P.grid.n0 - 2);
        int j = min(max(rn_int(wf - 0.5f), 0), P.grid.n1 - 2);
        unsigned w = __ldg(occ + i * P.occ_wpr + (j >> 5));
        return (w >> (j & 31)) & 1u;
    } else if (KIND == 2) {
        float rho2 = fmaf(x, x, fmaf(y, y, z * z));
        float cz = z * rsqrt_approx(fmaxf(rho2, 1e-30f));
        return rho2 > pc.r2lo && rho2 < pc.r2hi && cz > pc.czlo && cz < pc.czhi;
    } else {
        float tx = (x - pc.lo[0]) * pc.inv_d[0], ty = (y - pc.lo[1]) * pc.inv_d[1], tz = (z - pc.lo[2]) * pc.inv_d[2];
        bool in = tx > -1.0f && tx < (float)P.grid.n0 && ty > -1.0f && ty < (float)P.grid.n1 && tz > -1.0f &&
                  tz < (float)P.grid.n2;
        if (!in) return false;
        if (!P.use_occ) return true;
        int I = min(max(rn_int(tx - 0.5f), 0), P.grid.n0 - 2) >> 2;
        int J = min(max(rn_int(ty - 0.5f), 0), P.grid.n1 - 2) >> 2;
        int Lb = min(max(rn_int(tz - 0.5f), 0), P.grid.n2 - 2) >> 2;
        unsigned w = __ldg(occ + (I * P.occ_nbj + J) * P.occ_wpr + (Lb >> 5));
        return (w >> (Lb & 31)) & 1u;
    }
}

// Compact the active steps of this batch (march order) into slot pairs {2i, 2i+1}.  A pair is evaluated in ONE
// 32-channel group that must contain the union [ulo, uhi] of its two line windows; the group itself is chosen in
// phase B (hysteresis: the lanes keep their channels while the union still fits).  An odd count is completed with a
// no-op entry (K2 = 0).  Returns the number of pairs; `wide` tells that some pair's union is wider than 32
// channels (the caller then runs one pass per fixed 32-channel block, `blk` >= 0).
__device__ __forceinline__ int write_entries(WinShared &S, int lane, bool act, int blk, const StepState &st, float K2,
                                         bool &wide, int &pos_out)
{
    const unsigned mask = __ballot_sync(FULL, act);
    wide = false;
    if (mask == 0u) return 0;
    const int cnt = __popc(mask);
    const int pos = __popc(mask & ((1u << lane) - 1u));
    pos_out = pos;
    int ulo = blk, uhi = blk + 31;
    if (blk < 0) {
        if (act) S.win[pos] = make_int2(st.wlo, st.whi);
        __syncwarp();
        ulo = st.wlo; uhi = st.whi;
        if (act && (pos ^ 1) < cnt) {
            const int2 pw = S.win[pos ^ 1];
            ulo = min(ulo, pw.x); uhi = max(uhi, pw.y);
        }
        wide = __any_sync(FULL, act && uhi - ulo > 31);
        if (wide) return 0;
    }
    float *fa = reinterpret_cast<float *>(S.a), *fb = reinterpret_cast<float *>(S.b), *fc = reinterpret_cast<float *>(S.c);
    if (act) {
        const int q = (pos >> 1) * 4 + (pos & 1);
        fa[q] = st.u0; fa[q + 2] = st.dvA;
        fb[q] = K2; fb[q + 2] = st.S;
        fc[q] = (float)st.cref;
        if (!(pos & 1)) {
            fc[q + 2] = __int_as_float(ulo);
            fc[q + 3] = __int_as_float(uhi);
            if (pos == cnt - 1) { fa[q + 1] = 0.f; fa[q + 3] = 0.f; fb[q + 1] = 0.f; fb[q + 3] = 0.f; fc[q + 1] = 0.f; }
        }
    }
    __syncwarp();
    return (cnt + 1) >> 1;
}

// The pair's union window [ulo, uhi] no longer fits the current group [cur, cur + 32)?
__device__ __forceinline__ bool group_misses(int cur, int ulo, int uhi) { return ulo < cur || uhi > cur + 31; }
// New group for that union: centred, so that the line can drift either way before the lanes change channel again.
__device__ __forceinline__ int group_for(int ulo, int uhi) { return ulo - ((31 - (uhi - ulo)) >> 1); }

// Per-lane channel state of the forward window march.  The (I, T) of all channels of the ray live in shared
// memory (channel c is only ever touched by lane c & 31); the lane keeps the pair of the ONE channel it serves in
// the current group [cur, cur + 32) in registers.
// COMP (the caller passed cube_lo): the rounding errors of the sum I += c are collected in a low-order word Ls, which the
// adjoint uses to form R_k = I - I_{<=k} without the cancellation noise of the fp32 sum.
template <bool COMP>
struct LaneState {
    float Is, Ts, cf, Ls;
    int cur, myc;
    float *sI, *sT, *sL;
    __device__ __forceinline__ void init(float *sI_, float *sT_, int lane, int ng)
    {
        sI = sI_; sT = sT_; sL = sT_ + 32 * ng;
        for (int g = 0; g < ng; ++g) {
            sI[lane + 32 * g] = 0.f; sT[lane + 32 * g] = 1.f;
            if (COMP) sL[lane + 32 * g] = 0.f;
        }
        Is = 0.f; Ts = 1.f; cf = 0.f; Ls = 0.f; cur = NO_GROUP; myc = -1;
    }
    __device__ __forceinline__ void put_back()
    {
        if (myc >= 0) {
            sI[myc] = Is; sT[myc] = Ts;
            if (COMP) sL[myc] = Ls;
        }
    }
    // the group moved: put the lane's channel state back, take the new channel's
    __device__ __forceinline__ void regroup(int clo, int lane, int nchan)
    {
        put_back();
        const int c = clo + ((lane - clo) & 31);
        myc = (unsigned)c < (unsigned)nchan ? c : -1;
        cf = (float)c;
        Is = 0.f; Ts = 1.f; Ls = 0.f;
        if (myc >= 0) {
            Is = sI[c]; Ts = sT[c];
            if (COMP) Ls = sL[c];
        }
        cur = clo;
    }
};

// u' of the lane's channel (cf, as a float) for the two steps of a pair: u'(c) = u0 + (c - c_ref) dvA
__device__ __forceinline__ f2 pair_u_win(const float4 &qa, const float4 &qc, float cf)
{
    return fma2(sub2(pk1(cf), pk(qc.x, qc.y)), pk(qa.z, qa.w), pk(qa.x, qa.y));
}

// O9 for the two steps of a pair, in march order.  c = S ((1-e) T) and I += c with fixed roundings: the adjoint
// re-march repeats exactly this sequence and so reproduces the partial sums bit for bit.
template <bool COMP>
__device__ __forceinline__ void fwd_pair(const float4 &qa, const float4 &qb, const float4 &qc, float cf, float &Is, float &Ts,
                                         float &Ls)
{
    Pair s;
    pair_eval(pair_u_win(qa, qc, cf), pk(qb.x, qb.y), s);
    float om0, om1, e0, e1;
    upk(s.om, om0, om1);
    upk(s.e, e0, e1);
    const float m0 = __fmul_rn(om0, Ts);
    const float I1 = __fmaf_rn(qb.z, m0, Is);
    // rounding error of I1 = fl(S m + Is): Is - I1 is exact whenever the contribution is small against the sum, which
    // is when it matters
    if (COMP) Ls += __fmaf_rn(qb.z, m0, __fsub_rn(Is, I1));
    Ts = __fmul_rn(Ts, e0);
    const float m1 = __fmul_rn(om1, Ts);
    const float I2 = __fmaf_rn(qb.w, m1, I1);
    if (COMP) Ls += __fmaf_rn(qb.w, m1, __fsub_rn(I1, I2));
    Is = I2;
    Ts = __fmul_rn(Ts, e1);
}

// Candidate steps of the ray, compacted over 32-step blocks: fills S.cand until it holds >= 32 or the ray ends.
template <int KIND>
__device__ __forceinline__ void gather_candidates(const MarchParams &P, const PreCtx &pc, const unsigned *occ, WinShared &S,
                                                  const RayCtx &rc, int lane, int &ncand, int &kb)
{
    const unsigned lt = (1u << lane) - 1u;
    while (ncand < 32 && kb < rc.k_hi) {
        const int k = kb + lane;
        const bool cnd = k >= rc.k_lo && k < rc.k_hi && prefilter<KIND>(P, pc, occ, k);
        const unsigned m = __ballot_sync(FULL, cnd);
        if (cnd) S.cand[ncand + __popc(m & lt)] = k;
        ncand += __popc(m);
        kb += 32;
    }
}

// Take up to 32 candidates (march order) out of S.cand; lanes beyond the count get k = nstep (outside).
__device__ __forceinline__ int take_candidates(WinShared &S, int lane, int &ncand, int nstep)
{
    __syncwarp();
    const int n = min(ncand, 32);
    const int k = lane < n ? S.cand[lane] : nstep;
    const int kx = lane + 32 < ncand ? S.cand[lane + 32] : 0;
    __syncwarp();
    if (lane + 32 < ncand) S.cand[lane] = kx;
    ncand -= n;
    return k;
}

extern __shared__ __align__(16) unsigned char win_smem[];

// ---------------------------------------------------------------------------------------------
// K2 / K3 forward march.  Dynamic shared memory per warp: WinShared + (I, T) of 32 ngroups channels.
// ---------------------------------------------------------------------------------------------
static size_t fwd_warp_bytes(int ng, bool comp) { return sizeof(WinShared) + (size_t)ng * (comp ? 384 : 256); }

template <int KIND, bool COMP>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32, RADT_WIN_MINB_FWD) k_march_fwd_w(const __grid_constant__ MarchParams P)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RayCtx rc;
    if (!ray_setup(P, rc, warp)) return;
    const int ng = P.line.ngroups;
    unsigned char *base = win_smem + (size_t)warp * (sizeof(WinShared) + (size_t)ng * (COMP ? 384 : 256));
    WinShared &S = *reinterpret_cast<WinShared *>(base);
    float *sI = reinterpret_cast<float *>(base + sizeof(WinShared)), *sT = sI + 32 * ng;
    const DevGeom &G = P.geom[rc.b];
    const int nchan = P.line.nchan;
    float *out = P.cube + rc.ray * (size_t)nchan;
    LaneState<COMP> L;
    L.init(sI, sT, lane, ng);
    if (P.target) loss_prefetch(P, rc.ray * (size_t)nchan, nchan, lane);
    unsigned n_steps = 0, n_mufu = 0;
    if (rc.ds != 0.0) {
        const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
        const unsigned *occ = P.ws.occ + (size_t)(P.b0 + rc.b) * (size_t)P.occ_words;
        PreCtx pc;
        pre_setup<KIND>(P, G, rc, pc);
        int ncand = 0, kb = rc.k_lo & ~31;
        while (true) {
            gather_candidates<KIND>(P, pc, occ, S, rc, lane, ncand, kb);
            if (ncand == 0) break;
            const int k = take_candidates(S, lane, ncand, P.nstep);

            StepState st;
            phase_a<KIND, true, true>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, k, st);
            const bool act = st.inside && (st.K2 > K2_EMPTY || !P.opt_skip_empty) && st.whi >= 0 && st.wlo < nchan;
            n_steps += __popc(__ballot_sync(FULL, act));
            bool wide;
            int pos;
            int npairs = write_entries(S, lane, act, -1, st, st.K2, wide, pos);
            const int npass = wide ? ng : 1;
#pragma unroll 1
            for (int p = 0; p < npass; ++p) {
                if (wide) {
                    bool w2;
                    npairs = write_entries(S, lane, act && st.wlo <= 32 * p + 31 && st.whi >= 32 * p, 32 * p, st, st.K2, w2, pos);
                }
                if (npairs == 0) continue;
#pragma unroll 2
                for (int i = 0; i < npairs; ++i) {
                    const float4 qa = S.a[i], qb = S.b[i], qc = S.c[i];
                    const int ulo = __float_as_int(qc.z), uhi = __float_as_int(qc.w);
                    if (group_misses(L.cur, ulo, uhi)) L.regroup(group_for(ulo, uhi), lane, nchan);
                    fwd_pair<COMP>(qa, qb, qc, L.cf, L.Is, L.Ts, L.Ls);
                }
                n_mufu += 4 * npairs;
                __syncwarp();
            }
        }
        L.put_back();
    }
    double r2 = 0.0;
    for (int g = 0; g < ng; ++g) {
        const int c = lane + 32 * g;
        if (c < nchan) {
            const float Ic = sI[c];
            out[c] = Ic;
            if (COMP) P.cube_lo[rc.ray * (size_t)nchan + c] = L.sL[c];
            if (P.target) r2 += loss_voxel(P, rc.ray * (size_t)nchan + c, Ic);
        }
    }
    if (P.target) loss_report(P, r2, lane);
    if (lane == 0 && n_steps) {
        atomicAdd(P.ws.counters + 0, (unsigned long long)n_steps);
        atomicAdd(P.ws.counters + 1, (unsigned long long)n_mufu);
    }
}

// ---------------------------------------------------------------------------------------------
// K4 / K5 adjoint march: front-to-back re-march with the saved cube
//   dL/d dtau_k,c = G_c (T_{k+1,c} S_k - R_k,c),  R_k = I - I_{<=k}        dL/dS_k = sum_c G_c (1-e_k,c) T_k,c
// Entries with K2 = 0 are zero-opacity steps (LINEAR density grids): they leave the ray state untouched and
// feed dL/dn only.  Per step every lane writes its partial sums {w, w u', w u'^2, G (1-e) T} (one float4; one float
// in batches of zero-opacity steps) to shared memory; after BWD_SUB pairs the lanes sum them over the channels.
// ---------------------------------------------------------------------------------------------
#define BWD_SUB 4            // pairs per reduction batch

// Per-lane channel state of the adjoint window march: transmittance and partial sum of all channels live in shared
// memory; the saved intensity and dL/dI of the served channel are re-read (L1) when the group moves.
template <bool COMP>
struct BwdLane {
    float Ts, Ps, Is, Gs, cf;                     // transmittance, partial sum, saved I, dL/dI of the served channel
    float Qs, Ils;                                // COMP: low-order words of the partial sum and of the saved I
    int cur, myc;
    float *sT, *sP, *sQ;
    const float *Isave, *Gin, *Ilo;
    __device__ __forceinline__ void put_back()
    {
        if (myc >= 0) {
            sT[myc] = Ts; sP[myc] = Ps;
            if (COMP) sQ[myc] = Qs;
        }
    }
    __device__ __forceinline__ void regroup(int clo, int lane, int nchan)
    {
        put_back();
        const int c = clo + ((lane - clo) & 31);
        myc = (unsigned)c < (unsigned)nchan ? c : -1;
        cf = (float)c;
        Ts = 1.f; Ps = 0.f; Is = 0.f; Gs = 0.f;    // lanes without a channel contribute nothing (G = 0)
        Qs = 0.f; Ils = 0.f;
        if (myc >= 0) {
            Ts = sT[c]; Ps = sP[c]; Is = __ldg(Isave + c); Gs = __ldg(Gin + c);
            if (COMP) { Qs = sQ[c]; Ils = __ldg(Ilo + c); }
        }
        cur = clo;
    }
    // -R = (P - I) + (P_lo - I_lo) of the served channel
    __device__ __forceinline__ float neg_r() const { return COMP ? (Ps - Is) + (Qs - Ils) : Ps - Is; }
};

// Partial sums of a reduction batch, rows padded by one element so that both the per-lane writes and the per-step
// reads are free of bank conflicts with plain immediate offsets:
//   emitting batches   float4 [2 BWD_SUB steps][33]   {w, w u', w u'^2, G (1-e) T} per (step, lane)
//   zero-opacity runs  float  [32 steps][33]          w per (step, lane)
#define RED_ROW 33
typedef float4 RedBuf[2 * BWD_SUB][RED_ROW];

// A pair with at least one emitting step.  Repeats the forward's O9 sequence bit for bit (fwd_pair).
template <bool COMP>
__device__ __forceinline__ void bwd_pair_e(const float4 &qa, const float4 &qb, const float4 &qc, BwdLane<COMP> &L,
                                           float nsmax, float4 (*red)[RED_ROW], int lane)
{
    Pair s;
    pair_eval(pair_u_win(qa, qc, L.cf), pk(qb.x, qb.y), s);
    float om0, om1, e0, e1;
    upk(s.om, om0, om1);
    upk(s.e, e0, e1);
    const float c0 = __fmul_rn(om0, L.Ts);
    const float P0 = __fmaf_rn(qb.z, c0, L.Ps);
    const float T1 = __fmul_rn(L.Ts, e0);
    const float c1 = __fmul_rn(om1, T1);
    const float P1 = __fmaf_rn(qb.w, c1, P0);
    const float T2 = __fmul_rn(T1, e1);
    const f2 Tn = pk(T1, T2), G2 = pk1(L.Gs);
    f2 PmI = sub2(pk(P0, P1), pk1(L.Is));
    if (COMP) {
        // the same error words the forward collected (fwd_pair), so that P + Q tracks the exact partial sum
        const float Q0 = L.Qs + __fmaf_rn(qb.z, c0, __fsub_rn(L.Ps, P0));
        const float Q1 = Q0 + __fmaf_rn(qb.w, c1, __fsub_rn(P0, P1));
        PmI = add2(PmI, sub2(pk(Q0, Q1), pk1(L.Ils)));
        L.Qs = Q1;
    }
    const f2 nR = clamp_nR(PmI, Tn, pk1(nsmax));
    const f2 a = mul2(G2, fma2(Tn, pk(qb.z, qb.w), nR));          // dL/d dtau
    const f2 w = mul2(a, s.g), wu = mul2(w, s.u), wuu = mul2(wu, s.u), gc = mul2(G2, pk(c0, c1));
    float w0, w1, x0, x1, y0, y1, z0, z1;
    upk(w, w0, w1); upk(wu, x0, x1); upk(wuu, y0, y1); upk(gc, z0, z1);
    red[0][lane] = make_float4(w0, x0, y0, z0);
    red[1][lane] = make_float4(w1, x1, y1, z1);
    L.Ts = T2; L.Ps = P1;
}

// Zero-opacity steps leave T and P untouched, so G T and G R are fixed while the lane keeps its channel; only
// sum w = sum (G T S_k - G R) g is needed.  {GT, GnR} of the served channel:
template <bool COMP>
__device__ __forceinline__ float2 z_frozen(const BwdLane<COMP> &L, float nsmax)
{
    return make_float2(L.Gs * L.Ts, L.Gs * fminf(fmaxf(L.neg_r(), L.Ts * nsmax), 0.f));
}
__device__ __forceinline__ f2 z_pair_w(const float4 &qa, float Sa, float Sb, const float4 &qc, float cf, float2 fr)
{
    const f2 u = pair_u_win(qa, qc, cf);
    float t0, t1;
    upk(mul2(u, u), t0, t1);
    const f2 g = pk(ex2_approx(-t0), ex2_approx(-t1));
    return mul2(fma2(pk1(fr.x), pk(Sa, Sb), pk1(fr.y)), g);
}

// Sum the partials of nb <= BWD_SUB pairs (2 nb steps) over the 32 lanes.  Lane (s = lane & 7, h = lane >> 3) adds
// the source lanes 8h .. 8h+7 of step s, two shuffle rounds combine the four quarters, and lane s < 2 nb stores the
// four sums of step s.
__device__ __forceinline__ void reduce_steps_e(const RedBuf &red, int nb, float4 *out, int lane)
{
    // rows as pairs of packed f32x2: one FADD2 per two sums
    const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(&red[lane & 7][lane & 24]);
    ulonglong2 a = row[0];
#pragma unroll
    for (int i = 1; i < 8; ++i) {
        const ulonglong2 v = row[i];
        a.x = add2(a.x, v.x); a.y = add2(a.y, v.y);
    }
    float4 acc;
    upk(a.x, acc.x, acc.y); upk(a.y, acc.z, acc.w);
#pragma unroll
    for (int m = 8; m <= 16; m <<= 1) {
        acc.x += __shfl_xor_sync(FULL, acc.x, m);
        acc.y += __shfl_xor_sync(FULL, acc.y, m);
        acc.z += __shfl_xor_sync(FULL, acc.z, m);
        acc.w += __shfl_xor_sync(FULL, acc.w, m);
    }
    if (lane < 2 * nb) out[lane] = acc;
}
// A run of nz <= 16 zero-opacity pairs: lane s < 2 nz sums the 32 partials of step s.
__device__ __forceinline__ void reduce_steps_z(const float (*redz)[RED_ROW], int nz, float4 *out, int lane)
{
    if (lane < 2 * nz) {
        const float *row = redz[lane];
        float a0 = row[0], a1 = row[1], a2 = row[2], a3 = row[3];
#pragma unroll
        for (int i = 4; i < 32; i += 4) { a0 += row[i]; a1 += row[i + 1]; a2 += row[i + 2]; a3 += row[i + 3]; }
        out[lane] = make_float4((a0 + a1) + (a2 + a3), 0.f, 0.f, 0.f);
    }
}

struct __align__(16) BwdShared {          // per warp, followed by (T, P) of 32 ngroups channels
    WinShared w;
    RedBuf red;                           // 8 x 33 float4 = 32 x 33 float
    float4 sum[32];                       // channel sums of the compacted steps
};
static size_t bwd_warp_bytes(int ng, bool comp) { return sizeof(BwdShared) + (size_t)ng * (comp ? 384 : 256); }

template <int KIND, bool COMP>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32, RADT_WIN_MINB_BWD) k_march_bwd_w(const __grid_constant__ MarchParams P)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RayCtx rc;
    if (!ray_setup(P, rc, warp)) return;
    if (rc.ds == 0.0) return;
    const int ng = P.line.ngroups;
    unsigned char *base = win_smem + (size_t)warp * (sizeof(BwdShared) + (size_t)ng * (COMP ? 384 : 256));
    BwdShared &B = *reinterpret_cast<BwdShared *>(base);
    WinShared &S = B.w;
    const DevGeom &G = P.geom[rc.b];
    const DevLine &Ln = P.line;
    const int nchan = Ln.nchan;
    BwdLane<COMP> L;
    L.sT = reinterpret_cast<float *>(base + sizeof(BwdShared)); L.sP = L.sT + 32 * ng; L.sQ = L.sP + 32 * ng;
    L.Ilo = P.cube_lo + rc.ray * (size_t)nchan;
    L.Isave = P.cube + rc.ray * (size_t)nchan;
    L.Gin = P.dl_dcube + rc.ray * (size_t)nchan;
    bool anyg = false;
    for (int g = 0; g < ng; ++g) {
        const int c = lane + 32 * g;
        L.sT[c] = 1.f; L.sP[c] = 0.f;
        if (COMP) L.sQ[c] = 0.f;
        anyg |= c < nchan && __ldg(L.Gin + c) != 0.f;
    }
    L.Ts = 1.f; L.Ps = 0.f; L.Is = 0.f; L.Gs = 0.f; L.cf = 0.f; L.Qs = 0.f; L.Ils = 0.f; L.cur = NO_GROUP; L.myc = -1;
    if (!__any_sync(FULL, anyg)) return;     // dL/dcube vanishes on this ray: no gradient
    const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    const unsigned *occ = P.ws.occ + (size_t)(P.b0 + rc.b) * (size_t)P.occ_words;
    float4 *grad = P.ws.grad + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    // upper bound of the source function anywhere on the grid (S grows with T)
    const float tmax = fmaxf(__int_as_float(*reinterpret_cast<const int *>(P.ws.counters + 4)), 1.0f);
    const float nsmax = -G.sunit * 1.0001f / (ex2_approx(Ln.T0l2 / tmax) - 1.0f);
    const float kthr = P.opt_skip_empty ? K2_EMPTY : 0.f;    // the forward's own test for an emitting step
    PreCtx pc;
    pre_setup<KIND>(P, G, rc, pc);
    unsigned n_steps = 0, n_mufu = 0;
    int ncand = 0, kb = rc.k_lo & ~31;
    while (true) {
        gather_candidates<KIND>(P, pc, occ, S, rc, lane, ncand, kb);
        if (ncand == 0) break;
        const int k = take_candidates(S, lane, ncand, P.nstep);

        StepState st;
        phase_a<KIND, false, true>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, k, st);
        const bool isE = st.inside && st.K2 > kthr;
        // zero-opacity steps still carry dL/dn when the grid stores n itself (LINEAR)
        const bool act = st.inside && (isE || (P.grid.dens_mode == 0 && P.opt_zero_grad)) && st.whi >= 0 && st.wlo < nchan;
        const float K2e = isE ? st.K2 : 0.f;
        n_steps += __popc(__ballot_sync(FULL, act));
        bool wide;
        int pos;
        int npairs = write_entries(S, lane, act, -1, st, K2e, wide, pos);
        const int npass = wide ? ng : 1;
        float4 sm = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 1
        for (int p = 0; p < npass; ++p) {
            bool a = act;
            if (wide) {
                bool w2;
                a = act && st.wlo <= 32 * p + 31 && st.whi >= 32 * p;
                npairs = write_entries(S, lane, a, 32 * p, st, K2e, w2, pos);
            }
            if (npairs == 0) continue;
            // pairs that hold an emitting step
            const unsigned emask = __ballot_sync(FULL, lane < npairs && (S.b[lane].x > 0.f || S.b[lane].y > 0.f));
            int base_i = 0;
#pragma unroll 1
            while (base_i < npairs) {
                const unsigned erest = emask >> base_i;
                if (!(erest & 1u)) {
                    // a run of zero-opacity pairs (up to the whole batch): the ray state is frozen
                    const int nz = min(erest ? __ffs(erest) - 1 : 32, npairs - base_i);
                    float (*redz)[RED_ROW] = reinterpret_cast<float (*)[RED_ROW]>(&B.red[0][0]);
                    float2 fr = z_frozen(L, nsmax);
#pragma unroll 1
                    for (int jj = 0; jj < nz; ++jj) {
                        const int i = base_i + jj;
                        const float4 qa = S.a[i], qc = S.c[i];
                        const float2 Sab = *reinterpret_cast<const float2 *>(&S.b[i].z);
                        const int ulo = __float_as_int(qc.z), uhi = __float_as_int(qc.w);
                        if (group_misses(L.cur, ulo, uhi)) {
                            L.regroup(group_for(ulo, uhi), lane, nchan);
                            fr = z_frozen(L, nsmax);
                        }
                        float w0, w1;
                        upk(z_pair_w(qa, Sab.x, Sab.y, qc, L.cf, fr), w0, w1);
                        redz[2 * jj][lane] = w0;
                        redz[2 * jj + 1][lane] = w1;
                    }
                    n_mufu += 2 * nz;
                    __syncwarp();
                    reduce_steps_z(redz, nz, &B.sum[2 * base_i], lane);
                    __syncwarp();
                    base_i += nz;
                    continue;
                }
                // up to BWD_SUB consecutive pairs that hold an emitting step
                const int nb = min(min(BWD_SUB, __ffs(~erest) - 1), npairs - base_i);
#pragma unroll 1
                for (int jj = 0; jj < nb; ++jj) {
                    const int i = base_i + jj;
                    const float4 qa = S.a[i], qb = S.b[i], qc = S.c[i];
                    const int ulo = __float_as_int(qc.z), uhi = __float_as_int(qc.w);
                    if (group_misses(L.cur, ulo, uhi)) L.regroup(group_for(ulo, uhi), lane, nchan);
                    bwd_pair_e<COMP>(qa, qb, qc, L, nsmax, &B.red[2 * jj], lane);
                }
                n_mufu += 4 * nb;
                __syncwarp();
                reduce_steps_e(B.red, nb, &B.sum[2 * base_i], lane);
                __syncwarp();
                base_i += nb;
            }
            if (a) {
                const float4 v = B.sum[pos];
                sm.x += v.x; sm.y += v.y; sm.z += v.z; sm.w += v.w;
            }
            __syncwarp();
        }
        // ---- phase C: chain rule to (n, T, v_phi) at this lane's step, scatter to the grid (O11) ----
        if (act) phase_c<KIND>(P, st, sm, isE, grad);
    }
    if (lane == 0 && n_steps) {
        atomicAdd(P.ws.counters + 2, (unsigned long long)n_steps);
        atomicAdd(P.ws.counters + 3, (unsigned long long)n_mufu);
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
template <typename K>
static cudaError_t launch_w(K kern, const MarchParams &P, int nbatch, size_t warp_bytes, cudaStream_t st)
{
    const size_t smem = warp_bytes * RADT_WARPS_PER_CTA;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(P.tiles_x * P.tiles_y, nbatch);
    kern<<<grid, RADT_WARPS_PER_CTA * 32, smem, st>>>(P);
    return cudaGetLastError();
}

cudaError_t radt_launch_march_fwd_win(const MarchParams &P, int nbatch, cudaStream_t st)
{
    const bool comp = P.cube_lo != nullptr;
    const size_t wb = fwd_warp_bytes(P.line.ngroups, comp);
    if (comp)
        return P.grid.kind == 0 ? launch_w(k_march_fwd_w<0, true>, P, nbatch, wb, st)
             : P.grid.kind == 1 ? launch_w(k_march_fwd_w<1, true>, P, nbatch, wb, st)
                                : launch_w(k_march_fwd_w<2, true>, P, nbatch, wb, st);
    return P.grid.kind == 0 ? launch_w(k_march_fwd_w<0, false>, P, nbatch, wb, st)
         : P.grid.kind == 1 ? launch_w(k_march_fwd_w<1, false>, P, nbatch, wb, st)
                            : launch_w(k_march_fwd_w<2, false>, P, nbatch, wb, st);
}

cudaError_t radt_launch_march_bwd_win(const MarchParams &P, int nbatch, cudaStream_t st)
{
    const bool comp = P.cube_lo != nullptr;
    const size_t wb = bwd_warp_bytes(P.line.ngroups, comp);
    if (comp)
        return P.grid.kind == 0 ? launch_w(k_march_bwd_w<0, true>, P, nbatch, wb, st)
             : P.grid.kind == 1 ? launch_w(k_march_bwd_w<1, true>, P, nbatch, wb, st)
                                : launch_w(k_march_bwd_w<2, true>, P, nbatch, wb, st);
    return P.grid.kind == 0 ? launch_w(k_march_bwd_w<0, false>, P, nbatch, wb, st)
         : P.grid.kind == 1 ? launch_w(k_march_bwd_w<1, false>, P, nbatch, wb, st)
                            : launch_w(k_march_bwd_w<2, false>, P, nbatch, wb, st);
}
