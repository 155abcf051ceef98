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

#ifndef RADT_WIN_MINB_FWD
#define RADT_WIN_MINB_FWD 8     // CTAs (of 4 warps) per SM the kernels are compiled for: 64 and 80 registers per thread
                                // (measured: 72 registers and 7 CTAs for the adjoint is slower, the spills cost more)
#endif
#ifndef RADT_WIN_MINB_BWD
#define RADT_WIN_MINB_BWD 6
#endif
#define WIN_PAIRS 16         // slot pairs per batch of 32 steps
#define NO_GROUP 0x7fffffff

struct __align__(16) WinShared {          // per warp
    float4 a[WIN_PAIRS];                  // {u0_a, u0_b, dvA_a, dvA_b}
    float4 b[WIN_PAIRS];                  // {K2_a, K2_b, S_a, S_b}
    float4 c[WIN_PAIRS];                  // {c_ref_a, c_ref_b, bits of u_lo, bits of 31 - (u_hi - u_lo)}: union window of the pair
    int cand[64];                         // candidate step indices waiting for phase A (circular queue)
    int2 win[32];                         // channel windows of the compacted steps
    double ray[6];                        // ox, oy, oz, s0, ds of the ray (fp64: read once per batch by phase A)
};

// fp32 copy of the ray for the prefilter (the grid mapping and the ray direction come as fp32 kernel parameters)
struct PreRay {
    float ox, oy, oz, s0, ds;
};

// Can step k lie in a cell that matters?  A superset test in fp32: positions are good to ~1e-4 au, the test
// accepts one cell of margin around the grid and the bitmap is dilated accordingly (radt_setup.cu).
template <int KIND>
__device__ __forceinline__ bool prefilter(const MarchParams &P, const DevGeom &G, const PreRay &pr, const unsigned *__restrict__ occ,
                                          int k)
{
    const DevGrid &g = P.grid;
    const float s = fmaf((float)k + 0.5f, pr.ds, pr.s0);
    const float x = fmaf(s, G.wxf, pr.ox), y = fmaf(s, G.wyf, pr.oy), z = fmaf(s, G.wzf, pr.oz);
    if (KIND == 0) {
        const float r2 = fmaxf(fmaf(x, x, y * y), 1e-30f);
        const float zr = z * rsqrt_approx(r2);
        const float uf = fmaf(lg2_approx(r2), g.pre_us_half, g.pre_uoff);
        const float wf = fmaf(g.mirror ? fabsf(zr) : zr, g.pre_wscale, g.pre_woff);
        const bool in = uf > -1.0f && uf < g.pre_n0f && wf > -1.0f && wf < g.pre_n1f;
        if (!in) return false;
        if (!P.use_occ) return true;
        // bit (I, J) = (floor(u) + 1, floor(w) + 1): no clamps, the bitmap has the extra row and column
        const int I = rn_int(uf + 0.5f), J = rn_int(wf + 0.5f);
        const unsigned w = __ldg(occ + (I * P.occ_wpr + (J >> 5)));
        return (w >> (J & 31)) & 1u;
    } else if (KIND == 2) {
        const float rho2 = fmaxf(fmaf(x, x, fmaf(y, y, z * z)), 1e-30f);
        const float cz = z * rsqrt_approx(rho2);
        const float uf = fmaf(lg2_approx(rho2), g.pre_us_half, g.pre_uoff);
        const bool in = uf > -1.0f && uf < g.pre_n0f && cz > g.pre_czlo && cz < g.pre_czhi;
        if (!in) return false;
        if (!P.use_occ) return true;
        // bit (I, C) = (floor(u) + 1, bin of cos theta), any phi
        const int I = rn_int(uf + 0.5f), C = rn_int(fmaf(cz - g.pre_czlo, g.pre_cscale, -0.5f));
        const unsigned w = __ldg(occ + (I * P.occ_wpr + (C >> 5)));
        return (w >> (C & 31)) & 1u;
    } else {
        const float tx = (x - g.pre_lo[0]) * g.pre_inv_d[0], ty = (y - g.pre_lo[1]) * g.pre_inv_d[1],
                    tz = (z - g.pre_lo[2]) * g.pre_inv_d[2];
        const bool in = tx > -1.0f && tx < g.pre_n0f && ty > -1.0f && ty < g.pre_n1f && tz > -1.0f && tz < g.pre_n2f;
        if (!in) return false;
        if (!P.use_occ) return true;
        const int I = min(max(rn_int(tx - 0.5f), 0), g.n0 - 2) >> 2;
        const int J = min(max(rn_int(ty - 0.5f), 0), g.n1 - 2) >> 2;
        const int Lb = min(max(rn_int(tz - 0.5f), 0), g.n2 - 2) >> 2;
        const unsigned w = __ldg(occ + ((I * P.occ_nbj + J) * P.occ_wpr + (Lb >> 5)));
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
            fc[q + 3] = __int_as_float(31 - (uhi - ulo));
            if (pos == cnt - 1) { fa[q + 1] = 0.f; fa[q + 3] = 0.f; fb[q + 1] = 0.f; fb[q + 3] = 0.f; fc[q + 1] = 0.f; }
        }
    }
    __syncwarp();
    return (cnt + 1) >> 1;
}

// The pair's union window [ulo, uhi] (given as ulo and lim = 31 - (uhi - ulo) >= 0) no longer fits the current group
// [cur, cur + 32)?  It fits iff 0 <= ulo - cur <= lim: one unsigned comparison (cur = NO_GROUP always misses).
__device__ __forceinline__ bool group_misses(int cur, int ulo, int lim) { return (unsigned)(ulo - cur) > (unsigned)lim; }
// New group for that union: centred, so that the line can drift either way before the lanes change channel again.
__device__ __forceinline__ int group_for(int ulo, int lim) { return ulo - (lim >> 1); }

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
    Ts = __fmul_rn(Ts, e0);
    const float m1 = __fmul_rn(om1, Ts);
    const float I2 = __fmaf_rn(qb.w, m1, I1);
    if (COMP) {
        // rounding errors of I1 = fl(S m + Is) and I2: Is - I1 is exact whenever the contribution is small against the
        // sum, which is when it matters; both steps in one packed subtraction and one packed fma (the same values as the
        // adjoint's scalar ones)
        float r0, r1;
        upk(fma2(pk(qb.z, qb.w), pk(m0, m1), sub2(pk(Is, I1), pk(I1, I2))), r0, r1);
        Ls = (Ls + r0) + r1;
    }
    Is = I2;
    Ts = __fmul_rn(Ts, e1);
}

// Candidate steps of the ray, compacted over 32-step blocks into a circular queue of 64 entries (head `ch`, `ncand` waiting):
// filled until it holds >= 32 or the ray ends.
template <int KIND>
__device__ __forceinline__ void gather_candidates(const MarchParams &P, const DevGeom &G, const PreRay &pr, const unsigned *occ,
                                                  WinShared &S, int k_lo, int k_hi, int lane, int ch, int &ncand, int &kb)
{
    const unsigned lt = (1u << lane) - 1u;
    while (ncand < 32 && kb < k_hi) {
        const int k = kb + lane;
        const bool cnd = k >= k_lo && k < k_hi && prefilter<KIND>(P, G, pr, occ, k);
        const unsigned m = __ballot_sync(FULL, cnd);
        if (cnd) S.cand[(ch + ncand + __popc(m & lt)) & 63] = k;
        ncand += __popc(m);
        kb += 32;
    }
}

// Take up to 32 candidates (march order) from the head of the queue; lanes beyond the count get k = nstep (outside).
__device__ __forceinline__ int take_candidates(WinShared &S, int lane, int &ch, int &ncand, int nstep)
{
    __syncwarp();
    const int n = min(ncand, 32);
    const int k = lane < n ? S.cand[(ch + lane) & 63] : nstep;
    __syncwarp();                   // the next fill may wrap around onto the slots just read
    ch = (ch + n) & 63;
    ncand -= n;
    return k;
}

// The ray's fp64 origin and interval go to shared memory (phase A reads them once per batch); the prefilter keeps fp32 copies.
__device__ __forceinline__ PreRay stash_ray(WinShared &S, const RayCtx &rc, int lane)
{
    if (lane == 0) { S.ray[0] = rc.ox; S.ray[1] = rc.oy; S.ray[2] = rc.oz; S.ray[3] = rc.s0; S.ray[4] = rc.ds; }
    PreRay pr;
    pr.ox = (float)rc.ox; pr.oy = (float)rc.oy; pr.oz = (float)rc.oz; pr.s0 = (float)rc.s0; pr.ds = (float)rc.ds;
    __syncwarp();
    return pr;
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
    unsigned n_steps = 0, n_mufu = 0, n_useful = 0;
    if (rc.ds != 0.0) {
        const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
        const unsigned *occ = P.ws.occ + (size_t)(P.b0 + rc.b) * (size_t)P.occ_words;
        const PreRay pr = stash_ray(S, rc, lane);
        const int k_lo = rc.k_lo, k_hi = rc.k_hi;
        int ncand = 0, ch = 0, kb = k_lo & ~31;
        while (true) {
            gather_candidates<KIND>(P, G, pr, occ, S, k_lo, k_hi, lane, ch, ncand, kb);
            if (ncand == 0) break;
            const int k = take_candidates(S, lane, ch, ncand, P.nstep);

            StepState st;
            phase_a<KIND, true, true>(P, G, cells, S.ray[0], S.ray[1], S.ray[2], S.ray[3], S.ray[4], k, st);
            const bool act = st.inside && (st.K2 > K2_EMPTY || !P.opt_skip_empty) && st.whi >= 0 && st.wlo < nchan;
            n_steps += __popc(__ballot_sync(FULL, act));
            n_useful += __reduce_add_sync(FULL, act ? min(st.whi, nchan - 1) - max(st.wlo, 0) + 1 : 0);
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
                    const int ulo = __float_as_int(qc.z), lim = __float_as_int(qc.w);
                    if (group_misses(L.cur, ulo, lim)) L.regroup(group_for(ulo, lim), lane, nchan);
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
        atomicAdd(P.ws.counters + RADT_CNT_USEFUL, (unsigned long long)n_useful);
    }
}

// ---------------------------------------------------------------------------------------------
// K4 / K5 adjoint march: front-to-back re-march with the saved cube
//   dL/d dtau_k,c = G_c (T_{k+1,c} S_k - R_k,c),  R_k = I - I_{<=k}        dL/dS_k = sum_c G_c (1-e_k,c) T_k,c
// Emitting steps run as pairs with lanes over channels: every lane writes its partial sums {w, w u', w u'^2, G (1-e) T}
// (one float4 per step) to shared memory and after BWD_SUB pairs the lanes sum them over the channels.  Zero-opacity steps
// (LINEAR density grids) leave the ray state untouched, feed dL/dn only and run with lanes over steps (refresh_frozen).
// ---------------------------------------------------------------------------------------------
#define BWD_SUB 4            // pairs per reduction batch

// Per-lane channel state of the adjoint window march: transmittance and partial sum of all channels live in shared
// memory; the saved intensity and dL/dI of the served channel are re-read (L1) when the group moves.
template <bool COMP>
struct BwdLane {
    float Ts, Ps, Is, Gs, cf;                     // transmittance, partial sum, saved I, dL/dI of the served channel
    float Qs;                                     // COMP: low-order word of the partial sum MINUS that of the saved I (the
                                                  // word starts at -I_lo instead of 0: only the difference is ever used)
    int cur, myc;
    float *sT, *sP, *sQ;
    const float *Isave, *Gin;
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
        Qs = 0.f;
        if (myc >= 0) {
            Ts = sT[c]; Ps = sP[c]; Is = __ldg(Isave + c); Gs = __ldg(Gin + c);
            if (COMP) Qs = sQ[c];
        }
        cur = clo;
    }
};

// Partial sums of a reduction batch of BWD_SUB pairs: 4 BWD_SUB rows (pair jj, component q of {w, w u', w u'^2, G (1-e) T}),
// one float2 {step a, step b} per lane, i.e. exactly the packed f32x2 registers the pair evaluation ends with (one
// 8-byte store per component, no repacking).  A row is two half-rows of 16 lanes with 16 bytes of padding after each
// (RED_ROW_BYTES = 288, RED_HALF_BYTES = 144): the 16-byte reads of reduce_steps_e are then free of bank conflicts.
#define RED_ROW_BYTES 288
#define RED_HALF_BYTES 144
#define RED_BYTES (4 * BWD_SUB * RED_ROW_BYTES)

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sts_f2(unsigned addr, f2 v) { asm volatile("st.shared.b64 [%0], %1;" ::"r"(addr), "l"(v) : "memory"); }
__device__ __forceinline__ void lds_2f2(unsigned addr, f2 &a, f2 &b)
{
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr) : "memory");
}

// A pair of emitting steps (or one and a no-op entry).  Repeats the forward's O9 sequence bit for bit (fwd_pair).
// `red_lane` = shared address of this lane's float2 in row 0 of the pair's four rows.
template <bool COMP>
__device__ __forceinline__ void bwd_pair_e(const float4 &qa, const float4 &qb, const float4 &qc, BwdLane<COMP> &L,
                                           float nsmax, unsigned red_lane)
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
    f2 nR = sub2(pk(P0, P1), pk1(L.Is));               // -R = P - I_saved
    if (COMP) {
        // the same error words the forward collected (fwd_pair), so that P + Q tracks the exact partial sum; with
        // them the difference is good to ~1e-14 I and needs no clamp
        const float Q0 = L.Qs + __fmaf_rn(qb.z, c0, __fsub_rn(L.Ps, P0));
        const float Q1 = Q0 + __fmaf_rn(qb.w, c1, __fsub_rn(P0, P1));
        nR = add2(nR, pk(Q0, Q1));
        L.Qs = Q1;
    } else {
        nR = clamp_nR(nR, Tn, pk1(nsmax));
    }
    const f2 a = mul2(G2, fma2(Tn, pk(qb.z, qb.w), nR));          // dL/d dtau
    const f2 w = mul2(a, s.g), wu = mul2(w, s.u);
    sts_f2(red_lane, w);
    sts_f2(red_lane + RED_ROW_BYTES, wu);
    sts_f2(red_lane + 2 * RED_ROW_BYTES, mul2(wu, s.u));
    sts_f2(red_lane + 3 * RED_ROW_BYTES, mul2(G2, pk(c0, c1)));
    L.Ts = T2; L.Ps = P1;
}

// Zero-opacity steps (LINEAR density grids) leave T and P untouched and feed only dL/dn = kappa sum_c (G T S_k - G R) g_c.
// While no emitting step intervenes, G T and G R of every channel are frozen: they are written once to shared memory
// ({G T, -G R} per channel) and a whole run of such steps is then evaluated with LANES OVER STEPS, each lane looping
// over the channels of its own step's line window.  Its sum lands in the lane that runs phase C for that step: no
// partials, no reduction over lanes (the earlier lanes-over-channels pairs cost 41 + 4 instructions per pair; this
// loop costs ~8 per channel for 32 steps at once).
template <bool COMP>
__device__ __forceinline__ void refresh_frozen(BwdLane<COMP> &L, float2 *sF, float nsmax, int ng, int nchan, int lane)
{
    L.put_back();                                  // (channel c is only ever touched by lane c & 31)
    for (int g = 0; g < ng; ++g) {
        const int c = lane + 32 * g;
        if (c < nchan) {
            const float T = L.sT[c], Gc = __ldg(L.Gin + c);
            float nr = L.sP[c] - __ldg(L.Isave + c);
            if (COMP) nr += L.sQ[c];
            else nr = fminf(fmaxf(nr, T * nsmax), 0.f);       // same clamp as clamp_nR
            sF[c] = make_float2(Gc * T, Gc * nr);
        }
    }
    __syncwarp();
}
// sum_c (G T S + (-G R)) g_c over every `stride`-th channel from c0 + q of the window [c0, c1]; u'(c) as in pair_u_win
__device__ __forceinline__ float z_slice_sum(float u0, float dvA, float Ss, int cref, int c0, int c1, int q, int stride,
                                             const float2 *__restrict__ sF)
{
    // two channels (c, c + stride) per trip in packed f32x2 arithmetic; an odd last channel on its own
    int c = c0 + q;
    const float cf0 = (float)(c - cref), df = (float)stride;
    f2 cf2 = pk(cf0, cf0 + df), acc2 = pk1(0.f);
    const f2 d2 = pk1(2.0f * df), dvA2 = pk1(dvA), u02 = pk1(u0), S2 = pk1(Ss);
    for (; c + stride <= c1; c += 2 * stride) {
        const f2 u = fma2(cf2, dvA2, u02);
        float t0, t1;
        upk(mul2(u, u), t0, t1);
        const float2 fa = sF[c], fb = sF[c + stride];
        acc2 = fma2(fma2(pk(fa.x, fb.x), S2, pk(fa.y, fb.y)), pk(ex2_approx(-t0), ex2_approx(-t1)), acc2);
        cf2 = add2(cf2, d2);
    }
    float a0, a1;
    upk(acc2, a0, a1);
    float acc = a0 + a1;
    if (c <= c1) {
        float cfl, dummy;
        upk(cf2, cfl, dummy);
        const float u = fmaf(cfl, dvA, u0);
        const float2 f = sF[c];
        acc = fmaf(fmaf(f.x, Ss, f.y), ex2_approx(-u * u), acc);
    }
    return acc;
}
// A run of m zero-opacity steps (lanes `inrun`, r-th step of the run in lane order): 32 >> ceil(log2 m) lanes share one
// step, each taking a slice of its window; the step's sum returns to the lane that holds the step.
__device__ __forceinline__ float z_run(WinShared &S, const StepState &st, bool inrun, int r, int m, const float2 *__restrict__ sF,
                                       int nchan, int lane, unsigned &n_mufu)
{
    const int c0 = max(st.wlo, 0), c1 = min(st.whi, nchan - 1);
    if (m > 16) {                                    // one lane per step
        const float v = inrun ? z_slice_sum(st.u0, st.dvA, st.S, st.cref, c0, c1, 0, 1, sF) : 0.f;
        n_mufu += __reduce_max_sync(FULL, inrun ? c1 - c0 + 1 : 0);
        return v;
    }
    const int sh = 5 - (32 - __clz(m - 1));          // log2 of the lanes per step: m = 1 -> 5, 2 -> 4, 3..4 -> 3, ... 9..16 -> 1
    if (inrun) {
        S.a[r] = make_float4(st.u0, st.dvA, st.S, (float)st.cref);       // (|c_ref| <= 1e6: exact)
        S.win[r] = make_int2(c0, c1);
    }
    __syncwarp();
    const int myr = lane >> sh, q = lane & ((1 << sh) - 1);
    float acc = 0.f;
    int trips = 0;
    if (myr < m) {
        const float4 e = S.a[myr];
        const int2 w = S.win[myr];
        acc = z_slice_sum(e.x, e.y, e.z, (int)e.w, w.x, w.y, q, 1 << sh, sF);
        trips = (w.y - w.x - q + (1 << sh)) >> sh;
    }
    n_mufu += __reduce_max_sync(FULL, max(trips, 0));
    for (int o = (1 << sh) >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(FULL, acc, o);
    const float v = __shfl_sync(FULL, acc, (r << sh) & 31);
    __syncwarp();
    return v;
}

// Sum the partials of nb <= BWD_SUB pairs over the 32 lanes.  Lane l adds the 16 source lanes of half (l & 1) of row
// l >> 1 (eight 16-byte reads, packed adds), one shuffle round joins the halves, and the even lane of a row stores the two
// sums {step a, step b} of (pair jj = row >> 2, component q = row & 3) into sum[2 (base_i + jj) + {0, 1}].q.
__device__ __forceinline__ void reduce_steps_e(unsigned red, int nb, float *sum_base, int lane)
{
    const unsigned src = red + (lane >> 1) * RED_ROW_BYTES + (lane & 1) * RED_HALF_BYTES;
    f2 a, b;
    lds_2f2(src, a, b);
#pragma unroll
    for (int i = 1; i < 8; ++i) {
        f2 c, d;
        lds_2f2(src + 16 * i, c, d);
        a = add2(a, c); b = add2(b, d);
    }
    a = add2(a, b);
    float x, y;
    upk(a, x, y);
    x += __shfl_xor_sync(FULL, x, 1);
    y += __shfl_xor_sync(FULL, y, 1);
    const int jj = lane >> 3, q = (lane >> 1) & 3;
    if (!(lane & 1) && jj < nb) {
        sum_base[8 * jj + q] = x;
        sum_base[8 * jj + 4 + q] = y;
    }
}

struct __align__(16) BwdShared {          // per warp, followed by (T, P[, Q]) and the frozen {G T, -G R} of 32 ngroups channels
    WinShared w;
    unsigned char red[RED_BYTES];         // partial sums of a reduction batch (layout above)
    float4 sum[32];                       // channel sums of the compacted steps
};
#define BWD_CHAN_BYTES(comp) ((comp) ? 640 : 512)      // per 32 channels: T, P (, Q) floats and {G T, -G R} float2
static size_t bwd_warp_bytes(int ng, bool comp) { return sizeof(BwdShared) + (size_t)ng * BWD_CHAN_BYTES(comp); }

template <int KIND, bool COMP>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32, RADT_WIN_MINB_BWD) k_march_bwd_w(const __grid_constant__ MarchParams P)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    RayCtx rc;
    if (!ray_setup(P, rc, warp)) return;
    if (rc.ds == 0.0) return;
    const int ng = P.line.ngroups;
    unsigned char *base = win_smem + (size_t)warp * (sizeof(BwdShared) + (size_t)ng * BWD_CHAN_BYTES(COMP));
    BwdShared &B = *reinterpret_cast<BwdShared *>(base);
    WinShared &S = B.w;
    const DevGeom &G = P.geom[rc.b];
    const DevLine &Ln = P.line;
    const int nchan = Ln.nchan;
    BwdLane<COMP> L;
    L.sT = reinterpret_cast<float *>(base + sizeof(BwdShared)); L.sP = L.sT + 32 * ng; L.sQ = L.sP + 32 * ng;
    float2 *sF = reinterpret_cast<float2 *>(L.sP + (COMP ? 64 : 32) * ng);
    L.Isave = P.cube + rc.ray * (size_t)nchan;
    L.Gin = P.dl_dcube + rc.ray * (size_t)nchan;
    bool anyg = false;
    for (int g = 0; g < ng; ++g) {
        const int c = lane + 32 * g;
        L.sT[c] = 1.f; L.sP[c] = 0.f;
        if (COMP) L.sQ[c] = c < nchan ? -__ldg(P.cube_lo + rc.ray * (size_t)nchan + c) : 0.f;
        anyg |= c < nchan && __ldg(L.Gin + c) != 0.f;
    }
    L.Ts = 1.f; L.Ps = 0.f; L.Is = 0.f; L.Gs = 0.f; L.cf = 0.f; L.Qs = 0.f; L.cur = NO_GROUP; L.myc = -1;
    if (!__any_sync(FULL, anyg)) return;     // dL/dcube vanishes on this ray: no gradient
    const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    const unsigned *occ = P.ws.occ + (size_t)(P.b0 + rc.b) * (size_t)P.occ_words;
    float4 *grad = P.ws.grad + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    // upper bound of the source function anywhere on the grid (S grows with T)
    const float tmax = fmaxf(__int_as_float(*reinterpret_cast<const int *>(P.ws.counters + RADT_CNT_TMAX)), 1.0f);
    const float nsmax = -G.sunit * 1.0001f / (ex2_approx(Ln.T0l2 / tmax) - 1.0f);
    const float kthr = P.opt_skip_empty ? K2_EMPTY : 0.f;    // the forward's own test for an emitting step
    const bool zsteps = P.grid.dens_mode == 0 && P.opt_zero_grad;      // zero-opacity steps carry dL/dn (LINEAR grids)
    const PreRay pr = stash_ray(S, rc, lane);
    const int k_lo = rc.k_lo, k_hi = rc.k_hi;
    const unsigned lt = (1u << lane) - 1u;
    const unsigned red0 = smem_u32(B.red), red_lane = red0 + (lane >> 4) * RED_HALF_BYTES + (lane & 15) * 8;
    unsigned n_steps = 0, n_mufu = 0;
    bool zdirty = true;                      // the frozen {G T, -G R} in shared memory are stale
    int ncand = 0, ch = 0, kb = k_lo & ~31;
    while (true) {
        gather_candidates<KIND>(P, G, pr, occ, S, k_lo, k_hi, lane, ch, ncand, kb);
        if (ncand == 0) break;
        const int k = take_candidates(S, lane, ch, ncand, P.nstep);

        StepState st;
        phase_a<KIND, false, true>(P, G, cells, S.ray[0], S.ray[1], S.ray[2], S.ray[3], S.ray[4], k, st);
        const bool inwin = st.inside && st.whi >= 0 && st.wlo < nchan;
        const bool isE = inwin && st.K2 > kthr;
        const bool isZ = inwin && !isE && zsteps;
        const unsigned emask = __ballot_sync(FULL, isE), zmask = __ballot_sync(FULL, isZ);
        n_steps += __popc(emask | zmask);
        float4 sm = make_float4(0.f, 0.f, 0.f, 0.f);
        // Runs of emitting steps and runs of zero-opacity steps, in march order (lane order): a zero-opacity step sees the
        // ray state left by every emitting step before it.
        unsigned rem = emask | zmask;
#pragma unroll 1
        while (rem) {
            const int first = __ffs(rem) - 1;
            const bool kindE = (emask >> first) & 1u;
            const unsigned other = (kindE ? zmask : emask) & ~((1u << first) - 1u);
            const unsigned run = other ? rem & ((1u << (__ffs(other) - 1)) - 1u) : rem;
            rem &= ~run;
            const bool inrun = (run >> lane) & 1u;
            if (!kindE) {
                if (zdirty) {
                    refresh_frozen<COMP>(L, sF, nsmax, ng, nchan, lane);
                    zdirty = false;
                }
                const float v = z_run(S, st, inrun, __popc(run & lt), __popc(run), sF, nchan, lane, n_mufu);
                if (inrun) sm.x = v;
                continue;
            }
            zdirty = true;
            bool wide;
            int pos;
            int npairs = write_entries(S, lane, inrun, -1, st, st.K2, wide, pos);
            const int npass = wide ? ng : 1;
#pragma unroll 1
            for (int p = 0; p < npass; ++p) {
                bool a = inrun;
                if (wide) {
                    bool w2;
                    a = inrun && st.wlo <= 32 * p + 31 && st.whi >= 32 * p;
                    npairs = write_entries(S, lane, a, 32 * p, st, st.K2, w2, pos);
                }
                if (npairs == 0) continue;
#pragma unroll 1
                for (int base_i = 0; base_i < npairs; base_i += BWD_SUB) {
                    const int nb = min(BWD_SUB, npairs - base_i);
#pragma unroll 1
                    for (int jj = 0; jj < nb; ++jj) {
                        const int i = base_i + jj;
                        const float4 qa = S.a[i], qb = S.b[i], qc = S.c[i];
                        const int ulo = __float_as_int(qc.z), lim = __float_as_int(qc.w);
                        if (group_misses(L.cur, ulo, lim)) L.regroup(group_for(ulo, lim), lane, nchan);
                        bwd_pair_e<COMP>(qa, qb, qc, L, nsmax, red_lane + jj * (4 * RED_ROW_BYTES));
                    }
                    n_mufu += 4 * nb;
                    __syncwarp();
                    reduce_steps_e(red0, nb, reinterpret_cast<float *>(&B.sum[2 * base_i]), lane);
                    __syncwarp();
                }
                if (a) {
                    const float4 v = B.sum[pos];
                    sm.x += v.x; sm.y += v.y; sm.z += v.z; sm.w += v.w;
                }
                __syncwarp();
            }
        }
        // ---- phase C: chain rule to (n, T, v_phi) at this lane's step, scatter to the grid (O11) ----
        if (isE || isZ) phase_c<KIND>(P, st, sm, isE, grad);
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
    dim3 grid(P.tiles_x, P.launch_ty, nbatch);
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
