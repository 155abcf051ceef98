// radt_march.cu -- forward march (K2/K3) and memory-free adjoint march (K4/K5) for sm_100a.
//
// Mapping: one warp per ray.  Every 32-step block runs in two phases:
//   phase A  lanes over STEPS   : position (fp64), grid lookup, LTE thermodynamics -> 4 scalars/step
//   phase B  lanes over CHANNELS: for each active step, broadcast the 4 scalars from shared memory,
//                                 2 x MUFU.EX2 per (channel, step) sample, accumulate in registers
//   phase C  (adjoint) lanes over STEPS again: chain rule + vector atomics into the packed gradient.
// Algorithm: DESIGN.md O4-O11; PAPER.md:262-294 (Eq. 11-17).
#include "radt_march.cuh"


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
// COMP (the caller passed cube_lo): the rounding errors of every I += c are collected in a low-order word per channel,
// which the adjoint uses to form R_k = I - I_{<=k} without the cancellation noise of the fp32 sum.
template <int KIND, int NP, bool CL, bool COMP>
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
    if (P.target) loss_prefetch(P, rc.ray * (size_t)nchan, nchan, lane);
    f2 I[NP], T[NP], vcs[NP], vcl[NP], Lw[COMP ? NP : 1];
    float vmin, vmax;
    load_channels<NP>(P.ws.vcs + (size_t)(P.b0 + rc.b) * RADT_MAXCHAN, nchan, lane, vcs, vcl, vmin, vmax);
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        I[p] = pk(0.f, 0.f); T[p] = pk(1.f, 1.f);
        if (COMP) Lw[p] = pk(0.f, 0.f);
    }
    unsigned n_steps = 0, n_mufu = 0;
    if (rc.ds != 0.0) {
        const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
        // only the 32-step blocks that can hold in-grid samples (K1's conservative step range)
        for (int kb = rc.k_lo & ~31; kb < rc.k_hi; kb += 32) {
            StepState st;
            phase_a<KIND, true, false>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, kb + lane, st);
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
                    const f2 m = mul2(s.om, T[p]);
                    const f2 In = fma2(S2, m, I[p]);
                    // rounding error of In = fl(S m + I): I - In is exact whenever the contribution is small against the
                    // sum, which is when it matters
                    if (COMP) Lw[p] = add2(Lw[p], fma2(S2, m, sub2(I[p], In)));
                    I[p] = In;
                    T[p] = mul2(T[p], s.e);
                }
            }
            __syncwarp();
        }
    }
    double r2 = 0.0;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        int c0 = lane + 64 * p, c1 = c0 + 32;
        float i0, i1;
        upk(I[p], i0, i1);
        if (c0 < nchan) out[c0] = i0;
        if (c1 < nchan) out[c1] = i1;
        if (COMP) {
            float l0, l1;
            upk(Lw[p], l0, l1);
            float *lo = P.cube_lo + rc.ray * (size_t)nchan;
            if (c0 < nchan) lo[c0] = l0;
            if (c1 < nchan) lo[c1] = l1;
        }
        if (P.target) {
            if (c0 < nchan) r2 += loss_voxel(P, rc.ray * (size_t)nchan + c0, i0);
            if (c1 < nchan) r2 += loss_voxel(P, rc.ray * (size_t)nchan + c1, i1);
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
// Steps come in two kinds: E (emitting, K > 0) update the transmittance and the partial sums and feed all four
// channel sums; Z (zero opacity, LINEAR density grids) leave the ray state untouched and feed dL/dn only.
// Channel sums are written per lane to shared memory and reduced for RADT_NS steps at a time.
// ---------------------------------------------------------------------------------------------
#define RADT_NS 8

template <int NP, bool CL, bool COMP, int NQ>
__device__ __forceinline__ float4 bwd_estep(const float4 q, const float S, const float nsmax, const bool window,
                                            f2 (&T)[NP], f2 (&Pp)[NP], f2 (&Qp)[NQ], const f2 (&Isv)[NP], const f2 (&Ilo)[NQ],
                                            const f2 (&Gc)[NP], const f2 (&vcs)[NP], const f2 (&vcl)[NP], unsigned &n_mufu)
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
        const f2 Pn = fma2(S2, omT, Pp[p]);           // = the forward's partial sum I_{<=k}, bit for bit
        f2 PmI = sub2(Pn, Isv[p]);
        if (COMP) {
            // the same error words the forward collected, so that P + Q tracks the exact partial sum
            Qp[p] = add2(Qp[p], fma2(S2, omT, sub2(Pp[p], Pn)));
            PmI = add2(PmI, sub2(Qp[p], Ilo[p]));
        }
        Pp[p] = Pn;
        f2 Tn = mul2(T[p], s.e);
        f2 nR = clamp_nR(PmI, Tn, nsm2);
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

template <int KIND, int NP, bool CL, bool COMP>
__global__ void __launch_bounds__(RADT_WARPS_PER_CTA * 32, (COMP && NP == 4) ? 4 : 6) k_march_bwd(const __grid_constant__ MarchParams P)
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
    constexpr int NQ = COMP ? NP : 1;
    f2 Isv[NP], Pp[NP], T[NP], vcs[NP], vcl[NP], Gc[NP], Qp[NQ], Ilo[NQ];
    const float *Lsave = COMP ? P.cube_lo + rc.ray * (size_t)nchan : nullptr;
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
        if (COMP) {
            Qp[p] = pk(0.f, 0.f);
            Ilo[p] = pk(ok0 ? __ldg(Lsave + c0) : 0.f, ok1 ? __ldg(Lsave + c1) : 0.f);
        }
        Gc[p] = pk(g0, g1);
        anyg |= (g0 != 0.f) || (g1 != 0.f);
    }
    if (!__any_sync(FULL, anyg)) return;     // dL/dcube vanishes on this ray: no gradient
    const float4 *cells = P.ws.cells + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    float4 *grad = P.ws.grad + (size_t)(P.b0 + rc.b) * (size_t)P.grid.cells;
    // upper bound of the source function anywhere on the grid (S grows with T)
    const float tmax = fmaxf(__int_as_float(*reinterpret_cast<const int *>(P.ws.counters + RADT_CNT_TMAX)), 1.0f);
    const float nsmax = -G.sunit * 1.0001f / (ex2_approx(L.T0l2 / tmax) - 1.0f);
    const float kthr = P.opt_skip_empty ? K2_EMPTY : 0.f;    // the forward's own test for an emitting step
    const bool window = P.opt_window;
    unsigned n_steps = 0, n_mufu = 0;
    for (int kb = rc.k_lo & ~31; kb < rc.k_hi; kb += 32) {
        StepState st;
        phase_a<KIND, false, false>(P, G, cells, rc.ox, rc.oy, rc.oz, rc.s0, rc.ds, kb + lane, st);
        const bool isE = st.inside && st.K2 > kthr;
        // zero-opacity steps still carry dL/dn when the grid stores n itself (LINEAR)
        const bool active = st.inside && (isE || (P.grid.dens_mode == 0 && P.opt_zero_grad)) && (!window || line_hits_span(st, vmin, vmax));
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
                    sh_red[warp][jj][lane] = bwd_estep<NP, CL, COMP, NQ>(q, S, nsmax, window, T, Pp, Qp, Isv, Ilo, Gc, vcs, vcl, n_mufu);
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
                    f2 PmI = sub2(Pp[p], Isv[p]);
                    if (COMP) PmI = add2(PmI, sub2(Qp[p], Ilo[p]));
                    GnR[p] = mul2(Gc[p], clamp_nR(PmI, T[p], nsm2));
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
        if (active) phase_c<KIND>(P, st, sh_sum[warp][pos], isE, grad);
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
    dim3 grid(P.tiles_x, P.launch_ty, nbatch);
    const bool comp = P.cube_lo != nullptr;
    if (P.chan_lo && comp) k_march_fwd<KIND, NP, true, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else if (P.chan_lo) k_march_fwd<KIND, NP, true, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else if (comp) k_march_fwd<KIND, NP, false, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else k_march_fwd<KIND, NP, false, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    return cudaGetLastError();
}

template <int KIND, int NP>
static cudaError_t launch_bwd_t(const MarchParams &P, int nbatch, cudaStream_t st)
{
    dim3 grid(P.tiles_x, P.launch_ty, nbatch);
    const bool comp = P.cube_lo != nullptr;
    if (P.chan_lo && comp) k_march_bwd<KIND, NP, true, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else if (P.chan_lo) k_march_bwd<KIND, NP, true, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else if (comp) k_march_bwd<KIND, NP, false, true><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    else k_march_bwd<KIND, NP, false, false><<<grid, RADT_WARPS_PER_CTA * 32, 0, st>>>(P);
    return cudaGetLastError();
}

#define RADT_DISPATCH(fn)                                                        \
    int np = (P.line.ngroups + 1) / 2;                                           \
    if (P.grid.kind == 0) {                                                      \
        if (np <= 1) return fn<0, 1>(P, nbatch, st);                             \
        if (np <= 2) return fn<0, 2>(P, nbatch, st);                             \
        return fn<0, 4>(P, nbatch, st);                                          \
    }                                                                            \
    if (P.grid.kind == 2) {                                                      \
        if (np <= 1) return fn<2, 1>(P, nbatch, st);                             \
        if (np <= 2) return fn<2, 2>(P, nbatch, st);                             \
        return fn<2, 4>(P, nbatch, st);                                          \
    }                                                                            \
    if (np <= 1) return fn<1, 1>(P, nbatch, st);                                 \
    if (np <= 2) return fn<1, 2>(P, nbatch, st);                                 \
    return fn<1, 4>(P, nbatch, st);

cudaError_t radt_launch_march_fwd(const MarchParams &P, int nbatch, cudaStream_t st) { RADT_DISPATCH(launch_fwd_t) }
cudaError_t radt_launch_march_bwd(const MarchParams &P, int nbatch, cudaStream_t st) { RADT_DISPATCH(launch_bwd_t) }
