// radt_mlp.cu -- symmetric MLP temperature field on the nodes of the (r, zeta) grid and its adjoint w.r.t. the
// parameters (Eq. 10).  Algorithm M1-M4 of DESIGN.md section 9: normalised grid
// coordinates -> positional encoding of degree L -> 4 x 64 ReLU layers -> sigmoid scaled to [t_lo, t_hi].
// fp32 FMA (packed FFMA2); activations in shared memory ([unit][node], so both the per-node and the per-unit passes
// read without bank conflicts), parameters staged in shared memory and read as warp-wide broadcasts; the hidden
// layers serve two nodes per thread so that each broadcast feeds both.  Shares nothing with oracle/.
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define MLP_W 64                       // hidden width
#define MLP_H 4                        // hidden layers
#define MLP_TF 128                     // nodes per block, forward
#define MLP_TB 64                      // nodes per block, adjoint
#define MLP_S 4                        // threads per node: each computes MLP_W / MLP_S units of a layer
#define MLP_PW (MLP_W / MLP_S)
#define MLP_SA (MLP_TB + 1)            // activation row stride (adjoint): scalar reads by unit are conflict free
#define MLP_SD (MLP_TB + 4)            // delta row stride: 16-byte aligned rows for broadcast float4 reads

// packed f32x2 FMA (sm_100): every dot product below runs as two interleaved partial sums, one FFMA2 per two terms
typedef unsigned long long f2;
__device__ __forceinline__ f2 mlp_pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float mlp_sum2(f2 v) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); return lo + hi; }
__device__ __forceinline__ f2 mlp_fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }

struct MlpOff {
    int W[MLP_H + 1], b[MLP_H + 1], D;
};
__device__ __forceinline__ MlpOff mlp_offsets(int L)
{
    MlpOff o;
    o.D = 2 + 4 * L;
    int off = 0, fan = o.D;
    for (int l = 0; l <= MLP_H; ++l) {
        const int out = l < MLP_H ? MLP_W : 1;
        o.W[l] = off; off += out * fan;
        o.b[l] = off; off += out;
        fan = MLP_W;
    }
    return o;
}

// M1-M2: encoding of node (i, j) into column `node` of act[unit][stride]
__device__ __forceinline__ void mlp_encode(const MlpParamsDev &Q, int i, int j, float *act, int stride, int node)
{
    const float p0 = (float)i / (float)(Q.nr - 1), p1 = (float)j / (float)(Q.nz - 1);
    act[0 * stride + node] = p0;
    act[1 * stride + node] = p1;
    float f = 1.0f;
    for (int k = 0; k < Q.L; ++k) {
        act[(2 + 4 * k + 0) * stride + node] = sinpif(f * p0);
        act[(2 + 4 * k + 1) * stride + node] = cospif(f * p0);
        act[(2 + 4 * k + 2) * stride + node] = sinpif(f * p1);
        act[(2 + 4 * k + 3) * stride + node] = cospif(f * p1);
        f *= 2.0f;
    }
}

// M3, first layer: fan-in D (rows are not 16-byte aligned: scalar uniform loads)
__device__ __forceinline__ void mlp_layer_first(const float *__restrict__ W, const float *__restrict__ b, int D,
                                                const float *in, float *out, int stride, int node, int part)
{
    float h[34];
#pragma unroll
    for (int i = 0; i < 34; ++i) h[i] = i < D ? in[i * stride + node] : 0.f;
#pragma unroll 4
    for (int o = part * MLP_PW; o < (part + 1) * MLP_PW; ++o) {
        float acc = b[o];
#pragma unroll
        for (int i = 0; i < 34; ++i)
            if (i < D) acc = fmaf(W[o * D + i], h[i], acc);
        out[o * stride + node] = fmaxf(acc, 0.f);
    }
}

// M3, hidden layer 64 -> 64: the node's inputs in registers, one output unit at a time, weight rows as float4
__device__ __forceinline__ void mlp_layer(const float *__restrict__ W, const float *__restrict__ b, const float *in,
                                          float *out, int stride, int node, int part)
{
    f2 h[MLP_W / 2];
#pragma unroll
    for (int i = 0; i < MLP_W / 2; ++i) h[i] = mlp_pk(in[2 * i * stride + node], in[(2 * i + 1) * stride + node]);
#pragma unroll 4
    for (int o = part * MLP_PW; o < (part + 1) * MLP_PW; ++o) {
        const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(W + o * MLP_W);
        f2 a0 = mlp_pk(b[o], 0.f), a1 = mlp_pk(0.f, 0.f);
#pragma unroll
        for (int q = 0; q < MLP_W / 4; ++q) {
            const ulonglong2 w = row[q];
            a0 = mlp_fma2(w.x, h[2 * q], a0);
            a1 = mlp_fma2(w.y, h[2 * q + 1], a1);
        }
        out[o * stride + node] = fmaxf(mlp_sum2(a0) + mlp_sum2(a1), 0.f);
    }
}

// M3, hidden layer 64 -> 64 for TWO nodes per thread and 8 of the 64 output units (part = 0..7): every broadcast weight
// load feeds both nodes (the one-node version is bound by shared-memory wavefronts: 16 LDS.128 per 32 FFMA2), inputs
// in two chunks of 32 so that the 16 accumulator pairs and the inputs of both nodes fit the register file.
#define MLP_P8 8
__device__ __forceinline__ void mlp_layer2(const float *__restrict__ W, const float *__restrict__ b, const float *in,
                                           float *out, int stride, int n0, int n1, int part)
{
    const int o0 = part * MLP_P8;
    f2 acc0[MLP_P8], acc1[MLP_P8];
#pragma unroll
    for (int o = 0; o < MLP_P8; ++o) { acc0[o] = mlp_pk(b[o0 + o], 0.f); acc1[o] = acc0[o]; }
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        f2 h0[16], h1[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float *p = in + (32 * c + 2 * i) * stride;
            h0[i] = mlp_pk(p[n0], p[stride + n0]);
            h1[i] = mlp_pk(p[n1], p[stride + n1]);
        }
#pragma unroll
        for (int o = 0; o < MLP_P8; ++o) {
            const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(W + (o0 + o) * MLP_W + 32 * c);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const ulonglong2 w = row[q];
                acc0[o] = mlp_fma2(w.x, h0[2 * q], acc0[o]);
                acc1[o] = mlp_fma2(w.x, h1[2 * q], acc1[o]);
                acc0[o] = mlp_fma2(w.y, h0[2 * q + 1], acc0[o]);
                acc1[o] = mlp_fma2(w.y, h1[2 * q + 1], acc1[o]);
            }
        }
    }
#pragma unroll
    for (int o = 0; o < MLP_P8; ++o) {
        out[(o0 + o) * stride + n0] = fmaxf(mlp_sum2(acc0[o]), 0.f);
        out[(o0 + o) * stride + n1] = fmaxf(mlp_sum2(acc1[o]), 0.f);
    }
}

// output unit and M4; returns the sigmoid
__device__ __forceinline__ float mlp_head(const float *__restrict__ w5, float b5, const float *in, int stride, int node)
{
    float o = b5;
#pragma unroll 8
    for (int i = 0; i < MLP_W; ++i) o = fmaf(w5[i], in[i * stride + node], o);
    return 1.0f / (1.0f + __expf(-o));
}

extern __shared__ __align__(16) float mlp_smem[];

// cooperative copy of `count` floats into shared memory (src and dst 16-byte aligned)
__device__ __forceinline__ void mlp_stage(float *dst, const float *__restrict__ src, int count, int nthreads)
{
    const float4 *s4 = reinterpret_cast<const float4 *>(src);
    float4 *d4 = reinterpret_cast<float4 *>(dst);
    for (int q = threadIdx.x; q < count / 4; q += nthreads) d4[q] = __ldg(s4 + q);
    for (int q = (count & ~3) + threadIdx.x; q < count; q += nthreads) dst[q] = __ldg(src + q);
}

// (The forward pass runs on the tensor cores: radt_mlp_tc.cu.  The helpers above serve the adjoint's recompute.)

// dW[o][i] = sum_n delta[o][n] a[i][n] for this block's nodes; thread t owns input unit i = t (its activations over
// the nodes sit in registers), output units one at a time with broadcast float4 reads of the delta rows.
__device__ __forceinline__ void mlp_grad_weights(const float *act, const float *delta, int fan_in, float *gW, float *gb,
                                                 int nout, int t, int part)
{
    if (t < fan_in) {
        f2 a[MLP_TB / 2];
#pragma unroll
        for (int n = 0; n < MLP_TB / 2; ++n) a[n] = mlp_pk(act[t * MLP_SA + 2 * n], act[t * MLP_SA + 2 * n + 1]);
#pragma unroll 2
        for (int o = part * MLP_PW; o < (part + 1) * MLP_PW; ++o) {
            const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(delta + o * MLP_SD);
            f2 s0 = mlp_pk(0.f, 0.f), s1 = s0;
#pragma unroll
            for (int q = 0; q < MLP_TB / 4; ++q) {
                const ulonglong2 d = row[q];
                s0 = mlp_fma2(d.x, a[2 * q], s0);
                s1 = mlp_fma2(d.y, a[2 * q + 1], s1);
            }
            atomicAdd(gW + o * fan_in + t, mlp_sum2(s0) + mlp_sum2(s1));
        }
    }
    if (part == 0 && t < nout) {
        const float4 *row = reinterpret_cast<const float4 *>(delta + t * MLP_SD);
        float s = 0.f;
#pragma unroll
        for (int q = 0; q < MLP_TB / 4; ++q) {
            const float4 d = row[q];
            s += (d.x + d.y) + (d.z + d.w);
        }
        atomicAdd(gb + t, s);
    }
}

// delta_in[i][node] = relu'(a_in[i][node]) sum_o W[o][i] delta_out[o][node] for the input units i of this thread's
// part; in place (din = dout): every part reads the whole column first, the block synchronises, then writes.
__device__ __forceinline__ void mlp_back_layer(const float *__restrict__ W, float *dl, const float *ain, int node, int part)
{
    f2 acc2[MLP_PW / 2];
#pragma unroll
    for (int i = 0; i < MLP_PW / 2; ++i) acc2[i] = mlp_pk(0.f, 0.f);
#pragma unroll 4
    for (int o = 0; o < MLP_W; ++o) {
        const float d = dl[o * MLP_SD + node];
        const f2 dd = mlp_pk(d, d);
        const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(W + o * MLP_W + part * MLP_PW);
#pragma unroll
        for (int q = 0; q < MLP_PW / 4; ++q) {
            const ulonglong2 w = row[q];
            acc2[2 * q] = mlp_fma2(w.x, dd, acc2[2 * q]);
            acc2[2 * q + 1] = mlp_fma2(w.y, dd, acc2[2 * q + 1]);
        }
    }
    float acc[MLP_PW];
#pragma unroll
    for (int i = 0; i < MLP_PW / 2; ++i) asm("mov.b64 {%0, %1}, %2;" : "=f"(acc[2 * i]), "=f"(acc[2 * i + 1]) : "l"(acc2[i]));
    __syncthreads();
#pragma unroll
    for (int i = 0; i < MLP_PW; ++i) {
        const int u = part * MLP_PW + i;
        dl[u * MLP_SD + node] = ain[u * MLP_SA + node] > 0.f ? acc[i] : 0.f;
    }
}

// Two-node / two-unit versions of the adjoint's inner routines (same arithmetic; every broadcast row load feeds two
// accumulator sets, which halves the shared-memory wavefronts per FMA as in mlp_layer2).
// dW[o][i] for units i = u0, u1 and the 8 output units of `part`, nodes in two chunks of 32.
__device__ __forceinline__ void mlp_grad_weights2(const float *act, const float *delta, float *gW, int u0, int u1, int part)
{
    const int o0 = part * MLP_P8;
    f2 s0[MLP_P8], s1[MLP_P8];
#pragma unroll
    for (int o = 0; o < MLP_P8; ++o) { s0[o] = mlp_pk(0.f, 0.f); s1[o] = s0[o]; }
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        f2 a0[16], a1[16];
#pragma unroll
        for (int n = 0; n < 16; ++n) {
            a0[n] = mlp_pk(act[u0 * MLP_SA + 32 * c + 2 * n], act[u0 * MLP_SA + 32 * c + 2 * n + 1]);
            a1[n] = mlp_pk(act[u1 * MLP_SA + 32 * c + 2 * n], act[u1 * MLP_SA + 32 * c + 2 * n + 1]);
        }
#pragma unroll
        for (int o = 0; o < MLP_P8; ++o) {
            const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(delta + (o0 + o) * MLP_SD + 32 * c);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const ulonglong2 d = row[q];
                s0[o] = mlp_fma2(d.x, a0[2 * q], s0[o]);
                s1[o] = mlp_fma2(d.x, a1[2 * q], s1[o]);
                s0[o] = mlp_fma2(d.y, a0[2 * q + 1], s0[o]);
                s1[o] = mlp_fma2(d.y, a1[2 * q + 1], s1[o]);
            }
        }
    }
#pragma unroll
    for (int o = 0; o < MLP_P8; ++o) {
        atomicAdd(gW + (o0 + o) * MLP_W + u0, mlp_sum2(s0[o]));
        atomicAdd(gW + (o0 + o) * MLP_W + u1, mlp_sum2(s1[o]));
    }
}

// delta_in for nodes n0, n1 and the 8 input units of `part`; in place like mlp_back_layer
__device__ __forceinline__ void mlp_back_layer2(const float *__restrict__ W, float *dl, const float *ain, int n0, int n1, int part)
{
    const int i0 = part * MLP_P8;
    f2 acc0[MLP_P8 / 2], acc1[MLP_P8 / 2];
#pragma unroll
    for (int i = 0; i < MLP_P8 / 2; ++i) { acc0[i] = mlp_pk(0.f, 0.f); acc1[i] = acc0[i]; }
#pragma unroll 8
    for (int o = 0; o < MLP_W; ++o) {
        const float d0 = dl[o * MLP_SD + n0], d1 = dl[o * MLP_SD + n1];
        const f2 dd0 = mlp_pk(d0, d0), dd1 = mlp_pk(d1, d1);
        const ulonglong2 *row = reinterpret_cast<const ulonglong2 *>(W + o * MLP_W + i0);
#pragma unroll
        for (int q = 0; q < MLP_P8 / 4; ++q) {
            const ulonglong2 w = row[q];
            acc0[2 * q] = mlp_fma2(w.x, dd0, acc0[2 * q]); acc1[2 * q] = mlp_fma2(w.x, dd1, acc1[2 * q]);
            acc0[2 * q + 1] = mlp_fma2(w.y, dd0, acc0[2 * q + 1]); acc1[2 * q + 1] = mlp_fma2(w.y, dd1, acc1[2 * q + 1]);
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < MLP_P8 / 2; ++i) {
        float a, b;
        const int u = i0 + 2 * i;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(acc0[i]));
        dl[u * MLP_SD + n0] = ain[u * MLP_SA + n0] > 0.f ? a : 0.f;
        dl[(u + 1) * MLP_SD + n0] = ain[(u + 1) * MLP_SA + n0] > 0.f ? b : 0.f;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(acc1[i]));
        dl[u * MLP_SD + n1] = ain[u * MLP_SA + n1] > 0.f ? a : 0.f;
        dl[(u + 1) * MLP_SD + n1] = ain[(u + 1) * MLP_SA + n1] > 0.f ? b : 0.f;
    }
}

// Adjoint: recomputes the activations of its 64 nodes (nothing is stored between the passes), then walks the layers
// backwards; parameter gradients leave the block as float atomics.  Shared memory: all activations, ONE delta buffer
// (a node's column is private to its thread, so the back-propagation runs in place) and the weights of the layer
// at hand.
#define MLP_WBUF (MLP_W * MLP_W + MLP_W)
__global__ void __launch_bounds__(MLP_TB * MLP_S, 2) k_mlp_bwd(const __grid_constant__ MlpParamsDev Q)
{
    const int node = threadIdx.x & (MLP_TB - 1), part = threadIdx.x / MLP_TB;   // part is warp uniform
    const int q = blockIdx.x * MLP_TB + node, n = Q.nr * Q.nz;
    const int qq = min(q, n - 1), i = qq / Q.nz, j = qq - i * Q.nz;
    const MlpOff F = mlp_offsets(Q.L);
    float *sW = mlp_smem;                                  // [MLP_WBUF] W_l | b_l of the layer at hand
    float *a0 = sW + MLP_WBUF;                             // [34][SA]
    float *a1 = a0 + 34 * MLP_SA;                          // a_l = a1 + (l - 1) 64 SA, l = 1..4
    float *dl = a1 + MLP_H * MLP_W * MLP_SA;
    dl += (4 - ((dl - mlp_smem) & 3)) & 3;                 // 16-byte aligned rows
    float *go = dl + MLP_W * MLP_SD;
    auto act = [&](int l) { return l == 0 ? a0 : a1 + (l - 1) * MLP_W * MLP_SA; };
    // layer l: W at F.W[l] (64 x fan) followed by b at F.b[l] = F.W[l] + 64 fan: one contiguous block
    auto stage = [&](int l) {
        __syncthreads();
        const int fan = l == 0 ? F.D : MLP_W, cnt = l < MLP_H ? MLP_W * fan + MLP_W : MLP_W + 1;
        const int lead = F.W[l] & 3;                       // keep the 16-byte phase of the source
        for (int t = threadIdx.x; t < cnt; t += MLP_TB * MLP_S) sW[lead + t] = __ldg(Q.params + F.W[l] + t);
        __syncthreads();
        return sW + lead;
    };
    if (part == 0) mlp_encode(Q, i, j, a0, MLP_SA, node);
    {
        const float *w = stage(0);
        mlp_layer_first(w, w + MLP_W * F.D, F.D, a0, a1, MLP_SA, node, part);
    }
    {
        // hidden layers with two nodes per thread: 32 node pairs x 8 parts (radt_mlp.cu mlp_layer2)
        const int pair = threadIdx.x & (MLP_TB / 2 - 1), part8 = threadIdx.x / (MLP_TB / 2);
        for (int l = 1; l < MLP_H; ++l) {
            const float *w = stage(l);                     // (its barriers also order the layers)
            mlp_layer2(w, w + MLP_W * MLP_W, act(l), act(l + 1), MLP_SA, pair, pair + MLP_TB / 2, part8);
        }
    }
    const float *w5 = stage(MLP_H);
    const float *a4 = act(MLP_H);
    const float s = mlp_head(w5, w5[MLP_W], a4, MLP_SA, node);
    // M4 and the output unit
    const float g_o = q < n ? __ldg(Q.g_temp + q) * (Q.t_hi - Q.t_lo) * s * (1.0f - s) : 0.f;
    if (part == 0) go[node] = g_o;
    for (int o = part * MLP_PW; o < (part + 1) * MLP_PW; ++o)
        dl[o * MLP_SD + node] = a4[o * MLP_SA + node] > 0.f ? g_o * w5[o] : 0.f;
    __syncthreads();
    if (part == 0) {
        float s5 = 0.f, sb = 0.f;
        for (int m = 0; m < MLP_TB; ++m) {
            const float g = go[m];
            s5 = fmaf(g, a4[node * MLP_SA + m], s5);
            sb += g;
        }
        atomicAdd(Q.g_params + F.W[MLP_H] + node, s5);     // node doubles as the unit index here (MLP_TB == MLP_W)
        if (node == 0) atomicAdd(Q.g_params + F.b[MLP_H], sb);
    }
    for (int l = MLP_H - 1; l >= 0; --l) {
        const int pair = threadIdx.x & (MLP_TB / 2 - 1), part8 = threadIdx.x / (MLP_TB / 2);
        if (l == 0) {
            mlp_grad_weights(act(0), dl, F.D, Q.g_params + F.W[0], Q.g_params + F.b[0], MLP_W, node, part);
        } else {
            mlp_grad_weights2(act(l), dl, Q.g_params + F.W[l], pair, pair + MLP_TB / 2, part8);
            if (threadIdx.x < MLP_W) {                     // bias gradients: one unit per thread
                const float4 *row = reinterpret_cast<const float4 *>(dl + threadIdx.x * MLP_SD);
                float sb = 0.f;
#pragma unroll
                for (int q = 0; q < MLP_TB / 4; ++q) {
                    const float4 d = row[q];
                    sb += (d.x + d.y) + (d.z + d.w);
                }
                atomicAdd(Q.g_params + F.b[l] + threadIdx.x, sb);
            }
            const float *w = stage(l);                     // (its barriers also fence the reads of dl above)
            mlp_back_layer2(w, dl, act(l), pair, pair + MLP_TB / 2, part8);
            __syncthreads();
        }
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static size_t mlp_bwd_smem() { return (size_t)(MLP_WBUF + 4 + 34 * MLP_SA + MLP_H * MLP_W * MLP_SA + 4 + MLP_W * MLP_SD + MLP_TB) * sizeof(float); }

cudaError_t radt_launch_mlp_bwd(const MlpParamsDev &Q, int nparams, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(Q.g_params, 0, (size_t)nparams * sizeof(float), st);
    if (e != cudaSuccess) return e;
    const size_t smem = mlp_bwd_smem();
    e = cudaFuncSetAttribute(k_mlp_bwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int n = Q.nr * Q.nz;
    k_mlp_bwd<<<(n + MLP_TB - 1) / MLP_TB, MLP_TB * MLP_S, smem, st>>>(Q);
    return cudaGetLastError();
}
