// radt_mlp.cu -- symmetric MLP temperature field on the nodes of the (r, zeta) grid and its adjoint w.r.t. the
// parameters (Eq. 10).  Algorithm M1-M4 of DESIGN.md section 9: normalised grid
// coordinates -> positional encoding of degree L -> 4 x 64 ReLU layers -> sigmoid scaled to [t_lo, t_hi].
// fp32 FMA; one node per thread, activations in shared memory ([unit][node], so both the per-node and the
// per-unit passes read without bank conflicts), weights through uniform L1 loads.  Shares nothing with oracle/.
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define MLP_W 64                       // hidden width
#define MLP_H 4                        // hidden layers
#define MLP_TF 128                     // nodes per block, forward
#define MLP_TB 64                      // nodes per block, adjoint
#define MLP_SA (MLP_TB + 1)            // activation row stride (adjoint): scalar reads by unit are conflict free
#define MLP_SD (MLP_TB + 4)            // delta row stride: 16-byte aligned rows for broadcast float4 reads

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
                                                const float *in, float *out, int stride, int node)
{
    float h[34];
#pragma unroll
    for (int i = 0; i < 34; ++i) h[i] = i < D ? in[i * stride + node] : 0.f;
#pragma unroll 2
    for (int o = 0; o < MLP_W; ++o) {
        float acc = __ldg(b + o);
#pragma unroll
        for (int i = 0; i < 34; ++i)
            if (i < D) acc = fmaf(__ldg(W + o * D + i), h[i], acc);
        out[o * stride + node] = fmaxf(acc, 0.f);
    }
}

// M3, hidden layer 64 -> 64: the node's inputs in registers, one output unit at a time, weight rows as float4
__device__ __forceinline__ void mlp_layer(const float *__restrict__ W, const float *__restrict__ b, const float *in,
                                          float *out, int stride, int node)
{
    float h[MLP_W];
#pragma unroll
    for (int i = 0; i < MLP_W; ++i) h[i] = in[i * stride + node];
#pragma unroll 2
    for (int o = 0; o < MLP_W; ++o) {
        const float4 *row = reinterpret_cast<const float4 *>(W + o * MLP_W);
        float a0 = __ldg(b + o), a1 = 0.f;
#pragma unroll
        for (int q = 0; q < MLP_W / 4; ++q) {
            const float4 w = __ldg(row + q);
            a0 = fmaf(w.x, h[4 * q], a0); a1 = fmaf(w.y, h[4 * q + 1], a1);
            a0 = fmaf(w.z, h[4 * q + 2], a0); a1 = fmaf(w.w, h[4 * q + 3], a1);
        }
        out[o * stride + node] = fmaxf(a0 + a1, 0.f);
    }
}

// output unit and M4; returns the sigmoid
__device__ __forceinline__ float mlp_head(const float *__restrict__ w5, float b5, const float *in, int stride, int node)
{
    float o = b5;
#pragma unroll 8
    for (int i = 0; i < MLP_W; ++i) o = fmaf(__ldg(w5 + i), in[i * stride + node], o);
    return 1.0f / (1.0f + __expf(-o));
}

extern __shared__ __align__(16) float mlp_smem[];

__global__ void __launch_bounds__(MLP_TF) k_mlp_fwd(const __grid_constant__ MlpParamsDev Q)
{
    const int node = threadIdx.x, q = blockIdx.x * MLP_TF + node, n = Q.nr * Q.nz;
    const int qq = min(q, n - 1), i = qq / Q.nz, j = qq - i * Q.nz;
    const MlpOff F = mlp_offsets(Q.L);
    float *A = mlp_smem, *B = mlp_smem + MLP_W * MLP_TF;           // ping-pong [unit][node]
    mlp_encode(Q, i, j, A, MLP_TF, node);
    mlp_layer_first(Q.params + F.W[0], Q.params + F.b[0], F.D, A, B, MLP_TF, node);
    mlp_layer(Q.params + F.W[1], Q.params + F.b[1], B, A, MLP_TF, node);
    mlp_layer(Q.params + F.W[2], Q.params + F.b[2], A, B, MLP_TF, node);
    mlp_layer(Q.params + F.W[3], Q.params + F.b[3], B, A, MLP_TF, node);
    const float s = mlp_head(Q.params + F.W[4], __ldg(Q.params + F.b[4]), A, MLP_TF, node);
    if (q < n) Q.temp_out[q] = fmaf(Q.t_hi - Q.t_lo, s, Q.t_lo);
}

// dW[o][i] = sum_n delta[o][n] a[i][n] for this block's nodes; thread t owns input unit i = t (its activations over
// the nodes sit in registers), output units one at a time with broadcast float4 reads of the delta rows.
__device__ __forceinline__ void mlp_grad_weights(const float *act, const float *delta, int fan_in, float *gW, float *gb,
                                                 int nout, int t)
{
    if (t < fan_in) {
        float a[MLP_TB];
#pragma unroll
        for (int n = 0; n < MLP_TB; ++n) a[n] = act[t * MLP_SA + n];
#pragma unroll 2
        for (int o = 0; o < nout; ++o) {
            const float4 *row = reinterpret_cast<const float4 *>(delta + o * MLP_SD);
            float s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int q = 0; q < MLP_TB / 4; ++q) {
                const float4 d = row[q];
                s0 = fmaf(d.x, a[4 * q], s0); s1 = fmaf(d.y, a[4 * q + 1], s1);
                s0 = fmaf(d.z, a[4 * q + 2], s0); s1 = fmaf(d.w, a[4 * q + 3], s1);
            }
            atomicAdd(gW + o * fan_in + t, s0 + s1);
        }
    }
    if (t < nout) {
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

// delta_in[i][node] = relu'(a_in[i][node]) sum_o W[o][i] delta_out[o][node]
__device__ __forceinline__ void mlp_back_layer(const float *__restrict__ W, const float *dout, const float *ain, float *din,
                                               int node)
{
    float acc[MLP_W];
#pragma unroll
    for (int i = 0; i < MLP_W; ++i) acc[i] = 0.f;
#pragma unroll 2
    for (int o = 0; o < MLP_W; ++o) {
        const float d = dout[o * MLP_SD + node];
        const float4 *row = reinterpret_cast<const float4 *>(W + o * MLP_W);
#pragma unroll
        for (int q = 0; q < MLP_W / 4; ++q) {
            const float4 w = __ldg(row + q);
            acc[4 * q] = fmaf(w.x, d, acc[4 * q]); acc[4 * q + 1] = fmaf(w.y, d, acc[4 * q + 1]);
            acc[4 * q + 2] = fmaf(w.z, d, acc[4 * q + 2]); acc[4 * q + 3] = fmaf(w.w, d, acc[4 * q + 3]);
        }
    }
#pragma unroll
    for (int i = 0; i < MLP_W; ++i) din[i * MLP_SD + node] = ain[i * MLP_SA + node] > 0.f ? acc[i] : 0.f;
}

// Adjoint: recomputes the activations of its 64 nodes (nothing is stored between the passes), then walks the layers
// backwards; parameter gradients leave the block as float atomics.
__global__ void __launch_bounds__(MLP_TB) k_mlp_bwd(const __grid_constant__ MlpParamsDev Q)
{
    const int node = threadIdx.x, q = blockIdx.x * MLP_TB + node, n = Q.nr * Q.nz;
    const int qq = min(q, n - 1), i = qq / Q.nz, j = qq - i * Q.nz;
    const MlpOff F = mlp_offsets(Q.L);
    float *a0 = mlp_smem;                                  // [34][SA]
    float *a[MLP_H + 1];
    a[0] = a0;
    for (int l = 1; l <= MLP_H; ++l) a[l] = a0 + 34 * MLP_SA + (l - 1) * MLP_W * MLP_SA;
    float *dA = a0 + 34 * MLP_SA + MLP_H * MLP_W * MLP_SA;
    dA += (4 - ((dA - mlp_smem) & 3)) & 3;                 // 16-byte aligned rows
    float *dB = dA + MLP_W * MLP_SD, *go = dB + MLP_W * MLP_SD;
    mlp_encode(Q, i, j, a[0], MLP_SA, node);
    mlp_layer_first(Q.params + F.W[0], Q.params + F.b[0], F.D, a[0], a[1], MLP_SA, node);
    for (int l = 1; l < MLP_H; ++l) mlp_layer(Q.params + F.W[l], Q.params + F.b[l], a[l], a[l + 1], MLP_SA, node);
    const float s = mlp_head(Q.params + F.W[MLP_H], __ldg(Q.params + F.b[MLP_H]), a[MLP_H], MLP_SA, node);
    // M4 and the output unit
    const float g_o = q < n ? __ldg(Q.g_temp + q) * (Q.t_hi - Q.t_lo) * s * (1.0f - s) : 0.f;
    go[node] = g_o;
    for (int o = 0; o < MLP_W; ++o)
        dA[o * MLP_SD + node] = a[MLP_H][o * MLP_SA + node] > 0.f ? g_o * __ldg(Q.params + F.W[MLP_H] + o) : 0.f;
    __syncthreads();
    {
        float s5 = 0.f, sb = 0.f;
        for (int m = 0; m < MLP_TB; ++m) {
            const float g = go[m];
            s5 = fmaf(g, a[MLP_H][node * MLP_SA + m], s5);
            sb += g;
        }
        atomicAdd(Q.g_params + F.W[MLP_H] + node, s5);     // node doubles as the unit index here (MLP_TB == MLP_W)
        if (node == 0) atomicAdd(Q.g_params + F.b[MLP_H], sb);
    }
    float *dcur = dA, *dnext = dB;
    for (int l = MLP_H - 1; l >= 0; --l) {
        mlp_grad_weights(a[l], dcur, l == 0 ? F.D : MLP_W, Q.g_params + F.W[l], Q.g_params + F.b[l], MLP_W, node);
        if (l > 0) {
            mlp_back_layer(Q.params + F.W[l], dcur, a[l], dnext, node);
            float *t = dcur; dcur = dnext; dnext = t;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static size_t mlp_bwd_smem() { return (size_t)(34 * MLP_SA + MLP_H * MLP_W * MLP_SA + 4 + 2 * MLP_W * MLP_SD + MLP_TB) * sizeof(float); }

cudaError_t radt_launch_mlp_fwd(const MlpParamsDev &Q, cudaStream_t st)
{
    const size_t smem = (size_t)2 * MLP_W * MLP_TF * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(k_mlp_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int n = Q.nr * Q.nz;
    k_mlp_fwd<<<(n + MLP_TF - 1) / MLP_TF, MLP_TF, smem, st>>>(Q);
    return cudaGetLastError();
}

cudaError_t radt_launch_mlp_bwd(const MlpParamsDev &Q, int nparams, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(Q.g_params, 0, (size_t)nparams * sizeof(float), st);
    if (e != cudaSuccess) return e;
    const size_t smem = mlp_bwd_smem();
    e = cudaFuncSetAttribute(k_mlp_bwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int n = Q.nr * Q.nz;
    k_mlp_bwd<<<(n + MLP_TB - 1) / MLP_TB, MLP_TB, smem, st>>>(Q);
    return cudaGetLastError();
}
