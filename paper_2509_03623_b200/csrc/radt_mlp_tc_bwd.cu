// radt_mlp_tc_bwd.cu -- adjoint of the symmetric MLP temperature field w.r.t. its parameters (Eq. 10; DESIGN.md
// section 9, M1-M4) on the 5th-generation tensor cores of sm_100a: every contraction of the back-propagation is a tcgen05.mma
// (kind::f16 on bf16 operands, 3-product split: x = x_1 + x_2, two bf16 terms carry 16 mantissa bits, D = A_2 B_1 + A_1 B_2 +
// A_1 B_1 with fp32 accumulation in tensor memory; the dropped terms are 2^-16 of the product, the gradient tolerance is 1e-3).
//
// Per tile of 128 grid nodes (node r is served by threads r and r + 128: units 0-31 / 32-63), one CTA per SM, persistent:
//   recompute   a_l = relu(a_{l-1} W_l^T + b_l), l = 1..4; every a_l is written once, by the node's own threads, as a K-major
//               operand tile [node][unit] in shared memory (16-byte chunks of 8 units; 32 consecutive nodes store 512
//               contiguous bytes) and STAYS there for the backward sweep;
//   head        o = w_5 . a_4 + b_5, T = t_lo + (t_hi - t_lo) sigmoid(o); delta_4 = g_T dT/do w_5 relu'(a_4); dw_5, db_5 by a
//               transposing shuffle reduction over the nodes of each warp;
//   for l = 4..1, ONE batch of MMAs per layer:
//     back-prop   delta_{l-1} = (delta_l W_l) relu'(a_{l-1}): A = the delta_l tile [node][unit] (K-major), B = the SAME weight
//                 tile W_l [o][i] the recompute reads K-major, now read through an MN-major descriptor as [i][o];
//     dW_l^T      = a_{l-1}^T delta_l, [i x o], the NODE dimension is K = 128: A = the a_{l-1} tile and B = the delta_l tile, both
//                 read MN-major.  No operand is ever transposed or copied: for 16-bit operands without swizzle the K-major tile
//                 [r][k] IS the MN-major tile [k][r] with the two byte offsets of the descriptor exchanged (8 x 8 core
//                 matrices of 128 bytes either way).  (kind::tf32 allows MN-major operands only in the 128B/32B-swizzled
//                 layout - measured: the plain layout returns zeros - which is why this kernel splits into bf16 terms.)
//                 The accumulator's lane is the input unit, so its read-out adds 32 consecutive addresses of dW_l per warp
//                 instruction; db_l comes from the shuffle reduction of delta_l.
// Parameter gradients leave the CTA as float atomics per tile.  Shares nothing with oracle/.
#include <cuda_bf16.h>
#include "radt_tc.cuh"

#define TB_THREADS 256
#define TB_K1 48                        // first-layer fan-in padded to a multiple of 16 (D = 2 + 4 L <= 34)
#define TB_COL_D 0                      // TMEM columns: forward / back-prop accumulator, dW^T accumulator
#define TB_COL_DW 64
#define TB_COLS 128
// operand tiles (bytes).  K-major, no swizzle, 16-bit: chunk kc (8 K elements = 16 bytes) of row r at kc LBO + r 16, i.e.
// 8 rows x 16 bytes = one 128-byte core matrix, SBO = 128 between groups of 8 rows, LBO = rows x 16 between chunks.
#define TB_ACT_LBO (TC_M * 16)          // activation / delta tiles: 128 rows
#define TB_ACT_BYTES (8 * TB_ACT_LBO)   // 64 units: 16 KB per term
#define TB_A0_BYTES (6 * TB_ACT_LBO)    // 48 features: 12 KB per term
#define TB_W_LBO (TC_W * 16)            // weight tiles: 64 rows
#define TB_W_BYTES (8 * TB_W_LBO)       // 8 KB per term
#define TB_W1_BYTES (6 * TB_W_LBO)      // 6 KB per term
#define TB_OFF_W1 0                                            // {hi, lo}
#define TB_OFF_W (TB_OFF_W1 + 2 * TB_W1_BYTES)                 // layers 2-4 x {hi, lo}
#define TB_OFF_BIAS (TB_OFF_W + 6 * TB_W_BYTES)                // 4 x 64 biases, 64 output weights, output bias
#define TB_OFF_PART (TB_OFF_BIAS + (5 * TC_W + 4) * 4)         // partial output sums of the upper half-rows [128]
#define TB_OFF_GO (TB_OFF_PART + TC_M * 4)                     // dL/do per node [128]
#define TB_OFF_BAR (TB_OFF_GO + TC_M * 4)                      // mbarrier, TMEM base address
#define TB_OFF_A0 ((TB_OFF_BAR + 32 + 127) & ~127)             // a_0 {hi, lo}
#define TB_OFF_ACT (TB_OFF_A0 + 2 * TB_A0_BYTES)               // a_1, a_2, a_3 x {hi, lo}
#define TB_OFF_DL (TB_OFF_ACT + 6 * TB_ACT_BYTES)              // delta_l {hi, lo}; also what the M = 128 rows of the a_3 read alias
#define TB_SMEM_BYTES (TB_OFF_DL + 2 * TB_ACT_BYTES)

// instruction descriptor of kind::f16: D fp32, A and B bf16, N = 64, M = 128; bit 15 / 16: A / B is MN-major
#define TB_IDESC ((1u << 4) | (1u << 7) | (1u << 10) | ((TC_W >> 3) << 17) | ((TC_M >> 4) << 24))
#define TB_A_MN (1u << 15)
#define TB_B_MN (1u << 16)

// D[tmem] (+)= A[smem] B[smem]
__device__ __forceinline__ void tb_mma(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned idesc,
                                       unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
                 "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
}
// the three products of one K step; the descriptors advance by `astep` / `bstep` bytes
__device__ __forceinline__ void tb_mma3(unsigned tmem_d, unsigned long long &a_hi, unsigned long long &a_lo, unsigned long long &b_hi,
                                        unsigned long long &b_lo, unsigned idesc, unsigned &acc, unsigned astep, unsigned bstep)
{
    tb_mma(tmem_d, a_lo, b_hi, idesc, acc);          // small terms first
    tb_mma(tmem_d, a_hi, b_lo, idesc, 1u);
    tb_mma(tmem_d, a_hi, b_hi, idesc, 1u);
    acc = 1u;
    a_hi += astep >> 4; a_lo += astep >> 4;
    b_hi += bstep >> 4; b_lo += bstep >> 4;
}
// generic-proxy writes to shared memory -> visible to the tensor core's (async proxy) operand reads
__device__ __forceinline__ void tb_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// eight consecutive K elements of row `row` (chunk kc) into the hi and lo terms of a K-major tile
__device__ __forceinline__ void tb_store8(unsigned char *hi, unsigned char *lo, int lbo, int kc, int row, const float *x)
{
    unsigned h[4], l[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const __nv_bfloat162 hh = __floats2bfloat162_rn(x[2 * e], x[2 * e + 1]);          // .x = lower address = lower K
        const float2 hf = __bfloat1622float2(hh);
        const __nv_bfloat162 ll = __floats2bfloat162_rn(x[2 * e] - hf.x, x[2 * e + 1] - hf.y);
        h[e] = *reinterpret_cast<const unsigned *>(&hh);
        l[e] = *reinterpret_cast<const unsigned *>(&ll);
    }
    const int off = kc * lbo + row * 16;
    *reinterpret_cast<uint4 *>(hi + off) = make_uint4(h[0], h[1], h[2], h[3]);
    *reinterpret_cast<uint4 *>(lo + off) = make_uint4(l[0], l[1], l[2], l[3]);
}

// column sums over the 32 lanes of a warp: on return lane j holds sum_lanes v[j] (31 shuffles: the lanes halve the columns
// they keep in every round); v is destroyed
__device__ __forceinline__ float tb_column_sums(float (&v)[32], int lane)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const bool up = lane & s;
#pragma unroll
        for (int k = 0; k < s; ++k) {
            const float keep = up ? v[k + s] : v[k], send = up ? v[k] : v[k + s];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, s);
        }
    }
    return v[0];
}

extern __shared__ __align__(128) unsigned char tb_smem[];

__global__ void __launch_bounds__(TB_THREADS, 1) k_mlp_bwd_tc(const __grid_constant__ MlpParamsDev Q, int ntiles)
{
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31, row = t & (TC_M - 1), half = t >> 7;
    const int D = 2 + 4 * Q.L;
    unsigned char *sm = tb_smem;
    float *sBias = reinterpret_cast<float *>(sm + TB_OFF_BIAS), *sPart = reinterpret_cast<float *>(sm + TB_OFF_PART);
    float *sGo = reinterpret_cast<float *>(sm + TB_OFF_GO);
    const unsigned bar = tc_smem_u32(sm + TB_OFF_BAR);
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(sm + TB_OFF_BAR + 16);
    // parameter vector: [W1 (64 x D) | b1 | W2 | b2 | W3 | b3 | W4 | b4 | w_out | b_out]
    const int off2 = TC_W * D + TC_W, lstride = TC_W * TC_W + TC_W, off5 = off2 + 3 * lstride;

    // ---- one-time set-up: TMEM allocation (warp 0), mbarrier, weights split into bf16 hi / lo K-major tiles [o][i]
    if (t < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc_smem_u32(tmem_slot)), "r"(TB_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (t == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        const float *p = Q.params;
        // layers 2-4: 3 x 64 rows x 8 chunks of 8 inputs; rows fastest over the threads (16-byte stores of a quarter-warp fall
        // into different banks), six chunks (12 float4 loads) in flight per thread
#pragma unroll 1
        for (int pass = 0; pass < 1536 / (TB_THREADS * 6); ++pass) {
            float4 v[6][2];
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                const int g = t + TB_THREADS * (6 * pass + i), l = g >> 9, r = g & 511, o = r & (TC_W - 1), kc = r >> 6;
                const float4 *src = reinterpret_cast<const float4 *>(p + off2 + l * lstride + o * TC_W + 8 * kc);
                v[i][0] = __ldg(src); v[i][1] = __ldg(src + 1);
            }
#pragma unroll
            for (int i = 0; i < 6; ++i) {
                const int g = t + TB_THREADS * (6 * pass + i), l = g >> 9, r = g & 511, o = r & (TC_W - 1), kc = r >> 6;
                const float x[8] = {v[i][0].x, v[i][0].y, v[i][0].z, v[i][0].w, v[i][1].x, v[i][1].y, v[i][1].z, v[i][1].w};
                tb_store8(sm + TB_OFF_W + 2 * l * TB_W_BYTES, sm + TB_OFF_W + (2 * l + 1) * TB_W_BYTES, TB_W_LBO, kc, o, x);
            }
        }
        for (int q = t; q < 4 * TC_W; q += TB_THREADS)             // biases of the four layers
            sBias[q] = __ldg(p + (q < TC_W ? TC_W * D + q : off2 + ((q >> 6) - 1) * lstride + TC_W * TC_W + (q & (TC_W - 1))));
        for (int q = t; q < TC_W; q += TB_THREADS) sBias[4 * TC_W + q] = __ldg(p + off5 + q);       // output weights
        if (t == 0) sBias[5 * TC_W] = __ldg(p + off5 + TC_W);                                       // output bias
        for (int q = t; q < TC_W * (TB_K1 / 8); q += TB_THREADS) {       // first layer: rows o, chunks of 8 inputs, zero padded
            const int o = q % TC_W, kc = q / TC_W;
            float x[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) x[e] = (8 * kc + e) < D ? __ldg(p + o * D + 8 * kc + e) : 0.f;
            tb_store8(sm + TB_OFF_W1, sm + TB_OFF_W1 + TB_W1_BYTES, TB_W_LBO, kc, o, x);
        }
    }
    tb_fence_async();
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = *tmem_slot;
    const unsigned tlane = tmem + ((unsigned)((warp & 3) * 32) << 16);                  // this thread's TMEM lane, column 0
    unsigned parity = 0;
    const int n = Q.nr * Q.nz;
    const bool issuer = warp == 0;
    const unsigned s_a0 = tc_smem_u32(sm + TB_OFF_A0), s_act = tc_smem_u32(sm + TB_OFF_ACT), s_dl = tc_smem_u32(sm + TB_OFF_DL);
    const unsigned s_w1 = tc_smem_u32(sm + TB_OFF_W1), s_w = tc_smem_u32(sm + TB_OFF_W);

    // operand tiles written by all threads -> one elected lane issues a batch of MMAs and commits it -> every thread waits
#define TB_ISSUE_BEGIN()                                                           \
    tb_fence_async();                                                              \
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");               \
    __syncthreads();                                                               \
    if (issuer && tc_elect()) {                                                    \
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#define TB_ISSUE_END()                                                             \
        tc_commit(bar);                                                            \
    }                                                                              \
    tc_wait(bar, parity);                                                          \
    parity ^= 1u;                                                                  \
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int q = tile * TC_M + row, qq = min(q, n - 1);
        const int gi = qq / Q.nz, gj = qq - gi * Q.nz;
        const float p0 = (float)gi / (float)(Q.nr - 1), p1 = (float)gj / (float)(Q.nz - 1);
        // ---- M1-M2: gamma = (p0, p1, {sin, cos (2^k pi p0), sin, cos (2^k pi p1)}_k) into the a_0 tile: chunk kc holds features
        // 8 kc .. 8 kc + 7; the two threads of a row take chunks {0, 1, 2} and {3, 4, 5}
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            const int kc = 3 * half + cc;
            float x[8];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2) {
                const int c = 2 * kc + e2;                       // features 4 c .. 4 c + 3
                float s1, c1, s0, c0;
                sincospif(__int_as_float((126 + c) << 23) * p1, &s1, &c1);       // 2^(c-1) p1
                sincospif(__int_as_float((127 + c) << 23) * p0, &s0, &c0);       // 2^c p0
                if (c == 0) { s1 = p0; c1 = p1; }
                if (4 * c + 2 >= D) { s0 = 0.f; c0 = 0.f; }                      // zero padding beyond the D features
                if (4 * c >= D) { s1 = 0.f; c1 = 0.f; }
                x[4 * e2] = s1; x[4 * e2 + 1] = c1; x[4 * e2 + 2] = s0; x[4 * e2 + 3] = c0;
            }
            tb_store8(sm + TB_OFF_A0, sm + TB_OFF_A0 + TB_A0_BYTES, TB_ACT_LBO, kc, row, x);
        }
        // ---- recompute the activations: a_1..a_3 into their tiles (and their sign patterns into registers), a_4 in registers
        float v[32];
        unsigned mask[3];
#pragma unroll
        for (int l = 0; l < 4; ++l) {
            TB_ISSUE_BEGIN()
                const unsigned abase = l == 0 ? s_a0 : s_act + 2 * (l - 1) * TB_ACT_BYTES, asize = l == 0 ? TB_A0_BYTES : TB_ACT_BYTES;
                const unsigned wbase = l == 0 ? s_w1 : s_w + 2 * (l - 1) * TB_W_BYTES, wsize = l == 0 ? TB_W1_BYTES : TB_W_BYTES;
                unsigned long long a_hi = tc_desc(abase, TB_ACT_LBO, TC_SBO), a_lo = tc_desc(abase + asize, TB_ACT_LBO, TC_SBO);
                unsigned long long b_hi = tc_desc(wbase, TB_W_LBO, TC_SBO), b_lo = tc_desc(wbase + wsize, TB_W_LBO, TC_SBO);
                unsigned acc = 0;
                const int ksteps = (l == 0 ? TB_K1 : TC_W) / 16;
                for (int s = 0; s < ksteps; ++s)
                    tb_mma3(tmem + TB_COL_D, a_hi, a_lo, b_hi, b_lo, TB_IDESC, acc, 2 * TB_ACT_LBO, 2 * TB_W_LBO);
            TB_ISSUE_END()
            const float *bias = sBias + l * TC_W + 32 * half;
            tc_ld32(tlane + TB_COL_D + 32 * half, v);
            unsigned m = 0;
#pragma unroll
            for (int c = 0; c < 32; ++c) {
                v[c] = fmaxf(v[c] + bias[c], 0.f);
                m |= (v[c] > 0.f ? 1u : 0u) << c;
            }
            if (l < 3) {
                mask[l] = m;
                unsigned char *dst = sm + TB_OFF_ACT + 2 * l * TB_ACT_BYTES;
#pragma unroll
                for (int j = 0; j < 4; ++j) tb_store8(dst, dst + TB_ACT_BYTES, TB_ACT_LBO, 4 * half + j, row, v + 8 * j);
            }
        }
        // ---- head: M3 output unit, M4 sigmoid, dL/do; delta_4; dw_5 and db_5
        float dl[32];
        {
            const float *w5 = sBias + 4 * TC_W + 32 * half;
            float o = 0.f;
#pragma unroll
            for (int c = 0; c < 32; ++c) o = fmaf(w5[c], v[c], o);
            if (half) sPart[row] = o;
            __syncthreads();
            if (!half) {
                o += sPart[row] + sBias[5 * TC_W];
                const float s = 1.0f / (1.0f + __expf(-o));
                sGo[row] = q < n ? __ldg(Q.g_temp + q) * (Q.t_hi - Q.t_lo) * s * (1.0f - s) : 0.f;
            }
            __syncthreads();
            const float g_o = sGo[row];
            float pr[32];
#pragma unroll
            for (int c = 0; c < 32; ++c) {
                dl[c] = v[c] > 0.f ? g_o * w5[c] : 0.f;
                pr[c] = g_o * v[c];
            }
            const float cs = tb_column_sums(pr, lane);
            atomicAdd(Q.g_params + off5 + 32 * half + lane, cs);
            if (!half) {
                float gs = g_o;
#pragma unroll
                for (int m = 16; m > 0; m >>= 1) gs += __shfl_xor_sync(0xffffffffu, gs, m);
                if (lane == 0) atomicAdd(Q.g_params + off5 + TC_W, gs);
            }
        }
        // ---- back-propagation, layer by layer
#pragma unroll
        for (int l = 4; l >= 1; --l) {
            const int fan = l == 1 ? D : TC_W;
            float *gW = Q.g_params + (l == 1 ? 0 : off2 + (l - 2) * lstride);
            // delta_l into its tile; db_l = its column sums
#pragma unroll
            for (int j = 0; j < 4; ++j) tb_store8(sm + TB_OFF_DL, sm + TB_OFF_DL + TB_ACT_BYTES, TB_ACT_LBO, 4 * half + j, row, dl + 8 * j);
            {
                const float cs = tb_column_sums(dl, lane);          // (dl is dead from here on: the tile holds it)
                atomicAdd(gW + TC_W * fan + 32 * half + lane, cs);
            }
            TB_ISSUE_BEGIN()
                const unsigned d_hi0 = s_dl, d_lo0 = s_dl + TB_ACT_BYTES;
                if (l > 1) {
                    // delta_{l-1} (pre-mask) = delta_l W_l: K = the 64 output units of layer l.  A: delta tile, K-major; B: the weight
                    // tile [o][i] read MN-major as [i][o]: 16-byte atoms of 8 inputs at SBO = the tile's chunk stride, K groups of 8
                    // outputs at LBO = 128
                    const unsigned wbase = s_w + 2 * (l - 2) * TB_W_BYTES;
                    unsigned long long a_hi = tc_desc(d_hi0, TB_ACT_LBO, TC_SBO), a_lo = tc_desc(d_lo0, TB_ACT_LBO, TC_SBO);
                    unsigned long long b_hi = tc_desc(wbase, 128, TB_W_LBO), b_lo = tc_desc(wbase + TB_W_BYTES, 128, TB_W_LBO);
                    unsigned acc = 0;
                    for (int s = 0; s < TC_W / 16; ++s)
                        tb_mma3(tmem + TB_COL_D, a_hi, a_lo, b_hi, b_lo, TB_IDESC | TB_B_MN, acc, 2 * TB_ACT_LBO, 256);
                }
                {
                    // dW_l^T = a_{l-1}^T delta_l: K = the 128 nodes of the tile; both tiles [node][unit] read MN-major as [unit][node]
                    const unsigned abase = l == 1 ? s_a0 : s_act + 2 * (l - 2) * TB_ACT_BYTES, asize = l == 1 ? TB_A0_BYTES : TB_ACT_BYTES;
                    unsigned long long a_hi = tc_desc(abase, 128, TB_ACT_LBO), a_lo = tc_desc(abase + asize, 128, TB_ACT_LBO);
                    unsigned long long b_hi = tc_desc(d_hi0, 128, TB_ACT_LBO), b_lo = tc_desc(d_lo0, 128, TB_ACT_LBO);
                    unsigned acc = 0;
                    for (int s = 0; s < TC_M / 16; ++s)
                        tb_mma3(tmem + TB_COL_DW, a_hi, a_lo, b_hi, b_lo, TB_IDESC | TB_A_MN | TB_B_MN, acc, 256, 256);
                }
            TB_ISSUE_END()
            // delta_{l-1} = relu'(a_{l-1}) (delta_l W_l)
            if (l > 1) {
                tc_ld32(tlane + TB_COL_D + 32 * half, dl);
                const unsigned m = mask[l - 2];
#pragma unroll
                for (int c = 0; c < 32; ++c) dl[c] = (m >> c) & 1u ? dl[c] : 0.f;
            }
            // dW_l^T: TMEM lane = input unit, column = output unit: 32 consecutive addresses per reduction
            if ((warp & 3) < 2) {
                float w[32];
                tc_ld32(tlane + TB_COL_DW + 32 * half, w);
                if (row < fan) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) atomicAdd(gW + (32 * half + c) * fan + row, w[c]);
                }
            }
        }
    }
    // ---- teardown: every thread is done with tensor memory before warp 0 frees it
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (t < 32) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TB_COLS));
    }
}

cudaError_t radt_launch_mlp_bwd(const MlpParamsDev &Q, int nparams, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(Q.g_params, 0, (size_t)nparams * sizeof(float), st);
    if (e != cudaSuccess) return e;
    const int n = Q.nr * Q.nz, ntiles = (n + TC_M - 1) / TC_M;
    e = cudaFuncSetAttribute(k_mlp_bwd_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, TB_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    k_mlp_bwd_tc<<<ntiles < sms ? ntiles : sms, TB_THREADS, TB_SMEM_BYTES, st>>>(Q, ntiles);
    return cudaGetLastError();
}
