// radt_mlp_tc.cu -- forward of the symmetric MLP temperature field (Eq. 10, M1-M4) on
// the 5th-generation tensor cores of sm_100a: tcgen05.mma (kind::tf32) with the accumulators in tensor memory.
//
// The four hidden layers are dense 64-wide contractions: per tile of 128 grid nodes, h_l [128 x 64] = relu(h_{l-1} W_l^T + b_l).
//   - one CTA = 128 threads = one tile of 128 nodes at a time (persistent over tiles); thread t owns node row t, which is
//     TMEM lane t of the accumulator D [128 lanes x 64 fp32 columns];
//   - operands live in shared memory in the canonical K-major, no-swizzle UMMA layout: the tile is cut into chunks of 4 K
//     elements (16 bytes), chunk j of row r at  j * (rows * 16) + r * 16  (8 rows x 16 bytes = one 128-byte core matrix;
//     leading byte offset = rows * 16 between K-adjacent core matrices, stride byte offset = 128 between groups of 8 rows);
//   - fp32 accuracy from TF32 tensor cores by the 3-product split: x = x_hi + x_lo with x_hi = rna_tf32(x), x_lo = x - x_hi
//     (exact), D = A_hi B_hi + A_lo B_hi + A_hi B_lo, the dropped A_lo B_lo term is 2^-22 of the product;
//   - one elected thread issues the K/8 x 3 MMAs of a layer and commits them to an mbarrier; all threads then read their
//     row of D with tcgen05.ld (32x32b.x32), add the bias, apply the ReLU, split and write the next layer's A operand;
//     the activations never leave the SM between layers;
//   - weights (hi and lo copies of all four layers, 108 KB) are converted and staged once per CTA.
// The output unit (64 -> 1) and the sigmoid are a dot product per thread in the last epilogue.  Shares nothing with oracle/.
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define TC_M 128                        // nodes per tile = TMEM lanes = threads
#define TC_W 64                         // hidden width = UMMA N
#define TC_KMAX1 40                     // first-layer fan-in padded to a multiple of 8 (D = 2 + 4 L <= 34)
#define TC_A_CHUNK (TC_M * 16)          // bytes of one 4-wide K chunk of an A tile   (leading byte offset of A)
#define TC_B_CHUNK (TC_W * 16)          // bytes of one 4-wide K chunk of a weight tile (leading byte offset of B)
#define TC_SBO 128                      // 8 rows x 16 bytes

// shared-memory map (bytes)
#define TC_OFF_AHI 0
#define TC_OFF_ALO (TC_OFF_AHI + 16 * TC_A_CHUNK)                  // 32 KB each
#define TC_OFF_W1HI (TC_OFF_ALO + 16 * TC_A_CHUNK)
#define TC_OFF_W1LO (TC_OFF_W1HI + (TC_KMAX1 / 4) * TC_B_CHUNK)    // 10 KB each
#define TC_OFF_WHI (TC_OFF_W1LO + (TC_KMAX1 / 4) * TC_B_CHUNK)     // layers 2-4: 3 x 16 KB
#define TC_OFF_WLO (TC_OFF_WHI + 3 * 16 * TC_B_CHUNK)
#define TC_OFF_BIAS (TC_OFF_WLO + 3 * 16 * TC_B_CHUNK)             // 4 x 64 biases, 64 output weights, output bias
#define TC_OFF_BAR (TC_OFF_BIAS + (5 * TC_W + 4) * 4)
#define TC_SMEM_BYTES (TC_OFF_BAR + 16)

__device__ __forceinline__ unsigned tc_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// K-major, SWIZZLE_NONE shared-memory matrix descriptor (sm_100 version field = 1); all offsets in units of 16 bytes
__device__ __forceinline__ unsigned long long tc_desc(unsigned saddr, unsigned lbo_bytes, unsigned sbo_bytes)
{
    return (unsigned long long)((saddr >> 4) & 0x3FFF) | ((unsigned long long)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((unsigned long long)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46);
}
// instruction descriptor of kind::tf32: D fp32, A and B TF32, both K-major, N = 64, M = 128
#define TC_IDESC ((1u << 4) | (2u << 7) | (2u << 10) | ((TC_W >> 3) << 17) | ((TC_M >> 4) << 24))

__device__ __forceinline__ void tc_mma(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
                 "l"(adesc), "l"(bdesc), "r"(TC_IDESC), "r"(accumulate)
                 : "memory");
}
__device__ __forceinline__ void tc_commit(unsigned bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_wait(unsigned bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@!p bra WAIT_%=;\n\t}\n" ::"r"(bar),
                 "r"(parity)
                 : "memory");
}
// 32 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tc_ld32(unsigned taddr, float (&v)[32])
{
    unsigned r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, "
                 "%24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
                   "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
                   "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float tc_tf32(float x)
{
    unsigned y;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(y) : "f"(x));
    return __uint_as_float(y);
}
// four consecutive K elements of row `row` into the hi and lo copies of an operand tile
__device__ __forceinline__ void tc_store4(unsigned char *hi, unsigned char *lo, int chunk_bytes, int chunk, int row, float a, float b,
                                          float c, float d)
{
    const float ah = tc_tf32(a), bh = tc_tf32(b), ch = tc_tf32(c), dh = tc_tf32(d);
    const int off = chunk * chunk_bytes + row * 16;
    *reinterpret_cast<float4 *>(hi + off) = make_float4(ah, bh, ch, dh);
    *reinterpret_cast<float4 *>(lo + off) = make_float4(a - ah, b - bh, c - ch, d - dh);
}

extern __shared__ __align__(128) unsigned char tc_smem[];

__global__ void __launch_bounds__(TC_M, 1) k_mlp_fwd_tc(const __grid_constant__ MlpParamsDev Q, int ntiles)
{
    const int t = threadIdx.x, warp = t >> 5;
    const int D = 2 + 4 * Q.L, K1 = (D + 7) & ~7;
    unsigned char *sm = tc_smem;
    float *sBias = reinterpret_cast<float *>(sm + TC_OFF_BIAS);
    const unsigned bar = tc_smem_u32(sm + TC_OFF_BAR);
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(sm + TC_OFF_BAR + 8);

    // ---- one-time set-up: TMEM allocation (warp 0), mbarrier, weights split into hi / lo operand tiles
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc_smem_u32(tmem_slot)), "r"(64));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (t == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        // parameter vector: [W1 (64 x D) | b1 | W2 | b2 | W3 | b3 | W4 | b4 | w_out | b_out]
        const float *p = Q.params;
        for (int q = t; q < TC_W * (K1 / 4); q += TC_M) {          // first layer: rows n, chunks of 4 inputs, zero padded
            const int n = q % TC_W, j = q / TC_W;
            float v[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = (4 * j + e) < D ? __ldg(p + n * D + 4 * j + e) : 0.f;
            tc_store4(sm + TC_OFF_W1HI, sm + TC_OFF_W1LO, TC_B_CHUNK, j, n, v[0], v[1], v[2], v[3]);
        }
        int off = TC_W * D;
        for (int q = t; q < TC_W; q += TC_M) sBias[q] = __ldg(p + off + q);
        off += TC_W;
        for (int l = 0; l < 3; ++l) {
            for (int q = t; q < TC_W * 16; q += TC_M) {
                const int n = q % TC_W, j = q / TC_W;
                const float4 v = __ldg(reinterpret_cast<const float4 *>(p + off + n * TC_W) + j);     // (offsets are multiples of 4 iff D is even: it is)
                tc_store4(sm + TC_OFF_WHI + l * 16 * TC_B_CHUNK, sm + TC_OFF_WLO + l * 16 * TC_B_CHUNK, TC_B_CHUNK, j, n, v.x, v.y,
                          v.z, v.w);
            }
            off += TC_W * TC_W;
            for (int q = t; q < TC_W; q += TC_M) sBias[(l + 1) * TC_W + q] = __ldg(p + off + q);
            off += TC_W;
        }
        for (int q = t; q < TC_W; q += TC_M) sBias[4 * TC_W + q] = __ldg(p + off + q);        // output weights
        if (t == 0) sBias[5 * TC_W] = __ldg(p + off + TC_W);                                  // output bias
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = *tmem_slot;
    const unsigned taddr = tmem + ((unsigned)(warp * 32) << 16);          // this warp's lane quadrant
    const unsigned sA_hi = tc_smem_u32(sm + TC_OFF_AHI), sA_lo = tc_smem_u32(sm + TC_OFF_ALO);
    unsigned parity = 0;
    const int n = Q.nr * Q.nz;

    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        // ---- M1-M2: encoding of this thread's node into the layer-1 A operand (K1 columns, zero padded)
        {
            const int qq = min(tile * TC_M + t, n - 1);
            const int i = qq / Q.nz, j = qq - i * Q.nz;
            const float p0 = (float)i / (float)(Q.nr - 1), p1 = (float)j / (float)(Q.nz - 1);
            float f[TC_KMAX1];
#pragma unroll
            for (int e = 0; e < TC_KMAX1; ++e) f[e] = 0.f;
            f[0] = p0; f[1] = p1;
            float fr = 1.0f;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (k < Q.L) {
                    f[2 + 4 * k + 0] = sinpif(fr * p0); f[2 + 4 * k + 1] = cospif(fr * p0);
                    f[2 + 4 * k + 2] = sinpif(fr * p1); f[2 + 4 * k + 3] = cospif(fr * p1);
                }
                fr *= 2.0f;
            }
#pragma unroll
            for (int c = 0; c < TC_KMAX1 / 4; ++c)
                if (4 * c < K1) tc_store4(sm + TC_OFF_AHI, sm + TC_OFF_ALO, TC_A_CHUNK, c, t, f[4 * c], f[4 * c + 1], f[4 * c + 2], f[4 * c + 3]);
        }
        float temp_out = 0.f;
#pragma unroll 1
        for (int l = 0; l < 4; ++l) {
            // the A operand written by the generic proxy must be visible to the tensor core's async proxy; every thread has
            // also finished reading the previous accumulator
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (t == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const int ksteps = (l == 0 ? K1 : TC_W) / 8;
                const unsigned w_hi = tc_smem_u32(sm + (l == 0 ? TC_OFF_W1HI : TC_OFF_WHI + (l - 1) * 16 * TC_B_CHUNK));
                const unsigned w_lo = tc_smem_u32(sm + (l == 0 ? TC_OFF_W1LO : TC_OFF_WLO + (l - 1) * 16 * TC_B_CHUNK));
                unsigned acc = 0;
                for (int s = 0; s < ksteps; ++s) {
                    const unsigned long long a_hi = tc_desc(sA_hi + 2 * s * TC_A_CHUNK, TC_A_CHUNK, TC_SBO);
                    const unsigned long long a_lo = tc_desc(sA_lo + 2 * s * TC_A_CHUNK, TC_A_CHUNK, TC_SBO);
                    const unsigned long long b_hi = tc_desc(w_hi + 2 * s * TC_B_CHUNK, TC_B_CHUNK, TC_SBO);
                    const unsigned long long b_lo = tc_desc(w_lo + 2 * s * TC_B_CHUNK, TC_B_CHUNK, TC_SBO);
                    tc_mma(tmem, a_lo, b_hi, acc);          // small terms first
                    tc_mma(tmem, a_hi, b_lo, 1u);
                    tc_mma(tmem, a_hi, b_hi, 1u);
                    acc = 1u;
                }
                tc_commit(bar);                              // arrives on the mbarrier when these MMAs have completed
            }
            tc_wait(bar, parity);
            parity ^= 1u;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const float *bias = sBias + l * TC_W;
            if (l < 3) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    float v[32];
                    tc_ld32(taddr + 32 * h, v);
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const int u = 32 * h + 4 * c;
                        tc_store4(sm + TC_OFF_AHI, sm + TC_OFF_ALO, TC_A_CHUNK, u >> 2, t, fmaxf(v[4 * c] + bias[u], 0.f),
                                  fmaxf(v[4 * c + 1] + bias[u + 1], 0.f), fmaxf(v[4 * c + 2] + bias[u + 2], 0.f),
                                  fmaxf(v[4 * c + 3] + bias[u + 3], 0.f));
                    }
                }
            } else {
                // M3 output unit and M4: sigmoid scaled to [t_lo, t_hi]
                const float *w5 = sBias + 4 * TC_W;
                float o = sBias[5 * TC_W];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    float v[32];
                    tc_ld32(taddr + 32 * h, v);
#pragma unroll
                    for (int c = 0; c < 32; ++c) o = fmaf(w5[32 * h + c], fmaxf(v[c] + bias[32 * h + c], 0.f), o);
                }
                temp_out = fmaf(Q.t_hi - Q.t_lo, 1.0f / (1.0f + __expf(-o)), Q.t_lo);
            }
        }
        const int q = tile * TC_M + t;
        if (q < n) Q.temp_out[q] = temp_out;
    }
    // ---- teardown: every thread is done with the accumulator before warp 0 frees it
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(64));
    }
}

cudaError_t radt_launch_mlp_fwd(const MlpParamsDev &Q, cudaStream_t st)
{
    const int n = Q.nr * Q.nz, ntiles = (n + TC_M - 1) / TC_M;
    cudaError_t e = cudaFuncSetAttribute(k_mlp_fwd_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    k_mlp_fwd_tc<<<ntiles < sms ? ntiles : sms, TC_M, TC_SMEM_BYTES, st>>>(Q, ntiles);
    return cudaGetLastError();
}
