// radt_mlp_tc.cu -- forward of the symmetric MLP temperature field (Eq. 10, M1-M4) on
// the 5th-generation tensor cores of sm_100a: tcgen05.mma (kind::tf32) with the accumulators in tensor memory.
//
// The four hidden layers are dense 64-wide contractions: per tile of 128 grid nodes, h_l [128 x 64] = relu(h_{l-1} W_l^T + b_l).
//   - one CTA = 2 groups of 256 threads, each group with its own tile of 128 nodes in flight (persistent over tiles; the
//     tensor core works on one group's layer while the other group converts its accumulator); node row r is TMEM lane r of the
//     accumulator D [128 lanes x 64 fp32 columns] and is served by threads r (columns 0-31) and r + 128 (columns 32-63): two
//     warps per scheduler, so that one warp's TMEM loads and conversions overlap the other's;
//   - the A operand (activations, [128 x K]) lives in TENSOR MEMORY as well (lane = node row, one column per K element):
//     with only 8 K elements per tf32 MMA, an A operand in shared memory made the MMAs wait on 4 KB of operand reads each
//     (100 cycles per MMA against the 32-cycle floor of a 128 x 64 tile);
//   - the B operand (weights, [64 x K]) lives in shared memory in the canonical K-major, no-swizzle UMMA layout: chunks of 4
//     K elements (16 bytes), chunk j of row r at  j * 1024 + r * 16  (8 rows x 16 bytes = one 128-byte core matrix; leading
//     byte offset = 1024 between K-adjacent core matrices, stride byte offset = 128 between groups of 8 rows);
//   - fp32 accuracy from TF32 tensor cores by the 3-product split: x = x_hi + x_lo with x_hi = rna_tf32(x), x_lo = x - x_hi
//     (exact), D = A_hi B_hi + A_lo B_hi + A_hi B_lo, the dropped A_lo B_lo term is 2^-22 of the product;
//   - one elected thread issues the K/8 x 3 MMAs of a layer and commits them to an mbarrier; all threads then read their
//     row of D with tcgen05.ld (32x32b.x32), add the bias, apply the ReLU, split and write the next layer's A operand
//     back with tcgen05.st; the activations never leave tensor memory / registers between layers;
//   - weights (hi and lo copies of all four layers, 108 KB) are converted and staged once per CTA.
// The output unit (64 -> 1) and the sigmoid are a dot product per thread in the last epilogue.  Shares nothing with oracle/.
#include "radt_tc.cuh"

extern __shared__ __align__(128) unsigned char tc_smem[];

__global__ void __launch_bounds__(TC_THREADS, 1) k_mlp_fwd_tc(const __grid_constant__ MlpParamsDev Q, int ntiles)
{
    const int t = threadIdx.x, group = t >> 8, tg = t & (TC_GROUP - 1), warp = tg >> 5, row = tg & (TC_M - 1), half = tg >> 7;
    const int D = 2 + 4 * Q.L, K1 = (D + 7) & ~7;
    unsigned char *sm = tc_smem;
    float *sBias = reinterpret_cast<float *>(sm + TC_OFF_BIAS), *sPart = reinterpret_cast<float *>(sm + TC_OFF_PART) + TC_M * group;
    const unsigned bar = tc_smem_u32(sm + TC_OFF_BAR) + 8 * group;
    unsigned *tmem_slot = reinterpret_cast<unsigned *>(sm + TC_OFF_BAR + 16);

    // ---- one-time set-up: TMEM allocation (warp 0), mbarrier, weights split into hi / lo operand tiles
    if (t < 32) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc_smem_u32(tmem_slot)), "r"(TC_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tg == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {
        // parameter vector: [W1 (64 x D) | b1 | W2 | b2 | W3 | b3 | W4 | b4 | w_out | b_out]
        const float *p = Q.params;
        // layers 2-4: 3 x 1024 float4, six per thread, all loads in flight before the first conversion (a load-convert-
        // store loop left the CTA waiting on L2 for 5 cycles per issued instruction); rows fastest over the threads, so that
        // the 16-byte stores of a quarter-warp fall into different banks
        const int off2 = TC_W * D + TC_W, lstride = TC_W * TC_W + TC_W;
        float4 v[6];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const int g = t + TC_THREADS * i, l = g >> 10, r = g & 1023, n = r & (TC_W - 1), j = r >> 6;
            v[i] = __ldg(reinterpret_cast<const float4 *>(p + off2 + l * lstride + n * TC_W) + j);     // (offsets are multiples of 4: D is even)
        }
        for (int q = t; q < 4 * TC_W; q += TC_THREADS)             // biases of the four layers
            sBias[q] = __ldg(p + (q < TC_W ? TC_W * D + q : off2 + ((q >> 6) - 1) * lstride + TC_W * TC_W + (q & (TC_W - 1))));
        const int off5 = off2 + 3 * lstride;
        for (int q = t; q < TC_W; q += TC_THREADS) sBias[4 * TC_W + q] = __ldg(p + off5 + q);       // output weights
        if (t == 0) sBias[5 * TC_W] = __ldg(p + off5 + TC_W);                                       // output bias
        for (int q = t; q < TC_W * (K1 / 4); q += TC_THREADS) {          // first layer: rows n, chunks of 4 inputs, zero padded
            const int n = q % TC_W, j = q / TC_W;
            float v[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) v[e] = (4 * j + e) < D ? __ldg(p + n * D + 4 * j + e) : 0.f;
            tc_store4(sm + TC_OFF_W1HI, sm + TC_OFF_W1LO, TC_B_CHUNK, j, n, v[0], v[1], v[2], v[3]);
        }
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const int g = t + TC_THREADS * i, l = g >> 10, r = g & 1023, n = r & (TC_W - 1), j = r >> 6;
            tc_store4(sm + TC_OFF_WHI + l * 16 * TC_B_CHUNK, sm + TC_OFF_WLO + l * 16 * TC_B_CHUNK, TC_B_CHUNK, j, n, v[i].x, v[i].y,
                      v[i].z, v[i].w);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = *tmem_slot + TC_COLS_GROUP * group;          // this group's columns
    const unsigned taddr = tmem + ((unsigned)((warp & 3) * 32) << 16) + TC_COL_D + 32 * half;      // this warp's lane quadrant, this half's columns of D
    const unsigned tlane = tmem + ((unsigned)((warp & 3) * 32) << 16);                  // this thread's TMEM lane, column 0
    unsigned parity = 0;
    const int n = Q.nr * Q.nz;

    for (int tile = 2 * blockIdx.x + group; tile < ntiles; tile += 2 * gridDim.x) {
        // ---- M1-M2: encoding of this thread's node into the layer-1 A operand (K1 columns, zero padded)
        {
            const int qq = min(tile * TC_M + row, n - 1);
            const int i = qq / Q.nz, j = qq - i * Q.nz;
            const float p0 = (float)i / (float)(Q.nr - 1), p1 = (float)j / (float)(Q.nz - 1);
            // chunk c holds features 4c .. 4c+3 of gamma = (p0, p1, {sin, cos (2^k pi p0), sin, cos (2^k pi p1)}_k); the two
            // threads of a row write alternate chunks c = 2 cc + half: entries {0, 1} are sin, cos of 2^(c-1) pi p1 (chunk 0:
            // p0, p1 themselves) and entries {2, 3} are sin, cos of 2^c pi p0 -- one sincospi per pair
#pragma unroll
            for (int cc = 0; cc < TC_KMAX1 / 8; ++cc) {
                const int c = 2 * cc + half;
                if (4 * c < K1) {
                    float s1, c1, s0, c0;
                    sincospif(__int_as_float((126 + c) << 23) * p1, &s1, &c1);       // 2^(c-1) p1
                    sincospif(__int_as_float((127 + c) << 23) * p0, &s0, &c0);       // 2^c p0
                    if (c == 0) { s1 = p0; c1 = p1; }
                    if (4 * c + 2 >= D) { s0 = 0.f; c0 = 0.f; }                      // zero padding beyond the D features
                    if (4 * c >= D) { s1 = 0.f; c1 = 0.f; }
                    const float h0 = tc_tf32(s1), h1 = tc_tf32(c1), h2 = tc_tf32(s0), h3 = tc_tf32(c0);
                    tc_st4(tlane + TC_COL_AHI + 4 * c, h0, h1, h2, h3);
                    tc_st4(tlane + TC_COL_ALO + 4 * c, s1 - h0, c1 - h1, s0 - h2, c0 - h3);
                }
            }
        }
        float temp_out = 0.f;
#pragma unroll 1
        for (int l = 0; l < 4; ++l) {
            // every thread's A columns are in tensor memory and every thread has finished reading the previous accumulator
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            asm volatile("bar.sync %0, %1;" ::"r"(1 + group), "r"(TC_GROUP) : "memory");        // this group's threads only
            if (warp == 0 && tc_elect()) {                   // one elected lane of warp 0 issues (warp-uniform operands)
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const int ksteps = (l == 0 ? K1 : TC_W) / 8;
                const unsigned w_hi = tc_smem_u32(sm + (l == 0 ? TC_OFF_W1HI : TC_OFF_WHI + (l - 1) * 16 * TC_B_CHUNK));
                const unsigned w_lo = tc_smem_u32(sm + (l == 0 ? TC_OFF_W1LO : TC_OFF_WLO + (l - 1) * 16 * TC_B_CHUNK));
                // a K step of 8 elements: 8 TMEM columns of A, two chunks of B (start-address field of the descriptor)
                unsigned a_hi = tmem + TC_COL_AHI, a_lo = tmem + TC_COL_ALO;
                unsigned long long b_hi = tc_desc(w_hi, TC_B_CHUNK, TC_SBO), b_lo = tc_desc(w_lo, TC_B_CHUNK, TC_SBO);
                unsigned acc = 0;
#pragma unroll 2
                for (int s = 0; s < ksteps; ++s) {
                    tc_mma(tmem + TC_COL_D, a_lo, b_hi, acc);          // small terms first
                    tc_mma(tmem + TC_COL_D, a_hi, b_lo, 1u);
                    tc_mma(tmem + TC_COL_D, a_hi, b_hi, 1u);
                    acc = 1u;
                    a_hi += 8; a_lo += 8;
                    b_hi += (2 * TC_B_CHUNK) >> 4; b_lo += (2 * TC_B_CHUNK) >> 4;
                }
                tc_commit(bar);                              // arrives on the mbarrier when these MMAs have completed
            }
            tc_wait(bar, parity);
            parity ^= 1u;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const float *bias = sBias + l * TC_W + 32 * half;
            float v[32];
            tc_ld32(taddr, v);
            if (l < 3) {
                float hi[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) {
                    v[c] = fmaxf(v[c] + bias[c], 0.f);
                    hi[c] = tc_tf32(v[c]);
                    v[c] -= hi[c];
                }
                tc_st32(tlane + TC_COL_AHI + 32 * half, hi);
                tc_st32(tlane + TC_COL_ALO + 32 * half, v);
            } else {
                // M3 output unit and M4: each half-row's share of the dot product, then the sigmoid scaled to [t_lo, t_hi]
                const float *w5 = sBias + 4 * TC_W + 32 * half;
                float o = 0.f;
#pragma unroll
                for (int c = 0; c < 32; ++c) o = fmaf(w5[c], fmaxf(v[c] + bias[c], 0.f), o);
                if (half) sPart[row] = o;
                asm volatile("bar.sync %0, %1;" ::"r"(1 + group), "r"(TC_GROUP) : "memory");
                if (!half) {
                    o += sPart[row] + sBias[5 * TC_W];
                    temp_out = fmaf(Q.t_hi - Q.t_lo, 1.0f / (1.0f + __expf(-o)), Q.t_lo);
                }
            }
        }
        const int q = tile * TC_M + row;
        if (!half && q < n) Q.temp_out[q] = temp_out;
    }
    // ---- teardown: every thread is done with the accumulator before warp 0 frees it
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (t < 32) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TC_COLS));
    }
}

cudaError_t radt_launch_mlp_fwd(const MlpParamsDev &Q, cudaStream_t st)
{
    const int n = Q.nr * Q.nz, ntiles = (n + TC_M - 1) / TC_M;
    cudaError_t e = cudaFuncSetAttribute(k_mlp_fwd_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int pairs = (ntiles + 1) / 2;
    k_mlp_fwd_tc<<<pairs < sms ? pairs : sms, TC_THREADS, TC_SMEM_BYTES, st>>>(Q, ntiles);
    return cudaGetLastError();
}
