// radt_tc.cuh -- tcgen05 / tensor-memory helpers shared by the tensor-core MLP kernels (radt_mlp_tc.cu: forward,
// radt_mlp_tc_bwd.cu: adjoint): operand tile geometry, shared-memory matrix descriptors, MMA issue, TMEM loads and stores,
// the TF32 hi / lo split.  sm_100a only.  Shares nothing with oracle/.
#pragma once
#include "radt_dev.cuh"
#include "radt_kernels.h"

#define TC_M 128                        // nodes per tile = TMEM lanes
#define TC_GROUP 256                    // threads per tile: two per node row
#define TC_THREADS 512                  // two groups per CTA, each with its own tile in flight: one group's epilogue runs under
                                        // the other's MMAs
#define TC_W 64                         // hidden width = UMMA N
#define TC_KMAX1 40                     // first-layer fan-in padded to a multiple of 8 (D = 2 + 4 L <= 34)
#define TC_B_CHUNK (TC_W * 16)          // bytes of one 4-wide K chunk of a weight tile (leading byte offset of B)
#define TC_SBO 128                      // 8 rows x 16 bytes
#define TC_COL_D 0                      // TMEM columns: accumulator, A_hi, A_lo (64 fp32 columns each; 256 allocated)
#define TC_COL_AHI 64
#define TC_COL_ALO 128
#define TC_COLS_GROUP 192               // per group
#define TC_COLS 512

// shared-memory map (bytes)
#define TC_OFF_W1HI 0
#define TC_OFF_W1LO (TC_OFF_W1HI + (TC_KMAX1 / 4) * TC_B_CHUNK)    // 10 KB each
#define TC_OFF_WHI (TC_OFF_W1LO + (TC_KMAX1 / 4) * TC_B_CHUNK)     // layers 2-4: 3 x 16 KB
#define TC_OFF_WLO (TC_OFF_WHI + 3 * 16 * TC_B_CHUNK)
#define TC_OFF_BIAS (TC_OFF_WLO + 3 * 16 * TC_B_CHUNK)             // 4 x 64 biases, 64 output weights, output bias
#define TC_OFF_PART (TC_OFF_BIAS + (5 * TC_W + 4) * 4)              // partial output sums of the upper half-rows
#define TC_OFF_BAR (TC_OFF_PART + 2 * TC_M * 4)                   // two mbarriers, TMEM base address
#define TC_SMEM_BYTES (TC_OFF_BAR + 32)

__device__ __forceinline__ unsigned tc_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// K-major, SWIZZLE_NONE shared-memory matrix descriptor (sm_100 version field = 1); all offsets in units of 16 bytes
__device__ __forceinline__ unsigned long long tc_desc(unsigned saddr, unsigned lbo_bytes, unsigned sbo_bytes)
{
    return (unsigned long long)((saddr >> 4) & 0x3FFF) | ((unsigned long long)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((unsigned long long)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46);
}
// instruction descriptor of kind::tf32: D fp32, A and B TF32, both K-major, N = 64, M = 128
#define TC_IDESC ((1u << 4) | (2u << 7) | (2u << 10) | ((TC_W >> 3) << 17) | ((TC_M >> 4) << 24))

__device__ __forceinline__ bool tc_elect()
{
    unsigned pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.b32 %0, 1, 0, P;\n\t}\n" : "=r"(pred));
    return pred != 0;
}
// D[tmem] (+)= A[tmem] B[smem]^T
__device__ __forceinline__ void tc_mma(unsigned tmem_d, unsigned tmem_a, unsigned long long bdesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(tmem_d),
                 "r"(tmem_a), "l"(bdesc), "r"(TC_IDESC), "r"(accumulate)
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
// four / thirty-two consecutive columns of this thread's TMEM lane
__device__ __forceinline__ void tc_st4(unsigned taddr, float a, float b, float c, float d)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(__float_as_uint(a)),
                 "r"(__float_as_uint(b)), "r"(__float_as_uint(c)), "r"(__float_as_uint(d))
                 : "memory");
}
__device__ __forceinline__ void tc_st32(unsigned taddr, const float (&v)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
                 "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, "
                 "%24, %25, %26, %27, %28, %29, %30, %31};" ::"r"(__float_as_uint(v[0])),
                 "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])),
                 "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])), "r"(__float_as_uint(v[8])),
                 "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])), "r"(__float_as_uint(v[12])),
                 "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15])), "r"(__float_as_uint(v[16])),
                 "r"(__float_as_uint(v[17])), "r"(__float_as_uint(v[18])), "r"(__float_as_uint(v[19])), "r"(__float_as_uint(v[20])),
                 "r"(__float_as_uint(v[21])), "r"(__float_as_uint(v[22])), "r"(__float_as_uint(v[23])), "r"(__float_as_uint(v[24])),
                 "r"(__float_as_uint(v[25])), "r"(__float_as_uint(v[26])), "r"(__float_as_uint(v[27])), "r"(__float_as_uint(v[28])),
                 "r"(__float_as_uint(v[29])), "r"(__float_as_uint(v[30])), "r"(__float_as_uint(v[31])), "r"(taddr)
                 : "memory");
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

