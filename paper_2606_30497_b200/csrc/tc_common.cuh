// tc_common.cuh -- tcgen05 / TMEM / TMA helpers shared by the tensor-core kernels (eval_tc.cu, train_tc.cu).
// Product code only; nothing here is used by, or shared with, oracle/.
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "internal.h"

namespace mlp {

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tmap, int c0, int c1,
                                            uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                 : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc], fp32 operands read as TF32
__device__ __forceinline__ void mma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                         uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// the same with 16-bit operands (kind::f16; the instruction descriptor says BF16), fp32 accumulate
__device__ __forceinline__ void mma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                        uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// 32 lanes x 32 consecutive columns: thread t of the warp gets lane (base + t), columns c..c+31
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
          "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]),
          "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]),
          "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, 128-byte-swizzled operand descriptor (8-row x 128-byte atoms, 1024 bytes apart)
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}

// MN-major 16-bit operand in the same layout (rows = K index, the 128 bytes of a row = 64 M or N elements; groups of 8 K rows,
// 1,024 bytes apart; +2,048 bytes (16 rows) per K = 16; instruction-descriptor bit 15 (A) / 16 (B)): measured with a probe kernel
__device__ __forceinline__ uint64_t smem_desc_sw128_mn16(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (64ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// The same tile geometry with the "128-byte swizzle, 32-byte atom" (CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B; UMMA layout type 1):
// the 32-byte chunk index is XORed with (row & 3), the pattern repeats every 4 rows (512 bytes).  It is the layout in which
// a TF32 operand can be read in EITHER orientation (measured with a probe kernel, profiles/r02_microbench.md section 4):
//   K-major  (rows = M or N index, the 128 bytes of a row = 32 K elements): groups of 4 rows, SBO = 512 bytes; +32 bytes per K = 8;
//   MN-major (rows = K index, the 128 bytes of a row = 32 M or N elements): groups of 4 K rows, SBO = 512 bytes, LBO = distance
//            between 32-element column blocks of M / N; +1,024 bytes (8 rows) per K = 8; instruction-descriptor bit 15 (A) / 16 (B).
// (The 16-byte-atom swizzle of smem_desc_sw128 gives all-zero results for MN-major TF32 operands; LBO must be 32-byte aligned.)
__device__ __forceinline__ uint64_t smem_desc_sw128_a32(uint32_t saddr, uint32_t lbo_bytes) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | (32ull << 32) | (1ull << 46) | (1ull << 61);
}
// byte offset of the 16-byte half h of the 32-byte chunk g of row r in such a tile
__device__ __forceinline__ int swz32(int r, int g, int h) { return r * 128 + ((g ^ (r & 3)) << 5) + (h << 4); }
constexpr uint32_t kIdescAMajorMN = 1u << 15, kIdescBMajorMN = 1u << 16;

// byte offset of the 16-byte chunk c of row r in a [rows][128 B] tile with the 128-byte swizzle
__device__ __forceinline__ int swz(int r, int c) { return r * 128 + ((c ^ (r & 7)) << 4); }
// two fp32 -> packed bf16x2 (round to nearest even); `lo` lands in the low half
__device__ __forceinline__ uint32_t bf16x2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
// fp32 -> the TF32 value the tensor core would use (low 13 mantissa bits dropped), and what that drops (exact in fp32)
__device__ __forceinline__ float tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
__device__ __forceinline__ float tf32_residual(float x) { return x - tf32_trunc(x); }
// instruction descriptor of tcgen05.mma: fp32 accumulate, both operands K-major, A/B format `fmt`
// (kind::tf32: 2 = TF32; kind::f16: 1 = BF16), N and M extents
__host__ __device__ constexpr uint32_t mma_idesc(uint32_t fmt, int M, int N) {
    return (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

}  // namespace mlp
