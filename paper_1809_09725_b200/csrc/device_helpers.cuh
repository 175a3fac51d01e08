// Device helpers shared by the tensor-core and TMA-staged projector kernels (sm_100a): mma.sync / ldmatrix wrappers, the
// split-bf16 pair, and the mbarrier + 1-D bulk-copy idioms.  Internal to libcp4d.so.
#pragma once
#include <cuda_bf16.h>
#include <stdint.h>

namespace cp4d {

// D[16 x 8] += A[16 x 16] * B[16 x 8], bf16 operands, fp32 accumulation (SASS HMMA.16816.F32.BF16)
__device__ __forceinline__ void mma16816(float (&d)[4], const unsigned (&a)[4], unsigned b0, unsigned b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// D[16 x 8] += A[16 x 32] * B[32 x 8] with A 2:4 sparse along K (two kept elements per group of four, as a 16 x 16 compressed
// matrix in the layout of the dense m16n8k16 A fragment; SASS HMMA.SP.16832.F32.BF16).  Metadata e (selector 0): lane 4g holds
// the 2-bit positions of row g's compressed elements 0..7 in its low half and of row g + 8's in its high half, lane 4g + 1 the
// same for the compressed elements 8..15 (element c at bits 2c; positions of a group in ascending order); lanes 4g + 2, 4g + 3
// are not read.  Measured on B200 (profiles/r2_microbench.md): 9.7 clk per instruction and sub-partition against 8.7 for the dense
// m16n8k16, i.e. 1.8 x the products per clock.
__device__ __forceinline__ void mma_sp16832(float (&d)[4], const unsigned (&a)[4], const unsigned (&b)[4], unsigned e) {
    asm volatile("mma.sp::ordered_metadata.sync.aligned.m16n8k32.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9,%10,%11}, "
                 "{%0,%1,%2,%3}, %12, 0x0;\n"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]), "r"(e));
}
// four 8 x 8 b16 matrices, transposed on the way: lane l gives the row address of matrix l / 8, row l % 8 (SASS LDSM.16.MT88.4)
__device__ __forceinline__ void ldsm4t(unsigned (&a)[4], unsigned addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]) : "r"(addr));
}
// (x, y) -> bf16 pairs hi, lo with x = hi.x + lo.x + O(2^-18 x); low half = first element
__device__ __forceinline__ void split2(float x, float y, unsigned &hi, unsigned &lo) {
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;\n" : "=r"(hi) : "f"(y), "f"(x));
    const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xffff0000u);       // bf16 -> fp32 is a shift
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;\n" : "=r"(lo) : "f"(y - hy), "f"(x - hx));
}

// ---- TMA 1-D bulk copy global -> shared, completion on an mbarrier (SASS UBLKCP / SYNCS) ----
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

}  // namespace cp4d
