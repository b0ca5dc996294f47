// tc_tmem.cuh -- tensor memory (TMEM, 512 columns x 128 lanes x 32 bit per SM) used as a parking buffer between the
// consumer warps of the W-builder and its flusher warps.  FP64 has no tcgen05.mma kind, so TMEM holds no accumulators
// here: it is 256 KB of on-chip storage next to a full shared memory.
// Shape 32x32b: thread t of warp w owns lane 32 (w % 4) + t; .x64 moves 64 consecutive 32-bit columns of that lane.
#pragma once

#include "tc_common.cuh"

__device__ __forceinline__ void tmem_alloc(uint32_t smem_result_addr, uint32_t ncols) {   // one full warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_result_addr), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {            // the same warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// 32 doubles of this thread -> 64 columns at taddr (lane field = this warp's quarter).  The source registers are read at issue;
// tmem_wait_st() before the data is read back (tcgen05.ld by this thread, or a hand-over to other warps).
__device__ __forceinline__ void tmem_store32(uint32_t taddr, const double (&x)[32]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x64.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63, %64};"
                 ::"r"(taddr), "r"(__double2loint(x[0])), "r"(__double2hiint(x[0])), "r"(__double2loint(x[1])), "r"(__double2hiint(x[1])), "r"(__double2loint(x[2])), "r"(__double2hiint(x[2])), "r"(__double2loint(x[3])), "r"(__double2hiint(x[3])), "r"(__double2loint(x[4])), "r"(__double2hiint(x[4])), "r"(__double2loint(x[5])), "r"(__double2hiint(x[5])), "r"(__double2loint(x[6])), "r"(__double2hiint(x[6])), "r"(__double2loint(x[7])), "r"(__double2hiint(x[7])), "r"(__double2loint(x[8])), "r"(__double2hiint(x[8])), "r"(__double2loint(x[9])), "r"(__double2hiint(x[9])), "r"(__double2loint(x[10])), "r"(__double2hiint(x[10])), "r"(__double2loint(x[11])), "r"(__double2hiint(x[11])), "r"(__double2loint(x[12])), "r"(__double2hiint(x[12])), "r"(__double2loint(x[13])), "r"(__double2hiint(x[13])), "r"(__double2loint(x[14])), "r"(__double2hiint(x[14])), "r"(__double2loint(x[15])), "r"(__double2hiint(x[15])), "r"(__double2loint(x[16])), "r"(__double2hiint(x[16])), "r"(__double2loint(x[17])), "r"(__double2hiint(x[17])), "r"(__double2loint(x[18])), "r"(__double2hiint(x[18])), "r"(__double2loint(x[19])), "r"(__double2hiint(x[19])), "r"(__double2loint(x[20])), "r"(__double2hiint(x[20])), "r"(__double2loint(x[21])), "r"(__double2hiint(x[21])), "r"(__double2loint(x[22])), "r"(__double2hiint(x[22])), "r"(__double2loint(x[23])), "r"(__double2hiint(x[23])), "r"(__double2loint(x[24])), "r"(__double2hiint(x[24])), "r"(__double2loint(x[25])), "r"(__double2hiint(x[25])), "r"(__double2loint(x[26])), "r"(__double2hiint(x[26])), "r"(__double2loint(x[27])), "r"(__double2hiint(x[27])), "r"(__double2loint(x[28])), "r"(__double2hiint(x[28])), "r"(__double2loint(x[29])), "r"(__double2hiint(x[29])), "r"(__double2loint(x[30])), "r"(__double2hiint(x[30])), "r"(__double2loint(x[31])), "r"(__double2hiint(x[31]))
                 : "memory");
}
// 64 columns at taddr -> 32 doubles of this thread
__device__ __forceinline__ void tmem_load32(uint32_t taddr, double (&x)[32]) {
    uint32_t r[64];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x64.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63}, [%64];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]), "=r"(r[32]), "=r"(r[33]), "=r"(r[34]), "=r"(r[35]), "=r"(r[36]), "=r"(r[37]), "=r"(r[38]), "=r"(r[39]), "=r"(r[40]), "=r"(r[41]), "=r"(r[42]), "=r"(r[43]), "=r"(r[44]), "=r"(r[45]), "=r"(r[46]), "=r"(r[47]), "=r"(r[48]), "=r"(r[49]), "=r"(r[50]), "=r"(r[51]), "=r"(r[52]), "=r"(r[53]), "=r"(r[54]), "=r"(r[55]), "=r"(r[56]), "=r"(r[57]), "=r"(r[58]), "=r"(r[59]), "=r"(r[60]), "=r"(r[61]), "=r"(r[62]), "=r"(r[63])
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; i++) x[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
}
// 32 columns at taddr -> 16 doubles of this thread
__device__ __forceinline__ void tmem_load16(uint32_t taddr, double (&x)[16]) {
    uint32_t r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; i++) x[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
}

// Two 32-column loads in flight together, one wait; returns the NEGATED doubles (sign bit flipped in the integer pipe: hole
// sums enter W with a minus sign and the FP64 pipe belongs to the DMMAs).
__device__ __forceinline__ void tmem_load16_neg_pair(uint32_t taddr0, uint32_t taddr1, double (&x0)[16], double (&x1)[16]) {
    uint32_t r[32], q[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(taddr0)
                 : "memory");
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                 : "=r"(q[0]), "=r"(q[1]), "=r"(q[2]), "=r"(q[3]), "=r"(q[4]), "=r"(q[5]), "=r"(q[6]), "=r"(q[7]), "=r"(q[8]), "=r"(q[9]), "=r"(q[10]), "=r"(q[11]), "=r"(q[12]), "=r"(q[13]), "=r"(q[14]), "=r"(q[15]), "=r"(q[16]), "=r"(q[17]), "=r"(q[18]), "=r"(q[19]), "=r"(q[20]), "=r"(q[21]), "=r"(q[22]), "=r"(q[23]), "=r"(q[24]), "=r"(q[25]), "=r"(q[26]), "=r"(q[27]), "=r"(q[28]), "=r"(q[29]), "=r"(q[30]), "=r"(q[31])
                 : "r"(taddr1)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; i++) {
        x0[i] = __hiloint2double((int)(r[2 * i + 1] ^ 0x80000000u), (int)r[2 * i]);
        x1[i] = __hiloint2double((int)(q[2 * i + 1] ^ 0x80000000u), (int)q[2 * i]);
    }
}
