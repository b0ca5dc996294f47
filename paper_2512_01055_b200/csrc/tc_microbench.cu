// tc_microbench.cu -- the roofline denominators, measured on the device the library runs on:
//   * FP64 tensor-core peak: register-resident mma.sync m8n8k4 f64 (SASS DMMA.8x8x4) chains,
//   * FP64 FMA peak: register-resident DFMA chains,
//   * device copy bandwidth,
//   * what the W-builder's consumer loop can reach (tc_bench_ring_peak): the production warp tile and operand ring
//     without flush and epilogue, in three steps (bare LDS + DMMA, + mbarrier ring, + TMA producers).
// BASELINE.json north_star: "each against the chip's peak as measured by a DMMA
// microbenchmark and a copy microbenchmark".
#include <algorithm>

#include "tc_tma.cuh"

namespace {

constexpr int kChains = 8;  // independent accumulator pairs per warp (DMMA) / per thread x2 (DFMA)

__global__ void __launch_bounds__(1024) k_dmma_chain(int iters, double* sink) {
    double c0[kChains], c1[kChains];
    const double a = 1.0 + 1e-9 * (threadIdx.x & 31);
    const double b = 1e-9 * (threadIdx.x & 7);
#pragma unroll
    for (int n = 0; n < kChains; n++) {
        c0[n] = n;
        c1[n] = -n;
    }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int n = 0; n < kChains; n++) dmma884(c0[n], c1[n], a, b);
    }
    double s = 0;
#pragma unroll
    for (int n = 0; n < kChains; n++) s += c0[n] + c1[n];
    if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;  // never true; keeps the chain alive
}

__global__ void __launch_bounds__(1024) k_dfma_chain(int iters, double* sink) {
    double c[2 * kChains];
    const double a = 1.0 + 1e-12 * (threadIdx.x & 31);
    const double b = 1e-9 * (threadIdx.x & 7);
#pragma unroll
    for (int n = 0; n < 2 * kChains; n++) c[n] = n;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int n = 0; n < 2 * kChains; n++) c[n] = fma(c[n], a, b);
    }
    double s = 0;
#pragma unroll
    for (int n = 0; n < 2 * kChains; n++) s += c[n];
    if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_copy(double2* __restrict__ dst, const double2* __restrict__ src, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (; i + 3 * stride < n; i += 4 * stride) {
        double2 x0 = src[i], x1 = src[i + stride], x2 = src[i + 2 * stride], x3 = src[i + 3 * stride];
        dst[i] = x0;
        dst[i + stride] = x1;
        dst[i + 2 * stride] = x2;
        dst[i + 3 * stride] = x3;
    }
    for (; i < n; i += stride) dst[i] = src[i];
}

}  // namespace

// warps_per_sm in {4,8,16,32,64}: threads per block = min(1024, 32*warps_per_sm), blocks per SM accordingly
static void micro_cfg(int warps_per_sm, int sm_count, dim3* grid, dim3* block) {
    int tpb = warps_per_sm * 32;
    int bps = 1;
    while (tpb > 1024) {
        tpb /= 2;
        bps *= 2;
    }
    *grid = dim3(sm_count * bps);
    *block = dim3(tpb);
}

static int g_dmma_wps = 16, g_dfma_wps = 16;

cudaError_t tc_micro_dmma(int sm_count, int iters, double* sink, cudaStream_t stream, double* flop_out) {
    dim3 g, b;
    micro_cfg(g_dmma_wps, sm_count, &g, &b);
    k_dmma_chain<<<g, b, 0, stream>>>(iters, sink);
    // one DMMA.8x8x4 = 8*8*4 FMA = 512 flop per warp instruction
    *flop_out = (double)g.x * (b.x / 32) * (double)iters * kChains * 512.0;
    return cudaGetLastError();
}

cudaError_t tc_micro_dfma(int sm_count, int iters, double* sink, cudaStream_t stream, double* flop_out) {
    dim3 g, b;
    micro_cfg(g_dfma_wps, sm_count, &g, &b);
    k_dfma_chain<<<g, b, 0, stream>>>(iters, sink);
    *flop_out = (double)g.x * b.x * (double)iters * (2 * kChains) * 2.0;
    return cudaGetLastError();
}

cudaError_t tc_micro_copy(void* dst, const void* src, size_t bytes, int sm_count, cudaStream_t stream) {
    k_copy<<<sm_count * 16, 256, 0, stream>>>((double2*)dst, (const double2*)src, bytes / sizeof(double2));
    return cudaGetLastError();
}

// ---- C-ABI ------------------------------------------------------------------------------

typedef cudaError_t (*micro_fn)(int, int, double*, cudaStream_t, double*);

static tc_status run_peak(tc_ctx* ctx, micro_fn fn, int* wps_var, double seconds, double* sustained, double* burst) {
    if (!ctx || !sustained || !burst || !(seconds > 0)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad argument");
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    double* sink = nullptr;
    TC_CUDA(ctx, cudaMalloc(&sink, sizeof(double) * 64));  // never written (guard is false)
    cudaEvent_t e0 = ctx->ev_t0, e1 = ctx->ev_t1;
    double best_rate = 0;
    int best_wps = 16;
    const int cand[5] = {4, 8, 16, 32, 64};
    // calibration: pick the occupancy with the best single-launch rate (~10 ms launches)
    for (int c = 0; c < 5; c++) {
        *wps_var = cand[c];
        double flop = 0;
        int iters = 4096;
        for (int rep = 0; rep < 3; rep++) {
            cudaEventRecord(e0, 0);
            cudaError_t e = fn(ctx->sm_count, iters, sink, 0, &flop);
            cudaEventRecord(e1, 0);
            if (e != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) {
                cudaFree(sink);
                TC_FAIL(ctx, TC_ERR_CUDA, "microbenchmark launch failed: %s", cudaGetErrorString(cudaGetLastError()));
            }
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            double rate = flop / (ms * 1e-3);
            if (rate > best_rate) {
                best_rate = rate;
                best_wps = cand[c];
            }
            if (ms < 5.0f) iters *= 4;
        }
    }
    *wps_var = best_wps;
    // size one launch to ~20 ms, then run back to back for `seconds`
    double flop1 = 0;
    int iters = 1 << 14;
    {
        cudaEventRecord(e0, 0);
        fn(ctx->sm_count, iters, sink, 0, &flop1);
        cudaEventRecord(e1, 0);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        double scale = 20.0 / (ms > 1e-3f ? ms : 1e-3f);
        long long it2 = (long long)(iters * scale);
        if (it2 < 1024) it2 = 1024;
        if (it2 > (1 << 26)) it2 = 1 << 26;
        iters = (int)it2;
    }
    int launches = (int)(seconds / 0.020) + 1;
    double total_flop = 0;
    cudaEventRecord(e0, 0);
    for (int n = 0; n < launches; n++) {
        fn(ctx->sm_count, iters, sink, 0, &flop1);
        total_flop += flop1;
    }
    cudaEventRecord(e1, 0);
    cudaError_t e = cudaEventSynchronize(e1);
    cudaFree(sink);
    if (e != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "microbenchmark failed: %s", cudaGetErrorString(e));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    *sustained = total_flop / (ms * 1e-3) * 1e-12;
    *burst = best_rate * 1e-12;
    return TC_OK;
}

extern "C" tc_status tc_bench_dmma_peak(tc_ctx* ctx, double seconds, double* tflops_sustained, double* tflops_burst) {
    return run_peak(ctx, tc_micro_dmma, &g_dmma_wps, seconds, tflops_sustained, tflops_burst);
}

extern "C" tc_status tc_bench_dfma_peak(tc_ctx* ctx, double seconds, double* tflops_sustained, double* tflops_burst) {
    return run_peak(ctx, tc_micro_dfma, &g_dfma_wps, seconds, tflops_sustained, tflops_burst);
}

extern "C" tc_status tc_bench_copy_bw(tc_ctx* ctx, void* dst_dev, const void* src_dev, size_t bytes, int reps, double* gbs) {
    if (!ctx || !dst_dev || !src_dev || bytes < 4096 || reps < 1 || !gbs) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad argument");
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    tc_micro_copy(dst_dev, src_dev, bytes, ctx->sm_count, 0);  // warm-up
    double best = 0;
    for (int r = 0; r < reps; r++) {
        cudaEventRecord(ctx->ev_t0, 0);
        TC_CUDA(ctx, tc_micro_copy(dst_dev, src_dev, bytes, ctx->sm_count, 0));
        cudaEventRecord(ctx->ev_t1, 0);
        TC_CUDA(ctx, cudaEventSynchronize(ctx->ev_t1));
        float ms = 0;
        cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1);
        double rate = 2.0 * (double)bytes / (ms * 1e-3) * 1e-9;
        if (rate > best) best = rate;
    }
    *gbs = best;
    return TC_OK;
}

// ---- the W-builder's consumer loop, stand-alone ------------------------------------------------------------------
// Same shape as k_wbuild_tma's particle phase: 8 consumer warps with 32 x 32 warp tiles, K chunk 4, a 3-stage ring of
// [2][16][4][8] B fragments and [4][8][4] A fragments, 4 producer warps with one operand stream each.
namespace {

constexpr int RB_STAGES = 3;
constexpr int RB_B_STAGE = 2 * 16 * 4 * 8;   // doubles
constexpr int RB_A_STAGE = 4 * 32;
constexpr int RB_V = 128;                    // the scratch buffer is viewed as slices / amplitude blocks of v = 128

struct __align__(128) RingSmem {
    double B[RB_STAGES][RB_B_STAGE];
    double A[RB_STAGES][RB_A_STAGE];
    unsigned long long full[RB_STAGES];
    unsigned long long empty[RB_STAGES];
};

template <int VARIANT>
__global__ void __launch_bounds__(384, 1)
k_ring(int chunks, int nslots, double* sink, const __grid_constant__ CUtensorMap mapB, const __grid_constant__ CUtensorMap mapA) {
    extern __shared__ unsigned char ring_raw[];
    RingSmem& s = *reinterpret_cast<RingSmem*>(((uintptr_t)ring_raw + 127) & ~(uintptr_t)127);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int n = tid; n < RB_STAGES * RB_B_STAGE; n += 384) (&s.B[0][0])[n] = 1e-3 * (n & 15);
    for (int n = tid; n < RB_STAGES * RB_A_STAGE; n += 384) (&s.A[0][0])[n] = 1.0 + 1e-3 * (n & 7);
    if (tid == 0) {
        for (int n = 0; n < RB_STAGES; n++) {
            mbar_init(smem_u32(&s.full[n]), 1);
            mbar_init(smem_u32(&s.empty[n]), 8);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t full0 = smem_u32(&s.full[0]), empty0 = smem_u32(&s.empty[0]);
    if (warp >= 8) {
        if (VARIANT == 0) return;
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        const int pw = warp - 8;
        const bool leader = elect_one();
        const uint32_t B0 = smem_u32(&s.B[0][0]), A0 = smem_u32(&s.A[0][0]);
        int stage = 0;
        uint32_t wrap = 0;
        for (int r = 0; r < chunks; r++) {
            if (wrap > 0) mbar_wait(empty0 + stage * 8, (wrap - 1) & 1);
            if (leader) {
                const uint32_t full = full0 + stage * 8;
                if (VARIANT == 1) {
                    if (pw == 0) mbar_arrive(full);
                } else {
                    // walk K (d) of one (n1, n2) tile pair, then the next pair, then the next slot
                    const int k0 = (r * 4) % RB_V, tile = (r * 4) / RB_V;
                    const int U0 = (tile % 8) * 16, V0 = ((tile / 8) % 8) * 16, slot = (blockIdx.x + tile / 64) % nslots;
                    if (pw == 0) mbar_expect_tx(full, 2 * 4096 + 2 * 512);
                    if (pw < 2) tma_load_4d(B0 + stage * (RB_B_STAGE * 8) + pw * 4096, &mapB, V0 + 8 * pw, k0, U0, slot, full);
                    else tma_load_4d(A0 + stage * (RB_A_STAGE * 8) + (pw - 2) * 512, &mapA, k0, U0, (tile + pw) % RB_V, slot, full);
                }
            }
            if (++stage == RB_STAGES) {
                stage = 0;
                wrap++;
            }
        }
        return;
    }
    if (VARIANT != 0) asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    const int fr = lane >> 2, fk = lane & 3;
    const uint32_t bB = opaque(smem_u32(&s.B[0][0]) + ((warp * 4 + fk) * 8 + fr) * 8);
    const uint32_t bA = opaque(smem_u32(&s.A[0][0]) + (fr * 4 + fk) * 8);
    double acc[4][2][2][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) acc[x][y][z][0] = acc[x][y][z][1] = 0.0;
    int stage = 0;
    uint32_t parity = 0;
    for (int r = 0; r < chunks; r++) {
        if (VARIANT != 0) mbar_wait(full0 + stage * 8, parity);
        const uint32_t pa = bA + stage * (RB_A_STAGE * 8), pb = bB + stage * (RB_B_STAGE * 8);
        double fa[4], fb[2][2];
#pragma unroll
        for (int x = 0; x < 4; x++) fa[x] = lds64(pa + x * 256);
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) fb[y][z] = lds64(pb + z * 4096 + y * 2048);
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int y = 0; y < 2; y++)
#pragma unroll
                for (int z = 0; z < 2; z++) dmma884(acc[x][y][z][0], acc[x][y][z][1], fa[x], fb[y][z]);
        if (VARIANT != 0) {
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + stage * 8);
        }
        if (++stage == RB_STAGES) {
            stage = 0;
            parity ^= 1;
        }
    }
    double sum = 0;
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) sum += acc[x][y][z][0] + acc[x][y][z][1];
    if (sum == 123.456) sink[blockIdx.x * 256 + tid] = sum;   // never true; keeps the chains alive
}

constexpr int kRingSmem = (int)sizeof(RingSmem) + 128;

}  // namespace

cudaError_t tc_microbench_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_ring<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_ring<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_ring<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem);
    return e;
}

extern "C" tc_status tc_bench_ring_peak(tc_ctx* ctx, int variant, double seconds, void* scratch_dev, size_t scratch_bytes, double* tflops) {
    if (!ctx || !tflops || variant < 0 || variant > 2 || !(seconds > 0)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad argument");
    const size_t slot_bytes = sizeof(double) * RB_V * RB_V * RB_V;   // 16 MB
    if (variant == 2 && (!scratch_dev || scratch_bytes < 4 * slot_bytes)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "variant 2 needs >= 64 MB of device scratch");
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    CUtensorMap mapB, mapA;
    memset(&mapB, 0, sizeof(mapB));
    memset(&mapA, 0, sizeof(mapA));
    int nslots = 1;
    if (variant == 2) {
        nslots = (int)std::min<size_t>(scratch_bytes / slot_bytes, 64);
        TC_CUDA(ctx, cudaMemsetAsync(scratch_dev, 0, (size_t)nslots * slot_bytes, 0));
        const cuuint64_t V = RB_V;
        const cuuint64_t dimB[4] = {V, V, V, (cuuint64_t)nslots}, strB[3] = {V * V, V, V * V * V};   // slice [slot][d][b][c] as (c, d, b, slot)
        const cuuint32_t boxB[4] = {8, 4, 16, 1};
        const cuuint64_t dimA[4] = {V, V, V, (cuuint64_t)nslots}, strA[3] = {V, V * V, V * V * V};   // t2 [x][y][m][d] as (d, m, y, x)
        const cuuint32_t boxA[4] = {4, 16, 1, 1};
        if (!tctma::encode4(&mapB, (const double*)scratch_dev, dimB, strB, boxB) || !tctma::encode4(&mapA, (const double*)scratch_dev, dimA, strA, boxA))
            TC_FAIL(ctx, TC_ERR_CUDA, "cuTensorMapEncodeTiled failed");
    }
    double* sink = nullptr;
    TC_CUDA(ctx, cudaMalloc(&sink, sizeof(double) * 64));
    auto launch = [&](int chunks) -> cudaError_t {
        if (variant == 0) k_ring<0><<<ctx->sm_count, 384, kRingSmem, 0>>>(chunks, nslots, sink, mapB, mapA);
        else if (variant == 1) k_ring<1><<<ctx->sm_count, 384, kRingSmem, 0>>>(chunks, nslots, sink, mapB, mapA);
        else k_ring<2><<<ctx->sm_count, 384, kRingSmem, 0>>>(chunks, nslots, sink, mapB, mapA);
        return cudaGetLastError();
    };
    const int chunks = 1 << 16;   // ~17 ms per launch at the DMMA peak
    const double flop1 = (double)ctx->sm_count * 8.0 * chunks * 16.0 * 512.0;
    cudaError_t e = launch(chunks);   // warm-up
    int launches = (int)(seconds / 0.018) + 1;
    cudaEventRecord(ctx->ev_t0, 0);
    for (int n = 0; n < launches && e == cudaSuccess; n++) e = launch(chunks);
    cudaEventRecord(ctx->ev_t1, 0);
    if (e == cudaSuccess) e = cudaEventSynchronize(ctx->ev_t1);
    cudaFree(sink);
    if (e != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "ring microbenchmark failed: %s", cudaGetErrorString(e));
    float ms = 0;
    cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1);
    *tflops = flop1 * launches / (ms * 1e-3) * 1e-12;
    return TC_OK;
}
