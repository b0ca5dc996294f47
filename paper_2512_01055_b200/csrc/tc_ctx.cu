// tc_ctx.cu -- context lifetime, status strings, statistics.
#include <stdlib.h>

#include "tc_common.cuh"

extern "C" const char* tc_status_string(tc_status s) {
    switch (s) {
        case TC_OK: return "TC_OK";
        case TC_ERR_INVALID_ARG: return "TC_ERR_INVALID_ARG";
        case TC_ERR_UNSUPPORTED_DEVICE: return "TC_ERR_UNSUPPORTED_DEVICE";
        case TC_ERR_WORKSPACE_TOO_SMALL: return "TC_ERR_WORKSPACE_TOO_SMALL";
        case TC_ERR_CUDA: return "TC_ERR_CUDA";
        case TC_ERR_INTERNAL: return "TC_ERR_INTERNAL";
    }
    return "TC_ERR_UNKNOWN";
}

extern "C" const char* tc_last_error(const tc_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" tc_status tc_create(tc_ctx** out, int device) {
    if (!out) return TC_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return TC_ERR_UNSUPPORTED_DEVICE;  // no CUDA device: there is no fallback path by design
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return TC_ERR_CUDA;
    if (prop.major != 10) return TC_ERR_UNSUPPORTED_DEVICE;  // kernels are built for sm_100a only
    tc_ctx* ctx = (tc_ctx*)calloc(1, sizeof(tc_ctx));
    if (!ctx) return TC_ERR_INTERNAL;
    ctx->device = device;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->cc_major = prop.major;
    ctx->cc_minor = prop.minor;
    ctx->smem_optin = prop.sharedMemPerBlockOptin;
    ctx->l2_bytes = (size_t)prop.l2CacheSize;
    ctx->err[0] = 0;
    bool ok = cudaSetDevice(device) == cudaSuccess;
    {
        // the staging stream outranks the caller's: its GEMM CTAs are dispatched as soon as SMs free up, so the operands of
        // block n+1 are in place long before the W-builder of block n (hundreds of thousands of queued CTAs) has drained
        int prio_least = 0, prio_greatest = 0;
        ok = ok && cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest) == cudaSuccess;
        ok = ok && cudaStreamCreateWithPriority(&ctx->side_stream, cudaStreamNonBlocking, prio_greatest) == cudaSuccess;
    }
    ok = ok && cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess;
    for (int n = 0; n < TC_EV_RING; n++) {
        ok = ok && cudaEventCreateWithFlags(&ctx->ev_staged[n], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&ctx->ev_done[n], cudaEventDisableTiming) == cudaSuccess;
    }
    for (int n = 0; n < TC_TIMING_RING; n++) {
        ok = ok && cudaEventCreate(&ctx->ev_k0[n]) == cudaSuccess && cudaEventCreate(&ctx->ev_k1[n]) == cudaSuccess;
        ok = ok && cudaEventCreate(&ctx->ev_g0[n]) == cudaSuccess && cudaEventCreate(&ctx->ev_g1[n]) == cudaSuccess;
    }
    cudaEvent_t* timed[6] = {&ctx->ev_t0, &ctx->ev_t1, &ctx->ev_s0, &ctx->ev_s1, &ctx->ev_c0, &ctx->ev_c1};
    for (int n = 0; n < 6; n++) ok = ok && cudaEventCreate(timed[n]) == cudaSuccess;
    ok = ok && cudaMallocHost(&ctx->pinned, 64 * sizeof(double)) == cudaSuccess;
    // opt-in shared memory of the kernels: a per-device attribute, set here for this context's device
    ok = ok && tc_wbuild_configure() == cudaSuccess &&
         tc_stager_configure() == cudaSuccess && tc_microbench_configure() == cudaSuccess;
    if (!ok) {
        tc_destroy(ctx);
        return TC_ERR_CUDA;
    }
    *out = ctx;
    return TC_OK;
}

extern "C" tc_status tc_destroy(tc_ctx* ctx) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    cudaSetDevice(ctx->device);
    if (ctx->side_stream) cudaStreamDestroy(ctx->side_stream);
    cudaEvent_t evs[7] = {ctx->ev_fork, ctx->ev_t0, ctx->ev_t1, ctx->ev_s0, ctx->ev_s1, ctx->ev_c0, ctx->ev_c1};
    for (int n = 0; n < 7; n++)
        if (evs[n]) cudaEventDestroy(evs[n]);
    for (int n = 0; n < TC_EV_RING; n++) {
        if (ctx->ev_staged[n]) cudaEventDestroy(ctx->ev_staged[n]);
        if (ctx->ev_done[n]) cudaEventDestroy(ctx->ev_done[n]);
    }
    for (int n = 0; n < TC_TIMING_RING; n++) {
        cudaEvent_t t4[4] = {ctx->ev_k0[n], ctx->ev_k1[n], ctx->ev_g0[n], ctx->ev_g1[n]};
        for (int q = 0; q < 4; q++)
            if (t4[q]) cudaEventDestroy(t4[q]);
    }
    if (ctx->pinned) cudaFreeHost(ctx->pinned);
    if (ctx->plan_host) cudaFreeHost(ctx->plan_host);
    if (ctx->host_slab) cudaFree(ctx->host_slab);
    free(ctx);
    return TC_OK;
}

extern "C" tc_status tc_get_stats(const tc_ctx* ctx, tc_stats* out) {
    if (!ctx || !out) return TC_ERR_INVALID_ARG;
    *out = ctx->stats;
    return TC_OK;
}
