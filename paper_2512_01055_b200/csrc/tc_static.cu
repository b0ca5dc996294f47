// tc_static.cu -- tc_triples_energy_static: the (T) energy of a triplet range with NO allocation anywhere on its path.
//
// For callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
// Everything the kernels of the energy call use as scratch (triplet records, per-unit partial sums, S_ijk, the assembled
// (ov|oo)^T / (ov|ov) blocks, the tiled (vv|v.) slices, the padded t2 copy for odd v -- the workspace of tc_workspace_bytes)
// lives in ONE file-scope device array of TC_STATIC_SCRATCH_BYTES.  Every GPU that loads the library holds that array until the
// process exits.  The caller still passes inputs and outputs.
//
// The array's name is a host-side stand-in in host code, not a device address: its device address is resolved here with
// cudaGetSymbolAddress, once per device and with that device current, and that pointer is what the kernels get.
//
// Sharing: every call on a device uses the same array and finds the previous call's contents in it.  The call clears the part
// it is going to use before anything else is enqueued, so a result never depends on an earlier call; two calls that OVERLAP on
// one GPU (different streams, different threads) race on the array -- serialise them.
#include <mutex>

#include "tc_common.cuh"

namespace {

static __device__ __align__(256) unsigned char g_static_scratch[TC_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void* g_scratch_addr[kMaxDevices];   // device address of g_static_scratch on device n (NULL: not resolved yet)
std::mutex g_scratch_mutex;

// the device address of the scratch array on the CURRENT device (ctx->device has been made current by the caller)
tc_status scratch_address(tc_ctx* ctx, void** out) {
    const int dev = ctx->device;
    if (dev < 0 || dev >= kMaxDevices) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "device %d outside [0,%d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        TC_CUDA(ctx, cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (uintptr_t)p % 256 != 0) TC_FAIL(ctx, TC_ERR_INTERNAL, "static scratch resolved to %p", p);
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return TC_OK;
}

}  // namespace

extern "C" tc_status tc_triples_energy_static(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                              const double* t1, const double* t2, const tc_int_blocks* blocks,
                                              const tc_df_factors* df, void* stream, long long first, long long count,
                                              double* S_dev, double* E_partial_out) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "o and v must be >= 1 (got o=%d v=%d)", o, v);
    if ((blocks != nullptr) == (df != nullptr)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "exactly one of blocks / df must be given");
    if (df && df->naux < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "df->naux must be >= 1");
    // everything resident (no slice cache, hence no schedule tables either): the size tc_workspace_bytes reports without a budget
    size_t need = 0;
    tc_status st = tc_workspace_bytes(ctx, o, v, df ? df->naux : 0, 0, &need);
    if (st != TC_OK) return st;
    if (need > (size_t)TC_STATIC_SCRATCH_BYTES)
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL,
                "tc_triples_energy_static: o=%d v=%d needs %zu bytes of scratch, the static scratch holds %zu "
                "(TC_STATIC_SCRATCH_BYTES); use tc_triples_energy_slice with a caller-allocated workspace",
                o, v, need, (size_t)TC_STATIC_SCRATCH_BYTES);
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    void* scratch = nullptr;
    st = scratch_address(ctx, &scratch);
    if (st != TC_OK) return st;
    // the array keeps the last call's contents: start from zeros (stream ordered, ahead of everything the call enqueues)
    TC_CUDA(ctx, cudaMemsetAsync(scratch, 0, need, (cudaStream_t)stream));
    return tc_triples_energy_slice(ctx, o, v, eps_occ, eps_vir, t1, t2, blocks, df, scratch, (size_t)TC_STATIC_SCRATCH_BYTES, stream,
                                   first, count, S_dev, E_partial_out);
}
