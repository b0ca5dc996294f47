// tc_common.cuh -- shared declarations of the (T) library's translation units.
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/tc_triples.h"

constexpr int TC_EV_RING = 16;     // fork/join events of the staging pipeline (blocked schedule)
constexpr int TC_TIMING_RING = 64;  // timing-event pairs harvested as they are recycled

struct tc_ctx {
    int device;
    int sm_count;
    int cc_major, cc_minor;
    size_t smem_optin;
    size_t l2_bytes;
    // a2 on a side stream (blocked schedule): the slices / amplitude rows of block n+1 are staged here while the
    // W-builder of block n runs on the caller's stream
    cudaStream_t side_stream;
    cudaEvent_t ev_fork;                    // caller's stream -> side stream at the start of a call
    cudaEvent_t ev_staged[TC_EV_RING];      // side -> main: the operands of block n are in place
    cudaEvent_t ev_done[TC_EV_RING];        // main -> side: the W-builder of block n has finished (its slots may be reused)
    cudaEvent_t ev_k0[TC_TIMING_RING], ev_k1[TC_TIMING_RING];   // W-builder launch brackets (main stream)
    cudaEvent_t ev_g0[TC_TIMING_RING], ev_g1[TC_TIMING_RING];   // staging brackets (side stream)
    cudaEvent_t ev_t0, ev_t1, ev_s0, ev_s1, ev_c0, ev_c1;
    double* pinned;                // a few doubles of pinned host memory for scalar results
    void* host_slab;               // device slab of tc_triples_energy_host, kept between calls (grow-only)
    size_t host_slab_bytes;
    void* plan_host;               // pinned host staging of the blocked schedule's tables (grow-only)
    size_t plan_host_bytes;
    tc_stats stats;
    char err[512];
};

#define TC_FAIL(ctx, code, ...)                                        \
    do {                                                               \
        if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__); \
        return (code);                                                 \
    } while (0)

#define TC_CUDA(ctx, call)                                                                  \
    do {                                                                                    \
        cudaError_t e__ = (call);                                                           \
        if (e__ != cudaSuccess)                                                             \
            TC_FAIL(ctx, TC_ERR_CUDA, "%s:%d: %s -> %s", __FILE__, __LINE__, #call,         \
                    cudaGetErrorString(e__));                                               \
    } while (0)

// ---- FP64 tensor-core primitive -------------------------------------------------------
// mma.sync m8n8k4 f64: the only FP64 MMA shape that is a single native instruction on
// sm_100a (SASS DMMA.8x8x4).  Fragment layout (PTX ISA):
//   A[row = lane>>2][k = lane&3], B[k = lane&3][col = lane>>2],
//   C[row = lane>>2][col = 2*(lane&3) + {0,1}].
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// ---- cp.async helpers (LDGSTS) --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
// 16-byte copy, src_bytes in [0,16] valid bytes, the rest zero-filled.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes));
}
// 8-byte copy, src_bytes in {0,8}.
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, int src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// ---- internal entry points (defined in the other .cu files) ---------------------------

// a2: C = A^T B with K-major operands and a 2-level output index map (tc_stager.cu).
//   A[K][M], B[K][N] (leading dimensions lda, ldb), row = r1*R2 + r2, col = c1*C2 + c2,
//   C[r1*sr1 + r2*sr2 + c1*sc1 + c2*sc2] = sum_k A[k][row] B[k][col].
cudaError_t tc_launch_df_gemm(const double* A, size_t lda, const double* B, size_t ldb, int M, int N, int K,
                              int R2, long long sr1, long long sr2, int C2, long long sc1, long long sc2,
                              double* C, cudaStream_t stream);
// a2 for the W-builder: slices x0 .. x0+nx-1, I_x[d][b][c] = (bd|cx) = sum_Q Bvv[Q][d][b] Bov[Q][x][c], written in the tiled
// layout (slice x at dst + (x - x0) * slice_stride; the zero padding is NOT written: the caller clears the slots once).
cudaError_t tc_launch_df_slices_tiled(const double* Bvv, const double* Bov, int o, int v, int naux, int x0, int nx,
                                      double* dst, size_t slice_stride, cudaStream_t stream);
// abcijk schedule: the tile-restricted parts of all o slices for one tile orbit (A, B, C), chunk layout over the 3 x 3 local tile
// pairs [lu][lv][K chunk][z][n1][k][n2 8]; x at dst + x * x_stride
cudaError_t tc_launch_df_slices_orbit(const double* Bvv, const double* Bov, int o, int v, int naux, int tA, int tB, int tC, double* dst,
                                      size_t x_stride, cudaStream_t stream);
// the same layout from a materialised array src[k][b][c] (K rows k, row length ld >= v): a slice of the caller's (vv|vo)
// block (K = v) or an amplitude row t2[y] (K = o); writes the padding too
cudaError_t tc_launch_tile_slice(const double* src, int K, int v, size_t ld, double* dst, cudaStream_t stream);
// (ov|oo)^T[z][x][m][ldo] from the caller's block ovoo[z][x][l][m] (blocks input); the pad column is zeroed
cudaError_t tc_launch_transpose_ovoo(const double* ovoo, int o, int v, int ldo, double* dst, cudaStream_t stream);

// K chunks (of 4) per tile pair in the tiled slice layout: rounded up to even, so that the steps that consume two K chunks per
// ring stage (ragged n1 / n2 tiles, tc_wbuild_tma.cu "paired" modes) never read past a tile; the extra chunk is zero padding
__host__ __device__ inline int tc_tiled_kchunks(int K) {
    const int n = (K + 3) / 4;
    return n + (n & 1);
}

// a3-a6: fused W-builder + epilogue over a list of triplets (tc_wbuild_tma.cu, tc_wbuild.cu).
// One record per triplet.  The slots say where the per-occupied-index operands of the triplet live: slice slot s[p]
// holds the (vv|v.) slice of occ[p], amplitude slot t[p] holds the row t2[occ[p]][:][:][:] (slot = index when
// everything is resident; the blocked schedule and the host-resident t2 path cache them in fewer slots).
struct tc_trip_rec {
    int occ[3];   // i >= j >= k (tc_debug_W_triplet: any order)
    int row;      // row of partial[]
    int s[3];     // slice slots of i, j, k
    int pad0;
    int t[3];     // amplitude-row slots of i, j, k
    int pad1;
};
static_assert(sizeof(tc_trip_rec) == 48, "tc_trip_rec is read as three int4");

struct tc_wbuild_args {
    int o, v;
    int ldv;                         // row length (doubles) of t2: v, or v + 1 for odd v (zero-padded copy)
    int ldo;                         // row length of (ov|oo)^T: o rounded up to even
    const double* eps_occ;
    const double* eps_vir;
    const double* t1;
    const double* t2;                // [tslot][y][a][ldv], amplitude rows t2_row_stride doubles apart
    size_t t2_row_stride;
    const double* slices;            // slot s at slices + s * slice_stride, in the W-builder's tiled layout
                                     // [n1 tile][n2 tile][K chunk][z][n1 16][k 4][n2 8], zero padded (tc_wbuild_slice_doubles)
    size_t slice_stride;             // doubles
    int orbit_local;                 // 1 (abcijk schedule): the slices hold only the 3 x 3 tile pairs of each tile orbit of the launch,
                                     // pair (lu, lv) = positions of the n1 / n2 tile in (A, B, C)
    size_t orbit_stride;             // orbit_local: doubles between the slice sets of consecutive orbits of the launch
    const double* ovooT;             // [z][x][m][ldo] = (l z | x m): the (ov|oo) block with the contracted index fastest
    const double* ovov;              // [j][k][b][c] (natural layout; read by the epilogue only)
    const tc_trip_rec* recs;         // device array [n_trip]
    int n_trip;
    double* partial;                 // device [n_trip][n_orbits] per-unit partial sums
    int n_orbits;
    double* W_debug;                 // optional v^3 output of W for n_trip == 1
};
// TMA descriptors of the tensor-box operand streams (tc_wbuild_tma.cu); the slices are read with plain bulk copies.
struct tc_wbuild_maps {
    CUtensorMap T2h;    // t2 as hole B        [tslot][l][n1][n2], box of 16 n1 rows
    CUtensorMap T2h8;   // the same with a box of 8 n1 rows (steps whose n1 tile has at most 8 valid indices)
    CUtensorMap T2p;    // t2 as particle A    [tslot][y][m][d]
    CUtensorMap OvooT;  // (ov|oo)^T as hole A [z][x][m][l]
    bool valid;
};
// n_tslots amplitude rows behind a.t2.
cudaError_t tc_wbuild_make_maps(const tc_wbuild_args& a, int n_tslots, tc_wbuild_maps* out);
int tc_wbuild_tile();                                  // virtual tile edge T
int tc_wbuild_num_orbits(int v);                       // nb(nb+1)(nb+2)/6
size_t tc_wbuild_slice_doubles(int v);                 // doubles of one slice in the tiled layout
cudaError_t tc_launch_wbuild(const tc_wbuild_args& a, const tc_wbuild_maps* maps,
                             const int4* orbits /*device [n_orbits]: (A,B,C,0), A>=B>=C*/, cudaStream_t stream);
// per-device kernel attributes (opt-in shared memory); called by tc_create with the device current
cudaError_t tc_wbuild_configure();
cudaError_t tc_stager_configure();
cudaError_t tc_microbench_configure();

// dst[r][0..v) = src[r][0..v), dst rows ldd doubles apart (ldd >= v; the pad is zeroed): TMA needs 16-byte row strides
cudaError_t tc_launch_pad_rows(double* dst, size_t ldd, const double* src, size_t lds, size_t nrows, int v, cudaStream_t stream);

// a7: deterministic reductions (tc_reduce.cu).
//   recs[t] = decode(first + t) with row = t and slots = indices; w[t] = 2 - d_ij - d_jk
cudaError_t tc_launch_make_triplets(int o, long long first, int n, tc_trip_rec* recs, double* w, cudaStream_t stream);
//   S[dest ? dest[t] : t] = sum_u partial[t][u], fixed order
cudaError_t tc_launch_reduce_units(const double* partial, int n_trip, int n_units, const int* dest, double* S, cudaStream_t stream);
//   abcijk schedule: S[t] = (first ? 0 : S[t]) + partial[t];  *E_orbit = sum_t w[t] * partial[t] (fixed order, one block)
cudaError_t tc_launch_accumulate_orbit(const double* partial, int stride, const double* w, long long n, int first, double* S,
                                       double* E_orbit, cudaStream_t stream);
//   *E = sum_t w[t] * S[t], fixed order, one block
cudaError_t tc_launch_reduce_energy(const double* S, const double* w, long long n, double* E, cudaStream_t stream);

// microbenchmarks (tc_microbench.cu)
cudaError_t tc_micro_dmma(int sm_count, int iters, double* sink, cudaStream_t stream, double* flop_out);
cudaError_t tc_micro_dfma(int sm_count, int iters, double* sink, cudaStream_t stream, double* flop_out);
cudaError_t tc_micro_copy(void* dst, const void* src, size_t bytes, int sm_count, cudaStream_t stream);
