/*
 * tc_triples.h -- C-ABI of the B200-native closed-shell (T) energy library.
 *
 * What it computes (arxiv 2512.01055, "Accelerating CCSD(T) on GPUs"; citations are
 * PAPER.md line numbers):
 *
 *   E(T) = sum_{i>=j>=k} (2 - d_ij - d_jk) S_ijk                        eq. (1)
 *   S_ijk = sum_abc (W_abc + Vd_abc) R_abc / D_abc                      (virtual-index form of eq. (1))
 *   W_ijk^abc = P [ sum_d t_ij^ad (bd|ck) - sum_l t_il^ab (lj|kc) ]     eqs. (2),(5)
 *   Vd_ijk^abc = t_i^a (jb|kc) + t_j^b (ia|kc) + t_k^c (ia|jb)          eq. (3)
 *   D_ijk^abc = e_i + e_j + e_k - e_a - e_b - e_c                       Fig. 4 l.23
 *   R_abc = 4W_abc + W_bca + W_cab - 2W_acb - 2W_cba - 2W_bac           eq. (1) weights
 *   (pq|rs) = sum_Q B^Q_pq B^Q_rs                                       eq. (6)
 *
 * All arithmetic is FP64 and runs in hand-written sm_100a kernels; there is no CPU
 * fallback: on a machine without a compute-capability-10.x device every compute call
 * returns TC_ERR_UNSUPPORTED_DEVICE.
 *
 * Conventions common to all calls
 *   - No exceptions cross the boundary; every call returns a tc_status.  On error the
 *     output arguments are untouched and tc_last_error(ctx) describes the failure.
 *   - "device" pointers are CUDA device memory on the context's device, owned by the
 *     caller, read-only to the library unless stated, and must stay valid until the
 *     call returns.  "host" pointers are ordinary host memory.
 *   - All arrays are FP64 ("double"), dense, C order (last index fastest).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Work is enqueued on it.  When the (vv|vo) slices (or, for the streamed call, the
 *     amplitudes) do not all fit in the workspace, the library runs a blocked schedule
 *     and stages the operands of the next block on a side stream it owns while the
 *     current block's contraction runs on `stream`; that side stream is forked from and
 *     joined to `stream` with events, so the caller sees single-stream semantics.  In
 *     every other case all work is on `stream` itself.  Calls that return a host scalar
 *     synchronise `stream` once before returning.
 *   - The library performs no device allocation inside the compute calls: scratch
 *     space is the caller-allocated `workspace` (the paper's "pre-allocate and reuse"
 *     rule).  tc_workspace_bytes tells how much is needed.
 *
 * Triplet linear index (defines "a contiguous slice of triplets"):
 *   idx(i,j,k) = i(i+1)(i+2)/6 + j(j+1)/2 + k   for i >= j >= k >= 0.
 */
#ifndef TC_TRIPLES_H
#define TC_TRIPLES_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TC_OK = 0,
    TC_ERR_INVALID_ARG = 1,
    TC_ERR_UNSUPPORTED_DEVICE = 2,
    TC_ERR_WORKSPACE_TOO_SMALL = 3,
    TC_ERR_CUDA = 4,
    TC_ERR_INTERNAL = 5
} tc_status;

typedef struct tc_ctx tc_ctx; /* opaque; owns streams/events and a few KB of pinned memory */

/* Materialised integral blocks (device pointers). */
typedef struct {
    const double* vvvo; /* [x][d][b][c] = (bd|cx), o*v^3; slice x is contiguous (the paper's (vv|vo) block) */
    const double* ovoo; /* [j][k][l][c] = (lj|kc), o^3*v */
    const double* ovov; /* [j][k][b][c] = (jb|kc), o^2*v^2 */
} tc_int_blocks;

/* Density-fitting (or Cholesky, eq. (6)) factors (device pointers). */
typedef struct {
    int naux;
    const double* Boo; /* [Q][i][j] */
    const double* Bov; /* [Q][i][a] */
    const double* Bvv; /* [Q][a][b], symmetric in a,b */
} tc_df_factors;

/* ---- context ------------------------------------------------------------------- */

/* Create a context on CUDA device `device`.  Fails with TC_ERR_UNSUPPORTED_DEVICE if
 * there is no such device or its compute capability is not 10.x. */
tc_status tc_create(tc_ctx** ctx, int device);
tc_status tc_destroy(tc_ctx* ctx);
const char* tc_status_string(tc_status s);
const char* tc_last_error(const tc_ctx* ctx); /* never NULL; valid until the next call on ctx */

/* ---- a1: triplet scheduler (host, no GPU needed) -------------------------------- */

/* o(o+1)(o+2)/6, or -1 if o < 1. */
long long tc_triplet_count(int o);
/* idx -> (i,j,k) and the degeneracy weight 2 - d_ij - d_jk (0 for i=j=k). */
tc_status tc_triplet_decode(int o, long long idx, int* i, int* j, int* k, double* weight);
/* (i,j,k), i>=j>=k -> idx, or -1 if the arguments are not an ordered triplet below o. */
long long tc_triplet_index(int o, int i, int j, int k);
/* Multi-GPU sharding (the paper hands independent tile batches to the GPUs and sums the partial
 * energies): the contiguous range [first, first+count) of the linear triplet index
 * owned by `rank` of `world`.  The ranges tile [0, N_trip) and differ in size by at most one; each
 * rank runs tc_triples_energy_slice on its range with replicated inputs and the partial energies are
 * summed (one scalar all-reduce).  Host only. */
tc_status tc_triplet_partition(int o, int world, int rank, long long* first, long long* count);

/* ---- workspace ------------------------------------------------------------------ */

/* Bytes of device workspace tc_triples_energy / _slice need for a problem of this size.
 *   naux_or_0   : naux when DF factors will be passed, 0 when integral blocks are passed.
 *   hbm_budget  : upper bound the caller is willing to give (0 = no bound).  With DF
 *                 input the library materialises all (vv|vo) slices if they fit in the
 *                 budget, else it sizes an LRU cache of per-occupied-index slices.
 * Returns TC_ERR_WORKSPACE_TOO_SMALL if even the minimum does not fit the budget. */
tc_status tc_workspace_bytes(tc_ctx* ctx, int o, int v, int naux_or_0, size_t hbm_budget, size_t* bytes);

/* The same for tc_triples_energy_streamed (t2 stays on the host; DF input only). */
tc_status tc_workspace_bytes_streamed(tc_ctx* ctx, int o, int v, int naux, size_t hbm_budget, size_t* bytes);

/* The blocked schedule (what the library does when the per-occupied-index operands -- (vv|v.) slices,
 * amplitude rows -- are cached in `nslots` < o slots): the triplets are cut into blocks of bi x bj x bk occupied
 * indices, the operands of a block are made resident (LRU eviction), and the next block's missing operands are
 * staged while the current block computes.  This host-only call reports the plan for a triplet range:
 * number of blocks (= W-builder launches), operand loads (slice assemblies), and the block shape chosen.
 * Any output pointer may be NULL.  Returns TC_ERR_INVALID_ARG if nslots < 3 (a triplet needs three slices). */
tc_status tc_plan_summary(int o, long long first, long long count, int nslots,
                          long long* n_blocks, long long* n_loads, int* bi, int* bj, int* bk);

/* The plan itself, for validation (host only): recs_out[count][8] = (i, j, k, index of the triplet in the range,
 * block, slot of i, slot of j, slot of k) in execution order; loads_out[n_loads][4] = (block, occupied index,
 * slot, last block that used the slot or -1) -- n_loads from tc_plan_summary, TC_ERR_WORKSPACE_TOO_SMALL if
 * loads_capacity is less. */
tc_status tc_plan_dump(int o, long long first, long long count, int nslots,
                       int* recs_out, int* loads_out, long long loads_capacity);

/* ---- a2: integral staging from DF factors --------------------------------------- */

/* Assemble integral blocks on the device from DF factors with the library's FP64
 * tensor-core GEMM (eq. (6)).  Each output pointer may be NULL (skipped):
 *   vvvo_out [x0 <= x < x0+nx][d][b][c] (nx*v^3), ovoo_out (o^3 v), ovov_out (o^2 v^2).
 * Asynchronous on `stream`. */
tc_status tc_build_blocks(tc_ctx* ctx, int o, int v, const tc_df_factors* df,
                          int x0, int nx, double* vvvo_out, double* ovoo_out, double* ovov_out,
                          void* stream);

/* ---- a3-a7: the (T) energy ------------------------------------------------------ */

/* E(T) over all triplets.  Exactly one of `blocks` / `df` is non-NULL.
 *   eps_occ[o], eps_vir[v], t1[i][a], t2[i][j][a][b] (= t_ij^ab; precondition
 *   t_ij^ab == t_ji^ba): device.  t2 must be 16-byte aligned (it is a TMA operand; CUDA allocators
 *   return at least 256-byte alignment), else TC_ERR_INVALID_ARG.  Any o, v >= 1: odd v runs on the
 *   same kernel through a zero-padded copy of t2 in the workspace.  E_out: host.  */
tc_status tc_triples_energy(tc_ctx* ctx, int o, int v,
                            const double* eps_occ, const double* eps_vir,
                            const double* t1, const double* t2,
                            const tc_int_blocks* blocks, const tc_df_factors* df,
                            void* workspace, size_t workspace_bytes,
                            void* stream, double* E_out);

/* The same over triplets first .. first+count-1 of the linear index.
 *   S_dev (device, [count], optional): receives S_ijk of each triplet (0 for i=j=k).
 *   E_partial_out (host): sum of weight * S_ijk over the range. */
tc_status tc_triples_energy_slice(tc_ctx* ctx, int o, int v,
                                  const double* eps_occ, const double* eps_vir,
                                  const double* t1, const double* t2,
                                  const tc_int_blocks* blocks, const tc_df_factors* df,
                                  void* workspace, size_t workspace_bytes,
                                  void* stream, long long first, long long count,
                                  double* S_dev, double* E_partial_out);

/* The same with NO allocation anywhere on its path, for callers that cannot allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the scratch the kernels use (what `workspace` is above) lives in
 * one file-scope device array of TC_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds
 * until the process exits.  The caller passes only inputs and outputs (arguments as in tc_triples_energy_slice).
 *   Limit: the problem must fit the array with everything resident, i.e. tc_workspace_bytes(ctx, o, v, naux_or_0, 0) <=
 *   TC_STATIC_SCRATCH_BYTES (e.g. (o,v,naux) = (8,40,120), (6,72,24), (10,48,150)); beyond that TC_ERR_WORKSPACE_TOO_SMALL with
 *   the two sizes in tc_last_error, and nothing is launched.
 *   Sharing: all calls on a device use the same array and find the last call's contents in it.  The call clears the part it
 *   uses first (stream ordered), so a result never depends on an earlier call; calls that OVERLAP on one GPU (different
 *   streams or threads) race on the array: serialise them.
 *   Calls no cudaMalloc / cudaFree / allocating library routine; synchronises `stream` once to return the host double, like
 *   the other energy calls. */
#define TC_STATIC_SCRATCH_BYTES (64u << 20)
tc_status tc_triples_energy_static(tc_ctx* ctx, int o, int v,
                                   const double* eps_occ, const double* eps_vir,
                                   const double* t1, const double* t2,
                                   const tc_int_blocks* blocks, const tc_df_factors* df,
                                   void* stream, long long first, long long count,
                                   double* S_dev, double* E_partial_out);

/* Host-resident amplitudes (the paper streams t2 pieces with cudaMemcpyAsync under the integral
 * build, Fig. 2 l.6, 9: at o=150, v=1150 the amplitudes are 238 GB).  As
 * tc_triples_energy_slice with DF input, except that `t2_host` is HOST memory (pinned for the copies to
 * overlap; pageable works but serialises) and is never resident as a whole: the rows t2[x][:][:][:] that
 * a block of triplets needs are copied into a device ring of slots on the library's side stream while the
 * previous block computes, next to the slice cache.  eps, t1, DF factors: device.  Workspace size:
 * tc_workspace_bytes_streamed. */
tc_status tc_triples_energy_streamed(tc_ctx* ctx, int o, int v,
                                     const double* eps_occ, const double* eps_vir,
                                     const double* t1, const double* t2_host,
                                     const tc_df_factors* df,
                                     void* workspace, size_t workspace_bytes,
                                     void* stream, long long first, long long count,
                                     double* S_dev, double* E_partial_out);

/* The paper's own loop order (the abcijk scheme; Fig. 1; Fig. 2): virtual tile
 * orbits {A >= B >= C} (tile edge 16) outer, all triplets i >= j >= k inner.  For each orbit the (vv|vo) integrals are
 * rebuilt from the DF factors restricted to the orbit's tiles (Fig. 2 l.7, 10), so the footprint beside t2 and (ov|ov) is
 * O(o v 16^2) instead of o v^3; a launch takes two orbits (all triplets x each), and the next launch's integrals are
 * assembled on the library's side stream while the current one's contraction runs (two sets of staging buffers).  Same kernels, same result as tc_triples_energy: E = sum over orbits of the orbit's energy
 *   E_orbit = sum_{i>=j>=k} (2 - d_ij - d_jk) sum_{(a,b,c) in orbit} (W + Vd) R / D.
 * Orbits orbit_first .. orbit_first+orbit_count-1 of the enumeration A >= B >= C (A slowest) are computed;
 * E_orbit_dev (device, [orbit_count], optional) receives their energies, E_out (host) their sum.  DF input only;
 * t2 device-resident, 16-byte aligned.  Workspace: tc_workspace_bytes_abcijk.  tc_tile_orbit_count(v) = nb(nb+1)(nb+2)/6,
 * nb = ceil(v/16). */
long long tc_tile_orbit_count(int v);
tc_status tc_workspace_bytes_abcijk(tc_ctx* ctx, int o, int v, int naux, size_t* bytes);
tc_status tc_triples_energy_abcijk(tc_ctx* ctx, int o, int v,
                                   const double* eps_occ, const double* eps_vir,
                                   const double* t1, const double* t2,
                                   const tc_df_factors* df,
                                   void* workspace, size_t workspace_bytes,
                                   void* stream, long long orbit_first, long long orbit_count,
                                   double* E_orbit_dev, double* E_out);

/* End-to-end variant with HOST inputs: copies the DF factors, amplitudes and orbital
 * energies to the device, assembles the integrals, computes E(T) over triplets
 * first .. first+count-1, returns it on the host.  This is the one call that allocates
 * device memory: a single slab (inputs + workspace) owned by the context, kept between
 * calls, grown when a larger problem arrives and freed by tc_destroy.
 * If bytes_h2d != NULL it receives the bytes copied host->device. */
tc_status tc_triples_energy_host(tc_ctx* ctx, int o, int v, int naux,
                                 const double* eps_occ, const double* eps_vir,
                                 const double* t1, const double* t2,
                                 const double* Boo, const double* Bov, const double* Bvv,
                                 long long first, long long count,
                                 double* E_out, size_t* bytes_h2d);

/* Debug/validation: W_ijk^abc (eqs. (2),(5)) of one triplet written to W_dev[a][b][c]
 * (device, v^3) by the same tile kernels that feed the fused epilogue.  Any order of
 * i,j,k is accepted.  Used by the parity tests only (allocates its own scratch). */
tc_status tc_debug_W_triplet(tc_ctx* ctx, int o, int v, int i, int j, int k,
                             const double* t2, const tc_int_blocks* blocks,
                             double* W_dev, void* stream);
#define TC_KERNEL_TMA 1 /* tc_stats.kernel: the TMA/mbarrier/TMEM W-builder (the only one there is) */

/* ---- statistics of the last energy call ----------------------------------------- */

typedef struct {
    long long n_triplets;        /* triplets in the range with non-zero weight          */
    long long n_work_units;      /* (triplet, virtual tile orbit) units executed         */
    long long n_kernel_launches; /* kernels this library launched during the call        */
    double    flop_contraction;  /* executed o^3v^4 + o^4v^3 contraction flop (useful)   */
    double    ms_total;          /* device time of the whole call (CUDA events)          */
    double    ms_contraction;    /* device time of the fused W-builder kernels           */
    double    ms_staging;        /* device time of DF->block assembly (0 with blocks)    */
    long long slices_built;      /* (vv|v.) slices assembled from DF during the call     */
    int       kernel;            /* W-builder that ran: TC_KERNEL_TMA (0 if the range was empty) */
    int       padded;            /* 1: odd v, t2 used through a zero-padded copy (row length v+1) */
    long long n_blocks;          /* blocked schedule: W-builder launches (0 = everything resident) */
    long long t2_rows_copied;    /* streamed call: amplitude rows copied host->device    */
    double    bytes_h2d;         /* streamed call: bytes copied host->device             */
    double    ms_kernels;        /* sum of the W-builder launches alone (events around each launch)         */
    double    ms_staging_side;   /* blocked schedule: device time of the side-stream staging (sum of spans)  */
    double    staging_first_ms, staging_last_ms;          /* side-stream staging interval, relative to call start */
    double    contraction_first_ms, contraction_last_ms;  /* first W-builder start / last W-builder end          */
} tc_stats;
tc_status tc_get_stats(const tc_ctx* ctx, tc_stats* out);

/* ---- microbenchmarks: the roofline denominators ---------------------------------- */

/* Register-resident FP64 tensor-core (mma.sync m8n8k4 f64 -> DMMA.8x8x4) throughput.
 * Runs for about `seconds`; returns sustained TFLOP/s and the best single-launch
 * (burst) TFLOP/s. */
tc_status tc_bench_dmma_peak(tc_ctx* ctx, double seconds, double* tflops_sustained, double* tflops_burst);
/* The same with scalar FP64 FMA (DFMA). */
tc_status tc_bench_dfma_peak(tc_ctx* ctx, double seconds, double* tflops_sustained, double* tflops_burst);
/* Device copy bandwidth (read+write bytes / time), GB/s, over `bytes` per direction
 * of caller-provided device buffers. */
tc_status tc_bench_copy_bw(tc_ctx* ctx, void* dst_dev, const void* src_dev, size_t bytes, int reps, double* gbs);
/* What the W-builder's consumer loop can reach: stand-alone kernels with the production kernel's warp
 * tile (8 warps x 32 x 32, K chunk 4: 8 LDS.64 + 16 DMMA.8x8x4 per chunk), no flush, no epilogue.
 *   variant 0: fragments from shared memory, no synchronisation      (the LDS + DMMA floor)
 *   variant 1: + the 3-stage full/empty mbarrier ring, producers only arrive
 *   variant 2: + real TMA producers streaming a device buffer (the production operand path)
 * Returns TFLOP/s over about `seconds`.  `scratch_dev` (>= 64 MB, device) is the buffer variant 2 streams. */
tc_status tc_bench_ring_peak(tc_ctx* ctx, int variant, double seconds, void* scratch_dev, size_t scratch_bytes, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* TC_TRIPLES_H */
