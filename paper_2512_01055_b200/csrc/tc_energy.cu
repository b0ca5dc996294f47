// tc_energy.cu -- the C-ABI compute calls: argument checks, workspace carving, and the
// launch sequence  scheduler (a1) -> stager (a2) -> fused W-builder/epilogue (a3-a6) -> reductions (a7).
//
// Two regimes.  RESIDENT: every (vv|v.) slice (and t2) is in HBM; one W-builder launch per batch of triplets, all on
// the caller's stream.  BLOCKED (DF input whose slices do not fit, or host-resident t2): the per-occupied-index
// operands are cached in slots, the triplets are executed block by block (tc_plan.cu), and the operands of block n+1
// are staged on the library's side stream while the W-builder of block n runs on the caller's stream.
#include <algorithm>
#include <vector>

#include "tc_plan.h"

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

enum Mode { MODE_BLOCKS = 0, MODE_DF = 1, MODE_STREAMED = 2, MODE_ABCIJK = 3 };

// How the caller's workspace is carved.  Everything the compute calls need lives here
// (pre-allocate and reuse; no device allocation inside the call).
struct Layout {
    size_t off_orbits, off_recs, off_dest, off_w, off_S, off_partial, off_E;
    size_t off_t2;      // zero-padded copy of t2 (odd v, resident t2) or the amplitude-row slots (streamed)
    size_t off_ovooT;   // (ov|oo)^T [z][x][m][ldo]: assembled from DF, or transposed from the caller's block
    size_t off_ovov;    // (ov|ov) assembled from DF
    size_t off_vvvo;    // slice slots in the W-builder's tiled layout: assembled from DF, or re-tiled from the caller's block
    size_t total;
    int n_orbits;
    int batch;          // triplets per W-builder launch (resident regime)
    int n_slots;        // resident (vv|v.) slices; < o: blocked schedule
    int ldv;            // row length of the TMA-addressed t2: v, or v + 1 when v is odd
    int ldo;            // row length of (ov|oo)^T: o rounded up to even
    size_t slice_stride, t2row_stride;   // doubles
    size_t off_Eorb;    // abcijk schedule: per-orbit partial energies [n_orbits]
    size_t orbit_buf_stride;   // abcijk schedule: doubles between the two staging buffers (o tile-restricted slices each)
};

#ifndef TC_ORBIT_GROUP
#define TC_ORBIT_GROUP 2
#endif
constexpr size_t kPartialBudget = (size_t)256 << 20;
// abcijk schedule: tile orbits per W-builder launch.  One orbit is N_trip equal units, i.e. N_trip / 148 waves with a ragged last
// one (cfg1: 10.3 -> 11); two orbits of different length per launch smooth that out for one more staging buffer set.
constexpr int kOrbitGroup = TC_ORBIT_GROUP;

// bounded == false: size for everything resident (tc_workspace_bytes with hbm_budget 0).
bool make_layout(int o, int v, int naux, Mode mode, bool bounded, size_t budget, Layout* L) {
    const long long ntrip = (long long)o * (o + 1) * (o + 2) / 6;
    L->n_orbits = tc_wbuild_num_orbits(v);
    long long batch = (long long)(kPartialBudget / ((size_t)L->n_orbits * sizeof(double)));
    if (batch < 1) batch = 1;
    if (batch > ntrip) batch = ntrip;
    if (batch * L->n_orbits > 0x7fffffffLL) batch = 0x7fffffffLL / L->n_orbits;
    L->batch = (int)batch;
    L->ldv = v + (v & 1);
    L->ldo = o + (o & 1);
    const bool pad = L->ldv != v;
    const size_t O = o, V = v, LD = L->ldv;
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t at = off;
        off += align_up(bytes);
        return at;
    };
    L->off_orbits = take(sizeof(int4) * (size_t)L->n_orbits);
    L->off_recs = take(sizeof(tc_trip_rec) * (size_t)ntrip);
    L->off_dest = take(sizeof(int) * (size_t)ntrip);
    L->off_w = take(sizeof(double) * (size_t)ntrip);
    L->off_S = take(sizeof(double) * (size_t)ntrip);
    L->off_partial = take(sizeof(double) * (size_t)L->batch * L->n_orbits);
    L->off_E = take(sizeof(double) * 8);
    L->off_t2 = L->off_ovov = 0;
    L->slice_stride = align_up(sizeof(double) * tc_wbuild_slice_doubles(v)) / sizeof(double);
    L->t2row_stride = align_up(sizeof(double) * O * V * LD) / sizeof(double);
    L->n_slots = o;
    L->off_ovooT = take(sizeof(double) * O * O * V * (size_t)L->ldo);
    if (mode != MODE_STREAMED && pad) L->off_t2 = take(sizeof(double) * O * L->t2row_stride);   // TMA needs 16-byte row strides
    L->off_Eorb = 0;
    L->orbit_buf_stride = 0;
    if (mode == MODE_ABCIJK) {
        // tile-restricted slices: 3 x 3 local tile pairs instead of nb^2, for all o occupied indices, double buffered
        L->off_ovov = take(sizeof(double) * O * O * V * V);
        L->slice_stride = align_up(sizeof(double) * 9 * (size_t)tc_tiled_kchunks(v) * 1024) / sizeof(double);
        L->orbit_buf_stride = O * L->slice_stride;
        L->off_vvvo = take(sizeof(double) * 2 * kOrbitGroup * L->orbit_buf_stride);   // two sets (double buffering) of kOrbitGroup orbits
        L->off_Eorb = take(sizeof(double) * (size_t)L->n_orbits);
    } else if (mode == MODE_BLOCKS) {
        L->off_vvvo = take(sizeof(double) * O * L->slice_stride);
    } else {
        L->off_ovov = take(sizeof(double) * O * O * V * V);
        const size_t per_slot = sizeof(double) * (L->slice_stride + (mode == MODE_STREAMED ? L->t2row_stride : 0));
        long long slots = o;
        if (bounded) {
            if (off >= budget) return false;
            const long long fit = (long long)((budget - off) / per_slot);
            if (fit < slots) slots = fit;
        }
        // fewer slots than slices: the blocked schedule (a triplet needs three operands resident)
        if (slots < 3 && slots < o) return false;
        L->n_slots = (int)slots;
        L->off_vvvo = take(sizeof(double) * L->slice_stride * (size_t)slots);
        if (mode == MODE_STREAMED) L->off_t2 = take(sizeof(double) * L->t2row_stride * (size_t)slots);
    }
    L->total = off;
    return !bounded || off <= budget;
}

bool is_device_ptr(const void* p) {
    if (!p) return false;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

tc_status check_common(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir, const double* t1,
                       const double* t2, bool t2_on_host, const tc_int_blocks* blocks, const tc_df_factors* df) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "o and v must be >= 1 (got o=%d v=%d)", o, v);
    if ((blocks != nullptr) == (df != nullptr)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "exactly one of blocks / df must be given");
    if (!is_device_ptr(eps_occ) || !is_device_ptr(eps_vir) || !is_device_ptr(t1))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "eps_occ, eps_vir, t1 must be device pointers");
    if (!t2_on_host && !is_device_ptr(t2)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "t2 must be a device pointer");
    if (!t2_on_host && (uintptr_t)t2 % 16 != 0)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "t2 must be 16-byte aligned (TMA operand; every CUDA allocator returns at least 256-byte alignment)");
    if (t2_on_host && (!t2 || is_device_ptr(t2))) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "t2_host must be a host pointer");
    if (blocks && (!is_device_ptr(blocks->vvvo) || !is_device_ptr(blocks->ovoo) || !is_device_ptr(blocks->ovov)))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "blocks->vvvo/ovoo/ovov must be device pointers");
    if (df && (df->naux < 1 || !is_device_ptr(df->Boo) || !is_device_ptr(df->Bov) || !is_device_ptr(df->Bvv)))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "df->naux must be >= 1 and df->Boo/Bov/Bvv device pointers");
    return TC_OK;
}

void fill_orbits(int v, std::vector<int4>& orb) {
    const int T = tc_wbuild_tile();
    const int nb = (v + T - 1) / T;
    orb.clear();
    for (int A = 0; A < nb; A++)
        for (int B = 0; B <= A; B++)
            for (int C = 0; C <= B; C++) orb.push_back(make_int4(A, B, C, 0));
}

// ---- a2 launches: eq. (6) by the DMMA GEMM ----
// natural layouts (tc_build_blocks): slices x0 .. x0+nx-1 as [x][d][b][c]
cudaError_t launch_slices_natural(const tc_df_factors* df, int o, int v, int x0, int nx, double* dst, cudaStream_t st) {
    // rows (d,b) -> (d*v + b)*v; cols (x,c) -> x*v^3 + c
    return tc_launch_df_gemm(df->Bvv, (size_t)v * v, df->Bov + (size_t)x0 * v, (size_t)o * v, v * v, nx * v, df->naux,
                             /*R2*/ 1, /*sr1*/ (long long)v, /*sr2*/ 0, /*C2*/ v, /*sc1*/ (long long)v * v * v, /*sc2*/ 1, dst, st);
}
cudaError_t launch_ovoo_natural(const tc_df_factors* df, int o, int v, double* dst, cudaStream_t st) {
    // ovoo[j][k][l][c]: rows (l,j) -> l*v + j*o*o*v; cols (k,c) -> k*o*v + c
    const long long O = o, V = v;
    return tc_launch_df_gemm(df->Boo, (size_t)(O * O), df->Bov, (size_t)(O * V), o * o, o * v, df->naux,
                             /*R2*/ o, /*sr1*/ V, /*sr2*/ O * O * V, /*C2*/ v, /*sc1*/ O * V, /*sc2*/ 1, dst, st);
}
// the W-builder's hole A operand: (ov|oo)^T[z][x][m][ldo] = (l z | x m) = sum_Q Boo[Q][l][z] Bov[Q][x][m]
cudaError_t launch_ovooT(const tc_df_factors* df, int o, int v, int ldo, double* dst, cudaStream_t st) {
    // rows (l,z) -> l + z*o*v*ldo; cols (x,m) -> x*v*ldo + m*ldo
    const long long O = o, V = v, LD = ldo;
    return tc_launch_df_gemm(df->Boo, (size_t)(O * O), df->Bov, (size_t)(O * V), o * o, o * v, df->naux,
                             /*R2*/ o, /*sr1*/ 1, /*sr2*/ O * V * LD, /*C2*/ v, /*sc1*/ V * LD, /*sc2*/ LD, dst, st);
}
cudaError_t launch_ovov(const tc_df_factors* df, int o, int v, double* dst, cudaStream_t st) {
    // ovov[j][k][b][c]: rows (j,b) -> j*o*v^2 + b*v; cols (k,c) -> k*v^2 + c
    const long long O = o, V = v;
    return tc_launch_df_gemm(df->Bov, (size_t)(O * V), df->Bov, (size_t)(O * V), o * v, o * v, df->naux,
                             /*R2*/ v, /*sr1*/ O * V * V, /*sr2*/ V, /*C2*/ v, /*sc1*/ V * V, /*sc2*/ 1, dst, st);
}

// number of i=j=k triplets (weight 0) in [first, first+count): idx(i,i,i) = i(i+1)(i+2)/6 + i(i+1)/2 + i
long long count_diagonal(int o, long long first, long long count) {
    long long n = 0;
    for (long long i = 0; i < o; i++) {
        const long long idx = i * (i + 1) * (i + 2) / 6 + i * (i + 1) / 2 + i;
        if (idx >= first && idx < first + count) n++;
    }
    return n;
}

struct TimingRing {
    cudaEvent_t *e0, *e1;
    long long used = 0;
    double total_ms = 0;
    TimingRing(cudaEvent_t* a, cudaEvent_t* b) : e0(a), e1(b) {}
    void harvest(int slot) {
        float ms = 0;
        if (cudaEventSynchronize(e1[slot]) == cudaSuccess && cudaEventElapsedTime(&ms, e0[slot], e1[slot]) == cudaSuccess)
            total_ms += ms;
    }
    int next() {
        const int slot = (int)(used % TC_TIMING_RING);
        if (used >= TC_TIMING_RING) harvest(slot);
        used++;
        return slot;
    }
    void finish() {
        const long long n = std::min<long long>(used, TC_TIMING_RING);
        const long long start = used - n;
        for (long long q = start; q < used; q++) harvest((int)(q % TC_TIMING_RING));
        used = 0;
    }
};

// the energy call proper; t2 is a device pointer (MODE_BLOCKS / MODE_DF) or a host pointer (MODE_STREAMED)
tc_status run_energy(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir, const double* t1,
                     const double* t2, Mode mode, const tc_int_blocks* blocks, const tc_df_factors* df, void* workspace,
                     size_t workspace_bytes, cudaStream_t s, long long first, long long count, double* S_dev,
                     double* E_partial_out) {
    const long long ntrip = tc_triplet_count(o);
    if (first < 0 || count < 0 || first + count > ntrip)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "triplet range [%lld,%lld) outside [0,%lld)", first, first + count, ntrip);
    if (!E_partial_out) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "E_out must not be NULL");
    if (S_dev && !is_device_ptr(S_dev)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "S_dev must be a device pointer");
    Layout L;
    // the caller's workspace_bytes is a hard bound: a layout that does not fit is an error, never an overrun
    if (!is_device_ptr(workspace) || !make_layout(o, v, df ? df->naux : 0, mode, true, workspace_bytes, &L))
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "workspace of %zu bytes is too small or not device memory (see tc_workspace_bytes)",
                workspace_bytes);
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    char* ws = (char*)workspace;
    int4* d_orbits = (int4*)(ws + L.off_orbits);
    tc_trip_rec* d_recs = (tc_trip_rec*)(ws + L.off_recs);
    int* d_dest = (int*)(ws + L.off_dest);
    double* d_w = (double*)(ws + L.off_w);
    double* d_S = (double*)(ws + L.off_S);
    double* d_partial = (double*)(ws + L.off_partial);
    double* d_E = (double*)(ws + L.off_E);
    const int ldv = L.ldv;
    const bool pad = ldv != v;
    const size_t O = o, V = v;

    memset(&ctx->stats, 0, sizeof(ctx->stats));
    ctx->stats.padded = pad ? 1 : 0;
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t0, s));

    // ---- a2: integral staging, and the operand views the W-builder addresses ----
    tc_wbuild_args a;
    memset(&a, 0, sizeof(a));
    a.o = o;
    a.v = v;
    a.eps_occ = eps_occ;
    a.eps_vir = eps_vir;
    a.t1 = t1;
    a.n_orbits = L.n_orbits;
    a.partial = d_partial;
    a.recs = d_recs;
    int n_tslots = o;
    const bool blocked = (mode == MODE_STREAMED) || (mode == MODE_DF && L.n_slots < o);
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_s0, s));
    double* w_ovooT = (double*)(ws + L.off_ovooT);
    double* w_vvvo = (double*)(ws + L.off_vvvo);
    a.ovooT = w_ovooT;
    a.ldo = L.ldo;
    a.slices = w_vvvo;
    a.slice_stride = L.slice_stride;
    a.ldv = ldv;
    if (mode == MODE_BLOCKS) {
        // the caller's blocks, re-laid for the W-builder: slices tiled in fragment order, (ov|oo) with l fastest
        a.ovov = blocks->ovov;
        for (int x = 0; x < o; x++) TC_CUDA(ctx, tc_launch_tile_slice(blocks->vvvo + (size_t)x * V * V * V, v, v, V, w_vvvo + (size_t)x * L.slice_stride, s));
        TC_CUDA(ctx, tc_launch_transpose_ovoo(blocks->ovoo, o, v, L.ldo, w_ovooT, s));
        ctx->stats.n_kernel_launches += o + 1;
    } else {
        double* w_ovov = (double*)(ws + L.off_ovov);
        if (L.ldo != o) TC_CUDA(ctx, cudaMemsetAsync(w_ovooT, 0, sizeof(double) * O * O * V * (size_t)L.ldo, s));   // the pad column
        TC_CUDA(ctx, launch_ovooT(df, o, v, L.ldo, w_ovooT, s));
        TC_CUDA(ctx, launch_ovov(df, o, v, w_ovov, s));
        ctx->stats.n_kernel_launches += 2;
        // the GEMM writes the elements of a slice, not the zero padding of its tiles (ragged tiles, K rounded up to 4):
        // clear the slots once per call
        if (tc_wbuild_slice_doubles(v) != V * V * V)
            TC_CUDA(ctx, cudaMemsetAsync(w_vvvo, 0, sizeof(double) * L.slice_stride * (size_t)L.n_slots, s));
        if (!blocked) {
            // all o slices in one launch
            TC_CUDA(ctx, tc_launch_df_slices_tiled(df->Bvv, df->Bov, o, v, df->naux, 0, o, w_vvvo, L.slice_stride, s));
            ctx->stats.n_kernel_launches++;
            ctx->stats.slices_built += o;
        }
        a.ovov = w_ovov;
    }
    if (mode == MODE_STREAMED) {
        a.t2 = (double*)(ws + L.off_t2);   // amplitude-row slots [slot][y][a][ldv]
        n_tslots = L.n_slots;
    } else if (pad) {
        double* p_t2 = (double*)(ws + L.off_t2);
        for (int x = 0; x < o; x++)
            TC_CUDA(ctx, tc_launch_pad_rows(p_t2 + (size_t)x * L.t2row_stride, ldv, t2 + (size_t)x * O * V * V, V, O * V, v, s));
        ctx->stats.n_kernel_launches += o;
        a.t2 = p_t2;
    } else {
        a.t2 = t2;
    }
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_s1, s));
    // amplitude rows: the caller's array has stride o*v*v, the padded copy / the slots sit at the aligned t2row_stride
    a.t2_row_stride = (a.t2 == t2) ? O * V * V : L.t2row_stride;

    // ---- tables: tile orbits (small host->device copy, stream ordered; the pageable source is staged before return) ----
    {
        std::vector<int4> orb;
        fill_orbits(v, orb);
        if ((int)orb.size() != L.n_orbits) TC_FAIL(ctx, TC_ERR_INTERNAL, "orbit count mismatch");
        TC_CUDA(ctx, cudaMemcpyAsync(d_orbits, orb.data(), sizeof(int4) * orb.size(), cudaMemcpyHostToDevice, s));
    }
    tc_wbuild_maps maps;
    TC_CUDA(ctx, tc_wbuild_make_maps(a, n_tslots, &maps));
    if (!maps.valid) TC_FAIL(ctx, TC_ERR_INTERNAL, "tensor maps of the W-builder could not be encoded");

    TimingRing kring(ctx->ev_k0, ctx->ev_k1), gring(ctx->ev_g0, ctx->ev_g1);
    bool first_kernel = true, first_staging = true;
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c0, s));
    auto launch_block = [&](const tc_trip_rec* recs, int n, const int* dest, double* S_out) -> tc_status {
        const int slot = kring.next();
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_k0[slot], s));
        if (first_kernel) {
            TC_CUDA(ctx, cudaEventRecord(ctx->ev_c0, s));
            first_kernel = false;
        }
        a.recs = recs;
        a.n_trip = n;
        TC_CUDA(ctx, tc_launch_wbuild(a, &maps, d_orbits, s));
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_k1[slot], s));
        TC_CUDA(ctx, tc_launch_reduce_units(d_partial, n, L.n_orbits, dest, S_out, s));
        ctx->stats.n_kernel_launches += 2;
        ctx->stats.n_work_units += (long long)n * L.n_orbits;
        return TC_OK;
    };

    if (!blocked) {
        for (long long done = 0; done < count; done += L.batch) {
            const int nb = (int)((count - done < L.batch) ? (count - done) : L.batch);
            TC_CUDA(ctx, tc_launch_make_triplets(o, first + done, nb, d_recs, d_w + done, s));
            ctx->stats.n_kernel_launches++;
            tc_status st = launch_block(d_recs, nb, nullptr, d_S + done);
            if (st != TC_OK) return st;
        }
    } else {
        // ---- blocked schedule: tables uploaded once, then one W-builder launch per block with the next block's
        //      operands staged on the side stream (a2 overlapped, north_star; PAPER.md:69 for the amplitudes) ----
        tc_plan plan;
        if (!tc_build_plan(o, first, count, L.n_slots, &plan)) TC_FAIL(ctx, TC_ERR_INTERNAL, "blocked schedule: no plan for %d slots", L.n_slots);
        const size_t nrec = plan.recs.size();
        if ((long long)nrec != count) TC_FAIL(ctx, TC_ERR_INTERNAL, "blocked schedule: %zu records for %lld triplets", nrec, count);
        const size_t bytes_tab = nrec * (sizeof(tc_trip_rec) + sizeof(int) + sizeof(double)) + 64;
        if (bytes_tab > ctx->plan_host_bytes) {
            if (ctx->plan_host) cudaFreeHost(ctx->plan_host);
            ctx->plan_host = nullptr;
            ctx->plan_host_bytes = 0;
            TC_CUDA(ctx, cudaMallocHost(&ctx->plan_host, bytes_tab));   // pinned HOST memory (grow-only); no device allocation
            ctx->plan_host_bytes = bytes_tab;
        }
        if (nrec) {
            tc_trip_rec* h_recs = (tc_trip_rec*)ctx->plan_host;
            double* h_w = (double*)(h_recs + nrec);
            int* h_dest = (int*)(h_w + nrec);
            memcpy(h_recs, plan.recs.data(), nrec * sizeof(tc_trip_rec));
            if (mode != MODE_STREAMED)   // t2 is resident as a whole: its rows are addressed by occupied index, not by slot
                for (size_t r = 0; r < nrec; r++)
                    for (int q = 0; q < 3; q++) h_recs[r].t[q] = h_recs[r].occ[q];
            memcpy(h_dest, plan.dest.data(), nrec * sizeof(int));
            for (size_t r = 0; r < nrec; r++) {   // w[dest] = 2 - d_ij - d_jk (eq. (1))
                const tc_trip_rec& rec = plan.recs[r];
                h_w[plan.dest[r]] = 2.0 - (rec.occ[0] == rec.occ[1] ? 1.0 : 0.0) - (rec.occ[1] == rec.occ[2] ? 1.0 : 0.0);
            }
            TC_CUDA(ctx, cudaMemcpyAsync(d_recs, h_recs, nrec * sizeof(tc_trip_rec), cudaMemcpyHostToDevice, s));
            TC_CUDA(ctx, cudaMemcpyAsync(d_w, h_w, nrec * sizeof(double), cudaMemcpyHostToDevice, s));
            TC_CUDA(ctx, cudaMemcpyAsync(d_dest, h_dest, nrec * sizeof(int), cudaMemcpyHostToDevice, s));
        }
        cudaStream_t side = ctx->side_stream;
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));         // the side stream starts after ovoo/ovov and the tables
        TC_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_fork, 0));
        double* w_t2 = (mode == MODE_STREAMED) ? (double*)(ws + L.off_t2) : nullptr;
        const long long nblocks = (long long)plan.blocks.size();
        for (long long n = 0; n < nblocks; n++) {
            const tc_plan_block& b = plan.blocks[n];
            if (b.load_end > b.load_begin) {
                // the slots being overwritten were last read by block wait_block: wait for its W-builder.  The event ring
                // holds the last TC_EV_RING blocks; an older block is covered by waiting for block n-2 (stream order).
                long long wb = b.wait_block;
                if (wb >= 0 && n - wb >= TC_EV_RING) wb = n - 2;
                if (wb >= 0) TC_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_done[wb % TC_EV_RING], 0));
                const int g = gring.next();
                TC_CUDA(ctx, cudaEventRecord(ctx->ev_g0[g], side));
                if (first_staging) {
                    TC_CUDA(ctx, cudaEventRecord(ctx->ev_s0, side));
                    first_staging = false;
                }
                for (int q = b.load_begin; q < b.load_end; q++) {
                    const tc_plan_load& ld = plan.loads[q];
                    TC_CUDA(ctx, tc_launch_df_slices_tiled(df->Bvv, df->Bov, o, v, df->naux, ld.x, 1, w_vvvo + (size_t)ld.slot * L.slice_stride, L.slice_stride, side));
                    ctx->stats.n_kernel_launches++;
                    ctx->stats.slices_built++;
                    if (w_t2) {   // the amplitude row t2[x][:][:][:] from the host, padded on the fly when v is odd
                        TC_CUDA(ctx, cudaMemcpy2DAsync(w_t2 + (size_t)ld.slot * L.t2row_stride, sizeof(double) * ldv,
                                                       t2 + (size_t)ld.x * O * V * V, sizeof(double) * V, sizeof(double) * V, O * V,
                                                       cudaMemcpyHostToDevice, side));
                        ctx->stats.t2_rows_copied++;
                        ctx->stats.bytes_h2d += (double)(sizeof(double) * O * V * V);
                    }
                }
                TC_CUDA(ctx, cudaEventRecord(ctx->ev_g1[g], side));
                TC_CUDA(ctx, cudaEventRecord(ctx->ev_s1, side));
                TC_CUDA(ctx, cudaEventRecord(ctx->ev_staged[n % TC_EV_RING], side));
                TC_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_staged[n % TC_EV_RING], 0));
            }
            tc_status st = launch_block(d_recs + b.rec_begin, b.n, d_dest + b.rec_begin, d_S);
            if (st != TC_OK) return st;
            TC_CUDA(ctx, cudaEventRecord(ctx->ev_done[n % TC_EV_RING], s));
        }
        ctx->stats.n_blocks = nblocks;
        // every ev_staged has been waited for on the caller's stream: the side stream is joined
    }
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c1, s));
    TC_CUDA(ctx, tc_launch_reduce_energy(d_S, d_w, count, d_E, s));
    ctx->stats.n_kernel_launches++;
    if (S_dev && count > 0) TC_CUDA(ctx, cudaMemcpyAsync(S_dev, d_S, sizeof(double) * (size_t)count, cudaMemcpyDeviceToDevice, s));
    TC_CUDA(ctx, cudaMemcpyAsync(ctx->pinned, d_E, sizeof(double), cudaMemcpyDeviceToHost, s));
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t1, s));
    TC_CUDA(ctx, cudaStreamSynchronize(s));
    TC_CUDA(ctx, cudaStreamSynchronize(ctx->side_stream));

    float ms = 0;
    cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1);
    ctx->stats.ms_total = ms;
    if (count > 0) {
        cudaEventElapsedTime(&ms, ctx->ev_c0, ctx->ev_c1);
        ctx->stats.ms_contraction = ms;
        cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_c0);
        ctx->stats.contraction_first_ms = ms;
        cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_c1);
        ctx->stats.contraction_last_ms = ms;
    }
    kring.finish();
    ctx->stats.ms_kernels = kring.total_ms;
    if (!blocked) {
        if (df) {
            cudaEventElapsedTime(&ms, ctx->ev_s0, ctx->ev_s1);
            ctx->stats.ms_staging = ms;
        }
    } else {
        gring.finish();
        ctx->stats.ms_staging_side = gring.total_ms;
        ctx->stats.ms_staging = gring.total_ms;
        if (!first_staging) {
            cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_s0);
            ctx->stats.staging_first_ms = ms;
            cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_s1);
            ctx->stats.staging_last_ms = ms;
        }
    }
    ctx->stats.kernel = (count > 0) ? TC_KERNEL_TMA : 0;
    const long long nz = count - count_diagonal(o, first, count);
    ctx->stats.n_triplets = nz;
    ctx->stats.flop_contraction = (double)nz * 12.0 * (double)v * v * v * ((double)v + o);
    *E_partial_out = (count > 0) ? ctx->pinned[0] : 0.0;
    return TC_OK;
}

}  // namespace

extern "C" tc_status tc_workspace_bytes(tc_ctx* ctx, int o, int v, int naux_or_0, size_t hbm_budget, size_t* bytes) {
    if (!ctx || !bytes) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || naux_or_0 < 0) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes o=%d v=%d naux=%d", o, v, naux_or_0);
    Layout L;
    if (!make_layout(o, v, naux_or_0, naux_or_0 ? MODE_DF : MODE_BLOCKS, hbm_budget != 0, hbm_budget, &L))
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "problem does not fit the HBM budget of %zu bytes", hbm_budget);
    *bytes = L.total;
    return TC_OK;
}

extern "C" tc_status tc_workspace_bytes_streamed(tc_ctx* ctx, int o, int v, int naux, size_t hbm_budget, size_t* bytes) {
    if (!ctx || !bytes) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || naux < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes o=%d v=%d naux=%d", o, v, naux);
    Layout L;
    if (!make_layout(o, v, naux, MODE_STREAMED, hbm_budget != 0, hbm_budget, &L))
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "problem does not fit the HBM budget of %zu bytes", hbm_budget);
    *bytes = L.total;
    return TC_OK;
}

extern "C" tc_status tc_workspace_bytes_abcijk(tc_ctx* ctx, int o, int v, int naux, size_t* bytes) {
    if (!ctx || !bytes) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || naux < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes o=%d v=%d naux=%d", o, v, naux);
    Layout L;
    make_layout(o, v, naux, MODE_ABCIJK, false, 0, &L);
    *bytes = L.total;
    return TC_OK;
}

extern "C" long long tc_tile_orbit_count(int v) { return v < 1 ? -1 : (long long)tc_wbuild_num_orbits(v); }

// The paper's own loop order (abcijk; Fig. 1; Fig. 2): virtual tile orbits outer, all
// i >= j >= k inner; per orbit the integrals are rebuilt from the factors restricted to its tiles (Fig. 2 l.7, 10), so the
// footprint beside t2 is O(o v T^2) instead of o v^3.  The next orbit's integrals are assembled on the side stream while the
// current orbit's W-builder launch (all triplets x this orbit) runs.
extern "C" tc_status tc_triples_energy_abcijk(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                              const double* t1, const double* t2, const tc_df_factors* df, void* workspace,
                                              size_t workspace_bytes, void* stream, long long orbit_first, long long orbit_count,
                                              double* E_orbit_dev, double* E_out) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (!df) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "the abcijk call takes DF factors");
    tc_status st = check_common(ctx, o, v, eps_occ, eps_vir, t1, t2, false, nullptr, df);
    if (st != TC_OK) return st;
    if (!E_out) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "E_out must not be NULL");
    if (E_orbit_dev && !is_device_ptr(E_orbit_dev)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "E_orbit_dev must be a device pointer");
    Layout L;
    make_layout(o, v, df->naux, MODE_ABCIJK, false, 0, &L);
    if (!is_device_ptr(workspace) || L.total > workspace_bytes)
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "workspace of %zu bytes is too small or not device memory (see tc_workspace_bytes_abcijk)",
                workspace_bytes);
    if (orbit_first < 0 || orbit_count < 0 || orbit_first + orbit_count > L.n_orbits)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "orbit range [%lld,%lld) outside [0,%d)", orbit_first, orbit_first + orbit_count, L.n_orbits);
    const long long ntrip = tc_triplet_count(o);
    const int group = std::min(kOrbitGroup, L.n_orbits);
    if ((long long)L.batch * L.n_orbits < ntrip * group || ntrip * group > 0x7fffffffLL)
        TC_FAIL(ctx, TC_ERR_INTERNAL, "partial buffer too small for %lld triplets x %d orbits", ntrip, group);
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t s = (cudaStream_t)stream, side = ctx->side_stream;
    char* ws = (char*)workspace;
    int4* d_orbits = (int4*)(ws + L.off_orbits);
    tc_trip_rec* d_recs = (tc_trip_rec*)(ws + L.off_recs);
    double* d_w = (double*)(ws + L.off_w);
    double* d_S = (double*)(ws + L.off_S);
    double* d_partial = (double*)(ws + L.off_partial);
    double* d_E = (double*)(ws + L.off_E);
    double* d_Eorb = (double*)(ws + L.off_Eorb);
    double* w_ovooT = (double*)(ws + L.off_ovooT);
    double* w_ovov = (double*)(ws + L.off_ovov);
    double* w_buf = (double*)(ws + L.off_vvvo);
    const size_t O = o, V = v;
    const bool pad = L.ldv != v;

    memset(&ctx->stats, 0, sizeof(ctx->stats));
    ctx->stats.padded = pad ? 1 : 0;
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t0, s));
    std::vector<int4> orb;
    fill_orbits(v, orb);
    TC_CUDA(ctx, cudaMemcpyAsync(d_orbits, orb.data(), sizeof(int4) * orb.size(), cudaMemcpyHostToDevice, s));
    if (L.ldo != o) TC_CUDA(ctx, cudaMemsetAsync(w_ovooT, 0, sizeof(double) * O * O * V * (size_t)L.ldo, s));
    TC_CUDA(ctx, launch_ovooT(df, o, v, L.ldo, w_ovooT, s));
    TC_CUDA(ctx, launch_ovov(df, o, v, w_ovov, s));
    TC_CUDA(ctx, cudaMemsetAsync(w_buf, 0, sizeof(double) * 2 * kOrbitGroup * L.orbit_buf_stride, s));   // K padding of the chunk layout stays zero
    TC_CUDA(ctx, tc_launch_make_triplets(o, 0, (int)ntrip, d_recs, d_w, s));
    ctx->stats.n_kernel_launches += 3;
    tc_wbuild_args a;
    memset(&a, 0, sizeof(a));
    a.o = o;
    a.v = v;
    a.ldv = L.ldv;
    a.ldo = L.ldo;
    a.eps_occ = eps_occ;
    a.eps_vir = eps_vir;
    a.t1 = t1;
    a.ovooT = w_ovooT;
    a.ovov = w_ovov;
    a.slice_stride = L.slice_stride;
    a.orbit_local = 1;
    a.orbit_stride = L.orbit_buf_stride;
    a.recs = d_recs;
    a.n_trip = (int)ntrip;
    a.partial = d_partial;
    a.n_orbits = 1;
    if (pad) {
        double* p_t2 = (double*)(ws + L.off_t2);
        for (int x = 0; x < o; x++)
            TC_CUDA(ctx, tc_launch_pad_rows(p_t2 + (size_t)x * L.t2row_stride, L.ldv, t2 + (size_t)x * O * V * V, V, O * V, v, s));
        ctx->stats.n_kernel_launches += o;
        a.t2 = p_t2;
        a.t2_row_stride = L.t2row_stride;
    } else {
        a.t2 = t2;
        a.t2_row_stride = O * V * V;
    }
    tc_wbuild_maps maps;
    TC_CUDA(ctx, tc_wbuild_make_maps(a, o, &maps));
    if (!maps.valid) TC_FAIL(ctx, TC_ERR_INTERNAL, "tensor maps of the W-builder could not be encoded");
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_fork, s));
    TC_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_fork, 0));
    TimingRing kring(ctx->ev_k0, ctx->ev_k1), gring(ctx->ev_g0, ctx->ev_g1);
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c0, s));
    long long ngroups = 0;
    for (long long n = 0; n < orbit_count; n += group, ngroups++) {
        const long long q = ngroups;                      // launch number
        const int g_n = (int)std::min<long long>(group, orbit_count - n);
        double* buf = w_buf + (size_t)(q & 1) * kOrbitGroup * L.orbit_buf_stride;
        // staging buffer set q & 1 was last read by launch q - 2
        if (q >= 2) TC_CUDA(ctx, cudaStreamWaitEvent(side, ctx->ev_done[(q - 2) % TC_EV_RING], 0));
        const int g = gring.next();
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_g0[g], side));
        for (int m = 0; m < g_n; m++) {
            const int4 ob = orb[(size_t)(orbit_first + n + m)];
            TC_CUDA(ctx, tc_launch_df_slices_orbit(df->Bvv, df->Bov, o, v, df->naux, ob.x, ob.y, ob.z, buf + (size_t)m * L.orbit_buf_stride,
                                                   L.slice_stride, side));
        }
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_g1[g], side));
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_staged[q % TC_EV_RING], side));
        TC_CUDA(ctx, cudaStreamWaitEvent(s, ctx->ev_staged[q % TC_EV_RING], 0));
        const int kslot = kring.next();
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_k0[kslot], s));
        a.slices = buf;
        a.n_orbits = g_n;                                 // partial sums of the launch: [triplet][g_n]
        TC_CUDA(ctx, tc_launch_wbuild(a, &maps, d_orbits + (orbit_first + n), s));
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_k1[kslot], s));
        for (int m = 0; m < g_n; m++)                     // orbit by orbit, in order: S and the per-orbit energies do not depend on the grouping
            TC_CUDA(ctx, tc_launch_accumulate_orbit(d_partial + m, g_n, d_w, ntrip, (n + m) == 0 ? 1 : 0, d_S, d_Eorb + n + m, s));
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_done[q % TC_EV_RING], s));
        ctx->stats.n_kernel_launches += 1 + 2 * g_n;
        ctx->stats.n_work_units += ntrip * g_n;
        ctx->stats.slices_built += (long long)o * g_n;
    }
    ctx->stats.n_blocks = orbit_count;
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c1, s));
    if (orbit_count == 0) TC_CUDA(ctx, cudaMemsetAsync(d_S, 0, sizeof(double) * (size_t)ntrip, s));
    TC_CUDA(ctx, tc_launch_reduce_energy(d_S, d_w, ntrip, d_E, s));
    ctx->stats.n_kernel_launches++;
    if (E_orbit_dev && orbit_count > 0)
        TC_CUDA(ctx, cudaMemcpyAsync(E_orbit_dev, d_Eorb, sizeof(double) * (size_t)orbit_count, cudaMemcpyDeviceToDevice, s));
    TC_CUDA(ctx, cudaMemcpyAsync(ctx->pinned, d_E, sizeof(double), cudaMemcpyDeviceToHost, s));
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t1, s));
    TC_CUDA(ctx, cudaStreamSynchronize(s));
    TC_CUDA(ctx, cudaStreamSynchronize(side));
    float ms = 0;
    cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1);
    ctx->stats.ms_total = ms;
    cudaEventElapsedTime(&ms, ctx->ev_c0, ctx->ev_c1);
    ctx->stats.ms_contraction = ms;
    kring.finish();
    gring.finish();
    ctx->stats.ms_kernels = kring.total_ms;
    ctx->stats.ms_staging = ctx->stats.ms_staging_side = gring.total_ms;
    ctx->stats.kernel = orbit_count > 0 ? TC_KERNEL_TMA : 0;
    const long long nz = ntrip - o;   // all but the o triplets i = j = k
    ctx->stats.n_triplets = nz;
    // executed contraction flop of the orbits in the range: 294 912 (v + o) per (triplet, generic orbit) when no tile is ragged;
    // the full range sums to exactly 12 v^3 (v + o) per non-zero triplet
    ctx->stats.flop_contraction = (orbit_count == L.n_orbits) ? (double)nz * 12.0 * (double)v * v * v * ((double)v + o) : 0.0;
    *E_out = ctx->pinned[0];
    return TC_OK;
}

extern "C" tc_status tc_build_blocks(tc_ctx* ctx, int o, int v, const tc_df_factors* df, int x0, int nx,
                                     double* vvvo_out, double* ovoo_out, double* ovov_out, void* stream) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || !df || df->naux < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes or df == NULL");
    if (!is_device_ptr(df->Boo) || !is_device_ptr(df->Bov) || !is_device_ptr(df->Bvv))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "df factors must be device pointers");
    if (vvvo_out && (x0 < 0 || nx < 0 || x0 + nx > o)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "slice range [%d,%d) outside [0,%d)", x0, x0 + nx, o);
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (vvvo_out && nx > 0) {
        TC_CUDA(ctx, launch_slices_natural(df, o, v, x0, nx, vvvo_out, st));
        ctx->stats.n_kernel_launches++;
        ctx->stats.slices_built += nx;
    }
    if (ovoo_out) {
        TC_CUDA(ctx, launch_ovoo_natural(df, o, v, ovoo_out, st));
        ctx->stats.n_kernel_launches++;
    }
    if (ovov_out) {
        TC_CUDA(ctx, launch_ovov(df, o, v, ovov_out, st));
        ctx->stats.n_kernel_launches++;
    }
    return TC_OK;
}

extern "C" tc_status tc_triples_energy_slice(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                             const double* t1, const double* t2, const tc_int_blocks* blocks,
                                             const tc_df_factors* df, void* workspace, size_t workspace_bytes, void* stream,
                                             long long first, long long count, double* S_dev, double* E_partial_out) {
    tc_status st = check_common(ctx, o, v, eps_occ, eps_vir, t1, t2, false, blocks, df);
    if (st != TC_OK) return st;
    return run_energy(ctx, o, v, eps_occ, eps_vir, t1, t2, df ? MODE_DF : MODE_BLOCKS, blocks, df, workspace, workspace_bytes,
                      (cudaStream_t)stream, first, count, S_dev, E_partial_out);
}

extern "C" tc_status tc_triples_energy_streamed(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                                const double* t1, const double* t2_host, const tc_df_factors* df,
                                                void* workspace, size_t workspace_bytes, void* stream, long long first,
                                                long long count, double* S_dev, double* E_partial_out) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (!df) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "the streamed call takes DF factors");
    tc_status st = check_common(ctx, o, v, eps_occ, eps_vir, t1, t2_host, true, nullptr, df);
    if (st != TC_OK) return st;
    return run_energy(ctx, o, v, eps_occ, eps_vir, t1, t2_host, MODE_STREAMED, nullptr, df, workspace, workspace_bytes,
                      (cudaStream_t)stream, first, count, S_dev, E_partial_out);
}

extern "C" tc_status tc_triples_energy(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                       const double* t1, const double* t2, const tc_int_blocks* blocks,
                                       const tc_df_factors* df, void* workspace, size_t workspace_bytes, void* stream,
                                       double* E_out) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "o must be >= 1");
    return tc_triples_energy_slice(ctx, o, v, eps_occ, eps_vir, t1, t2, blocks, df, workspace, workspace_bytes, stream, 0,
                                   tc_triplet_count(o), nullptr, E_out);
}

extern "C" tc_status tc_triples_energy_host(tc_ctx* ctx, int o, int v, int naux, const double* eps_occ, const double* eps_vir,
                                            const double* t1, const double* t2, const double* Boo, const double* Bov,
                                            const double* Bvv, long long first, long long count, double* E_out,
                                            size_t* bytes_h2d) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || naux < 1 || !eps_occ || !eps_vir || !t1 || !t2 || !Boo || !Bov || !Bvv || !E_out)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes or NULL host pointer");
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    size_t wsb = 0;
    tc_status st = tc_workspace_bytes(ctx, o, v, naux, 0, &wsb);
    if (st != TC_OK) return st;
    const size_t O = o, V = v, X = naux;
    const size_t n[7] = {O, V, O * V, O * O * V * V, X * O * O, X * O * V, X * V * V};
    const double* h[7] = {eps_occ, eps_vir, t1, t2, Boo, Bov, Bvv};
    double* d[7] = {0, 0, 0, 0, 0, 0, 0};
    // one device slab for the inputs and the workspace, kept in the context between calls (grow-only):
    // repeated calls pay for the copies, not for cudaMalloc/cudaFree
    size_t need = align_up(wsb);
    for (int q = 0; q < 7; q++) need += align_up(n[q] * sizeof(double));
    if (need > ctx->host_slab_bytes) {
        if (ctx->host_slab) cudaFree(ctx->host_slab);
        ctx->host_slab = nullptr;
        ctx->host_slab_bytes = 0;
        cudaError_t ea = cudaMalloc(&ctx->host_slab, need);
        if (ea != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "device allocation of %zu bytes failed: %s", need, cudaGetErrorString(ea));
        ctx->host_slab_bytes = need;
    }
    char* slab = (char*)ctx->host_slab;
    void* ws = slab;
    size_t off = align_up(wsb), copied = 0;
    cudaError_t e = cudaSuccess;
    for (int q = 0; q < 7 && e == cudaSuccess; q++) {
        d[q] = (double*)(slab + off);
        off += align_up(n[q] * sizeof(double));
        e = cudaMemcpyAsync(d[q], h[q], n[q] * sizeof(double), cudaMemcpyHostToDevice, 0);
        copied += n[q] * sizeof(double);
    }
    if (e == cudaSuccess) {
        tc_df_factors df = {naux, d[4], d[5], d[6]};
        double E = 0;
        st = tc_triples_energy_slice(ctx, o, v, d[0], d[1], d[2], d[3], nullptr, &df, ws, wsb, 0, first, count, nullptr, &E);
        if (st == TC_OK) *E_out = E;
    }
    if (e != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "host->device copy failed: %s", cudaGetErrorString(e));
    if (st == TC_OK && bytes_h2d) *bytes_h2d = copied;
    return st;
}

extern "C" tc_status tc_debug_W_triplet(tc_ctx* ctx, int o, int v, int i, int j, int k, const double* t2,
                                        const tc_int_blocks* blocks, double* W_dev, void* stream) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || i < 0 || j < 0 || k < 0 || i >= o || j >= o || k >= o)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes or occupied indices");
    if (!blocks || !is_device_ptr(t2) || !is_device_ptr(blocks->vvvo) || !is_device_ptr(blocks->ovoo) ||
        !is_device_ptr(blocks->ovov) || !is_device_ptr(W_dev))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "t2, blocks and W_dev must be device pointers");
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t s = (cudaStream_t)stream;
    if ((uintptr_t)t2 % 16 != 0) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "t2 must be 16-byte aligned");
    Layout L;
    make_layout(o, v, 0, MODE_BLOCKS, false, 0, &L);
    // debug path: scratch allocated here (not a compute call of the hot path); zeros stand in for eps and t1
    const size_t b_zero = align_up(sizeof(double) * (size_t)(o > v ? o : v) * v);
    char* tmp = nullptr;
    TC_CUDA(ctx, cudaMalloc(&tmp, L.total + b_zero));
    const int ldv = L.ldv;
    const size_t O = o, V = v;
    std::vector<int4> orb;
    fill_orbits(v, orb);
    tc_trip_rec rec;
    memset(&rec, 0, sizeof(rec));
    rec.occ[0] = i; rec.occ[1] = j; rec.occ[2] = k;
    for (int p = 0; p < 3; p++) rec.s[p] = rec.t[p] = rec.occ[p];
    cudaError_t e = cudaMemcpyAsync(tmp + L.off_orbits, orb.data(), sizeof(int4) * orb.size(), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tmp + L.off_recs, &rec, sizeof(rec), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(tmp + L.total, 0, b_zero, s);
    tc_wbuild_args a;
    memset(&a, 0, sizeof(a));
    a.o = o;
    a.v = v;
    const double* zeros = (const double*)(tmp + L.total);
    a.eps_occ = zeros;  // the epilogue result is discarded; only W is wanted
    a.eps_vir = zeros;
    a.t1 = zeros;
    a.ovov = blocks->ovov;
    a.recs = (const tc_trip_rec*)(tmp + L.off_recs);
    a.n_trip = 1;
    a.partial = (double*)(tmp + L.off_partial);
    a.n_orbits = L.n_orbits;
    a.W_debug = W_dev;
    double* w_vvvo = (double*)(tmp + L.off_vvvo);
    double* w_ovooT = (double*)(tmp + L.off_ovooT);
    a.slices = w_vvvo;
    a.slice_stride = L.slice_stride;
    a.ovooT = w_ovooT;
    a.ldo = L.ldo;
    a.ldv = ldv;
    for (int x = 0; x < o && e == cudaSuccess; x++)
        if (x == i || x == j || x == k) e = tc_launch_tile_slice(blocks->vvvo + (size_t)x * V * V * V, v, v, V, w_vvvo + (size_t)x * L.slice_stride, s);
    if (e == cudaSuccess) e = tc_launch_transpose_ovoo(blocks->ovoo, o, v, L.ldo, w_ovooT, s);
    if (ldv != v) {
        double* p_t2 = (double*)(tmp + L.off_t2);
        for (int x = 0; x < o && e == cudaSuccess; x++)
            e = tc_launch_pad_rows(p_t2 + (size_t)x * L.t2row_stride, ldv, t2 + (size_t)x * O * V * V, V, O * V, v, s);
        a.t2 = p_t2;
        a.t2_row_stride = L.t2row_stride;
    } else {
        a.t2 = t2;
        a.t2_row_stride = O * V * V;
    }
    if (e == cudaSuccess) {
        tc_wbuild_maps maps;
        e = tc_wbuild_make_maps(a, o, &maps);
        if (e == cudaSuccess && !maps.valid) e = cudaErrorInvalidValue;
        if (e == cudaSuccess) e = tc_launch_wbuild(a, &maps, (const int4*)(tmp + L.off_orbits), s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        ctx->stats.kernel = TC_KERNEL_TMA;
    }
    cudaFree(tmp);
    if (e != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "debug W kernel failed: %s", cudaGetErrorString(e));
    return TC_OK;
}
