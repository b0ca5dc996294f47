// tc_energy.cu -- the C-ABI compute calls: argument checks, workspace carving, and the
// launch sequence  scheduler (a1) -> stager (a2) -> fused W-builder/epilogue (a3-a6) -> reductions (a7).
#include <stdlib.h>

#include <algorithm>
#include <vector>

#include "tc_common.cuh"

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// How the caller's workspace is carved.  Everything the compute calls need lives here
// (pre-allocate and reuse; no device allocation inside the call).
struct Layout {
    size_t off_orbits, off_sliceptr, off_sliceslot, off_trip, off_dest, off_w, off_S, off_partial, off_E, off_ovoo, off_ovov, off_vvvo;
    size_t total;
    int n_orbits;
    int batch;      // triplets per W-builder launch
    int n_slots;    // resident (vv|v.) slices (DF input): o = all materialised
};

constexpr size_t kPartialBudget = (size_t)256 << 20;

bool make_layout(int o, int v, int naux, size_t budget, Layout* L) {
    const long long ntrip = (long long)o * (o + 1) * (o + 2) / 6;
    L->n_orbits = tc_wbuild_num_orbits(v);
    long long batch = (long long)(kPartialBudget / ((size_t)L->n_orbits * sizeof(double)));
    if (batch < 1) batch = 1;
    if (batch > ntrip) batch = ntrip;
    if (batch * L->n_orbits > 0x7fffffffLL) batch = 0x7fffffffLL / L->n_orbits;
    L->batch = (int)batch;
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t at = off;
        off += align_up(bytes);
        return at;
    };
    L->off_orbits = take(sizeof(int4) * (size_t)L->n_orbits);
    L->off_sliceptr = take(sizeof(double*) * (size_t)o);
    L->off_sliceslot = take(sizeof(int) * (size_t)o);
    L->off_trip = take(sizeof(int4) * (size_t)L->batch);
    L->off_dest = take(sizeof(int) * (size_t)L->batch);
    L->off_w = take(sizeof(double) * (size_t)ntrip);
    L->off_S = take(sizeof(double) * (size_t)ntrip);
    L->off_partial = take(sizeof(double) * (size_t)L->batch * L->n_orbits);
    L->off_E = take(sizeof(double) * 8);
    L->off_ovoo = L->off_ovov = L->off_vvvo = 0;
    L->n_slots = 0;
    if (naux > 0) {
        const size_t v3 = (size_t)v * v * v;
        L->off_ovoo = take(sizeof(double) * (size_t)o * o * o * v);
        L->off_ovov = take(sizeof(double) * (size_t)o * o * v * v);
        const size_t slice_bytes = align_up(sizeof(double) * v3);
        long long slots = o;
        if (budget) {
            if (off >= budget) return false;
            const long long fit = (long long)((budget - off) / slice_bytes);
            if (fit < slots) slots = fit;
        }
        // fewer slots than slices: the slice cache of the blocked schedule (needs i + one j + one k slice)
        if (slots < 3 && slots < o) return false;
        L->n_slots = (int)slots;
        L->off_vvvo = take(slice_bytes * (size_t)slots);
    }
    L->total = off;
    return budget == 0 || off <= budget;
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
                       const double* t2, const tc_int_blocks* blocks, const tc_df_factors* df) {
    if (!ctx) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "o and v must be >= 1 (got o=%d v=%d)", o, v);
    if ((blocks != nullptr) == (df != nullptr)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "exactly one of blocks / df must be given");
    if (!is_device_ptr(eps_occ) || !is_device_ptr(eps_vir) || !is_device_ptr(t1) || !is_device_ptr(t2))
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "eps_occ, eps_vir, t1, t2 must be device pointers");
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

}  // namespace

extern "C" tc_status tc_workspace_bytes(tc_ctx* ctx, int o, int v, int naux_or_0, size_t hbm_budget, size_t* bytes) {
    if (!ctx || !bytes) return TC_ERR_INVALID_ARG;
    if (o < 1 || v < 1 || naux_or_0 < 0) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "bad sizes o=%d v=%d naux=%d", o, v, naux_or_0);
    Layout L;
    if (!make_layout(o, v, naux_or_0, hbm_budget, &L))
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "problem does not fit the HBM budget of %zu bytes", hbm_budget);
    *bytes = L.total;
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
    const int naux = df->naux;
    const long long V = v, O = o;
    if (vvvo_out && nx > 0) {
        // rows (d,b) -> d*v + b (row*v), cols (x,c) -> x*v^3 + c
        TC_CUDA(ctx, tc_launch_df_gemm(df->Bvv, (size_t)(V * V), df->Bov + (size_t)x0 * v, (size_t)(O * V), v * v, nx * v, naux,
                                       /*R2*/ 1, /*sr1*/ V, /*sr2*/ 0, /*C2*/ v, /*sc1*/ V * V * V, /*sc2*/ 1, vvvo_out, st));
        ctx->stats.n_kernel_launches++;
        ctx->stats.slices_built += nx;
    }
    if (ovoo_out) {
        // rows (l,j): l*v + j*o^2*v; cols (k,c): k*o*v + c
        TC_CUDA(ctx, tc_launch_df_gemm(df->Boo, (size_t)(O * O), df->Bov, (size_t)(O * V), o * o, o * v, naux,
                                       /*R2*/ o, /*sr1*/ V, /*sr2*/ O * O * V, /*C2*/ v, /*sc1*/ O * V, /*sc2*/ 1, ovoo_out, st));
        ctx->stats.n_kernel_launches++;
    }
    if (ovov_out) {
        // rows (j,b): j*o*v^2 + b*v; cols (k,c): k*v^2 + c
        TC_CUDA(ctx, tc_launch_df_gemm(df->Bov, (size_t)(O * V), df->Bov, (size_t)(O * V), o * v, o * v, naux,
                                       /*R2*/ v, /*sr1*/ O * V * V, /*sr2*/ V, /*C2*/ v, /*sc1*/ V * V, /*sc2*/ 1, ovov_out, st));
        ctx->stats.n_kernel_launches++;
    }
    return TC_OK;
}

extern "C" tc_status tc_triples_energy_slice(tc_ctx* ctx, int o, int v, const double* eps_occ, const double* eps_vir,
                                             const double* t1, const double* t2, const tc_int_blocks* blocks,
                                             const tc_df_factors* df, void* workspace, size_t workspace_bytes, void* stream,
                                             long long first, long long count, double* S_dev, double* E_partial_out) {
    tc_status st = check_common(ctx, o, v, eps_occ, eps_vir, t1, t2, blocks, df);
    if (st != TC_OK) return st;
    const long long ntrip = tc_triplet_count(o);
    if (first < 0 || count < 0 || first + count > ntrip)
        TC_FAIL(ctx, TC_ERR_INVALID_ARG, "triplet range [%lld,%lld) outside [0,%lld)", first, first + count, ntrip);
    if (!E_partial_out) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "E_out must not be NULL");
    if (S_dev && !is_device_ptr(S_dev)) TC_FAIL(ctx, TC_ERR_INVALID_ARG, "S_dev must be a device pointer");
    Layout L;
    if (!make_layout(o, v, df ? df->naux : 0, workspace_bytes, &L) || !is_device_ptr(workspace))
        TC_FAIL(ctx, TC_ERR_WORKSPACE_TOO_SMALL, "workspace of %zu bytes is too small or not device memory (see tc_workspace_bytes)",
                workspace_bytes);
    TC_CUDA(ctx, cudaSetDevice(ctx->device));
    cudaStream_t s = (cudaStream_t)stream;
    char* ws = (char*)workspace;
    int4* d_orbits = (int4*)(ws + L.off_orbits);
    const double** d_sliceptr = (const double**)(ws + L.off_sliceptr);
    int* d_sliceslot = (int*)(ws + L.off_sliceslot);
    int4* d_trip = (int4*)(ws + L.off_trip);
    int* d_dest = (int*)(ws + L.off_dest);
    double* d_w = (double*)(ws + L.off_w);
    double* d_S = (double*)(ws + L.off_S);
    double* d_partial = (double*)(ws + L.off_partial);
    double* d_E = (double*)(ws + L.off_E);

    memset(&ctx->stats, 0, sizeof(ctx->stats));
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t0, s));

    // ---- a2: integral staging ----
    const double *ovoo, *ovov, *vvvo;
    size_t slice_stride;
    if (df) {
        double* w_ovoo = (double*)(ws + L.off_ovoo);
        double* w_ovov = (double*)(ws + L.off_ovov);
        double* w_vvvo = (double*)(ws + L.off_vvvo);
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_s0, s));
        st = tc_build_blocks(ctx, o, v, df, 0, o, nullptr, w_ovoo, w_ovov, s);
        if (st != TC_OK) return st;
        // slices land at an aligned stride so each starts on a 256-byte boundary
        slice_stride = align_up(sizeof(double) * (size_t)v * v * v) / sizeof(double);
        if (L.n_slots >= o) {
            // all o slices in one launch: column (x, c) of the v^2 x (o v) product lands at x * slice_stride + c
            TC_CUDA(ctx, tc_launch_df_gemm(df->Bvv, (size_t)v * v, df->Bov, (size_t)o * v, v * v, o * v, df->naux, 1, (long long)v, 0,
                                           v, (long long)slice_stride, 1, w_vvvo, s));
            ctx->stats.n_kernel_launches++;
            ctx->stats.slices_built += o;
        }
        TC_CUDA(ctx, cudaEventRecord(ctx->ev_s1, s));
        ovoo = w_ovoo;
        ovov = w_ovov;
        vvvo = w_vvvo;
    } else {
        ovoo = blocks->ovoo;
        ovov = blocks->ovov;
        vvvo = blocks->vvvo;
        slice_stride = (size_t)v * v * v;
    }

    // ---- tables: tile orbits and slice pointers (small host->device copies, stream ordered) ----
    {
        std::vector<int4> orb;
        fill_orbits(v, orb);
        if ((int)orb.size() != L.n_orbits) TC_FAIL(ctx, TC_ERR_INTERNAL, "orbit count mismatch");
        std::vector<const double*> sp(o);
        std::vector<int> slot(o);
        for (int x = 0; x < o; x++) {
            sp[x] = vvvo + (size_t)x * slice_stride;
            slot[x] = x;  // all slices resident, slice x in slot x
        }
        TC_CUDA(ctx, cudaMemcpyAsync(d_sliceslot, slot.data(), sizeof(int) * slot.size(), cudaMemcpyHostToDevice, s));
        // pageable sources: cudaMemcpyAsync stages them before returning, so the vectors may die here
        TC_CUDA(ctx, cudaMemcpyAsync(d_orbits, orb.data(), sizeof(int4) * orb.size(), cudaMemcpyHostToDevice, s));
        TC_CUDA(ctx, cudaMemcpyAsync(d_sliceptr, sp.data(), sizeof(double*) * sp.size(), cudaMemcpyHostToDevice, s));
        TC_CUDA(ctx, cudaStreamSynchronize(s));
    }

    // ---- a1 + a3..a7 over batches of triplets ----
    tc_wbuild_args a;
    a.o = o;
    a.v = v;
    a.eps_occ = eps_occ;
    a.eps_vir = eps_vir;
    a.t1 = t1;
    a.t2 = t2;
    a.slice_ptr = d_sliceptr;
    a.slices_aligned16 = ((uintptr_t)vvvo % 16 == 0) && ((slice_stride * sizeof(double)) % 16 == 0);
    a.ovoo = ovoo;
    a.ovov = ovov;
    a.triplets = d_trip;
    a.partial = d_partial;
    a.n_orbits = L.n_orbits;
    a.slice_slot = d_sliceslot;
    a.W_debug = nullptr;
    const bool blocked = df && L.n_slots < o;
    const int nslots = blocked ? L.n_slots : o;
    tc_wbuild_maps maps;
    TC_CUDA(ctx, tc_wbuild_make_maps(a, vvvo, slice_stride, nslots, &maps));
    if (getenv("TC_FORCE_CPASYNC")) maps.valid = false;  // testing aid: exercise the fallback kernel on even v
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c0, s));
    if (!blocked) {
        for (long long done = 0; done < count; done += L.batch) {
            const int nb = (int)((count - done < L.batch) ? (count - done) : L.batch);
            TC_CUDA(ctx, tc_launch_make_triplets(o, first + done, nb, d_trip, d_w + done, s));
            a.n_trip = nb;
            TC_CUDA(ctx, tc_launch_wbuild(a, &maps, d_orbits, s));
            TC_CUDA(ctx, tc_launch_reduce_units(d_partial, nb, L.n_orbits, nullptr, d_S + done, s));
            ctx->stats.n_kernel_launches += 3;
            ctx->stats.n_work_units += (long long)nb * L.n_orbits;
        }
    } else {
        // ---- blocked schedule with a slice cache ("LRU of slots" for cfg4-size problems) ----
        // The (vv|v.) slices do not all fit: nslots slots hold the slices a block of triplets needs.  For each
        // i the (j,k) plane is cut into b x b blocks, b = (nslots-1)/2: slice i stays pinned, a block of j slices
        // stays while the k blocks stream through, so a block of up to b^2 triplets costs at most b new slices.
        // Missing slices are assembled from the DF factors (eq. (6)) right before the launch that needs them.
        for (long long done = 0; done < count; done += L.batch) {  // weights of the whole range
            const int nb = (int)((count - done < L.batch) ? (count - done) : L.batch);
            TC_CUDA(ctx, tc_launch_make_triplets(o, first + done, nb, d_trip, d_w + done, s));
            ctx->stats.n_kernel_launches++;
        }
        double* w_vvvo = (double*)(ws + L.off_vvvo);
        const int b = std::max(1, (nslots - 1) / 2);
        std::vector<int> slot_of(o, -1), owner(nslots, -1);
        std::vector<long long> stamp(nslots, 0);
        long long tick = 0;
        std::vector<const double*> sp(o, nullptr);
        std::vector<int4> list;
        std::vector<int> dest;
        auto flush_list = [&]() -> tc_status {
            for (size_t at = 0; at < list.size(); at += (size_t)L.batch) {
                const int nb = (int)std::min((size_t)L.batch, list.size() - at);
                for (int t = 0; t < nb; t++) list[at + t].w = t;
                TC_CUDA(ctx, cudaMemcpyAsync(d_trip, list.data() + at, sizeof(int4) * nb, cudaMemcpyHostToDevice, s));
                TC_CUDA(ctx, cudaMemcpyAsync(d_dest, dest.data() + at, sizeof(int) * nb, cudaMemcpyHostToDevice, s));
                TC_CUDA(ctx, cudaMemcpyAsync(d_sliceslot, slot_of.data(), sizeof(int) * o, cudaMemcpyHostToDevice, s));
                TC_CUDA(ctx, cudaMemcpyAsync(d_sliceptr, sp.data(), sizeof(double*) * o, cudaMemcpyHostToDevice, s));
                a.n_trip = nb;
                TC_CUDA(ctx, tc_launch_wbuild(a, &maps, d_orbits, s));
                TC_CUDA(ctx, tc_launch_reduce_units(d_partial, nb, L.n_orbits, d_dest, d_S, s));
                ctx->stats.n_kernel_launches += 2;
                ctx->stats.n_work_units += (long long)nb * L.n_orbits;
            }
            list.clear();
            dest.clear();
            return TC_OK;
        };
        // make slice x resident without evicting any slice of `keep`
        auto ensure = [&](int x, const std::vector<int>& keep) -> tc_status {
            if (slot_of[x] >= 0) {
                stamp[slot_of[x]] = ++tick;
                return TC_OK;
            }
            int victim = -1;
            for (int q = 0; q < nslots; q++) {
                if (owner[q] >= 0 && std::find(keep.begin(), keep.end(), owner[q]) != keep.end()) continue;
                if (victim < 0 || owner[q] < 0 || (owner[victim] >= 0 && stamp[q] < stamp[victim])) victim = q;
                if (owner[q] < 0) break;
            }
            if (victim < 0) TC_FAIL(ctx, TC_ERR_INTERNAL, "slice cache: no evictable slot");
            if (owner[victim] >= 0) {
                slot_of[owner[victim]] = -1;
                sp[owner[victim]] = nullptr;
            }
            double* dst = w_vvvo + (size_t)victim * slice_stride;
            TC_CUDA(ctx, tc_launch_df_gemm(df->Bvv, (size_t)v * v, df->Bov + (size_t)x * v, (size_t)o * v, v * v, v, df->naux, 1,
                                           (long long)v, 0, v, 0, 1, dst, s));
            ctx->stats.n_kernel_launches++;
            ctx->stats.slices_built++;
            owner[victim] = x;
            slot_of[x] = victim;
            sp[x] = dst;
            stamp[victim] = ++tick;
            return TC_OK;
        };
        long long idx = first;
        const long long end = first + count;
        while (idx < end) {
            int i, j, k;
            tc_triplet_decode(o, idx, &i, &j, &k, nullptr);
            // the (j,k) pairs of this i inside the range: idx .. min(end, start of i+1)
            const long long next_i = (long long)(i + 1) * (i + 2) * (i + 3) / 6;
            const long long stop = std::min(end, next_i);
            std::vector<int4> pairs;  // (j, k, dest, 0)
            for (long long n = idx; n < stop; n++) {
                int ii, jj, kk;
                tc_triplet_decode(o, n, &ii, &jj, &kk, nullptr);
                pairs.push_back(make_int4(jj, kk, (int)(n - first), 0));
            }
            const int jmin = pairs.front().x, jmax = pairs.back().x;
            for (int j0 = (jmin / b) * b; j0 <= jmax; j0 += b) {
                for (int k0 = 0; k0 <= std::min(j0 + b - 1, jmax); k0 += b) {
                    std::vector<int> need(1, i);
                    for (const int4& pr : pairs) {
                        if (pr.x < j0 || pr.x >= j0 + b || pr.y < k0 || pr.y >= k0 + b) continue;
                        list.push_back(make_int4(i, pr.x, pr.y, 0));
                        dest.push_back(pr.z);
                        if (std::find(need.begin(), need.end(), pr.x) == need.end()) need.push_back(pr.x);
                        if (std::find(need.begin(), need.end(), pr.y) == need.end()) need.push_back(pr.y);
                    }
                    if (list.empty()) continue;
                    for (int x : need) {
                        st = ensure(x, need);
                        if (st != TC_OK) return st;
                    }
                    st = flush_list();
                    if (st != TC_OK) return st;
                }
            }
            idx = stop;
        }
    }
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_c1, s));
    TC_CUDA(ctx, tc_launch_reduce_energy(d_S, d_w, count, d_E, s));
    ctx->stats.n_kernel_launches++;
    if (S_dev && count > 0) TC_CUDA(ctx, cudaMemcpyAsync(S_dev, d_S, sizeof(double) * (size_t)count, cudaMemcpyDeviceToDevice, s));
    TC_CUDA(ctx, cudaMemcpyAsync(ctx->pinned, d_E, sizeof(double), cudaMemcpyDeviceToHost, s));
    TC_CUDA(ctx, cudaEventRecord(ctx->ev_t1, s));
    TC_CUDA(ctx, cudaStreamSynchronize(s));

    float ms = 0;
    cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1);
    ctx->stats.ms_total = ms;
    cudaEventElapsedTime(&ms, ctx->ev_c0, ctx->ev_c1);
    ctx->stats.ms_contraction = ms;
    if (df) {
        cudaEventElapsedTime(&ms, ctx->ev_s0, ctx->ev_s1);
        ctx->stats.ms_staging = ms;
    }
    long long nz = 0;
    for (long long n = 0; n < count; n++) {
        int i, j, k;
        double w;
        tc_triplet_decode(o, first + n, &i, &j, &k, &w);
        if (w != 0.0) nz++;
    }
    ctx->stats.n_triplets = nz;
    ctx->stats.flop_contraction = (double)nz * 12.0 * (double)v * v * v * ((double)v + o);
    *E_partial_out = (count > 0) ? ctx->pinned[0] : 0.0;
    return TC_OK;
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
    std::vector<int4> orb;
    fill_orbits(v, orb);
    std::vector<const double*> sp(o);
    for (int x = 0; x < o; x++) sp[x] = blocks->vvvo + (size_t)x * v * v * v;
    // debug path: small temporaries allocated here (not a compute call of the hot path)
    char* tmp = nullptr;
    const size_t b_orb = align_up(sizeof(int4) * orb.size()), b_sp = align_up(sizeof(double*) * o + sizeof(int) * o);
    const size_t b_part = align_up(sizeof(double) * orb.size());
    const size_t b_dummy = align_up(sizeof(double) * (size_t)(o > v ? o : v) * v);
    TC_CUDA(ctx, cudaMalloc(&tmp, b_orb + b_sp + 256 + b_part + b_dummy));
    int4 trip = make_int4(i, j, k, 0);
    cudaError_t e = cudaMemcpyAsync(tmp, orb.data(), sizeof(int4) * orb.size(), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tmp + b_orb, sp.data(), sizeof(double*) * o, cudaMemcpyHostToDevice, s);
    std::vector<int> slot(o);
    for (int x = 0; x < o; x++) slot[x] = x;
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(tmp + b_orb + sizeof(double*) * o, slot.data(), sizeof(int) * o, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tmp + b_orb + b_sp, &trip, sizeof(int4), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(tmp + b_orb + b_sp + 256 + b_part, 0, b_dummy, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) {
        tc_wbuild_args a;
        a.o = o;
        a.v = v;
        const double* zeros = (const double*)(tmp + b_orb + b_sp + 256 + b_part);
        a.eps_occ = zeros;  // the epilogue result is discarded; only W is wanted
        a.eps_vir = zeros;
        a.t1 = zeros;
        a.t2 = t2;
        a.slice_ptr = (const double* const*)(tmp + b_orb);
        a.slices_aligned16 = ((uintptr_t)blocks->vvvo % 16 == 0) && (((size_t)v * v * v * sizeof(double)) % 16 == 0);
        a.ovoo = blocks->ovoo;
        a.ovov = blocks->ovov;
        a.triplets = (const int4*)(tmp + b_orb + b_sp);
        a.n_trip = 1;
        a.partial = (double*)(tmp + b_orb + b_sp + 256);
        a.n_orbits = (int)orb.size();
        a.slice_slot = (const int*)(tmp + b_orb + sizeof(double*) * o);
        a.W_debug = W_dev;
        tc_wbuild_maps maps;
        e = tc_wbuild_make_maps(a, blocks->vvvo, (size_t)v * v * v, o, &maps);
        if (getenv("TC_FORCE_CPASYNC")) maps.valid = false;
        if (e == cudaSuccess) e = tc_launch_wbuild(a, &maps, (const int4*)tmp, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    }
    cudaFree(tmp);
    if (e != cudaSuccess) TC_FAIL(ctx, TC_ERR_CUDA, "debug W kernel failed: %s", cudaGetErrorString(e));
    return TC_OK;
}
