// tc_plan.cu -- a1/a2 host logic: the blocked schedule used when the per-occupied-index operands (the (vv|v.)
// slices I_x and, for host-resident amplitudes, the rows t2[x]) are cached in fewer slots than there are occupied
// indices (SURVEY 8(a) a2 "LRU of slots"; the paper bounds memory by tiling and rebuilds integrals from Cholesky
// pieces on the device).
//
// The triplets of the range are cut into blocks of bi x bj x bk occupied indices (i slowest, k fastest).  A block needs
// the operands of its i's, j's and k's; missing ones are loaded into slots chosen by LRU among the slots the block
// does not need.  The i and j blocks stay while the k blocks stream through, so a block of bi*bj*bk triplets costs
// about bk loads: one streamed operand is reused over the bi x bj footprint.  The shape is chosen by simulation: of
// the candidates with bi + bj + 2 bk <= nslots (room to stage block n+1 while block n computes) the one with the
// fewest loads.  Every load records the last block that used its slot: the side stream
// must not overwrite the slot before that block's W-builder has finished.
#include <algorithm>

#include "tc_plan.h"

namespace {

struct Sim {
    int o, nslots;
    std::vector<int> slot_of, owner;
    std::vector<long long> stamp, last_use;
    long long tick = 0;
    Sim(int o_, int n) : o(o_), nslots(n), slot_of(o_, -1), owner(n, -1), stamp(n, 0), last_use(n, -1) {}
};

// runs the schedule; emit == nullptr: count only
bool run_schedule(int o, long long first, long long count, int nslots, int bi, int bj, int bk, tc_plan* emit,
                  long long* n_blocks, long long* n_loads) {
    Sim sm(o, nslots);
    long long blocks = 0, loads = 0;
    std::vector<char> needed(o, 0);
    std::vector<int> need;
    const long long end = first + count;
    if (count <= 0) {
        if (n_blocks) *n_blocks = 0;
        if (n_loads) *n_loads = 0;
        return true;
    }
    int i_lo, i_hi, jj, kk;
    if (tc_triplet_decode(o, first, &i_lo, &jj, &kk, nullptr) != TC_OK) return false;
    if (tc_triplet_decode(o, end - 1, &i_hi, &jj, &kk, nullptr) != TC_OK) return false;
    auto mark = [&](int x) {
        if (!needed[x]) {
            needed[x] = 1;
            need.push_back(x);
        }
    };
    for (int i0 = (i_lo / bi) * bi; i0 <= i_hi; i0 += bi) {
        const int i1 = std::min(i0 + bi - 1, i_hi);
        for (int j0 = 0; j0 <= i1; j0 += bj) {
            const int j1 = std::min(j0 + bj - 1, i1);
            for (int k0 = 0; k0 <= j1; k0 += bk) {
                const int k1 = std::min(k0 + bk - 1, j1);
                need.clear();
                const long long rec_begin = emit ? (long long)emit->recs.size() : 0;
                int n_in_block = 0;
                // k slowest inside the block: consecutive CTAs of a launch then share the k slice, and mostly i or j
                for (int k = k0; k <= k1; k++)
                    for (int i = std::max(i0, i_lo); i <= i1; i++)
                        for (int j = std::max(j0, k); j <= std::min(j1, i); j++) {
                            const long long idx = (long long)i * (i + 1) * (i + 2) / 6 + (long long)j * (j + 1) / 2 + k;
                            if (idx < first || idx >= end) continue;
                            n_in_block++;
                            mark(i);
                            mark(j);
                            mark(k);
                            if (emit) {
                                tc_trip_rec r;
                                r.occ[0] = i; r.occ[1] = j; r.occ[2] = k;
                                r.row = 0;
                                r.pad0 = r.pad1 = 0;
                                emit->recs.push_back(r);
                                emit->dest.push_back((int)(idx - first));
                            }
                        }
                if (n_in_block == 0) continue;
                if ((int)need.size() > nslots) return false;
                const int load_begin = emit ? (int)emit->loads.size() : 0;
                long long wait_block = -1;
                for (int x : need) {
                    if (sm.slot_of[x] >= 0) continue;
                    int victim = -1;
                    for (int q = 0; q < nslots; q++) {
                        if (sm.owner[q] < 0) { victim = q; break; }
                        if (needed[sm.owner[q]]) continue;
                        if (victim < 0 || sm.stamp[q] < sm.stamp[victim]) victim = q;
                    }
                    if (victim < 0) return false;
                    if (sm.owner[victim] >= 0) sm.slot_of[sm.owner[victim]] = -1;
                    sm.owner[victim] = x;
                    sm.slot_of[x] = victim;
                    wait_block = std::max(wait_block, sm.last_use[victim]);
                    loads++;
                    if (emit) emit->loads.push_back({x, victim});
                }
                for (int x : need) {
                    const int q = sm.slot_of[x];
                    sm.stamp[q] = ++sm.tick;
                    sm.last_use[q] = blocks;
                    needed[x] = 0;
                }
                if (emit) {
                    for (long long r = rec_begin; r < (long long)emit->recs.size(); r++) {
                        tc_trip_rec& rec = emit->recs[r];
                        rec.row = (int)(r - rec_begin);
                        for (int p = 0; p < 3; p++) rec.s[p] = rec.t[p] = sm.slot_of[rec.occ[p]];
                    }
                    tc_plan_block b;
                    b.rec_begin = rec_begin;
                    b.n = n_in_block;
                    b.load_begin = load_begin;
                    b.load_end = (int)emit->loads.size();
                    b.wait_block = wait_block;
                    emit->blocks.push_back(b);
                }
                blocks++;
            }
        }
    }
    if (n_blocks) *n_blocks = blocks;
    if (n_loads) *n_loads = loads;
    return true;
}

}  // namespace

bool tc_build_plan(int o, long long first, long long count, int nslots, tc_plan* out) {
    if (o < 1 || (nslots < 3 && nslots < o)) return false;
    if (nslots > o) nslots = o;
    int best[3] = {1, 1, 1};
    long long best_loads = -1, best_blocks = 0;
    auto consider = [&](int bi, int bj, int bk) {
        if (bi < 1 || bj < 1 || bk < 1) return;   // run_schedule rejects shapes whose blocks need more than nslots operands
        bi = std::min(bi, o);
        bj = std::min(bj, o);
        bk = std::min(bk, o);
        long long nb = 0, nl = 0;
        if (!run_schedule(o, first, count, nslots, bi, bj, bk, nullptr, &nb, &nl)) return;
        if (best_loads < 0 || nl < best_loads || (nl == best_loads && nb < best_blocks)) {
            best_loads = nl;
            best_blocks = nb;
            best[0] = bi;
            best[1] = bj;
            best[2] = bk;
        }
    };
    // candidate shapes.  With room to spare, bi + bj + 2 bk <= nslots: the next k block is staged while the current one
    // computes.  The i x j footprint is what a streamed k operand is reused over, so shapes from 1 x (n-3) to square.
    if (nslots >= o) {
        consider(o, o, o);
    } else if (nslots <= 4) {
        consider(1, 1, 1);
        consider(1, nslots - 2, 1);
    } else {
        for (int bk = 1; bk <= 2; bk++) {
            const int room = nslots - 2 * bk;   // bi + bj
            if (room < 2) continue;
            for (int bi = 1; bi <= room / 2; bi++) consider(bi, room - bi, bk);
        }
        consider((nslots - 1) / 3, (nslots - 1) / 3, (nslots - 1) / 3);
    }
    if (best_loads < 0 && count > 0) return false;
    out->recs.clear();
    out->dest.clear();
    out->loads.clear();
    out->blocks.clear();
    out->bi = best[0];
    out->bj = best[1];
    out->bk = best[2];
    out->nslots = nslots;
    if (count == 0) return true;
    return run_schedule(o, first, count, nslots, best[0], best[1], best[2], out, nullptr, nullptr);
}

extern "C" tc_status tc_plan_summary(int o, long long first, long long count, int nslots, long long* n_blocks,
                                     long long* n_loads, int* bi, int* bj, int* bk) {
    const long long ntrip = tc_triplet_count(o);
    if (o < 1 || first < 0 || count < 0 || first + count > ntrip || (nslots < 3 && nslots < o)) return TC_ERR_INVALID_ARG;
    tc_plan plan;
    if (!tc_build_plan(o, first, count, nslots, &plan)) return TC_ERR_INTERNAL;
    if (n_blocks) *n_blocks = (long long)plan.blocks.size();
    if (n_loads) *n_loads = (long long)plan.loads.size();
    if (bi) *bi = plan.bi;
    if (bj) *bj = plan.bj;
    if (bk) *bk = plan.bk;
    return TC_OK;
}

extern "C" tc_status tc_plan_dump(int o, long long first, long long count, int nslots, int* recs_out, int* loads_out,
                                  long long loads_capacity) {
    const long long ntrip = tc_triplet_count(o);
    if (o < 1 || first < 0 || count < 0 || first + count > ntrip || (nslots < 3 && nslots < o) || !recs_out || !loads_out)
        return TC_ERR_INVALID_ARG;
    tc_plan plan;
    if (!tc_build_plan(o, first, count, nslots, &plan)) return TC_ERR_INTERNAL;
    if ((long long)plan.loads.size() > loads_capacity) return TC_ERR_WORKSPACE_TOO_SMALL;
    for (size_t n = 0; n < plan.blocks.size(); n++) {
        const tc_plan_block& b = plan.blocks[n];
        for (long long r = b.rec_begin; r < b.rec_begin + b.n; r++) {
            const tc_trip_rec& rec = plan.recs[r];
            int* out = recs_out + 8 * r;
            out[0] = rec.occ[0]; out[1] = rec.occ[1]; out[2] = rec.occ[2];
            out[3] = plan.dest[r];
            out[4] = (int)n;
            out[5] = rec.s[0]; out[6] = rec.s[1]; out[7] = rec.s[2];
        }
        for (int q = b.load_begin; q < b.load_end; q++) {
            int* out = loads_out + 4 * q;
            out[0] = (int)n;
            out[1] = plan.loads[q].x;
            out[2] = plan.loads[q].slot;
            out[3] = (int)b.wait_block;
        }
    }
    return TC_OK;
}
