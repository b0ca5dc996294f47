// tc_plan.h -- the blocked schedule (host): see tc_plan.cu.
#pragma once

#include <vector>

#include "tc_common.cuh"

struct tc_plan_load {
    int x;     // occupied index whose operands (slice I_x, and the row t2[x] when t2 is host-resident) are loaded ...
    int slot;  // ... into this slot
};

struct tc_plan_block {
    long long rec_begin;      // first record of the block in tc_plan::recs
    int n;                    // triplets in the block (one W-builder launch)
    int load_begin, load_end; // its loads in tc_plan::loads
    long long wait_block;     // the loads overwrite slots last used by this block (-1: never used)
};

struct tc_plan {
    std::vector<tc_trip_rec> recs;   // execution order; row = position inside its block
    std::vector<int> dest;           // recs[r] is triplet first + dest[r] of the range
    std::vector<tc_plan_load> loads;
    std::vector<tc_plan_block> blocks;
    int bi, bj, bk, nslots;
};

// false: nslots cannot hold the three operands of a triplet
bool tc_build_plan(int o, long long first, long long count, int nslots, tc_plan* out);
