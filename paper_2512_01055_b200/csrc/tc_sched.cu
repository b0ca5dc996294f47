// tc_sched.cu -- a1: the triplet scheduler (host side).
// Enumerates i >= j >= k with the degeneracy weight 2 - d_ij - d_jk of eq. (1)
// (the paper writes the weight over a >= b >= c, SURVEY 8(c) item 6 shows the
// occupied form is sum-equivalent).  idx(i,j,k) = i(i+1)(i+2)/6 + j(j+1)/2 + k.
#include <math.h>

#include "tc_common.cuh"

static inline long long tet(long long i) { return i * (i + 1) * (i + 2) / 6; }
static inline long long tri(long long j) { return j * (j + 1) / 2; }

extern "C" long long tc_triplet_count(int o) {
    if (o < 1) return -1;
    return tet(o);
}

extern "C" long long tc_triplet_index(int o, int i, int j, int k) {
    if (o < 1 || i >= o || k < 0 || j > i || k > j) return -1;
    return tet(i) + tri(j) + k;
}

extern "C" tc_status tc_triplet_decode(int o, long long idx, int* pi, int* pj, int* pk, double* weight) {
    if (o < 1 || idx < 0 || idx >= tet(o) || !pi || !pj || !pk) return TC_ERR_INVALID_ARG;
    // closed-form estimate of the tetrahedral / triangular roots, then fix up by +-1
    long long i = (long long)floor(cbrt(6.0 * (double)idx));
    if (i < 0) i = 0;
    while (tet(i + 1) <= idx) i++;
    while (i > 0 && tet(i) > idx) i--;
    long long rest = idx - tet(i);
    long long j = (long long)floor((sqrt(8.0 * (double)rest + 1.0) - 1.0) * 0.5);
    if (j < 0) j = 0;
    while (tri(j + 1) <= rest) j++;
    while (j > 0 && tri(j) > rest) j--;
    long long k = rest - tri(j);
    *pi = (int)i;
    *pj = (int)j;
    *pk = (int)k;
    if (weight) *weight = 2.0 - (i == j ? 1.0 : 0.0) - (j == k ? 1.0 : 0.0);
    return TC_OK;
}

// Multi-GPU sharding: contiguous ranges of the linear triplet index, sizes differing by at most one.
extern "C" tc_status tc_triplet_partition(int o, int world, int rank, long long* first, long long* count) {
    if (o < 1 || world < 1 || rank < 0 || rank >= world || !first || !count) return TC_ERR_INVALID_ARG;
    const long long n = tet(o), base = n / world, rem = n % world;
    *first = rank * base + (rank < rem ? rank : rem);
    *count = base + (rank < rem ? 1 : 0);
    return TC_OK;
}
