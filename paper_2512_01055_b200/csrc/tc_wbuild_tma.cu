// tc_wbuild_tma.cu -- steps a3-a6 of the hot path: fused W-builder + epilogue (sm_100a).
//
// One CTA = one work unit = (occupied triplet i>=j>=k) x (S3-orbit of a virtual tile triple {A,B,C}, A>=B>=C,
// tile edge T=16).  The up-to-six permuted T^3 tiles of W_ijk (eqs. (2),(5)) live in shared memory
// for the whole unit (192 KB); W and Y never touch HBM.
//
// Contraction algebra.  Every step is one dense 32 x 256 x K GEMM on the FP64 tensor cores whose
// two 16-row halves are added into two W tiles with the index permutation folded into the shared-memory address (no
// PERMUTE kernel).  For an arrangement (m-tile, n1-tile, n2-tile) of the orbit:
//   particle step z:  P[m][n1][n2] = sum_d t2[x][y][m][d] * vvvo[z][d][n1][n2]    K = v   rows 0-15: (x,y), 16-31: (y,x)
//   hole step y:      H[m][n1][n2] = sum_l ovoo[z][x][l][m] * t2[y][l][n1][n2]    K = o   rows 0-15 / 16-31: the two (z,x)
//                                                                                          with {x,y,z} = {i,j,k} sharing y
// (the hole B operand depends on y only, so the six 16-row hole terms of an arrangement pair up into three 32-row
// steps).  Hole results enter W with a minus sign (eq. (2)).
//
// Six steps per arrangement, in the order H0 H1 P0 H2 P1 P2: each hole term is the hole part of one particle term, so a hole
// step's accumulators are parked in tensor memory and the particle steps START from them; one flush then carries both
// contractions of a (tile, orientation) pair.
//
// Roles (512 threads, 1 CTA per SM):
//   warps 0-7   consumers, warp tile 32 x 32: per ring stage  wait full -> 8 conflict-free LDS.64 -> 16 DMMA.8x8x4 -> release.
//               A stage is one K chunk of 4, or two K chunks when the n1 or n2 tile is ragged and half the B stage would be
//               idle (MODE_Z2 / MODE_Y2).  At the end of a step the 32 accumulators of each thread are PARKED in tensor memory
//               (tcgen05.st): a hole step for the particle steps of the same threads, a particle step for the flushers.
//   warps 8-11  producers, one operand stream each (B columns 0-7 + expect_tx, B columns 8-15, A rows 0-15, A rows 16-31)
//               into a 3-stage ring.  Particle B comes from slices the stager laid out in fragment order, 4 KB contiguous
//               per chunk and column half (cp.async.bulk); hole B and both A operands are cp.async.bulk.tensor boxes that
//               land in the same fragment order.  At the end they stage the epilogue's (ov|ov) blocks in the ring memory.
//   warps 12-15 flushers: read the parked particle steps back (tcgen05.ld) and add them into the W tiles, permutation in
//               the address -- off the consumers' critical path.
//   After the last step consumers and flushers run the fused epilogue (tcw::orbit_energy).
// Ragged tiles are zero-filled (TMA out-of-bounds fill, zero padding of the slices); 8-blocks entirely outside v are
// neither loaded nor multiplied.  CTA order: tile orbit slow, triplet fast (L2 reuse between concurrent CTAs).
#include <type_traits>

#include "tc_tma.cuh"
#include "tc_tmem.cuh"
#include "tc_wbuild_shared.cuh"

namespace {

using tcw::c_perm;
using tcw::T;
using tcw::TILE;

constexpr int KC = 4;                     // K chunk = one DMMA k-step
constexpr int STAGES = 3;                 // operand ring depth (smem: 192 KB of W tiles leave 35 KB)
constexpr int NCONS_WARPS = 8;
constexpr int NCONS = NCONS_WARPS * 32;   // consumer threads
constexpr int NFLUSH = 128;               // flusher threads (warps 12-15)
constexpr int NTHREADS = 512;
constexpr int B_STAGE = 2 * 16 * KC * 8;  // doubles: [z][n1][k][8]
constexpr int A_STAGE = 2 * 4 * 32;       // doubles: [K chunk 0/1][four 8-row blocks [m 8][k 4]]; chunk 1 only in the paired modes
constexpr int MAX_STEPS = 36;
constexpr uint32_t B_HALF_BYTES = 16 * KC * 8 * 8;  // 4096
constexpr uint32_t A_BOX_BYTES = KC * 16 * 8;       // 512
constexpr int TBUF_COLS = 128;            // one parked step: 2 consumer warps per lane quarter x 64 columns
constexpr int TB_HOLE = 0;                // TMEM buffers 0-2: the three hole steps of the current arrangement
constexpr int TB_PART = 3;                // TMEM buffer 3: the particle step handed to the flushers
constexpr int TMEM_COLS = 4 * TBUF_COLS;
constexpr int EPI_SPLIT = 11;             // epilogue: the consumers take la < 11 of their (lb, lc), the flushers la >= 11 of two pairs

// Step modes.  A step whose n2 (or n1) tile has at most 8 valid indices needs only half of the B stage per K chunk; it then packs
// TWO K chunks into every ring stage, so that a stage still carries 16 DMMAs per warp (a stage with 8 costs almost as much time:
// the per-stage synchronisation and the ring's depth in time do not shrink with it):
//   MODE_Z2: n2 ragged -- stage half kk holds the z = 0 half of chunk 2r + kk
//   MODE_Y2: n1 ragged -- rows 8 kk .. 8 kk + 7 of stage half z hold the rows n1 = 0..7 of chunk 2r + kk
// Steps whose m tile is ragged cannot do this (their B chunk is full size) and run with 8 DMMAs per stage.
constexpr int MODE_PLAIN = 0, MODE_Z2 = 1, MODE_Y2 = 2;

// (104 bytes: an odd number of 8-byte words.  The 36 table-building threads write their records at this stride; 112- or
// 128-byte records measured 1.5 % slower.)
struct Step {
    int nstages;       // ring stages of the step: K chunks, or pairs of K chunks in the paired modes
    int mode;
    int particle;      // 1: B = slice (bulk copies), A = t2 rows; 0: hole step, B = amplitude row (boxes), A = (ov|oo)^T
    int nxb, ny, nz;   // 8-blocks with at least one index below v: rows, n1, n2 (1 or 2)
    int W0, U0, V0;    // first virtual index of the m, n1 and n2 tiles
    const double* b_src;   // particle: chunk 0, column half 0 of the (n1, n2) tile of slice z (tiled layout); hole: NULL
    int b_c3;              // hole: slot of the amplitude row t2[y]
    int a_c2[2], a_c3[2];  // A box coordinates of the two halves: particle (y, slot of t2[x]); hole (x, z) of (ov|oo)^T
    int slot[2];           // shared-memory W tile receiving half h
    int sm[2], sn1[2], sn2[2];  // address strides of m, n1, n2 in that tile (0 for the rotated last coordinate)
};

static_assert(sizeof(Step) == 104, "see the comment at Step");
static_assert(STAGES * (B_STAGE + A_STAGE) >= tcw::KST_DOUBLES, "the epilogue stages its (ov|ov) blocks in the operand ring");

struct __align__(128) Smem {
    double tiles[6 * TILE];
    double B[STAGES][B_STAGE];
    double A[STAGES][A_STAGE];
    Step steps[MAX_STEPS];
    unsigned long long full[STAGES];
    unsigned long long empty[STAGES];
    unsigned long long tfull;          // consumers -> flushers: a particle step is parked
    unsigned long long tfree;          // flushers -> consumers: it has been read back
    unsigned long long tdone;          // flushers -> consumers: every step but the last is in the W tiles
    unsigned long long tlast;          // consumers -> flushers: the last step has read its hole terms, tensor memory is idle
    unsigned long long kready;         // producers -> epilogue: the (ov|ov) blocks are staged in the operand ring
    double red[NCONS_WARPS + NFLUSH / 32];
    int slot_of_perm[6];
    int nsteps;
    uint32_t tmem_base;
};

__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" ::"n"(NCONS) : "memory"); }
__device__ __forceinline__ void flusher_bar() { asm volatile("bar.sync 2, %0;" ::"n"(NFLUSH) : "memory"); }
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

// a[i] for a runtime i without putting the array into local memory
__device__ __forceinline__ int pick3(const int (&a)[3], int i) { return i == 0 ? a[0] : (i == 1 ? a[1] : a[2]); }

struct ConsumerState {
    int stage;        // ring position of the next chunk to consume
    uint32_t parity;  // its full-barrier parity
    int lane;
    uint32_t full0, empty0;  // shared addresses of full[0] / empty[0]
    uint32_t bB, bA;         // this thread's fragment addresses in stage 0
    uint32_t zero;           // 0, but not to the compiler (see release_stage)
};

// Hands a ring stage back to the producers.  The stage may be refilled as soon as every fragment of it is in registers, but
// "after the loads in program order" does not say that: a shared-memory load delivers its data asynchronously, and an mbarrier
// arrive issued behind it can become visible first (observed: with the arrive right behind the loads, about one unit in 20 000
// multiplied a fragment of the NEXT chunk when the refill was fast; tests/test_gpu_parity.py::test_abcijk_is_bit_reproducible).
// A DMMA reads its operands at issue and cannot issue before they have landed, so the arrive's address is made to depend on
// the results of DMMAs that between them take every fragment of the stage as an operand (`bits`, ANDed with a zero the compiler
// cannot see): wherever the assembler schedules the arrive, and in whatever order it issues the DMMAs, the loads have landed.
__device__ __forceinline__ uint32_t hi_bits(double x) { return (uint32_t)__double2hiint(x); }
__device__ __forceinline__ void release_stage(const ConsumerState& cs, uint32_t bits) {
    const uint32_t bar = cs.empty0 + cs.stage * 8 + (bits & cs.zero);
    __syncwarp();
    // lane 0 arrives; predicated, so that the address arithmetic stays outside a divergent branch
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.eq.u32 p, %1, 0;\n"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
        "}\n" ::"r"(bar),
        "r"(cs.lane)
        : "memory");
}

// One step of the consumer warps: n chunks of  wait full -> LDS -> DMMA -> release.
// NXB / NY / NZ = number of 8-blocks of rows (per half) / n1 / n2 that reach below v.
// The two warps of a scheduler may be up to STAGES-1 chunks apart in the ring and settle out of phase, so one warp's
// barrier/LDS latency is covered by the other's DMMAs (tc_bench_ring_peak measures this loop stand-alone).
template <int NXB, int NY, int NZ>
__device__ __forceinline__ void run_step(double (&acc)[4][2][2][2], ConsumerState& cs, int n) {
    constexpr uint32_t BST = B_STAGE * 8, AST = A_STAGE * 8;  // stage strides in bytes
#pragma unroll 2   // measured: +0.3 % over the rolled loop, 3 and 4 no better
    for (int r = 0; r < n; r++) {
        mbar_wait(cs.full0 + cs.stage * 8, cs.parity);
        const uint32_t pa = cs.bA + cs.stage * AST;
        const uint32_t pb = cs.bB + cs.stage * BST;
        double fa[2][NXB], fb[NY][NZ];
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int xb = 0; xb < NXB; xb++) fa[h][xb] = lds64(pa + (2 * h + xb) * 256);
#pragma unroll
        for (int y = 0; y < NY; y++)
#pragma unroll
            for (int z = 0; z < NZ; z++) fb[y][z] = lds64(pb + z * 4096 + y * 2048);
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int xb = 0; xb < NXB; xb++)
#pragma unroll
                for (int y = 0; y < NY; y++)
#pragma unroll
                    for (int z = 0; z < NZ; z++) dmma884(acc[2 * h + xb][y][z][0], acc[2 * h + xb][y][z][1], fa[h][xb], fb[y][z]);
        {
            // a covering set: NC = max(na, nb) blocks that between them take every row fragment and every column fragment as operands
            constexpr int NA = 2 * NXB, NB = NY * NZ, NC = NA > NB ? NA : NB;
            uint32_t bits = 0;
#pragma unroll
            for (int i = 0; i < NC; i++) {
                const int ia = (NC - 1 - i) % NA, ib = i % NB;   // the anti-diagonal: 0.3 % faster than the diagonal (scheduling)
                bits |= hi_bits(acc[2 * (ia / NXB) + ia % NXB][ib / NZ][ib % NZ][0]);
            }
            release_stage(cs, bits);
        }
        if (++cs.stage == STAGES) {
            cs.stage = 0;
            cs.parity ^= 1;
        }
    }
}

// The paired modes: two K chunks per stage.  MODE_Z2: fb[kk][y] from stage half kk, accumulators [..][y][0];
// MODE_Y2: fb[kk][z] from rows 8 kk.. of stage half z, accumulators [..][0][z].  NO = blocks of the other column index (1 or 2).
template <int NXB, int MODE, int NO>
__device__ __forceinline__ void run_step_paired(double (&acc)[4][2][2][2], ConsumerState& cs, int n) {
    constexpr uint32_t BST = B_STAGE * 8, AST = A_STAGE * 8;
#pragma unroll 2   // measured: +0.3 % over the rolled loop, 3 and 4 no better
    for (int r = 0; r < n; r++) {
        mbar_wait(cs.full0 + cs.stage * 8, cs.parity);
        const uint32_t pa = cs.bA + cs.stage * AST;
        const uint32_t pb = cs.bB + cs.stage * BST;
        double fa[2][2][NXB], fb[2][NO];
#pragma unroll
        for (int kk = 0; kk < 2; kk++)
#pragma unroll
            for (int h = 0; h < 2; h++)
#pragma unroll
                for (int xb = 0; xb < NXB; xb++) fa[kk][h][xb] = lds64(pa + kk * 1024 + (2 * h + xb) * 256);
#pragma unroll
        for (int kk = 0; kk < 2; kk++)
#pragma unroll
            for (int q = 0; q < NO; q++)
                fb[kk][q] = lds64(pb + (MODE == MODE_Z2 ? kk * 4096 + q * 2048 : q * 4096 + kk * 2048));
#pragma unroll
        for (int kk = 0; kk < 2; kk++)
#pragma unroll
            for (int h = 0; h < 2; h++)
#pragma unroll
                for (int xb = 0; xb < NXB; xb++)
#pragma unroll
                    for (int q = 0; q < NO; q++) {
                        if (MODE == MODE_Z2) dmma884(acc[2 * h + xb][q][0][0], acc[2 * h + xb][q][0][1], fa[kk][h][xb], fb[kk][q]);
                        else dmma884(acc[2 * h + xb][0][q][0], acc[2 * h + xb][0][q][1], fa[kk][h][xb], fb[kk][q]);
                    }
        {
            // every accumulator block is written by the K chunk kk = 1 last, after kk = 0 (a true dependency through the block):
            // a covering set of blocks therefore covers the fragments of both chunks
            constexpr int NA = 2 * NXB, NC = NA > NO ? NA : NO;
            uint32_t bits = 0;
#pragma unroll
            for (int i = 0; i < NC; i++) {
                const int ia = i % NA, q = i % NO;
                bits |= hi_bits(MODE == MODE_Z2 ? acc[2 * (ia / NXB) + ia % NXB][q][0][0] : acc[2 * (ia / NXB) + ia % NXB][0][q][0]);
            }
            release_stage(cs, bits);
        }
        if (++cs.stage == STAGES) {
            cs.stage = 0;
            cs.parity ^= 1;
        }
    }
}

// ---- the kernel ------------------------------------------------------------------------------
__global__ void __launch_bounds__(NTHREADS, 1)
k_wbuild_tma(const tc_wbuild_args a, const int4* __restrict__ orbits, const __grid_constant__ CUtensorMap mapT2h,
             const __grid_constant__ CUtensorMap mapT2h8, const __grid_constant__ CUtensorMap mapT2p,
             const __grid_constant__ CUtensorMap mapOvooT) {
    // no integer round trip in this cast: the compiler then knows that everything reached through `s` is shared memory (LDS / STS
    // with 32-bit addresses instead of generic loads)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    Smem& s = *reinterpret_cast<Smem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int o = a.o, v = a.v;

    // CTA order: tile orbit slow, triplet fast.  CTAs that run together then work on the same orbit for consecutive
    // triplets (i, j, k), (i, j, k+1), ...: they walk the same step sequence and share the tiles of the slices I_i and
    // I_j in L2.
    const int orbit = blockIdx.x / a.n_trip;
    const int trip = blockIdx.x - orbit * a.n_trip;
    const tc_trip_rec rec = a.recs[trip];
    const int occ[3] = {rec.occ[0], rec.occ[1], rec.occ[2]};
    const int4 ob = orbits[orbit];
    const int bv[3] = {ob.x, ob.y, ob.z};  // tile indices A >= B >= C
    if (occ[0] == occ[1] && occ[1] == occ[2] && !a.W_debug) {
        // weight 2 - d_ij - d_jk = 0 (and S_iii = 0 anyway: R vanishes by symmetry)
        if (tid == 0) a.partial[(size_t)rec.row * a.n_orbits + orbit] = 0.0;
        return;
    }
    const int nhc = (o + KC - 1) / KC;  // chunks of a hole step
    const int npc = (v + KC - 1) / KC;  // chunks of a particle step

    // ---- the step program: thread (q, n) writes step n of arrangement q.  Order H0 H1 P0 H2 P1 P2: hole step Hy (B = the
    //      amplitude row of occ[2 - y]) computes two 16-row terms that are the hole parts of two particle steps; each particle
    //      step Pz (slice role z) starts from the parked results of its two hole terms (see the consumers) ----
    if (tid < MAX_STEPS) {
        int sop[6];
        tcw::arrangement_slots(bv, sop);
        const int q = tid / 6, n = tid - 6 * q;
        int before = 0, distinct = 0, sop_pk = 0;   // sop packed four bits each: runtime lookups without a local array
#pragma unroll
        for (int q2 = 0; q2 < 6; q2++) {
            sop_pk |= sop[q2] << (4 * q2);
            if (sop[q2] == q2) {
                distinct++;
                if (q2 < q) before++;
            }
        }
        const int t3[3] = {rec.t[0], rec.t[1], rec.t[2]}, s3[3] = {rec.s[0], rec.s[1], rec.s[2]};
        if (tid == 0) {
            s.nsteps = 6 * distinct;
#pragma unroll
            for (int q2 = 0; q2 < 6; q2++) s.slot_of_perm[q2] = sop[q2];
        }
        if (((sop_pk >> (4 * q)) & 7) == q) {
            // c_perm and its inverse packed into constants: lookups with runtime indices by shifts instead of dependent
            // constant-memory loads (the step table is on every unit's critical path)
            constexpr unsigned long long PERM_PK = tcw::perm_packed();
            constexpr unsigned int PERM_INV = tcw::perm_inverse_packed();
            const int pw = (int)(PERM_PK >> (6 * q)) & 3, pu = (int)(PERM_PK >> (6 * q + 2)) & 3, pvv = (int)(PERM_PK >> (6 * q + 4)) & 3;  // which of (A,B,C) is the m / n1 / n2 tile
            Step& d = s.steps[6 * before + n];
            const int tU = pick3(bv, pu), tV = pick3(bv, pvv);
            d.W0 = pick3(bv, pw) * T;
            d.U0 = tU * T;
            d.V0 = tV * T;
            d.nxb = (v - d.W0 > 8) ? 2 : 1;
            d.ny = (v - d.U0 > 8) ? 2 : 1;
            d.nz = (v - d.V0 > 8) ? 2 : 1;
            const bool particle = (n == 2 || n >= 4);
            const int sub = (n < 2) ? n : (n == 2 ? 0 : (n == 3 ? 2 : n - 3));   // y of a hole step / z of a particle step
            d.particle = particle ? 1 : 0;
            d.mode = (d.nz == 1) ? MODE_Z2 : (d.ny == 1 ? MODE_Y2 : MODE_PLAIN);
            {
                const int nchunks = particle ? npc : nhc;
                d.nstages = (d.mode == MODE_PLAIN) ? nchunks : (nchunks + 1) / 2;
            }
            // the two (slice role zp, family h) terms this step computes in rows 0-15 and 16-31:
            //   family 0 of role zp: (x,y,z) = (occ[xp], occ[yp], occ[zp]),  m -> position xp, n1 -> yp, n2 -> zp
            //   family 1 of role zp: (y,x,z),                                m -> position yp, n1 -> xp, n2 -> zp
            int zps[2], hs[2];
            if (particle) {
                zps[0] = zps[1] = sub;
                hs[0] = 0;
                hs[1] = 1;
            } else {
                // hole steps pair the terms that share the amplitude row of B: occ[2]: (0,0),(1,0); occ[1]: (0,1),(2,0);
                // occ[0]: (1,1),(2,1)
                const int yy = sub;
                zps[0] = (yy == 2) ? 1 : 0;
                hs[0] = (yy == 0) ? 0 : 1;
                zps[1] = (yy == 0) ? 1 : 2;
                hs[1] = (yy == 2) ? 1 : 0;
            }
#pragma unroll
            for (int hh = 0; hh < 2; hh++) {
                const int zp = zps[hh], h = hs[hh];
                const int xp = (zp == 0) ? 1 : 0;
                const int yp = (zp == 2) ? 1 : 2;
                const int pm = h ? yp : xp, pn1 = h ? xp : yp, pn2 = zp;
                // the ordering that has tile role pw at position pm, pu at pn1, pvv at pn2
                const int a0 = (pm == 0) ? pw : (pn1 == 0 ? pu : pvv), a1 = (pm == 1) ? pw : (pn1 == 1 ? pu : pvv);
                const int qq = (int)(PERM_INV >> (3 * (4 * a0 + a1))) & 7;
                d.slot[hh] = (sop_pk >> (4 * qq)) & 7;
                d.sm[hh] = (pm == 0) ? T * T : (pm == 1 ? T : 0);
                d.sn1[hh] = (pn1 == 0) ? T * T : (pn1 == 1 ? T : 0);
                d.sn2[hh] = (pn2 == 0) ? T * T : (pn2 == 1 ? T : 0);
                if (particle) {   // A = t2[x][y][m][d] (family 0) or t2[y][x][m][d] (family 1): box coordinates (second index, row slot)
                    d.a_c2[hh] = h ? pick3(occ, xp) : pick3(occ, yp);
                    d.a_c3[hh] = h ? pick3(t3, yp) : pick3(t3, xp);
                } else {          // A = (ov|oo)^T[z][x'][m][l], x' = x (family 0) or y (family 1)
                    d.a_c2[hh] = h ? pick3(occ, yp) : pick3(occ, xp);
                    d.a_c3[hh] = pick3(occ, zp);
                    d.b_c3 = h ? pick3(t3, xp) : pick3(t3, yp);   // B = t2[y'][l][n1][n2], y' = y (family 0) or x (family 1): the same row for both halves
                }
            }
            if (particle) {
                const int zp = sub;
                const size_t nb = (size_t)((v + T - 1) / T);
                // tile pair (n1 tile, n2 tile): global tile indices, or (abcijk schedule) their positions in this orbit's (A, B, C)
                const size_t pair = a.orbit_local ? (size_t)(pu * 3 + pvv) : (size_t)tU * nb + tV;
                d.b_src = a.slices + (a.orbit_local ? (size_t)orbit * a.orbit_stride : 0) + (size_t)pick3(s3, zp) * a.slice_stride +
                          pair * (size_t)tc_tiled_kchunks(v) * B_STAGE;
                d.b_c3 = 0;
            } else {
                d.b_src = nullptr;
            }
        }
    }
    if (tid == 2 * 32) {   // a warp that builds no step: in parallel with the table
        for (int n = 0; n < STAGES; n++) {
            mbar_init(smem_u32(&s.full[n]), 1);
            mbar_init(smem_u32(&s.empty[n]), NCONS_WARPS);
        }
        mbar_init(smem_u32(&s.tfull), NCONS_WARPS);
        mbar_init(smem_u32(&s.tfree), NFLUSH / 32);
        mbar_init(smem_u32(&s.tdone), NFLUSH / 32);
        mbar_init(smem_u32(&s.tlast), NCONS_WARPS);
        mbar_init(smem_u32(&s.kready), 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 12) tmem_alloc(smem_u32(&s.tmem_base), TMEM_COLS);
    tmem_fence_before();
    __syncthreads();
    tmem_fence_after();

    const int nsteps = s.nsteps;
    const uint32_t tmem_base = s.tmem_base;

    if (warp >= 12) {
        // =========================== flushers: parked accumulators -> W tiles ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 120;");
        const int fw = warp - 12;   // lane quarter fw: the consumer warps fw and fw + 4 park here
        const int ft = tid - 384;
        for (int n = ft; n < 6 * TILE; n += NFLUSH) s.tiles[n] = 0.0;
        flusher_bar();
        const int fr = lane >> 2, fk = lane & 3;
        const uint32_t tiles0 = smem_u32(&s.tiles[0]);
        const uint32_t tfull0 = smem_u32(&s.tfull), tfree0 = smem_u32(&s.tfree);
        const uint32_t tlane = tmem_base + ((uint32_t)(fw * 32) << 16) + TB_PART * TBUF_COLS;
        // only the particle steps are flushed: they start from their hole terms (parked in TMEM by the same threads), so one
        // flush carries both contractions of a (tile, orientation) pair -- half the shared-memory traffic of flushing every step
        // ... except the unit's last step, which the consumers (idle by then) add in from their registers
        const int nflush = nsteps / 2 - 1;
        for (int p = 0; p < nflush; p++) {
            const int arr = p / 3, zp = p - 3 * arr;
            const Step& d = s.steps[6 * arr + (zp == 0 ? 2 : zp + 3)];
            mbar_wait(tfull0, p & 1);
            tmem_fence_after();
            // the step's flush parameters, once, in registers
            const int slot0 = d.slot[0], slot1 = d.slot[1];
            const int smv[2] = {d.sm[0], d.sm[1]}, sn1v[2] = {d.sn1[0], d.sn1[1]}, sn2v[2] = {d.sn2[0], d.sn2[1]};
            const bool same = slot0 == slot1;   // repeated tile indices: the halves meet on one tile
            // element (m, n1, n2) of half h sits in the thread (fr, fk) of consumer warp cw = n1 & 7 as acc[2h+xb][y][z][e]
            // with m = 8 xb + fr, n1 = cw + 8 y, n2 = 8 z + 2 fk + e
            const int npass = same ? 2 : 1;
            for (int pass = 0; pass < npass; pass++) {
                for (int c2 = 0; c2 < 2; c2++) {
                    const int cw = fw + 4 * c2;
#pragma unroll
                    for (int h = 0; h < 2; h++) {
                        if (same && h != pass) continue;
                        double x[16];   // half h of the thread (fr, fk) of consumer warp cw: columns 32 h .. 32 h + 31 of its 64
                        tmem_load16(tlane + c2 * 64 + h * 32, x);
                        if (c2 == 1 && (same ? pass == 1 : h == 1)) {   // last read of the buffer: the consumers may park into it again
                            tmem_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(tfree0);
                        }
                        const uint32_t tile = tiles0 + (uint32_t)(h ? slot1 : slot0) * (TILE * 8);
                        const int sm = smv[h], sn1 = sn1v[h], sn2 = sn2v[h];
                        // address of (m, n1, n2) = base + m sm + n1 sn1 + n2 sn2 + ((m + n1 + n2) & 15): the linear part is split
                        // into a per-thread base and compile-time multiples of the three strides
                        const int lin0 = fr * sm + cw * sn1 + 2 * fk * sn2;
                        const int rot0 = fr + cw + 2 * fk;
#pragma unroll
                        for (int xb = 0; xb < 2; xb++) {
                            uint32_t ad[2][2][2];
                            double old[2][2][2];
#pragma unroll
                            for (int y = 0; y < 2; y++)
#pragma unroll
                                for (int z = 0; z < 2; z++)
#pragma unroll
                                    for (int e = 0; e < 2; e++) {
                                        const int lin = lin0 + 8 * xb * sm + 8 * y * sn1 + (8 * z + e) * sn2;
                                        const int rot = (rot0 + 8 * xb + 8 * y + 8 * z + e) & (T - 1);
                                        ad[y][z][e] = tile + (uint32_t)(lin + rot) * 8;
                                        old[y][z][e] = lds64(ad[y][z][e]);
                                    }
#pragma unroll
                            for (int y = 0; y < 2; y++)
#pragma unroll
                                for (int z = 0; z < 2; z++)
#pragma unroll
                                    for (int e = 0; e < 2; e++) sts64(ad[y][z][e], old[y][z][e] + x[((xb * 2 + y) * 2 + z) * 2 + e]);
                        }
                    }
                }
                // two flusher threads add to the same tile element only from different (step, half) pairs: order them
                flusher_bar();
            }
        }
        tmem_fence_before();
        flusher_bar();
        if (lane == 0) mbar_arrive(smem_u32(&s.tdone));   // before the deallocation: nobody waits for that
        if (warp == 12) {
            mbar_wait(smem_u32(&s.tlast), 0);   // the consumers have read the hole terms of the last step: nobody uses tensor memory any more
            tmem_fence_after();
            tmem_dealloc(tmem_base, TMEM_COLS);
        }
        __syncwarp();
        // ---- the flushers' share of the fused epilogue: la >= EPI_SPLIT of the pairs ft and ft + 128 ----
        const tcw::EpiBC pre0 = tcw::epilogue_prefetch(bv, occ, a, ft), pre1 = tcw::epilogue_prefetch(bv, occ, a, ft + NFLUSH);
        mbar_wait(smem_u32(&s.kready), 0);
        asm volatile("bar.sync 4, %0;" ::"n"(NCONS + NFLUSH) : "memory");   // the consumers have added the last step in
        double sum = tcw::orbit_energy(s.tiles, &s.B[0][0], s.slot_of_perm, bv, a, pre0, ft, EPI_SPLIT, T) +
                     tcw::orbit_energy(s.tiles, &s.B[0][0], s.slot_of_perm, bv, a, pre1, ft + NFLUSH, EPI_SPLIT, T);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
        if (lane == 0) s.red[NCONS_WARPS + fw] = sum;
        asm volatile("bar.sync 3, %0;" ::"n"(NCONS + NFLUSH) : "memory");   // joins the consumers' final reduction
        return;
    }

    if (warp >= NCONS_WARPS) {
        // =========================== producers: four warps, one operand stream each ===========================
        //   stream 0: B columns 0-7 (+ the expect_tx of the whole stage)   stream 1: B columns 8-15
        //   stream 2: A rows 0-15                                          stream 3: A rows 16-31
        // The code is warp-uniform and one elected lane issues.  Registers are allocated per warp: this warpgroup
        // hands its share to the consumers.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const int pw = warp - NCONS_WARPS;
        const bool leader = elect_one();
        if (leader) {   // the descriptors this stream uses: keep their first use off the critical path
            const CUtensorMap* m0 = (pw < 2) ? &mapT2h : &mapT2p;
            asm volatile("prefetch.tensormap [%0];" ::"l"(m0) : "memory");
            if (pw >= 2) asm volatile("prefetch.tensormap [%0];" ::"l"(&mapOvooT) : "memory");
            else asm volatile("prefetch.tensormap [%0];" ::"l"(&mapT2h8) : "memory");
        }
        const uint32_t full0 = smem_u32(&s.full[0]), empty0 = smem_u32(&s.empty[0]);
        const uint32_t dstB = smem_u32(&s.B[0][0]) + pw * B_HALF_BYTES;
        const uint32_t dstA = smem_u32(&s.A[0][0]) + (pw - 2) * A_BOX_BYTES;
        int stage = 0;
        uint32_t wrap = 0;  // how many times the ring has wrapped
        for (int st = 0; st < nsteps; st++) {
            const Step& d = s.steps[st];
            const int n = d.nstages, mode = d.mode;
            const bool particle = d.particle != 0;
            // bytes per stage: plain 2 x 4 KB (B) + 2 x 512 B (A); paired modes 8 KB of B either way and two K chunks of A
            const uint32_t tx = (mode == MODE_PLAIN) ? 2 * B_HALF_BYTES + 2 * A_BOX_BYTES : 2 * B_HALF_BYTES + 4 * A_BOX_BYTES;
            const char* bsrc = (const char*)d.b_src;
            const int V0 = d.V0, U0 = d.U0, c3 = d.b_c3;
            const CUtensorMap* amap = particle ? &mapT2p : &mapOvooT;
            const int a2 = d.a_c2[pw & 1], a3 = d.a_c3[pw & 1], aw = d.W0;
            for (int r = 0; r < n; r++) {
                // every stream waits: a stream that ran ahead by two ring turns would alias the barrier's phase parity
                if (wrap > 0) mbar_wait(empty0 + stage * 8, (wrap - 1) & 1);
                if (leader) {
                    const uint32_t full = full0 + stage * 8;
                    if (pw == 0) mbar_expect_tx(full, tx);
                    if (pw < 2) {
                        const uint32_t dst = dstB + stage * (B_STAGE * 8);   // stage half pw
                        if (mode == MODE_PLAIN) {          // column half z = pw of chunk r
                            if (particle) bulk_load(dst, bsrc + (size_t)r * (B_STAGE * 8) + pw * B_HALF_BYTES, B_HALF_BYTES, full);
                            else tma_load_4d(dst, &mapT2h, V0 + 8 * pw, r * KC, U0, c3, full);
                        } else if (mode == MODE_Z2) {      // column half z = 0 of chunk 2r + pw
                            const int c = 2 * r + pw;
                            if (particle) bulk_load(dst, bsrc + (size_t)c * (B_STAGE * 8), B_HALF_BYTES, full);
                            else tma_load_4d(dst, &mapT2h, V0, c * KC, U0, c3, full);
                        } else {                            // MODE_Y2: rows n1 = 0..7 of column half z = pw, chunks 2r and 2r + 1
#pragma unroll
                            for (int kk = 0; kk < 2; kk++) {
                                const int c = 2 * r + kk;
                                if (particle) bulk_load(dst + kk * (B_HALF_BYTES / 2), bsrc + (size_t)c * (B_STAGE * 8) + pw * B_HALF_BYTES, B_HALF_BYTES / 2, full);
                                else tma_load_4d(dst + kk * (B_HALF_BYTES / 2), &mapT2h8, V0 + 8 * pw, c * KC, U0, c3, full);
                            }
                        }
                    } else {
                        const uint32_t dst = dstA + stage * (A_STAGE * 8);   // rows 16 (pw - 2) ..
                        if (mode == MODE_PLAIN) {
                            tma_load_4d(dst, amap, r * KC, aw, a2, a3, full);
                        } else {
                            tma_load_4d(dst, amap, 2 * r * KC, aw, a2, a3, full);
                            tma_load_4d(dst + (A_STAGE / 2) * 8, amap, (2 * r + 1) * KC, aw, a2, a3, full);
                        }
                    }
                }
                if (++stage == STAGES) {
                    stage = 0;
                    wrap++;
                }
            }
        }
        // ---- the ring is done: once the consumers have released its last chunks, stage the (ov|ov) blocks of the fused
        //      epilogue into it (this overlaps the flushers' tail) ----
        for (int q = 0; q < STAGES; q++) {
            const uint32_t fills = wrap + (q < stage ? 1u : 0u);
            if (fills > 0) mbar_wait(empty0 + q * 8, (fills - 1) & 1);
        }
        tcw::stage_panels(&s.B[0][0], bv, occ, a, tid - NCONS);
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&s.kready));
        return;
    }

    // =========================== consumers: 8 warps, LDS + DMMA only ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
    ConsumerState cs;
    cs.stage = 0;
    cs.parity = 0;
    cs.lane = lane;
    cs.zero = (uint32_t)a.n_trip >> 31;   // 0 (n_trip is positive); a kernel argument, so not foldable
    cs.full0 = opaque(smem_u32(&s.full[0]));
    cs.empty0 = opaque(smem_u32(&s.empty[0]));
    {
        const int fr = lane >> 2, fk = lane & 3;
        cs.bB = opaque(smem_u32(&s.B[0][0]) + ((warp * KC + fk) * 8 + fr) * 8);  // stage layout [z][n1][k][8]
        cs.bA = opaque(smem_u32(&s.A[0][0]) + (fr * KC + fk) * 8);               // A block [m 8][k 4]
    }
    // accumulators: [row block 0..3][n1 index 0..1][column block 0..1][2]
    double acc[4][2][2][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) acc[x][y][z][0] = acc[x][y][z][1] = 0.0;

    const uint32_t tfull0 = opaque(smem_u32(&s.tfull)), tfree0 = opaque(smem_u32(&s.tfree));
    const uint32_t tpark = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(warp >> 2) * 64;
    int nparked = 0;   // particle steps handed to the flushers so far
    for (int st = 0; st < nsteps; st++) {
        const Step& d = s.steps[st];
        const int n6 = st % 6;                       // position in the arrangement: H0 H1 P0 H2 P1 P2
        const bool particle = d.particle != 0;
        if (particle) {
            // ---- start from the hole terms of this particle step's two targets, parked by this thread: rows 0-15 <- term
            //      (z, family 0), rows 16-31 <- term (z, family 1); hole sums enter W with a minus sign (eq. (2)) ----
            //        P0: H0 rows 0-15,  H1 rows 0-15      P1: H0 rows 16-31, H2 rows 0-15      P2: H1 rows 16-31, H2 rows 16-31
            const int z = (n6 == 2) ? 0 : n6 - 3;
            const int b0 = (z == 2) ? 1 : 0, h0 = (z == 0) ? 0 : 1;
            const int b1 = (z == 0) ? 1 : 2, h1 = (z == 2) ? 1 : 0;
            double lo[16], hi[16];
            tmem_wait_st();   // the hole steps' parking stores of this thread
            tmem_load16_neg_pair(tpark + (TB_HOLE + b0) * TBUF_COLS + h0 * 32, tpark + (TB_HOLE + b1) * TBUF_COLS + h1 * 32, lo, hi);
#pragma unroll
            for (int q = 0; q < 16; q++) {
                (&acc[0][0][0][0])[q] = lo[q];
                (&acc[2][0][0][0])[q] = hi[q];
            }
            if (st == nsteps - 1) {   // this warp's last access to tensor memory: the flushers may deallocate it
                tmem_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&s.tlast));
            }
        }
        // dispatch on the mode and the ragged-block counts: the loops inside have compile-time trip counts, so the DMMAs carry
        // no predicates (predicated mma.sync costs a WARPSYNC + NOP each)
        const int n = d.nstages;
        if (d.mode == MODE_PLAIN) {          // ny == nz == 2
            if (d.nxb == 2) run_step<2, 2, 2>(acc, cs, n);
            else run_step<1, 2, 2>(acc, cs, n);
        } else if (d.mode == MODE_Z2) {
            const int code = (d.nxb - 1) * 2 + (d.ny - 1);
            switch (code) {
                case 3: run_step_paired<2, MODE_Z2, 2>(acc, cs, n); break;
                case 2: run_step_paired<2, MODE_Z2, 1>(acc, cs, n); break;
                case 1: run_step_paired<1, MODE_Z2, 2>(acc, cs, n); break;
                default: run_step_paired<1, MODE_Z2, 1>(acc, cs, n); break;
            }
        } else {                              // MODE_Y2: ny == 1, nz == 2
            if (d.nxb == 2) run_step_paired<2, MODE_Y2, 2>(acc, cs, n);
            else run_step_paired<1, MODE_Y2, 2>(acc, cs, n);
        }
        // ---- park the step's accumulators in tensor memory ----
        if (!particle) {
            // a hole step: kept for the two particle steps that start from it (same threads: no hand-over)
            const int y = (n6 < 2) ? n6 : 2;
            tmem_store32(tpark + (TB_HOLE + y) * TBUF_COLS, reinterpret_cast<const double(&)[32]>(acc));
        } else if (st == nsteps - 1) {
            // ---- the unit's last step: nothing is left to multiply, so the consumers add it into the W tiles themselves,
            //      straight from the registers (256 threads, no round trip through tensor memory) ----
            mbar_wait(smem_u32(&s.tdone), 0);   // every earlier step is in the tiles
            const int fr = lane >> 2, fk = lane & 3;
            const uint32_t tiles0 = smem_u32(&s.tiles[0]);
            const bool same = d.slot[0] == d.slot[1];
#pragma unroll
            for (int h = 0; h < 2; h++) {
                if (h == 1 && same) consumer_bar();   // the halves meet on one tile: one after the other
                const uint32_t tile = tiles0 + (uint32_t)d.slot[h] * (TILE * 8);
                const int sm = d.sm[h], sn1 = d.sn1[h], sn2 = d.sn2[h];
                // element acc[2h+xb][y][z][e] = (m, n1, n2) = (8 xb + fr, warp + 8 y, 8 z + 2 fk + e), as in the flushers
                const int lin0 = fr * sm + warp * sn1 + 2 * fk * sn2;
                const int rot0 = fr + warp + 2 * fk;
#pragma unroll
                for (int xb = 0; xb < 2; xb++) {
                    uint32_t ad[2][2][2];
                    double old[2][2][2];
#pragma unroll
                    for (int y = 0; y < 2; y++)
#pragma unroll
                        for (int z = 0; z < 2; z++)
#pragma unroll
                            for (int e = 0; e < 2; e++) {
                                const int lin = lin0 + 8 * xb * sm + 8 * y * sn1 + (8 * z + e) * sn2;
                                const int rot = (rot0 + 8 * xb + 8 * y + 8 * z + e) & (T - 1);
                                ad[y][z][e] = tile + (uint32_t)(lin + rot) * 8;
                                old[y][z][e] = lds64(ad[y][z][e]);
                            }
#pragma unroll
                    for (int y = 0; y < 2; y++)
#pragma unroll
                        for (int z = 0; z < 2; z++)
#pragma unroll
                            for (int e = 0; e < 2; e++) sts64(ad[y][z][e], old[y][z][e] + acc[2 * h + xb][y][z][e]);
                }
            }
        } else {
            // a particle step (hole terms included): the flushers fold it into the W tiles
            if (nparked > 0) mbar_wait(tfree0, (nparked - 1) & 1);   // the flushers have read the previous one
            tmem_fence_after();
            tmem_store32(tpark + TB_PART * TBUF_COLS, reinterpret_cast<const double(&)[32]>(acc));
            tmem_wait_st();
            tmem_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tfull0);
            nparked++;
        }
#pragma unroll
        for (int x = 0; x < 4; x++)
#pragma unroll
            for (int y = 0; y < 2; y++)
#pragma unroll
                for (int z = 0; z < 2; z++) acc[x][y][z][0] = acc[x][y][z][1] = 0.0;
    }
    const tcw::EpiBC pre = tcw::epilogue_prefetch(bv, occ, a, tid);   // in flight across the two waits below
    mbar_wait(smem_u32(&s.kready), 0);  // the epilogue's (ov|ov) blocks are staged
    asm volatile("bar.sync 4, %0;" ::"n"(NCONS + NFLUSH) : "memory");   // every step is in the W tiles (consumers + flushers)

    if (a.W_debug) tcw::dump_W(s.tiles, s.slot_of_perm, bv, v, a.W_debug, tid, NCONS);
    double sum = tcw::orbit_energy(s.tiles, &s.B[0][0], s.slot_of_perm, bv, a, pre, tid, 0, EPI_SPLIT);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
    if (lane == 0) s.red[warp] = sum;
    asm volatile("bar.sync 3, %0;" ::"n"(NCONS + NFLUSH) : "memory");   // consumers + flushers
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < NCONS_WARPS + NFLUSH / 32; w++) tot += s.red[w];
        a.partial[(size_t)rec.row * a.n_orbits + orbit] = tot;
    }
}

}  // namespace


cudaError_t tc_wbuild_make_maps(const tc_wbuild_args& a, int n_tslots, tc_wbuild_maps* out) {
    out->valid = false;
    const cuuint64_t o = a.o, v = a.v, ld = a.ldv, ldo = a.ldo;
    // TMA needs 16-byte aligned bases and strides: the energy calls guarantee it (even row lengths through padded
    // copies, library-built (ov|oo)^T and slices, 16-byte aligned caller pointers)
    if (ld % 2 != 0 || ldo % 2 != 0 || a.t2_row_stride % 2 != 0 || n_tslots < 1) return cudaSuccess;
    if ((((uintptr_t)a.t2) | ((uintptr_t)a.ovooT) | ((uintptr_t)a.slices)) % 16 != 0) return cudaSuccess;
    bool ok = true;
    {   // t2[tslot][l][n1][n2] viewed as dims (n2, l, n1, tslot): hole B, boxes land as [n1][k][8]
        const cuuint64_t dim[4] = {v, o, v, (cuuint64_t)n_tslots};
        const cuuint64_t str[3] = {v * ld, ld, (cuuint64_t)a.t2_row_stride};
        const cuuint32_t box[4] = {8, KC, 16, 1};
        ok = ok && tctma::encode4(&out->T2h, a.t2, dim, str, box);
    }
    {   // the same view with a box of 8 n1 rows (MODE_Y2 hole steps)
        const cuuint64_t dim[4] = {v, o, v, (cuuint64_t)n_tslots};
        const cuuint64_t str[3] = {v * ld, ld, (cuuint64_t)a.t2_row_stride};
        const cuuint32_t box[4] = {8, KC, 8, 1};
        ok = ok && tctma::encode4(&out->T2h8, a.t2, dim, str, box);
    }
    {   // t2[tslot][y][m][d] as dims (d, m, y, tslot): particle A, boxes land as [m][k]
        const cuuint64_t dim[4] = {v, v, o, (cuuint64_t)n_tslots};
        const cuuint64_t str[3] = {ld, v * ld, (cuuint64_t)a.t2_row_stride};
        const cuuint32_t box[4] = {KC, 16, 1, 1};
        ok = ok && tctma::encode4(&out->T2p, a.t2, dim, str, box);
    }
    {   // (ov|oo)^T[z][x][m][l] as dims (l, m, x, z): hole A, boxes land as [m][k]
        const cuuint64_t dim[4] = {o, v, o, o};
        const cuuint64_t str[3] = {ldo, v * ldo, o * v * ldo};
        const cuuint32_t box[4] = {KC, 16, 1, 1};
        ok = ok && tctma::encode4(&out->OvooT, a.ovooT, dim, str, box);
    }
    out->valid = ok;
    return cudaSuccess;
}

int tc_wbuild_tile() { return T; }
int tc_wbuild_num_orbits(int v) {
    const long long nb = (v + T - 1) / T;
    return (int)(nb * (nb + 1) * (nb + 2) / 6);
}
// one slice in the W-builder's layout: [n1 tile][n2 tile][K chunk][z][n1][k][n2 8], zero padded (doubles)
size_t tc_wbuild_slice_doubles(int v) {
    const size_t nb = (size_t)((v + T - 1) / T), nkq = (size_t)tc_tiled_kchunks(v);
    return nb * nb * nkq * B_STAGE;
}

constexpr int kSmemTma = (int)sizeof(Smem);
static_assert(kSmemTma <= 232448, "the unit must fit the 227 KB of opt-in shared memory of one SM");

// per device: called by tc_create with the device current (the attribute is per device, not per process)
cudaError_t tc_wbuild_configure() {
    return cudaFuncSetAttribute(k_wbuild_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTma);
}

cudaError_t tc_launch_wbuild(const tc_wbuild_args& a, const tc_wbuild_maps* maps, const int4* orbits, cudaStream_t stream) {
    if (!maps || !maps->valid) return cudaErrorInvalidValue;   // the energy calls never get here: see tc_wbuild_make_maps
    const long long nblocks = (long long)a.n_trip * a.n_orbits;
    if (nblocks <= 0) return cudaSuccess;
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_wbuild_tma<<<(unsigned)nblocks, NTHREADS, kSmemTma, stream>>>(a, orbits, maps->T2h, maps->T2h8, maps->T2p, maps->OvooT);
    return cudaGetLastError();
}
