// tc_wbuild_tma.cu -- steps a3-a6 of the hot path, main kernel: fused W-builder + epilogue with
// TMA operand staging and a warp-specialised mbarrier pipeline (sm_100a).
//
// One CTA = one work unit = (occupied triplet i>=j>=k) x (S3-orbit of a virtual tile triple
// {A,B,C}, A>=B>=C, tile edge T=16).  The up-to-six permuted T^3 tiles of W_ijk (eqs. (2),(5),
// PAPER.md:42-53) live in shared memory for the whole unit (192 KB); W and Y never touch HBM.
//
// Contraction algebra: for a slice role z and a tile pair (U,V) the
// families (x,y,z) and (y,x,z) share the B operand, so one step is a 32 x 256 x (v + 2o) GEMM
//   P[m][n1][n2] =  sum_d t2[x][y][m][d] * vvvo[z][d][n1][n2]      particle, K = v   (rows 0-15: (x,y), 16-31: (y,x))
//                 - sum_l ovoo[z][x][l][m] * t2[y][l][n1][n2]      hole,     K = o   (one 16-row half per phase)
// whose two 16-row halves are added into two W tiles with the index permutation folded into
// the shared-memory store address (no PERMUTE kernel).
//
// Roles (384 threads, 1 CTA per SM, setmaxnreg 40 / 232):
//   warps 8-11  producers, one operand stream each (B columns 0-7 + expect_tx, B columns 8-15, A half 0, A half 1):
//               per K chunk of 4 each issues one cp.async.bulk.tensor box into a 3-stage ring; the boxes land
//               directly in the fragment order of mma.sync m8n8k4 f64
//                 B stage [z][n1][k][8]  <- box (8 c, 4 d, 16 b) of the slice viewed as dims (c, d, b, slot)
//                 A stage [rowblock][..] <- box (4 d, 16 m) of t2 rows (particle) or (8 m, 4 l) of (ov|oo) (hole)
//   warps 0-7   consumers, warp tile 32 x 32: per chunk  wait full -> 8 conflict-free 256-byte LDS.64 ->
//               16 DMMA.8x8x4 -> release; after a step they add their accumulators into the W tiles
//               under the next step's hole phases (half 1 from its accumulators, half 0 from spare registers),
//               at the end they run the epilogue.
// Ragged tiles are zero-filled by TMA; 8-blocks that are entirely outside v are neither loaded nor multiplied.
// CTA order: tile orbit slow, triplet fast (L2 reuse of the I_i and I_j slabs between concurrent CTAs).
#include <type_traits>

#include "tc_tma.cuh"
#include "tc_wbuild_shared.cuh"

namespace {

using tcw::c_perm;
using tcw::T;
using tcw::TILE;

constexpr int KC = 4;                     // K chunk = one DMMA k-step
constexpr int STAGES = 3;                 // TMA pipeline depth (smem: 192 KB of W tiles leave 27 KB)
constexpr int NCONS_WARPS = 8;
constexpr int NCONS = NCONS_WARPS * 32;   // consumer threads
constexpr int NTHREADS = NCONS + 128;     // + producer warpgroup (one elected lane issues TMA)
constexpr int B_STAGE = 2 * 16 * KC * 8;  // doubles: [z][n1][k][8]
constexpr int A_STAGE = 4 * 32;           // doubles: four 8-row blocks of 32
constexpr int MAX_STEPS = 18;
constexpr uint32_t B_BOX_BYTES = 8 * KC * 16 * 8;  // 4096
constexpr uint32_t AP_BOX_BYTES = KC * 16 * 8;     // 512
constexpr uint32_t AH_BOX_BYTES = 8 * KC * 8;      // 256

struct Step {
    int U0, V0, W0;  // first virtual index of the n1, n2 and m tiles
    int ox, oy, oz;  // occupied indices in the roles x, y, z
    int zslot;       // slot of slice oz in the slice array
    int tsx, tsy;    // slots of the amplitude rows t2[ox], t2[oy]
    int nxb, ny, nz; // 8-blocks with at least one index below v: rows, n1, n2 (1 or 2)
    int slot[2];     // shared-memory W tile receiving half h
    int sm[2], sn1[2], sn2[2];  // address strides of m, n1, n2 in that tile (0 for the rotated last coordinate)
};

struct __align__(128) Smem {
    double tiles[6 * TILE];
    double B[STAGES][B_STAGE];
    double A[STAGES][A_STAGE];
    unsigned long long full[STAGES];
    unsigned long long empty[STAGES];
    Step steps[MAX_STEPS];
    double red[NCONS_WARPS];
    int slot_of_perm[6];
    int nsteps;
};

__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" ::"n"(NCONS) : "memory"); }


struct ConsumerState {
    int stage;        // ring position of the next chunk to consume
    uint32_t parity;  // its full-barrier parity
    int lane;
    int nhc, npc;     // chunks per hole phase / of the particle phase
    uint32_t full0, empty0;  // shared addresses of full[0] / empty[0]
    uint32_t bB, bAp, bAh;   // this thread's fragment addresses in stage 0 (B, particle A, hole A)
    bool skew;               // second warp of its scheduler (warps w and w+4 share one)
    // deferred flush of the previous step's half 1 (rows 16-31): folded into the W tile under the hole phase of
    // half 0, whose chunks carry only half the DMMAs and leave the warp idle most of the time
    bool pend_on;
    uint32_t pend_tile;      // shared address of the target tile
    int pend_sm, pend_sn1, pend_sn2;
    // ... and of its half 0, parked in spare registers (`hold`) and folded in under the hole phase of half 1
    bool pend0_on;
    uint32_t pend0_tile;
    int pend0_sm, pend0_sn1, pend0_sn2;
    int fr, fk, warp;        // place of this thread in the DMMA C fragment / of its warp in the column tile
};

__device__ __forceinline__ void cons_advance(ConsumerState& cs) {
    if (++cs.stage == STAGES) {
        cs.stage = 0;
        cs.parity ^= 1;
    }
}
// every DMMA that reads the stage's fragments has been issued: hand the stage back to the producer
__device__ __forceinline__ void cons_release(const ConsumerState& cs, int stage) {
    __syncwarp();
    if (cs.lane == 0) mbar_arrive(cs.empty0 + stage * 8);
}

// One slab step of the consumer warps: hole phase of half 0, hole phase of half 1, sign flip,
// particle phase.  NXB / NY / NZ = number of 8-blocks of rows / n1 / n2 that reach below v.
// Every chunk is: wait full -> 4-8 LDS.64 -> 8-16 DMMA.8x8x4 -> release.  Nothing cleverer is needed:
// the two warps of a scheduler may be up to STAGES-1 chunks apart in the ring and settle out of
// phase, so one warp's barrier/LDS latency is covered by the other's DMMAs (a bare LDS+DMMA loop of
// this shape measures 99 % of the DMMA peak, with the mbarrier ring and TMA producers 91 %;
// DESIGN.md "what the consumer loop can reach").
template <int NXB, int NY, int NZ>
__device__ __forceinline__ void run_step(double (&acc)[4][2][2][2], double (&hold)[2][2][2][2], ConsumerState& cs) {
    constexpr uint32_t BST = B_STAGE * 8, AST = A_STAGE * 8;  // stage strides in bytes
    // slice Q = (xb, y) of the pending half: the 4 accumulators acc[2+xb][y][z][e] (always full size: blocks a
    // ragged variant skipped are zero)
    auto flush_slice = [&](auto qc) {
        constexpr int Q = decltype(qc)::value;
        constexpr int xb = Q >> 1, y = Q & 1;
        uint32_t ad[2][2];
        double old[2][2];
#pragma unroll
        for (int z = 0; z < 2; z++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int m = xb * 8 + cs.fr, n1 = cs.warp + 8 * y, n2 = z * 8 + 2 * cs.fk + e;
                ad[z][e] = cs.pend_tile + (uint32_t)(m * cs.pend_sm + n1 * cs.pend_sn1 + n2 * cs.pend_sn2 + ((m + n1 + n2) & (T - 1))) * 8;
                old[z][e] = lds64(ad[z][e]);
            }
#pragma unroll
        for (int z = 0; z < 2; z++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                sts64(ad[z][e], old[z][e] + acc[2 + xb][y][z][e]);
                acc[2 + xb][y][z][e] = 0.0;
            }
    };
    auto flush_hold_slice = [&](auto qc) {
        constexpr int Q = decltype(qc)::value;
        constexpr int xb = Q >> 1, y = Q & 1;
#pragma unroll
        for (int z = 0; z < 2; z++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int m = xb * 8 + cs.fr, n1 = cs.warp + 8 * y, n2 = z * 8 + 2 * cs.fk + e;
                const uint32_t ad = cs.pend0_tile + (uint32_t)(m * cs.pend0_sm + n1 * cs.pend0_sn1 + n2 * cs.pend0_sn2 + ((m + n1 + n2) & (T - 1))) * 8;
                sts64(ad, lds64(ad) + hold[xb][y][z][e]);
            }
    };
    auto flush_hold_n = [&](int q) {
        switch (q) {
            case 0: flush_hold_slice(std::integral_constant<int, 0>{}); break;
            case 1: flush_hold_slice(std::integral_constant<int, 1>{}); break;
            case 2: flush_hold_slice(std::integral_constant<int, 2>{}); break;
            default: flush_hold_slice(std::integral_constant<int, 3>{}); break;
        }
    };
    auto flush_slice_n = [&](int q) {
        switch (q) {
            case 0: flush_slice(std::integral_constant<int, 0>{}); break;
            case 1: flush_slice(std::integral_constant<int, 1>{}); break;
            case 2: flush_slice(std::integral_constant<int, 2>{}); break;
            default: flush_slice(std::integral_constant<int, 3>{}); break;
        }
    };
    // ---- hole phases: rows of half h only, K = o ----
#pragma unroll
    for (int h = 0; h < 2; h++) {
        if (h == 1 && cs.pend_on) {   // fewer than four hole chunks: finish the pending half before its rows are reused
            for (int q = cs.nhc; q < 4; q++) flush_slice_n(q);
            cs.pend_on = false;
        }
        for (int r = 0; r < cs.nhc; r++) {
            mbar_wait(cs.full0 + cs.stage * 8, cs.parity);
            const uint32_t pa = cs.bAh + cs.stage * AST + (2 * h) * 256;
            const uint32_t pb = cs.bB + cs.stage * BST;
            double fa[NXB], fb[NY][NZ];
#pragma unroll
            for (int xb = 0; xb < NXB; xb++) fa[xb] = lds64(pa + xb * 256);
#pragma unroll
            for (int y = 0; y < NY; y++)
#pragma unroll
                for (int z = 0; z < NZ; z++) fb[y][z] = lds64(pb + z * 4096 + y * 2048);
#pragma unroll
            for (int xb = 0; xb < NXB; xb++)
#pragma unroll
                for (int y = 0; y < NY; y++)
#pragma unroll
                    for (int z = 0; z < NZ; z++) dmma884(acc[2 * h + xb][y][z][0], acc[2 * h + xb][y][z][1], fa[xb], fb[y][z]);
            cons_release(cs, cs.stage);
            if (h == 0 && cs.pend_on && r < 4) flush_slice_n(r);
            if (h == 1 && cs.pend0_on && r < 4) flush_hold_n(r);
            cons_advance(cs);
        }
    }
    if (cs.pend0_on) {   // fewer than four hole chunks: the rest of the parked half 0
        for (int q = cs.nhc; q < 4; q++) flush_hold_n(q);
        cs.pend0_on = false;
    }
    // the hole sums enter W with a minus sign (eq. (2))
#pragma unroll
    for (int h = 0; h < 2; h++)
#pragma unroll
        for (int xb = 0; xb < NXB; xb++)
#pragma unroll
            for (int y = 0; y < NY; y++)
#pragma unroll
                for (int z = 0; z < NZ; z++) {
                    acc[2 * h + xb][y][z][0] = -acc[2 * h + xb][y][z][0];
                    acc[2 * h + xb][y][z][1] = -acc[2 * h + xb][y][z][1];
                }

    // ---- particle phase: both halves, K = v ----
    if (cs.skew) {
        // The two warps of a scheduler leave the flush barrier in lockstep and need some ten chunks to
        // drift out of phase (in phase, their barrier/LDS latencies coincide and the tensor pipe idles).
        // Starting the second one a quarter chunk late gets there at once (+0.7 % on cfg1).
        const long long t0 = clock64();
        while (clock64() - t0 < 150) {}
    }
    for (int r = 0; r < cs.npc; r++) {
        mbar_wait(cs.full0 + cs.stage * 8, cs.parity);
        const uint32_t pa = cs.bAp + cs.stage * AST;
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
        // every DMMA that reads this chunk's fragments has been issued (operands are read at issue)
        cons_release(cs, cs.stage);
        cons_advance(cs);
    }
}

// ---- the kernel ------------------------------------------------------------------------------
__global__ void __launch_bounds__(NTHREADS, 1)
k_wbuild_tma(const tc_wbuild_args a, const int4* __restrict__ orbits, const __grid_constant__ CUtensorMap mapI,
             const __grid_constant__ CUtensorMap mapT2h, const __grid_constant__ CUtensorMap mapT2p,
             const __grid_constant__ CUtensorMap mapOvoo) {
    extern __shared__ unsigned char smem_raw[];
    Smem& s = *reinterpret_cast<Smem*>(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int o = a.o, v = a.v;

    // CTA order: tile orbit slow, triplet fast.  CTAs that run together then work on the same orbit for
    // consecutive triplets (i, j, k), (i, j, k+1), ...: they walk the same step sequence and share the slabs of
    // the slices I_i and I_j (12 of a unit's 18 slabs) in L2; with the triplet slow and the orbit fast,
    // neighbours share two tiles and hence only 6 of 18.
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

    // ---- the step program: thread (q, zp) writes the step of arrangement q with slice role zp ----
    if (tid < 18) {
        int sop[6];
        tcw::arrangement_slots(bv, sop);
        const int q = tid / 3, zp = tid - 3 * q;
        int before = 0, distinct = 0;
#pragma unroll
        for (int q2 = 0; q2 < 6; q2++) {
            if (sop[q2] == q2) {
                distinct++;
                if (q2 < q) before++;
            }
        }
        if (tid == 0) {
            s.nsteps = 3 * distinct;
#pragma unroll
            for (int q2 = 0; q2 < 6; q2++) s.slot_of_perm[q2] = sop[q2];
        }
        if (sop[q] == q) {
            const int pw = c_perm[q][0], pu = c_perm[q][1], pvv = c_perm[q][2];  // which of (A,B,C) is the m / n1 / n2 tile
            const int xp = (zp == 0) ? 1 : 0;
            const int yp = (zp == 2) ? 1 : 2;
            Step& d = s.steps[3 * before + zp];
            d.W0 = bv[pw] * T;
            d.U0 = bv[pu] * T;
            d.V0 = bv[pvv] * T;
            d.ox = occ[xp];
            d.oy = occ[yp];
            d.oz = occ[zp];
            d.zslot = rec.s[zp];
            d.tsx = rec.t[xp];
            d.tsy = rec.t[yp];
            d.nxb = (v - d.W0 > 8) ? 2 : 1;
            d.ny = (v - d.U0 > 8) ? 2 : 1;
            d.nz = (v - d.V0 > 8) ? 2 : 1;
#pragma unroll
            for (int h = 0; h < 2; h++) {
                // half 0: family (x,y,z): m -> position xp, n1 -> yp, n2 -> zp
                // half 1: family (y,x,z): m -> position yp, n1 -> xp, n2 -> zp
                const int pm = h ? yp : xp, pn1 = h ? xp : yp, pn2 = zp;
                int qq = 0;
#pragma unroll
                for (int q3 = 0; q3 < 6; q3++)
                    if (c_perm[q3][pm] == pw && c_perm[q3][pn1] == pu && c_perm[q3][pn2] == pvv) qq = q3;
                d.slot[h] = sop[qq];
                d.sm[h] = (pm == 0) ? T * T : (pm == 1 ? T : 0);
                d.sn1[h] = (pn1 == 0) ? T * T : (pn1 == 1 ? T : 0);
                d.sn2[h] = (pn2 == 0) ? T * T : (pn2 == 1 ? T : 0);
            }
        }
    }
    if (tid == 0) {
        for (int n = 0; n < STAGES; n++) {
            mbar_init(smem_u32(&s.full[n]), 1);
            mbar_init(smem_u32(&s.empty[n]), NCONS_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nsteps = s.nsteps;
    const int nhc = (o + KC - 1) / KC;  // chunks per hole phase
    const int npc = (v + KC - 1) / KC;  // chunks of the particle phase
    const int cps = 2 * nhc + npc;      // chunks per step

    if (warp >= NCONS_WARPS) {
        // =========================== producers: four warps, one operand stream each ===========================
        //   stream 0: B columns 0-7 (+ the expect_tx of the whole stage)   stream 1: B columns 8-15
        //   stream 2: A rows of half 0 (particle) / row block 0 (hole)      stream 3: A half 1 / row block 1
        // Splitting the issue work keeps the per-chunk instruction path of each producer short
        // (one wait, one UTMALDG); the code is warp-uniform and one elected lane issues.
        // Registers are allocated per scheduler partition: this warpgroup hands its share to the
        // consumers (168 -> 40 / 232 per thread).
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        const int pw = warp - NCONS_WARPS;
        const bool leader = elect_one();
        if (leader) {   // the descriptors this stream uses: keep their first use off the critical path
            const CUtensorMap* m0 = (pw < 2) ? &mapI : &mapT2p;
            const CUtensorMap* m1 = (pw < 2) ? &mapT2h : &mapOvoo;
            asm volatile("prefetch.tensormap [%0];" ::"l"(m0) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(m1) : "memory");
        }
        const uint32_t full0 = smem_u32(&s.full[0]), empty0 = smem_u32(&s.empty[0]);
        const uint32_t B0 = smem_u32(&s.B[0][0]), A0 = smem_u32(&s.A[0][0]);
        // A segment = one phase of one step as seen by this stream: n chunks along one K coordinate.
        struct Seg {
            const CUtensorMap* map;    // staging box (KC along K)
            int kdim, c0, c1, c2, c3, n;
            uint32_t dst0, dst_stride, tx;
            bool active;
        };
        auto get_seg = [&](int seg_i, Seg& g) {
            const int st = seg_i / 3, ph = seg_i - 3 * st;
            const Step& d = s.steps[st];
            if (ph < 2) {  // hole phase of half ph: B = t2[y or x][l][n1][n2], A = ovoo[z][x or y][l][m]
                const int yy = ph ? d.tsx : d.tsy, xx = ph ? d.oy : d.ox;   // B: amplitude row of y (by slot), A: (ov|oo) of x
                g.n = nhc;
                g.kdim = 1;
                g.tx = d.nz * B_BOX_BYTES + d.nxb * AH_BOX_BYTES;
                if (pw < 2) {
                    g.map = &mapT2h;
                    g.c0 = d.V0 + 8 * pw; g.c1 = 0; g.c2 = d.U0; g.c3 = yy;
                    g.dst0 = B0 + pw * B_BOX_BYTES; g.dst_stride = B_STAGE * 8;
                    g.active = pw < d.nz;
                } else {
                    g.map = &mapOvoo;
                    g.c0 = d.W0 + 8 * (pw - 2); g.c1 = 0; g.c2 = xx; g.c3 = d.oz;
                    g.dst0 = A0 + (2 * ph + pw - 2) * AH_BOX_BYTES; g.dst_stride = A_STAGE * 8;
                    g.active = pw - 2 < d.nxb;
                }
            } else {  // particle phase: B = vvvo[z][d][n1][n2], A = t2[x][y][m][d] (rows 0-15), t2[y][x][m][d] (rows 16-31)
                g.n = npc;
                g.tx = d.nz * B_BOX_BYTES + 2 * AP_BOX_BYTES;
                if (pw < 2) {
                    g.map = &mapI;
                    g.kdim = 1;
                    g.c0 = d.V0 + 8 * pw; g.c1 = 0; g.c2 = d.U0; g.c3 = d.zslot;
                    g.dst0 = B0 + pw * B_BOX_BYTES; g.dst_stride = B_STAGE * 8;
                    g.active = pw < d.nz;
                } else {
                    g.map = &mapT2p;
                    g.kdim = 0;
                    g.c0 = 0; g.c1 = d.W0; g.c2 = (pw == 2) ? d.oy : d.ox; g.c3 = (pw == 2) ? d.tsx : d.tsy;
                    g.dst0 = A0 + (pw - 2) * AP_BOX_BYTES; g.dst_stride = A_STAGE * 8;
                    g.active = true;
                }
            }
        };
        const int nseg = 3 * nsteps;
        int stage = 0;
        uint32_t wrap = 0;  // how many times the ring has wrapped
        for (int seg_i = 0; seg_i < nseg; seg_i++) {
            Seg g;
            get_seg(seg_i, g);
            for (int r = 0; r < g.n; r++) {
                // every stream waits, active or not: a stream that ran ahead by two ring turns would
                // alias the barrier's phase parity
                if (wrap > 0) mbar_wait(empty0 + stage * 8, (wrap - 1) & 1);
                if (leader) {
                    const uint32_t full = full0 + stage * 8;
                    if (pw == 0) mbar_expect_tx(full, g.tx);
                    if (g.active) tma_load_4d(g.dst0 + stage * g.dst_stride, g.map, g.kdim == 0 ? r * KC : g.c0, g.kdim == 1 ? r * KC : g.c1, g.c2, g.c3, full);
                }
                if (++stage == STAGES) {
                    stage = 0;
                    wrap++;
                }
            }
        }
        return;
    }

    // =========================== consumers: 8 warps, LDS + DMMA only ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    // zero the W tiles (overlaps the first TMA round trips)
    for (int n = tid; n < 6 * TILE; n += NCONS) s.tiles[n] = 0.0;

    ConsumerState cs;
    cs.stage = 0;
    cs.parity = 0;
    cs.lane = lane;
    cs.skew = (warp & 4) != 0;
    cs.pend_on = false;
    cs.pend0_on = false;
    cs.fr = lane >> 2;
    cs.fk = lane & 3;
    cs.warp = warp;
    cs.nhc = nhc;
    cs.npc = npc;
    cs.full0 = opaque(smem_u32(&s.full[0]));
    cs.empty0 = opaque(smem_u32(&s.empty[0]));
    {
        const int fr = lane >> 2, fk = lane & 3;
        cs.bB = opaque(smem_u32(&s.B[0][0]) + ((warp * KC + fk) * 8 + fr) * 8);  // stage layout [z][n1][k][8]
        cs.bAp = opaque(smem_u32(&s.A[0][0]) + (fr * KC + fk) * 8);              // particle A block [m 8][k 4]
        cs.bAh = opaque(smem_u32(&s.A[0][0]) + (fk * 8 + fr) * 8);               // hole A block     [k 4][m 8]
    }

    // accumulators: [row block 0..3][n1 index 0..1][column block 0..1][2]
    double acc[4][2][2][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) acc[x][y][z][0] = acc[x][y][z][1] = 0.0;

    const int fr = lane >> 2, fk = lane & 3;   // this thread's place in the DMMA C fragment
    const uint32_t tiles0 = opaque(smem_u32(&s.tiles[0]));
    double hold[2][2][2][2];   // half 0 of the previous step while it waits for the hole phase of half 1
    for (int st = 0; st < nsteps; st++) {
        const Step& d = s.steps[st];
        // dispatch on the ragged-block counts: the loops inside have compile-time trip counts, so
        // the DMMAs carry no predicates (predicated mma.sync costs a WARPSYNC + NOP each)
        const int code = (d.nxb - 1) * 4 + (d.ny - 1) * 2 + (d.nz - 1);
        switch (code) {
            case 7: run_step<2, 2, 2>(acc, hold, cs); break;
            case 6: run_step<2, 2, 1>(acc, hold, cs); break;
            case 5: run_step<2, 1, 2>(acc, hold, cs); break;
            case 4: run_step<2, 1, 1>(acc, hold, cs); break;
            case 3: run_step<1, 2, 2>(acc, hold, cs); break;
            case 2: run_step<1, 2, 1>(acc, hold, cs); break;
            case 1: run_step<1, 1, 2>(acc, hold, cs); break;
            default: run_step<1, 1, 1>(acc, hold, cs); break;
        }
        // ---- flush: add the two 16-row halves into their W tiles, permutation in the address ----
        // (explicit 32-bit shared addresses; per row block 16 loads in flight, then 16 adds and stores)
        // Half 1 can wait: the next step's first phase (hole, half 0) touches rows 0-15 only, so rows 16-31 are
        // folded into their tile under it, four accumulators per hole chunk (see run_step).  Not when the two halves
        // share a tile (they need the barrier between them) and not for very short steps (ring-ordering argument).
        // The ring-ordering argument needs cps >= nhc + 2*4 (the pending halves are folded in under the first four
        // chunks of each hole phase and must be done before a warp can be STAGES chunks ahead): cps = 2 nhc + npc >= 16
        // gives it for every o (npc >= 16 - 2 nhc  =>  cps - nhc - 8 = nhc + npc - 8 >= 0 when cps >= 16, nhc >= 1).
        static_assert(STAGES == 3, "the defer threshold below (cps >= 16) was derived for a 3-stage ring and a 4-chunk flush window");
        const bool defer = (cps >= 16) && (d.slot[0] != d.slot[1]);
        if (defer) {   // park half 0 in spare registers: nothing of the flush is left on the critical path
#pragma unroll
            for (int xb = 0; xb < 2; xb++)
#pragma unroll
                for (int y = 0; y < 2; y++)
#pragma unroll
                    for (int z = 0; z < 2; z++)
#pragma unroll
                        for (int e = 0; e < 2; e++) {
                            hold[xb][y][z][e] = acc[xb][y][z][e];
                            acc[xb][y][z][e] = 0.0;
                        }
            cs.pend0_on = true;
            cs.pend0_tile = tiles0 + (uint32_t)d.slot[0] * (TILE * 8);
            cs.pend0_sm = d.sm[0];
            cs.pend0_sn1 = d.sn1[0];
            cs.pend0_sn2 = d.sn2[0];
        }
#pragma unroll
        for (int h = 0; h < 2; h++) {
            if (h == 0 && defer) continue;
            if (h == 1 && defer) {
                cs.pend_on = true;
                cs.pend_tile = tiles0 + (uint32_t)d.slot[1] * (TILE * 8);
                cs.pend_sm = d.sm[1];
                cs.pend_sn1 = d.sn1[1];
                cs.pend_sn2 = d.sn2[1];
                break;
            }
            // Two threads add to the same tile element only from different (step, half) pairs.  Different
            // steps are ordered by the ring: a warp cannot pass chunk c+STAGES before every warp has released
            // chunk c, and a warp releases a step's chunks before it flushes the next step, so with at least
            // STAGES+1 chunks per step the adds of step s happen-before those of step s+1 (through the
            // empty/full barriers) without any CTA barrier -- the warps keep their phase offsets across steps.
            // The two halves of one step meet on a tile only when tile indices repeat.
            if (cps <= STAGES || (h == 1 && d.slot[0] == d.slot[1])) consumer_bar();
            const uint32_t tile = tiles0 + (uint32_t)d.slot[h] * (TILE * 8);
            const int sm = d.sm[h], sn1 = d.sn1[h], sn2 = d.sn2[h];
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
                            const int m = xb * 8 + fr, n1 = warp + 8 * y, n2 = z * 8 + 2 * fk + e;
                            ad[y][z][e] = tile + (uint32_t)(m * sm + n1 * sn1 + n2 * sn2 + ((m + n1 + n2) & (T - 1))) * 8;
                            old[y][z][e] = lds64(ad[y][z][e]);
                        }
#pragma unroll
                for (int y = 0; y < 2; y++)
#pragma unroll
                    for (int z = 0; z < 2; z++)
#pragma unroll
                        for (int e = 0; e < 2; e++) {
                            sts64(ad[y][z][e], old[y][z][e] + acc[2 * h + xb][y][z][e]);
                            acc[2 * h + xb][y][z][e] = 0.0;
                        }
            }
        }
    }
    if (cs.pend0_on) {   // the last step's half 0
#pragma unroll
        for (int xb = 0; xb < 2; xb++)
#pragma unroll
            for (int y = 0; y < 2; y++)
#pragma unroll
                for (int z = 0; z < 2; z++)
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        const int m = xb * 8 + fr, n1 = warp + 8 * y, n2 = z * 8 + 2 * fk + e;
                        const uint32_t ad = cs.pend0_tile + (uint32_t)(m * cs.pend0_sm + n1 * cs.pend0_sn1 + n2 * cs.pend0_sn2 + ((m + n1 + n2) & (T - 1))) * 8;
                        sts64(ad, lds64(ad) + hold[xb][y][z][e]);
                    }
    }
    if (cs.pend_on) {   // the last step's half 1
        for (int q = 0; q < 4; q++) {
            const int xb = q >> 1, y = q & 1;
#pragma unroll
            for (int z = 0; z < 2; z++)
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int m = xb * 8 + fr, n1 = warp + 8 * y, n2 = z * 8 + 2 * fk + e;
                    const uint32_t ad = cs.pend_tile + (uint32_t)(m * cs.pend_sm + n1 * cs.pend_sn1 + n2 * cs.pend_sn2 + ((m + n1 + n2) & (T - 1))) * 8;
                    double x = 0.0;
#pragma unroll
                    for (int qq = 0; qq < 4; qq++)
                        if (qq == q) x = acc[2 + (qq >> 1)][qq & 1][z][e];
                    sts64(ad, lds64(ad) + x);
                }
        }
    }
    consumer_bar();

    if (a.W_debug) tcw::dump_W(s.tiles, s.slot_of_perm, bv, v, a.W_debug, tid, NCONS);
    double sum = tcw::orbit_energy(s.tiles, s.slot_of_perm, bv, occ, a, tid, NCONS);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
    if (lane == 0) s.red[warp] = sum;
    consumer_bar();
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < NCONS_WARPS; w++) tot += s.red[w];
        a.partial[(size_t)rec.row * a.n_orbits + orbit] = tot;
    }
}

}  // namespace

cudaError_t tc_wbuild_make_maps(const tc_wbuild_args& a, int nslots, int n_tslots, tc_wbuild_maps* out) {
    out->valid = false;
    const cuuint64_t o = a.o, v = a.v, ld = a.ldv;
    // TMA needs 16-byte aligned bases and strides.  Odd v never gets here unpadded: the energy calls pass zero-padded
    // copies with ldv = v + 1, so only caller pointers that are not 16-byte aligned take the cp.async kernel.
    if (ld % 2 != 0 || a.slice_stride % 2 != 0 || a.t2_row_stride % 2 != 0 || nslots < 1 || n_tslots < 1) return cudaSuccess;
    if ((((uintptr_t)a.t2) | ((uintptr_t)a.ovoo) | ((uintptr_t)a.slices)) % 16 != 0) return cudaSuccess;
    bool ok = true;
    {   // slices [slot][d][b][c] viewed as dims (c, d, b, slot)
        const cuuint64_t dim[4] = {v, v, v, (cuuint64_t)nslots};
        const cuuint64_t str[3] = {v * ld, ld, (cuuint64_t)a.slice_stride};
        const cuuint32_t box[4] = {8, KC, 16, 1};
        ok = ok && tctma::encode4(&out->I, a.slices, dim, str, box);
    }
    {   // t2[tslot][l][n1][n2] viewed as dims (n2, l, n1, tslot)
        const cuuint64_t dim[4] = {v, o, v, (cuuint64_t)n_tslots};
        const cuuint64_t str[3] = {v * ld, ld, (cuuint64_t)a.t2_row_stride};
        const cuuint32_t box[4] = {8, KC, 16, 1};
        ok = ok && tctma::encode4(&out->T2h, a.t2, dim, str, box);
    }
    {   // t2[tslot][y][m][d] as dims (d, m, y, tslot)
        const cuuint64_t dim[4] = {v, v, o, (cuuint64_t)n_tslots};
        const cuuint64_t str[3] = {ld, v * ld, (cuuint64_t)a.t2_row_stride};
        const cuuint32_t box[4] = {KC, 16, 1, 1};
        ok = ok && tctma::encode4(&out->T2p, a.t2, dim, str, box);
    }
    {   // ovoo[z][x][l][m] as dims (m, l, x, z)
        const cuuint64_t dim[4] = {v, o, o, o};
        const cuuint64_t str[3] = {ld, o * ld, o * o * ld};
        const cuuint32_t box[4] = {8, KC, 1, 1};
        ok = ok && tctma::encode4(&out->Ovoo, a.ovoo, dim, str, box);
    }
    out->valid = ok;
    return cudaSuccess;
}

int tc_wbuild_tile() { return T; }
int tc_wbuild_num_orbits(int v) {
    const long long nb = (v + T - 1) / T;
    return (int)(nb * (nb + 1) * (nb + 2) / 6);
}

constexpr int kSmemTma = (int)sizeof(Smem) + 128;

// per device: called by tc_create with the device current (the attribute is per device, not per process)
cudaError_t tc_wbuild_configure() {
    return cudaFuncSetAttribute(k_wbuild_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemTma);
}

cudaError_t tc_launch_wbuild(const tc_wbuild_args& a, const tc_wbuild_maps* maps, const int4* orbits, cudaStream_t stream,
                             int* kernel_out) {
    if (!maps || !maps->valid) {
        if (kernel_out) *kernel_out = TC_KERNEL_CPASYNC;
        return tc_launch_wbuild_cpasync(a, orbits, stream);
    }
    if (kernel_out) *kernel_out = TC_KERNEL_TMA;
    const long long nblocks = (long long)a.n_trip * a.n_orbits;
    if (nblocks <= 0) return cudaSuccess;
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    k_wbuild_tma<<<(unsigned)nblocks, NTHREADS, kSmemTma, stream>>>(a, orbits, maps->I, maps->T2h, maps->T2p, maps->Ovoo);
    return cudaGetLastError();
}
