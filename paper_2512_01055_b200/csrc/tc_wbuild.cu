// tc_wbuild.cu -- steps a3-a6 of the hot path: the fused W-builder + epilogue, cp.async variant.
// This is the FALLBACK kernel for operands the TMA path cannot address: caller arrays whose base pointers are not
// 16-byte aligned (odd v no longer comes here: the energy calls pad the row length to v + 1 and use TMA).  It is also
// what tc_debug_force_kernel(TC_KERNEL_CPASYNC) selects, so the tests can compare the two kernels on any input.
// The main path is tc_wbuild_tma.cu; both share tc_wbuild_shared.cuh.
//
// One CTA = one work unit = (occupied triplet i>=j>=k) x (S3-orbit of a virtual tile
// triple {A,B,C}, A>=B>=C, tile edge T=16).  The CTA forms the up-to-six permuted
// T^3 tiles of W_ijk (eqs. (2),(5)) in shared memory with FP64
// tensor-core MMAs, then evaluates Y R / D (eqs. (1),(3),(4)) for every point of the
// orbit from shared memory and writes ONE double.  W and Y never touch HBM
// (the paper's PERMUTE kernel, Fig. 3, and the 36 global gathers of its energy
// kernel, Fig. 4, have no counterpart here).
//
// Contraction algebra used:
//   P_{xy,z}[m][n1][n2] =  sum_d t2[x][y][m][d] * vvvo[z][d][n1][n2]        particle, K = v
//                         - sum_l ovoo[z][x][l][m] * t2[y][l][n1][n2]        hole,     K = o
//   adds to W with the virtual index of position(x) = m, position(y) = n1, position(z) = n2,
//   where (x,y,z) is a permutation of the occupied positions (i,j,k) -- the six rows of the
//   table in SURVEY 8(c) step 2.  For a fixed slice z and tile pair (U,V) the families
//   (x,y,z) and (y,x,z) share the B operand vvvo[z][:, U, V] ("slab"), so one slab step
//   stacks them on M: a 32 x 256 x (v + 2o) DMMA GEMM whose two 16-row halves are added into
//   two shared-memory W tiles with the index permutation folded into the store address.
#include "tc_wbuild_shared.cuh"

namespace {

using tcw::T;
using tcw::TILE;
using tcw::c_perm;
using tcw::tile_addr;
constexpr int KC = 4;             // K chunk = one DMMA k-step
constexpr int STAGES = 3;         // cp.async pipeline depth
constexpr int NTHREADS = 256;
constexpr int NWARPS = NTHREADS / 32;
constexpr int SB = T * T + 4;     // doubles per k-row of a staged B chunk; == 4 mod 16 -> conflict-free B fragments
constexpr int A_STAGE = 32 * KC;  // doubles
constexpr int B_STAGE = KC * SB;  // doubles
constexpr int MAX_STEPS = 18;

struct StepDesc {
    // ld = row length of the operands (v, or v + 1 for the padded copies)
    const double* Bp;     // particle B: slice z + U0*ld + V0             (element + k*v*ld + n1*ld + n2)
    const double* Bh[2];  // hole B of half h: t2 row y or x + U0*ld + V0 (element + l*v*ld + n1*ld + n2)
    const double* Ap[2];  // particle A of half h: t2[x][y] (or [y][x]) + W0*ld   (element + m*ld + d)
    const double* Ah[2];  // hole A of half h: ovoo[z][x] (or [z][y]) + W0        (element + l*ld + m)
    int wW, wU, wV;       // valid extents of the m, n1, n2 tiles
    int slot[2];          // shared-memory W tile receiving half h
    int sm[2], sn1[2], sn2[2];  // address strides of m, n1, n2 in that tile (0 for the swizzled last coordinate)
};

struct Smem {
    double tiles[6 * TILE];
    double A[STAGES][A_STAGE];
    double B[STAGES][B_STAGE];
    StepDesc steps[MAX_STEPS];
    double red[NWARPS];
    int slot_of_perm[6];
    int nsteps;
};

// ---- loader: one K chunk of one slab step into a pipeline stage ------------------------------
template <int VEC>  // VEC = 2: 16-byte cp.async (v even), VEC = 1: 8-byte cp.async (any v)
__device__ __forceinline__ void issue_chunk(Smem& s, int stage, const StepDesc& d, int phase, int k0, int o, int v, int ld) {
    const int tid = threadIdx.x;
    const size_t vv = (size_t)v * ld;
    const int klim = (phase == 2) ? v : o;
    const double* Bsrc = (phase == 2) ? d.Bp : d.Bh[phase];
    double* Bs = s.B[stage];
    double* As = s.A[stage];
    // B chunk: KC x T x T doubles
    constexpr int NPIECE_B = KC * T * T / VEC;
#pragma unroll
    for (int p = tid; p < NPIECE_B; p += NTHREADS) {
        const int n2 = (p % (T / VEC)) * VEC;
        const int n1 = (p / (T / VEC)) % T;
        const int kk = p / (T * T / VEC);
        const bool row_ok = (k0 + kk < klim) && (n1 < d.wU);
        int nvalid = d.wV - n2;
        nvalid = row_ok ? (nvalid < 0 ? 0 : (nvalid > VEC ? VEC : nvalid)) : 0;
        const double* src = nvalid ? Bsrc + (size_t)(k0 + kk) * vv + (size_t)n1 * ld + n2 : Bsrc;
        const uint32_t dst = smem_u32(Bs + kk * SB + n1 * T + n2);
        if (VEC == 2) cp_async16(dst, src, nvalid * 8);
        else cp_async8(dst, src, nvalid * 8);
    }
    // A chunk
    if (phase == 2) {
        constexpr int NPIECE_A = 32 * KC / VEC;
        if (tid < NPIECE_A) {
            const int row = tid / (KC / VEC);
            const int kk = (tid % (KC / VEC)) * VEC;
            const int h = row >> 4, m = row & 15;
            int nvalid = v - (k0 + kk);
            nvalid = (m < d.wW) ? (nvalid < 0 ? 0 : (nvalid > VEC ? VEC : nvalid)) : 0;
            const double* src = nvalid ? d.Ap[h] + (size_t)m * ld + k0 + kk : d.Ap[h];
            const uint32_t dst = smem_u32(As + row * KC + kk);
            if (VEC == 2) cp_async16(dst, src, nvalid * 8);
            else cp_async8(dst, src, nvalid * 8);
        }
    } else {
        if (tid < 16 * KC) {
            const int m = tid & 15, kk = tid >> 4;
            const bool ok = (k0 + kk < o) && (m < d.wW);
            const double* src = ok ? d.Ah[phase] + (size_t)(k0 + kk) * ld + m : d.Ah[phase];
            cp_async8(smem_u32(As + (phase * 16 + m) * KC + kk), src, ok ? 8 : 0);
        }
    }
}

// ---- the kernel ----------------------------------------------------------------------------
template <int VEC>
__global__ void __launch_bounds__(NTHREADS, 1) k_wbuild(const tc_wbuild_args a, const int4* __restrict__ orbits) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Smem& s = *reinterpret_cast<Smem*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int o = a.o, v = a.v, ld = a.ldv;

    const int trip = blockIdx.x / a.n_orbits;
    const int orbit = blockIdx.x - trip * a.n_orbits;
    const tc_trip_rec rec = a.recs[trip];
    const int occ[3] = {rec.occ[0], rec.occ[1], rec.occ[2]};
    const int4 ob = orbits[orbit];
    const int bv[3] = {ob.x, ob.y, ob.z};  // tile indices A >= B >= C
    if (occ[0] == occ[1] && occ[1] == occ[2] && !a.W_debug) {
        // weight 2 - d_ij - d_jk = 0 (and S_iii = 0 anyway: R vanishes by symmetry)
        if (tid == 0) a.partial[(size_t)rec.row * a.n_orbits + orbit] = 0.0;
        return;
    }

    // ---- zero the W tiles; thread 0 builds the step program ----
    for (int n = tid; n < 6 * TILE; n += NTHREADS) s.tiles[n] = 0.0;
    if (tid == 0) {
        int sop[6];
        for (int q = 0; q < 6; q++) {
            sop[q] = q;
            for (int q2 = 0; q2 < q; q2++) {
                if (bv[c_perm[q2][0]] == bv[c_perm[q][0]] && bv[c_perm[q2][1]] == bv[c_perm[q][1]] &&
                    bv[c_perm[q2][2]] == bv[c_perm[q][2]]) {
                    sop[q] = q2;
                    break;
                }
            }
            s.slot_of_perm[q] = sop[q];
        }
        int ns = 0;
        const size_t vv = (size_t)v * ld;
        for (int q = 0; q < 6; q++) {
            if (sop[q] != q) continue;  // arrangement already covered
            const int pw = c_perm[q][0], pu = c_perm[q][1], pvv = c_perm[q][2];  // which of (A,B,C) is the m / n1 / n2 tile
            const int W0 = bv[pw] * T, U0 = bv[pu] * T, V0 = bv[pvv] * T;
            for (int zp = 0; zp < 3; zp++) {
                const int xp = (zp == 0) ? 1 : 0;
                const int yp = (zp == 2) ? 1 : 2;
                const int ox = occ[xp], oy = occ[yp], oz = occ[zp];
                StepDesc& d = s.steps[ns++];
                const double* t2x = a.t2 + (size_t)rec.t[xp] * a.t2_row_stride;   // amplitude rows by slot
                const double* t2y = a.t2 + (size_t)rec.t[yp] * a.t2_row_stride;
                d.Bp = a.slices + (size_t)rec.s[zp] * a.slice_stride + (size_t)U0 * ld + V0;
                d.Bh[0] = t2y + (size_t)U0 * ld + V0;
                d.Bh[1] = t2x + (size_t)U0 * ld + V0;
                d.Ap[0] = t2x + (size_t)oy * vv + (size_t)W0 * ld;
                d.Ap[1] = t2y + (size_t)ox * vv + (size_t)W0 * ld;
                d.Ah[0] = a.ovoo + ((size_t)oz * o + ox) * o * ld + W0;
                d.Ah[1] = a.ovoo + ((size_t)oz * o + oy) * o * ld + W0;
                d.wW = min(T, v - W0);
                d.wU = min(T, v - U0);
                d.wV = min(T, v - V0);
                for (int h = 0; h < 2; h++) {
                    // half 0: family (x,y,z): m -> position xp, n1 -> yp, n2 -> zp
                    // half 1: family (y,x,z): m -> position yp, n1 -> xp, n2 -> zp
                    const int pm = h ? yp : xp, pn1 = h ? xp : yp, pn2 = zp;
                    int rho[3];  // which of (A,B,C) sits at each position of the output tile
                    rho[pm] = pw;
                    rho[pn1] = pu;
                    rho[pn2] = pvv;
                    int qq = 0;
                    for (int q3 = 0; q3 < 6; q3++)
                        if (c_perm[q3][0] == rho[0] && c_perm[q3][1] == rho[1] && c_perm[q3][2] == rho[2]) qq = q3;
                    d.slot[h] = sop[qq];
                    const int strides[3] = {T * T, T, 0};
                    d.sm[h] = strides[pm];
                    d.sn1[h] = strides[pn1];
                    d.sn2[h] = strides[pn2];
                }
            }
        }
        s.nsteps = ns;
    }
    __syncthreads();

    const int nsteps = s.nsteps;
    const int nhc = (o + KC - 1) / KC;  // chunks per hole phase
    const int npc = (v + KC - 1) / KC;  // chunks of the particle phase
    const int cps = 2 * nhc + npc;      // chunks per step
    const int total = nsteps * cps;

    // accumulators: [row block 0..3][n1 index 0..1][column block 0..1][2]
    double acc[4][2][2][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) acc[x][y][z][0] = acc[x][y][z][1] = 0.0;

    // loader state (runs STAGES-1 chunks ahead of the consumer)
    int ld_step = 0, ld_r = 0, ld_c = 0;
    auto load_next = [&]() {
        if (ld_c < total) {
            const int phase = (ld_r < nhc) ? 0 : (ld_r < 2 * nhc ? 1 : 2);
            const int k0 = (ld_r - (phase == 0 ? 0 : phase == 1 ? nhc : 2 * nhc)) * KC;
            issue_chunk<VEC>(s, ld_c % STAGES, s.steps[ld_step], phase, k0, o, v, ld);
            ld_c++;
            if (++ld_r == cps) {
                ld_r = 0;
                ld_step++;
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int n = 0; n < STAGES - 1; n++) load_next();

    const int fr = lane >> 2, fk = lane & 3;
    int cs_step = 0, cs_r = 0;
    for (int c = 0; c < total; c++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        load_next();

        const int phase = (cs_r < nhc) ? 0 : (cs_r < 2 * nhc ? 1 : 2);
        if (cs_r == 2 * nhc) {  // the hole sums enter W with a minus sign (eq. (2))
#pragma unroll
            for (int x = 0; x < 4; x++)
#pragma unroll
                for (int y = 0; y < 2; y++)
#pragma unroll
                    for (int z = 0; z < 2; z++) {
                        acc[x][y][z][0] = -acc[x][y][z][0];
                        acc[x][y][z][1] = -acc[x][y][z][1];
                    }
        }
        const double* As = s.A[c % STAGES];
        const double* Bs = s.B[c % STAGES];
        double bf[2][2];
#pragma unroll
        for (int y = 0; y < 2; y++)
#pragma unroll
            for (int z = 0; z < 2; z++) bf[y][z] = Bs[fk * SB + (warp + 8 * y) * T + z * 8 + fr];
        if (phase != 1) {
#pragma unroll
            for (int x = 0; x < 2; x++) {
                const double af = As[(x * 8 + fr) * KC + fk];
#pragma unroll
                for (int y = 0; y < 2; y++)
#pragma unroll
                    for (int z = 0; z < 2; z++) dmma884(acc[x][y][z][0], acc[x][y][z][1], af, bf[y][z]);
            }
        }
        if (phase != 0) {
#pragma unroll
            for (int x = 2; x < 4; x++) {
                const double af = As[(x * 8 + fr) * KC + fk];
#pragma unroll
                for (int y = 0; y < 2; y++)
#pragma unroll
                    for (int z = 0; z < 2; z++) dmma884(acc[x][y][z][0], acc[x][y][z][1], af, bf[y][z]);
            }
        }

        if (++cs_r == cps) {
            // ---- flush: add the two 16-row halves into their W tiles, permutation in the address ----
            const StepDesc& d = s.steps[cs_step];
#pragma unroll
            for (int h = 0; h < 2; h++) {
                double* tile = s.tiles + d.slot[h] * TILE;
                const int sm = d.sm[h], sn1 = d.sn1[h], sn2 = d.sn2[h];
#pragma unroll
                for (int xb = 0; xb < 2; xb++)
#pragma unroll
                    for (int y = 0; y < 2; y++)
#pragma unroll
                        for (int z = 0; z < 2; z++)
#pragma unroll
                            for (int e = 0; e < 2; e++) {
                                const int m = xb * 8 + fr, n1 = warp + 8 * y, n2 = z * 8 + 2 * fk + e;
                                const int addr = m * sm + n1 * sn1 + n2 * sn2 + ((m + n1 + n2) & (T - 1));
                                tile[addr] += acc[2 * h + xb][y][z][e];
                                acc[2 * h + xb][y][z][e] = 0.0;
                            }
                __syncthreads();  // the two halves may hit the same tile (repeated tile index)
            }
            cs_r = 0;
            cs_step++;
        }
    }
    cp_async_wait<0>();
    __syncthreads();

    if (a.W_debug) tcw::dump_W(s.tiles, s.slot_of_perm, bv, v, a.W_debug, tid, NTHREADS);
    double sum = tcw::orbit_energy(s.tiles, s.slot_of_perm, bv, occ, a, tid, NTHREADS);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, off);
    if (lane == 0) s.red[warp] = sum;
    __syncthreads();
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < NWARPS; w++) tot += s.red[w];
        a.partial[(size_t)rec.row * a.n_orbits + orbit] = tot;
    }
}

}  // namespace

cudaError_t tc_wbuild_cpasync_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_wbuild<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_wbuild<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem));
}

cudaError_t tc_launch_wbuild_cpasync(const tc_wbuild_args& a, const int4* orbits, cudaStream_t stream) {
    const long long nblocks = (long long)a.n_trip * a.n_orbits;
    if (nblocks <= 0) return cudaSuccess;
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    // 16-byte cp.async needs 16-byte aligned rows: even row length and strides, 16-byte aligned base pointers
    const bool vec2 = (a.ldv % 2 == 0) && (a.slice_stride % 2 == 0) && (a.t2_row_stride % 2 == 0) &&
                      (((uintptr_t)a.t2 | (uintptr_t)a.ovoo | (uintptr_t)a.slices) % 16 == 0);
    if (vec2) k_wbuild<2><<<(unsigned)nblocks, NTHREADS, sizeof(Smem), stream>>>(a, orbits);
    else k_wbuild<1><<<(unsigned)nblocks, NTHREADS, sizeof(Smem), stream>>>(a, orbits);
    return cudaGetLastError();
}
