// tc_stager.cu -- step a2: integral blocks from DF / Cholesky factors, eq. (6):
//     (pq|rs) = sum_Q B^Q_pq B^Q_rs.
// One FP64 tensor-core GEMM kernel, C = A^T B with both operands K-major (the natural layout of
// B^Q_pq: Q is the slow index), and a two-level output index map so that the three blocks land
// directly in the layouts the W-builder consumes (no transposition pass):
//     vvvo[x][d][b][c] = sum_Q Bvv[Q][d][b] Bov[Q][x][c]      M = v^2, N = nx*v   (the paper's Fig. 2 l.10)
//     ovoo[j][k][l][c] = sum_Q Boo[Q][l][j] Bov[Q][k][c]      M = o^2, N = o*v    (Fig. 2 l.7)
//     ovov[j][k][b][c] = sum_Q Bov[Q][j][b] Bov[Q][k][c]      M = o*v, N = o*v    (Fig. 2 l.16-18)
// CTA tile 128 x 128, K chunk 32, 3-stage cp.async pipeline (198 KB of shared memory), 8 warps (4 x 2), warp tile 32 x 64
// = 4 x 8 DMMA.8x8x4 blocks per k-step (12 fragment loads per 32 MMAs).
#include <algorithm>

#include "tc_common.cuh"

namespace {

constexpr int BM = 128, BN = 128, BK = 32;   // BK 32 measured 4-6 % faster than 16 (half the block-wide syncs per flop)
constexpr int GSTAGES = 3;
constexpr int LDS_ = BM + 4;  // == 4 mod 16: the four k rows of a fragment hit disjoint banks
constexpr int GTHREADS = 256;

struct GemmSmem {
    double A[GSTAGES][BK][LDS_];
    double B[GSTAGES][BK][LDS_];
};

template <int VEC>
__device__ __forceinline__ void gemm_load(double (*dst)[LDS_], const double* src, size_t ld, int col0, int ncols, int k0, int K) {
    constexpr int PIECES = BK * BM / VEC;
#pragma unroll
    for (int p = threadIdx.x; p < PIECES; p += GTHREADS) {
        const int c = (p % (BM / VEC)) * VEC;
        const int kk = p / (BM / VEC);
        int nvalid = ncols - (col0 + c);
        nvalid = (k0 + kk < K) ? (nvalid < 0 ? 0 : (nvalid > VEC ? VEC : nvalid)) : 0;
        const double* s = nvalid ? src + (size_t)(k0 + kk) * ld + col0 + c : src;
        const uint32_t d = smem_u32(&dst[kk][c]);
        if (VEC == 2) cp_async16(d, s, nvalid * 8);
        else cp_async8(d, s, nvalid * 8);
    }
}

// Tile-restricted operand panels (the abcijk schedule): column col of the panel is element (col / 48, tile[(col / 16) % 3] * 16 +
// col % 16) of a [.][v] array, i.e. only the three 16-wide tiles of the second index; elements at or beyond v read as zero.
struct TileSel {
    int t[3];
};
template <int VEC>
__device__ __forceinline__ void gemm_load_tiles(double (*dst)[LDS_], const double* src, size_t ld, int col0, int ncols, int k0, int K,
                                                int v, TileSel ts) {
    constexpr int PIECES = BK * BM / VEC;
#pragma unroll
    for (int p = threadIdx.x; p < PIECES; p += GTHREADS) {
        const int c = (p % (BM / VEC)) * VEC;
        const int kk = p / (BM / VEC);
        const int col = col0 + c;
        const int g = col >> 4, within = col & 15, outer = g / 3, which = g - 3 * outer;
        const int idx = ts.t[which] * 16 + within;
        int nvalid = v - idx;
        nvalid = (k0 + kk < K && col < ncols) ? (nvalid < 0 ? 0 : (nvalid > VEC ? VEC : nvalid)) : 0;
        const double* s = nvalid ? src + (size_t)(k0 + kk) * ld + (size_t)outer * v + idx : src;
        const uint32_t d = smem_u32(&dst[kk][c]);
        if (VEC == 2) cp_async16(d, s, nvalid * 8);
        else cp_async8(d, s, nvalid * 8);
    }
}

// TILED = false: two-level linear output map.  TILED = true: rows are (d, b) = (row / v, row % v), columns (x, c) =
// (col / v, col % v) of slice x, written in the W-builder's tiled layout
//   [n1 tile b/16][n2 tile c/16][K chunk d/4][z = (c%16)/8][n1 = b%16][k = d%4][n2 = c%8]
// (R2 = C2 = v, sr1 = tiles per edge nb, sr2 = K chunks nkq, sc1 = slice stride): a K chunk of a tile pair is then
// 8 KB contiguous, in the fragment order of mma.sync m8n8k4, and the W-builder streams it with plain bulk copies.
// TILED = 2 (abcijk schedule): both operands are tile-restricted panels (TileSel), rows (d, lu, bl), columns (x, lv, cl); the
// output is the same chunk layout over the 3 x 3 local tile pairs: [lu][lv][K chunk][z][n1][k][n2 8] per x (sc1 = stride of x,
// sr2 = K chunks, R2 = v).
template <int VEC, int TILED>
__global__ void __launch_bounds__(GTHREADS, 1)
k_df_gemm(const double* __restrict__ A, size_t lda, const double* __restrict__ B, size_t ldb, int M, int N, int K,
          int R2, long long sr1, long long sr2, int C2, long long sc1, long long sc2, double* __restrict__ C, TileSel ts) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    GemmSmem& s = *reinterpret_cast<GemmSmem*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wm = warp >> 1, wn = warp & 1;  // 4 x 2 warps
    const int fr = lane >> 2, fk = lane & 3;
    const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
    const int nchunks = (K + BK - 1) / BK;

    double acc[4][8][2];
#pragma unroll
    for (int x = 0; x < 4; x++)
#pragma unroll
        for (int y = 0; y < 8; y++) acc[x][y][0] = acc[x][y][1] = 0.0;

    int ld_c = 0;
    auto load_next = [&]() {
        if (ld_c < nchunks) {
            if (TILED == 2) {
                gemm_load_tiles<VEC>(s.A[ld_c % GSTAGES], A, lda, m0, M, ld_c * BK, K, R2, ts);
                gemm_load_tiles<VEC>(s.B[ld_c % GSTAGES], B, ldb, n0, N, ld_c * BK, K, R2, ts);
            } else {
                gemm_load<VEC>(s.A[ld_c % GSTAGES], A, lda, m0, M, ld_c * BK, K);
                gemm_load<VEC>(s.B[ld_c % GSTAGES], B, ldb, n0, N, ld_c * BK, K);
            }
            ld_c++;
        }
        cp_async_commit();
    };
#pragma unroll
    for (int n = 0; n < GSTAGES - 1; n++) load_next();

    for (int c = 0; c < nchunks; c++) {
        cp_async_wait<GSTAGES - 2>();
        __syncthreads();
        load_next();
        const double(*As)[LDS_] = s.A[c % GSTAGES];
        const double(*Bs)[LDS_] = s.B[c % GSTAGES];
#pragma unroll
        for (int ks = 0; ks < BK; ks += 4) {
            double af[4], bf[8];
#pragma unroll
            for (int x = 0; x < 4; x++) af[x] = As[ks + fk][wm * 32 + x * 8 + fr];
#pragma unroll
            for (int y = 0; y < 8; y++) bf[y] = Bs[ks + fk][wn * 64 + y * 8 + fr];
#pragma unroll
            for (int x = 0; x < 4; x++)
#pragma unroll
                for (int y = 0; y < 8; y++) dmma884(acc[x][y][0], acc[x][y][1], af[x], bf[y]);
        }
    }
    cp_async_wait<0>();

    // store through the output index map
#pragma unroll
    for (int x = 0; x < 4; x++) {
        const int row = m0 + wm * 32 + x * 8 + fr;
        if (row >= M) continue;
        long long roff;
        if (TILED == 2) {
            const int d = row / 48, lb = row - d * 48;   // lb = 16 lu + bl
            roff = (((long long)(lb >> 4) * 3) * sr2 + (d >> 2)) * 1024 + (lb & 15) * 32 + (d & 3) * 8;
        } else if (TILED == 1) {
            const int d = row / R2, b = row - d * R2;
            roff = (((long long)(b >> 4) * sr1) * sr2 + (d >> 2)) * 1024 + (b & 15) * 32 + (d & 3) * 8;
        } else {
            roff = (long long)(row / R2) * sr1 + (long long)(row % R2) * sr2;
        }
#pragma unroll
        for (int y = 0; y < 8; y++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int col = n0 + wn * 64 + y * 8 + 2 * fk + e;
                if (col >= N) continue;
                if (TILED == 2) {
                    const int xs = col / 48, lc = col - xs * 48;   // lc = 16 lv + cl
                    C[roff + (long long)xs * sc1 + ((long long)(lc >> 4) * sr2) * 1024 + ((lc >> 3) & 1) * 512 + (lc & 7)] = acc[x][y][e];
                } else if (TILED == 1) {
                    const int xs = col / C2, c = col - xs * C2;
                    C[roff + (long long)xs * sc1 + ((long long)(c >> 4) * sr2) * 1024 + ((c >> 3) & 1) * 512 + (c & 7)] = acc[x][y][e];
                } else {
                    C[roff + (long long)(col / C2) * sc1 + (long long)(col % C2) * sc2] = acc[x][y][e];
                }
            }
    }
}

// materialised src[k][b][c] (K rows, row length ld) -> tiled layout, padding included (one thread per destination element)
__global__ void __launch_bounds__(256) k_tile_slice(const double* __restrict__ src, int K, int v, size_t ld, int nb, int nkq,
                                                    double* __restrict__ dst) {
    const size_t total = (size_t)nb * nb * nkq * 1024;
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < total; n += (size_t)gridDim.x * blockDim.x) {
        const int n2 = (int)(n & 7), k = (int)((n >> 3) & 3), n1 = (int)((n >> 5) & 15), z = (int)((n >> 9) & 1);
        size_t t = n >> 10;
        const int kq = (int)(t % nkq);
        t /= nkq;
        const int V = (int)(t % nb), U = (int)(t / nb);
        const int d = kq * 4 + k, b = U * 16 + n1, c = V * 16 + z * 8 + n2;
        dst[n] = (d < K && b < v && c < v) ? src[((size_t)d * v + b) * ld + c] : 0.0;
    }
}

// ovoo[z][x][l][m] -> dst[z][x][m][ldo] (l fastest, pad zeroed)
__global__ void __launch_bounds__(256) k_transpose_ovoo(const double* __restrict__ src, int o, int v, int ldo, size_t npanels,
                                                        double* __restrict__ dst) {
    const size_t per = (size_t)v * ldo, total = npanels * per;
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < total; n += (size_t)gridDim.x * blockDim.x) {
        const size_t panel = n / per;
        const int r = (int)(n - panel * per);
        const int m = r / ldo, l = r - m * ldo;
        dst[n] = (l < o) ? src[(panel * o + l) * v + m] : 0.0;
    }
}

}  // namespace

// per device: called by tc_create with the device current
cudaError_t tc_stager_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_df_gemm<1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_df_gemm<2, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_df_gemm<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_df_gemm<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_df_gemm<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_df_gemm<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    return e;
}

cudaError_t tc_launch_df_gemm(const double* A, size_t lda, const double* B, size_t ldb, int M, int N, int K,
                              int R2, long long sr1, long long sr2, int C2, long long sc1, long long sc2,
                              double* C, cudaStream_t stream) {
    if (M <= 0 || N <= 0 || K <= 0) return cudaSuccess;
    dim3 grid((N + BN - 1) / BN, (M + BM - 1) / BM);
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    const bool vec2 = (lda % 2 == 0) && (ldb % 2 == 0) && (((uintptr_t)A | (uintptr_t)B) % 16 == 0);
    if (vec2)
        k_df_gemm<2, 0><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(A, lda, B, ldb, M, N, K, R2, sr1, sr2, C2, sc1, sc2, C, TileSel{{0, 0, 0}});
    else
        k_df_gemm<1, 0><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(A, lda, B, ldb, M, N, K, R2, sr1, sr2, C2, sc1, sc2, C, TileSel{{0, 0, 0}});
    return cudaGetLastError();
}

cudaError_t tc_launch_df_slices_tiled(const double* Bvv, const double* Bov, int o, int v, int naux, int x0, int nx, double* dst,
                                      size_t slice_stride, cudaStream_t stream) {
    if (nx <= 0) return cudaSuccess;
    const int M = v * v, N = nx * v;
    const size_t lda = (size_t)v * v, ldb = (size_t)o * v;
    const double* B = Bov + (size_t)x0 * v;
    dim3 grid((N + BN - 1) / BN, (M + BM - 1) / BM);
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    const int nb = (v + 15) / 16, nkq = tc_tiled_kchunks(v);
    const bool vec2 = (lda % 2 == 0) && (ldb % 2 == 0) && (((uintptr_t)Bvv | (uintptr_t)B) % 16 == 0);
    if (vec2)
        k_df_gemm<2, 1><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(Bvv, lda, B, ldb, M, N, naux, v, nb, nkq, v, (long long)slice_stride, 0, dst, TileSel{{0, 0, 0}});
    else
        k_df_gemm<1, 1><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(Bvv, lda, B, ldb, M, N, naux, v, nb, nkq, v, (long long)slice_stride, 0, dst, TileSel{{0, 0, 0}});
    return cudaGetLastError();
}

// abcijk schedule: for every occupied x the part of I_x[d][b][c] = (bd|cx) with b and c in the three tiles (A, B, C) of one tile
// orbit, in the W-builder's chunk layout over the 3 x 3 local tile pairs (x at dst + x * x_stride).  One GEMM:
// M = 48 v rows (d, lu, bl), N = 48 o columns (x, lv, cl), K = naux.  Indices at or beyond v come out as zeros.
cudaError_t tc_launch_df_slices_orbit(const double* Bvv, const double* Bov, int o, int v, int naux, int tA, int tB, int tC, double* dst,
                                      size_t x_stride, cudaStream_t stream) {
    const int M = 48 * v, N = 48 * o;
    const size_t lda = (size_t)v * v, ldb = (size_t)o * v;
    dim3 grid((N + BN - 1) / BN, (M + BM - 1) / BM);
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    const int nkq = tc_tiled_kchunks(v);
    const TileSel ts{{tA, tB, tC}};
    const bool vec2 = (v % 2 == 0) && (((uintptr_t)Bvv | (uintptr_t)Bov) % 16 == 0);
    if (vec2)
        k_df_gemm<2, 2><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(Bvv, lda, Bov, ldb, M, N, naux, v, 0, nkq, v, (long long)x_stride, 0, dst, ts);
    else
        k_df_gemm<1, 2><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(Bvv, lda, Bov, ldb, M, N, naux, v, 0, nkq, v, (long long)x_stride, 0, dst, ts);
    return cudaGetLastError();
}

cudaError_t tc_launch_tile_slice(const double* src, int K, int v, size_t ld, double* dst, cudaStream_t stream) {
    const int nb = (v + 15) / 16, nkq = tc_tiled_kchunks(K);
    const size_t total = (size_t)nb * nb * nkq * 1024;
    const unsigned grid = (unsigned)std::min<size_t>((total + 255) / 256, 148 * 32);
    k_tile_slice<<<grid, 256, 0, stream>>>(src, K, v, ld, nb, nkq, dst);
    return cudaGetLastError();
}

cudaError_t tc_launch_transpose_ovoo(const double* ovoo, int o, int v, int ldo, double* dst, cudaStream_t stream) {
    const size_t npanels = (size_t)o * o, total = npanels * v * ldo;
    const unsigned grid = (unsigned)std::min<size_t>((total + 255) / 256, 148 * 32);
    k_transpose_ovoo<<<grid, 256, 0, stream>>>(ovoo, o, v, ldo, npanels, dst);
    return cudaGetLastError();
}
