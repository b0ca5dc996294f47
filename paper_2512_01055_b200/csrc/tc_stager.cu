// tc_stager.cu -- step a2: integral blocks from DF / Cholesky factors, eq. (6):
//     (pq|rs) = sum_Q B^Q_pq B^Q_rs.
// One FP64 tensor-core GEMM kernel, C = A^T B with both operands K-major (the natural layout of
// B^Q_pq: Q is the slow index), and a two-level output index map so that the three blocks land
// directly in the layouts the W-builder consumes (no transposition pass):
//     vvvo[x][d][b][c] = sum_Q Bvv[Q][d][b] Bov[Q][x][c]      M = v^2, N = nx*v   (the paper's Fig. 2 l.10)
//     ovoo[j][k][l][c] = sum_Q Boo[Q][l][j] Bov[Q][k][c]      M = o^2, N = o*v    (Fig. 2 l.7)
//     ovov[j][k][b][c] = sum_Q Bov[Q][j][b] Bov[Q][k][c]      M = o*v, N = o*v    (Fig. 2 l.16-18)
// CTA tile 128 x 128, K chunk 16, 3-stage cp.async pipeline, 8 warps (4 x 2), warp tile 32 x 64
// = 4 x 8 DMMA.8x8x4 blocks per k-step (12 fragment loads per 32 MMAs).
#include "tc_common.cuh"

namespace {

constexpr int BM = 128, BN = 128, BK = 16;
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

template <int VEC>
__global__ void __launch_bounds__(GTHREADS, 1)
k_df_gemm(const double* __restrict__ A, size_t lda, const double* __restrict__ B, size_t ldb, int M, int N, int K,
          int R2, long long sr1, long long sr2, int C2, long long sc1, long long sc2, double* __restrict__ C) {
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
            gemm_load<VEC>(s.A[ld_c % GSTAGES], A, lda, m0, M, ld_c * BK, K);
            gemm_load<VEC>(s.B[ld_c % GSTAGES], B, ldb, n0, N, ld_c * BK, K);
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
        const long long roff = (long long)(row / R2) * sr1 + (long long)(row % R2) * sr2;
#pragma unroll
        for (int y = 0; y < 8; y++)
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int col = n0 + wn * 64 + y * 8 + 2 * fk + e;
                if (col < N) C[roff + (long long)(col / C2) * sc1 + (long long)(col % C2) * sc2] = acc[x][y][e];
            }
    }
}

}  // namespace

// per device: called by tc_create with the device current
cudaError_t tc_stager_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_df_gemm<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_df_gemm<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GemmSmem));
}

cudaError_t tc_launch_df_gemm(const double* A, size_t lda, const double* B, size_t ldb, int M, int N, int K,
                              int R2, long long sr1, long long sr2, int C2, long long sc1, long long sc2,
                              double* C, cudaStream_t stream) {
    if (M <= 0 || N <= 0 || K <= 0) return cudaSuccess;
    dim3 grid((N + BN - 1) / BN, (M + BM - 1) / BM);
    if (grid.y > 65535) return cudaErrorInvalidConfiguration;
    const bool vec2 = (lda % 2 == 0) && (ldb % 2 == 0) && (((uintptr_t)A | (uintptr_t)B) % 16 == 0);
    if (vec2)
        k_df_gemm<2><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(A, lda, B, ldb, M, N, K, R2, sr1, sr2, C2, sc1, sc2, C);
    else
        k_df_gemm<1><<<grid, GTHREADS, sizeof(GemmSmem), stream>>>(A, lda, B, ldb, M, N, K, R2, sr1, sr2, C2, sc1, sc2, C);
    return cudaGetLastError();
}
