// tc_reduce.cu -- a1 (device side of the scheduler) and a7 (deterministic reductions).
//   per-unit partials -> S_ijk -> E = sum w_ijk S_ijk, all in a fixed summation order so that two
//   runs are bit-identical (the paper keeps a sum_ijk array and applies the Kronecker weights
//   afterwards; same here).
#include <algorithm>

#include "tc_common.cuh"

namespace {

__device__ __forceinline__ long long tet(long long i) { return i * (i + 1) * (i + 2) / 6; }
__device__ __forceinline__ long long tri(long long j) { return j * (j + 1) / 2; }

__global__ void k_make_triplets(int o, long long first, int n, tc_trip_rec* __restrict__ recs, double* __restrict__ w) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const long long idx = first + t;
    long long i = (long long)floor(cbrt(6.0 * (double)idx));
    if (i < 0) i = 0;
    while (tet(i + 1) <= idx) i++;
    while (i > 0 && tet(i) > idx) i--;
    const long long rest = idx - tet(i);
    long long j = (long long)floor((sqrt(8.0 * (double)rest + 1.0) - 1.0) * 0.5);
    if (j < 0) j = 0;
    while (tri(j + 1) <= rest) j++;
    while (j > 0 && tri(j) > rest) j--;
    const long long k = rest - tri(j);
    // everything resident: slice slot = amplitude-row slot = the occupied index itself
    int4* out = reinterpret_cast<int4*>(recs + t);
    out[0] = make_int4((int)i, (int)j, (int)k, t);
    out[1] = make_int4((int)i, (int)j, (int)k, 0);
    out[2] = make_int4((int)i, (int)j, (int)k, 0);
    w[t] = 2.0 - (i == j ? 1.0 : 0.0) - (j == k ? 1.0 : 0.0);  // eq. (1): 2 - d_ij - d_jk
}

// dst[r][c] = src[r][c] for c < v, 0 for v <= c < ldd (zero-padded copy with a 16-byte row stride for TMA)
__global__ void __launch_bounds__(256) k_pad_rows(double* __restrict__ dst, size_t ldd, const double* __restrict__ src, size_t lds,
                                                  size_t nrows, int v) {
    const size_t total = nrows * ldd;
    for (size_t n = (size_t)blockIdx.x * blockDim.x + threadIdx.x; n < total; n += (size_t)gridDim.x * blockDim.x) {
        const size_t r = n / ldd;
        const int c = (int)(n - r * ldd);
        dst[n] = (c < v) ? src[r * lds + c] : 0.0;
    }
}

constexpr int RT = 256;

__device__ __forceinline__ double block_sum_fixed(double x, double* sh) {
    sh[threadIdx.x] = x;
    __syncthreads();
    for (int s = blockDim.x / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    return sh[0];
}

__global__ void __launch_bounds__(RT) k_reduce_units(const double* __restrict__ partial, int n_units, const int* __restrict__ dest,
                                                      double* __restrict__ S) {
    __shared__ double sh[RT];
    const double* p = partial + (size_t)blockIdx.x * n_units;
    double x = 0.0;
    for (int u = threadIdx.x; u < n_units; u += RT) x += p[u];
    x = block_sum_fixed(x, sh);
    if (threadIdx.x == 0) S[dest ? dest[blockIdx.x] : (int)blockIdx.x] = x;
}

__global__ void __launch_bounds__(1024) k_reduce_energy(const double* __restrict__ S, const double* __restrict__ w, long long n,
                                                        double* __restrict__ E) {
    __shared__ double sh[1024];
    double x = 0.0, comp = 0.0;  // Kahan: |E| reaches 1e5..1e11 Eh with BASELINE's generators
    for (long long t = threadIdx.x; t < n; t += 1024) {
        const double y = w[t] * S[t] - comp;
        const double z = x + y;
        comp = (z - x) - y;
        x = z;
    }
    x = block_sum_fixed(x, sh);
    if (threadIdx.x == 0) *E = x;
}

// abcijk schedule: fold one tile orbit's per-triplet partials into S and form the orbit's partial energy
// (partial[t * stride]: the launch's partial sums are [triplet][orbit of the launch])
__global__ void __launch_bounds__(1024) k_accumulate_orbit(const double* __restrict__ partial, int stride, const double* __restrict__ w,
                                                           long long n, int first, double* __restrict__ S, double* __restrict__ E_orbit) {
    __shared__ double sh[1024];
    double x = 0.0, comp = 0.0;
    for (long long t = threadIdx.x; t < n; t += 1024) {
        const double p = partial[t * stride];
        S[t] = first ? p : S[t] + p;
        const double y = w[t] * p - comp;
        const double z = x + y;
        comp = (z - x) - y;
        x = z;
    }
    x = block_sum_fixed(x, sh);
    if (threadIdx.x == 0 && E_orbit) *E_orbit = x;
}

}  // namespace

cudaError_t tc_launch_accumulate_orbit(const double* partial, int stride, const double* w, long long n, int first, double* S,
                                       double* E_orbit, cudaStream_t stream) {
    k_accumulate_orbit<<<1, 1024, 0, stream>>>(partial, stride, w, n, first, S, E_orbit);
    return cudaGetLastError();
}

cudaError_t tc_launch_make_triplets(int o, long long first, int n, tc_trip_rec* recs, double* w, cudaStream_t stream) {
    if (n <= 0) return cudaSuccess;
    k_make_triplets<<<(n + 255) / 256, 256, 0, stream>>>(o, first, n, recs, w);
    return cudaGetLastError();
}

cudaError_t tc_launch_reduce_units(const double* partial, int n_trip, int n_units, const int* dest, double* S, cudaStream_t stream) {
    if (n_trip <= 0) return cudaSuccess;
    k_reduce_units<<<n_trip, RT, 0, stream>>>(partial, n_units, dest, S);
    return cudaGetLastError();
}

cudaError_t tc_launch_reduce_energy(const double* S, const double* w, long long n, double* E, cudaStream_t stream) {
    k_reduce_energy<<<1, 1024, 0, stream>>>(S, w, n, E);
    return cudaGetLastError();
}

cudaError_t tc_launch_pad_rows(double* dst, size_t ldd, const double* src, size_t lds, size_t nrows, int v, cudaStream_t stream) {
    if (nrows == 0) return cudaSuccess;
    const size_t total = nrows * ldd;
    const unsigned grid = (unsigned)std::min<size_t>((total + 255) / 256, 148 * 16);
    k_pad_rows<<<grid, 256, 0, stream>>>(dst, ldd, src, lds, nrows, v);
    return cudaGetLastError();
}
