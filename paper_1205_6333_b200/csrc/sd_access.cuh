// sd_access.cuh -- the paper's Appendix A on B200:
// minimal O(N^2) memory-access kernels.  N threads (128 per block, as in the paper); thread j
// reads and accumulates N array elements and stores the sum.  Three access patterns
//   linear     k -> k
//   strided    k -> k p mod N                      p = 131 (a prime > 128)
//   unordered  k -> (k p + j M) mod N              M = 32, j = global thread id of the READER
// and the staging schemes of Alg. 3 / Alg. 4 plus the one the product kernels use:
//   naive         every thread loads every element from global memory            (Alg. 3)
//   small-tiling  the first warp of the block copies 32 elements into shared memory, two
//                 __syncthreads per tile                                           (Alg. 4)
//   tiling        the same with the whole block copying 128 elements              (Alg. 4, text)
//   bulk          linear pattern only: 1-D bulk asynchronous copies (TMA engine) into a 4-stage
//                 shared-memory ring with mbarriers, as in sd_pairs_f32.cuh
// In the tiled schemes the element a thread copies is the image of ITS OWN map, exactly as in
// Alg. 4 (for the unordered pattern the tile therefore mixes the offsets of the copying threads).
// The accumulation is "a trivial computation": sum += element (x + y + z + w for
// float4).  With small-integer data every sum is exact, so results are compared bit for bit.
#pragma once
#include "sd_common.cuh"

namespace sd {

enum { ACC_LINEAR = 0, ACC_STRIDED = 1, ACC_UNORDERED = 2 };
enum { ACC_NAIVE = 0, ACC_SMALL_TILING = 1, ACC_TILING = 2, ACC_BULK = 3 };
constexpr int kAccThreads = 128;
constexpr unsigned kAccPrime = 131u;
constexpr unsigned kAccWarp = 32u;

template <int PATTERN>
__device__ __forceinline__ unsigned acc_map(const unsigned k, const unsigned j, const unsigned N) {
    if (PATTERN == ACC_LINEAR) return k;
    if (PATTERN == ACC_STRIDED) return static_cast<unsigned>((static_cast<unsigned long long>(k) * kAccPrime) % N);
    return static_cast<unsigned>((static_cast<unsigned long long>(k) * kAccPrime +
                                  static_cast<unsigned long long>(j) * kAccWarp) % N);
}

__device__ __forceinline__ float acc_value(const float v) { return v; }
__device__ __forceinline__ float acc_value(const float4 v) { return (v.x + v.y) + (v.z + v.w); }

template <typename T, int PATTERN>
__global__ void __launch_bounds__(kAccThreads)
access_naive_kernel(float* __restrict__ out, const T* __restrict__ in, const unsigned N) {
    const unsigned j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    float sum = acc_value(in[j]);
    for (unsigned k = 0; k < N; ++k) sum += acc_value(in[acc_map<PATTERN>(k, j, N)]);
    out[j] = sum;
}

// W = 32: small-tiling, W = 128: tiling.  Threads beyond N keep copying and synchronising.
template <typename T, int PATTERN, int W>
__global__ void __launch_bounds__(kAccThreads)
access_tiled_kernel(float* __restrict__ out, const T* __restrict__ in, const unsigned N) {
    __shared__ T s_data[W];
    const unsigned j = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned n = threadIdx.x;
    float sum = (j < N) ? acc_value(in[j]) : 0.f;
    for (unsigned m = 0; m < N; m += W) {
        if (n < W && m + n < N) s_data[n] = in[acc_map<PATTERN>(m + n, j, N)];
        __syncthreads();
        const unsigned cnt = min(static_cast<unsigned>(W), N - m);
        for (unsigned k = 0; k < cnt; ++k) sum += acc_value(s_data[k]);
        __syncthreads();
    }
    if (j < N) out[j] = sum;
}

// linear pattern through the bulk-copy ring of the product kernels: tiles of 128 elements
template <typename T>
__global__ void __launch_bounds__(kAccThreads)
access_bulk_kernel(float* __restrict__ out, const T* __restrict__ in, const unsigned N) {
    constexpr int W = 128, STAGES = 4, PREFETCH = 2;
    __shared__ __align__(128) T tiles[STAGES][W];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];
    const unsigned j = blockIdx.x * blockDim.x + threadIdx.x;
    const int tid = threadIdx.x, lane = tid & 31;
    const int n_tiles = static_cast<int>((N + W - 1) / W);
    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], kAccThreads / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();
    int pf = 0;
    auto produce = [&]() {
        const int s = pf % STAGES, q = pf / STAGES;
        if (q > 0) mbar_wait(&empty_bar[s], (q - 1) & 1);
        const unsigned cnt = min(static_cast<unsigned>(W), N - static_cast<unsigned>(pf) * W);
        const unsigned bytes = cnt * static_cast<unsigned>(sizeof(T));  // multiple of 16 (host checks)
        mbar_arrive_expect_tx(&full_bar[s], bytes);
        bulk_load(&tiles[s][0], in + static_cast<size_t>(pf) * W, bytes, &full_bar[s]);
        ++pf;
    };
    if (tid == 0)
        for (int q = 0; q < PREFETCH && pf < n_tiles; ++q) produce();
    float sum = (j < N) ? acc_value(in[j]) : 0.f;
    for (int t = 0; t < n_tiles; ++t) {
        if (tid == 0 && pf < n_tiles) produce();
        const int s = t % STAGES;
        mbar_wait(&full_bar[s], (t / STAGES) & 1);
        const unsigned cnt = min(static_cast<unsigned>(W), N - static_cast<unsigned>(t) * W);
        for (unsigned k = 0; k < cnt; ++k) sum += acc_value(tiles[s][k]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);
    }
    if (j < N) out[j] = sum;
}

}  // namespace sd
