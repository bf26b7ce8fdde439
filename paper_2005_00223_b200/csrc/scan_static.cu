// dp_scan_exclusive_static: the two-level exclusive prefix sum of the neighbour-list build (nlist.cu: bin offsets, row offsets)
// as an entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
// serving loops, harnesses that forbid it).  The existing path (dp_launch_scan, reached through dp_scan_exclusive below) takes
// its scratch (tile sums and tile offsets) from the caller's workspace; this variant keeps that scratch in a file-scope device
// array of fixed size, so the caller passes only the input and the output.
//
// Rules of the static scratch (also in include/dp.h):
//   * size: 2 * (DP_SCAN_STATIC_MAX / 4096 + 2) ints = 32,784 bytes; every GPU that loads the library holds it until exit;
//   * n > DP_SCAN_STATIC_MAX is rejected with DP_ENOMEM before anything is launched;
//   * every call shares the array and it keeps the last call's contents.  Nothing in it has to start at zero: every word a
//     kernel of one call reads (sums[0 .. nt), tile_start[0 .. nt]) was written earlier in the same call, by a kernel the
//     stream orders before it; words beyond nt are stale and never read;
//   * calls that overlap on the GPU (different streams, or several host threads on different streams) RACE on the array:
//     serialise them (one stream, or events).  Calls on one stream are ordered and safe;
//   * in host code the array's NAME is a host-side stand-in, not a device address: the device address is taken once per
//     device with cudaGetSymbolAddress, with that device current, and that pointer is what the kernels receive.
// No cudaMalloc, cudaFree or allocating library routine is called here.
#include <atomic>
#include <mutex>
#include "dp_internal.h"

namespace {

constexpr int ST_TILE = 4096;                                    // 1024 threads x 4 elements (as nlist.cu)
constexpr int ST_MAX_TILES = DP_SCAN_STATIC_MAX / ST_TILE;       // 4,096
constexpr int ST_WORDS = 2 * (ST_MAX_TILES + 2);                 // sums[nt + 1] | tile_start[nt + 1], nt <= ST_MAX_TILES
static_assert(DP_SCAN_STATIC_MAX % ST_TILE == 0, "the maximum is a whole number of tiles");

static __device__ __align__(256) int g_scan_scratch[ST_WORDS];

// inclusive scan over the 1024 threads of a block of one value per thread; returns the exclusive prefix of the thread
__device__ __forceinline__ int block_exclusive(int tsum, int *warp_sums, int *block_total) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int x = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        warp_sums[lane] = s;
    }
    __syncthreads();
    if (block_total) *block_total = warp_sums[31];
    return (wid ? warp_sums[wid - 1] : 0) + x - tsum;
}

// step 1: sums[tile] = sum of the tile's elements
__global__ void __launch_bounds__(1024) k_sscan_sums(int n, const int *__restrict__ cnt, int *__restrict__ scratch) {
    __shared__ int ws[32];
    const int i0 = blockIdx.x * ST_TILE + 4 * threadIdx.x;
    int v = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) v += i0 + k < n ? cnt[i0 + k] : 0;
    int total;
    (void)block_exclusive(v, ws, &total);
    if (threadIdx.x == 0) scratch[blockIdx.x] = total;
}

// step 2 (one block): tile_start[0 .. nt] = exclusive scan of sums[0 .. nt)
__global__ void __launch_bounds__(1024) k_sscan_top(int nt, int *__restrict__ scratch) {
    __shared__ int ws[32];
    __shared__ int carry;
    const int *sums = scratch;
    int *tile_start = scratch + nt + 1;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nt; base += ST_TILE) {
        const int i0 = base + 4 * threadIdx.x;
        int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = i0 + k < nt ? sums[i0 + k] : 0;
        int total;
        int prefix = carry + block_exclusive(v[0] + v[1] + v[2] + v[3], ws, &total);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (i0 + k < nt) tile_start[i0 + k] = prefix;
            prefix += v[k];
        }
        __syncthreads();
        if (threadIdx.x == 0) carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) tile_start[nt] = carry;
}

// step 3: every tile scans itself on top of its offset; the last tile writes the total
__global__ void __launch_bounds__(1024) k_sscan_tiles(int n, int nt, const int *__restrict__ cnt, const int *__restrict__ scratch,
                                                       int *__restrict__ start) {
    __shared__ int ws[32];
    const int *tile_start = scratch + nt + 1;
    const int i0 = blockIdx.x * ST_TILE + 4 * threadIdx.x;
    int v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = i0 + k < n ? cnt[i0 + k] : 0;
    int prefix = tile_start[blockIdx.x] + block_exclusive(v[0] + v[1] + v[2] + v[3], ws, nullptr);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (i0 + k < n) start[i0 + k] = prefix;
        prefix += v[k];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) start[n] = tile_start[nt];
}

// device address of the scratch array, per device ordinal, taken once with that device current
constexpr int ST_MAX_DEVICES = 64;
std::mutex st_mutex;
int *st_ptr[ST_MAX_DEVICES] = {nullptr};
std::atomic<bool> st_ready[ST_MAX_DEVICES];

cudaError_t scratch_of_current_device(int **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= ST_MAX_DEVICES) return cudaErrorInvalidDevice;
    if (!st_ready[dev].load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(st_mutex);
        if (!st_ready[dev].load(std::memory_order_relaxed)) {
            int *p = nullptr;
            e = cudaGetSymbolAddress((void **)&p, g_scan_scratch);      // the array's name is NOT a device pointer in host code
            if (e != cudaSuccess) return e;
            if (!p) return cudaErrorInvalidSymbol;
            st_ptr[dev] = p;
            st_ready[dev].store(true, std::memory_order_release);
        }
    }
    *out = st_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int dp_scan_exclusive_static(int n, const int *cnt_dev, int *start_dev, void *cuda_stream) {
    if (n <= 0 || !cnt_dev || !start_dev) return DP_EINVAL;
    if (n > DP_SCAN_STATIC_MAX) return DP_ENOMEM;              // the static scratch holds DP_SCAN_STATIC_MAX / 4096 tiles
    int *scratch = nullptr;
    if (scratch_of_current_device(&scratch) != cudaSuccess) return DP_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nt = (n + ST_TILE - 1) / ST_TILE;
    k_sscan_sums<<<nt, 1024, 0, st>>>(n, cnt_dev, scratch);
    k_sscan_top<<<1, 1024, 0, st>>>(nt, scratch);
    k_sscan_tiles<<<nt, 1024, 0, st>>>(n, nt, cnt_dev, scratch, start_dev);
    return cudaGetLastError() == cudaSuccess ? DP_OK : DP_ECUDA;
}

// the existing path (the scan dp_compute runs, nlist.cu) with caller-owned scratch, exported so that it can be called alone
extern "C" size_t dp_scan_scratch_bytes(int n) {
    return n > 0 ? sizeof(int) * 2 * ((size_t)n / ST_TILE + 2) : 0;
}
extern "C" int dp_scan_exclusive(int n, const int *cnt_dev, int *start_dev, void *scratch_dev, size_t scratch_bytes,
                                 void *cuda_stream) {
    if (n <= 0 || !cnt_dev || !start_dev || !scratch_dev) return DP_EINVAL;
    if (scratch_bytes < dp_scan_scratch_bytes(n)) return DP_ENOMEM;
    dp_launch_scan(n, cnt_dev, start_dev, (int *)scratch_dev, (cudaStream_t)cuda_stream);
    return cudaGetLastError() == cudaSuccess ? DP_OK : DP_ECUDA;
}
