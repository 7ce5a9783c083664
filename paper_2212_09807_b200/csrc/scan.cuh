// Device-wide exclusive prefix sum with an input transform (three launches: block sums, scan of the
// sums in one block, final scan; one launch of one block up to 32 768 elements).  Used for the pre-sizing offsets of S3, the tile / pair /
// active-pixel compaction and the hit compaction of S6.  Accumulates in 64-bit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

extern long long g_lartpc_launches;

namespace lscan {

constexpr int THREADS = 256;
constexpr int ITEMS = 8;
constexpr int TILE = THREADS * ITEMS;

__device__ __forceinline__ long long warp_incl_scan(long long v, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        long long o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// exclusive scan of one value per thread over the block; returns the exclusive prefix, *total = block sum
__device__ __forceinline__ long long block_excl_scan(long long v, long long *total)
{
    __shared__ long long wsum[THREADS / 32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    long long inc = warp_incl_scan(v, lane);
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        long long s = lane < THREADS / 32 ? wsum[lane] : 0;
        long long si = warp_incl_scan(s, lane);
        if (lane < THREADS / 32) wsum[lane] = si - s;
    }
    __syncthreads();
    long long off = wsum[w];
    // total = exclusive prefix of last warp + its sum
    __shared__ long long s_total;
    if (threadIdx.x == THREADS - 1) s_total = off + inc;
    __syncthreads();
    *total = s_total;
    long long r = off + inc - v;
    __syncthreads();
    return r;
}

template <typename F>
__global__ void block_sums_kernel(int64_t n, F f, long long *sums)
{
    int64_t base = (int64_t)blockIdx.x * TILE;
    long long v = 0;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        int64_t i = base + (int64_t)threadIdx.x * ITEMS + k;
        if (i < n) v += (long long)f(i);
    }
    long long total;
    block_excl_scan(v, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// single block: exclusive scan of sums[0..m) in place; writes the grand total to *total
static __global__ void scan_sums_kernel(long long *sums, int64_t m, long long *total)
{
    long long carry = 0;
    for (int64_t base = 0; base < m; base += THREADS) {
        int64_t i = base + threadIdx.x;
        long long v = i < m ? sums[i] : 0;
        long long tot;
        long long ex = block_excl_scan(v, &tot);
        if (i < m) sums[i] = carry + ex;
        carry += tot;
    }
    if (threadIdx.x == 0 && total) *total = carry;
}

template <typename F, typename Out>
__global__ void final_scan_kernel(int64_t n, F f, const long long *sums, Out *out, bool write_last)
{
    int64_t base = (int64_t)blockIdx.x * TILE;
    long long vals[ITEMS];
    long long v = 0;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        int64_t i = base + (int64_t)threadIdx.x * ITEMS + k;
        vals[k] = i < n ? (long long)f(i) : 0;
        v += vals[k];
    }
    long long total;
    long long ex = block_excl_scan(v, &total) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        int64_t i = base + (int64_t)threadIdx.x * ITEMS + k;
        if (i < n) out[i] = (Out)ex;
        ex += vals[k];
        if (write_last && i == n - 1) out[n] = (Out)ex;
    }
}

// small inputs (the plans of configs[0] / [1], every scan of a small spill): the three steps in one block, one launch
constexpr int64_t SMALL_N = 16 * TILE;
template <typename F, typename Out>
__global__ void small_scan_kernel(int64_t n, F f, Out *out, bool write_last, long long *total_dev)
{
    long long carry = 0;
    for (int64_t base = 0; base < n; base += TILE) {
        long long vals[ITEMS];
        long long v = 0;
#pragma unroll
        for (int k = 0; k < ITEMS; ++k) {
            const int64_t i = base + (int64_t)threadIdx.x * ITEMS + k;
            vals[k] = i < n ? (long long)f(i) : 0;
            v += vals[k];
        }
        long long total;
        long long ex = block_excl_scan(v, &total) + carry;
        if (out) {
#pragma unroll
            for (int k = 0; k < ITEMS; ++k) {
                const int64_t i = base + (int64_t)threadIdx.x * ITEMS + k;
                if (i < n) out[i] = (Out)ex;
                ex += vals[k];
            }
        }
        carry += total;
    }
    if (threadIdx.x == 0) {
        if (total_dev) *total_dev = carry;
        if (write_last && out) out[n] = (Out)carry;
    }
}

// out[i] = sum_{k<i} f(k) for i in [0, n) (and out[n] = grand total when write_last);
// *total_dev (optional) receives the grand total.  tmp must hold ceil(n / TILE) + 1 long longs.
template <typename F, typename Out>
inline cudaError_t exclusive_scan(int64_t n, F f, Out *out, bool write_last, long long *total_dev,
                                  long long *tmp, cudaStream_t st)
{
    if (n <= 0) {
        if (total_dev) cudaMemsetAsync(total_dev, 0, sizeof(long long), st);
        if (write_last && out) cudaMemsetAsync(out, 0, sizeof(Out), st);
        return cudaGetLastError();
    }
    if (n <= SMALL_N) {
        ++g_lartpc_launches;
        small_scan_kernel<<<1, THREADS, 0, st>>>(n, f, out, write_last, total_dev);
        return cudaGetLastError();
    }
    int64_t blocks = (n + TILE - 1) / TILE;
    ++g_lartpc_launches;
    block_sums_kernel<<<(unsigned)blocks, THREADS, 0, st>>>(n, f, tmp);
    ++g_lartpc_launches;
    scan_sums_kernel<<<1, THREADS, 0, st>>>(tmp, blocks, total_dev);
    if (out) { ++g_lartpc_launches; final_scan_kernel<<<(unsigned)blocks, THREADS, 0, st>>>(n, f, tmp, out, write_last); }
    return cudaGetLastError();
}

inline int64_t tmp_elems(int64_t n) { return (n + TILE - 1) / TILE + 1; }

}  // namespace lscan
