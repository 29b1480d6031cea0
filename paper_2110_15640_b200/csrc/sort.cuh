// sort.cuh -- counting sort of one pass of event records by (channel, cell), between the transport kernel and the
// peel-off kernel.  Peel-off rays of one observer are parallel, so events that start in the same cell of the same
// channel march through the same columns of the same extinction table for nearly the same number of segments:
// handing the peel kernel its events in (channel, cell) order turns 32 unrelated gathers per warp-load into one or
// two sectors and makes the lanes of a warp finish together.  Only a permutation is built (4 B per event); the
// 48 B records stay where the transport kernel wrote them.
//
//   key(e) = clamp(chan_run(e) - chan_lo, 0, c_fold - 1) * bins_per_chan + (k * nlat + j) * nlg + (i >> lev_shift)
//            (cells when a channel has >= 2 packets per cell; groups of 4 levels or whole columns for sparser runs)
//   ev_hist_kernel    hist[key]++   (global atomics; albedo runs count the bin while the record is written instead)
//   scan_*            exclusive prefix sum of hist in place        (tile reduce, scan of tile sums, tile scan)
//   ev_scatter_kernel perm[hist[key]++] = e
//
// chan_lo is the first channel this pass draws fresh packets from (resumed packets of earlier channels clamp to it)
// and c_fold the number of channels a pass can span; the clamped key keeps the order monotone in the channel, which
// the peel kernel's per-warp flux bins rely on, and bounds the histogram (<= 2^25 bins).
#pragma once
#include "device_common.cuh"

namespace gcmcrt {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;                       // per thread
constexpr int kScanTile = kScanThreads * kScanItems;  // 4096 bins per CTA

struct SortParams {
    const unsigned int* keys;    // [n] sort keys: stored with the event records (kernels.cuh write_event), or the
                                 // launch keys of the first flights
    const unsigned int* count;   // number of items on the device (events written this pass), or NULL -> n_host
    unsigned int cap, n_host;
    unsigned int* hist;          // [nbins]
    unsigned int* tile_sums;     // [n_tiles]
    unsigned int* perm;          // [cap]
    unsigned int nbins, n_tiles;
    int nlev, nlat, ncell, c_fold;
};

__global__ void __launch_bounds__(256) ev_hist_kernel(const SortParams p)
{
    const unsigned int n = p.count ? min(*p.count, p.cap) : p.n_host;
    for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x)
        atomicAdd(p.hist + __ldg(p.keys + e), 1u);
}

// Consecutive records were written by one warp of neighbouring packets and often share their (channel, cell) key:
// the lanes of a warp that hold the same key take their slots with one atomic (any order inside a bin is valid).
__global__ void __launch_bounds__(256) ev_scatter_kernel(const SortParams p)
{
    const unsigned int n = p.count ? min(*p.count, p.cap) : p.n_host;
    const unsigned int n_round = (n + 31u) & ~31u;
    for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < n_round; e += gridDim.x * blockDim.x) {
        const bool valid = e < n;
        const unsigned int key = valid ? __ldg(p.keys + e) : 0xffffffffu - lane_id();
        const unsigned int peers = __match_any_sync(kFullMask, key);
        const int leader = __ffs(peers) - 1;
        unsigned int base = 0;
        if (valid && lane_id() == leader) base = atomicAdd(p.hist + key, (unsigned int)__popc(peers));
        base = __shfl_sync(kFullMask, base, leader);
        GCMCRT_CHECK(!valid || (key < p.nbins && base + __popc(peers & ((1u << lane_id()) - 1u)) < n));
        if (valid) p.perm[base + __popc(peers & ((1u << lane_id()) - 1u))] = e;
    }
}

__device__ __forceinline__ unsigned int block_sum_u32(unsigned int v, unsigned int* warp_part)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
    if (lane_id() == 0) warp_part[threadIdx.x >> 5] = v;
    __syncthreads();
    unsigned int t = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += warp_part[w];
    __syncthreads();
    return t;
}

// tile_sums[b] = sum of hist over tile b
__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const SortParams p)
{
    __shared__ unsigned int warp_part[kScanThreads / 32];
    const unsigned int base = blockIdx.x * kScanTile;
    unsigned int s = 0;
#pragma unroll
    for (int m = 0; m < kScanItems; ++m) {
        const unsigned int idx = base + m * kScanThreads + threadIdx.x;
        if (idx < p.nbins) s += p.hist[idx];
    }
    s = block_sum_u32(s, warp_part);
    if (threadIdx.x == 0) p.tile_sums[blockIdx.x] = s;
}

// exclusive scan of tile_sums in place, one CTA
__global__ void __launch_bounds__(1024) scan_tiles_kernel(const SortParams p)
{
    __shared__ unsigned int warp_tot[32];
    __shared__ unsigned int carry_s;
    const int lane = lane_id(), wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (unsigned int base = 0; base < p.n_tiles; base += blockDim.x) {
        const unsigned int idx = base + threadIdx.x;
        const unsigned int x = idx < p.n_tiles ? p.tile_sums[idx] : 0u;
        unsigned int v = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int n = __shfl_up_sync(kFullMask, v, o);
            if (lane >= o) v += n;
        }
        if (lane == 31) warp_tot[wid] = v;
        __syncthreads();
        if (wid == 0) {
            unsigned int w = warp_tot[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int n = __shfl_up_sync(kFullMask, w, o);
                if (lane >= o) w += n;
            }
            warp_tot[lane] = w;
        }
        __syncthreads();
        const unsigned int carry = carry_s;
        const unsigned int incl = carry + (wid > 0 ? warp_tot[wid - 1] : 0u) + v;
        if (idx < p.n_tiles) p.tile_sums[idx] = incl - x;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry_s = incl;
        __syncthreads();
    }
}

// hist[idx] = tile offset + exclusive scan within the tile (each thread owns kScanItems consecutive bins)
__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(const SortParams p)
{
    __shared__ unsigned int warp_tot[kScanThreads / 32];
    const unsigned int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
    unsigned int x[kScanItems];
    unsigned int s = 0;
#pragma unroll
    for (int m = 0; m < kScanItems; ++m) {
        x[m] = (base + m < p.nbins) ? p.hist[base + m] : 0u;
        s += x[m];
    }
    const int lane = lane_id(), wid = threadIdx.x >> 5;
    unsigned int v = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int n = __shfl_up_sync(kFullMask, v, o);
        if (lane >= o) v += n;
    }
    if (lane == 31) warp_tot[wid] = v;
    __syncthreads();
    unsigned int off = p.tile_sums[blockIdx.x] + (v - s);
    for (int w = 0; w < wid; ++w) off += warp_tot[w];
#pragma unroll
    for (int m = 0; m < kScanItems; ++m) {
        if (base + m < p.nbins) p.hist[base + m] = off;
        off += x[m];
    }
}

}  // namespace gcmcrt
