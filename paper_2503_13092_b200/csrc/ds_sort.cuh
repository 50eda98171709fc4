// Pieces of the per-event counting sort of the UT hits (S1) shared by k_layout (ds_layout.cu) and k_event (ds_event.cu):
// the sort bin of a hit, a block-wide exclusive scan, and the staging of one input array into shared memory by a 1-D bulk
// async copy.
#pragma once

#include "ds_common.cuh"

namespace ds {

#ifndef DS_KSUB
#define DS_KSUB 4
#endif
constexpr int kSub = DS_KSUB;   // the sort cuts every x0 slice of the bin table into kSub sub-slices (a power of two)

// Sort bin of a hit: (layer, sector, x0 sub-slice).  t = (x0 + off) * scale is the same fp32 value xbin() floors, and
// 4t is exact, so floor(floor(kSub * t) / kSub) = floor(t): sub-slice s lies in table slice s / kSub, clamps included.
__device__ __forceinline__ int fine_bin(const DevConst &c, int id, float x0)
{
    int sec = min(id_sector(id), c.n_sectors - 1);
    return (id_layer(id) * c.n_sectors + sec) * (kXBins * kSub) + xslice<kXBins * kSub>(x0, c.xb_off, c.xb_scale);
}

// exclusive scan of v[0..n) in place (n <= a few thousand), v[n] = total.  All threads of the block call it.
__device__ inline void block_exclusive_scan(int *v, int n, int *warp_sums)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    const int per = (n + blockDim.x - 1) / blockDim.x;
    const int b = tid * per, e = min(b + per, n);
    int s = 0;
    for (int k = b; k < e; ++k) s += v[k];
    int inc = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = lane < nw ? warp_sums[lane] : 0, wi = ws;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= d) wi += t;
        }
        if (lane < nw) warp_sums[lane] = wi - ws;
        if (lane == 31) warp_sums[32] = wi;
    }
    __syncthreads();
    int run = warp_sums[wid] + inc - s;
    for (int k = b; k < e; ++k) {
        int t = v[k];
        v[k] = run;
        run += t;
    }
    if (tid == 0) v[n] = warp_sums[32];
    __syncthreads();
}

// Stage global src[h0 .. h0+n) into a shared buffer so that element i sits at buf[(h0 & 3) + i]: the part of the slice
// between 16-byte boundaries by one bulk async copy that completes on `bar` (issued by thread 0, which also arms the
// barrier), the up to three elements after the last boundary by ordinary loads (threads 32..34).  With `bulk` false
// (a source pointer that is not 16-byte aligned) everything is loaded by ordinary loads and the barrier only armed.
// Every thread of the block calls it; the buffer must be free (a __syncthreads after its last reader), and a
// __syncthreads plus mbar_wait(bar) must precede the first read.
template <typename T>
__device__ __forceinline__ void stage_field(T *buf, const T *__restrict__ src, int h0, int n, unsigned long long *bar,
                                            bool bulk);

// the same out of line for 4-byte elements of either type (k_event calls it five times per event)
__device__ void stage_words(void *buf, const void *src, int h0, int n, unsigned long long *bar, bool bulk);

template <typename T>
__device__ __forceinline__ void stage_field(T *buf, const T *__restrict__ src, int h0, int n, unsigned long long *bar,
                                            bool bulk)
{
    const int d = h0 & 3, h0a = h0 - d, h1 = h0 + n;
    const int h1dn = bulk ? max(h1 & ~3, h0a) : h0a;          // bulk part: [h0a, h1dn); it may start before h0
    if (threadIdx.x == 0) {
        const uint32_t bytes = 4u * (uint32_t)(h1dn - h0a);
        // the buffer may have been written and read by ordinary (generic-proxy) accesses of the whole block before the
        // __syncthreads that precedes this call: order them before the async-proxy write of the bulk copy
        fence_proxy_async();
        mbar_expect_tx(bar, bytes);
        if (bytes) bulk_g2s(buf, src + h0a, bytes, bar);
    }
    if (bulk) {
        const int t = (int)threadIdx.x - 32;
        if (t >= 0 && h1dn + t < h1 && h1dn + t >= h0) buf[h1dn + t - h0a] = src[h1dn + t];
    } else {
        for (int i = threadIdx.x; i < n; i += blockDim.x) buf[d + i] = src[h0 + i];
    }
}

}  // namespace ds
