// S1 / K1: event-batched layout of the UT hits: segmented sort by (layer, y-sector, x0, id) + per-event bin table.
// Paper: UT hits are grouped in Y sectors so that a seed only looks at compatible ones (P:109-P:111); the sort by x
// inside a sector and the x0 slices are this library's own layout (BASELINE north_star (1)).
//
// One thread block per event.  The sort is a counting sort on the fine bin (layer, sector, x0 slice) followed by a
// rank inside each fine bin (a handful of hits), so there is no comparison network and no global scratch:
//   A  histogram of the fine bins in shared memory (atomicAdd returns the hit's arrival slot in its bin)
//   B  block-wide exclusive scan -> bin starts (= the bin table that is written out)
//   C  arrival-ordered member list per bin
//   D  rank of every hit among the members of its bin by (x0, id, original index) -> final position q
//   E  field by field: scatter in[i] -> smem[q], then coalesced copy smem -> out (double buffered)
// Events larger than the shared-memory capacity chosen from the caller's hint take an O(n^2) rank over global
// memory (phase A/B identical), which yields the same permutation.
#include "ds_common.cuh"

namespace ds {

constexpr int kLayoutThreads = 512;
constexpr int kMaxBins = 4 * DS_MAX_SECTORS * kXBins;

__device__ __forceinline__ int fine_bin(const DevConst &c, int id, float x0)
{
    int sec = min(id_sector(id), c.n_sectors - 1);
    return (id_layer(id) * c.n_sectors + sec) * kXBins + xbin(x0, c.xb_off, c.xb_scale);
}

// exclusive scan of v[0..n) in place (n <= a few thousand), v[n] = total.  All threads of the block call it.
__device__ void block_exclusive_scan(int *v, int n, int *warp_sums)
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

template <typename T>
__device__ __forceinline__ void scatter_field(const T *__restrict__ in, T *buf, const uint32_t *q, int n)
{
    for (int i = threadIdx.x; i < n; i += blockDim.x) buf[q[i]] = in[i];
}

template <typename T>
__device__ __forceinline__ void copy_out(const T *buf, T *__restrict__ out, int n)
{
    for (int i = threadIdx.x; i < n; i += blockDim.x) out[i] = buf[i];
}

__global__ void __launch_bounds__(kLayoutThreads)
k_layout(const __grid_constant__ DevConst c, const LayoutPtrs p, const int32_t *__restrict__ hit_offsets, int cap)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int warp_sums[33];
    const int nb = c.n_bins;
    int *hist = reinterpret_cast<int *>(smem_raw);                    // [nb + 1]
    uint32_t *keyx = reinterpret_cast<uint32_t *>(hist + kMaxBins + 1); // [cap] orderable x0
    uint32_t *pk = keyx + cap;                                         // [cap] bin << 20 | slot, later q
    uint32_t *bufA = pk + cap, *bufB = bufA + cap;                     // [cap] staging
    uint16_t *lst = reinterpret_cast<uint16_t *>(bufB + cap);          // [cap] members of each bin, arrival order

    const int e = blockIdx.x;
    const int h0 = hit_offsets[e];
    const int n = hit_offsets[e + 1] - h0;
    const int tid = threadIdx.x;
    const bool fast = n <= cap;
    const float *x0 = p.x0 + h0;
    const int32_t *hid = p.id + h0;

    for (int b = tid; b <= nb; b += blockDim.x) hist[b] = 0;
    __syncthreads();
    // A
    for (int i = tid; i < n; i += blockDim.x) {
        float x = x0[i];
        int b = fine_bin(c, hid[i], x);
        int slot = atomicAdd(&hist[b], 1);
        if (fast) {
            keyx[i] = float_key(x);
            pk[i] = ((uint32_t)b << 20) | (uint32_t)slot;
        }
    }
    __syncthreads();
    // B
    block_exclusive_scan(hist, nb, warp_sums);
    int32_t *tab = p.bin_offsets + (size_t)e * (nb + 1);
    for (int b = tid; b <= nb; b += blockDim.x) tab[b] = hist[b];

    if (fast) {
        // C
        for (int i = tid; i < n; i += blockDim.x) {
            uint32_t v = pk[i];
            lst[hist[v >> 20] + (v & 0xfffffu)] = (uint16_t)i;
        }
        __syncthreads();
        // D
        for (int i = tid; i < n; i += blockDim.x) {
            const int b = pk[i] >> 20;
            const uint32_t ki = keyx[i];
            const int jb = hist[b], je = hist[b + 1];
            int rank = 0;
            for (int j = jb; j < je; ++j) {
                const int m = lst[j];
                const uint32_t km = keyx[m];
                bool less = km < ki;
                if (km == ki && m != i) {
                    const int im = hid[m], ii = hid[i];
                    less = im < ii || (im == ii && m < i);
                }
                rank += less ? 1 : 0;
            }
            pk[i] = (uint32_t)(jb + rank);   // q (pk[i] is only ever touched by the thread that owns hit i)
        }
        __syncthreads();
        // E: perm, x0, z, ymin, ymax, w, id
        for (int i = tid; i < n; i += blockDim.x) bufA[pk[i]] = (uint32_t)(h0 + i);
        __syncthreads();
        scatter_field(x0, reinterpret_cast<float *>(bufB), pk, n);
        copy_out(reinterpret_cast<int32_t *>(bufA), p.perm + h0, n);
        __syncthreads();
        scatter_field(p.z + h0, reinterpret_cast<float *>(bufA), pk, n);
        copy_out(reinterpret_cast<float *>(bufB), p.sx0 + h0, n);
        __syncthreads();
        scatter_field(p.ymin + h0, reinterpret_cast<float *>(bufB), pk, n);
        copy_out(reinterpret_cast<float *>(bufA), p.sz + h0, n);
        __syncthreads();
        scatter_field(p.ymax + h0, reinterpret_cast<float *>(bufA), pk, n);
        copy_out(reinterpret_cast<float *>(bufB), p.symin + h0, n);
        __syncthreads();
        scatter_field(p.w + h0, reinterpret_cast<float *>(bufB), pk, n);
        copy_out(reinterpret_cast<float *>(bufA), p.symax + h0, n);
        __syncthreads();
        scatter_field(hid, reinterpret_cast<int32_t *>(bufA), pk, n);
        copy_out(reinterpret_cast<float *>(bufB), p.sw + h0, n);
        __syncthreads();
        copy_out(reinterpret_cast<int32_t *>(bufA), p.sid + h0, n);
    } else {
        // oversize event: rank over the whole event straight from global memory, scattered writes
        for (int i = tid; i < n; i += blockDim.x) {
            const float xi = x0[i];
            const int ii = hid[i];
            const int b = fine_bin(c, ii, xi);
            const uint32_t ki = float_key(xi);
            int rank = 0;
            for (int m = 0; m < n; ++m) {
                const float xm = x0[m];
                const int im = hid[m];
                if (fine_bin(c, im, xm) != b) continue;
                const uint32_t km = float_key(xm);
                bool less = km < ki;
                if (km == ki && m != i) less = im < ii || (im == ii && m < i);
                rank += less ? 1 : 0;
            }
            const size_t q = (size_t)h0 + hist[b] + rank;
            p.perm[q] = h0 + i;
            p.sx0[q] = xi;
            p.sz[q] = p.z[h0 + i];
            p.symin[q] = p.ymin[h0 + i];
            p.symax[q] = p.ymax[h0 + i];
            p.sw[q] = p.w[h0 + i];
            p.sid[q] = ii;
        }
    }
}

static size_t layout_smem_bytes(int cap) { return sizeof(int) * (kMaxBins + 1) + (size_t)cap * (4 * 4 + 2) + 16; }

cudaError_t launch_layout(const DevConst &c, const LayoutPtrs &p, const int32_t *hit_offsets, int n_events,
                          int max_event_hits_hint, cudaStream_t st, Prof &prof)
{
    if (n_events <= 0) return cudaSuccess;
    int hint = max_event_hits_hint > 0 ? max_event_hits_hint : 4096;
    int cap = (hint + 255) & ~255;
    const int cap_max = (int)((227 * 1024 - sizeof(int) * (kMaxBins + 1) - 512) / 18) & ~255;   // 227 KB per CTA
    if (cap > cap_max) cap = cap_max;
    if (cap > 65536) cap = 65536;   // lst holds uint16 indices
    const size_t smem = layout_smem_bytes(cap);
    cudaError_t err = cudaFuncSetAttribute(k_layout, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    prof.begin(DS_K_LAYOUT, st);
    k_layout<<<n_events, kLayoutThreads, smem, st>>>(c, p, hit_offsets, cap);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
