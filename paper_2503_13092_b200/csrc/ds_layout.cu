// S1 / K1: event-batched layout of the UT hits: segmented sort by (layer, y-sector, x0, id) + per-event bin table.
// Paper: UT hits are grouped in Y sectors so that a seed only looks at compatible ones (P:109-P:111); the sort by x
// inside a sector and the x0 slices are this library's own layout (BASELINE north_star (1)).
//
// One thread block per event.  The sort is a counting sort on the fine bin (layer, sector, x0 slice) followed by a
// rank inside each fine bin (a handful of hits), so there is no comparison network and no global scratch.  The
// event's six input arrays are brought into shared memory by 1-D bulk async copies (cp.async.bulk + mbarrier), each
// exactly once: x0 and id up front (they make the sort key), z while the sort runs, ymin / ymax / w into buffers as
// they fall free, so that every load is in flight behind the work on the previous array:
//   A  histogram of the fine bins (atomicAdd returns the hit's arrival slot in its bin)
//   B  block-wide exclusive scan -> bin starts (= the bin table that is written out)
//   C  orderable x0 keys and hit indices laid out bin by bin, in arrival order
//   D  rank of every hit among the keys of its bin (ties: id, then original index) -> final position q; src[q] = hit
//   E  per array: out[q] = staged[src[q]], coalesced stores
// Events larger than the shared-memory capacity chosen from the caller's hint take an O(n^2) rank over global
// memory (phase A/B identical), which yields the same permutation.
//
// Two output forms.  ds_layout (public, S1 alone) writes the sorted SoA of include/ds.h: seven arrays.  Inside ds_reconstruct
// (kInternal) the consumer is k_track, and the layout is the one it reads best:
//   sx0    [n]  sorted x0 (the only array a window search scans)
//   aux    [n]  float4 (z, w, perm, id) of the hit at a sorted position: read only for hits that passed a window, and then
//               one 16-byte load brings all four (one DRAM sector instead of four)
//   ybounds [E][4 * n_sectors] (ymin, ymax) of each (layer, sector), and uniform[e] = 1 iff every hit of the event carries
//               exactly the bounds of its (layer, sector).  That is how detectors are built (A-2: a strip's y range is its
//               sector's), so y-compatibility becomes one test per (seed, sector) instead of one per hit and k_track stages
//               4 instead of 12 bytes per hit.  symin / symax (sorted per-hit bounds) are written only for events that are
//               not uniform; k_track then tests every hit with its own bounds.
#include "ds_sort.cuh"

namespace ds {

constexpr int kLayoutThreads = 512;
template <bool kInternal>
__global__ void __launch_bounds__(2 * kLayoutThreads)
k_layout(const __grid_constant__ DevConst c, const LayoutPtrs p, const int32_t *__restrict__ hit_offsets, int n_events, int cap,
         bool bulk, const int32_t *__restrict__ only)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int warp_sums[33];
    __shared__ __align__(8) unsigned long long bars[3];
    __shared__ float2 s_ref[kLayers * DS_MAX_SECTORS];   // kInternal: (ymin, ymax) of the first hit of each (layer, sector)
    __shared__ int s_nonuni;
    const int nb = c.n_bins, nfine = nb * kSub;
    // cap is a multiple of 4, so every array starts on a 16-byte boundary
    float *s_x0 = reinterpret_cast<float *>(smem_raw);                 // [cap] x0, later ymin
    int32_t *s_id = reinterpret_cast<int32_t *>(s_x0 + cap);           // [cap] id, later ymax
    uint32_t *s_pk = reinterpret_cast<uint32_t *>(s_id + cap);         // [cap] bin << 20 | slot, later q
    uint32_t *s_buf = s_pk + cap;                                      // [cap] keys in bin order, later z, later w
    uint16_t *s_src = reinterpret_cast<uint16_t *>(s_buf + cap);       // [cap] hits in bin order, later src[q]
    int *hist = reinterpret_cast<int *>(s_src + cap);                  // [nfine + 1]
    unsigned long long *bar_x = &bars[0], *bar_i = &bars[1], *bar_b = &bars[2];

    if (only) {   // normally nothing is left over: all marks of this block's events in one round of loads, then out
        bool any = false;
        for (int e = blockIdx.x + threadIdx.x * gridDim.x; e < n_events; e += blockDim.x * gridDim.x) any |= only[e] != 0;
        if (!__syncthreads_or(any)) return;
    }
    // one event per block; with `only` (the events k_event has left over) a small grid walks the event list and a block may
    // meet several marked events: the launcher then passes cap = 0, so that none of them takes the staged path (whose
    // mbarriers are armed once per block)
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
    if (only && only[e] == 0) continue;
    __syncthreads();   // the previous event of this block is finished
    const int h0 = hit_offsets[e];
    const int n = hit_offsets[e + 1] - h0;
    const int tid = threadIdx.x;
    const int d = h0 & 3;
    const bool fast = n + 3 <= cap;

    if (tid == 0 && fast) {
        mbar_init(bar_x, 1);
        mbar_init(bar_i, 1);
        mbar_init(bar_b, 1);
    }
    for (int b = tid; b <= nfine; b += blockDim.x) hist[b] = 0;
    __syncthreads();

    if (fast) {
        stage_field(s_x0, p.x0, h0, n, bar_x, bulk);
        stage_field(s_id, p.id, h0, n, bar_i, bulk);
        __syncthreads();
        mbar_wait(bar_x, 0);
        mbar_wait(bar_i, 0);
        // A
        for (int i = tid; i < n; i += blockDim.x) {
            const int b = fine_bin(c, s_id[d + i], s_x0[d + i]);
            const int slot = atomicAdd(&hist[b], 1);
            s_pk[i] = ((uint32_t)b << 20) | (uint32_t)slot;
        }
        __syncthreads();
    } else {
        for (int i = tid; i < n; i += blockDim.x) atomicAdd(&hist[fine_bin(c, p.id[h0 + i], p.x0[h0 + i])], 1);
        __syncthreads();
    }
    // B
    block_exclusive_scan(hist, nfine, warp_sums);
    int32_t *tab = p.bin_offsets + (size_t)e * (nb + 1);
    for (int b = tid; b <= nb; b += blockDim.x) tab[b] = hist[b * kSub];

    if (fast) {
        // C
        for (int i = tid; i < n; i += blockDim.x) {
            const uint32_t v = s_pk[i];
            const int pos = hist[v >> 20] + (int)(v & 0xfffffu);
            s_buf[pos] = float_key(s_x0[d + i]);
            s_src[pos] = (uint16_t)i;
        }
        __syncthreads();
        // D
        for (int i = tid; i < n; i += blockDim.x) {
            const int b = s_pk[i] >> 20;
            const uint32_t ki = float_key(s_x0[d + i]);
            const int jb = hist[b], je = hist[b + 1];
            int rank = 0, eq = 0;
            for (int j = jb; j < je; j += 4) {   // four keys at a time (a sub-slice holds about one)
                uint32_t km[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) km[u] = s_buf[min(j + u, je - 1)];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const bool in = j + u < je;
                    rank += (in & (km[u] < ki)) ? 1 : 0;
                    eq += (in & (km[u] == ki)) ? 1 : 0;
                }
            }
            if (eq > 1) {   // equal x0 inside the bin: order by (id, original index)
                const int ii = s_id[d + i];
                for (int j = jb; j < je; ++j) {
                    const int m = s_src[j];
                    if (s_buf[j] == ki && m != i) {
                        const int im = s_id[d + m];
                        rank += (im < ii || (im == ii && m < i)) ? 1 : 0;
                    }
                }
            }
            s_pk[i] = (uint32_t)(jb + rank);   // q
        }
        __syncthreads();
        for (int i = tid; i < n; i += blockDim.x) s_src[s_pk[i]] = (uint16_t)i;
        __syncthreads();
        if (!kInternal) {
            // E: z is loaded while perm, x0 and id go out; ymin, ymax, w follow into the buffers that fall free
            stage_field(reinterpret_cast<float *>(s_buf), p.z, h0, n, bar_b, bulk);
            for (int q = tid; q < n; q += blockDim.x) {
                const int i = s_src[q];
                p.perm[h0 + q] = h0 + i;
                p.sx0[h0 + q] = s_x0[d + i];
                p.sid[h0 + q] = s_id[d + i];
            }
            __syncthreads();
            stage_field(s_x0, p.ymin, h0, n, bar_x, bulk);
            stage_field(reinterpret_cast<float *>(s_id), p.ymax, h0, n, bar_i, bulk);
            mbar_wait(bar_b, 0);
            for (int q = tid; q < n; q += blockDim.x) p.sz[h0 + q] = reinterpret_cast<float *>(s_buf)[d + s_src[q]];
            __syncthreads();
            stage_field(reinterpret_cast<float *>(s_buf), p.w, h0, n, bar_b, bulk);
            mbar_wait(bar_x, 1);
            mbar_wait(bar_i, 1);
            for (int q = tid; q < n; q += blockDim.x) {
                const int i = d + s_src[q];
                p.symin[h0 + q] = s_x0[i];
                p.symax[h0 + q] = reinterpret_cast<float *>(s_id)[i];
            }
            __syncthreads();
            mbar_wait(bar_b, 1);
            for (int q = tid; q < n; q += blockDim.x) p.sw[h0 + q] = reinterpret_cast<float *>(s_buf)[d + s_src[q]];
        } else {
            // E (internal form): z and w are loaded (into the key and rank buffers, both free now) while x0 goes out; ymin
            // follows into the x0 buffer while the aux records (z, w, perm, id) go out; ymax into the key buffer
            float *b_z = reinterpret_cast<float *>(s_buf), *b_w = reinterpret_cast<float *>(s_pk);
            stage_field(b_z, p.z, h0, n, bar_b, bulk);
            stage_field(b_w, p.w, h0, n, bar_x, bulk);            // bar_x: second use (phase 1)
            const int ncoarse = kLayers * c.n_sectors;
            if (tid < kLayers * DS_MAX_SECTORS) s_ref[tid] = make_float2(0.f, 0.f);
            if (tid == 0) s_nonuni = 0;
            for (int q = tid; q < n; q += blockDim.x) p.sx0[h0 + q] = s_x0[d + s_src[q]];
            __syncthreads();
            stage_field(s_x0, p.ymin, h0, n, bar_i, bulk);        // bar_i: second use (phase 1)
            mbar_wait(bar_b, 0);
            mbar_wait(bar_x, 1);
            for (int q = tid; q < n; q += blockDim.x) {
                const int i = s_src[q];
                p.aux[h0 + q] = make_float4(b_z[d + i], b_w[d + i], __int_as_float(h0 + i), __int_as_float(s_id[d + i]));
            }
            __syncthreads();
            float *b_ymin = s_x0, *b_ymax = reinterpret_cast<float *>(s_buf);
            stage_field(b_ymax, p.ymax, h0, n, bar_b, bulk);      // bar_b: second use (phase 1)
            mbar_wait(bar_i, 1);
            mbar_wait(bar_b, 1);
            __syncthreads();   // the tail elements of ymax were stored by ordinary stores of other threads
            // reference bounds of a (layer, sector): those of its first hit in sorted order; then every hit against them
            if (tid < ncoarse) {
                const int qb = hist[tid * (kXBins * kSub)], qe = hist[(tid + 1) * (kXBins * kSub)];
                if (qb < qe) {
                    const int i = s_src[qb];
                    s_ref[tid] = make_float2(b_ymin[d + i], b_ymax[d + i]);
                }
            }
            __syncthreads();
            bool differs = false;
            for (int i = tid; i < n; i += blockDim.x) {
                const int id = s_id[d + i];
                const float2 r = s_ref[id_layer(id) * c.n_sectors + min(id_sector(id), c.n_sectors - 1)];
                differs |= (b_ymin[d + i] != r.x) | (b_ymax[d + i] != r.y);
            }
            if (differs) s_nonuni = 1;
            __syncthreads();
            const bool nonuni = s_nonuni != 0;
            if (tid < ncoarse) p.ybounds[(size_t)e * ncoarse + tid] = s_ref[tid];
            if (tid == 0) p.uniform[e] = nonuni ? 0 : 1;
            if (nonuni) {
                for (int q = tid; q < n; q += blockDim.x) {
                    const int i = d + s_src[q];
                    p.symin[h0 + q] = b_ymin[i];
                    p.symax[h0 + q] = b_ymax[i];
                }
            }
        }
    } else {
        // oversize event: rank over the whole event straight from global memory, scattered writes
        const float *x0 = p.x0 + h0;
        const int32_t *hid = p.id + h0;
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
            p.sx0[q] = xi;
            p.symin[q] = p.ymin[h0 + i];
            p.symax[q] = p.ymax[h0 + i];
            if (kInternal) {
                p.aux[q] = make_float4(p.z[h0 + i], p.w[h0 + i], __int_as_float(h0 + i), __int_as_float(ii));
            } else {
                p.perm[q] = h0 + i;
                p.sz[q] = p.z[h0 + i];
                p.sw[q] = p.w[h0 + i];
                p.sid[q] = ii;
            }
        }
        if (kInternal) {   // an event that is not staged is never declared uniform: k_track tests its hits one by one
            if (tid < kLayers * c.n_sectors) p.ybounds[(size_t)e * (kLayers * c.n_sectors) + tid] = make_float2(0.f, 0.f);
            if (tid == 0) p.uniform[e] = 0;
        }
    }
    }   // events of this block
}


static size_t layout_smem_bytes(int cap, int n_bins) { return (size_t)cap * 18 + sizeof(int) * ((size_t)n_bins * kSub + 1) + 16; }

cudaError_t launch_layout(const DevConst &c, const LayoutPtrs &p, const int32_t *hit_offsets, int n_events,
                          int max_event_hits_hint, const int32_t *only, cudaStream_t st, Prof &prof)
{
    if (n_events <= 0) return cudaSuccess;
    // staging capacity in hits: a multiple of 4 with room for the alignment slack, 18 bytes each; hit indices inside an
    // event are kept as uint16_t
    const int hint = max_event_hits_hint > 0 ? max_event_hits_hint : 4096;
    int cap = ((hint + 3) & ~3) + 8;
    int cap_max = (int)((227 * 1024 - sizeof(int) * ((size_t)c.n_bins * kSub + 1) - 1024) / 18) & ~3;   // 227 KB per CTA, static part included
    if (cap_max > 65532) cap_max = 65532;
    if (cap > cap_max) cap = cap_max;
    const size_t smem = layout_smem_bytes(cap, c.n_bins);
    const bool internal = p.aux != nullptr;
    static unsigned long long opted[2] = {0, 0};
    const cudaError_t aerr = internal ? opt_in_max_smem(k_layout<true>, &opted[1]) : opt_in_max_smem(k_layout<false>, &opted[0]);
    if (aerr != cudaSuccess) return aerr;
    // the bulk copies need 16-byte aligned sources (offsets inside the arrays are handled by the kernel)
    const uintptr_t bits = reinterpret_cast<uintptr_t>(p.x0) | reinterpret_cast<uintptr_t>(p.z) |
                           reinterpret_cast<uintptr_t>(p.ymin) | reinterpret_cast<uintptr_t>(p.ymax) |
                           reinterpret_cast<uintptr_t>(p.w) | reinterpret_cast<uintptr_t>(p.id);
    const bool bulk = (bits & 15) == 0;
    prof.begin(DS_K_LAYOUT, st);
    // events so large that one block fills an SM's shared memory get twice the threads (every loop strides by blockDim.x)
    const int threads = smem + 1024 > (228 * 1024) / 2 ? 2 * kLayoutThreads : kLayoutThreads;
    const int grid = only ? (n_events < kRedoGrid ? n_events : kRedoGrid) : n_events;
    if (only) cap = 0;
    if (internal) k_layout<true><<<grid, threads, smem, st>>>(c, p, hit_offsets, n_events, cap, bulk, only);
    else k_layout<false><<<grid, threads, smem, st>>>(c, p, hit_offsets, n_events, cap, bulk, only);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
