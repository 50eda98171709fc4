// S2..S6 / K2+K3: seed extrapolation, window search, candidate fit and best-candidate choice.
// Paper: magnet point from the seed state; first search window in UTbX, <= 10 closest hits;
// per first hit a new trajectory through (hit, magnet point) and refined windows in UTaX/UTaU/UTbV keeping the
// closest 1/2/2 hits; one final candidate per SciFi seed by score.  Readings A-1..A-9 in DESIGN.md.
//
// Mapping: one thread block per event.  The event's slice of the sorted x0 array (what a window search scans) is staged in
// shared memory by a 1-D bulk async copy (cp.async.bulk + mbarrier), issued by one thread while the block loads the bin
// table and the event's per-sector y bounds.  y-compatibility: k_layout has checked whether every hit of the event carries
// exactly the y range of its (layer, sector) (the normal case, A-2); then a seed tests each sector once (a bit mask per
// layer, computed in phase A) and no per-hit bounds are read at all; otherwise every hit in a window is tested with its own
// bounds from the sorted global arrays.  The work is then flattened over the block in rounds of three phases:
//   A  thread per seed:      S2, first window in UTbX (S3) -> the seed's <= max_first first hits appended to a block-wide
//                            list (block scan of the counts; only if more hits pass than are tried, a selection by
//                            (distance, id))
//   B  thread per first hit: the three refined windows (S4), the <= 4 fits (S5) -> best score of this first hit
//   C  thread per seed:      best first hit (S6; exact score ties resolved by (more hits, ids)), the winner's fit is
//                            evaluated once more and the track record written, coalesced over the seeds
// z, w, id and perm are read from global memory only for hits that passed a window: one 16-byte aux record per hit (see
// ds_layout.cu).  Events larger than the staging buffer run the same code on the global arrays.
// All of this arithmetic is fp64 in registers on fp32 inputs (the deciding comparisons must agree with an fp64
// reference to ~1e-5 relative; fp32 would not: one ulp of x at 800 mm is 6e-5 mm).
#include <cstdlib>

#include "ds_track.cuh"

namespace ds {

// Development aid: DS_TRACK_BLOCKS=3|4 forces the blocks-per-SM configuration of k_track (0 / unset: automatic).
static int track_blocks_override()
{
    static int v = -1;
    if (v < 0) {
        const char *e = getenv("DS_TRACK_BLOCKS");
        v = e ? atoi(e) : 0;
    }
    return v;
}

__global__ void k_extrapolate(const __grid_constant__ DevConst c, const ds_seeds seeds, double *__restrict__ out)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= seeds.n) return;
    S2 r = extrapolate_seed(c, seeds.x[s], seeds.y[s], seeds.tx[s], seeds.ty[s], seeds.qop[s]);
    double *o = out + 12 * s;
    o[0] = r.zm; o[1] = r.xm; o[2] = r.ym; o[3] = r.y0; o[4] = r.y1; o[5] = r.y2; o[6] = r.y3;
    o[7] = r.txp; o[8] = r.xc3; o[9] = r.w0; o[10] = r.w1; o[11] = 0.0;
}

cudaError_t launch_extrapolate(const DevConst &c, const ds_seeds &seeds, double *out, cudaStream_t st)
{
    if (seeds.n <= 0) return cudaSuccess;
    k_extrapolate<<<(unsigned)((seeds.n + 255) / 256), 256, 0, st>>>(c, seeds, out);
    return cudaGetLastError();
}

// Block-shared state of k_track (carved from dynamic shared memory, followed by the staged hit arrays); W warps.
template <typename Idx, bool kDv1, int W>
struct TrackShared {
    unsigned long long bar;
    WarpShared<Idx, kDv1> warp[W];
    float2 yb[kLayers * DS_MAX_SECTORS];  // (ymin, ymax) of each (layer, sector) of the event (uniform events)
    Idx tab[kMaxBins + 1];                // the event's bin table
};
static_assert(kFirstCap <= 512 && kFitCap < 0xfff, "packing of task[] and ffit[]");


// W warps per block and kMinBlocks blocks per SM follow the staging size (launch_track): the Run-3-like event sizes run
// 5 warps x 4 blocks; events whose staging leaves room for fewer blocks get more warps per block, so that an SM keeps
// about the same number of warps busy
template <bool kDv1, int W, int kMinBlocks>
__global__ void __launch_bounds__(32 * W, kMinBlocks)
k_track(const __grid_constant__ DevConst c, const LayoutPtrs L, const ds_seeds seeds,
        const int32_t *__restrict__ hit_offsets, const int32_t *__restrict__ seed_offsets, const ds_tracks out, int n_events,
        int cap, const int32_t *__restrict__ only)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int kThreads = 32 * W;
    using Staged = TrackShared<uint16_t, kDv1, W>;
    using Direct = TrackShared<int, kDv1, W>;
    constexpr size_t kHitsAt = (sizeof(Staged) + 15) & ~(size_t)15;
    float *st_x0 = reinterpret_cast<float *>(smem_raw + kHitsAt);   // [cap]

    const int tid = threadIdx.x;
    if (only) {   // normally nothing is left over: all marks of this block's events in one round of loads, then out
        bool any = false;
        for (int e = blockIdx.x + threadIdx.x * gridDim.x; e < n_events; e += blockDim.x * gridDim.x) any |= only[e] != 0;
        if (!__syncthreads_or(any)) return;
    }
    // one event per block; with `only` (the events k_event has left over) a small grid walks the event list and a block may
    // meet several marked events: the launcher then passes cap = 0, so that none of them is staged (the mbarrier is armed
    // once per block)
    for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
    if (only && only[e] == 0) continue;
    __syncthreads();   // the previous event of this block is finished
    const int s_begin = seed_offsets[e], s_end = seed_offsets[e + 1];
    if (s_begin == s_end) continue;
    const int h0 = hit_offsets[e], h1 = hit_offsets[e + 1];
    const bool uni = L.uniform[e] != 0;
    // staged range: the event's slice widened to 16-byte boundaries (the sorted arrays are 256-byte aligned and padded)
    const int h0a = h0 & ~3, cnt = ((h1 + 3) & ~3) - h0a;
    const bool staged = cnt <= cap;   // cap < 65535 (see launch_track)
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(smem_raw);   // first member of both layouts
    if (tid == 0 && staged) {
        mbar_init(bar, 1);
        const uint32_t bytes = 4u * (uint32_t)cnt;
        mbar_expect_tx(bar, bytes);
        if (bytes) bulk_g2s(st_x0, L.sx0 + h0a, bytes, bar);
    }
    // the lane's first seed, fetched now so that the load is in flight with the table and the hits
    SeedPre pre;
    {
        const int chunk = seed_chunk<W>(s_begin, s_end);
        const int s = s_begin + (tid >> 5) * chunk + (tid & 31);
        pre = load_seed(seeds, s, !kDv1 && (tid & 31) < chunk && s < s_end);
    }
    const int nb = c.n_bins;
    const int32_t *gtab = L.bin_offsets + (size_t)e * (nb + 1);
    const int nyb = kLayers * c.n_sectors;
    if (staged) {
        Staged &sh = *reinterpret_cast<Staged *>(smem_raw);
        constexpr int kPer = (kMaxBins + kThreads) / kThreads;
        int v[kPer];
#pragma unroll
        for (int u = 0; u < kPer; ++u) v[u] = gtab[min(tid + u * kThreads, nb)];
        float2 ybv = make_float2(0.f, 0.f);
        if (tid < nyb) ybv = L.ybounds[(size_t)e * nyb + tid];
#pragma unroll
        for (int u = 0; u < kPer; ++u)
            if (tid + u * kThreads <= nb) sh.tab[tid + u * kThreads] = (uint16_t)v[u];
        if (tid < nyb) sh.yb[tid] = ybv;
    } else {
        Direct &sh = *reinterpret_cast<Direct *>(smem_raw);
        for (int b = tid; b <= nb; b += kThreads) sh.tab[b] = gtab[b];
        if (tid < nyb) sh.yb[tid] = L.ybounds[(size_t)e * nyb + tid];
    }
    __syncthreads();

    HitsSorted H;
    H.ymin = L.symin + h0; H.ymax = L.symax + h0; H.aux = L.aux + h0;
    if (staged) {
        mbar_wait(bar, 0);
        H.x0 = st_x0 + (h0 - h0a);
        Staged &sh = *reinterpret_cast<Staged *>(smem_raw);
        const BinTable<uint16_t, kXBins, true> tab{sh.tab};
        if (uni) track_event<uint16_t, kDv1, true, W>(c, sh.warp, tab, sh.yb, H, seeds, s_begin, s_end, out, pre);
        else track_event<uint16_t, kDv1, false, W>(c, sh.warp, tab, sh.yb, H, seeds, s_begin, s_end, out, pre);
    } else {
        H.x0 = L.sx0 + h0;
        Direct &sh = *reinterpret_cast<Direct *>(smem_raw);
        const BinTable<int, kXBins, true> tab{sh.tab};
        if (uni) track_event<int, kDv1, true, W>(c, sh.warp, tab, sh.yb, H, seeds, s_begin, s_end, out, pre);
        else track_event<int, kDv1, false, W>(c, sh.warp, tab, sh.yb, H, seeds, s_begin, s_end, out, pre);
    }
    }   // events of this block
}

// Threads and blocks per SM tried for a staging size, most blocks first (see launch_track)
template <bool kDv1, int W, int kMinBlocks>
static cudaError_t launch_one(const DevConst &c, const LayoutPtrs &lay, const ds_seeds &seeds, const int32_t *hit_offsets,
                              const int32_t *seed_offsets, int n_events, int cap, size_t smem, const int32_t *only,
                              const ds_tracks &out, cudaStream_t st, Prof &prof)
{
    static unsigned long long opted = 0;
    const cudaError_t aerr = opt_in_max_smem(k_track<kDv1, W, kMinBlocks>, &opted);
    if (aerr != cudaSuccess) return aerr;
    prof.begin(DS_K_TRACK, st);
    const int grid = only ? (n_events < kRedoGrid ? n_events : kRedoGrid) : n_events;
    k_track<kDv1, W, kMinBlocks><<<grid, 32 * W, smem, st>>>(c, lay, seeds, hit_offsets, seed_offsets, out, n_events, only ? 0 : cap, only);
    prof.end(st);
    return cudaGetLastError();
}

template <bool kDv1, int W>
static size_t track_smem(int cap)
{
    const size_t fixed = (sizeof(TrackShared<uint16_t, kDv1, W>) + 15) & ~(size_t)15;
    const size_t staged = fixed + (size_t)cap * 4, direct = sizeof(TrackShared<int, kDv1, W>);
    return staged > direct ? staged : direct;
}

template <bool kDv1>
static cudaError_t launch_track_t(const DevConst &c, const LayoutPtrs &lay, const ds_seeds &seeds, const int32_t *hit_offsets,
                                  const int32_t *seed_offsets, int n_events, int hint, const int32_t *only, const ds_tracks &out,
                                  cudaStream_t st, Prof &prof)
{
    // staging capacity in hits (a multiple of 4, with room for the alignment slack): 4 bytes each; positions of a staged
    // event are stored as uint16_t with 0xffff = none
    int cap = ((hint + 3) & ~3) + 8;
    const size_t kSm = 227 * 1024, kPerBlock = 1024;   // usable shared memory of an SM; reserved per resident block
    // configuration: as many blocks per SM as the staging allows (more resident warps hide more latency)
    const int want = track_blocks_override();
    if ((want == 0 || want == 4) && 4 * (track_smem<kDv1, 5>(cap) + kPerBlock) <= kSm + 1024)
        return launch_one<kDv1, 5, 4>(c, lay, seeds, hit_offsets, seed_offsets, n_events, cap, track_smem<kDv1, 5>(cap), only, out, st, prof);
    if ((want == 0 || want == 3) && 3 * (track_smem<kDv1, 5>(cap) + kPerBlock) <= kSm + 1024)
        return launch_one<kDv1, 5, 3>(c, lay, seeds, hit_offsets, seed_offsets, n_events, cap, track_smem<kDv1, 5>(cap), only, out, st, prof);
    if (2 * (track_smem<kDv1, 8>(cap) + kPerBlock) <= kSm + 1024)
        return launch_one<kDv1, 8, 2>(c, lay, seeds, hit_offsets, seed_offsets, n_events, cap, track_smem<kDv1, 8>(cap), only, out, st, prof);
    const size_t fixed = (sizeof(TrackShared<uint16_t, kDv1, 12>) + 15) & ~(size_t)15;
    int cap_max = (int)((kSm - fixed) / 4) & ~3;
    if (cap_max > 65528) cap_max = 65528;
    if (cap > cap_max) cap = cap_max;
    return launch_one<kDv1, 12, 1>(c, lay, seeds, hit_offsets, seed_offsets, n_events, cap, track_smem<kDv1, 12>(cap), only, out, st, prof);
}

cudaError_t launch_track(const DevConst &c, const LayoutPtrs &lay, const ds_seeds &seeds, const int32_t *hit_offsets,
                         const int32_t *seed_offsets, int n_events, int max_event_hits_hint, const int32_t *only,
                         const ds_tracks &out, cudaStream_t st, Prof &prof)
{
    if (n_events <= 0) return cudaSuccess;
    const int hint = max_event_hits_hint > 0 ? max_event_hits_hint : 4096;
    // Dv1 (triplet search, P:107-P:111) and Dv0 are separate instantiations: the Dv0 hot path carries none of the other's code
    return c.dv1 ? launch_track_t<true>(c, lay, seeds, hit_offsets, seed_offsets, n_events, hint, only, out, st, prof)
                 : launch_track_t<false>(c, lay, seeds, hit_offsets, seed_offsets, n_events, hint, only, out, st, prof);
}

}  // namespace ds
