// S1..S6 in ONE kernel, one thread block per event: the block sorts the event's UT hits into (layer, sector, x0 slice) bins
// in shared memory (S1) and goes straight on to the seed extrapolation, window searches, fits and best-candidate choice
// (S2..S6) on the copy it holds -- the sorted arrays, the permutation and the bin table never travel to global memory and
// back (k_layout + k_track: 20 B/hit written and re-read; here every input array is read exactly once, 24 B/hit).
// Paper: hits grouped in Y sectors (P:109-P:111), hits cached in shared memory for the combinatorics, search and
// candidate choice P:93-P:115.  This is the Dv0 hot path of ds_reconstruct; Dv1 and events that do not fit the staging
// capacity take k_layout + k_track (ds_layout.cu, ds_track.cu), which also document the phases of S2..S6.
//
// Phases of a block (T = 32 W threads):
//   load   x0, id, ymin, ymax of the event by 1-D bulk async copies (cp.async.bulk + mbarrier); the event's w array is
//          prefetched into L2 (cp.async.bulk.prefetch.L2): it is read later, only for the few hits that enter a fit
//   A      histogram of the sort bins (layer, sector, x0 slice; kFine = 64 slices per (layer, sector), about one hit each);
//          the counts are 16-bit halves of 32-bit words, atomicAdd returns the hit's arrival slot in its bin; the first hit
//          to arrive in a bin leaves its (ymin, ymax) as the reference of its (layer, sector)
//   B      block-wide exclusive scan -> bin starts = the bin table the searches use (uint16, in place)
//   Y      uniform y bounds?  every hit is compared with the reference of its (layer, sector): if all agree (A-2: a strip's y
//          range is its sector's) y-compatibility is decided once per (seed, sector) and no per-hit bounds are read again
//   C      scatter: x0 in bin order and the permutation src[] (position -> index inside the event).  Inside a bin the hits
//          stay in arrival order: a search looks at every hit of the slices its window touches and picks by the total
//          order (distance, id, index in the caller's arrays), so the result does not depend on that order
//   z      bulk copy of z into the buffer the unsorted x0 leaves free (read through src[]), in flight during the first searches
//   track  S2..S6 by the block's warps, each on its share of the event's seeds (event_chunk)
#include <cstdlib>

#include "ds_sort.cuh"
#include "ds_track.cuh"

namespace ds {

constexpr int kFine = kXBins * kSub;   // x0 slices per (layer, sector) of the sort = of the table the searches use here
constexpr int kFineLog2 = kFine == 64 ? 6 : (kFine == 32 ? 5 : (kFine == 128 ? 7 : -1));
static_assert((1 << kFineLog2) == kFine, "coarse bin = fine bin >> kFineLog2");
constexpr int kEvFirstCap = 64;   // first hits a warp handles per round (96 / 128 / 160 measured: no faster, a round rarely overflows)
static_assert(kEvFirstCap >= DS_MAX_FIRST_HITS && kEvFirstCap <= 512, "a seed's first hits fit a round; f packs into 9 bits");
constexpr int kSelCap = 64;            // hits of an over-full first window that the warp ranks together

// State of one warp of k_event (cf. WarpShared of ds_track.cuh; no fit results are kept: the lane that fits the best
// combination of a seed writes the track record itself)
// What the later phases need of the warp's 32 seeds (SeedRec of ds_track.cuh), one array per field: lanes that read or
// write their own seed, or first hits that read their seeds, then meet no shared-memory bank conflict by layout
struct SeedRecs {
    double xm[32], zm[32], w1[32], y[4][32];
    unsigned short mask[4][32];
    __device__ __forceinline__ SeedRec get(int o) const
    {
        SeedRec r;
        r.xm = xm[o]; r.zm = zm[o]; r.w1 = w1[o];
        r.y[0] = y[0][o]; r.y[1] = y[1][o]; r.y[2] = y[2][o]; r.y[3] = y[3][o];
        r.mask[0] = mask[0][o]; r.mask[1] = mask[1][o]; r.mask[2] = mask[2][o]; r.mask[3] = mask[3][o];
        return r;
    }
};

struct EventWarp {
    SeedRecs rec;
    unsigned long long best_bits[32];     // per seed: smallest score among its fits (bits of the non-negative double)
    uint16_t near[3 * kEvFirstCap][2];      // phase B: closest / second closest hit of (first hit, layer); phase A: ranking lists
    float z3[kEvFirstCap];                  // z of the first hit
    int n_best[32];                       // per seed: fits with that score (+ 2 for every first hit left to the seed's thread)
    int n_fit;                            // fit tasks appended this round (may exceed kFitCap)
    int fit_end;                          // tasks [0, fit_end) are queued; later appends did not fit the queue
    uint16_t slot[32 * kMaxFirst];        // phase A: the seed's first hits (positions in the event's bin-ordered x0)
    unsigned short foff[32];              // where the seed's first hits start in the round's list
    unsigned short fs[kEvFirstCap];         // first-hit list: index into slot[]
    unsigned short ffit[kEvFirstCap];       // first fit task of the first hit (| combinations << 12), kFitNone or kFitInline
    unsigned short task[kFitCap];         // fit task: first hit | i1 << 9 | i2 << 10
};
static_assert(sizeof(EventWarp) % 8 == 0 && sizeof(EventWarp::near) >= kSelCap * (sizeof(double) + sizeof(uint16_t)), "ranking lists fit near[]");

struct EventHead {
    unsigned long long bars[5];
    long long warp_sums[34];
    int nonuni;
    int pad_;
    float2 yb[kLayers * DS_MAX_SECTORS];   // (ymin, ymax) of each (layer, sector)
    double2 ye[kLayers * DS_MAX_SECTORS];  // uniform events: (ymin - y_tol, ymax + y_tol), what a track's y is compared with
};

// Byte offsets of the regions of the dynamic shared memory; cap is a multiple of 8.
//   HI  bin counts, then bin starts: uint16 [nfine + 1] (two per 32-bit word)
//   S   ymin, then x0 in bin order             Z  x0 (staged), then z (staged)
//   Y   ymax, then src (uint16, first half)    P  id, then bin << 20 | slot
//   WS  the warps' lists (S2..S6): from the second half of Y over P, both dead by then
struct EventLayout {
    uint32_t HI, S, Z, Y, P, WS, total;
};

template <int W>
static EventLayout event_layout(int cap, int nfine)
{
    auto up16 = [](size_t v) { return (uint32_t)((v + 15) & ~(size_t)15); };
    EventLayout L;
    const uint32_t c4 = 4 * (uint32_t)cap;
    L.HI = up16(sizeof(EventHead));
    L.S = L.HI + up16(4 * ((size_t)nfine / 2 + 1));
    L.Z = L.S + c4;
    L.Y = L.Z + c4;
    L.P = L.Y + c4;
    L.WS = L.Y + c4 / 2;
    const uint32_t sort_end = L.P + c4, ws_end = L.WS + W * (uint32_t)sizeof(EventWarp);
    L.total = sort_end > ws_end ? sort_end : ws_end;
    return L;
}

__device__ __forceinline__ void stage_words(void *buf, const void *src, int h0, int n, unsigned long long *bar, bool bulk)
{
    stage_field(static_cast<uint32_t *>(buf), static_cast<const uint32_t *>(src), h0, n, bar, bulk);
}

__device__ __forceinline__ void l2_prefetch(const void *p, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// ---- S2..S6 of k_event ---------------------------------------------------------------------------------------------------------
// What the searches of a block share
struct EventCtx {
    HitsFused H;
    const uint16_t *tab;   // bin starts, kFine slices per (layer, sector)
    const float2 *yb;      // (ymin, ymax) of each (layer, sector)
    const double2 *ye;     // (ymin - y_tol, ymax + y_tol) of each (layer, sector)
    bool uni;              // every hit carries the bounds of its (layer, sector)
    int n_hits;            // hits of the event (checked build)
    int rsec;              // sectors looked at on either side of the one a track's y falls into; 0: only the nearer neighbour
};

// Events whose hits do not all carry their sector's bounds (rare: out of line): the sectors a track at height y can touch;
// every hit is then tested with its own bounds
__device__ __forceinline__ unsigned ev_sector_mask_any(const DevConst &c, int layer, double y)
{
    return sector_mask<false>(c, nullptr, layer, y);
}

__device__ __forceinline__ bool ev_y_hit(const DevConst &c, const float *gymin, const float *gymax, int i, double y)
{
    const double lo = (double)gymin[i] - c.y_tol, hi = (double)gymax[i] + c.y_tol;
    return (lo <= y) & (y <= hi);
}

// Bit s set: sector s of `layer` is y-compatible with a track at height y (see sector_mask of ds_track.cuh).  Uniform
// event: the test of O-S3 itself (ymin - y_tol <= y <= ymax + y_tol) on the sectors around the one y falls into.
__device__ __forceinline__ unsigned ev_sector_mask(const DevConst &c, const EventCtx &E, int layer, double y)
{
    if (!E.uni) return ev_sector_mask_any(c, layer, y);
    const double u = (y - c.y0) * c.inv_h;
    const int sc = __double2int_rd(u);   // NaN -> 0: the tests below then fail
    int lo = sc - E.rsec, hi = sc + E.rsec;
    if (E.rsec == 0) {   // y_tol below half a sector: besides its own sector only the neighbour y is nearer to can be compatible
        const bool upper = u - (double)sc >= 0.5;
        lo = upper ? sc : sc - 1;
        hi = upper ? sc + 1 : sc;
    }
    lo = max(lo, 0);
    hi = min(hi, c.n_sectors - 1);
    unsigned m = 0;
#pragma unroll 1
    for (int s = lo; s <= hi; ++s) {
        const double2 b = E.ye[layer * c.n_sectors + s];
        m |= ((b.x <= y) & (y <= b.y)) ? 1u << s : 0u;
    }
    return m;
}

__device__ __forceinline__ bool ev_y_ok(const DevConst &c, const EventCtx &E, int j, double y)
{
    return E.uni || ev_y_hit(c, E.H.gymin, E.H.gymax, (int)E.H.src[j], y);
}

// Positions [a, b) of the slices of (layer, sector) that the (widened, fp32) window of pf touches
__device__ __forceinline__ void ev_slices(const DevConst &c, const EventCtx &E, int layer, int sector, int fl, int fh, int &a, int &b)
{
    const int base = (layer * c.n_sectors + sector) * kFine;
    a = E.tab[base + fl];
    b = E.tab[base + fh + 1];
    DS_ASSERT(fl >= 0 && fl <= fh && fh < kFine && a <= b && b <= E.n_hits);
}

// S4: closest and second closest y-compatible hit of layer l within w1 of the prediction xp; -1 = none
__device__ __forceinline__ int2 ev_search(const DevConst &c, const EventCtx &E, int l, double xp, double y, double w1, unsigned mask)
{
    int j0 = -1, j1 = -1;
    double d0 = 1e300, d1 = 1e300;
    const double off = c.dxdy[l] * y;
    const Prefilter pf = make_prefilter(xp - off, w1);
    const int fl = xslice<kFine>(pf.t - pf.w, c.xb_off, c.xb_scale), fh = xslice<kFine>(pf.t + pf.w, c.xb_off, c.xb_scale);
    for (unsigned m = mask; m; m &= m - 1) {
        int a, b;
        ev_slices(c, E, l, __ffs(m) - 1, fl, fh, a, b);
#pragma unroll 1
        for (int j = a; j < b; ++j) {
            const float xj = E.H.x0[j];
            if (!(fabsf(xj - pf.t) <= pf.w)) continue;
            const double d = fabs(((double)xj + off) - xp);
            if ((d <= w1) && ev_y_ok(c, E, j, y)) {
                if (closer(E.H, d, j, d0, j0)) {
                    d1 = d0; j1 = j0;
                    d0 = d; j0 = j;
                } else if (closer(E.H, d, j, d1, j1)) {
                    d1 = d; j1 = j;
                }
            }
        }
    }
    DS_ASSERT(j0 < E.n_hits && j1 < E.n_hits && (j0 < 0 || j0 != j1));
    return make_int2(j0, j1);
}

// More than max_first hits in a first window and more than the warp ranks together: max_first selection passes by the
// seed's own lane (each pass: the closest hit after the previous pick)
__device__ __noinline__ void ev_select_serial(const DevConst &c, const EventCtx &E, unsigned mask3, int fl, int fh, double off3,
                                              double xc3, double w0, double y3, int max_first, uint16_t *dst)
{
    double last_d = -1.0;
    int last_j = -1;
    for (int k = 0; k < max_first; ++k) {
        double bd = 1e300;
        int bj = -1;
        for (unsigned m = mask3; m; m &= m - 1) {
            int a, b;
            ev_slices(c, E, 3, __ffs(m) - 1, fl, fh, a, b);
            for (int j = a; j < b; ++j) {
                const double d = fabs(((double)E.H.x0[j] + off3) - xc3);
                if ((d <= w0) && ev_y_ok(c, E, j, y3)) {
                    const bool after = last_j < 0 || (j != last_j && closer(E.H, last_d, last_j, d, j));
                    if (after && closer(E.H, d, j, bd, bj)) { bd = d; bj = j; }
                }
            }
        }
        dst[k] = (uint16_t)bj;
        last_d = bd;
        last_j = bj;
    }
}

// S6 output: the track of seed s from its best candidate (state at z_ref; y and ty are the seed's, A-8)
__device__ __forceinline__ void ev_write_track(const DevConst &c, const HitsFused &H, const ds_seeds &seeds, const ds_tracks &out, int s,
                                               const Candidate &best)
{
    const double ys = (double)seeds.y[s], txs = (double)seeds.tx[s], tys = (double)seeds.ty[s];
    out.x[s] = (float)best.a;
    out.y[s] = (float)(ys + tys * (c.z_ref - c.z_seed));
    out.tx[s] = (float)best.b;
    out.ty[s] = (float)tys;
    out.qop[s] = (float)((txs - best.b) / c.kick);
    out.chi2[s] = (float)best.chi2;
    out.nhits[s] = best.nh;
    out.found[s] = 1;
    int4 hv;
    hv.x = best.j0 >= 0 ? hit_perm(H, best.j0) : -1;
    hv.y = best.j1 >= 0 ? hit_perm(H, best.j1) : -1;
    hv.z = best.j2 >= 0 ? hit_perm(H, best.j2) : -1;
    hv.w = hit_perm(H, best.j3);
    reinterpret_cast<int4 *>(out.hit)[s] = hv;
}

// S6 in full for one seed (first hits f0 .. f0+nF-1 of the warp's list, seed in lane o): every combination fitted in turn,
// equal scores resolved by (more hits, ids, indices) (A-9)
__device__ __forceinline__ Candidate ev_choose_general(const DevConst &c, const EventWarp &sh, const HitsFused &H, int f0, int nF, int o)
{
    Candidate best;
    best.score = kNoScore; best.a = 0.0; best.b = 0.0; best.chi2 = 0.0;
    best.nh = 0; best.j0 = -1; best.j1 = -1; best.j2 = -1; best.j3 = -1;
    const SeedRec s2 = sh.rec.get(o);
    for (int k = 0; k < nF; ++k) {
        const int f = f0 + k;
        if (sh.ffit[f] == kFitNone) continue;
        const int j0 = idx_get(sh.near[3 * f][0]), j3 = (int)sh.slot[sh.fs[f]];
        const int j1a = idx_get(sh.near[3 * f + 1][0]), j1b = idx_get(sh.near[3 * f + 1][1]);
        const int j2a = idx_get(sh.near[3 * f + 2][0]), j2b = idx_get(sh.near[3 * f + 2][1]);
        const int m1 = j1b >= 0 ? 2 : 1, m2 = j2b >= 0 ? 2 : 1;
        const int nh = 1 + (j0 >= 0) + (j1a >= 0) + (j2a >= 0);
        for (int i = 0; i < m1 * m2; ++i) {
            const int j1 = i / m2 ? j1b : j1a, j2 = i % m2 ? j2b : j2a;
            const FitRes r = fit_combo(c, H, s2, j0, j1, j2, j3, (double)sh.z3[f], (double)H.gw[H.src[j3]]);
            if (r.score == kNoScore) continue;
            Candidate cand;
            cand.score = r.score; cand.a = r.a; cand.b = r.b; cand.chi2 = r.chi2;
            cand.nh = nh; cand.j0 = j0; cand.j1 = j1; cand.j2 = j2; cand.j3 = j3;
            if (cand.score < best.score || (cand.score == best.score && tie_better(H, cand, best))) best = cand;
        }
    }
    return best;
}

// A first window with more than max_first hits (seed of lane o), by the whole warp: lanes over the hits of the window, every
// passing hit is ranked among all of them by (distance, id, index); the max_first closest go to the seed's slots in that order
__device__ __forceinline__ void ev_select_warp(const DevConst &c, const EventCtx &E, EventWarp &sh, int o, unsigned mask3, float pt, float pw,
                                            double off3, double xc3, double w0, double y3, int max_first)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const HitsFused &H = E.H;
    const int fl = xslice<kFine>(pt - pw, c.xb_off, c.xb_scale), fh = xslice<kFine>(pt + pw, c.xb_off, c.xb_scale);
    double *cd = reinterpret_cast<double *>(&sh.near[0][0]);          // near[] is free in phase A: the distances,
    uint16_t *cj = reinterpret_cast<uint16_t *>(cd + kSelCap);        //                            the hits
    int n_list = 0;
    for (unsigned m = mask3; m; m &= m - 1) {
        int a, b;
        ev_slices(c, E, 3, __ffs(m) - 1, fl, fh, a, b);
        for (int jb = a; jb < b; jb += 32) {
            const int j = jb + lane;
            bool pass = false;
            double d = 0.0;
            if (j < b) {
                d = fabs(((double)H.x0[j] + off3) - xc3);
                pass = (d <= w0) && ev_y_ok(c, E, j, y3);
            }
            const unsigned pm = __ballot_sync(FULL, pass);
            const int at = n_list + __popc(pm & lanemask_lt());
            if (pass && at < kSelCap) { cj[at] = (uint16_t)j; cd[at] = d; }
            n_list += __popc(pm);
        }
    }
    __syncwarp();
    if (n_list > kSelCap) {
        if (lane == o) ev_select_serial(c, E, mask3, fl, fh, off3, xc3, w0, y3, max_first, sh.slot + o * kMaxFirst);
    } else {
        for (int i = lane; i < n_list; i += 32) {
            const double di = cd[i];
            const int ji = cj[i];
            int rank = 0;
            for (int q = 0; q < n_list; ++q) rank += (q != i && closer(H, cd[q], (int)cj[q], di, ji)) ? 1 : 0;
            DS_ASSERT(rank >= 0 && rank < n_list);
            if (rank < max_first) sh.slot[o * kMaxFirst + rank] = (uint16_t)ji;
        }
    }
    __syncwarp();
}

__device__ __forceinline__ void ev_general_track(const DevConst &c, const EventWarp &sh, const HitsFused &H, const ds_seeds &seeds,
                                              const ds_tracks &out, int s, int f0, int nF, int o)
{
    const Candidate best = ev_choose_general(c, sh, H, f0, nF, o);
    if (best.score == kNoScore) write_not_found(out, s);
    else ev_write_track(c, H, seeds, out, s, best);
}

// Seeds [cb, ce) (at most 32) of the event, by one warp on its own, in rounds of the phases of track_chunk (ds_track.cuh):
//   A  lane per seed: S2, first window in UTbX (S3); a window with more than max_first hits is ranked by the whole warp
//   B  lane per first hit: the three refined windows (S4), the lane queues the fits
//   F  lane per queued combination: fit (S5); the lane that holds a seed's one best fit writes the track record (S6)
//   C  lane per seed: seeds without a track; seeds with exact score ties or more combinations than the queue holds
__device__ __forceinline__ void event_chunk(const DevConst &c, EventWarp &sh, const EventCtx &E, const ds_seeds &seeds,
                                            int cb, int ce, const ds_tracks &out, const SeedPre &pre)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int max_first = c.max_first;
    const HitsFused &H = E.H;
    uint16_t *my_slot = sh.slot + lane * kMaxFirst;
    int s_base = cb;
    while (s_base < ce) {
        // ---- phase A -----------------------------------------------------------------------------------------------------------
        const int s = s_base + lane;
        const bool act = s < ce;
        int nF = 0;
        double a_xc3 = 0.0, a_off3 = 0.0, a_w0 = 0.0, a_y3 = 0.0;   // the window, kept for the warp's ranking
        unsigned a_mask3 = 0;
        float a_pt = 0.f, a_pw = 0.f;
        if (lane == 0) { sh.n_fit = 0; sh.fit_end = kFitCap; }
        sh.best_bits[lane] = (unsigned long long)__double_as_longlong(kNoScore);
        sh.n_best[lane] = 0;
        if (act) {
            const SeedPre sp = pre.s == s ? pre : load_seed(seeds, s, true);
            const S2 s2 = extrapolate_seed(c, sp.x, sp.y, sp.tx, sp.ty, sp.qop);
            SeedRecs &r = sh.rec;
            r.xm[lane] = s2.xm; r.zm[lane] = s2.zm; r.w1[lane] = s2.w1;
            r.y[0][lane] = s2.y0; r.y[1][lane] = s2.y1; r.y[2][lane] = s2.y2; r.y[3][lane] = s2.y3;
#pragma unroll 1
            for (int l = 0; l < 4; ++l) r.mask[l][lane] = (unsigned short)ev_sector_mask(c, E, l, r.y[l][lane]);
            a_mask3 = r.mask[3][lane];
            a_y3 = s2.y3; a_xc3 = s2.xc3; a_w0 = s2.w0;
            a_off3 = c.dxdy[3] * s2.y3;
            const Prefilter pf = make_prefilter(a_xc3 - a_off3, a_w0);
            a_pt = pf.t; a_pw = pf.w;
            const int fl = xslice<kFine>(pf.t - pf.w, c.xb_off, c.xb_scale), fh = xslice<kFine>(pf.t + pf.w, c.xb_off, c.xb_scale);
            for (unsigned m = a_mask3; m; m &= m - 1) {
                int a, b;
                ev_slices(c, E, 3, __ffs(m) - 1, fl, fh, a, b);
#pragma unroll 1
                for (int j = a; j < b; ++j) {
                    const float xj = H.x0[j];
                    if (!(fabsf(xj - pf.t) <= pf.w)) continue;
                    const double d = fabs(((double)xj + a_off3) - a_xc3);
                    if ((d <= a_w0) && ev_y_ok(c, E, j, a_y3)) {
                        if (nF < max_first) my_slot[nF] = (uint16_t)j;
                        ++nF;
                    }
                }
            }
        }
        // more hits in a window than are tried: the max_first closest by (distance, id).  The warp takes these
        // seeds one by one: lanes over the hits of the window, every passing hit is ranked among all of them
        for (unsigned over = __ballot_sync(FULL, nF > max_first); over; over &= over - 1) {
            const int o = __ffs(over) - 1;
            const double xc3 = __shfl_sync(FULL, a_xc3, o), off3 = __shfl_sync(FULL, a_off3, o), w0 = __shfl_sync(FULL, a_w0, o),
                         y3 = __shfl_sync(FULL, a_y3, o);
            const unsigned mask3 = __shfl_sync(FULL, a_mask3, o);
            const float pt = __shfl_sync(FULL, a_pt, o), pw = __shfl_sync(FULL, a_pw, o);
            ev_select_warp(c, E, sh, o, mask3, pt, pw, off3, xc3, w0, y3, max_first);
        }
        hits_zw_ready(H);
        const int nFc = min(nF, max_first);
        int incl = nFc;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += t;
        }
        // the seeds taken this round are the longest prefix whose first hits fit the list
        const bool take = act && incl <= kEvFirstCap;
        const unsigned take_mask = __ballot_sync(FULL, take);
        const int n_take = __popc(take_mask);
        const int n_first = __shfl_sync(FULL, incl, n_take - 1);
        if (take) {
            const int pos = incl - nFc;
            sh.foff[lane] = (unsigned short)pos;
            for (int k = 0; k < nFc; ++k) {
                DS_ASSERT(pos + k < kEvFirstCap && (int)my_slot[k] < E.n_hits);
                sh.fs[pos + k] = (unsigned short)(lane * kMaxFirst + k);
                sh.z3[pos + k] = hit_z(H, (int)my_slot[k]);
            }
        }
        __syncwarp();
        // ---- phase B -----------------------------------------------------------------------------------------------------------
        for (int fb = 0; fb < n_first; fb += 32) {
            const int f = fb + lane;
            if (f < n_first) {
                const int sl = sh.fs[f], o = sl / kMaxFirst;
                const int j3 = (int)sh.slot[sl];
                const SeedRecs &t2 = sh.rec;
                const double xm = t2.xm[o], zm = t2.zm[o], w1 = t2.w1[o];
                // trajectory through (first hit, magnet point), refined windows
                const double x3 = (double)H.x0[j3] + c.dxdy[3] * t2.y[3][o];
                const double txc = (x3 - xm) / ((double)sh.z3[f] - zm);
                int nh = 1, m1 = 1, m2 = 1;
#pragma unroll 1
                for (int l = 0; l < 3; ++l) {
                    const double xp = xm + txc * (c.z_layer[l] - zm);
                    int2 r = ev_search(c, E, l, xp, t2.y[l][o], w1, (unsigned)t2.mask[l][o]);
                    if (l == 0) r.y = -1;   // UTaX keeps the closest hit only
                    *reinterpret_cast<uint32_t *>(&sh.near[3 * f + l][0]) = ((uint32_t)r.x & 0xffffu) | ((uint32_t)r.y << 16);
                    if (r.x >= 0) { hit_prefetch(H, r.x); ++nh; }
                    if (r.y >= 0) { hit_prefetch(H, r.y); if (l == 1) m1 = 2; else m2 = 2; }
                }
                unsigned short ff = kFitNone;
                if (nh >= c.min_hits) {
                    hit_prefetch(H, j3);
                    const int base = atomicAdd(&sh.n_fit, m1 * m2);
                    if (base + m1 * m2 <= kFitCap) {
                        DS_ASSERT(base >= 0 && f < 512);
                        ff = (unsigned short)(base | ((m1 * m2) << 12));
                        for (int i1 = 0; i1 < m1; ++i1)
                            for (int i2 = 0; i2 < m2; ++i2)
                                sh.task[base + i1 * m2 + i2] = (unsigned short)(f | (i1 << 9) | (i2 << 10));
                    } else {
                        ff = kFitInline;
                        atomicMin(&sh.fit_end, base);
                        atomicAdd(&sh.n_best[o], 2);
                    }
                }
                sh.ffit[f] = ff;
            }
        }
        __syncwarp();
        // ---- fit phase: lane per queued combination; the lane with a seed's one best fit writes its track record ---------------------
        const int n_fit = min(sh.n_fit, sh.fit_end);
        {
            unsigned long long bits = (unsigned long long)__double_as_longlong(kNoScore);
            int o = 0;
            Candidate cand;
            cand.score = kNoScore;
            if (lane < n_fit) {
                const int tk = sh.task[lane], f = tk & 511, i1 = (tk >> 9) & 1, i2 = (tk >> 10) & 1;
                const int sl = sh.fs[f];
                o = sl / kMaxFirst;
                cand.j0 = idx_get(sh.near[3 * f][0]);
                cand.j1 = idx_get(sh.near[3 * f + 1][i1]);
                cand.j2 = idx_get(sh.near[3 * f + 2][i2]);
                cand.j3 = (int)sh.slot[sl];
                cand.nh = 1 + (cand.j0 >= 0) + (cand.j1 >= 0) + (cand.j2 >= 0);
                const FitRes r = fit_combo(c, H, sh.rec.get(o), cand.j0, cand.j1, cand.j2, cand.j3, (double)sh.z3[f], (double)H.gw[H.src[cand.j3]]);
                cand.score = r.score; cand.a = r.a; cand.b = r.b; cand.chi2 = r.chi2;
                if (r.score != kNoScore) {
                    bits = (unsigned long long)__double_as_longlong(r.score);   // scores are >= +0: bit order = value order
                    atomicMin(&sh.best_bits[o], bits);
                }
            }
            __syncwarp();
            const bool top = cand.score != kNoScore && bits == sh.best_bits[o];
            if (top) atomicAdd(&sh.n_best[o], 1);
            __syncwarp();
            // one fit with the smallest score and every combination of the seed queued: that is the track
            if (top && sh.n_best[o] == 1) ev_write_track(c, H, seeds, out, s_base + o, cand);
        }
        // ---- phase C: seeds without a track; exact score ties and fits that were not queued: the general comparison ---------
        if (take) {
            const int nb = sh.n_best[lane];
            if (nb == 0) {
                write_not_found(out, s);
            } else if (nb >= 2) {
                ev_general_track(c, sh, H, seeds, out, s, sh.foff[lane], nFc, lane);
            }
        }
        s_base += n_take;
        __syncwarp();   // the lists are rewritten by the next round
    }
}

// ---- the sort passes over four neighbouring elements k0 .. k0+3 of the staged buffers (element i of the event sits at index
//      d + i; kFull: all four belong to the event, which is every group but the first and the last) ---------------------------
template <bool kFull>
__device__ __forceinline__ void ev_hist4(const DevConst &c, uint32_t *hist, float2 *yb, int32_t *b_p, const float *b_z, const float *b_s,
                                         const float *b_y, int k0, int d, int kend)
{
    const int4 id4 = *reinterpret_cast<const int4 *>(b_p + k0);
    const float4 x4 = *reinterpret_cast<const float4 *>(b_z + k0), lo4 = *reinterpret_cast<const float4 *>(b_s + k0),
                 hi4 = *reinterpret_cast<const float4 *>(b_y + k0);
    const int idv[4] = {id4.x, id4.y, id4.z, id4.w};
    const float xv[4] = {x4.x, x4.y, x4.z, x4.w}, lov[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hiv[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
    int pk[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int k = k0 + u;
        pk[u] = 0;
        if (kFull || (k >= d && k < kend)) {
            const int b = fine_bin(c, idv[u], xv[u]);
            const int sh16 = (b & 1) * 16;
            const uint32_t old = atomicAdd(&hist[b >> 1], 1u << sh16);
            const uint32_t slot = (old >> sh16) & 0xffffu;
            DS_ASSERT(b >= 0 && b < c.n_bins * kSub && slot < 0xffffu);
            pk[u] = (int)(((uint32_t)b << 20) | slot);
            if (slot == 0) yb[b >> kFineLog2] = make_float2(lov[u], hiv[u]);   // reference bounds of the (layer, sector)
        }
    }
    *reinterpret_cast<int4 *>(b_p + k0) = make_int4(pk[0], pk[1], pk[2], pk[3]);
}

template <bool kFull>
__device__ __forceinline__ bool ev_check4(const float2 *yb, const int32_t *b_p, const float *b_s, const float *b_y, int k0, int d, int kend)
{
    const int4 pk4 = *reinterpret_cast<const int4 *>(b_p + k0);
    const float4 lo4 = *reinterpret_cast<const float4 *>(b_s + k0), hi4 = *reinterpret_cast<const float4 *>(b_y + k0);
    const int pkv[4] = {pk4.x, pk4.y, pk4.z, pk4.w};
    const float lov[4] = {lo4.x, lo4.y, lo4.z, lo4.w}, hiv[4] = {hi4.x, hi4.y, hi4.z, hi4.w};
    bool differs = false;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int k = k0 + u;
        const float2 r = yb[(uint32_t)pkv[u] >> (20 + kFineLog2)];
        differs |= (kFull || (k >= d && k < kend)) & ((lov[u] != r.x) | (hiv[u] != r.y));
    }
    return differs;
}

template <bool kFull>
__device__ __forceinline__ void ev_scatter4(const uint16_t *tab, const int32_t *b_p, const float *b_z, float *b_s, uint16_t *src, int k0,
                                            int d, int kend)
{
    const int4 pk4 = *reinterpret_cast<const int4 *>(b_p + k0);
    const float4 x4 = *reinterpret_cast<const float4 *>(b_z + k0);
    const uint32_t pkv[4] = {(uint32_t)pk4.x, (uint32_t)pk4.y, (uint32_t)pk4.z, (uint32_t)pk4.w};
    const float xv[4] = {x4.x, x4.y, x4.z, x4.w};
    int pos[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) pos[u] = (int)tab[pkv[u] >> 20] + (int)(pkv[u] & 0xfffffu);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int k = k0 + u;
        if (kFull || (k >= d && k < kend)) {
            DS_ASSERT(pos[u] >= 0 && pos[u] < kend - d);
            b_s[pos[u]] = xv[u];
            src[pos[u]] = (uint16_t)(k - d);
        }
    }
}

// ---- the kernel -------------------------------------------------------------------------------------------------------------------
template <int W, int kMinBlocks>
__global__ void __launch_bounds__(32 * W, kMinBlocks)
k_event(const __grid_constant__ DevConst c, const ds_hits hits, const ds_seeds seeds, const int32_t *__restrict__ hit_offsets,
        const int32_t *__restrict__ seed_offsets, const ds_tracks out, const EventLayout L, int cap, int bulk,
        int32_t *__restrict__ redo)
{
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int T = 32 * W;
    const int e = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int s_begin = seed_offsets[e], s_end = seed_offsets[e + 1];
    const int h0 = hit_offsets[e], n = hit_offsets[e + 1] - h0;
    // an event without seeds has no output; an event above the staging capacity is left to k_layout + k_track
    const bool mine = s_begin == s_end || n + 3 <= cap;
    if (tid == 0) redo[e] = mine ? 0 : 1;
    if (s_begin == s_end || !mine) return;

    const int nfine = c.n_bins * kSub, nw = nfine / 2;   // nw words hold the nfine counts; word nw takes the total
    EventHead &hd = *reinterpret_cast<EventHead *>(smem);
    uint32_t *hist = reinterpret_cast<uint32_t *>(smem + L.HI);
    float *b_s = reinterpret_cast<float *>(smem + L.S);
    float *b_z = reinterpret_cast<float *>(smem + L.Z);
    float *b_y = reinterpret_cast<float *>(smem + L.Y);
    int32_t *b_p = reinterpret_cast<int32_t *>(smem + L.P);
    uint16_t *src = reinterpret_cast<uint16_t *>(b_y);
    const uint16_t *tab = reinterpret_cast<const uint16_t *>(hist);
    const bool stagers = !bulk || tid < 64;   // a bulk copy is issued by thread 0, the few elements after it by threads 32..34
    const int d = h0 & 3, kend = d + n;   // element i of the event sits at index d + i of a staged buffer

    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < 5; ++k) mbar_init(&hd.bars[k], 1);
        hd.nonuni = 0;
        if (bulk && n > 0) {   // w is read much later, for fitted hits only: bring the event's slice into L2 now;
            const int a0 = h0 & ~3, a1 = (h0 + n) & ~3;       // whole 16-byte groups inside the arrays
            if (a1 > a0) {
                l2_prefetch(hits.w + a0, 4u * (uint32_t)(a1 - a0));
                l2_prefetch(hits.z + a0, 4u * (uint32_t)(a1 - a0));
            }   // z follows once the unsorted x0 has left its buffer
        }
    }
    for (int k = tid; k < (nw + 4) / 4; k += T) reinterpret_cast<uint4 *>(hist)[k] = make_uint4(0u, 0u, 0u, 0u);
    if (tid < kLayers * DS_MAX_SECTORS) hd.yb[tid] = make_float2(0.f, 0.f);
    __syncthreads();
    if (stagers) stage_words(b_z, hits.x0, h0, n, &hd.bars[0], bulk != 0);
    if (stagers) stage_words(b_p, hits.id, h0, n, &hd.bars[1], bulk != 0);
    if (stagers) stage_words(b_s, hits.ymin, h0, n, &hd.bars[2], bulk != 0);
    if (stagers) stage_words(b_y, hits.ymax, h0, n, &hd.bars[3], bulk != 0);
    // the lane's first seed, fetched now so that the load is in flight with the hits
    SeedPre pre;
    {
        const int chunk = seed_chunk<W>(s_begin, s_end);
        const int s = s_begin + wid * chunk + lane;
        pre = load_seed(seeds, s, lane < chunk && s < s_end);
    }
    __syncthreads();   // the elements after the last 16-byte boundary were stored by ordinary stores
#pragma unroll
    for (int k = 0; k < 4; ++k) mbar_wait(&hd.bars[k], 0);
    // ---- A: histogram; a thread takes four neighbouring elements of the staged buffers at a time (ev_hist4) -------------------
    for (int k0 = 4 * tid; k0 < kend; k0 += 4 * T) {
        if (k0 >= d && k0 + 4 <= kend) ev_hist4<true>(c, hist, hd.yb, b_p, b_z, b_s, b_y, k0, d, kend);
        else ev_hist4<false>(c, hist, hd.yb, b_p, b_z, b_s, b_y, k0, d, kend);
    }
    __syncthreads();
    // ---- B: exclusive scan of the counts, two 16-bit counts per word -> bin starts ---------------------------------------------
    {
        // a thread takes per4 neighbouring groups of four words (128-bit accesses; 12 words apart for 160 threads and 14
        // sectors: no bank conflict) and keeps them in registers between the two passes
        constexpr int kQ = (4 * DS_MAX_SECTORS * kFine / 8 + T - 1) / T;
        const int nq = nw / 4, per4 = (nq + T - 1) / T;
        uint4 *h4 = reinterpret_cast<uint4 *>(hist);
        uint4 q[kQ];
        uint32_t sum = 0;
#pragma unroll
        for (int u = 0; u < kQ; ++u) {
            const int idx = tid * per4 + u;
            q[u] = (u < per4 && idx < nq) ? h4[idx] : make_uint4(0u, 0u, 0u, 0u);
            sum += (q[u].x & 0xffffu) + (q[u].x >> 16) + (q[u].y & 0xffffu) + (q[u].y >> 16) + (q[u].z & 0xffffu) + (q[u].z >> 16) +
                   (q[u].w & 0xffffu) + (q[u].w >> 16);
        }
        uint32_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        int *ws = reinterpret_cast<int *>(hd.warp_sums);
        if (lane == 31) ws[wid] = (int)inc;
        __syncthreads();
        uint32_t run = inc - sum;
        for (int w = 0; w < wid; ++w) run += (uint32_t)ws[w];
        auto scan_word = [&run](uint32_t w) {
            const uint32_t c0 = w & 0xffffu, c1 = w >> 16, r = run | ((run + c0) << 16);
            run += c0 + c1;
            return r;
        };
#pragma unroll
        for (int u = 0; u < kQ; ++u) {
            const int idx = tid * per4 + u;
            uint4 r;
            r.x = scan_word(q[u].x); r.y = scan_word(q[u].y); r.z = scan_word(q[u].z); r.w = scan_word(q[u].w);
            if (u < per4 && idx < nq) h4[idx] = r;
        }
        if (tid == T - 1) hist[nw] = run;   // tab[nfine] = n
    }
    __syncthreads();
    // ---- Y: does every hit carry the bounds of its (layer, sector)? ------------------------------------------------------------------
    {
        bool differs = false;
        for (int k0 = 4 * tid; k0 < kend; k0 += 4 * T) {
            if (k0 >= d && k0 + 4 <= kend) differs |= ev_check4<true>(hd.yb, b_p, b_s, b_y, k0, d, kend);
            else differs |= ev_check4<false>(hd.yb, b_p, b_s, b_y, k0, d, kend);
        }
        if (differs) hd.nonuni = 1;
    }
    __syncthreads();   // ymin and ymax are dead from here: their buffers take the x0 in bin order and src
    // ---- C: scatter into bin order ------------------------------------------------------------------------------------------------
    for (int k0 = 4 * tid; k0 < kend; k0 += 4 * T) {
        if (k0 >= d && k0 + 4 <= kend) ev_scatter4<true>(tab, b_p, b_z, b_s, src, k0, d, kend);
        else ev_scatter4<false>(tab, b_p, b_z, b_s, src, k0, d, kend);
    }
    if (tid < kLayers * DS_MAX_SECTORS) {
        const float2 b = hd.yb[tid];
        hd.ye[tid] = make_double2((double)b.x - c.y_tol, (double)b.y + c.y_tol);
    }
    __syncthreads();
    // the unsorted x0 is dead: its buffer takes z (by index inside the event); the searches start while it is in flight
    if (stagers) stage_words(b_z, hits.z, h0, n, &hd.bars[4], bulk != 0);
    __syncthreads();   // its last elements come by ordinary stores

    // ---- S2..S6 on the shared-memory copy ---------------------------------------------------------------------------------------------
    EventCtx E;
    E.H.x0 = b_s; E.H.src = src; E.H.z = b_z + d;
    E.H.gw = hits.w + h0; E.H.gymin = hits.ymin + h0; E.H.gymax = hits.ymax + h0; E.H.gid = hits.id + h0; E.H.h0 = h0;
    E.H.zbar = &hd.bars[4];
    E.tab = tab;
    E.yb = hd.yb;
    E.ye = hd.ye;
    E.uni = hd.nonuni == 0;
    E.n_hits = n;
    DS_ASSERT((int)tab[nfine] == n && (int)tab[0] == 0);
    E.rsec = (c.y_rsec == 1 && c.y_tol * c.inv_h < 0.5) ? 0 : c.y_rsec;
    EventWarp *warps = reinterpret_cast<EventWarp *>(smem + L.WS);
    const int chunk = seed_chunk<W>(s_begin, s_end);
    for (int cb = s_begin + wid * chunk; cb < s_end; cb += W * chunk)
        event_chunk(c, warps[wid], E, seeds, cb, min(cb + chunk, s_end), out, pre);
}

// Development aid: DS_EVENT_W=6|7 runs the 3-blocks-per-SM configuration with that many warps per block
static int event_warps_override()
{
    static int v = -1;
    if (v < 0) {
        const char *e = getenv("DS_EVENT_W");
        v = e ? atoi(e) : 0;
    }
    return v;
}

template <int W, int kMinBlocks>
static cudaError_t launch_event_one(const DevConst &c, const ds_hits &hits, const ds_seeds &seeds, const int32_t *hit_offsets,
                                    const int32_t *seed_offsets, int n_events, int cap, size_t smem, int bulk, const ds_tracks &out,
                                    int32_t *redo, cudaStream_t st, Prof &prof)
{
    static unsigned long long opted = 0;
    const cudaError_t aerr = opt_in_max_smem(k_event<W, kMinBlocks>, &opted);
    if (aerr != cudaSuccess) return aerr;
    prof.begin(DS_K_EVENT, st);
    k_event<W, kMinBlocks><<<n_events, 32 * W, smem, st>>>(c, hits, seeds, hit_offsets, seed_offsets, out, event_layout<W>(cap, c.n_bins * kSub),
                                                           cap, bulk, redo);
    prof.end(st);
    return cudaGetLastError();
}

cudaError_t launch_event(const DevConst &c, const ds_hits &hits, const ds_seeds &seeds, const int32_t *hit_offsets,
                         const int32_t *seed_offsets, int n_events, int max_event_hits_hint, const ds_tracks &out, int32_t *redo,
                         cudaStream_t st, Prof &prof)
{
    if (n_events <= 0) return cudaSuccess;
    const int hint = max_event_hits_hint > 0 ? max_event_hits_hint : 4096;
    int cap = ((hint + 7) & ~7) + 8;   // a multiple of 8 with room for the alignment slack
    const int nfine = c.n_bins * kSub;
    const size_t kSm = 227 * 1024, kPerBlock = 1024;   // usable shared memory of an SM; reserved per resident block
    const uintptr_t bits = reinterpret_cast<uintptr_t>(hits.x0) | reinterpret_cast<uintptr_t>(hits.z) |
                           reinterpret_cast<uintptr_t>(hits.ymin) | reinterpret_cast<uintptr_t>(hits.ymax) |
                           reinterpret_cast<uintptr_t>(hits.w) | reinterpret_cast<uintptr_t>(hits.id);
    const int bulk = (bits & 15) == 0;
    const int want = event_warps_override();
    size_t sm = event_layout<7>(cap, nfine).total;
    if (want == 7 && 3 * (sm + kPerBlock) <= kSm + 1024)
        return launch_event_one<7, 3>(c, hits, seeds, hit_offsets, seed_offsets, n_events, cap, sm, bulk, out, redo, st, prof);
    sm = event_layout<6>(cap, nfine).total;
    if (want == 6 && 3 * (sm + kPerBlock) <= kSm + 1024)
        return launch_event_one<6, 3>(c, hits, seeds, hit_offsets, seed_offsets, n_events, cap, sm, bulk, out, redo, st, prof);
    sm = event_layout<5>(cap, nfine).total;
    if (3 * (sm + kPerBlock) <= kSm + 1024)
        return launch_event_one<5, 3>(c, hits, seeds, hit_offsets, seed_offsets, n_events, cap, sm, bulk, out, redo, st, prof);
    // two blocks per SM: the largest capacity that still fits them (event_kernel_wanted has checked that the hint does)
    while (2 * (event_layout<8>(cap, nfine).total + kPerBlock) > kSm + 1024) cap -= 8;
    sm = event_layout<8>(cap, nfine).total;
    return launch_event_one<8, 2>(c, hits, seeds, hit_offsets, seed_offsets, n_events, cap, sm, bulk, out, redo, st, prof);
}

// k_event pays when at least two blocks share an SM (one block's loads and sort overlap the other's searches).  Events so
// large that only one would fit (cfg2-like, 8 000 hits: measured 0.36 ms per 1000 events against 0.33 ms) run k_layout +
// k_track, whose sort has the SM's full thread count to itself.
bool event_kernel_wanted(const DevConst &c, int max_event_hits_hint)
{
    const int hint = max_event_hits_hint > 0 ? max_event_hits_hint : 4096;
    const int cap = ((hint + 7) & ~7) + 8;
    const size_t kSm = 227 * 1024, kPerBlock = 1024;
    return 2 * (event_layout<8>(cap, c.n_bins * kSub).total + kPerBlock) <= kSm + 1024;
}

}  // namespace ds
