// S2..S6 device code shared by k_track (ds_track.cu: after k_layout, hits in the sorted global layout) and k_event
// (ds_event.cu: S1 in the same block, hits in shared memory).  See ds_track.cu for the mapping of the work.
#pragma once

#include "ds_common.cuh"

namespace ds {

constexpr int kMaxBins = 4 * DS_MAX_SECTORS * kXBins;

struct S2 {
    double zm, xm, ym, y0, y1, y2, y3, txp, xc3, w0, w1;
};

// S2 (thin-kick model: BASELINE cfg0)
__device__ __forceinline__ S2 extrapolate_seed(const DevConst &c, double xs, double ys, double txs, double tys,
                                               double qop)
{
    S2 r;
    r.zm = c.zmag_c[0] + c.zmag_c[1] * tys * tys + c.zmag_c[2] * txs * txs + c.zmag_c[3] * qop * qop;
    r.xm = xs + txs * (r.zm - c.z_seed);
    r.ym = ys + tys * (r.zm - c.z_seed);
    r.y0 = ys + tys * (c.z_layer[0] - c.z_seed);
    r.y1 = ys + tys * (c.z_layer[1] - c.z_seed);
    r.y2 = ys + tys * (c.z_layer[2] - c.z_seed);
    r.y3 = ys + tys * (c.z_layer[3] - c.z_seed);
    r.txp = txs - c.kick * qop;
    r.xc3 = r.xm + r.txp * (c.z_layer[3] - r.zm);
    r.w0 = fmin(c.w0_max, c.w0_a + c.w0_b * fabs(qop));
    r.w1 = c.w1_a + c.w1_b * fabs(qop);
    return r;
}

// Sectors whose y range, widened by y_tol, contains y (a superset: every hit is re-checked with its own ymin/ymax).
__device__ __forceinline__ void sector_range(const DevConst &c, double y, int &s_lo, int &s_hi)
{
    const double u = (y - c.y0) * c.inv_h, t = c.y_tol * c.inv_h;
    double lo = ceil(u - t - 1.0 - 1e-9), hi = floor(u + t + 1e-9);
    lo = fmax(lo, 0.0);
    hi = fmin(hi, (double)(c.n_sectors - 1));
    if (!(lo <= hi)) { s_lo = 0; s_hi = -1; return; }   // also catches NaN
    s_lo = (int)lo;
    s_hi = (int)hi;
}

// Bit s set: sector s of `layer` is y-compatible with a track at height y.  kUni (every hit of the event carries the bounds
// yb[layer * n_sectors + s] of its sector): the test of O-S3 itself, ymin - y_tol <= y <= ymax + y_tol, once per sector.
// Otherwise the superset of sector_range; every hit is then tested with its own bounds.
template <bool kUni>
__device__ __forceinline__ unsigned sector_mask(const DevConst &c, const float2 *yb, int layer, double y)
{
    int lo, hi;
    sector_range(c, y, lo, hi);
    unsigned m = 0;
    for (int s = lo; s <= hi; ++s) {
        if (kUni) {
            const float2 b = yb[layer * c.n_sectors + s];
            const double ylo = (double)b.x - c.y_tol, yhi = (double)b.y + c.y_tol;
            m |= ((ylo <= y) & (y <= yhi)) ? 1u << s : 0u;
        } else {
            m |= 1u << s;
        }
    }
    return m;
}

// Positions [a, b) (relative to the event) of the x0 slices of (layer, sector) that the x0 interval [lo, hi] touches.
template <typename TabT>
__device__ __forceinline__ void slice_range(const DevConst &c, const TabT &tab, int layer, int sector, double lo,
                                            double hi, int &a, int &b)
{
    const int base = (layer * c.n_sectors + sector) * TabT::kSlices;
    const int xl = xslice<TabT::kSlices>(__double2float_rd(lo), c.xb_off, c.xb_scale);
    const int xh = xslice<TabT::kSlices>(__double2float_ru(hi), c.xb_off, c.xb_scale);
    a = tab[base + xl];
    b = tab[base + xh + 1];
}


constexpr int kFirstCap = 64;    // first hits a warp handles per round (>= DS_MAX_FIRST_HITS)
constexpr int kFitCap = 32;      // fits of the warp's fit phase per round; the rest are fitted by the seed's thread
constexpr double kNoScore = 1e300;
constexpr unsigned short kFitNone = 0xffffu, kFitInline = 0xfffeu;

struct FitRes {
    double score, a, b, chi2;   // score = kNoScore: the combination fails the chi2/ndf cut
};

// State of one warp of k_track: the warp takes up to 32 seeds of the event through all phases on its own.  Idx is the
// type hit positions inside the event are stored in: uint16_t when the event is staged (it then has < 65535 hits),
// int otherwise.  (Idx)-1 = none.
// What the later phases need of a seed (S2, computed once in phase A): magnet point, y at the four planes, refined
// window half-width, and the mask of y-compatible sectors of each layer (sector_mask).
struct SeedRec {
    double xm, zm, w1, y[4];
    unsigned short mask[4];
};
static_assert(sizeof(SeedRec) == 64 && DS_MAX_SECTORS <= 16, "sector masks are 16 bits");

// Dv1 only: the (seed, UTbX hit) items
template <typename Idx, bool kDv1>
struct DvShared {};
template <typename Idx>
struct DvShared<Idx, true> {
    int dv_off[32], dv_a[32];             // first item and first UTbX candidate of the seed
    float cand_z[kFirstCap];              // items that passed the fp32 pre-test: z of the UTbX hit,
    Idx cand_j3[kFirstCap];               //      the hit,
    unsigned char cand_o[kFirstCap];      //      the seed (lane)
};

template <typename Idx, bool kDv1>
struct WarpShared : DvShared<Idx, kDv1> {
    FitRes res[kFitCap];                  // fit phase: result of fit task i
    SeedRec rec[32];
    float2 zw3[kFirstCap];                // (z, w) of the first hit
    int n_fit;                            // fit tasks appended this round (may exceed kFitCap)
    int fit_end;                          // tasks [0, fit_end) are queued; later appends did not fit the queue
    Idx slot[32 * kMaxFirst];             // phase A: the seed's first hits (positions in the event's sorted slice)
    Idx near[3 * kFirstCap][2];           // phase B: closest / second closest hit of (first hit, layer)
    unsigned short foff[32];              // where the seed's first hits start in the round's list
    unsigned short fs[kFirstCap];         // first-hit list: index into slot[]
    unsigned short ffit[kFirstCap];       // first fit task of the first hit (| combinations << 12), kFitNone or kFitInline
    unsigned short task[kFitCap];         // fit task: first hit | i1 << 9 | i2 << 10
    unsigned long long best_bits[32];     // per seed: smallest score among its fits (bits of the non-negative double)
    int best_fit[32];                     // per seed: first fit task with that score
    int n_best[32];                       // per seed: fits with that score (+ 2 for every first hit left to the seed's thread)
    // Dv1 keeps at most kFirstCap triplets in slot[]; the rest of it holds the fit queue (4 per triplet)
    __device__ __forceinline__ unsigned short *dv_task_ptr() { return reinterpret_cast<unsigned short *>(slot + kFirstCap); }
};
static_assert((32 * kMaxFirst - kFirstCap) * 2 >= 4 * kFirstCap * 2, "slot[] holds the Dv1 triplets and their fit queue");

// The event's hits as the searches see them.  Two layouts; every function below is a template on the layout (HitsT) and
// reaches the hit fields only through x0[] and the accessors hit_zw / hit_z / hit_perm / hit_id / hit_ymin / hit_ymax /
// hit_prefetch.  Indices are relative to the event's sorted slice.
// HitsSorted (k_track after k_layout): x0 from the staging buffer (or global for an oversize event), the rest from the
// sorted global arrays: per-hit y bounds (read only when the event is not uniform) and the aux record (z, w, perm, id).
struct HitsSorted {
    const float *x0;             // shared or global
    const float *ymin, *ymax;    // global
    const float4 *aux;           // global
};

__device__ __forceinline__ float2 hit_zw(const HitsSorted &H, int j) { return *reinterpret_cast<const float2 *>(H.aux + j); }
__device__ __forceinline__ float hit_z(const HitsSorted &H, int j) { return H.aux[j].x; }
__device__ __forceinline__ int hit_perm(const HitsSorted &H, int j) { return __float_as_int(H.aux[j].z); }
__device__ __forceinline__ int hit_id(const HitsSorted &H, int j) { return __float_as_int(H.aux[j].w); }
__device__ __forceinline__ float hit_ymin(const HitsSorted &H, int j) { return H.ymin[j]; }
__device__ __forceinline__ float hit_ymax(const HitsSorted &H, int j) { return H.ymax[j]; }

// z, w, id and perm of a hit live in global memory and are read only for hits that passed a window -- a phase later than
// the window test that picked them.  The test issues an L1 prefetch so that the later read does not wait on DRAM.
__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
__device__ __forceinline__ void hit_prefetch(const HitsSorted &H, int j) { prefetch_l1(H.aux + j); }
// (z, w) of a first hit as phase A keeps it, and its w as the fit wants it
__device__ __forceinline__ float2 first_zw(const HitsSorted &H, int j) { return hit_zw(H, j); }
__device__ __forceinline__ float first_w(const HitsSorted &, float2 zw, int) { return zw.y; }
// called by every warp before its first read of z or w
__device__ __forceinline__ void hits_zw_ready(const HitsSorted &) {}

// HitsFused (k_event: S1 runs in the same block): sorted x0, the sort permutation src[] (sorted position -> index inside
// the event) and z (by index inside the event) in shared memory; w, id and the per-hit y bounds from the caller's unsorted
// arrays through src[] (w only for fitted hits, id only on exact ties, bounds only in events that are not uniform).
struct HitsFused {
    const float *x0;             // shared, sorted
    const uint16_t *src;         // shared
    const float *z;              // shared, by index inside the event (the staging offset is folded into the pointer)
    const float *gw, *gymin, *gymax;   // global: the event's slice of the caller's arrays
    const int32_t *gid;          // global: the event's slice
    int h0;                      // first hit of the event in the caller's arrays
    unsigned long long *zbar;    // mbarrier the bulk copy of z completes on (phase 0)
};

__device__ __forceinline__ float2 hit_zw(const HitsFused &H, int j) { const int i = H.src[j]; return make_float2(H.z[i], H.gw[i]); }
__device__ __forceinline__ float hit_z(const HitsFused &H, int j) { return H.z[H.src[j]]; }
__device__ __forceinline__ int hit_perm(const HitsFused &H, int j) { return H.h0 + (int)H.src[j]; }
__device__ __forceinline__ int hit_id(const HitsFused &H, int j) { return H.gid[H.src[j]]; }
__device__ __forceinline__ float hit_ymin(const HitsFused &H, int j) { return H.gymin[H.src[j]]; }
__device__ __forceinline__ float hit_ymax(const HitsFused &H, int j) { return H.gymax[H.src[j]]; }
__device__ __forceinline__ void hit_prefetch(const HitsFused &H, int j) { prefetch_l1(H.gw + H.src[j]); }
// phase A keeps z only (shared memory); w comes from global memory when (and if) the first hit enters a fit
__device__ __forceinline__ float2 first_zw(const HitsFused &H, int j) { return make_float2(hit_z(H, j), 0.f); }
__device__ __forceinline__ float first_w(const HitsFused &H, float2, int j) { return H.gw[H.src[j]]; }
// z is still in flight when the searches start (they only look at x0): wait for its bulk copy
__device__ __forceinline__ void hits_zw_ready(const HitsFused &H) { mbar_wait(H.zbar, 0); }

// The event's bin table: positions (relative to the event) where the x0 slices of each (layer, sector) start.  kSlices
// slices per (layer, sector): DS_XBINS in the table k_layout writes, kXBins * kSub in the sort histogram of k_event.
// kSorted: the hits of a slice are in (x0, id, index) order (k_layout); otherwise only the slices are ordered (k_event: a
// slice holds about one hit, and every hit of the slices a window touches is looked at -- no order inside is needed).
template <typename T, int kSlices_, bool kSorted_>
struct BinTable {
    static constexpr int kSlices = kSlices_;
    static constexpr bool kSorted = kSorted_;
    const T *p;
    __device__ __forceinline__ int operator[](int i) const { return (int)p[i]; }
};

template <typename Idx>
__device__ __forceinline__ int idx_get(Idx v) { return v == (Idx)-1 ? -1 : (int)v; }

// y-compatibility of hit j (O-S3: ymin - y_tol <= y <= ymax + y_tol); no short circuit: both loads are always issued.
// kUni: decided per sector already (sector_mask), nothing to read.
template <bool kUni, typename HitsT>
__device__ __forceinline__ bool y_compatible(const DevConst &c, const HitsT &H, int j, double y)
{
    if (kUni) return true;
    const double lo = (double)hit_ymin(H, j) - c.y_tol, hi = (double)hit_ymax(H, j) + c.y_tol;
    return (lo <= y) & (y <= hi);
}

// Equal distances: smaller id, then (duplicates) the hit that comes first in the caller's arrays
template <typename HitsT>
__device__ __forceinline__ bool closer_tie(const HitsT &H, int j1, int j2)
{
    const int i1 = hit_id(H, j1), i2 = hit_id(H, j2);
    if (i1 != i2) return i1 < i2;
    return hit_perm(H, j1) < hit_perm(H, j2);
}

// (distance, id, index in the caller's arrays) order of the "closest hits" rules: a total order, so the result does
// not depend on the order the hits are looked at; ids are only read on an exact distance tie
template <typename HitsT>
__device__ __forceinline__ bool closer(const HitsT &H, double d1, int j1, double d2, int j2)
{
    if (d1 != d2) return d1 < d2;
    if (j2 < 0) return true;
    return closer_tie(H, j1, j2);
}

// fp32 superset test of "|x0 + off - x| <= w" (decided in fp64 afterwards): |x0 - t| <= w', with t = (float)(x - off)
// and w' = w widened by far more than the fp32 rounding of the difference (a few ulp of |t|)
struct Prefilter {
    float t, w;
};

__device__ __forceinline__ Prefilter make_prefilter(double target_x0, double w)
{
    Prefilter p;
    p.t = (float)target_x0;
    p.w = (float)w * 1.0001f + 0.01f + 2e-6f * fabsf(p.t);
    return p;
}

// First position in [a, b) of the x0-sorted slice whose x0 is not below xl
__device__ __forceinline__ int lower_bound_x0(const float *x0, int a, int b, float xl)
{
    while (a < b) {
        const int mid = (a + b) >> 1;
        if (x0[mid] < xl) a = mid + 1; else b = mid;
    }
    return a;
}

// S4: closest and second closest y-compatible hit of layer l (sectors tl..th) within w1 of the prediction xp;
// -1 = none.  Inside a sector the hits are x0-sorted: binary search to the lower edge of the (fp32, widened) window,
// then only the hits inside it are looked at in fp64.
template <bool kUni, typename HitsT, typename TabT>
__device__ __forceinline__ int2 search_layer(const DevConst &c, const HitsT &H, const TabT &tab, int l, double xp,
                                             double y, double w1, unsigned mask)
{
    int j0 = -1, j1 = -1;
    double d0 = 1e300, d1 = 1e300;
    const double off = c.dxdy[l] * y;
    const double lo = xp - off - w1, hi = xp - off + w1;
    const Prefilter pf = make_prefilter(xp - off, w1);
    const float xl = pf.t - pf.w, xh = pf.t + pf.w;
    for (unsigned m = mask; m; m &= m - 1) {
        const int sec = __ffs(m) - 1;
        int a, b;
        slice_range(c, tab, l, sec, lo, hi, a, b);
        int j = TabT::kSorted ? lower_bound_x0(H.x0, a, b, xl) : a;
        for (; j < b; ++j) {
            const float xj = H.x0[j];
            if (TabT::kSorted) { if (!(xj <= xh)) break; }
            else if (!(fabsf(xj - pf.t) <= pf.w)) continue;
            const double d = fabs(((double)xj + off) - xp);
            const bool pass = (d <= w1) & y_compatible<kUni>(c, H, j, y);
            if (pass) {
                if (closer(H, d, j, d0, j0)) {
                    d1 = d0; j1 = j0;
                    d0 = d; j0 = j;
                } else if (closer(H, d, j, d1, j1)) {
                    d1 = d; j1 = j;
                }
            }
        }
    }
    return make_int2(j0, j1);
}

// The max_first closest of the more than max_first hits in the first window, by (distance, id), for a window
// that touches one or two sectors: every sector is an x0-sorted range, so the closest hits are found by walking
// outwards from the window centre, one left and one right head per sector, always taking the closest head.  Returns
// false (dst not valid) when it meets equal x0 on a left side, where the walk order is not the id order.
template <bool kUni, typename Idx, typename HitsT, typename TabT>
__device__ __noinline__ bool select_first_walk(const DevConst &c, const HitsT &H, const TabT &tab, int sec_a, int sec_b,
                                               double off3, double xc, double w0, double y, int max_first, Idx *dst)
{
    int hj[4], hend[4];
    double hd[4];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        int A = 0, B = 0;
        const int sec = k ? sec_b : sec_a;   // -1: none
        if (sec >= 0) {
            const int base = (3 * c.n_sectors + sec) * TabT::kSlices;
            A = tab[base];
            B = tab[base + TabT::kSlices];
        }
        int lo = A, hi = B;   // first j in [A, B) with x0[j] + off3 >= xc
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if ((double)H.x0[mid] + off3 >= xc) hi = mid; else lo = mid + 1;
        }
        hj[2 * k] = lo - 1; hend[2 * k] = A - 1;
        hj[2 * k + 1] = lo; hend[2 * k + 1] = B;
    }
    // move head h to the next y-compatible hit inside the window (or to its end)
    auto settle = [&](int &j, int end, int step, double &d) {
        for (; j != end; j += step) {
            d = fabs(((double)H.x0[j] + off3) - xc);
            if (d > w0) { j = end; break; }
            if (y_compatible<kUni>(c, H, j, y)) break;
        }
    };
#pragma unroll
    for (int h = 0; h < 4; ++h) { hd[h] = 1e300; settle(hj[h], hend[h], (h & 1) ? 1 : -1, hd[h]); }
    for (int k = 0; k < max_first; ++k) {
        int pick = -1, pj = -1;
        double pd = 1e300;
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            if (hj[h] != hend[h] && (pick < 0 || closer(H, hd[h], hj[h], pd, pj))) { pick = h; pj = hj[h]; pd = hd[h]; }
        }
        if (pick < 0) return false;   // fewer hits than the caller counted: cannot happen
        dst[k] = (Idx)pj;
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            if (h == pick) {
                if (!(h & 1) && pj - 1 != hend[h] && H.x0[pj - 1] == H.x0[pj]) return false;
                hj[h] += (h & 1) ? 1 : -1;
                settle(hj[h], hend[h], (h & 1) ? 1 : -1, hd[h]);
            }
        }
    }
    return true;
}

// A candidate: fit result and chosen hits (positions in the event's sorted slice, -1 = layer missing)
struct Candidate {
    double score, a, b, chi2;   // score = kNoScore: none
    int nh, j0, j1, j2, j3;
};

// A-9 order of two candidates with the same score: more hits, then smaller (id3, id0, id1, id2); missing = INT32_MAX
template <typename HitsT>
__device__ __noinline__ bool tie_better(const HitsT &H, const Candidate &p, const Candidate &q)
{
    if (p.nh != q.nh) return p.nh > q.nh;
    const int pj[4] = {p.j3, p.j0, p.j1, p.j2}, qj[4] = {q.j3, q.j0, q.j1, q.j2};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int pi = pj[k] >= 0 ? hit_id(H, pj[k]) : INT32_MAX, qi = qj[k] >= 0 ? hit_id(H, qj[k]) : INT32_MAX;
        if (pi != qi) return pi < qi;
    }
    // the same ids (duplicate hits): the candidate whose hits come first in the caller's arrays
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int pi = pj[k] >= 0 ? hit_perm(H, pj[k]) : INT32_MAX, qi = qj[k] >= 0 ? hit_perm(H, qj[k]) : INT32_MAX;
        if (pi != qi) return pi < qi;
    }
    return false;
}

// S5: weighted straight line x(z - z_ref) through the first hit (z3, w3 given), the refined-window hits j0, j1, j2
// (-1 = missing) and the magnet point as pseudo-measurement (A-8); chi2; chi2/ndf cut and score (A-9)
template <typename HitsT>
__device__ __forceinline__ FitRes fit_combo(const DevConst &c, const HitsT &H, const SeedRec &s2, int j0, int j1, int j2,
                                            int j3, double z3, double w3)
{
    // all loads first (z, w come from global memory)
    const int k0 = max(j0, 0), k1 = max(j1, 0), k2 = max(j2, 0);
    const float2 zw0 = hit_zw(H, k0), zw1 = hit_zw(H, k1), zw2 = hit_zw(H, k2);
    const float fz0 = zw0.x, fw0 = zw0.y, fz1 = zw1.x, fw1 = zw1.y, fz2 = zw2.x, fw2 = zw2.y;
    const float fx0 = H.x0[k0], fx1 = H.x0[k1], fx2 = H.x0[k2], fx3 = H.x0[j3];
    const bool u0 = j0 >= 0, u1 = j1 >= 0, u2 = j2 >= 0;
    const int nh = 1 + u0 + u1 + u2;
    const double pz[5] = {u0 ? (double)fz0 - c.z_ref : 0.0, u1 ? (double)fz1 - c.z_ref : 0.0,
                          u2 ? (double)fz2 - c.z_ref : 0.0, z3 - c.z_ref, s2.zm - c.z_ref};
    const double px[5] = {u0 ? (double)fx0 + c.dxdy[0] * s2.y[0] : 0.0, u1 ? (double)fx1 + c.dxdy[1] * s2.y[1] : 0.0,
                          u2 ? (double)fx2 + c.dxdy[2] * s2.y[2] : 0.0, (double)fx3 + c.dxdy[3] * s2.y[3], s2.xm};
    const double pw[5] = {u0 ? (double)fw0 : 0.0, u1 ? (double)fw1 : 0.0, u2 ? (double)fw2 : 0.0, w3, c.w_mag};
    double S = 0, Sz = 0, Szz = 0, Sx = 0, Sxz = 0;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        S += pw[k];
        Sz += pw[k] * pz[k];
        Szz += pw[k] * pz[k] * pz[k];
        Sx += pw[k] * px[k];
        Sxz += pw[k] * px[k] * pz[k];
    }
    const double D = S * Szz - Sz * Sz;
    FitRes r;
    r.b = (S * Sxz - Sz * Sx) / D;
    r.a = (Szz * Sx - Sz * Sxz) / D;
    double chi2 = 0.0;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const double e = px[k] - r.a - r.b * pz[k];
        chi2 += pw[k] * e * e;
    }
    r.chi2 = chi2;
    const double ndf = (double)(nh - 1);
    r.score = (chi2 / ndf <= c.chi2ndf_max) ? chi2 + c.miss_penalty * (double)(4 - nh) : kNoScore;
    return r;
}

__device__ __forceinline__ void write_not_found(const ds_tracks &out, int64_t s)
{
    out.x[s] = 0.f; out.y[s] = 0.f; out.tx[s] = 0.f; out.ty[s] = 0.f; out.qop[s] = 0.f; out.chi2[s] = 0.f;
    out.nhits[s] = 0; out.found[s] = 0;
    reinterpret_cast<int4 *>(out.hit)[s] = make_int4(-1, -1, -1, -1);
}

// S6 in full for one seed (first hits f0 .. f0+nF-1 of the warp's list, seed in lane o): every combination in turn,
// equal scores resolved by (more hits, ids) (A-9), combinations that the fit phase did not take fitted here.
template <typename Idx, bool kDv1, typename HitsT>
__device__ __noinline__ Candidate choose_general(const DevConst &c, const WarpShared<Idx, kDv1> &sh, const HitsT &H, int f0,
                                                 int nF, int o)
{
    Candidate best;
    best.score = kNoScore; best.a = 0.0; best.b = 0.0; best.chi2 = 0.0;
    best.nh = 0; best.j0 = -1; best.j1 = -1; best.j2 = -1; best.j3 = -1;
    const SeedRec &s2 = sh.rec[o];
    for (int k = 0; k < nF; ++k) {
        const int f = f0 + k;
        const unsigned short ff = sh.ffit[f];
        if (ff == kFitNone) continue;
        const int j0 = idx_get(sh.near[3 * f][0]), j3 = (int)sh.slot[sh.fs[f]];
        const int j1a = idx_get(sh.near[3 * f + 1][0]), j1b = idx_get(sh.near[3 * f + 1][1]);
        const int j2a = idx_get(sh.near[3 * f + 2][0]), j2b = idx_get(sh.near[3 * f + 2][1]);
        const int m1 = j1b >= 0 ? 2 : 1, m2 = j2b >= 0 ? 2 : 1;
        const int nh = 1 + (j0 >= 0) + (j1a >= 0) + (j2a >= 0);
        for (int i1 = 0; i1 < m1; ++i1) {
            for (int i2 = 0; i2 < m2; ++i2) {
                const int j1 = i1 ? j1b : j1a, j2 = i2 ? j2b : j2a;
                const FitRes r = ff != kFitInline ? sh.res[(ff & 0xfff) + i1 * m2 + i2]
                                                  : fit_combo(c, H, s2, j0, j1, j2, j3, (double)sh.zw3[f].x, (double)first_w(H, sh.zw3[f], j3));
                if (r.score == kNoScore) continue;
                Candidate cand;
                cand.score = r.score; cand.a = r.a; cand.b = r.b; cand.chi2 = r.chi2;
                cand.nh = nh; cand.j0 = j0; cand.j1 = j1; cand.j2 = j2; cand.j3 = j3;
                if (cand.score < best.score || (cand.score == best.score && tie_better(H, cand, best))) best = cand;
            }
        }
    }
    return best;
}

// A lane's seed state, read before the block waits for its table and hits (the loads overlap that wait)
struct SeedPre {
    float x, y, tx, ty, qop;
    int s;   // the seed these values belong to, -1 = none
};

__device__ __forceinline__ SeedPre load_seed(const ds_seeds &seeds, int s, bool valid)
{
    SeedPre p;
    p.s = valid ? s : -1;
    p.x = valid ? seeds.x[s] : 0.f; p.y = valid ? seeds.y[s] : 0.f; p.tx = valid ? seeds.tx[s] : 0.f;
    p.ty = valid ? seeds.ty[s] : 0.f; p.qop = valid ? seeds.qop[s] : 0.f;
    return p;
}

// Seeds [cb, ce) (at most 32) of one event, by one warp on its own: rounds of
//   A  lane per seed:       S2, first window in UTbX (S3) -> the seed's <= max_first first hits; warp scan of the counts
//   B  three lanes per first hit, one per layer: refined windows (S4); the first lane of the three queues the fits
//   F  lane per queued combination: fit (S5)
//   C  lane per seed:       best candidate (S6), track record
// A round takes the longest prefix of the remaining seeds whose first hits fit the warp's list.
template <typename Idx, bool kUni, typename HitsT, typename TabT>
__device__ __forceinline__ void track_chunk(const DevConst &c, WarpShared<Idx, false> &sh, const TabT &tab, const float2 *yb,
                                            const HitsT &H, const ds_seeds &seeds, int cb, int ce, const ds_tracks &out,
                                            const SeedPre &pre)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int max_first = c.max_first;
    Idx *my_slot = sh.slot + lane * kMaxFirst;
    int s_base = cb;
    while (s_base < ce) {
        // ---- phase A: lane per seed -- S2, S3 ----------------------------------------------------------------------------
        const int s = s_base + lane;
        const bool act = s < ce;
        int nF = 0;
        float fy = 0.f, ftx = 0.f, fty = 0.f;   // kept for the track record (phase C)
        if (lane == 0) { sh.n_fit = 0; sh.fit_end = kFitCap; }
        sh.best_bits[lane] = (unsigned long long)__double_as_longlong(kNoScore);
        sh.best_fit[lane] = INT32_MAX;
        sh.n_best[lane] = 0;
        if (act) {
            const SeedPre sp = pre.s == s ? pre : load_seed(seeds, s, true);
            const float fx = sp.x, fq = sp.qop;
            fy = sp.y; ftx = sp.tx; fty = sp.ty;
            const S2 s2 = extrapolate_seed(c, fx, fy, ftx, fty, fq);
            const unsigned mask3 = sector_mask<kUni>(c, yb, 3, s2.y3);
            {
                SeedRec &r = sh.rec[lane];
                r.xm = s2.xm; r.zm = s2.zm; r.w1 = s2.w1;
                r.y[0] = s2.y0; r.y[1] = s2.y1; r.y[2] = s2.y2; r.y[3] = s2.y3;
#pragma unroll
                for (int l = 0; l < 3; ++l)
                    r.mask[l] = (unsigned short)sector_mask<kUni>(c, yb, l, l == 0 ? s2.y0 : (l == 1 ? s2.y1 : s2.y2));
                r.mask[3] = (unsigned short)mask3;
            }
            const double off3 = c.dxdy[3] * s2.y3;
            const double lo3 = s2.xc3 - off3 - s2.w0, hi3 = s2.xc3 - off3 + s2.w0;
            const Prefilter pf = make_prefilter(s2.xc3 - off3, s2.w0);
            const float xl = pf.t - pf.w, xh = pf.t + pf.w;
            for (unsigned m = mask3; m; m &= m - 1) {
                const int sec = __ffs(m) - 1;
                int a, b;
                slice_range(c, tab, 3, sec, lo3, hi3, a, b);
                int j = TabT::kSorted ? lower_bound_x0(H.x0, a, b, xl) : a;
                for (; j < b; ++j) {
                    const float xj = H.x0[j];
                    if (TabT::kSorted) { if (!(xj <= xh)) break; }
                    else if (!(fabsf(xj - pf.t) <= pf.w)) continue;
                    const double d = fabs(((double)xj + off3) - s2.xc3);
                    if ((d <= s2.w0) & y_compatible<kUni>(c, H, j, s2.y3)) {
                        if (nF < max_first) {
                            my_slot[nF] = (Idx)j;
                            hit_prefetch(H, j);
                        }
                        ++nF;
                    }
                }
            }
            if (nF > max_first) {
                // more hits in the window than are tried: the max_first closest by (distance, id)
                bool done = false;
                if (TabT::kSorted && __popc(mask3) <= 2) {
                    const int sec_a = __ffs(mask3) - 1, sec_b = __ffs(mask3 & (mask3 - 1)) - 1;
                    done = select_first_walk<kUni, Idx>(c, H, tab, sec_a, sec_b, off3, s2.xc3, s2.w0, s2.y3, max_first, my_slot);
                }
                if (!done) {   // general case: max_first selection passes over the window
                    double last_d = -1.0;
                    int last_j = -1;
                    for (int k = 0; k < max_first; ++k) {
                        double bd = 1e300;
                        int bj = -1;
                        for (unsigned m = mask3; m; m &= m - 1) {
                            const int sec = __ffs(m) - 1;
                            int a, b;
                            slice_range(c, tab, 3, sec, lo3, hi3, a, b);
                            for (int j = a; j < b; ++j) {
                                const double d = fabs(((double)H.x0[j] + off3) - s2.xc3);
                                if ((d <= s2.w0) & y_compatible<kUni>(c, H, j, s2.y3)) {
                                    // strictly after the previous pick, and before the best so far
                                    const bool after = last_j < 0 || (j != last_j && closer(H, last_d, last_j, d, j));
                                    if (after && closer(H, d, j, bd, bj)) { bd = d; bj = j; }
                                }
                            }
                        }
                        my_slot[k] = (Idx)bj;
                        last_d = bd;
                        last_j = bj;
                    }
                }
            }
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
        const bool take = act && incl <= kFirstCap;
        const unsigned take_mask = __ballot_sync(FULL, take);
        const int n_take = __popc(take_mask);
        const int n_first = __shfl_sync(FULL, incl, n_take - 1);
        if (take) {
            const int pos = incl - nFc;
            sh.foff[lane] = (unsigned short)pos;
            for (int k0 = 0; k0 < nFc; k0 += 5) {   // (z, w) of the first hits: five loads in flight at a time
                float2 v[5];
#pragma unroll
                for (int u = 0; u < 5; ++u) v[u] = first_zw(H, (int)my_slot[min(k0 + u, nFc - 1)]);
#pragma unroll
                for (int u = 0; u < 5; ++u) {
                    if (k0 + u < nFc) {
                        sh.fs[pos + k0 + u] = (unsigned short)(lane * kMaxFirst + k0 + u);
                        sh.zw3[pos + k0 + u] = v[u];
                    }
                }
            }
        }
        __syncwarp();
        // ---- phase B: lane per first hit -- S4 in UTaX, UTaU, UTbV one after the other; the lane queues the fits --------------
        for (int fb = 0; fb < n_first; fb += 32) {
            const int f = fb + lane;
            if (f < n_first) {
                const int sl = sh.fs[f], o = sl / kMaxFirst;
                const int j3 = (int)sh.slot[sl];
                const SeedRec &t2 = sh.rec[o];
                // trajectory through (first hit, magnet point), refined windows
                const double x3 = (double)H.x0[j3] + c.dxdy[3] * t2.y[3];
                const double txc = (x3 - t2.xm) / ((double)sh.zw3[f].x - t2.zm);
                int2 r[3];
#pragma unroll
                for (int l = 0; l < 3; ++l) {
                    const double xp = t2.xm + txc * (c.z_layer[l] - t2.zm);
                    r[l] = search_layer<kUni>(c, H, tab, l, xp, t2.y[l], t2.w1, (unsigned)t2.mask[l]);
                }
                r[0].y = -1;   // UTaX keeps the closest hit only
#pragma unroll
                for (int l = 0; l < 3; ++l) {
                    sh.near[3 * f + l][0] = (Idx)r[l].x;
                    sh.near[3 * f + l][1] = (Idx)r[l].y;
                    if (r[l].x >= 0) hit_prefetch(H, r[l].x);
                    if (r[l].y >= 0) hit_prefetch(H, r[l].y);
                }
                const int nh = 1 + (r[0].x >= 0) + (r[1].x >= 0) + (r[2].x >= 0);
                unsigned short ff = kFitNone;
                if (nh >= c.min_hits) {
                    const int m1 = r[1].y >= 0 ? 2 : 1, m2 = r[2].y >= 0 ? 2 : 1;
                    const int base = atomicAdd(&sh.n_fit, m1 * m2);
                    if (base + m1 * m2 <= kFitCap) {
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
        // ---- fit phase: lane per queued combination -- S5; per seed the smallest score, its first fit and how many share it
        const int n_fit = min(sh.n_fit, sh.fit_end);
        {
            unsigned long long bits = (unsigned long long)__double_as_longlong(kNoScore);
            int o = 0;
            if (lane < n_fit) {
                const int tk = sh.task[lane], f = tk & 511, i1 = (tk >> 9) & 1, i2 = (tk >> 10) & 1;
                const int sl = sh.fs[f];
                o = sl / kMaxFirst;
                const float2 zw = sh.zw3[f];
                const FitRes r = fit_combo(c, H, sh.rec[o], idx_get(sh.near[3 * f][0]), idx_get(sh.near[3 * f + 1][i1]),
                                           idx_get(sh.near[3 * f + 2][i2]), (int)sh.slot[sl], (double)zw.x,
                                           (double)first_w(H, zw, (int)sh.slot[sl]));
                sh.res[lane] = r;
                if (r.score != kNoScore) {
                    bits = (unsigned long long)__double_as_longlong(r.score);   // scores are >= +0: bit order = value order
                    atomicMin(&sh.best_bits[o], bits);
                }
            }
            __syncwarp();
            if (lane < n_fit && bits != (unsigned long long)__double_as_longlong(kNoScore) && bits == sh.best_bits[o]) {
                atomicMin(&sh.best_fit[o], lane);
                atomicAdd(&sh.n_best[o], 1);
            }
        }
        __syncwarp();
        // ---- phase C: lane per seed -- S6 and the track record -----------------------------------------------------------
        if (take) {
            const int f0 = sh.foff[lane];
            // one fit with the smallest score: that is the track; exact ties and fits that were not queued go through the
            // general comparison
            const int nb = sh.n_best[lane];
            const bool general = nb >= 2;
            const int bt = nb == 1 ? sh.best_fit[lane] : -1;
            Candidate best;
            best.score = kNoScore;
            if (general) {
                best = choose_general<Idx, false>(c, sh, H, f0, nFc, lane);
            } else if (bt >= 0) {
                const FitRes r = sh.res[bt];
                const int tk = sh.task[bt], bf = tk & 511, i1 = (tk >> 9) & 1, i2 = (tk >> 10) & 1;
                best.score = r.score; best.a = r.a; best.b = r.b; best.chi2 = r.chi2;
                best.j0 = idx_get(sh.near[3 * bf][0]);
                best.j1 = idx_get(sh.near[3 * bf + 1][i1]);
                best.j2 = idx_get(sh.near[3 * bf + 2][i2]);
                best.j3 = (int)sh.slot[sh.fs[bf]];
                best.nh = 1 + (best.j0 >= 0) + (best.j1 >= 0) + (best.j2 >= 0);
            }
            if (best.score == kNoScore) {
                write_not_found(out, s);
            } else {
                const double ys = (double)fy, txs = (double)ftx, tys = (double)fty;
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
        }
        s_base += n_take;
        __syncwarp();   // the lists are rewritten by the next round
    }
}

// ---- Dv1 (P:107-P:111, reading A-32): triplet search ---------------------------------------------------
// No first window: every UTbX hit of the seed's y-compatible sectors starts a candidate, and the candidate needs a UTaX
// hit collinear (within w1) with that hit and the magnet point -- the triplet.  The sectors s_lo..s_hi of UTbX are one
// contiguous range of the sorted slice, so a seed's candidates are (range start, count); the warp walks the items
// (seed, UTbX hit) of its <= 32 seeds 32 at a time:
//   T  lane per item: y-compatibility of the UTbX hit, trajectory through it and the magnet point, UTaX search;
//      items with a UTaX hit are compacted into the triplet list (the first-hit list of Dv0, filled by ballots)
//   whenever >= 32 triplets wait (and at the end):
//   S  two lanes per triplet, UTaU / UTbV searches (closest 2); the lane of UTaU queues the <= 4 fits
//   F  lane per queued fit, 32 at a time; per seed the best fit of the window (atomicMin on the score bits) is compared
//      by the seed's lane with the best candidate it holds so far (exact ties: full (hits, ids) comparison)
// and each seed's lane writes its track record at the end.
template <typename Idx>
__device__ __forceinline__ Candidate make_candidate(const WarpShared<Idx, true> &sh, const FitRes &r, int tk)
{
    const int f = tk & 511, i1 = (tk >> 9) & 1, i2 = (tk >> 10) & 1;
    Candidate cand;
    cand.score = r.score; cand.a = r.a; cand.b = r.b; cand.chi2 = r.chi2;
    cand.j0 = idx_get(sh.near[3 * f][0]);
    cand.j1 = idx_get(sh.near[3 * f + 1][i1]);
    cand.j2 = idx_get(sh.near[3 * f + 2][i2]);
    cand.j3 = (int)sh.slot[f];
    cand.nh = 1 + (cand.j0 >= 0) + (cand.j1 >= 0) + (cand.j2 >= 0);
    return cand;
}

template <typename Idx, typename HitsT>
__device__ __forceinline__ FitRes fit_task(const DevConst &c, const WarpShared<Idx, true> &sh, const HitsT &H, int tk)
{
    const int f = tk & 511, i1 = (tk >> 9) & 1, i2 = (tk >> 10) & 1;
    const int j3 = (int)sh.slot[f];
    return fit_combo(c, H, sh.rec[sh.fs[f]], idx_get(sh.near[3 * f][0]), idx_get(sh.near[3 * f + 1][i1]),
                     idx_get(sh.near[3 * f + 2][i2]), j3, (double)sh.zw3[f].x, (double)hit_zw(H, j3).y);
}

// S + F for the triplets [0, n_trip) of the warp's list (fs = owner lane, slot = UTbX hit, near[3f] = UTaX hit, zw3);
// `best` is the candidate the calling lane's seed holds so far.
template <typename Idx, bool kUni, typename HitsT, typename TabT>
__device__ __forceinline__ void dv1_flush(const DevConst &c, WarpShared<Idx, true> &sh, const TabT &tab, const HitsT &H,
                                          int n_trip, Candidate &best)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    if (lane == 0) sh.n_fit = 0;
    __syncwarp();
    // ---- S: stereo layers, two lanes per triplet ---------------------------------------------------------------------------
    for (int fb = 0; fb < n_trip; fb += 16) {
        const int g = lane >> 1, l = 1 + (lane & 1);
        const int f = fb + g;
        const bool on = f < n_trip;
        int2 r = make_int2(-1, -1);
        if (on) {
            const SeedRec &t2 = sh.rec[sh.fs[f]];
            const int j3 = (int)sh.slot[f];
            const double x3 = (double)H.x0[j3] + c.dxdy[3] * t2.y[3];
            const double txc = (x3 - t2.xm) / ((double)sh.zw3[f].x - t2.zm);
            const double xp = t2.xm + txc * (c.z_layer[l] - t2.zm);
            r = search_layer<kUni>(c, H, tab, l, xp, t2.y[l], t2.w1, (unsigned)t2.mask[l]);
            sh.near[3 * f + l][0] = (Idx)r.x;
            sh.near[3 * f + l][1] = (Idx)r.y;
        }
        const unsigned has1 = __ballot_sync(FULL, r.x >= 0), has2 = __ballot_sync(FULL, r.y >= 0);
        if (on && l == 1) {
            const int nh = 2 + ((has1 >> (2 * g)) & 1) + ((has1 >> (2 * g + 1)) & 1);   // UTbX + UTaX + stereo hits
            if (nh >= c.min_hits) {
                const int m1 = 1 + ((has2 >> (2 * g)) & 1), m2 = 1 + ((has2 >> (2 * g + 1)) & 1);
                const int base = atomicAdd(&sh.n_fit, m1 * m2);
                for (int i1 = 0; i1 < m1; ++i1)
                    for (int i2 = 0; i2 < m2; ++i2)
                        sh.dv_task_ptr()[base + i1 * m2 + i2] = (unsigned short)(f | (i1 << 9) | (i2 << 10));
            }
        }
    }
    __syncwarp();
    // ---- F: fits, 32 at a time; per seed the best of the window against the seed's best so far ---------------------------------
    const int n_fit = sh.n_fit;
    for (int tb = 0; tb < n_fit; tb += 32) {
        sh.best_bits[lane] = (unsigned long long)__double_as_longlong(kNoScore);
        sh.best_fit[lane] = INT32_MAX;
        sh.n_best[lane] = 0;
        __syncwarp();
        const int t = tb + lane;
        unsigned long long bits = (unsigned long long)__double_as_longlong(kNoScore);
        int o = 0, tk = 0;
        FitRes r;
        r.score = kNoScore;
        if (t < n_fit) {
            tk = sh.dv_task_ptr()[t];
            o = sh.fs[tk & 511];
            r = fit_task<Idx>(c, sh, H, tk);
            if (r.score != kNoScore) {
                bits = (unsigned long long)__double_as_longlong(r.score);
                atomicMin(&sh.best_bits[o], bits);
            }
        }
        __syncwarp();
        const bool top = t < n_fit && r.score != kNoScore && bits == sh.best_bits[o];
        if (top) {
            atomicMin(&sh.best_fit[o], lane);
            atomicAdd(&sh.n_best[o], 1);
        }
        __syncwarp();
        if (top && sh.best_fit[o] == lane) sh.res[o] = r;   // the window's best fit of seed o (first of equal ones)
        __syncwarp();
        const int nb = sh.n_best[lane];
        if (nb == 1) {
            const Candidate cand = make_candidate<Idx>(sh, sh.res[lane], sh.dv_task_ptr()[tb + sh.best_fit[lane]]);
            if (cand.score < best.score || (cand.score == best.score && tie_better(H, cand, best))) best = cand;
        } else if (nb >= 2) {   // equal scores inside the window: every fit of this seed once more, full comparison
            for (int q = tb; q < min(tb + 32, n_fit); ++q) {
                const int tq = sh.dv_task_ptr()[q];
                if (sh.fs[tq & 511] != lane) continue;
                const FitRes rq = fit_task<Idx>(c, sh, H, tq);
                if (rq.score == kNoScore) continue;
                const Candidate cand = make_candidate<Idx>(sh, rq, tq);
                if (cand.score < best.score || (cand.score == best.score && tie_better(H, cand, best))) best = cand;
            }
        }
        __syncwarp();
    }
}

// Seeds [cb, ce) (at most 32) of one event with the Dv1 triplet search, by one warp on its own.
template <typename Idx, bool kUni, typename HitsT, typename TabT>
__device__ __forceinline__ void track_chunk_dv1(const DevConst &c, WarpShared<Idx, true> &sh, const TabT &tab, const float2 *yb,
                                                const HitsT &H, const ds_seeds &seeds, int cb, int ce, const ds_tracks &out)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int s = cb + lane;
    const bool act = s < ce;
    // ---- per seed: S2 and the range of its UTbX candidates ----------------------------------------------------------------------
    float fy = 0.f, ftx = 0.f, fty = 0.f;
    int a_o = 0, n_o = 0;
    if (act) {
        const float fx = seeds.x[s], fq = seeds.qop[s];
        fy = seeds.y[s]; ftx = seeds.tx[s]; fty = seeds.ty[s];
        const S2 s2 = extrapolate_seed(c, fx, fy, ftx, fty, fq);
        SeedRec &r = sh.rec[lane];
        r.xm = s2.xm; r.zm = s2.zm; r.w1 = s2.w1;
        r.y[0] = s2.y0; r.y[1] = s2.y1; r.y[2] = s2.y2; r.y[3] = s2.y3;
#pragma unroll
        for (int l = 0; l < 3; ++l)
            r.mask[l] = (unsigned short)sector_mask<kUni>(c, yb, l, l == 0 ? s2.y0 : (l == 1 ? s2.y1 : s2.y2));
        const unsigned mask3 = sector_mask<kUni>(c, yb, 3, s2.y3);
        r.mask[3] = (unsigned short)mask3;
        if (mask3) {   // the sectors of a layer follow each other in the sorted slice: one range from the lowest to the
                       // highest compatible sector (a sector in between that is not compatible is sorted out per item)
            const int s_lo = __ffs(mask3) - 1, s_hi = 31 - __clz(mask3);
            a_o = (int)tab[(3 * c.n_sectors + s_lo) * TabT::kSlices];
            n_o = (int)tab[(3 * c.n_sectors + s_hi + 1) * TabT::kSlices] - a_o;
        }
    }
    int incl = n_o;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += t;
    }
    const int total = __shfl_sync(FULL, incl, 31);
    sh.dv_off[lane] = incl - n_o;
    sh.dv_a[lane] = a_o;
    __syncwarp();

    Candidate best;
    best.score = kNoScore; best.a = 0.0; best.b = 0.0; best.chi2 = 0.0;
    best.nh = 0; best.j0 = -1; best.j1 = -1; best.j2 = -1; best.j3 = -1;
    int n_trip = 0;
    // ---- T: lane per item (seed, UTbX hit) -----------------------------------------------------------------------------------------
    // item t -> (seed, UTbX hit); z of the hit comes from global memory and is fetched one round ahead
    auto item = [&](int t, int &o, int &j3, float &z3) {
        // last seed whose first item is <= t (seeds without items share the offset of the next); a lane's items only go up
        while (o < 31 && sh.dv_off[o + 1] <= t) ++o;
        j3 = sh.dv_a[o] + (t - sh.dv_off[o]);
        z3 = hit_z(H, j3);
    };
    int o_nx = 0, j3_nx = 0;
    float z3_nx = 0.f;
    if (lane < total) item(lane, o_nx, j3_nx, z3_nx);
    // T2: the exact (fp64) triplet test for the last `cnt` (<= 32) queued items, a lane each; triplets are compacted into the list
    int n_cand = 0;
    auto exact_round = [&](int cnt) {
        __syncwarp();
        bool has = false;
        int o = 0, j3 = 0, j0 = -1;
        float z3 = 0.f;
        if (lane < cnt) {
            const int q = n_cand - cnt + lane;
            o = sh.cand_o[q]; j3 = (int)sh.cand_j3[q]; z3 = sh.cand_z[q];
            const SeedRec &t2 = sh.rec[o];
            if (y_compatible<kUni>(c, H, j3, t2.y[3])) {   // kUni: the pre-test has decided it (exactly, by sector)
                const double x3 = (double)H.x0[j3] + c.dxdy[3] * t2.y[3];
                const double txc = (x3 - t2.xm) / ((double)z3 - t2.zm);
                const double xp = t2.xm + txc * (c.z_layer[0] - t2.zm);
                j0 = search_layer<kUni>(c, H, tab, 0, xp, t2.y[0], t2.w1, (unsigned)t2.mask[0]).x;
                has = j0 >= 0;
            }
        }
        n_cand -= cnt;
        const unsigned m = __ballot_sync(FULL, has);
        if (has) {
            const int f = n_trip + __popc(m & lanemask_lt());
            sh.fs[f] = (unsigned short)o;
            sh.slot[f] = (Idx)j3;
            sh.near[3 * f][0] = (Idx)j0;
            sh.near[3 * f][1] = (Idx)-1;
            sh.zw3[f] = make_float2(z3, 0.f);   // w of the UTbX hit is read by the fit
        }
        n_trip += __popc(m);
        if (n_trip >= 32) {   // the list holds 64: room for one more round is guaranteed after this
            dv1_flush<Idx, kUni>(c, sh, tab, H, n_trip, best);
            n_trip = 0;
        }
    };
    // T1: fp32 pre-test, a superset of the exact one (margins far above the fp32 rounding of the prediction, ~1e-3 mm):
    // y-compatibility of the UTbX hit and "is there a UTaX hit near the line through the hit and the magnet point".
    // About one item in eight passes; only those pay for the fp64 division and search.
    const float ytol_f = (float)c.y_tol + 0.01f, zl0_f = (float)c.z_layer[0];
    for (int t0 = 0; t0 < total; t0 += 32) {
        const int t = t0 + lane;
        const int o = o_nx, j3 = j3_nx;
        const float z3 = z3_nx;
        if (t + 32 < total) item(t + 32, o_nx, j3_nx, z3_nx);
        bool cand = false;
        if (t < total) {
            const SeedRec &t2 = sh.rec[o];
            const float y3 = (float)t2.y[3];
            bool y_ok;
            if (kUni) {   // the hit's sector: the last one of the seed's range that starts at or before the hit
                const unsigned mask3 = t2.mask[3];
                int sec = __ffs(mask3) - 1;
                const int s_hi = 31 - __clz(mask3);
                while (sec < s_hi && j3 >= (int)tab[(3 * c.n_sectors + sec + 1) * TabT::kSlices]) ++sec;
                y_ok = (mask3 >> sec) & 1u;
            } else {
                y_ok = hit_ymin(H, j3) - ytol_f <= y3 && y3 <= hit_ymax(H, j3) + ytol_f;
            }
            if (y_ok) {
                const float xm = (float)t2.xm, zm = (float)t2.zm;
                const float x3 = H.x0[j3] + (float)(c.dxdy[3] * t2.y[3]);
                const float xp = xm + (x3 - xm) * ((zl0_f - zm) / (z3 - zm));
                const float tg = xp - (float)(c.dxdy[0] * t2.y[0]);                 // in x0 coordinates of UTaX
                const float wf = (float)t2.w1 * 1.0001f + 0.05f + 4e-6f * fabsf(tg);
                const float xl = tg - wf, xh = tg + wf;
                const int bl = xslice<TabT::kSlices>(xl, c.xb_off, c.xb_scale), bh = xslice<TabT::kSlices>(xh, c.xb_off, c.xb_scale);
                for (unsigned m0 = t2.mask[0]; m0 && !cand; m0 &= m0 - 1) {
                    const int base = (__ffs(m0) - 1) * TabT::kSlices;   // layer 0
                    const int a = (int)tab[base + bl], b = (int)tab[base + bh + 1];
                    const int j = lower_bound_x0(H.x0, a, b, xl);
                    cand = j < b && H.x0[j] <= xh;
                }
                cand = cand || !(xp == xp);   // a prediction that is not a number goes to the exact test as it is
            }
        }
        const unsigned m = __ballot_sync(FULL, cand);
        if (m == 0) continue;
        if (cand) {
            const int q = n_cand + __popc(m & lanemask_lt());
            sh.cand_o[q] = (unsigned char)o;
            sh.cand_j3[q] = (Idx)j3;
            sh.cand_z[q] = z3;
        }
        n_cand += __popc(m);
        if (n_cand >= 32) exact_round(32);
    }
    if (n_cand > 0) exact_round(n_cand);
    if (n_trip > 0) dv1_flush<Idx, kUni>(c, sh, tab, H, n_trip, best);
    // ---- track record ------------------------------------------------------------------------------------------------------------
    if (act) {
        if (best.score == kNoScore) {
            write_not_found(out, s);
        } else {
            const double ys = (double)fy, txs = (double)ftx, tys = (double)fty;
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
    }
    __syncwarp();   // the lists are rewritten by the warp's next chunk
}

// All seeds of one event: every warp of the block takes an equal share (at most 32 at a time).
template <int W>
__device__ __forceinline__ int seed_chunk(int s_begin, int s_end)
{
    return min(32, (s_end - s_begin + W - 1) / W);
}

template <typename Idx, bool kDv1, bool kUni, int W, typename HitsT, typename TabT>
__device__ __forceinline__ void track_event(const DevConst &c, WarpShared<Idx, kDv1> *warps, const TabT &tab, const float2 *yb,
                                            const HitsT &H, const ds_seeds &seeds, int s_begin, int s_end, const ds_tracks &out,
                                            const SeedPre &pre)
{
    const int wid = threadIdx.x >> 5;
    const int chunk = seed_chunk<W>(s_begin, s_end);
    for (int cb = s_begin + wid * chunk; cb < s_end; cb += W * chunk) {
        if constexpr (kDv1) track_chunk_dv1<Idx, kUni>(c, warps[wid], tab, yb, H, seeds, cb, min(cb + chunk, s_end), out);
        else track_chunk<Idx, kUni>(c, warps[wid], tab, yb, H, seeds, cb, min(cb + chunk, s_end), out, pre);
    }
}

}  // namespace ds
