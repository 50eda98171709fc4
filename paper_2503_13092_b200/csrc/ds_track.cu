// S2..S6 / K2+K3: seed extrapolation, window search, candidate fit and best-candidate choice.
// Paper: magnet point from the seed state; first search window in UTbX, <= 10 closest hits;
// per first hit a new trajectory through (hit, magnet point) and refined windows in UTaX/UTaU/UTbV keeping the
// closest 1/2/2 hits; one final candidate per SciFi seed by score.  Readings A-1..A-9 in DESIGN.md.
//
// Mapping: one thread block per event.  Seeds are taken in chunks of blockDim.x: a thread-per-seed prefilter (S2 and
// "is there any hit in the x0 slices the first window touches") rejects most fake seeds at once and queues the rest
// in shared memory; then each warp takes queued seeds one at a time and works on them cooperatively:
//   S3  lanes over the candidate hits of the window (coalesced x0 reads of the sorted SoA), ballot compaction;
//       only if more than max_first hits pass, max_first selection passes by (distance, id)
//   S4  lanes over (first hit, layer): 3 * n_first independent searches of a few hits each
//   S5  lanes over combinations (first hit, i1, i2): every lane fits its own candidate
//   S6  warp argmin of the score, ties resolved by (more hits, ids)
// All of this arithmetic is fp64 in registers on fp32 inputs (the deciding comparisons must agree with an fp64
// reference to ~1e-5 relative; fp32 would not: one ulp of x at 800 mm is 6e-5 mm).
#include "ds_common.cuh"

namespace ds {

constexpr int kTrackThreads = 128;
constexpr int kTrackWarps = kTrackThreads / 32;
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

// Positions [a, b) (relative to the event) of the x0 slices of (layer, sector) that the x0 interval [lo, hi] touches.
__device__ __forceinline__ void slice_range(const DevConst &c, const int *tab, int layer, int sector, double lo,
                                            double hi, int &a, int &b)
{
    const int base = (layer * c.n_sectors + sector) * kXBins;
    const int xl = xbin(__double2float_rd(lo), c.xb_off, c.xb_scale);
    const int xh = xbin(__double2float_ru(hi), c.xb_off, c.xb_scale);
    a = tab[base + xl];
    b = tab[base + xh + 1];
}

struct Cand {
    double xh;   // measured x at the track's y
    int idx;     // position in the event's sorted slice
    int id;
};

struct WarpScratch {
    Cand first[kMaxFirst];
    Cand task[3 * kMaxFirst][2];
    int tn[3 * kMaxFirst];
};

__device__ __forceinline__ bool key_less(double d1, int id1, double d2, int id2)
{
    return d1 < d2 || (d1 == d2 && id1 < id2);
}

struct SortedHits {   // the event's slice of the sorted SoA
    const float *x0, *z, *ymin, *ymax, *w;
    const int32_t *id, *perm;
};

// y-compatibility of hit j (O-S3: ymin - y_tol <= y <= ymax + y_tol)
__device__ __forceinline__ bool y_compatible(const DevConst &c, const SortedHits &H, int j, double y)
{
    return ((double)H.ymin[j] - c.y_tol <= y) && (y <= (double)H.ymax[j] + c.y_tol);
}

__device__ __forceinline__ void write_not_found(const ds_tracks &out, int64_t s)
{
    out.x[s] = 0.f; out.y[s] = 0.f; out.tx[s] = 0.f; out.ty[s] = 0.f; out.qop[s] = 0.f; out.chi2[s] = 0.f;
    out.nhits[s] = 0; out.found[s] = 0;
    reinterpret_cast<int4 *>(out.hit)[s] = make_int4(-1, -1, -1, -1);
}

// One seed, whole warp.  Returns through `out` slot s.
__device__ void reconstruct_seed(const DevConst &c, const SortedHits &H, const int *tab, WarpScratch &ws, const S2 &s2,
                                 double ys, double txs, double tys, int64_t s, const ds_tracks &out)
{
    const int lane = threadIdx.x & 31;
    const unsigned FULL = 0xffffffffu;
    const int max_first = c.max_first;

    // ---- S3: first window in UTbX (layer 3) -------------------------------------------------------------------
    int s_lo, s_hi;
    sector_range(c, s2.y3, s_lo, s_hi);
    const double off3 = c.dxdy[3] * s2.y3;
    const double lo3 = s2.xc3 - off3 - s2.w0, hi3 = s2.xc3 - off3 + s2.w0;
    int nF = 0;
    for (int sec = s_lo; sec <= s_hi; ++sec) {
        int a, b;
        slice_range(c, tab, 3, sec, lo3, hi3, a, b);
        for (int base = a; base < b; base += 32) {
            const int j = base + lane;
            bool pass = false;
            double xh = 0.0;
            if (j < b) {
                xh = (double)H.x0[j] + off3;
                pass = fabs(xh - s2.xc3) <= s2.w0 && y_compatible(c, H, j, s2.y3);
            }
            const unsigned m = __ballot_sync(FULL, pass);
            if (pass) {
                const int pos = nF + __popc(m & lanemask_lt());
                if (pos < max_first) ws.first[pos] = Cand{xh, j, 0};
            }
            nF += __popc(m);
        }
    }
    if (nF == 0) {
        if (lane == 0) write_not_found(out, s);
        return;
    }
    if (nF > max_first) {
        // more hits in the window than are tried: keep the max_first closest by (distance, id)
        double last_d = -1.0;
        int last_id = INT32_MIN;
        for (int k = 0; k < max_first; ++k) {
            double bd = 1e300, bxh = 0.0;
            int bid = INT32_MAX, bj = -1;
            for (int sec = s_lo; sec <= s_hi; ++sec) {
                int a, b;
                slice_range(c, tab, 3, sec, lo3, hi3, a, b);
                for (int j = a + lane; j < b; j += 32) {
                    const double xh = (double)H.x0[j] + off3;
                    const double d = fabs(xh - s2.xc3);
                    if (d <= s2.w0 && y_compatible(c, H, j, s2.y3)) {
                        const int id = H.id[j];
                        if (key_less(last_d, last_id, d, id) && key_less(d, id, bd, bid)) {
                            bd = d; bid = id; bj = j; bxh = xh;
                        }
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double od = __shfl_xor_sync(FULL, bd, o), oxh = __shfl_xor_sync(FULL, bxh, o);
                const int oid = __shfl_xor_sync(FULL, bid, o), oj = __shfl_xor_sync(FULL, bj, o);
                if (key_less(od, oid, bd, bid)) { bd = od; bid = oid; bj = oj; bxh = oxh; }
            }
            if (lane == 0) ws.first[k] = Cand{bxh, bj, bid};
            last_d = bd;
            last_id = bid;
        }
        nF = max_first;
    }
    __syncwarp();

    // ---- S4: refined windows, lanes over (first hit, layer) -----------------------------------------------------------
    const int nT = 3 * nF;
    if (lane < nT) {
        const int f = lane / 3, l = lane - 3 * f;
        const Cand fh = ws.first[f];
        const double zf = (double)H.z[fh.idx];
        const double txc = (fh.xh - s2.xm) / (zf - s2.zm);
        const double xp = s2.xm + txc * (c.z_layer[l] - s2.zm);
        const double y = l == 0 ? s2.y0 : (l == 1 ? s2.y1 : s2.y2);
        const double off = c.dxdy[l] * y;
        const double lo = xp - off - s2.w1, hi = xp - off + s2.w1;
        const int keepn = l == 0 ? 1 : 2;
        double d0 = 1e300, d1 = 1e300;
        Cand c0 = Cand{0.0, -1, INT32_MAX}, c1 = c0;
        int n = 0, tl, th;
        sector_range(c, y, tl, th);
        for (int sec = tl; sec <= th; ++sec) {
            int a, b;
            slice_range(c, tab, l, sec, lo, hi, a, b);
            for (int j = a; j < b; ++j) {
                const double xh = (double)H.x0[j] + off;
                const double d = fabs(xh - xp);
                if (d <= s2.w1 && y_compatible(c, H, j, y)) {
                    const int id = H.id[j];
                    if (key_less(d, id, d0, c0.id)) {
                        d1 = d0; c1 = c0;
                        d0 = d; c0 = Cand{xh, j, id};
                    } else if (key_less(d, id, d1, c1.id)) {
                        d1 = d; c1 = Cand{xh, j, id};
                    }
                    ++n;
                }
            }
        }
        ws.tn[lane] = min(n, keepn);
        ws.task[lane][0] = c0;
        ws.task[lane][1] = c1;
    }
    __syncwarp();

    // ---- S5: lanes over combinations (first hit f, i1, i2); S6: best by (score, more hits, id3, id0, id1, id2) -----------------
    double b_score = 1e300, b_a = 0.0, b_b = 0.0, b_chi2 = 0.0;
    int b_nh = 0, b_i0 = -1, b_i1 = -1, b_i2 = -1, b_i3 = -1;
    int b_id0 = INT32_MAX, b_id1 = INT32_MAX, b_id2 = INT32_MAX, b_id3 = INT32_MAX;
    bool b_ok = false;
    for (int cb = lane; cb < 4 * nF; cb += 32) {
        const int f = cb >> 2, i1 = (cb >> 1) & 1, i2 = cb & 1;
        const int n0 = ws.tn[3 * f], n1 = ws.tn[3 * f + 1], n2 = ws.tn[3 * f + 2];
        if (i1 >= max(n1, 1) || i2 >= max(n2, 1)) continue;
        const int nh = 1 + (n0 > 0) + (n1 > 0) + (n2 > 0);
        if (nh < c.min_hits) continue;
        Cand h[4];
        h[0] = ws.task[3 * f][0];
        h[1] = ws.task[3 * f + 1][i1];
        h[2] = ws.task[3 * f + 2][i2];
        h[3] = ws.first[f];
        if (n0 == 0) h[0].idx = -1;
        if (n1 == 0) h[1].idx = -1;
        if (n2 == 0) h[2].idx = -1;
        double pz[5], px[5], pw[5];
        double S = 0, Sz = 0, Szz = 0, Sx = 0, Sxz = 0;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            bool use = true;
            if (k < 4) {
                use = h[k].idx >= 0;
                const int j = use ? h[k].idx : 0;
                pz[k] = (double)H.z[j] - c.z_ref;
                px[k] = h[k].xh;
                pw[k] = use ? (double)H.w[j] : 0.0;
            } else {   // magnet point pseudo-measurement (A-8)
                pz[k] = s2.zm - c.z_ref;
                px[k] = s2.xm;
                pw[k] = c.w_mag;
            }
            if (!use) px[k] = 0.0;
            S += pw[k];
            Sz += pw[k] * pz[k];
            Szz += pw[k] * pz[k] * pz[k];
            Sx += pw[k] * px[k];
            Sxz += pw[k] * px[k] * pz[k];
        }
        const double D = S * Szz - Sz * Sz;
        const double fb = (S * Sxz - Sz * Sx) / D;
        const double fa = (Szz * Sx - Sz * Sxz) / D;
        double chi2 = 0.0;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const double r = px[k] - fa - fb * pz[k];
            chi2 += pw[k] * r * r;
        }
        const double ndf = (double)(nh - 1);
        if (!(chi2 / ndf <= c.chi2ndf_max)) continue;
        const double score = chi2 + c.miss_penalty * (double)(4 - nh);
        const int id0 = h[0].idx >= 0 ? h[0].id : INT32_MAX;
        const int id1 = h[1].idx >= 0 ? h[1].id : INT32_MAX;
        const int id2 = h[2].idx >= 0 ? h[2].id : INT32_MAX;
        const int id3 = H.id[h[3].idx];
        bool better = !b_ok;
        if (b_ok) {
            if (score != b_score) better = score < b_score;
            else if (nh != b_nh) better = nh > b_nh;
            else if (id3 != b_id3) better = id3 < b_id3;
            else if (id0 != b_id0) better = id0 < b_id0;
            else if (id1 != b_id1) better = id1 < b_id1;
            else better = id2 < b_id2;
        }
        if (better) {
            b_ok = true; b_score = score; b_a = fa; b_b = fb; b_chi2 = chi2; b_nh = nh;
            b_i0 = h[0].idx; b_i1 = h[1].idx; b_i2 = h[2].idx; b_i3 = h[3].idx;
            b_id0 = id0; b_id1 = id1; b_id2 = id2; b_id3 = id3;
        }
    }
    // warp argmin
    double smin = b_ok ? b_score : 1e300;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smin = fmin(smin, __shfl_xor_sync(FULL, smin, o));
    unsigned tied = __ballot_sync(FULL, b_ok && b_score == smin);
    if (tied == 0) {
        if (lane == 0) write_not_found(out, s);
        return;
    }
    int win = __ffs(tied) - 1;
    unsigned rest = tied & (tied - 1);
    while (rest) {   // equal scores (duplicate hits): more hits, then (id3, id0, id1, id2)
        const int t = __ffs(rest) - 1;
        rest &= rest - 1;
        const int nh_t = __shfl_sync(FULL, b_nh, t), nh_w = __shfl_sync(FULL, b_nh, win);
        const int a3 = __shfl_sync(FULL, b_id3, t), w3 = __shfl_sync(FULL, b_id3, win);
        const int a0 = __shfl_sync(FULL, b_id0, t), w0 = __shfl_sync(FULL, b_id0, win);
        const int a1 = __shfl_sync(FULL, b_id1, t), w1 = __shfl_sync(FULL, b_id1, win);
        const int a2 = __shfl_sync(FULL, b_id2, t), w2 = __shfl_sync(FULL, b_id2, win);
        bool better;
        if (nh_t != nh_w) better = nh_t > nh_w;
        else if (a3 != w3) better = a3 < w3;
        else if (a0 != w0) better = a0 < w0;
        else if (a1 != w1) better = a1 < w1;
        else better = a2 < w2;
        if (better) win = t;
    }
    if (lane == win) {
        out.x[s] = (float)b_a;
        out.y[s] = (float)(ys + tys * (c.z_ref - c.z_seed));
        out.tx[s] = (float)b_b;
        out.ty[s] = (float)tys;
        out.qop[s] = (float)((txs - b_b) / c.kick);
        out.chi2[s] = (float)b_chi2;
        out.nhits[s] = b_nh;
        out.found[s] = 1;
        int4 hv;
        hv.x = b_i0 >= 0 ? H.perm[b_i0] : -1;
        hv.y = b_i1 >= 0 ? H.perm[b_i1] : -1;
        hv.z = b_i2 >= 0 ? H.perm[b_i2] : -1;
        hv.w = H.perm[b_i3];
        reinterpret_cast<int4 *>(out.hit)[s] = hv;
    }
}

__global__ void __launch_bounds__(kTrackThreads)
k_track(const __grid_constant__ DevConst c, const LayoutPtrs L, const ds_seeds seeds,
        const int32_t *__restrict__ hit_offsets, const int32_t *__restrict__ seed_offsets, const ds_tracks out)
{
    __shared__ int tab[kMaxBins + 1];
    __shared__ int queue[kTrackThreads];
    __shared__ int n_queue;
    __shared__ WarpScratch scratch[kTrackWarps];

    const int e = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int h0 = hit_offsets[e];
    const int s_begin = seed_offsets[e], s_end = seed_offsets[e + 1];
    if (s_begin == s_end) return;
    const int nb = c.n_bins;
    const int32_t *gtab = L.bin_offsets + (size_t)e * (nb + 1);
    for (int b = tid; b <= nb; b += kTrackThreads) tab[b] = gtab[b];
    SortedHits H;
    H.x0 = L.sx0 + h0; H.z = L.sz + h0; H.ymin = L.symin + h0; H.ymax = L.symax + h0; H.w = L.sw + h0;
    H.id = L.sid + h0; H.perm = L.perm + h0;

    for (int chunk = s_begin; chunk < s_end; chunk += kTrackThreads) {
        if (tid == 0) n_queue = 0;
        __syncthreads();   // also orders the table load before its first use
        // ---- prefilter: thread per seed (S2 + any hit in the slices of the first window?) ----------------------------
        const int s = chunk + tid;
        if (s < s_end) {
            const S2 s2 = extrapolate_seed(c, seeds.x[s], seeds.y[s], seeds.tx[s], seeds.ty[s], seeds.qop[s]);
            int s_lo, s_hi, cnt = 0;
            sector_range(c, s2.y3, s_lo, s_hi);
            const double off3 = c.dxdy[3] * s2.y3;
            for (int sec = s_lo; sec <= s_hi; ++sec) {
                int a, b;
                slice_range(c, tab, 3, sec, s2.xc3 - off3 - s2.w0, s2.xc3 - off3 + s2.w0, a, b);
                cnt += b - a;
            }
            if (cnt > 0) queue[atomicAdd(&n_queue, 1)] = s;
            else write_not_found(out, s);
        }
        __syncthreads();
        // ---- warp per queued seed ------------------------------------------------------------------------------------
        const int nq = n_queue;
        for (int q = wid; q < nq; q += kTrackWarps) {
            const int sq = queue[q];
            const double xs = seeds.x[sq], ys = seeds.y[sq], txs = seeds.tx[sq], tys = seeds.ty[sq], qop = seeds.qop[sq];
            const S2 s2 = extrapolate_seed(c, xs, ys, txs, tys, qop);
            reconstruct_seed(c, H, tab, scratch[wid], s2, ys, txs, tys, sq, out);
            __syncwarp();
        }
        __syncthreads();
    }
    (void)lane;
}

cudaError_t launch_track(const DevConst &c, const LayoutPtrs &lay, const ds_seeds &seeds, const int32_t *hit_offsets,
                         const int32_t *seed_offsets, int n_events, const ds_tracks &out, cudaStream_t st, Prof &prof)
{
    if (n_events <= 0) return cudaSuccess;
    prof.begin(DS_K_TRACK, st);
    k_track<<<n_events, kTrackThreads, 0, st>>>(c, lay, seeds, hit_offsets, seed_offsets, out);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
