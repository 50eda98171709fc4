// S8..S10 / K5: two-track vertexing of the kept downstream tracks.
// Paper: secondary vertex = point of closest approach of the two extrapolated tracks, trajectory model
// Eq. 4 with gamma = 0 in the field-free synthetic geometry, so the Newton-Raphson iteration of P:269 reduces to
// the closed-form two-line solution (A-20); opposite charges; invariant mass under the pi-pi and p-pi hypotheses
// (Fig. 18; proton = larger momentum, A-15); cuts from BASELINE cfg3.
//
// Three launches, all deterministic (count -> scan -> write, BASELINE north_star (5)):
//   k_vertex_count  block per event: ordered compaction of the kept positive / negative tracks into a per-event list
//                   (workspace) and, with the per-track terms of the masses (|d|, p/|d|, E_pi, E_p), into shared
//                   memory; then all (pos, neg) pairs, lanes over pairs, masses only for pairs that pass the DOCA and
//                   z cuts; number of passing pairs per event
//   k_vertex_scan   one block: exclusive scan of the per-event counts -> offsets (int64), overflow count
//   k_vertex_write  block per event: the pairs again, block-ordered compaction of the passing ones -> (ia, ib) order
// Pair arithmetic is fp64 in registers (cuts decide list membership); results are stored as fp32.
#include "ds_common.cuh"

namespace ds {

constexpr int kVtxThreads = 128;
constexpr int kVtxWarps = kVtxThreads / 32;
constexpr int kVtxCap = 512;   // seeds of an event whose kept tracks are staged in shared memory
constexpr int kSmallEventSeeds = 256;   // batches with at most this many seeds per event on average: warp per event

struct VtxOut {
    double x, y, z, doca, m_pipi, m_ppi;
    int flags;
};

// A kept track as the pair loop sees it: state at z_ref and the per-track terms of the invariant masses
// (|d| = sqrt(tx^2 + ty^2 + 1), p in MeV, k = p / |d|, E under the pion and the proton hypothesis).
struct VtxTrack {
    double x, y, tx, ty, p, k, e_pi, e_p;
    double g;   // gamma of Eq. 3: curvature of x(z) upstream of the UT; 0 with magnet_polarity = 0
};

__device__ __forceinline__ VtxTrack make_track(const DevConst &c, const ds_tracks &t, int i)
{
    VtxTrack r;
    r.x = t.x[i]; r.y = t.y[i]; r.tx = t.tx[i]; r.ty = t.ty[i];
    const double q = t.qop[i];
    r.p = 1000.0 / fabs(q);   // MeV
    r.k = r.p / sqrt(r.tx * r.tx + r.ty * r.ty + 1.0);
    r.e_pi = sqrt(r.p * r.p + c.m_pi * c.m_pi);
    r.e_p = sqrt(r.p * r.p + c.m_p * c.m_p);
    r.g = -c.vtx_mp * (c.gamma_c0 + c.gamma_c1 * (q / 1000.0));   // q/p in 1/GeV, the parametrisation in 1/MeV (A-27)
    return r;
}

// Kept tracks of one event in shared memory (positive tracks from the front, negative tracks from the back).
struct VtxShared {
    float x[kVtxCap], y[kVtxCap], tx[kVtxCap], ty[kVtxCap];
    double p[kVtxCap], k[kVtxCap], e_pi[kVtxCap], e_p[kVtxCap], g[kVtxCap];
    __device__ __forceinline__ void put(int pos, const VtxTrack &r)
    {
        x[pos] = (float)r.x; y[pos] = (float)r.y; tx[pos] = (float)r.tx; ty[pos] = (float)r.ty;   // exact: they were fp32
        p[pos] = r.p; k[pos] = r.k; e_pi[pos] = r.e_pi; e_p[pos] = r.e_p; g[pos] = r.g;
    }
    __device__ __forceinline__ VtxTrack get(int pos) const
    {
        VtxTrack r;
        r.x = x[pos]; r.y = y[pos]; r.tx = tx[pos]; r.ty = ty[pos];
        r.p = p[pos]; r.k = k[pos]; r.e_pi = e_pi[pos]; r.e_p = e_p[pos]; r.g = g[pos];
        return r;
    }
};

// a = positive track, b = negative track.  Returns true iff the pair passes every cut; o is complete only then.
template <bool kCurved>
__device__ __forceinline__ bool vertex_pair(const DevConst &c, const VtxTrack &a, const VtxTrack &b, VtxOut &o)
{
    // n = d_a x d_b with d = (tx, ty, 1): built from slope differences; |n|^2 = A*C - B^2 (Lagrange) without cancellation
    const double nx = a.ty - b.ty, ny = b.tx - a.tx, nz = a.tx * b.ty - a.ty * b.tx;
    const double n2 = nx * nx + ny * ny + nz * nz;
    if (n2 < c.n2_min) return false;
    const double A = a.tx * a.tx + a.ty * a.ty + 1.0, B = a.tx * b.tx + a.ty * b.ty + 1.0, C = b.tx * b.tx + b.ty * b.ty + 1.0;
    const double rx = a.x - b.x, ry = a.y - b.y;
    const double Dd = a.tx * rx + a.ty * ry, Ee = b.tx * rx + b.ty * ry;
    const double inv_n2 = 1.0 / n2;   // one division for both line parameters
    double sa = (B * Ee - C * Dd) * inv_n2, sb = (A * Ee - B * Dd) * inv_n2;
    constexpr bool curved = kCurved;   // the launcher instantiates the straight-track kernels for magnet_polarity = 0
    if (curved) {
        // Newton-Raphson on F(u, v) = |Traj_a(z_ref + u) - Traj_b(z_ref + v)|^2 with the parabolas of Eq. 4, from the
        // straight-line solution (A-28); gradient and Hessian of F / 2
        for (int it = 0; it < c.vtx_iters; ++it) {
            const double Dx = a.x + a.tx * sa + a.g * sa * sa - (b.x + b.tx * sb + b.g * sb * sb);
            const double Dy = a.y + a.ty * sa - (b.y + b.ty * sb), Dz = sa - sb;
            const double dax = a.tx + 2.0 * a.g * sa, dbx = b.tx + 2.0 * b.g * sb;
            const double gu = Dx * dax + Dy * a.ty + Dz, gv = -(Dx * dbx + Dy * b.ty + Dz);
            const double Huu = dax * dax + a.ty * a.ty + 1.0 + Dx * 2.0 * a.g;
            const double Hvv = dbx * dbx + b.ty * b.ty + 1.0 - Dx * 2.0 * b.g;
            const double Huv = -(dax * dbx + a.ty * b.ty + 1.0);
            const double det = Huu * Hvv - Huv * Huv;
            if (det == 0.0) break;
            const double inv = 1.0 / det;   // one division for both components
            sa -= (Hvv * gu - Huv * gv) * inv;
            sb -= (Huu * gv - Huv * gu) * inv;
        }
    }
    const double qax = a.x + sa * a.tx + a.g * sa * sa, qay = a.y + sa * a.ty, qaz = c.z_ref + sa;
    const double qbx = b.x + sb * b.tx + b.g * sb * sb, qby = b.y + sb * b.ty, qbz = c.z_ref + sb;
    const double dx = qax - qbx, dy = qay - qby, dz = qaz - qbz;
    o.x = 0.5 * (qax + qbx);
    o.y = 0.5 * (qay + qby);
    o.z = 0.5 * (qaz + qbz);
    // the cuts first, on the squared distance: most pairs end here, without the square root
    const double d2 = dx * dx + dy * dy + dz * dz;
    if (!(d2 < c.doca_max * c.doca_max && c.zv_min <= o.z && o.z <= c.zv_max)) return false;
    o.doca = sqrt(d2);
    if (!(o.doca < c.doca_max)) return false;   // the cut as defined (decides the last ulp)
    // invariant masses: same momentum sum under both hypotheses; proton = larger momentum (A-15)
    double atx = a.tx, btx = b.tx, ak = a.k, bk = b.k;
    if (curved) {   // slopes dx/dz at the vertex z (Eq. 2) and with them the direction normalisation
        atx = a.tx + 2.0 * a.g * (o.z - c.z_ref);
        btx = b.tx + 2.0 * b.g * (o.z - c.z_ref);
        ak = a.p / sqrt(atx * atx + a.ty * a.ty + 1.0);
        bk = b.p / sqrt(btx * btx + b.ty * b.ty + 1.0);
    }
    const double px = ak * atx + bk * btx, py = ak * a.ty + bk * b.ty, pz = ak + bk;
    const double p2 = px * px + py * py + pz * pz;
    const double e1 = a.e_pi + b.e_pi, e2 = a.p >= b.p ? a.e_p + b.e_pi : a.e_pi + b.e_p;
    const double m1 = e1 * e1 - p2, m2 = e2 * e2 - p2;
    o.m_pipi = m1 > 0.0 ? sqrt(m1) : 0.0;
    o.m_ppi = m2 > 0.0 ? sqrt(m2) : 0.0;
    o.flags = (fabs(o.m_pipi - c.m_ks) < c.dm_ks ? 1 : 0) | (fabs(o.m_ppi - c.m_lambda) < c.dm_lambda ? 2 : 0);
    return o.flags != 0;
}

struct PairLists {
    int32_t *list;   // [n_seeds]: event e (seeds [s0, s1)) keeps its positive tracks at s0, s0+1, ... and its negative
                     // tracks at s1-1, s1-2, ..., both in seed order
    int32_t *npos;   // [n_events]
    int32_t *nneg;   // [n_events]
};

// Track of pair k = a * nneg + b of the event: from shared memory if the event is staged, else from global memory.
struct PairSource {
    const VtxShared *sh;   // nullptr: not staged
    const int32_t *list;   // the event's slice of PairLists::list
    int n_seeds, nneg;
};

__device__ __forceinline__ void pair_tracks(const DevConst &c, const ds_tracks &t, const PairSource &ps, int64_t k,
                                            VtxTrack &ta, VtxTrack &tb, int &ia, int &ib)
{
    int pa, pb;
    if (k <= 0xffffffffLL) {   // 32-bit division when it fits
        const unsigned a = (unsigned)k / (unsigned)ps.nneg;
        pa = (int)a;
        pb = ps.n_seeds - 1 - (int)((unsigned)k - a * (unsigned)ps.nneg);
    } else {
        const int64_t a = k / ps.nneg;
        pa = (int)a;
        pb = ps.n_seeds - 1 - (int)(k - a * ps.nneg);
    }
    ia = ps.list[pa];
    ib = ps.list[pb];
    if (ps.sh) {
        ta = ps.sh->get(pa);
        tb = ps.sh->get(pb);
    } else {
        ta = make_track(c, t, ia);
        tb = make_track(c, t, ib);
    }
}

// Exclusive offsets of this thread's two flags inside the block (thread order) and the block totals.
__device__ __forceinline__ void block_ordered_offsets(bool f0, bool f1, int (*warp_cnt)[2], int &off0, int &off1,
                                                      int &tot0, int &tot1)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned m0 = __ballot_sync(0xffffffffu, f0), m1 = __ballot_sync(0xffffffffu, f1);
    if (lane == 0) { warp_cnt[wid][0] = __popc(m0); warp_cnt[wid][1] = __popc(m1); }
    __syncthreads();
    int b0 = 0, b1 = 0, t0 = 0, t1 = 0;
#pragma unroll
    for (int w = 0; w < kVtxWarps; ++w) {
        const int c0 = warp_cnt[w][0], c1 = warp_cnt[w][1];
        if (w < wid) { b0 += c0; b1 += c1; }
        t0 += c0; t1 += c1;
    }
    __syncthreads();
    tot0 = t0; tot1 = t1;
    off0 = b0 + __popc(m0 & lanemask_lt());
    off1 = b1 + __popc(m1 & lanemask_lt());
}

template <bool kCurved>
__global__ void __launch_bounds__(kVtxThreads)
k_vertex_count(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
               PairLists pl, unsigned long long *__restrict__ masks, int32_t *__restrict__ n_per_event)
{
    __shared__ VtxShared sh;
    __shared__ int warp_cnt[kVtxWarps][2];
    __shared__ int red[kVtxWarps];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int s0 = seed_offsets[e], s1 = seed_offsets[e + 1];
    const int n_seeds = s1 - s0;
    const bool staged = n_seeds <= kVtxCap;
    int32_t *list = pl.list + s0;
    // S8: kept tracks, positive to the front and negative to the back of the event's list slice, both in seed order
    int npos = 0, nneg = 0;
    for (int chunk = s0; chunk < s1; chunk += kVtxThreads) {
        const int s = chunk + tid;
        bool fp = false, fn = false;
        if (s < s1 && trk.keep[s]) {
            const float q = trk.qop[s];
            fp = q > 0.f;
            fn = q < 0.f;
        }
        int op, on, tp, tn;
        block_ordered_offsets(fp, fn, warp_cnt, op, on, tp, tn);
        if (fp | fn) {
            const int pos = fp ? npos + op : n_seeds - 1 - (nneg + on);
            list[pos] = s;
            if (staged) sh.put(pos, make_track(c, trk, s));
        }
        npos += tp;
        nneg += tn;
    }
    if (tid == 0) { pl.npos[e] = npos; pl.nneg[e] = nneg; }
    __syncthreads();   // list and shared-memory writes of this block are visible to this block
    // S9: all (positive, negative) pairs, lanes over pairs
    PairSource ps;
    ps.sh = staged ? &sh : nullptr; ps.list = list; ps.n_seeds = n_seeds; ps.nneg = nneg;
    const int64_t npairs = (int64_t)npos * nneg;
    int mine = 0, it = 0;
    unsigned long long mask = 0ull;   // bit `it`: pair it * kVtxThreads + tid passes (the write kernel computes only those again)
    for (int64_t k = tid; k < npairs; k += kVtxThreads, ++it) {
        VtxTrack ta, tb;
        int ia, ib;
        pair_tracks(c, trk, ps, k, ta, tb, ia, ib);
        VtxOut o;
        if (vertex_pair<kCurved>(c, ta, tb, o)) {
            ++mine;
            if (it < 64) mask |= 1ull << it;
        }
    }
    masks[(size_t)e * kVtxThreads + tid] = mask;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((tid & 31) == 0) red[tid >> 5] = mine;
    __syncthreads();
    if (tid == 0) {
        int t = 0;
        for (int w = 0; w < kVtxWarps; ++w) t += red[w];
        n_per_event[e] = t;
    }
}

constexpr int kScanThreads = 1024;

__global__ void __launch_bounds__(kScanThreads)
k_vertex_scan(const int32_t *__restrict__ n_per_event, int n_events, int64_t *__restrict__ offsets, int64_t capacity,
              int32_t *__restrict__ overflow)
{
    __shared__ long long warp_sums[33];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int per = (n_events + kScanThreads - 1) / kScanThreads;
    const int b = min(tid * per, n_events), e = min(b + per, n_events);
    long long s = 0;
    for (int k = b; k < e; ++k) s += n_per_event[k];
    long long inc = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const long long t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const long long ws = warp_sums[lane];
        long long wi = ws;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const long long t = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= d) wi += t;
        }
        warp_sums[lane] = wi - ws;
        if (lane == 31) warp_sums[32] = wi;
    }
    __syncthreads();
    long long run = warp_sums[wid] + inc - s;
    for (int k = b; k < e; ++k) {
        offsets[k] = run;
        run += n_per_event[k];
    }
    if (tid == 0) {
        const long long total = warp_sums[32];
        offsets[n_events] = total;
        const long long over = total > capacity ? total - capacity : 0;
        overflow[0] = (int32_t)(over > 2147483647LL ? 2147483647LL : over);
    }
}

template <bool kCurved>
__global__ void __launch_bounds__(kVtxThreads)
k_vertex_write(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
               PairLists pl, const unsigned long long *__restrict__ masks, const ds_vertices out)
{
    __shared__ VtxShared sh;
    __shared__ int warp_cnt[kVtxWarps][2];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t o0 = out.offsets[e];
    if (out.offsets[e + 1] == o0) return;
    const int s0 = seed_offsets[e], n_seeds = seed_offsets[e + 1] - s0;
    const int npos = pl.npos[e], nneg = pl.nneg[e];
    const bool staged = n_seeds <= kVtxCap;
    const int32_t *list = pl.list + s0;
    if (staged) {
        for (int t = tid; t < npos + nneg; t += kVtxThreads) {
            const int pos = t < npos ? t : n_seeds - 1 - (t - npos);
            sh.put(pos, make_track(c, trk, list[pos]));
        }
        __syncthreads();
    }
    PairSource ps;
    ps.sh = staged ? &sh : nullptr; ps.list = list; ps.n_seeds = n_seeds; ps.nneg = nneg;
    const int64_t npairs = (int64_t)npos * nneg;
    const unsigned long long mask = masks[(size_t)e * kVtxThreads + tid];
    // S10 for the first 64 tiles from the masks alone: per tile and warp the number of passing pairs (ballots, no pair
    // arithmetic), one barrier, a prefix over (tile, warp) -- every passing pair then knows its output position, and S9 is
    // computed again for those pairs only, each by the thread that owns it
    __shared__ int s_cnt[64][kVtxWarps];   // then: offset of (tile, warp) inside the event
    __shared__ int s_total;
    const int lane = tid & 31, wid = tid >> 5;
    const int64_t tiles = (npairs + kVtxThreads - 1) / kVtxThreads;
    const int mtiles = (int)(tiles < 64 ? tiles : 64);
    for (int it = 0; it < mtiles; ++it) {
        const unsigned m = __ballot_sync(0xffffffffu, ((mask >> it) & 1ull) != 0);
        if (lane == 0) s_cnt[it][wid] = __popc(m);
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        for (int it = 0; it < mtiles; ++it)
            for (int w = 0; w < kVtxWarps; ++w) {
                const int n = s_cnt[it][w];
                s_cnt[it][w] = run;
                run += n;
            }
        s_total = run;
    }
    __syncthreads();
    for (int it = 0; it < mtiles; ++it) {
        const bool bit = ((mask >> it) & 1ull) != 0;
        const unsigned m = __ballot_sync(0xffffffffu, bit);
        if (!bit) continue;
        VtxTrack ta, tb;
        VtxOut o;
        int ia, ib;
        pair_tracks(c, trk, ps, (int64_t)it * kVtxThreads + tid, ta, tb, ia, ib);
        vertex_pair<kCurved>(c, ta, tb, o);   // passes again: same arithmetic
        const int64_t pos = o0 + s_cnt[it][wid] + __popc(m & lanemask_lt());
        if (pos < out.capacity) {
            out.evt[pos] = e; out.ia[pos] = ia; out.ib[pos] = ib; out.flags[pos] = o.flags;
            out.x[pos] = (float)o.x; out.y[pos] = (float)o.y; out.z[pos] = (float)o.z; out.doca[pos] = (float)o.doca;
            out.m_pipi[pos] = (float)o.m_pipi; out.m_ppi[pos] = (float)o.m_ppi;
        }
    }
    // tiles beyond the reach of the mask: every pair again, block-ordered compaction tile by tile
    int64_t written = s_total;
    for (int64_t tile = (int64_t)64 * kVtxThreads; tile < npairs; tile += kVtxThreads) {
        const int64_t k = tile + tid;
        bool pass = false;
        VtxOut o;
        int ia = 0, ib = 0;
        if (k < npairs) {
            VtxTrack ta, tb;
            pair_tracks(c, trk, ps, k, ta, tb, ia, ib);
            pass = vertex_pair<kCurved>(c, ta, tb, o);
        }
        int off, off1, tot, tot1;
        block_ordered_offsets(pass, false, warp_cnt, off, off1, tot, tot1);
        const int64_t pos = o0 + written + off;
        if (pass && pos < out.capacity) {
            out.evt[pos] = e; out.ia[pos] = ia; out.ib[pos] = ib; out.flags[pos] = o.flags;
            out.x[pos] = (float)o.x; out.y[pos] = (float)o.y; out.z[pos] = (float)o.z; out.doca[pos] = (float)o.doca;
            out.m_pipi[pos] = (float)o.m_pipi; out.m_ppi[pos] = (float)o.m_ppi;
        }
        written += tot;
    }
}


// ---- warp-per-event variant (batches of small events: a block per event would leave most of its threads idle) -------
// k_vertex_count_w  warp per event: charge split by ballots into the event's list, kept tracks with their mass terms
//                   into the warp's shared memory, lanes over pairs; every lane keeps a bit mask of its passing pairs
//                   (pair k = 32 * iteration + lane -> bit `iteration`), stored for the write kernel; per-event count
//                   and the sum of the counts of every group of kGroup events (atomicAdd)
// k_vertex_write_w  warp per event: offset = counts of the earlier groups + counts of the earlier events of the group;
//                   only the pairs whose mask bit is set are computed again and written, in pair order
constexpr int kWThreads = 32;    // 32 / 64 / 128 / 256 measured on cfg4: 0.041 / 0.042 / 0.043 / 0.047 ms per 10 000 events
constexpr int kWWarps = kWThreads / 32;
constexpr int kWCap = 96;       // kept tracks of an event staged per warp
constexpr int kGroup = 256;     // events per group sum
constexpr int kMaskIters = 64;  // pair iterations covered by the 64-bit lane mask (events above: all pairs again)

struct WarpTracks {
    float x[kWCap], y[kWCap], tx[kWCap], ty[kWCap];
    double p[kWCap], k[kWCap], e_pi[kWCap], e_p[kWCap], g[kWCap];
    __device__ __forceinline__ void put(int pos, const VtxTrack &r)
    {
        x[pos] = (float)r.x; y[pos] = (float)r.y; tx[pos] = (float)r.tx; ty[pos] = (float)r.ty;   // exact: they were fp32
        p[pos] = r.p; k[pos] = r.k; e_pi[pos] = r.e_pi; e_p[pos] = r.e_p; g[pos] = r.g;
    }
    __device__ __forceinline__ VtxTrack get(int pos) const
    {
        VtxTrack r;
        r.x = x[pos]; r.y = y[pos]; r.tx = tx[pos]; r.ty = ty[pos];
        r.p = p[pos]; r.k = k[pos]; r.e_pi = e_pi[pos]; r.e_p = e_p[pos]; r.g = g[pos];
        return r;
    }
};

struct WarpWork {
    unsigned long long *masks;   // [n_events][32]
    int32_t *group_sums;         // [ceil(n_events / kGroup)], zeroed before k_vertex_count_w
};

// pair k of the event -> (a, b) with 32-bit division when it fits
__device__ __forceinline__ void pair_index(int64_t k, int nneg, int &a, int &b)
{
    if (k <= 0xffffffffLL) {
        const unsigned ua = (unsigned)k / (unsigned)nneg;
        a = (int)ua;
        b = (int)((unsigned)k - ua * (unsigned)nneg);
    } else {
        const int64_t la = k / nneg;
        a = (int)la;
        b = (int)(k - la * nneg);
    }
}

template <bool kCurved>
__global__ void __launch_bounds__(kWThreads)
k_vertex_count_w(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
                 int n_events, PairLists pl, WarpWork ww, int32_t *__restrict__ n_per_event)
{
    __shared__ WarpTracks tracks[kWWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int e = blockIdx.x * kWWarps + wid;
    if (e >= n_events) return;
    const unsigned FULL = 0xffffffffu;
    WarpTracks &sh = tracks[wid];
    const int s0 = seed_offsets[e], s1 = seed_offsets[e + 1];
    const int n_seeds = s1 - s0;
    int32_t *list = pl.list + s0;
    // S8: kept tracks, positive to the front and negative to the back of the event's list slice, both in seed order
    int npos = 0, nneg = 0;
    for (int chunk0 = s0; chunk0 < s1; chunk0 += 8 * 32) {   // eight chunks of 32 seeds with their loads in flight together
        int kp[8];
        float qp[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int s = chunk0 + u * 32 + lane;
            kp[u] = s < s1 ? trk.keep[s] : 0;
            qp[u] = s < s1 ? trk.qop[s] : 0.f;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (chunk0 + u * 32 >= s1) break;
            const int s = chunk0 + u * 32 + lane;
            const bool fp = kp[u] != 0 && qp[u] > 0.f, fn = kp[u] != 0 && qp[u] < 0.f;
            const unsigned mp = __ballot_sync(FULL, fp), mn = __ballot_sync(FULL, fn);
            if (fp) list[npos + __popc(mp & lanemask_lt())] = s;
            if (fn) list[n_seeds - 1 - (nneg + __popc(mn & lanemask_lt()))] = s;
            npos += __popc(mp);
            nneg += __popc(mn);
        }
    }
    if (lane == 0) { pl.npos[e] = npos; pl.nneg[e] = nneg; }
    __syncwarp();   // the list written by this warp is read by this warp
    const bool staged = npos + nneg <= kWCap;
    if (staged) {   // positive tracks at [0, npos), negative tracks at [npos, npos + nneg)
        for (int t = lane; t < npos + nneg; t += 32) sh.put(t, make_track(c, trk, t < npos ? list[t] : list[n_seeds - 1 - (t - npos)]));
        __syncwarp();
    }
    // S9: all (positive, negative) pairs, lanes over pairs
    const int64_t npairs = (int64_t)npos * nneg;
    unsigned long long mask = 0ull;
    int mine = 0, it = 0;
    for (int64_t k = lane; k < npairs; k += 32, ++it) {
        int a, b;
        pair_index(k, nneg, a, b);
        VtxTrack ta, tb;
        if (staged) {
            ta = sh.get(a);
            tb = sh.get(npos + b);
        } else {
            ta = make_track(c, trk, list[a]);
            tb = make_track(c, trk, list[n_seeds - 1 - b]);
        }
        VtxOut o;
        if (vertex_pair<kCurved>(c, ta, tb, o)) {
            ++mine;
            if (it < kMaskIters) mask |= 1ull << it;
        }
    }
    ww.masks[(size_t)e * 32 + lane] = mask;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(FULL, mine, o);
    if (lane == 0) {
        n_per_event[e] = mine;
        if (mine) atomicAdd(&ww.group_sums[e / kGroup], mine);
    }
}

constexpr int kW2Threads = 32;   // 32 / 64 / 128 / 256 / 512 measured: 0.027 / 0.030 / 0.027 / 0.031 / 0.035 ms
constexpr int kW2Warps = kW2Threads / 32;
static_assert(kGroup % kW2Warps == 0, "a block of k_vertex_write_w stays inside one group");

template <bool kCurved>
__global__ void __launch_bounds__(kW2Threads)
k_vertex_write_w(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
                 int n_events, PairLists pl, WarpWork ww, const ds_vertices out)
{
    __shared__ long long warp_part[kW2Warps];
    __shared__ int cnt[kW2Warps];
    __shared__ int pairbuf[kW2Warps][32];
    const unsigned FULL = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int e0 = blockIdx.x * kW2Warps, e = e0 + wid;
    // S10: vertices of all earlier events = sums of the earlier groups + counts of the earlier events of this group
    const int g0 = e0 / kGroup;
    long long part = 0;
    for (int g = tid; g < g0; g += kW2Threads) part += ww.group_sums[g];
    for (int i = g0 * kGroup + tid; i < e0; i += kW2Threads) part += out.n_per_event[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(FULL, part, o);
    if (lane == 0) {
        warp_part[wid] = part;
        cnt[wid] = e < n_events ? out.n_per_event[e] : 0;
    }
    __syncthreads();
    if (e >= n_events) return;
    long long o0 = 0;
#pragma unroll
    for (int w = 0; w < kW2Warps; ++w) o0 += warp_part[w] + (w < wid ? cnt[w] : 0);
    const int mine = cnt[wid];
    if (lane == 0) {
        out.offsets[e] = o0;
        if (e == n_events - 1) {
            const long long total = o0 + mine;
            out.offsets[n_events] = total;
            const long long over = total > out.capacity ? total - out.capacity : 0;
            out.overflow[0] = (int32_t)(over > 2147483647LL ? 2147483647LL : over);
        }
    }
    if (mine == 0) return;
    const int s0 = seed_offsets[e], n_seeds = seed_offsets[e + 1] - s0;
    const int npos = pl.npos[e], nneg = pl.nneg[e];
    const int32_t *list = pl.list + s0;
    const unsigned long long mask = ww.masks[(size_t)e * 32 + lane];
    const int64_t npairs = (int64_t)npos * nneg;
    const int64_t iters = (npairs + 31) / 32;
    // S9 again for the pairs that passed, a lane per passing pair: the pair indices are compacted from the masks (32 at a
    // time, in pair order) so that their tracks are fetched and their vertices computed side by side
    int *buf = pairbuf[wid];
    int64_t written = 0;
    int nbuf = 0;
    auto flush = [&]() {
        __syncwarp();
        if (lane < nbuf) {
            int a, b;
            pair_index(buf[lane], nneg, a, b);
            const int ia = list[a], ib = list[n_seeds - 1 - b];
            VtxOut o;
            vertex_pair<kCurved>(c, make_track(c, trk, ia), make_track(c, trk, ib), o);   // passes again: same arithmetic
            const int64_t pos = o0 + written + lane;
            if (pos < out.capacity) {
                out.evt[pos] = e; out.ia[pos] = ia; out.ib[pos] = ib; out.flags[pos] = o.flags;
                out.x[pos] = (float)o.x; out.y[pos] = (float)o.y; out.z[pos] = (float)o.z; out.doca[pos] = (float)o.doca;
                out.m_pipi[pos] = (float)o.m_pipi; out.m_ppi[pos] = (float)o.m_ppi;
            }
        }
        written += nbuf;
        nbuf = 0;
        __syncwarp();
    };
    const int mask_iters = (int)(iters < kMaskIters ? iters : kMaskIters);
    for (int it = 0; it < mask_iters; ++it) {
        const bool bit = ((mask >> it) & 1ull) != 0;
        const unsigned m = __ballot_sync(FULL, bit);
        if (m == 0) continue;
        if (nbuf + __popc(m) > 32) flush();
        if (bit) buf[nbuf + __popc(m & lanemask_lt())] = it * 32 + lane;
        nbuf += __popc(m);
    }
    flush();
    // pairs beyond the reach of the mask: every one is tried again
    for (int64_t it = kMaskIters; it < iters; ++it) {
        const int64_t k = it * 32 + lane;
        bool pass = false;
        VtxOut o;
        int ia = 0, ib = 0;
        if (k < npairs) {
            int a, b;
            pair_index(k, nneg, a, b);
            ia = list[a];
            ib = list[n_seeds - 1 - b];
            pass = vertex_pair<kCurved>(c, make_track(c, trk, ia), make_track(c, trk, ib), o);
        }
        const unsigned m = __ballot_sync(FULL, pass);
        const int64_t pos = o0 + written + __popc(m & lanemask_lt());
        if (pass && pos < out.capacity) {
            out.evt[pos] = e; out.ia[pos] = ia; out.ib[pos] = ib; out.flags[pos] = o.flags;
            out.x[pos] = (float)o.x; out.y[pos] = (float)o.y; out.z[pos] = (float)o.z; out.doca[pos] = (float)o.doca;
            out.m_pipi[pos] = (float)o.m_pipi; out.m_ppi[pos] = (float)o.m_ppi;
        }
        written += __popc(m);
    }
}

// Workspace: list [n_seeds], npos [E], nneg [E], pass masks [E][kVtxThreads] (the warp-per-event variant uses [E][32] of it), group sums
static size_t up256v(size_t v) { return (v + 255) & ~(size_t)255; }

size_t vertex_workspace_bytes(int n_events, int64_t n_seeds)
{
    const size_t ne = (size_t)(n_events > 0 ? n_events : 1), ns = (size_t)(n_seeds > 0 ? n_seeds : 1);
    return up256v(sizeof(int32_t) * ns) + 2 * up256v(sizeof(int32_t) * ne) + up256v(sizeof(unsigned long long) * kVtxThreads * ne) +
           up256v(sizeof(int32_t) * ((ne + kGroup - 1) / kGroup));
}

cudaError_t launch_vertex(const DevConst &c, const ds_tracks &trk, const int32_t *seed_offsets, int n_events,
                          const ds_vertices &out, void *workspace, cudaStream_t st, Prof &prof)
{
    const size_t ne = (size_t)(n_events > 0 ? n_events : 1), ns = (size_t)(trk.n > 0 ? trk.n : 1);
    PairLists pl;
    WarpWork ww;
    unsigned char *w = static_cast<unsigned char *>(workspace);
    pl.list = reinterpret_cast<int32_t *>(w);
    w += up256v(sizeof(int32_t) * ns);
    pl.npos = reinterpret_cast<int32_t *>(w);
    w += up256v(sizeof(int32_t) * ne);
    pl.nneg = reinterpret_cast<int32_t *>(w);
    w += up256v(sizeof(int32_t) * ne);
    ww.masks = reinterpret_cast<unsigned long long *>(w);
    w += up256v(sizeof(unsigned long long) * kVtxThreads * ne);
    ww.group_sums = reinterpret_cast<int32_t *>(w);
    const size_t n_groups = (ne + kGroup - 1) / kGroup;
    cudaError_t err = cudaSuccess;
    // batches of small events (the Run-3-like configurations): a warp per event; large events: a block per event
    const bool small_events = n_events > 0 && trk.n / n_events <= kSmallEventSeeds;
    const bool curved = c.vtx_mp != 0.0;   // parabolic trajectories + Newton-Raphson (P:255-P:269); else straight tracks
    if (n_events <= 0) {
        prof.begin(DS_K_VTX_SCAN, st);
        k_vertex_scan<<<1, kScanThreads, 0, st>>>(out.n_per_event, n_events, out.offsets, out.capacity, out.overflow);
        prof.end(st);
        return cudaGetLastError();
    }
    if (small_events) {
        err = cudaMemsetAsync(ww.group_sums, 0, sizeof(int32_t) * n_groups, st);
        if (err != cudaSuccess) return err;
        prof.begin(DS_K_VTX_COUNT, st);
        if (curved)
            k_vertex_count_w<true><<<(n_events + kWWarps - 1) / kWWarps, kWThreads, 0, st>>>(c, trk, seed_offsets, n_events, pl, ww,
                                                                                             out.n_per_event);
        else
            k_vertex_count_w<false><<<(n_events + kWWarps - 1) / kWWarps, kWThreads, 0, st>>>(c, trk, seed_offsets, n_events, pl,
                                                                                              ww, out.n_per_event);
        prof.end(st);
        err = cudaGetLastError();
        if (err != cudaSuccess) return err;
        prof.begin(DS_K_VTX_WRITE, st);
        if (curved)
            k_vertex_write_w<true><<<(n_events + kW2Warps - 1) / kW2Warps, kW2Threads, 0, st>>>(c, trk, seed_offsets, n_events, pl, ww, out);
        else
            k_vertex_write_w<false><<<(n_events + kW2Warps - 1) / kW2Warps, kW2Threads, 0, st>>>(c, trk, seed_offsets, n_events, pl, ww, out);
        prof.end(st);
        return cudaGetLastError();
    }
    prof.begin(DS_K_VTX_COUNT, st);
    if (curved)
        k_vertex_count<true><<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, ww.masks, out.n_per_event);
    else
        k_vertex_count<false><<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, ww.masks, out.n_per_event);
    prof.end(st);
    err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    prof.begin(DS_K_VTX_SCAN, st);
    k_vertex_scan<<<1, kScanThreads, 0, st>>>(out.n_per_event, n_events, out.offsets, out.capacity, out.overflow);
    prof.end(st);
    err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    prof.begin(DS_K_VTX_WRITE, st);
    if (curved)
        k_vertex_write<true><<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, ww.masks, out);
    else
        k_vertex_write<false><<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, ww.masks, out);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
