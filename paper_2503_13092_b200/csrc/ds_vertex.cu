// S8..S10 / K5: two-track vertexing of the kept downstream tracks.
// Paper: secondary vertex = point of closest approach of the two extrapolated tracks, trajectory model
// Eq. 4 with gamma = 0 in the field-free synthetic geometry, so the Newton-Raphson iteration of P:269 reduces to
// the closed-form two-line solution (A-20); opposite charges; invariant mass under the pi-pi and p-pi hypotheses
// (Fig. 18; proton = larger momentum, A-15); cuts from BASELINE cfg3.
//
// Three launches, all deterministic (count -> scan -> write, BASELINE north_star (5)):
//   k_vertex_count  block per event: ordered compaction of the kept positive / negative tracks into a per-event list
//                   (workspace), then all (pos, neg) pairs, lanes over pairs; number of passing pairs per event
//   k_vertex_scan   one block: exclusive scan of the per-event counts -> offsets (int64), overflow count
//   k_vertex_write  block per event: the pairs again, block-ordered compaction of the passing ones -> (ia, ib) order
// Pair arithmetic is fp64 in registers (cuts decide list membership); results are stored as fp32.
#include "ds_common.cuh"

namespace ds {

constexpr int kVtxThreads = 256;
constexpr int kVtxWarps = kVtxThreads / 32;

struct VtxOut {
    double x, y, z, doca, m_pipi, m_ppi;
    int flags;
};

__device__ __forceinline__ double inv_mass(double tx1, double ty1, double p1, double m1, double tx2, double ty2,
                                           double p2, double m2)
{
    const double n1 = sqrt(tx1 * tx1 + ty1 * ty1 + 1.0), n2 = sqrt(tx2 * tx2 + ty2 * ty2 + 1.0);
    const double k1 = p1 / n1, k2 = p2 / n2;
    const double px = k1 * tx1 + k2 * tx2, py = k1 * ty1 + k2 * ty2, pz = k1 + k2;
    const double E = sqrt(p1 * p1 + m1 * m1) + sqrt(p2 * p2 + m2 * m2);
    const double M2 = E * E - (px * px + py * py + pz * pz);
    return M2 > 0.0 ? sqrt(M2) : 0.0;
}

// a = positive track, b = negative track.  Returns true iff the pair passes every cut.
__device__ __forceinline__ bool vertex_pair(const DevConst &c, double xa, double ya, double txa, double tya, double qa,
                                            double xb, double yb, double txb, double tyb, double qb, VtxOut &o)
{
    // n = d_a x d_b with d = (tx, ty, 1): built from slope differences; |n|^2 = A*C - B^2 (Lagrange) without cancellation
    const double nx = tya - tyb, ny = txb - txa, nz = txa * tyb - tya * txb;
    const double n2 = nx * nx + ny * ny + nz * nz;
    if (n2 < c.n2_min) return false;
    const double A = txa * txa + tya * tya + 1.0, B = txa * txb + tya * tyb + 1.0, C = txb * txb + tyb * tyb + 1.0;
    const double rx = xa - xb, ry = ya - yb;
    const double Dd = txa * rx + tya * ry, Ee = txb * rx + tyb * ry;
    const double sa = (B * Ee - C * Dd) / n2, sb = (A * Ee - B * Dd) / n2;
    const double qax = xa + sa * txa, qay = ya + sa * tya, qaz = c.z_ref + sa;
    const double qbx = xb + sb * txb, qby = yb + sb * tyb, qbz = c.z_ref + sb;
    const double dx = qax - qbx, dy = qay - qby, dz = qaz - qbz;
    o.x = 0.5 * (qax + qbx);
    o.y = 0.5 * (qay + qby);
    o.z = 0.5 * (qaz + qbz);
    o.doca = sqrt(dx * dx + dy * dy + dz * dz);
    const double pa = 1000.0 / fabs(qa), pb = 1000.0 / fabs(qb);   // MeV
    o.m_pipi = inv_mass(txa, tya, pa, c.m_pi, txb, tyb, pb, c.m_pi);
    o.m_ppi = pa >= pb ? inv_mass(txa, tya, pa, c.m_p, txb, tyb, pb, c.m_pi)
                       : inv_mass(txa, tya, pa, c.m_pi, txb, tyb, pb, c.m_p);
    o.flags = (fabs(o.m_pipi - c.m_ks) < c.dm_ks ? 1 : 0) | (fabs(o.m_ppi - c.m_lambda) < c.dm_lambda ? 2 : 0);
    return o.doca < c.doca_max && c.zv_min <= o.z && o.z <= c.zv_max && o.flags != 0;
}

// Exclusive offset of this thread's flag inside the block (thread order) and the block total.
__device__ __forceinline__ int block_ordered_offset(bool flag, int *warp_cnt, int &total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned m = __ballot_sync(0xffffffffu, flag);
    if (lane == 0) warp_cnt[wid] = __popc(m);
    __syncthreads();
    int before = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < kVtxWarps; ++w) {
        const int cw = warp_cnt[w];
        if (w < wid) before += cw;
        tot += cw;
    }
    __syncthreads();
    total = tot;
    return before + __popc(m & lanemask_lt());
}

struct PairLists {
    int32_t *list;   // [n_seeds]: event e keeps its positive tracks at [s0, s0+npos), negative at [s0+npos, s0+npos+nneg)
    int32_t *npos;   // [n_events]
    int32_t *nneg;   // [n_events]
};

__device__ __forceinline__ void load_pair(const ds_tracks &t, int ia, int ib, double &xa, double &ya, double &txa,
                                          double &tya, double &qa, double &xb, double &yb, double &txb, double &tyb,
                                          double &qb)
{
    xa = t.x[ia]; ya = t.y[ia]; txa = t.tx[ia]; tya = t.ty[ia]; qa = t.qop[ia];
    xb = t.x[ib]; yb = t.y[ib]; txb = t.tx[ib]; tyb = t.ty[ib]; qb = t.qop[ib];
}

__global__ void __launch_bounds__(kVtxThreads)
k_vertex_count(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
               PairLists pl, int32_t *__restrict__ n_per_event)
{
    __shared__ int warp_cnt[kVtxWarps];
    __shared__ int red[kVtxWarps];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int s0 = seed_offsets[e], s1 = seed_offsets[e + 1];
    // pass 1: positive tracks to the front of the event's list slice, in seed order
    int npos = 0, nneg = 0;
    for (int sign = 0; sign < 2; ++sign) {
        int base = sign == 0 ? s0 : s0 + npos, cnt = 0;
        for (int chunk = s0; chunk < s1; chunk += kVtxThreads) {
            const int s = chunk + tid;
            bool f = false;
            if (s < s1 && trk.keep[s]) {
                const float q = trk.qop[s];
                f = sign == 0 ? q > 0.f : q < 0.f;
            }
            int tot;
            const int off = block_ordered_offset(f, warp_cnt, tot);
            if (f) pl.list[base + cnt + off] = s;
            cnt += tot;
        }
        if (sign == 0) npos = cnt; else nneg = cnt;
    }
    if (tid == 0) { pl.npos[e] = npos; pl.nneg[e] = nneg; }
    __syncthreads();   // list writes of this block are visible to this block
    const int64_t npairs = (int64_t)npos * nneg;
    int mine = 0;
    for (int64_t k = tid; k < npairs; k += kVtxThreads) {
        const int a = (int)(k / nneg), b = (int)(k - (int64_t)a * nneg);
        const int ia = pl.list[s0 + a], ib = pl.list[s0 + npos + b];
        double xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb;
        load_pair(trk, ia, ib, xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb);
        VtxOut o;
        mine += vertex_pair(c, xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb, o) ? 1 : 0;
    }
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

__global__ void __launch_bounds__(kVtxThreads)
k_vertex_write(const __grid_constant__ DevConst c, const ds_tracks trk, const int32_t *__restrict__ seed_offsets,
               PairLists pl, const ds_vertices out)
{
    __shared__ int warp_cnt[kVtxWarps];
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t o0 = out.offsets[e];
    if (out.offsets[e + 1] == o0) return;
    const int s0 = seed_offsets[e];
    const int npos = pl.npos[e], nneg = pl.nneg[e];
    const int64_t npairs = (int64_t)npos * nneg;
    int64_t written = 0;
    for (int64_t tile = 0; tile < npairs; tile += kVtxThreads) {
        const int64_t k = tile + tid;
        bool pass = false;
        VtxOut o;
        int ia = 0, ib = 0;
        if (k < npairs) {
            const int a = (int)(k / nneg), b = (int)(k - (int64_t)a * nneg);
            ia = pl.list[s0 + a];
            ib = pl.list[s0 + npos + b];
            double xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb;
            load_pair(trk, ia, ib, xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb);
            pass = vertex_pair(c, xa, ya, txa, tya, qa, xb, yb, txb, tyb, qb, o);
        }
        int tot;
        const int off = block_ordered_offset(pass, warp_cnt, tot);
        const int64_t pos = o0 + written + off;
        if (pass && pos < out.capacity) {
            out.evt[pos] = e; out.ia[pos] = ia; out.ib[pos] = ib; out.flags[pos] = o.flags;
            out.x[pos] = (float)o.x; out.y[pos] = (float)o.y; out.z[pos] = (float)o.z; out.doca[pos] = (float)o.doca;
            out.m_pipi[pos] = (float)o.m_pipi; out.m_ppi[pos] = (float)o.m_ppi;
        }
        written += tot;
    }
}

size_t vertex_workspace_bytes(int n_events, int64_t n_seeds)
{
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    return up(sizeof(int32_t) * (size_t)(n_seeds > 0 ? n_seeds : 1)) + 2 * up(sizeof(int32_t) * (size_t)(n_events > 0 ? n_events : 1));
}

cudaError_t launch_vertex(const DevConst &c, const ds_tracks &trk, const int32_t *seed_offsets, int n_events,
                          const ds_vertices &out, void *workspace, cudaStream_t st, Prof &prof)
{
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    PairLists pl;
    unsigned char *w = static_cast<unsigned char *>(workspace);
    pl.list = reinterpret_cast<int32_t *>(w);
    w += up(sizeof(int32_t) * (size_t)(trk.n > 0 ? trk.n : 1));
    pl.npos = reinterpret_cast<int32_t *>(w);
    w += up(sizeof(int32_t) * (size_t)(n_events > 0 ? n_events : 1));
    pl.nneg = reinterpret_cast<int32_t *>(w);
    if (n_events > 0) {
        prof.begin(DS_K_VTX_COUNT, st);
        k_vertex_count<<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, out.n_per_event);
        prof.end(st);
        cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) return err;
    }
    prof.begin(DS_K_VTX_SCAN, st);
    k_vertex_scan<<<1, kScanThreads, 0, st>>>(out.n_per_event, n_events, out.offsets, out.capacity, out.overflow);
    prof.end(st);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess) return err;
    if (n_events > 0) {
        prof.begin(DS_K_VTX_WRITE, st);
        k_vertex_write<<<n_events, kVtxThreads, 0, st>>>(c, trk, seed_offsets, pl, out);
        prof.end(st);
        err = cudaGetLastError();
    }
    return err;
}

}  // namespace ds
