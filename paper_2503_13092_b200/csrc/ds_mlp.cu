// S7 / K4: ghost-killer feed-forward network (inputs = downstream state (x, y, tx, ty, q/p, chi2) + SciFi
// (q/p, chi2); ReLU hidden layers, sigmoid output).  Two architectures, both fixed at compile time so that the activations
// live in registers ("static structs"):
//   8 -> 32 -> 16 -> 1   BASELINE cfg0 (ds_upload_geometry), the one the metric is quoted on
//   8 -> 14 -> 1         the paper's own ("a single hidden layer with 14 neurons"; ds_upload_mlp_single)
// and two arithmetic flavours of each: IEEE expf and division (the default; the parity bound is 1e-4), or the paper's fast
// intrinsics __expf / __fdividef (ds_params.mlp_fast_math = 1, outside the parity bound: bench.py --mlp-fast-math
// reports the time and the score differences).
//
// Thread per found track (found slots are compacted warp by warp, see k_mlp), weights staged once per block in shared
// memory and read as broadcast float4.  fp32 FMA on CUDA cores: the contraction per track is [1x8][8x32] + [1x32][32x16] +
// [1x16][16x1] = 784 MAC (126 for the paper's network) -- far too thin for tensor cores.  A score within 1e-3 relative of
// the threshold is re-evaluated in fp64 so that the keep decision equals an fp64 evaluation.
#include "ds_common.cuh"

namespace ds {

constexpr int kMlpThreads = 128;
constexpr int kMlpSpan = 512;   // seed slots per warp (128..1024 measured: 512 is the fastest on cfg4)

// Network in shared memory.  H2 = 0: a single hidden layer, W3 acts on it.
template <int H1, int H2>
struct Net {
    static constexpr int kOut = H2 > 0 ? H2 : H1;
    float W1[H1 * DS_MLP_IN], b1[H1];
    float W2[(H2 > 0 ? H2 : 1) * H1], b2[H2 > 0 ? H2 : 1];
    float W3[kOut], b3;
    float mu[DS_MLP_IN], inv_sigma[DS_MLP_IN];
};

template <int H1, int H2>
__device__ __forceinline__ void load_net(Net<H1, H2> &m, const void *g)
{
    if constexpr (H2 > 0) {
        const DevMlp *s = static_cast<const DevMlp *>(g);
        for (int i = threadIdx.x; i < H1 * DS_MLP_IN; i += kMlpThreads) m.W1[i] = s->W1[i];
        for (int i = threadIdx.x; i < H2 * H1; i += kMlpThreads) m.W2[i] = s->W2[i];
        if (threadIdx.x < H1) m.b1[threadIdx.x] = s->b1[threadIdx.x];
        if (threadIdx.x < H2) { m.b2[threadIdx.x] = s->b2[threadIdx.x]; m.W3[threadIdx.x] = s->W3[threadIdx.x]; }
        if (threadIdx.x < DS_MLP_IN) { m.mu[threadIdx.x] = s->mu[threadIdx.x]; m.inv_sigma[threadIdx.x] = s->inv_sigma[threadIdx.x]; }
        if (threadIdx.x == 0) m.b3 = s->b3;
    } else {
        const DevMlpSingle *s = static_cast<const DevMlpSingle *>(g);
        for (int i = threadIdx.x; i < H1 * DS_MLP_IN; i += kMlpThreads) m.W1[i] = s->W1[i];
        if (threadIdx.x < H1) { m.b1[threadIdx.x] = s->b1[threadIdx.x]; m.W3[threadIdx.x] = s->W3[threadIdx.x]; }
        if (threadIdx.x < DS_MLP_IN) { m.mu[threadIdx.x] = s->mu[threadIdx.x]; m.inv_sigma[threadIdx.x] = s->inv_sigma[threadIdx.x]; }
        if (threadIdx.x == 0) m.b3 = s->b3;
    }
}

// fp64 evaluation for the rare score that sits on the threshold: rolled loops, out of line (keeps the fp32 path lean)
template <int H1, int H2>
__device__ __noinline__ double mlp_forward_f64(const Net<H1, H2> &m, const float *v)
{
    double f[DS_MLP_IN], h1[H1];
    for (int i = 0; i < DS_MLP_IN; ++i) f[i] = ((double)v[i] - (double)m.mu[i]) * (double)m.inv_sigma[i];
#pragma unroll 1
    for (int j = 0; j < H1; ++j) {
        double t = (double)m.b1[j];
#pragma unroll 1
        for (int i = 0; i < DS_MLP_IN; ++i) t += (double)m.W1[j * DS_MLP_IN + i] * f[i];
        h1[j] = t > 0.0 ? t : 0.0;
    }
    double t = (double)m.b3;
    if constexpr (H2 > 0) {
        double h2[H2];
#pragma unroll 1
        for (int j = 0; j < H2; ++j) {
            double u = (double)m.b2[j];
#pragma unroll 1
            for (int i = 0; i < H1; ++i) u += (double)m.W2[j * H1 + i] * h1[i];
            h2[j] = u > 0.0 ? u : 0.0;
        }
#pragma unroll 1
        for (int i = 0; i < H2; ++i) t += (double)m.W3[i] * h2[i];
    } else {
#pragma unroll 1
        for (int i = 0; i < H1; ++i) t += (double)m.W3[i] * h1[i];
    }
    return t;
}

template <int H1, int H2>
__device__ __forceinline__ float mlp_forward(const Net<H1, H2> &m, const float (&v)[DS_MLP_IN])
{
    float f[DS_MLP_IN], h1[H1];
#pragma unroll
    for (int i = 0; i < DS_MLP_IN; ++i) f[i] = (v[i] - m.mu[i]) * m.inv_sigma[i];
#pragma unroll
    for (int j = 0; j < H1; ++j) {
        float t = m.b1[j];
        const float4 *w = reinterpret_cast<const float4 *>(m.W1 + j * DS_MLP_IN);
#pragma unroll
        for (int i = 0; i < DS_MLP_IN / 4; ++i) {
            const float4 q = w[i];
            t = fmaf(q.x, f[4 * i], t); t = fmaf(q.y, f[4 * i + 1], t); t = fmaf(q.z, f[4 * i + 2], t); t = fmaf(q.w, f[4 * i + 3], t);
        }
        h1[j] = t > 0.f ? t : 0.f;
    }
    float t = m.b3;
    if constexpr (H2 > 0) {
        static_assert(H2 == 0 || H1 % 4 == 0, "rows of W2 are read as float4");
        float h2[H2 > 0 ? H2 : 1];
#pragma unroll
        for (int j = 0; j < H2; ++j) {
            float u = m.b2[j];
            const float4 *w = reinterpret_cast<const float4 *>(m.W2 + j * H1);
#pragma unroll
            for (int i = 0; i < H1 / 4; ++i) {
                const float4 q = w[i];
                u = fmaf(q.x, h1[4 * i], u); u = fmaf(q.y, h1[4 * i + 1], u); u = fmaf(q.z, h1[4 * i + 2], u); u = fmaf(q.w, h1[4 * i + 3], u);
            }
            h2[j] = u > 0.f ? u : 0.f;
        }
#pragma unroll
        for (int i = 0; i < H2; ++i) t += m.W3[i] * h2[i];
    } else {
#pragma unroll
        for (int i = 0; i < H1; ++i) t += m.W3[i] * h1[i];
    }
    return t;
}

// One found track: features in the order of P:121, fp32 forward pass, sigmoid, threshold (fp64 re-evaluation next to the
// threshold; with kFast the paper's intrinsics and no re-evaluation).
template <int H1, int H2, bool kFast>
__device__ __forceinline__ void score_track(const DevConst &c, const Net<H1, H2> &m, const ds_seeds &seeds, const ds_tracks &trk,
                                            int64_t s)
{
    float v[DS_MLP_IN];
    v[0] = trk.x[s]; v[1] = trk.y[s]; v[2] = trk.tx[s]; v[3] = trk.ty[s]; v[4] = trk.qop[s]; v[5] = trk.chi2[s];
    v[6] = seeds.qop[s];
    v[7] = seeds.chi2 ? seeds.chi2[s] : 0.f;
    const float t = mlp_forward<H1, H2>(m, v);
    float score;
    double sd;
    if (kFast) {
        score = __fdividef(1.0f, 1.0f + __expf(-t));
        sd = (double)score;
    } else {
        score = 1.0f / (1.0f + expf(-t));
        sd = (double)score;
        if (fabs(sd - c.mlp_thr) <= 1e-3 * fabs(c.mlp_thr)) {
            const double td = mlp_forward_f64<H1, H2>(m, v);
            sd = 1.0 / (1.0 + exp(-td));
            score = (float)sd;
        }
    }
    trk.score[s] = score;
    trk.keep[s] = c.mlp_keep_above ? (sd > c.mlp_thr) : (sd < c.mlp_thr);
}

// Each warp walks kMlpSpan consecutive seed slots, 32 at a time: slots without a track get score = keep = 0 at once,
// the found ones are queued (ballot compaction) and scored 32 at a time, so that the forward pass runs on full warps
// although only one slot in six holds a track.
template <int H1, int H2, bool kFast>
__global__ void __launch_bounds__(kMlpThreads)
k_mlp(const __grid_constant__ DevConst c, const void *__restrict__ gm, const ds_seeds seeds, const ds_tracks trk)
{
    __shared__ __align__(16) Net<H1, H2> m;
    __shared__ int queue[kMlpThreads / 32][64];
    load_net<H1, H2>(m, gm);
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int *q = queue[wid];
    const int64_t begin = ((int64_t)blockIdx.x * (kMlpThreads / 32) + wid) * kMlpSpan;
    const int64_t end = begin + kMlpSpan < trk.n ? begin + kMlpSpan : trk.n;
    int nq = 0;
    // the found flags of the lane's kMlpSpan / 32 slots in one round of loads (one after the other they are a chain of
    // DRAM latencies: the ballots below keep the compiler from hoisting them)
    static_assert(kMlpSpan / 32 <= 32, "one bit per slot of the lane");
    unsigned bits = 0;
    {
        int fl[kMlpSpan / 32];
#pragma unroll
        for (int u = 0; u < kMlpSpan / 32; ++u) {
            const int64_t s = begin + u * 32 + lane;
            fl[u] = s < end ? trk.found[s] : 0;
        }
#pragma unroll
        for (int u = 0; u < kMlpSpan / 32; ++u) bits |= fl[u] != 0 ? 1u << u : 0u;
    }
#pragma unroll 1
    for (int u = 0; u < kMlpSpan / 32; ++u) {
        const int64_t base = begin + u * 32;
        if (base >= end) break;
        const int64_t s = base + lane;
        const bool f = s < end && ((bits >> u) & 1u) != 0;
        if (s < end && !f) { trk.score[s] = 0.f; trk.keep[s] = 0; }
        const unsigned mask = __ballot_sync(0xffffffffu, f);
        if (f) q[nq + __popc(mask & lanemask_lt())] = (int)(s - begin);
        nq += __popc(mask);
        __syncwarp();
        if (nq >= 32) {
            score_track<H1, H2, kFast>(c, m, seeds, trk, begin + q[lane]);
            const int rest = lane < nq - 32 ? q[32 + lane] : 0;
            __syncwarp();
            q[lane] = rest;
            nq -= 32;
            __syncwarp();
        }
    }
    if (lane < nq) score_track<H1, H2, kFast>(c, m, seeds, trk, begin + q[lane]);
}

cudaError_t launch_mlp(const DevConst &c, const DevMlp *mlp, const DevMlpSingle *single, const ds_seeds &seeds,
                       const ds_tracks &trk, cudaStream_t st, Prof &prof)
{
    if (trk.n <= 0) return cudaSuccess;
    const int64_t per_block = (int64_t)(kMlpThreads / 32) * kMlpSpan;
    const unsigned grid = (unsigned)((trk.n + per_block - 1) / per_block);
    prof.begin(DS_K_MLP, st);
    if (single) {   // the paper's 8 -> 14 -> 1 (ds_upload_mlp_single)
        if (c.mlp_fast_math) k_mlp<DS_MLP_SINGLE_H, 0, true><<<grid, kMlpThreads, 0, st>>>(c, single, seeds, trk);
        else k_mlp<DS_MLP_SINGLE_H, 0, false><<<grid, kMlpThreads, 0, st>>>(c, single, seeds, trk);
    } else {
        if (c.mlp_fast_math) k_mlp<DS_MLP_H1, DS_MLP_H2, true><<<grid, kMlpThreads, 0, st>>>(c, mlp, seeds, trk);
        else k_mlp<DS_MLP_H1, DS_MLP_H2, false><<<grid, kMlpThreads, 0, st>>>(c, mlp, seeds, trk);
    }
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
