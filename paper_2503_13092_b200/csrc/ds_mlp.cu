// S7 / K4: ghost-killer feed-forward network (inputs = downstream state (x, y, tx, ty, q/p, chi2) + SciFi
// (q/p, chi2); ReLU hidden layers, sigmoid output).  Architecture 8 -> 32 -> 16 -> 1 from BASELINE cfg0, fixed at
// compile time so that the activations live in registers ("static structs").
//
// Thread per found track (found slots are compacted warp by warp, see k_mlp), weights staged once per block in shared
// memory and read as broadcast float4.  fp32 FMA on
// CUDA cores: the contraction per track is [1x8][8x32] + [1x32][32x16] + [1x16][16x1] = 784 MAC -- far too thin for
// tensor cores.  IEEE expf and division (no fast-math intrinsics, unlike P:157: parity bound is 1e-4).  A score within
// 1e-3 relative of the threshold is re-evaluated in fp64 so that the keep decision equals an fp64 evaluation.
#include "ds_common.cuh"

namespace ds {

constexpr int kMlpThreads = 128;
constexpr int kMlpSpan = 512;   // seed slots per warp (128..1024 measured: 512 is the fastest on cfg4)

// fp64 evaluation for the rare score that sits on the threshold: rolled loops, out of line (keeps the fp32 path lean)
__device__ __noinline__ double mlp_forward_f64(const DevMlp &m, const float *v)
{
    double f[DS_MLP_IN], h1[DS_MLP_H1], h2[DS_MLP_H2];
    for (int i = 0; i < DS_MLP_IN; ++i) f[i] = ((double)v[i] - (double)m.mu[i]) * (double)m.inv_sigma[i];
#pragma unroll 1
    for (int j = 0; j < DS_MLP_H1; ++j) {
        double t = (double)m.b1[j];
#pragma unroll 1
        for (int i = 0; i < DS_MLP_IN; ++i) t += (double)m.W1[j * DS_MLP_IN + i] * f[i];
        h1[j] = t > 0.0 ? t : 0.0;
    }
#pragma unroll 1
    for (int j = 0; j < DS_MLP_H2; ++j) {
        double t = (double)m.b2[j];
#pragma unroll 1
        for (int i = 0; i < DS_MLP_H1; ++i) t += (double)m.W2[j * DS_MLP_H1 + i] * h1[i];
        h2[j] = t > 0.0 ? t : 0.0;
    }
    double t = (double)m.b3;
#pragma unroll 1
    for (int i = 0; i < DS_MLP_H2; ++i) t += (double)m.W3[i] * h2[i];
    return t;
}

template <typename T>
__device__ __forceinline__ T mlp_forward(const DevMlp &m, const float (&v)[DS_MLP_IN])
{
    T f[DS_MLP_IN], h1[DS_MLP_H1], h2[DS_MLP_H2];
#pragma unroll
    for (int i = 0; i < DS_MLP_IN; ++i) f[i] = ((T)v[i] - (T)m.mu[i]) * (T)m.inv_sigma[i];
#pragma unroll
    for (int j = 0; j < DS_MLP_H1; ++j) {
        T t = (T)m.b1[j];
        const float4 *w = reinterpret_cast<const float4 *>(m.W1 + j * DS_MLP_IN);
#pragma unroll
        for (int i = 0; i < DS_MLP_IN / 4; ++i) {
            const float4 q = w[i];
            t += (T)q.x * f[4 * i] + (T)q.y * f[4 * i + 1] + (T)q.z * f[4 * i + 2] + (T)q.w * f[4 * i + 3];
        }
        h1[j] = t > (T)0 ? t : (T)0;
    }
#pragma unroll
    for (int j = 0; j < DS_MLP_H2; ++j) {
        T t = (T)m.b2[j];
        const float4 *w = reinterpret_cast<const float4 *>(m.W2 + j * DS_MLP_H1);
#pragma unroll
        for (int i = 0; i < DS_MLP_H1 / 4; ++i) {
            const float4 q = w[i];
            t += (T)q.x * h1[4 * i] + (T)q.y * h1[4 * i + 1] + (T)q.z * h1[4 * i + 2] + (T)q.w * h1[4 * i + 3];
        }
        h2[j] = t > (T)0 ? t : (T)0;
    }
    T t = (T)m.b3;
#pragma unroll
    for (int i = 0; i < DS_MLP_H2; ++i) t += (T)m.W3[i] * h2[i];
    return t;
}

// One found track: features, fp32 forward pass, sigmoid, threshold (fp64 re-evaluation next to the threshold).
__device__ __forceinline__ void score_track(const DevConst &c, const DevMlp &m, const ds_seeds &seeds, const ds_tracks &trk,
                                            int64_t s)
{
    float v[DS_MLP_IN];
    v[0] = trk.x[s]; v[1] = trk.y[s]; v[2] = trk.tx[s]; v[3] = trk.ty[s]; v[4] = trk.qop[s]; v[5] = trk.chi2[s];
    v[6] = seeds.qop[s];
    v[7] = seeds.chi2 ? seeds.chi2[s] : 0.f;
    const float t = mlp_forward<float>(m, v);
    float score = 1.0f / (1.0f + expf(-t));
    double sd = (double)score;
    if (fabs(sd - c.mlp_thr) <= 1e-3 * fabs(c.mlp_thr)) {
        const double td = mlp_forward_f64(m, v);
        sd = 1.0 / (1.0 + exp(-td));
        score = (float)sd;
    }
    trk.score[s] = score;
    trk.keep[s] = c.mlp_keep_above ? (sd > c.mlp_thr) : (sd < c.mlp_thr);
}

// Each warp walks kMlpSpan consecutive seed slots, 32 at a time: slots without a track get score = keep = 0 at once,
// the found ones are queued (ballot compaction) and scored 32 at a time, so that the forward pass runs on full warps
// although only one slot in six holds a track.
__global__ void __launch_bounds__(kMlpThreads)
k_mlp(const __grid_constant__ DevConst c, const DevMlp *__restrict__ gm, const ds_seeds seeds, const ds_tracks trk)
{
    __shared__ __align__(16) DevMlp m;
    __shared__ int queue[kMlpThreads / 32][64];
    {
        const float4 *src = reinterpret_cast<const float4 *>(gm);
        float4 *dst = reinterpret_cast<float4 *>(&m);
        for (int i = threadIdx.x; i < (int)(sizeof(DevMlp) / 16); i += kMlpThreads) dst[i] = src[i];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int *q = queue[wid];
    const int64_t begin = ((int64_t)blockIdx.x * (kMlpThreads / 32) + wid) * kMlpSpan;
    const int64_t end = begin + kMlpSpan < trk.n ? begin + kMlpSpan : trk.n;
    int nq = 0;
    for (int64_t base = begin; base < end; base += 32) {
        const int64_t s = base + lane;
        const bool f = s < end && trk.found[s] != 0;
        if (s < end && !f) { trk.score[s] = 0.f; trk.keep[s] = 0; }
        const unsigned mask = __ballot_sync(0xffffffffu, f);
        if (f) q[nq + __popc(mask & lanemask_lt())] = (int)(s - begin);
        nq += __popc(mask);
        __syncwarp();
        if (nq >= 32) {
            score_track(c, m, seeds, trk, begin + q[lane]);
            const int rest = lane < nq - 32 ? q[32 + lane] : 0;
            __syncwarp();
            q[lane] = rest;
            nq -= 32;
            __syncwarp();
        }
    }
    if (lane < nq) score_track(c, m, seeds, trk, begin + q[lane]);
}

cudaError_t launch_mlp(const DevConst &c, const DevMlp *mlp, const ds_seeds &seeds, const ds_tracks &trk,
                       cudaStream_t st, Prof &prof)
{
    if (trk.n <= 0) return cudaSuccess;
    const int64_t per_block = (int64_t)(kMlpThreads / 32) * kMlpSpan;
    prof.begin(DS_K_MLP, st);
    k_mlp<<<(unsigned)((trk.n + per_block - 1) / per_block), kMlpThreads, 0, st>>>(c, mlp, seeds, trk);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
