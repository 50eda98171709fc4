// the HLT1 line NNs on the two-track vertices (P:277-P:285).
// Paper: "four different fast NNs with similar architectures to the one described in Sec. 2.2 ... a single hidden layer
// with 32 nodes and an output layer with a single node", inputs "include track parameters of the two secondary tracks,
// vertex parameters, and parent track parameters", threshold 0.5.  The paper lists no inputs: reading A-33 fixes
// 16 of them (see line_features).
//
// Thread per vertex (grid-stride; the number of vertices is read from the device-side offsets), the four weight sets
// staged once per block in shared memory and read as broadcast float4; features in fp64 from the fp32 records, networks
// in fp32 FMA like the ghost killer; a score within 1e-3 relative of the threshold is evaluated again in fp64 so that the
// decision bit equals an fp64 evaluation.
#include "ds_common.cuh"

namespace ds {

constexpr int kLineThreads = 128;

// A-33: positive track (tx, ty, q/p, chi2), negative track (tx, ty, q/p, chi2), vertex (x, y, z, DOCA), parent
// (tx, ty, p [GeV], pT [GeV]); parent momentum = sum of the track momenta 1/|q/p| along (tx, ty, 1)
__device__ __forceinline__ void line_features(const ds_tracks &t, const ds_vertices &v, int64_t k, float (&f)[DS_LINE_IN])
{
    const int a = v.ia[k], b = v.ib[k];
    const double txa = t.tx[a], tya = t.ty[a], qa = t.qop[a], txb = t.tx[b], tyb = t.ty[b], qb = t.qop[b];
    const double pa = 1.0 / fabs(qa), pb = 1.0 / fabs(qb);
    const double na = sqrt(txa * txa + tya * tya + 1.0), nb = sqrt(txb * txb + tyb * tyb + 1.0);
    const double px = pa * txa / na + pb * txb / nb, py = pa * tya / na + pb * tyb / nb, pz = pa / na + pb / nb;
    f[0] = (float)txa; f[1] = (float)tya; f[2] = (float)qa; f[3] = t.chi2[a];
    f[4] = (float)txb; f[5] = (float)tyb; f[6] = (float)qb; f[7] = t.chi2[b];
    f[8] = v.x[k]; f[9] = v.y[k]; f[10] = v.z[k]; f[11] = v.doca[k];
    f[12] = (float)(px / pz); f[13] = (float)(py / pz);
    f[14] = (float)sqrt(px * px + py * py + pz * pz);
    f[15] = (float)sqrt(px * px + py * py);
}

template <typename T>
__device__ __forceinline__ T line_forward(const DevLines &m, int net, const float (&v)[DS_LINE_IN])
{
    T f[DS_LINE_IN];
#pragma unroll
    for (int i = 0; i < DS_LINE_IN; ++i) f[i] = ((T)v[i] - (T)m.mu[i]) * (T)m.inv_sigma[i];
    T out = (T)m.b3[net];
#pragma unroll 4
    for (int j = 0; j < DS_LINE_H; ++j) {
        T t = (T)m.b1[net][j];
        const float4 *w = reinterpret_cast<const float4 *>(m.W1[net][j]);
#pragma unroll
        for (int i = 0; i < DS_LINE_IN / 4; ++i) {
            const float4 q = w[i];
            t += (T)q.x * f[4 * i] + (T)q.y * f[4 * i + 1] + (T)q.z * f[4 * i + 2] + (T)q.w * f[4 * i + 3];
        }
        out += (T)m.W3[net][j] * (t > (T)0 ? t : (T)0);
    }
    return out;
}

__global__ void __launch_bounds__(kLineThreads)
k_lines(const DevLines *__restrict__ gm, const ds_tracks trk, const ds_vertices vtx, int n_events, double thr,
        float *__restrict__ scores, int32_t *__restrict__ bits)
{
    __shared__ __align__(16) DevLines m;
    {
        const float4 *src = reinterpret_cast<const float4 *>(gm);
        float4 *dst = reinterpret_cast<float4 *>(&m);
        for (int i = threadIdx.x; i < (int)(sizeof(DevLines) / 16); i += kLineThreads) dst[i] = src[i];
    }
    __syncthreads();
    const int64_t total = vtx.offsets[n_events];
    const int64_t n = total < vtx.capacity ? total : vtx.capacity;
    for (int64_t k = (int64_t)blockIdx.x * kLineThreads + threadIdx.x; k < n; k += (int64_t)gridDim.x * kLineThreads) {
        float f[DS_LINE_IN];
        line_features(trk, vtx, k, f);
        int b = 0;
#pragma unroll 1
        for (int net = 0; net < DS_N_LINES; ++net) {
            float score = 1.0f / (1.0f + expf(-line_forward<float>(m, net, f)));
            double sd = (double)score;
            if (fabs(sd - thr) <= 1e-3 * fabs(thr)) {
                sd = 1.0 / (1.0 + exp(-line_forward<double>(m, net, f)));
                score = (float)sd;
            }
            scores[4 * k + net] = score;
            b |= sd > thr ? (1 << net) : 0;
        }
        bits[k] = b;
    }
}

cudaError_t launch_lines(const DevLines *nets, const ds_tracks &trk, const ds_vertices &vtx, int n_events, double thr,
                         float *scores, int32_t *bits, int n_sm, cudaStream_t st, Prof &prof)
{
    if (vtx.capacity <= 0) return cudaSuccess;
    int64_t blocks = (vtx.capacity + kLineThreads - 1) / kLineThreads;
    const int64_t cap = (int64_t)(n_sm > 0 ? n_sm : 148) * 8;   // grid-stride: the vertex count lives on the device
    if (blocks > cap) blocks = cap;
    prof.begin(DS_K_LINES, st);
    k_lines<<<(unsigned)blocks, kLineThreads, 0, st>>>(nets, trk, vtx, n_events, thr, scores, bits);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
