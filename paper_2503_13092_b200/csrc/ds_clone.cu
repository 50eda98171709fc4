// S6b: clone killing across seeds.
// Paper: "Iterating over all possible track pairs that have more than two shared UT hits ..., the candidates with lower
// scores are killed.  This removes about 1% of the candidates.".  Reading A-31: two found tracks of an event
// share a hit when they hold the same hit index in the same layer; a pair with at least clone_min_shared (3) shared hits
// is a clone pair and its worse member -- larger chi2 + miss_penalty * (4 - nhits), ties: the later seed -- is removed;
// every pair is judged on the tracks as S6 left them, so the result does not depend on an iteration order.
//
// One thread block per event: the (hit[4], score, seed index) records of the event's FOUND tracks are compacted into
// shared memory (a handful out of ~150 seed slots), a thread per found track counts shared hits against every other one
// (integer compares; the scores in fp64 from the fp32 chi2 of the record), then the removed tracks are reset to the "not
// found" record (score and keep included).  Events with more found tracks than the staging holds are judged straight
// from the records in two passes.
#include "ds_common.cuh"

namespace ds {

constexpr int kCloneThreads = 128;
constexpr int kCloneCap = 1024;   // found tracks of an event staged in shared memory (28 B each)

__device__ __forceinline__ int shared_hits(const int4 &a, const int4 &b)
{
    return (a.x >= 0 && a.x == b.x) + (a.y >= 0 && a.y == b.y) + (a.z >= 0 && a.z == b.z) + (a.w >= 0 && a.w == b.w);
}

__global__ void __launch_bounds__(kCloneThreads)
k_clone(const __grid_constant__ DevConst c, const int32_t *__restrict__ seed_offsets, const ds_tracks trk)
{
    __shared__ int4 s_hit[kCloneCap];
    __shared__ double s_score[kCloneCap];
    __shared__ int s_idx[kCloneCap];
    __shared__ int n_found;
    const int e = blockIdx.x, tid = threadIdx.x;
    const int s0 = seed_offsets[e], n = seed_offsets[e + 1] - s0;
    if (n < 2) return;
    const int4 *ghit = reinterpret_cast<const int4 *>(trk.hit) + s0;
    const int min_shared = c.clone_min_shared;
    auto score_of = [&](int i) {   // S6 score (A-9) of seed slot i
        return (double)trk.chi2[s0 + i] + c.miss_penalty * (double)(4 - trk.nhits[s0 + i]);
    };
    auto reset = [&](int64_t s) {
        trk.x[s] = 0.f; trk.y[s] = 0.f; trk.tx[s] = 0.f; trk.ty[s] = 0.f; trk.qop[s] = 0.f; trk.chi2[s] = 0.f;
        trk.score[s] = 0.f; trk.nhits[s] = 0; trk.found[s] = 0; trk.keep[s] = 0;
        reinterpret_cast<int4 *>(trk.hit)[s] = make_int4(-1, -1, -1, -1);
    };
    if (tid == 0) n_found = 0;
    __syncthreads();
    for (int i = tid; i < n; i += kCloneThreads) {
        if (trk.found[s0 + i]) {
            const int pos = atomicAdd(&n_found, 1);   // any order: the tie-break uses the seed index kept in s_idx
            if (pos < kCloneCap) {
                s_idx[pos] = i;
                s_hit[pos] = ghit[i];
                s_score[pos] = score_of(i);
            }
        }
    }
    __syncthreads();
    const int nf = n_found;
    if (nf < 2) return;
    if (nf <= kCloneCap) {
        for (int a = tid; a < nf; a += kCloneThreads) {
            const int4 ha = s_hit[a];
            const double sa = s_score[a];
            const int ia = s_idx[a];
            bool killed = false;
            for (int b = 0; b < nf; ++b) {
                if (b == a || shared_hits(ha, s_hit[b]) < min_shared) continue;
                const double sb = s_score[b];
                if (sb < sa || (sb == sa && s_idx[b] < ia)) killed = true;
            }
            if (killed) reset(s0 + ia);   // the judgement reads the shared-memory copy: the record can go at once
        }
        return;
    }
    // more found tracks than the staging holds: judge from the records; a removed track is first only marked (found = 2:
    // the judgement only asks found != 0, and k_track has written the field), the records change after every thread has
    // read them
    for (int i = tid; i < n; i += kCloneThreads) {
        if (!trk.found[s0 + i]) continue;
        const int4 hi = ghit[i];
        const double si = score_of(i);
        bool killed = false;
        for (int j = 0; j < n; ++j) {
            if (j == i || !trk.found[s0 + j] || shared_hits(hi, ghit[j]) < min_shared) continue;
            const double sj = score_of(j);
            if (sj < si || (sj == si && j < i)) killed = true;
        }
        if (killed) trk.found[s0 + i] = 2;
    }
    __syncthreads();
    for (int i = tid; i < n; i += kCloneThreads)
        if (trk.found[s0 + i] == 2) reset(s0 + i);
}

cudaError_t launch_clone(const DevConst &c, const int32_t *seed_offsets, int n_events, const ds_tracks &trk, cudaStream_t st,
                         Prof &prof)
{
    if (n_events <= 0 || c.clone_min_shared <= 0) return cudaSuccess;
    prof.begin(DS_K_CLONE, st);
    k_clone<<<n_events, kCloneThreads, 0, st>>>(c, seed_offsets, trk);
    prof.end(st);
    return cudaGetLastError();
}

}  // namespace ds
