// S6b: clone killing across seeds.
// Paper: "Iterating over all possible track pairs that have more than two shared UT hits ..., the candidates with lower
// scores are killed.  This removes about 1% of the candidates.".  Reading A-31: two found tracks of an event
// share a hit when they hold the same hit index in the same layer; a pair with at least clone_min_shared (3) shared hits
// is a clone pair and its worse member -- larger chi2 + miss_penalty * (4 - nhits), ties: the later seed -- is removed;
// every pair is judged on the tracks as S6 left them, so the result does not depend on an iteration order.
//
// One thread block per event: the (hit[4], score, found) records of the event's seeds are staged in shared memory, a
// thread per track counts shared hits against every other found track (integer compares; the scores in fp64 from the
// fp32 chi2 of the record), then the removed tracks are reset to the "not found" record (score and keep included).
#include "ds_common.cuh"

namespace ds {

constexpr int kCloneThreads = 128;
constexpr int kCloneCap = 1024;   // seeds of an event staged in shared memory (24 B each)

__global__ void __launch_bounds__(kCloneThreads)
k_clone(const __grid_constant__ DevConst c, const int32_t *__restrict__ seed_offsets, const ds_tracks trk)
{
    __shared__ int4 s_hit[kCloneCap];
    __shared__ double s_score[kCloneCap];   // < 0: no track in this slot
    const int e = blockIdx.x, tid = threadIdx.x;
    const int s0 = seed_offsets[e], n = seed_offsets[e + 1] - s0;
    if (n < 2) return;
    const bool staged = n <= kCloneCap;
    const int4 *ghit = reinterpret_cast<const int4 *>(trk.hit) + s0;
    auto score_of = [&](int i) {   // S6 score (A-9) of seed slot i, -1 if it holds no track
        return trk.found[s0 + i] ? (double)trk.chi2[s0 + i] + c.miss_penalty * (double)(4 - trk.nhits[s0 + i]) : -1.0;
    };
    if (staged) {
        for (int i = tid; i < n; i += kCloneThreads) {
            s_hit[i] = ghit[i];
            s_score[i] = score_of(i);
        }
        __syncthreads();
    }
    const int min_shared = c.clone_min_shared;
    constexpr unsigned kMark = 0x7fc0c10eu;   // a NaN payload no sigmoid produces: "removed", parked in score between the passes
    auto reset = [&](int64_t s) {
        trk.x[s] = 0.f; trk.y[s] = 0.f; trk.tx[s] = 0.f; trk.ty[s] = 0.f; trk.qop[s] = 0.f; trk.chi2[s] = 0.f;
        trk.score[s] = 0.f; trk.nhits[s] = 0; trk.found[s] = 0; trk.keep[s] = 0;
        reinterpret_cast<int4 *>(trk.hit)[s] = make_int4(-1, -1, -1, -1);
    };
    for (int i0 = 0; i0 < n; i0 += kCloneThreads) {
        const int i = i0 + tid;
        bool killed = false;
        if (i < n) {
            const double si = staged ? s_score[i] : score_of(i);
            if (si >= 0.0) {
                const int4 hi = staged ? s_hit[i] : ghit[i];
                for (int j = 0; j < n; ++j) {
                    const double sj = staged ? s_score[j] : score_of(j);
                    if (j == i || sj < 0.0) continue;
                    const int4 hj = staged ? s_hit[j] : ghit[j];
                    const int shared = (hi.x >= 0 && hi.x == hj.x) + (hi.y >= 0 && hi.y == hj.y) + (hi.z >= 0 && hi.z == hj.z) +
                                       (hi.w >= 0 && hi.w == hj.w);
                    if (shared >= min_shared && (sj < si || (sj == si && j < i))) killed = true;
                }
            }
        }
        if (killed) {
            // staged: the judgement reads the shared-memory copy, the record can go at once; else the records are what
            // the other threads still read, so the track is only marked (in a field the judgement does not read)
            if (staged) reset(s0 + i);
            else trk.score[s0 + i] = __uint_as_float(kMark);
        }
    }
    if (!staged) {
        __syncthreads();
        for (int i = tid; i < n; i += kCloneThreads)
            if (__float_as_uint(trk.score[s0 + i]) == kMark) reset(s0 + i);
    }
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
