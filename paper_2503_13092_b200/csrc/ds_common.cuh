// Shared device-side definitions of libds (CUDA, sm_100a).  Not part of the C ABI.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/ds.h"

// Checked build (DS_NVCC_EXTRA=-DDS_CHECKED): device-side asserts on the shared-memory indices and list sizes of the kernels;
// a failing one traps and the call returns DS_E_CUDA.  Compiled out otherwise.
#ifdef DS_CHECKED
#include <cassert>
#define DS_ASSERT(x) assert(x)
#else
#define DS_ASSERT(x) ((void)0)
#endif

namespace ds {

constexpr int kLayers = 4;
constexpr int kXBins = DS_XBINS;
constexpr int kMaxFirst = DS_MAX_FIRST_HITS;
constexpr int kIdLayerShift = 24;
constexpr int kIdSectorShift = 20;
constexpr int kIdSeqMask = (1 << 20) - 1;
constexpr int kRedoGrid = 2 * 148;   // blocks of k_layout / k_track when they only take the events k_event has left over

// Geometry + parameters as the kernels see them (passed by value as a __grid_constant__ kernel argument).
struct DevConst {
    // geometry
    double z_layer[4], dxdy[4];
    double y0;            // -y_half: lower edge of sector 0
    double inv_h;         // 1 / sector_height
    double z_seed, z_ref, zmag_c[4], kick, inv_kick;
    int n_sectors, n_bins; // n_bins = 4 * n_sectors * kXBins
    float xb_off, xb_scale; // xbin(x0) = clamp(floor((x0 + xb_off) * xb_scale))
    // parameters
    double w0_a, w0_b, w0_max, w1_a, w1_b, y_tol, w_mag, chi2ndf_max, miss_penalty;
    int min_hits, max_first;
    double mlp_thr;
    int mlp_keep_above, pad_;
    double doca_max, zv_min, zv_max, m_pi, m_p, m_ks, m_lambda, dm_ks, dm_lambda, n2_min;
    double vtx_mp, gamma_c0, gamma_c1;   // curved-track vertexing: gamma = -vtx_mp * (gamma_c0 + gamma_c1 * qop / 1000)
    int vtx_iters, clone_min_shared;
    int dv1, mlp_fast_math;
    int y_rsec, pad2_;   // sectors on either side of the one a y falls into that can be y-compatible: floor(y_tol / height) + 1
};

// Device copy of the ghost-killer weights (global memory, staged to shared memory by the kernel).
struct DevMlp {
    float W1[DS_MLP_H1 * DS_MLP_IN], b1[DS_MLP_H1];
    float W2[DS_MLP_H2 * DS_MLP_H1], b2[DS_MLP_H2];
    float W3[DS_MLP_H2], b3;
    float mu[DS_MLP_IN], inv_sigma[DS_MLP_IN];
    float pad_[3];
};
static_assert(sizeof(DevMlp) % 16 == 0, "DevMlp is copied as float4");

// Device copy of the paper's 8 -> 14 -> 1 ghost killer (ds_upload_mlp_single)
struct DevMlpSingle {
    float W1[DS_MLP_SINGLE_H * DS_MLP_IN], b1[DS_MLP_SINGLE_H];
    float W3[DS_MLP_SINGLE_H], b3;
    float mu[DS_MLP_IN], inv_sigma[DS_MLP_IN];
};

// Device copy of the four HLT1 line NNs (global memory, staged to shared memory by k_lines)
struct DevLines {
    float W1[DS_N_LINES][DS_LINE_H][DS_LINE_IN], b1[DS_N_LINES][DS_LINE_H];
    float W3[DS_N_LINES][DS_LINE_H], b3[DS_N_LINES];
    float mu[DS_LINE_IN], inv_sigma[DS_LINE_IN];
};
static_assert(sizeof(DevLines) % 16 == 0, "DevLines is copied as float4");

__device__ __forceinline__ int id_layer(int id) { return (id >> kIdLayerShift) & 3; }
__device__ __forceinline__ int id_sector(int id) { return (id >> kIdSectorShift) & 15; }

// x0 slice of a hit inside its (layer, sector) bin.  fp32 and monotone non-decreasing in x0, so the slices respect
// the x0 order and a window [lo, hi] in x0 maps to the slice range [xbin(lo'), xbin(hi')] for any lo' <= lo, hi' >= hi.
__device__ __forceinline__ int xbin(float x0, float off, float scale)
{
    const int t = __float2int_rd((x0 + off) * scale);   // floor, saturating, NaN -> 0
    return min(max(t, 0), kXBins - 1);
}

// The same for a table with kSlices = kXBins * k slices per (layer, sector) (k a power of two): slice of x0 =
// clamp(floor(k * t)) with t = (x0 + off) * scale the fp32 value xbin() floors; k * t is exact, so slice / k = xbin.
template <int kSlices>
__device__ __forceinline__ int xslice(float x0, float off, float scale)
{
    static_assert(kSlices % kXBins == 0, "slices refine the DS_XBINS slices of the public table");
    // floor by the conversion itself (round down, saturating, NaN -> 0), then the clamp on the integer
    const int t = __float2int_rd((x0 + off) * scale * (float)(kSlices / kXBins));
    return min(max(t, 0), kSlices - 1);
}

// Order-preserving map float -> uint32 (-0.0 is first folded onto +0.0 so that it compares equal, like IEEE ==).
__device__ __forceinline__ uint32_t float_key(float x)
{
    uint32_t u = __float_as_uint(x + 0.0f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// ---- 1-D bulk async copy global -> shared, completion on an mbarrier (PTX ISA: cp.async.bulk, mbarrier) -------------
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// Orders this thread's earlier generic-proxy accesses to shared memory (and, after a barrier, those of the threads that
// arrived at it) before its later async-proxy operations (bulk copies) on the same bytes.
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}

// dst, src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_addr(dst)),
                 "l"(src), "r"(bytes), "r"(smem_addr(bar))
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity)
{
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(ok)
            : "r"(smem_addr(bar)), "r"(parity)
            : "memory");
    }
}

// Optional per-kernel device timing (ds_profile_enable / ds_profile_read): a pair of events around each launch, on the
// launching stream.  Host side only.
struct Prof {
    struct Rec { int k; cudaEvent_t a, b; };
    bool on = false;
    std::vector<Rec> recs;
    std::vector<cudaEvent_t> pool;
    cudaEvent_t get()
    {
        cudaEvent_t e = nullptr;
        if (!pool.empty()) { e = pool.back(); pool.pop_back(); }
        else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }
        return e;
    }
    void begin(int k, cudaStream_t st)
    {
        if (!on) return;
        Rec r{k, get(), get()};
        if (r.a && r.b) { cudaEventRecord(r.a, st); recs.push_back(r); }
    }
    void end(cudaStream_t st)
    {
        if (on && !recs.empty()) cudaEventRecord(recs.back().b, st);
    }
    void release()
    {
        for (auto &r : recs) { pool.push_back(r.a); pool.push_back(r.b); }
        recs.clear();
    }
    void destroy()
    {
        release();
        for (auto e : pool) cudaEventDestroy(e);
        pool.clear();
    }
};

// Opt a kernel in to the full 227 KB of dynamic shared memory, once per (kernel instantiation, device): `done` is a static
// bit mask per instantiation (bit = device ordinal; devices >= 64 simply repeat the call), so the two runtime calls are
// not paid at every launch.  Thread-safe: the attribute is idempotent, the mask only ever gains bits.
template <typename K>
inline cudaError_t opt_in_max_smem(K kernel, unsigned long long *done)
{
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    const unsigned long long bit = dev < 64 ? 1ull << dev : 0ull;
    if (bit && (__atomic_load_n(done, __ATOMIC_ACQUIRE) & bit)) return cudaSuccess;
    cudaFuncAttributes fa;
    err = cudaFuncGetAttributes(&fa, kernel);
    if (err != cudaSuccess) return err;
    err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - (int)fa.sharedSizeBytes);
    if (err != cudaSuccess) return err;
    if (bit) __atomic_fetch_or(done, bit, __ATOMIC_RELEASE);
    return cudaSuccess;
}

// ---- launchers (host side, defined in the .cu files; all enqueue on `st` and return the launch error) ------------
// Inputs and outputs of k_layout.  Public form (ds_layout): sx0, sz, symin, symax, sw, sid, perm.  Internal form (inside
// ds_reconstruct, aux != nullptr): sx0, aux = (z, w, perm, id) per sorted position, ybounds / uniform per event, and
// symin / symax only for events whose hits do not all carry their sector's bounds (see ds_layout.cu).
struct LayoutPtrs {
    const float *x0, *z, *ymin, *ymax, *w;
    const int32_t *id;
    float *sx0, *sz, *symin, *symax, *sw;
    int32_t *sid, *perm, *bin_offsets;
    float4 *aux;
    float2 *ybounds;
    int32_t *uniform;
    int32_t *redo;   // [E] written by k_event: 1 = the event is left to k_layout + k_track
};

// only != nullptr (here and in launch_track): only the events e with only[e] != 0 are processed
cudaError_t launch_layout(const DevConst &c, const LayoutPtrs &p, const int32_t *hit_offsets, int n_events,
                          int max_event_hits_hint, const int32_t *only, cudaStream_t st, Prof &prof);

// S1..S6 in one kernel (ds_event.cu), Dv0 only; redo[e] = 1 for the events it leaves to k_layout + k_track.
// event_kernel_wanted: false for hints so large that only one block of it would fit an SM (then k_layout + k_track run alone)
bool event_kernel_wanted(const DevConst &c, int max_event_hits_hint);
cudaError_t launch_event(const DevConst &c, const ds_hits &hits, const ds_seeds &seeds, const int32_t *hit_offsets,
                         const int32_t *seed_offsets, int n_events, int max_event_hits_hint, const ds_tracks &out, int32_t *redo,
                         cudaStream_t st, Prof &prof);

cudaError_t launch_extrapolate(const DevConst &c, const ds_seeds &seeds, double *out, cudaStream_t st);

cudaError_t launch_track(const DevConst &c, const LayoutPtrs &lay, const ds_seeds &seeds, const int32_t *hit_offsets,
                         const int32_t *seed_offsets, int n_events, int max_event_hits_hint, const int32_t *only,
                         const ds_tracks &out, cudaStream_t st, Prof &prof);

cudaError_t launch_clone(const DevConst &c, const int32_t *seed_offsets, int n_events, const ds_tracks &trk, cudaStream_t st,
                         Prof &prof);

// single != nullptr: the paper's 8 -> 14 -> 1 network instead of mlp
cudaError_t launch_mlp(const DevConst &c, const DevMlp *mlp, const DevMlpSingle *single, const ds_seeds &seeds,
                       const ds_tracks &trk, cudaStream_t st, Prof &prof);

cudaError_t launch_lines(const DevLines *nets, const ds_tracks &trk, const ds_vertices &vtx, int n_events, double thr,
                         float *scores, int32_t *bits, int n_sm, cudaStream_t st, Prof &prof);

cudaError_t launch_vertex(const DevConst &c, const ds_tracks &trk, const int32_t *seed_offsets, int n_events,
                          const ds_vertices &out, void *workspace, cudaStream_t st, Prof &prof);
size_t vertex_workspace_bytes(int n_events, int64_t n_seeds);

}  // namespace ds
