// C ABI of libds (include/ds.h): handle, argument checks, workspace carving, launch order, host-buffer path.
// No arithmetic of the method lives here.
#include <cstdlib>
#include <mutex>
#include <new>

#include "ds_common.cuh"

using namespace ds;

struct ds_handle {
    int device;
    bool has_geom;
    ds_geometry geom;
    DevMlp *d_mlp;
    DevMlpSingle *d_single;   // nullptr until ds_upload_mlp_single
    bool use_single;          // the ghost killer in use is d_single (until the next ds_upload_geometry)
    DevLines *d_lines;   // nullptr until ds_upload_line_nets
    int n_sm;
    // arena of the *_host path, grown on demand
    unsigned char *arena;
    size_t arena_bytes;
    Prof prof;
};

// Scratch of ds_vertex_static (include/ds.h): a fixed device array instead of a caller's workspace.  In host code this
// name is only a stand-in for the symbol, never a device address: the address comes from cudaGetSymbolAddress (below).
static __device__ __align__(256) unsigned char ds_static_scratch[DS_STATIC_SCRATCH_BYTES];

namespace {

// Device address of ds_static_scratch on device `dev`, which must be current: resolved once per device, then cached.
std::mutex g_static_mu;
void *g_static_ptr[64] = {};

cudaError_t static_scratch_address(int dev, void **ptr)
{
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        const cudaError_t err = cudaGetSymbolAddress(&p, ds_static_scratch);
        if (err != cudaSuccess) return err;
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = p;
    }
    *ptr = g_static_ptr[dev];
    return cudaSuccess;
}

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

// Development aid: DS_FUSED=0 takes k_layout + k_track for every event (the path of Dv1 and of oversize events)
bool fused_off()
{
    static int v = -1;
    if (v < 0) {
        const char *e = getenv("DS_FUSED");
        v = (e && e[0] == '0') ? 1 : 0;
    }
    return v == 1;
}

inline size_t up256(size_t v) { return (v + 255) & ~(size_t)255; }

int n_bins_of(const ds_geometry &g) { return 4 * g.n_sectors_y * kXBins; }

bool make_const(const ds_geometry &g, const ds_params *p, DevConst &c)
{
    if (!p || p->struct_size != sizeof(ds_params)) return false;
    if (p->max_first_hits < 1 || p->max_first_hits > DS_MAX_FIRST_HITS) return false;
    if (p->vtx_newton_iters < 0 || p->vtx_newton_iters > 16) return false;
    if (p->clone_min_shared < 0) return false;
    double dmax = 0.0;
    for (int l = 0; l < 4; ++l) {
        c.z_layer[l] = g.z_layer[l];
        c.dxdy[l] = g.dxdy[l];
        c.zmag_c[l] = g.zmag_c[l];
        const double a = g.dxdy[l] < 0 ? -g.dxdy[l] : g.dxdy[l];
        if (a > dmax) dmax = a;
    }
    c.y0 = -g.y_half;
    c.inv_h = 1.0 / g.sector_height;
    c.z_seed = g.z_seed;
    c.z_ref = g.z_ref;
    c.kick = g.kick;
    c.inv_kick = 1.0 / g.kick;
    c.n_sectors = g.n_sectors_y;
    c.n_bins = n_bins_of(g);
    const float X = (float)(g.x_half + g.y_half * dmax);
    c.xb_off = X;
    c.xb_scale = (float)kXBins / (2.0f * X);
    c.w0_a = p->w0_a; c.w0_b = p->w0_b; c.w0_max = p->w0_max; c.w1_a = p->w1_a; c.w1_b = p->w1_b;
    c.y_tol = p->y_tol; c.w_mag = p->w_mag; c.chi2ndf_max = p->chi2ndf_max; c.miss_penalty = p->miss_penalty;
    c.min_hits = p->min_hits; c.max_first = p->max_first_hits;
    c.mlp_thr = p->mlp_thr; c.mlp_keep_above = p->mlp_keep_above; c.pad_ = 0;
    c.doca_max = p->doca_max; c.zv_min = p->zv_min; c.zv_max = p->zv_max;
    c.m_pi = p->m_pi; c.m_p = p->m_p; c.m_ks = p->m_ks; c.m_lambda = p->m_lambda;
    c.dm_ks = p->dm_ks; c.dm_lambda = p->dm_lambda; c.n2_min = p->n2_min;
    c.vtx_mp = p->magnet_polarity; c.gamma_c0 = p->gamma_c0; c.gamma_c1 = p->gamma_c1;
    c.vtx_iters = p->vtx_newton_iters; c.clone_min_shared = p->clone_min_shared;
    c.dv1 = p->dv1 != 0; c.mlp_fast_math = p->mlp_fast_math != 0;
    c.y_rsec = (int)(p->y_tol / g.sector_height + 1e-9) + 1; c.pad2_ = 0;
    return true;
}

bool hits_ok(const ds_hits *h)
{
    if (!h || h->n < 0 || h->n >= ((int64_t)1 << 31)) return false;
    return h->n == 0 || (h->x0 && h->z && h->ymin && h->ymax && h->w && h->id);
}

bool seeds_ok(const ds_seeds *s)
{
    if (!s || s->n < 0 || s->n >= ((int64_t)1 << 31)) return false;
    return s->n == 0 || (s->x && s->y && s->tx && s->ty && s->qop);
}

bool tracks_ok(const ds_tracks *t, int64_t n)
{
    if (!t || t->n != n) return false;
    return n == 0 || (t->x && t->y && t->tx && t->ty && t->qop && t->chi2 && t->score && t->nhits && t->hit &&
                      t->found && t->keep && (reinterpret_cast<uintptr_t>(t->hit) & 15) == 0);
}

bool vertices_ok(const ds_vertices *v)
{
    if (!v || v->capacity < 0 || !v->n_per_event || !v->offsets || !v->overflow) return false;
    return v->capacity == 0 ||
           (v->evt && v->ia && v->ib && v->x && v->y && v->z && v->doca && v->m_pipi && v->m_ppi && v->flags);
}

// carve the internal S1 output (see LayoutPtrs) out of a workspace; returns the bytes used (ws may be null: sizing)
size_t carve_layout(void *ws, int n_bins, int n_events, int64_t n_hits, LayoutPtrs &L)
{
    const size_t nh = (size_t)(n_hits > 0 ? n_hits : 1) + 4, ne = (size_t)(n_events > 0 ? n_events : 1);
    unsigned char *base = static_cast<unsigned char *>(ws);
    size_t off = 0;
    auto take = [&](size_t bytes) { unsigned char *r = base + off; off += up256(bytes); return r; };
    L.sx0 = reinterpret_cast<float *>(take(4 * nh));
    L.symin = reinterpret_cast<float *>(take(4 * nh));
    L.symax = reinterpret_cast<float *>(take(4 * nh));
    L.aux = reinterpret_cast<float4 *>(take(16 * nh));
    L.bin_offsets = reinterpret_cast<int32_t *>(take(4 * ne * (n_bins + 1)));
    L.ybounds = reinterpret_cast<float2 *>(take(sizeof(float2) * ne * (n_bins / kXBins)));
    L.uniform = reinterpret_cast<int32_t *>(take(4 * ne));
    L.redo = reinterpret_cast<int32_t *>(take(4 * ne));
    L.sz = L.sw = nullptr;
    L.sid = L.perm = nullptr;
    return off;
}

size_t layout_bytes(int n_bins, int n_events, int64_t n_hits)
{
    LayoutPtrs L;
    return carve_layout(nullptr, n_bins, n_events, n_hits, L);
}

void set_inputs(LayoutPtrs &L, const ds_hits *hits)
{
    L.x0 = hits->x0; L.z = hits->z; L.ymin = hits->ymin; L.ymax = hits->ymax; L.w = hits->w; L.id = hits->id;
}

// S1..S6.  Dv0: k_event does S1..S6 for every event that fits its staging capacity and marks the others in L.redo; k_layout
// + k_track then run for the marked events only (their blocks for the other events leave at once).  Dv1: k_layout + k_track.
cudaError_t reconstruct_launches(ds_handle *h, const DevConst &c, const LayoutPtrs &L, const ds_hits &hits, const ds_seeds &seeds,
                                 const int32_t *hit_offsets, const int32_t *seed_offsets, int n_events, int hint, const ds_tracks &out,
                                 cudaStream_t st)
{
    const int32_t *only = nullptr;
    cudaError_t err = cudaSuccess;
    if (!c.dv1 && !fused_off() && event_kernel_wanted(c, hint)) {
        err = launch_event(c, hits, seeds, hit_offsets, seed_offsets, n_events, hint, out, L.redo, st, h->prof);
        only = L.redo;
    }
    if (err == cudaSuccess) err = launch_layout(c, L, hit_offsets, n_events, hint, only, st, h->prof);
    if (err == cudaSuccess) err = launch_track(c, L, seeds, hit_offsets, seed_offsets, n_events, hint, only, out, st, h->prof);
    return err;
}

}  // namespace

extern "C" {

int ds_version(void) { return DS_VERSION; }

const char *ds_error_string(int code)
{
    switch (code) {
        case DS_OK: return "ok";
        case DS_E_ARG: return "invalid argument";
        case DS_E_NOGEOM: return "geometry not uploaded";
        case DS_E_WORKSPACE: return "workspace missing or too small";
        case DS_E_CUDA: return "CUDA error";
        case DS_E_LIMIT: return "call larger than the fixed scratch of ds_vertex_static (DS_STATIC_MAX_EVENTS / DS_STATIC_MAX_SEEDS)";
        default: return "unknown error";
    }
}

int ds_create(ds_handle **h, int cuda_device)
{
    if (!h) return DS_E_ARG;
    *h = nullptr;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || cuda_device < 0 || cuda_device >= n) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    DeviceGuard guard(cuda_device);
    if (!guard.ok) return DS_E_CUDA;
    ds_handle *p = new (std::nothrow) ds_handle();
    if (!p) return DS_E_CUDA;
    p->device = cuda_device;
    p->has_geom = false;
    p->arena = nullptr;
    p->arena_bytes = 0;
    p->d_lines = nullptr;
    p->d_single = nullptr;
    p->use_single = false;
    p->n_sm = 0;
    cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, cuda_device);
    if (cudaMalloc(&p->d_mlp, sizeof(DevMlp)) != cudaSuccess) {
        cudaGetLastError();
        delete p;
        return DS_E_CUDA;
    }
    *h = p;
    return DS_OK;
}

void ds_destroy(ds_handle *h)
{
    if (!h) return;
    DeviceGuard guard(h->device);
    if (h->d_mlp) cudaFree(h->d_mlp);
    if (h->d_lines) cudaFree(h->d_lines);
    if (h->d_single) cudaFree(h->d_single);
    if (h->arena) cudaFree(h->arena);
    h->prof.destroy();
    delete h;
}

int ds_upload_geometry(ds_handle *h, const ds_geometry *g, const ds_mlp *m)
{
    if (!h || !g || !m) return DS_E_ARG;
    if (g->struct_size != sizeof(ds_geometry) || m->struct_size != sizeof(ds_mlp)) return DS_E_ARG;
    if (g->n_sectors_y < 1 || g->n_sectors_y > DS_MAX_SECTORS || !(g->sector_height > 0.0) || !(g->x_half > 0.0) ||
        !(g->y_half > 0.0) || g->kick == 0.0)
        return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    DevMlp host;
    for (int j = 0; j < DS_MLP_H1; ++j) {
        for (int i = 0; i < DS_MLP_IN; ++i) host.W1[j * DS_MLP_IN + i] = m->W1[j][i];
        host.b1[j] = m->b1[j];
    }
    for (int j = 0; j < DS_MLP_H2; ++j) {
        for (int i = 0; i < DS_MLP_H1; ++i) host.W2[j * DS_MLP_H1 + i] = m->W2[j][i];
        host.b2[j] = m->b2[j];
        host.W3[j] = m->W3[j];
    }
    host.b3 = m->b3;
    for (int i = 0; i < DS_MLP_IN; ++i) { host.mu[i] = m->mu[i]; host.inv_sigma[i] = m->inv_sigma[i]; }
    host.pad_[0] = host.pad_[1] = host.pad_[2] = 0.f;
    if (cudaMemcpy(h->d_mlp, &host, sizeof host, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    h->geom = *g;
    h->has_geom = true;
    h->use_single = false;
    return DS_OK;
}

int ds_upload_mlp_single(ds_handle *h, const ds_mlp_single *m)
{
    if (!h || !m || m->struct_size != sizeof(ds_mlp_single)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    static_assert(sizeof(DevMlpSingle) <= sizeof(ds_mlp_single) - offsetof(ds_mlp_single, W1) && offsetof(DevMlpSingle, inv_sigma) == offsetof(ds_mlp_single, inv_sigma) - offsetof(ds_mlp_single, W1), "same layout after struct_size");
    if (!h->d_single && cudaMalloc(&h->d_single, sizeof(DevMlpSingle)) != cudaSuccess) {
        cudaGetLastError();
        h->d_single = nullptr;
        return DS_E_CUDA;
    }
    if (cudaMemcpy(h->d_single, &m->W1, sizeof(DevMlpSingle), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    h->use_single = true;
    return DS_OK;
}

int ds_layout(ds_handle *h, const ds_hits *hits, const int32_t *hit_offsets, int n_events, const ds_params *p,
              ds_layout_out *out, void *cuda_stream)
{
    if (!h || !hits_ok(hits) || !hit_offsets || n_events < 0 || !out) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    if (out->n != hits->n || !out->bin_offsets) return DS_E_ARG;
    if (hits->n > 0 && !(out->x0 && out->z && out->ymin && out->ymax && out->w && out->id && out->perm)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    LayoutPtrs L;
    set_inputs(L, hits);
    L.sx0 = out->x0; L.sz = out->z; L.symin = out->ymin; L.symax = out->ymax; L.sw = out->w; L.sid = out->id;
    L.perm = out->perm; L.bin_offsets = out->bin_offsets;
    L.aux = nullptr; L.ybounds = nullptr; L.uniform = nullptr; L.redo = nullptr;   // the public SoA form
    if (launch_layout(c, L, hit_offsets, n_events, p->max_event_hits_hint, nullptr, (cudaStream_t)cuda_stream, h->prof) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_extrapolate(ds_handle *h, const ds_seeds *seeds, const ds_params *p, double *out, void *cuda_stream)
{
    if (!h || !seeds_ok(seeds) || (!out && seeds->n > 0)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    if (launch_extrapolate(c, *seeds, out, (cudaStream_t)cuda_stream) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

size_t ds_workspace_bytes(const ds_handle *h, int n_events, int64_t n_hits, int64_t n_seeds)
{
    (void)n_seeds;
    const int nb = (h && h->has_geom) ? n_bins_of(h->geom) : 4 * DS_MAX_SECTORS * kXBins;
    return layout_bytes(nb, n_events, n_hits);
}

int ds_ghost_killer(ds_handle *h, const ds_seeds *seeds, const ds_params *p, ds_tracks *trk, void *cuda_stream)
{
    if (!h || !seeds_ok(seeds) || !tracks_ok(trk, seeds ? seeds->n : 0)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    if (launch_mlp(c, h->d_mlp, h->use_single ? h->d_single : nullptr, *seeds, *trk, (cudaStream_t)cuda_stream, h->prof) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_clone_kill(ds_handle *h, const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *trk,
                  void *cuda_stream)
{
    if (!h || !seed_offsets || n_events < 0 || !trk || !tracks_ok(trk, trk->n)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c) || c.clone_min_shared <= 0) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    if (launch_clone(c, seed_offsets, n_events, *trk, (cudaStream_t)cuda_stream, h->prof) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_reconstruct(ds_handle *h, const ds_hits *hits, const ds_seeds *seeds, const int32_t *hit_offsets,
                   const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *out, void *workspace,
                   size_t workspace_bytes, void *cuda_stream)
{
    if (!h || !hits_ok(hits) || !seeds_ok(seeds) || !hit_offsets || !seed_offsets || n_events < 0) return DS_E_ARG;
    if (!tracks_ok(out, seeds->n)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255) != 0 ||
        workspace_bytes < layout_bytes(c.n_bins, n_events, hits->n))
        return DS_E_WORKSPACE;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LayoutPtrs L;
    set_inputs(L, hits);
    carve_layout(workspace, c.n_bins, n_events, hits->n, L);
    cudaError_t err = reconstruct_launches(h, c, L, *hits, *seeds, hit_offsets, seed_offsets, n_events, p->max_event_hits_hint, *out, st);
    if (err == cudaSuccess) err = launch_clone(c, seed_offsets, n_events, *out, st, h->prof);
    if (err == cudaSuccess) err = launch_mlp(c, h->d_mlp, h->use_single ? h->d_single : nullptr, *seeds, *out, st, h->prof);
    if (err != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

size_t ds_vertex_workspace_bytes(const ds_handle *h, int n_events, int64_t n_seeds)
{
    (void)h;
    return vertex_workspace_bytes(n_events, n_seeds);
}

int ds_upload_line_nets(ds_handle *h, const ds_line_nets *nets)
{
    if (!h || !nets || nets->struct_size != sizeof(ds_line_nets)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    static_assert(sizeof(DevLines) == sizeof(ds_line_nets) - offsetof(ds_line_nets, W1), "same layout after struct_size");
    if (!h->d_lines && cudaMalloc(&h->d_lines, sizeof(DevLines)) != cudaSuccess) {
        cudaGetLastError();
        h->d_lines = nullptr;
        return DS_E_CUDA;
    }
    if (cudaMemcpy(h->d_lines, &nets->W1, sizeof(DevLines), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_lines(ds_handle *h, const ds_tracks *trk, const ds_vertices *vtx, int n_events, double threshold, float *scores,
             int32_t *bits, void *cuda_stream)
{
    if (!h || !trk || trk->n < 0 || n_events < 0 || !vertices_ok(vtx)) return DS_E_ARG;
    if (trk->n > 0 && !(trk->tx && trk->ty && trk->qop && trk->chi2)) return DS_E_ARG;
    if (vtx->capacity > 0 && (!scores || !bits)) return DS_E_ARG;
    if (!h->d_lines) return DS_E_NOGEOM;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    if (launch_lines(h->d_lines, *trk, *vtx, n_events, threshold, scores, bits, h->n_sm, (cudaStream_t)cuda_stream, h->prof) !=
        cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_vertex(ds_handle *h, const ds_tracks *trk, const int32_t *seed_offsets, int n_events, const ds_params *p,
              ds_vertices *out, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!h || !trk || trk->n < 0 || !seed_offsets || n_events < 0 || !vertices_ok(out)) return DS_E_ARG;
    if (trk->n > 0 && !(trk->x && trk->y && trk->tx && trk->ty && trk->qop && trk->keep)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 255) != 0 ||
        workspace_bytes < vertex_workspace_bytes(n_events, trk->n))
        return DS_E_WORKSPACE;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    if (launch_vertex(c, *trk, seed_offsets, n_events, *out, workspace, (cudaStream_t)cuda_stream, h->prof) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_vertex_static_setup(ds_handle *h)
{
    if (!h) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    void *scratch = nullptr;
    if (static_scratch_address(h->device, &scratch) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_vertex_static(ds_handle *h, const ds_tracks *trk, const int32_t *seed_offsets, int n_events, const ds_params *p,
                     ds_vertices *out, void *cuda_stream)
{
    if (!h || !trk || trk->n < 0 || !seed_offsets || n_events < 0 || !vertices_ok(out)) return DS_E_ARG;
    if (trk->n > 0 && !(trk->x && trk->y && trk->tx && trk->ty && trk->qop && trk->keep)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    if (n_events > DS_STATIC_MAX_EVENTS || trk->n > DS_STATIC_MAX_SEEDS ||
        vertex_workspace_bytes(n_events, trk->n) > (size_t)DS_STATIC_SCRATCH_BYTES)
        return DS_E_LIMIT;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    void *scratch = nullptr;
    if (static_scratch_address(h->device, &scratch) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    Prof none;   // never on: no event is created or recorded for these launches
    // launch_vertex clears what has to start at zero (the group sums) on the stream, ahead of its kernels; everything
    // else it reads of the scratch it has written in the same call
    if (launch_vertex(c, *trk, seed_offsets, n_events, *out, scratch, (cudaStream_t)cuda_stream, none) != cudaSuccess) {
        cudaGetLastError();
        return DS_E_CUDA;
    }
    return DS_OK;
}

int ds_process_host(ds_handle *h, const ds_hits *hits, const ds_seeds *seeds, const int32_t *hit_offsets,
                    const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *out_tracks,
                    ds_vertices *out_vertices, int64_t *n_vertices_total, void *cuda_stream)
{
    if (!h || !hits_ok(hits) || !seeds_ok(seeds) || !hit_offsets || !seed_offsets || n_events < 0) return DS_E_ARG;
    if (!tracks_ok(out_tracks, seeds->n) || !vertices_ok(out_vertices)) return DS_E_ARG;
    if (!h->has_geom) return DS_E_NOGEOM;
    DevConst c;
    if (!make_const(h->geom, p, c)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nh = (size_t)hits->n, ns = (size_t)seeds->n, ne = (size_t)n_events, cap = (size_t)out_vertices->capacity;
    const size_t ws_rec = layout_bytes(c.n_bins, n_events, hits->n), ws_vtx = vertex_workspace_bytes(n_events, seeds->n);
    // The arena is carved by ONE piece of code, run twice: first on a null base to add up the bytes (so that the size
    // can never disagree with the carving), then on the arena.
    cudaError_t err = cudaSuccess;
    ds_hits dh;
    ds_seeds dsd;
    ds_tracks dt;
    ds_vertices dv;
    const int32_t *d_hoff = nullptr, *d_soff = nullptr;
    void *wrec = nullptr, *wvtx = nullptr;
    auto carve = [&](unsigned char *base, bool copy) -> size_t {
        size_t off = 0;
        auto take = [&](size_t bytes) { unsigned char *r = base + off; off += up256(bytes); return r; };
        auto h2d = [&](const void *src, size_t bytes) -> void * {
            void *d = take(bytes + 4);
            if (copy && bytes && err == cudaSuccess) err = cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st);
            return d;
        };
        dh.n = hits->n;
        dh.x0 = (const float *)h2d(hits->x0, 4 * nh); dh.z = (const float *)h2d(hits->z, 4 * nh);
        dh.ymin = (const float *)h2d(hits->ymin, 4 * nh); dh.ymax = (const float *)h2d(hits->ymax, 4 * nh);
        dh.w = (const float *)h2d(hits->w, 4 * nh); dh.id = (const int32_t *)h2d(hits->id, 4 * nh);
        dsd.n = seeds->n;
        dsd.x = (const float *)h2d(seeds->x, 4 * ns); dsd.y = (const float *)h2d(seeds->y, 4 * ns);
        dsd.tx = (const float *)h2d(seeds->tx, 4 * ns); dsd.ty = (const float *)h2d(seeds->ty, 4 * ns);
        dsd.qop = (const float *)h2d(seeds->qop, 4 * ns);
        {
            void *d = h2d(seeds->chi2, seeds->chi2 ? 4 * ns : 0);
            dsd.chi2 = seeds->chi2 ? (const float *)d : nullptr;
        }
        d_hoff = (const int32_t *)h2d(hit_offsets, 4 * (ne + 1));
        d_soff = (const int32_t *)h2d(seed_offsets, 4 * (ne + 1));
        dt.n = seeds->n;
        dt.x = (float *)take(4 * ns + 4); dt.y = (float *)take(4 * ns + 4); dt.tx = (float *)take(4 * ns + 4);
        dt.ty = (float *)take(4 * ns + 4); dt.qop = (float *)take(4 * ns + 4); dt.chi2 = (float *)take(4 * ns + 4);
        dt.score = (float *)take(4 * ns + 4); dt.nhits = (int32_t *)take(4 * ns + 4); dt.found = (int32_t *)take(4 * ns + 4);
        dt.keep = (int32_t *)take(4 * ns + 4); dt.hit = (int32_t *)take(16 * ns + 16);
        dv.capacity = out_vertices->capacity;
        dv.evt = (int32_t *)take(4 * cap + 4); dv.ia = (int32_t *)take(4 * cap + 4); dv.ib = (int32_t *)take(4 * cap + 4);
        dv.x = (float *)take(4 * cap + 4); dv.y = (float *)take(4 * cap + 4); dv.z = (float *)take(4 * cap + 4);
        dv.doca = (float *)take(4 * cap + 4); dv.m_pipi = (float *)take(4 * cap + 4); dv.m_ppi = (float *)take(4 * cap + 4);
        dv.flags = (int32_t *)take(4 * cap + 4);
        dv.n_per_event = (int32_t *)take(4 * ne + 4);
        dv.offsets = (int64_t *)take(8 * (ne + 1));
        dv.overflow = (int32_t *)take(256);
        wrec = take(ws_rec);
        wvtx = take(ws_vtx);
        return off;
    };
    const size_t need = carve(nullptr, false);
    if (need > h->arena_bytes) {
        if (h->arena) cudaFree(h->arena);
        h->arena = nullptr;
        h->arena_bytes = 0;
        const size_t want = need + need / 8;
        if (cudaMalloc(&h->arena, want) != cudaSuccess) {
            cudaGetLastError();
            return DS_E_CUDA;
        }
        h->arena_bytes = want;
    }
    carve(h->arena, true);
    if (err != cudaSuccess) { cudaGetLastError(); return DS_E_CUDA; }

    LayoutPtrs L;
    set_inputs(L, &dh);
    carve_layout(wrec, c.n_bins, n_events, hits->n, L);
    err = reconstruct_launches(h, c, L, dh, dsd, d_hoff, d_soff, n_events, p->max_event_hits_hint, dt, st);
    if (err == cudaSuccess) err = launch_clone(c, d_soff, n_events, dt, st, h->prof);
    if (err == cudaSuccess) err = launch_mlp(c, h->d_mlp, h->use_single ? h->d_single : nullptr, dsd, dt, st, h->prof);
    if (err == cudaSuccess) err = launch_vertex(c, dt, d_soff, n_events, dv, wvtx, st, h->prof);
    auto d2h = [&](void *dst, const void *src, size_t bytes) {
        if (bytes && err == cudaSuccess) err = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st);
    };
    d2h(out_vertices->offsets, dv.offsets, 8 * (ne + 1));
    d2h(out_vertices->n_per_event, dv.n_per_event, 4 * ne);
    d2h(out_vertices->overflow, dv.overflow, 4);
    d2h(out_tracks->x, dt.x, 4 * ns); d2h(out_tracks->y, dt.y, 4 * ns); d2h(out_tracks->tx, dt.tx, 4 * ns);
    d2h(out_tracks->ty, dt.ty, 4 * ns); d2h(out_tracks->qop, dt.qop, 4 * ns); d2h(out_tracks->chi2, dt.chi2, 4 * ns);
    d2h(out_tracks->score, dt.score, 4 * ns); d2h(out_tracks->nhits, dt.nhits, 4 * ns);
    d2h(out_tracks->found, dt.found, 4 * ns); d2h(out_tracks->keep, dt.keep, 4 * ns); d2h(out_tracks->hit, dt.hit, 16 * ns);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) { cudaGetLastError(); return DS_E_CUDA; }
    const int64_t total = out_vertices->offsets[n_events];
    if (n_vertices_total) *n_vertices_total = total;
    const size_t nv = (size_t)(total < out_vertices->capacity ? total : out_vertices->capacity);
    d2h(out_vertices->evt, dv.evt, 4 * nv); d2h(out_vertices->ia, dv.ia, 4 * nv); d2h(out_vertices->ib, dv.ib, 4 * nv);
    d2h(out_vertices->x, dv.x, 4 * nv); d2h(out_vertices->y, dv.y, 4 * nv); d2h(out_vertices->z, dv.z, 4 * nv);
    d2h(out_vertices->doca, dv.doca, 4 * nv); d2h(out_vertices->m_pipi, dv.m_pipi, 4 * nv);
    d2h(out_vertices->m_ppi, dv.m_ppi, 4 * nv); d2h(out_vertices->flags, dv.flags, 4 * nv);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) { cudaGetLastError(); return DS_E_CUDA; }
    return DS_OK;
}

int ds_profile_enable(ds_handle *h, int on)
{
    if (!h) return DS_E_ARG;
    h->prof.on = on != 0;
    return DS_OK;
}

int ds_profile_read(ds_handle *h, ds_profile *out)
{
    if (!h || !out || out->struct_size != sizeof(ds_profile)) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    for (int k = 0; k < DS_K_COUNT; ++k) { out->ms[k] = 0.0; out->launches[k] = 0; }
    int rc = DS_OK;
    for (auto &r : h->prof.recs) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess) {
            cudaGetLastError();
            rc = DS_E_CUDA;
            continue;
        }
        out->ms[r.k] += (double)ms;
        out->launches[r.k] += 1;
    }
    h->prof.release();
    return rc;
}

namespace {
__global__ void k_fma_peak(double *out, int iters)
{
    double a0 = threadIdx.x * 1e-9, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0, a4 = a0 + 4.0, a5 = a0 + 5.0, a6 = a0 + 6.0, a7 = a0 + 7.0;
    const double m = 1.0000001, b = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
        a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
    }
    if (a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 == -1.0) out[0] = a0;   // never true: keeps the loop alive
}
}  // namespace

int ds_measure_dfma_peak(ds_handle *h, double *tflops)
{
    if (!h || !tflops) return DS_E_ARG;
    DeviceGuard guard(h->device);
    if (!guard.ok) return DS_E_CUDA;
    double *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaMalloc(&d, sizeof(double)) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cudaGetLastError();
        if (d) cudaFree(d);
        if (e0) cudaEventDestroy(e0);
        return DS_E_CUDA;
    }
    const int sms = h->n_sm > 0 ? h->n_sm : 148, threads = 256, blocks = sms * 8, iters = 1 << 15;
    k_fma_peak<<<blocks, threads>>>(d, 256);   // warm-up
    cudaEventRecord(e0);
    k_fma_peak<<<blocks, threads>>>(d, iters);
    cudaEventRecord(e1);
    float ms = 0.f;
    const cudaError_t err = cudaEventSynchronize(e1) == cudaSuccess ? cudaEventElapsedTime(&ms, e0, e1) : cudaErrorUnknown;
    cudaFree(d);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess || !(ms > 0.f)) { cudaGetLastError(); return DS_E_CUDA; }
    *tflops = 2.0 * 8.0 * (double)iters * (double)threads * (double)blocks / ((double)ms * 1e-3) / 1e12;
    return DS_OK;
}

const char *ds_kernel_name(int k)
{
    static const char *names[DS_K_COUNT] = {"k_layout", "k_track", "k_mlp", "k_vertex_count", "k_vertex_scan", "k_vertex_write",
                                               "k_clone", "k_lines", "k_event"};
    return (k >= 0 && k < DS_K_COUNT) ? names[k] : nullptr;
}

}  // extern "C"
