// api.cu -- the C-ABI of libtridsk (include/tridsk.h): handles, host-side ligand packing, staging of
// host buffers, and the CUDA-graph-captured launch series of tridsk_dock (hot-path step a10).
// No arithmetic of the method runs on the host: every step of the path is in the kernels.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <omp.h>

#include <algorithm>
#include <cmath>
#include <new>

#include <nvtx3/nvToolsExt.h>

#include "internal.h"
#include <mutex>

// ---------------------------------------------------------------------------------------- helpers
// NVTX range around a C-ABI call: captures under nsys / ncu name the four hot-path calls.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};
// Every entry point makes the ctx's device current: handles of several devices can live in one process.
#define ENTER(ctx)                                                                                 \
    do {                                                                                           \
        int dev_ = -1;                                                                             \
        if (cudaGetDevice(&dev_) != cudaSuccess || dev_ != (ctx)->device) {                        \
            cudaError_t e_ = cudaSetDevice((ctx)->device);                                         \
            if (e_ != cudaSuccess) return fail((ctx), TRIDSK_ECUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e_)); \
        }                                                                                          \
    } while (0)
static int fail(tridsk_ctx* ctx, int code, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return code;
}
#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA,       \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

// tridsk_dock_static (end of this file): resolves the device address of its static scratch array on the current device
static cudaError_t dock_static_prepare(int device);

static bool is_device_ptr(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static int scratch(tridsk_ctx* ctx, int slot, size_t bytes, void** out) {
    if (bytes > ctx->scratch_bytes[slot]) {
        if (ctx->scratch[slot]) { CK(cudaStreamSynchronize(ctx->stream)); CK(cudaFree(ctx->scratch[slot])); }
        ctx->scratch[slot] = nullptr; ctx->scratch_bytes[slot] = 0;
        size_t cap = bytes + bytes / 4 + 256;
        CK(cudaMalloc(&ctx->scratch[slot], cap));
        ctx->scratch_bytes[slot] = cap;
    }
    *out = ctx->scratch[slot];
    return TRIDSK_OK;
}

// device view of an input buffer: the pointer itself if it is device memory, else a staged copy
static int stage_in(tridsk_ctx* ctx, int slot, const void* p, size_t bytes, const void** out) {
    if (is_device_ptr(p)) { *out = p; return TRIDSK_OK; }
    void* d;
    int rc = scratch(ctx, slot, bytes, &d);
    if (rc) return rc;
    CK(cudaMemcpyAsync(d, p, bytes, cudaMemcpyHostToDevice, ctx->stream));
    *out = d;
    return TRIDSK_OK;
}

// host poses: the quaternion of every pose must have a finite, non-zero norm (tridsk.h conventions)
static bool host_quats_ok(const float* poses, size_t n_pose, int pose_stride) {
    for (size_t i = 0; i < n_pose; ++i) {
        const float* q = poses + i * pose_stride + 3;
        const float n2 = q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];
        if (!(n2 > 0.f) || !std::isfinite(n2)) return false;
    }
    return true;
}

static void to_dparams(const tridsk_params* p, DParams* d) {
    d->w_long = p->w_long; d->w_clash = p->w_clash; d->w_hbond = p->w_hbond;
    d->long_mu = p->long_mu; d->long_inv_two_sigma2 = 1.0f / p->long_two_sigma2; d->long_dmax = p->long_dmax;
    d->hb_mu = p->hb_mu; d->hb_inv_two_sigma2 = 1.0f / (2.0f * p->hb_sigma * p->hb_sigma);
    d->hb_dmax = p->hb_dmax; d->hb_dclash = p->hb_dclash;
    d->d_floor = p->d_floor; d->k_wall = p->k_wall;
    d->beta = p->beta; d->lr = p->lr; d->adam_b1 = p->adam_b1; d->adam_b2 = p->adam_b2; d->adam_eps = p->adam_eps;
    d->pert_trans = p->pert_trans; d->pert_rot = p->pert_rot; d->w_tor = p->w_tor;
    d->n_refine = p->n_refine;
}

// the constants every kernel divides by or takes a logarithm / square root of
static int check_params(tridsk_ctx* ctx, const tridsk_params* p) {
    const float pos[] = {p->long_two_sigma2, p->hb_sigma, p->d_floor, p->hb_dclash, p->lr};
    for (float v : pos) if (!(v > 0.f) || !std::isfinite(v)) return fail(ctx, TRIDSK_EINVAL, "long_two_sigma2, hb_sigma, d_floor, hb_dclash and lr must be > 0");
    const float fin[] = {p->w_long, p->w_clash, p->w_hbond, p->long_mu, p->long_dmax, p->hb_mu, p->hb_dmax, p->k_wall, p->beta,
                         p->adam_b1, p->adam_b2, p->adam_eps, p->pert_trans, p->pert_rot, p->w_tor};
    for (float v : fin) if (!std::isfinite(v)) return fail(ctx, TRIDSK_EINVAL, "non-finite parameter");
    if (!(p->adam_b1 >= 0.f && p->adam_b1 < 1.f && p->adam_b2 >= 0.f && p->adam_b2 < 1.f)) return fail(ctx, TRIDSK_EINVAL, "adam_b1, adam_b2 must lie in [0, 1)");
    if (p->n_refine < 0) return fail(ctx, TRIDSK_EINVAL, "n_refine < 0");
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- lifetime
extern "C" void tridsk_default_params(tridsk_params* p) {
    p->w_long = 0.2f; p->w_clash = 10.0f; p->w_hbond = 0.6f;
    p->long_mu = 3.0f; p->long_two_sigma2 = 4.0f; p->long_dmax = 10.0f; /* P:113, G2 */
    p->hb_mu = 2.88f; p->hb_sigma = 0.3f; p->hb_dmax = 3.4f; p->hb_dclash = 2.6f;
    p->d_floor = 0.05f; p->k_wall = 10.0f;                              /* G4, G8 */
    p->beta = 0.069f; p->lr = 0.1f; p->adam_b1 = 0.9f; p->adam_b2 = 0.999f; p->adam_eps = 1e-8f;
    p->pert_trans = 2.0f; p->pert_rot = 0.5f;                           /* G11 */
    p->w_tor = 0.01f;
    p->n_refine = 1;
}

extern "C" int tridsk_create(tridsk_ctx** out, int device, void* cuda_stream) {
    if (!out) return TRIDSK_EINVAL;
    *out = nullptr;
    tridsk_ctx* ctx = new (std::nothrow) tridsk_ctx();
    if (!ctx) return TRIDSK_ENOMEM;
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaSetDevice(device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) {           // no CPU fallback: fail loudly
        fprintf(stderr, "tridsk_create: %s\n", cudaGetErrorString(e));
        delete ctx;
        return TRIDSK_ECUDA;
    }
    ctx->sm_count = prop.multiProcessorCount;
    // kernel attributes are per device: opt every kernel in to its shared-memory size on THIS device
    e = mc_lane_prepare(TRIDSK_SMEM_MAX_CTA);
    if (e == cudaSuccess) e = mc_cta_prepare();
    if (e == cudaSuccess) e = topk_prepare();
    if (e == cudaSuccess) e = dock_static_prepare(device);
    if (e != cudaSuccess) { fprintf(stderr, "tridsk_create: %s\n", cudaGetErrorString(e)); delete ctx; return TRIDSK_ECUDA; }
    if (!ctx->stream) {               // the legacy default stream cannot be captured into a graph: own one
        e = cudaStreamCreateWithFlags(&ctx->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { fprintf(stderr, "tridsk_create: %s\n", cudaGetErrorString(e)); delete ctx; return TRIDSK_ECUDA; }
        ctx->own_stream = true;
    }
    {
        cudaMemPoolProps pp;
        memset(&pp, 0, sizeof(pp));
        pp.allocType = cudaMemAllocationTypePinned;
        pp.location.type = cudaMemLocationTypeDevice;
        pp.location.id = device;
        e = cudaMemPoolCreate(&ctx->pool, &pp);
        if (e == cudaSuccess) {
            unsigned long long keep = ~0ULL;
            e = cudaMemPoolSetAttribute(ctx->pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        if (e != cudaSuccess) { fprintf(stderr, "tridsk_create: %s\n", cudaGetErrorString(e)); tridsk_destroy(ctx); return TRIDSK_ECUDA; }
    }
    *out = ctx;
    return TRIDSK_OK;
}

extern "C" void tridsk_destroy(tridsk_ctx* ctx) {
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    for (auto& ent : ctx->grid_cache) tridsk_free_grid(ent.grid);
    ctx->grid_cache.clear();
    *ctx->alive = false;
    if (ctx->pool) cudaMemPoolDestroy(ctx->pool);   // outstanding grids keep their memory until they are freed
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    for (int i = 0; i < 3; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    if (ctx->fork_ev) cudaEventDestroy(ctx->fork_ev);
    for (int i = 0; i < TRIDSK_BRANCHES; ++i) {
        if (ctx->join_ev[i]) cudaEventDestroy(ctx->join_ev[i]);
        if (ctx->side[i]) cudaStreamDestroy(ctx->side[i]);
    }
    for (int i = 0; i < TRIDSK_SCRATCH; ++i) if (ctx->scratch[i]) cudaFree(ctx->scratch[i]);
    if (ctx->pin) cudaFreeHost(ctx->pin);
    if (ctx->pin_ev) cudaEventDestroy(ctx->pin_ev);
    if (ctx->own_stream) cudaStreamDestroy(ctx->stream);
    delete ctx;
}

extern "C" const char* tridsk_last_error(const tridsk_ctx* ctx) { return ctx ? ctx->err.c_str() : "null ctx"; }
extern "C" long long tridsk_launch_count(const tridsk_ctx* ctx) { return ctx ? ctx->launches : 0; }
extern "C" int tridsk_synchronize(tridsk_ctx* ctx) {
    if (!ctx) return TRIDSK_EINVAL;
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- grid
static int check_types(tridsk_ctx* ctx, const tridsk_types* t) {
    if (!t || !t->radius || !t->hb_role || t->n_types < 1) return fail(ctx, TRIDSK_EINVAL, "bad type table");
    if (t->n_types > TRIDSK_MAX_TYPES) return fail(ctx, TRIDSK_ELIMIT, "n_types > 32");
    return TRIDSK_OK;
}

static int new_grid(tridsk_ctx* ctx, int n_types, const float origin[3], const int dims[3], float spacing, tridsk_grid** out) {
    if (!origin || !dims || dims[0] < 2 || dims[1] < 2 || dims[2] < 2 || !(spacing > 0.f) || n_types < 1)
        return fail(ctx, TRIDSK_EINVAL, "bad grid geometry");
    if (n_types > TRIDSK_MAX_TYPES) return fail(ctx, TRIDSK_ELIMIT, "n_types > 32");
    tridsk_grid* g = new (std::nothrow) tridsk_grid();
    if (!g) return fail(ctx, TRIDSK_ENOMEM, "host alloc");
    g->ctx = ctx; g->ctx_alive = ctx->alive;
    g->d.nx = dims[0]; g->d.ny = dims[1]; g->d.nz = dims[2]; g->d.n_types = n_types;
    g->d.plane = (size_t)dims[0] * dims[1] * dims[2];
    g->d.ox = origin[0]; g->d.oy = origin[1]; g->d.oz = origin[2];
    g->d.h = spacing; g->d.inv_h = 1.0f / spacing;
    cudaError_t e = cudaMallocFromPoolAsync((void**)&g->g, sizeof(float) * g->d.plane * n_types, ctx->pool, ctx->stream);
    if (e == cudaSuccess)                                                                  // cell-packed copy (DGrid::gp)
        e = cudaMallocFromPoolAsync((void**)&g->gp, 2 * sizeof(float4) * g->d.plane * n_types, ctx->pool, ctx->stream);
    if (e != cudaSuccess) {
        if (g->g) cudaFreeAsync(g->g, ctx->stream);
        delete g;
        return fail(ctx, TRIDSK_ENOMEM, std::string("grid alloc: ") + cudaGetErrorString(e));
    }
    g->d.g = g->g; g->d.gp = g->gp;
    *out = g;
    return TRIDSK_OK;
}

extern "C" int tridsk_build_grid(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec,
                                 const tridsk_types* types, const tridsk_params* params,
                                 const float origin[3], const int dims[3], float spacing, tridsk_grid** out) {
    if (!ctx || !out || !params || !rec_xyz || !rec_type || n_rec < 0) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_build_grid");
    if (int prc = check_params(ctx, params)) return prc;
    *out = nullptr;
    int rc = check_types(ctx, types);
    if (rc) return rc;
    const int nt = types->n_types;
    // type-pair table: operands of the pair function, not results
    std::vector<float> tab(4 * (size_t)nt * nt);
    float dc_max = params->hb_dmax;
    for (int s = 0; s < nt; ++s)
        for (int t = 0; t < nt; ++t) {
            const unsigned char rs = types->hb_role[s], rt = types->hb_role[t];
            const bool hb = ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
            const float dvdw = types->radius[s] + types->radius[t];
            const float dc = hb ? params->hb_dclash : dvdw;
            float* e = &tab[4 * ((size_t)s * nt + t)];
            e[0] = dvdw + params->long_mu; e[1] = dc; e[2] = hb ? 1.f : 0.f; e[3] = 1.0f / dc;
            dc_max = std::max(dc_max, dc);
        }
    tridsk_grid* g = nullptr;
    rc = new_grid(ctx, nt, origin, dims, spacing, &g);
    if (rc) return rc;
    // scratch 0: [bad flag (16 B) | float4 rec[n_rec]], scratch 1: table, scratch 4: staged host inputs
    char* d_rec0; void* d_tab;
    const void *d_xyz = nullptr, *d_typ = nullptr;
    if ((rc = scratch(ctx, 0, 16 + sizeof(float4) * std::max(n_rec, 1), (void**)&d_rec0)) ||
        (rc = scratch(ctx, 1, sizeof(float) * (tab.size() + nt), &d_tab))) { tridsk_free_grid(g); return rc; }
    const size_t b_xyz = (sizeof(float) * 3 * (size_t)n_rec + 15) / 16 * 16;
    const bool h_xyz = n_rec && !is_device_ptr(rec_xyz), h_typ = n_rec && !is_device_ptr(rec_type);
    char* stage = nullptr;
    if ((h_xyz || h_typ) && (rc = scratch(ctx, 4, b_xyz + sizeof(int) * n_rec, (void**)&stage))) { tridsk_free_grid(g); return rc; }
    DParams P;
    to_dparams(params, &P);
    int* d_bad = (int*)d_rec0;
    float4* d_rec = (float4*)(d_rec0 + 16);
    cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(int), ctx->stream);
    if (e == cudaSuccess && h_xyz) e = cudaMemcpyAsync(stage, rec_xyz, sizeof(float) * 3 * n_rec, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess && h_typ) e = cudaMemcpyAsync(stage + b_xyz, rec_type, sizeof(int) * n_rec, cudaMemcpyHostToDevice, ctx->stream);
    d_xyz = h_xyz ? (const void*)stage : (const void*)rec_xyz;
    d_typ = h_typ ? (const void*)(stage + b_xyz) : (const void*)rec_type;
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_tab, tab.data(), sizeof(float) * tab.size(), cudaMemcpyHostToDevice, ctx->stream);
    float* d_rad = (float*)d_tab + tab.size();
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_rad, types->radius, sizeof(float) * nt, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = launch_rec_pack(ctx->stream, (const float*)d_xyz, (const int*)d_typ, n_rec, nt, d_rec, d_bad);
    if (e == cudaSuccess) e = launch_grid_build(ctx->stream, d_rec, n_rec, (const float*)d_tab, nt, P, g->d, dc_max, types->radius, d_rad, g->g);
    if (e == cudaSuccess) e = launch_grid_pack(ctx->stream, g->d, g->gp);
    int bad = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);     // host staging (tab, bad) dies at return
    if (e != cudaSuccess) { tridsk_free_grid(g); return fail(ctx, TRIDSK_ECUDA, std::string("build_grid: ") + cudaGetErrorString(e)); }
    ctx->launches += 2 + (n_rec > 0 ? 1 : 0);
    if (bad) { tridsk_free_grid(g); return fail(ctx, TRIDSK_EINVAL, "receptor atom type out of range"); }
    *out = g;
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- per-receptor grid cache
static unsigned long long fnv1a(unsigned long long h, const void* p, size_t n) {
    const unsigned char* b = (const unsigned char*)p;
    for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ULL; }
    return h;
}
static void cache_trim(tridsk_ctx* ctx) {
    while (!ctx->grid_cache.empty() && ctx->cache_bytes > ctx->cache_budget) {
        ctx->cache_bytes -= ctx->grid_cache.back().bytes;
        tridsk_free_grid(ctx->grid_cache.back().grid);
        ctx->grid_cache.pop_back();
    }
}

extern "C" int tridsk_build_grid_cached(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec,
                                        const tridsk_types* types, const tridsk_params* params,
                                        const float origin[3], const int dims[3], float spacing, tridsk_grid** out) {
    if (!ctx || !out || !params || !rec_xyz || !rec_type || n_rec < 0 || !origin || !dims) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    *out = nullptr;
    int rc = check_types(ctx, types);
    if (rc) return rc;
    if (ctx->cache_budget == 0) return tridsk_build_grid(ctx, rec_xyz, rec_type, n_rec, types, params, origin, dims, spacing, out);
    // host view of the receptor for the key
    std::vector<float> hx;
    std::vector<int> ht;
    const float* kx = rec_xyz;
    const int* kt = rec_type;
    if (n_rec && is_device_ptr(rec_xyz)) { hx.resize(3 * (size_t)n_rec); CK(cudaMemcpyAsync(hx.data(), rec_xyz, sizeof(float) * hx.size(), cudaMemcpyDeviceToHost, ctx->stream)); kx = hx.data(); }
    if (n_rec && is_device_ptr(rec_type)) { ht.resize(n_rec); CK(cudaMemcpyAsync(ht.data(), rec_type, sizeof(int) * n_rec, cudaMemcpyDeviceToHost, ctx->stream)); kt = ht.data(); }
    if (!hx.empty() || !ht.empty()) CK(cudaStreamSynchronize(ctx->stream));
    unsigned long long key = 14695981039346656037ULL;
    key = fnv1a(key, &n_rec, sizeof(int));
    key = fnv1a(key, kx, sizeof(float) * 3 * (size_t)n_rec);
    key = fnv1a(key, kt, sizeof(int) * (size_t)n_rec);
    key = fnv1a(key, &types->n_types, sizeof(int));
    key = fnv1a(key, types->radius, sizeof(float) * types->n_types);
    key = fnv1a(key, types->hb_role, types->n_types);
    const float pf[] = {params->w_long, params->w_clash, params->w_hbond, params->long_mu, params->long_two_sigma2, params->long_dmax,
                        params->hb_mu, params->hb_sigma, params->hb_dmax, params->hb_dclash, params->d_floor, origin[0], origin[1], origin[2], spacing};
    key = fnv1a(key, pf, sizeof(pf));
    key = fnv1a(key, dims, 3 * sizeof(int));
    for (size_t i = 0; i < ctx->grid_cache.size(); ++i)
        if (ctx->grid_cache[i].key == key) {
            tridsk_ctx::CacheEnt ent = ctx->grid_cache[i];
            ctx->grid_cache.erase(ctx->grid_cache.begin() + i);
            ctx->grid_cache.insert(ctx->grid_cache.begin(), ent);          // most recently used first
            ++ent.grid->refs;
            ++ctx->cache_hits;
            *out = ent.grid;
            return TRIDSK_OK;
        }
    tridsk_grid* g = nullptr;
    rc = tridsk_build_grid(ctx, rec_xyz, rec_type, n_rec, types, params, origin, dims, spacing, &g);
    if (rc) return rc;
    ++ctx->cache_misses;
    const size_t bytes = (sizeof(float) + 2 * sizeof(float4)) * g->d.plane * g->d.n_types;
    if (bytes <= ctx->cache_budget) {
        ++g->refs;
        ctx->grid_cache.insert(ctx->grid_cache.begin(), {key, bytes, g});
        ctx->cache_bytes += bytes;
        cache_trim(ctx);
    }
    *out = g;
    return TRIDSK_OK;
}

extern "C" int tridsk_grid_cache_config(tridsk_ctx* ctx, long long budget_bytes, long long stats[4]) {
    if (!ctx) return TRIDSK_EINVAL;
    ENTER(ctx);
    if (budget_bytes >= 0) { ctx->cache_budget = (size_t)budget_bytes; cache_trim(ctx); }
    if (stats) { stats[0] = ctx->cache_hits; stats[1] = ctx->cache_misses; stats[2] = (long long)ctx->grid_cache.size(); stats[3] = (long long)ctx->cache_bytes; }
    return TRIDSK_OK;
}

extern "C" int tridsk_grid_from_values(tridsk_ctx* ctx, const float* values, int n_types,
                                       const float origin[3], const int dims[3], float spacing, tridsk_grid** out) {
    if (!ctx || !out || !values) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    *out = nullptr;
    tridsk_grid* g = nullptr;
    int rc = new_grid(ctx, n_types, origin, dims, spacing, &g);
    if (rc) return rc;
    cudaError_t e = cudaMemcpyAsync(g->g, values, sizeof(float) * g->d.plane * n_types, cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess) e = launch_grid_pack(ctx->stream, g->d, g->gp);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    ctx->launches += 1;
    if (e != cudaSuccess) { tridsk_free_grid(g); return fail(ctx, TRIDSK_ECUDA, std::string("grid copy: ") + cudaGetErrorString(e)); }
    *out = g;
    return TRIDSK_OK;
}

extern "C" int tridsk_grid_export(tridsk_ctx* ctx, const tridsk_grid* grid, float* dst) {
    if (!ctx || !grid || !dst) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    CK(cudaMemcpyAsync(dst, grid->g, sizeof(float) * grid->d.plane * grid->d.n_types, cudaMemcpyDefault, ctx->stream));
    if (!is_device_ptr(dst)) CK(cudaStreamSynchronize(ctx->stream));
    return TRIDSK_OK;
}

extern "C" int tridsk_grid_attach_receptor(tridsk_ctx* ctx, tridsk_grid* grid, const float* rec_xyz, const int* rec_type, int n_rec,
                                           const tridsk_types* types, const tridsk_params* params) {
    if (!ctx || !grid || !rec_xyz || !rec_type || n_rec < 1 || !params) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    int rc = check_types(ctx, types);
    if (rc) return rc;
    if ((rc = check_params(ctx, params))) return rc;
    if (types->n_types != grid->d.n_types) return fail(ctx, TRIDSK_EINVAL, "type table does not match the grid");
    // host view of the receptor (the cell sort is layout work, no arithmetic of the method)
    std::vector<float> hx(3 * (size_t)n_rec);
    std::vector<int> ht(n_rec);
    CK(cudaMemcpyAsync(hx.data(), rec_xyz, sizeof(float) * hx.size(), cudaMemcpyDefault, ctx->stream));
    CK(cudaMemcpyAsync(ht.data(), rec_type, sizeof(int) * n_rec, cudaMemcpyDefault, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    float cut = std::max(params->long_dmax, params->hb_dmax);
    for (int s = 0; s < types->n_types; ++s)
        for (int t = 0; t < types->n_types; ++t) {
            const unsigned char rs = types->hb_role[s], rt = types->hb_role[t];
            const bool hb = ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
            cut = std::max(cut, hb ? params->hb_dclash : types->radius[s] + types->radius[t]);
        }
    float lo[3] = {1e30f, 1e30f, 1e30f}, hi[3] = {-1e30f, -1e30f, -1e30f};
    for (int r = 0; r < n_rec; ++r) {
        if (ht[r] < 0 || ht[r] >= types->n_types) return fail(ctx, TRIDSK_EINVAL, "receptor atom type out of range");
        for (int c = 0; c < 3; ++c) { lo[c] = std::min(lo[c], hx[3 * r + c]); hi[c] = std::max(hi[c], hx[3 * r + c]); }
    }
    RecDev R;
    memset(&R, 0, sizeof(R));
    long long ncell = 1;
    // cells of a third of the range, x fastest: the atoms of a row of cells adjacent in x are one contiguous slice, so a ligand
    // atom visits, per (y, z) row within range, ONE slice trimmed to the x interval that can still lie inside the cut-off
    R.span = 3;                                             // measured on D2: span 1 81 ms, 2 49 ms, 3 42 ms, 4 43 ms, 5 46 ms
    const float cell = cut / (float)R.span;
    for (int c = 0; c < 3; ++c) { R.lo[c] = lo[c]; R.nc[c] = std::max(1, (int)std::floor((hi[c] - lo[c]) / cell) + 1); ncell *= R.nc[c]; }
    if (ncell > (1 << 22)) return fail(ctx, TRIDSK_ELIMIT, "receptor extent / cut-off gives too many cells");
    R.inv_cell = 1.f / cell; R.cell = cell; R.cut2 = cut * cut;
    auto cell_of = [&](int r) {
        int ci[3];
        for (int c = 0; c < 3; ++c) ci[c] = std::min(R.nc[c] - 1, std::max(0, (int)std::floor((hx[3 * r + c] - lo[c]) * R.inv_cell)));
        return (ci[2] * R.nc[1] + ci[1]) * R.nc[0] + ci[0];
    };
    std::vector<int> off((size_t)ncell + 1, 0), fillp;
    for (int r = 0; r < n_rec; ++r) off[cell_of(r) + 1]++;
    for (long long c = 0; c < ncell; ++c) off[c + 1] += off[c];
    fillp.assign(off.begin(), off.end() - 1);
    std::vector<float4> at(n_rec);
    for (int r = 0; r < n_rec; ++r) {                      // input order inside a cell
        float tb; memcpy(&tb, &ht[r], sizeof(tb));
        at[fillp[cell_of(r)]++] = make_float4(hx[3 * r], hx[3 * r + 1], hx[3 * r + 2], tb);
    }
    for (int i = 0; i < 4; ++i) if (grid->rd_buf[i]) { cudaFree(grid->rd_buf[i]); grid->rd_buf[i] = nullptr; }
    cudaError_t e = cudaMalloc(&grid->rd_buf[0], sizeof(float4) * n_rec);
    if (e == cudaSuccess) e = cudaMalloc(&grid->rd_buf[1], sizeof(int) * (ncell + 1));
    if (e == cudaSuccess) e = cudaMalloc(&grid->rd_buf[2], sizeof(float) * types->n_types);
    if (e == cudaSuccess) e = cudaMalloc(&grid->rd_buf[3], types->n_types);
    if (e == cudaSuccess) e = cudaMemcpyAsync(grid->rd_buf[0], at.data(), sizeof(float4) * n_rec, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(grid->rd_buf[1], off.data(), sizeof(int) * (ncell + 1), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(grid->rd_buf[2], types->radius, sizeof(float) * types->n_types, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(grid->rd_buf[3], types->hb_role, types->n_types, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return fail(ctx, e == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA, std::string("attach_receptor: ") + cudaGetErrorString(e));
    R.atoms = (const float4*)grid->rd_buf[0]; R.cell_off = (const int*)grid->rd_buf[1];
    R.radius = (const float*)grid->rd_buf[2]; R.role = (const unsigned char*)grid->rd_buf[3];
    grid->rd = R;
    return TRIDSK_OK;
}

extern "C" void tridsk_free_grid(tridsk_grid* g) {
    if (!g) return;
    if (--g->refs > 0) return;                       // the grid cache (or the caller) still holds it
    for (int i = 0; i < 4; ++i) if (g->rd_buf[i]) cudaFree(g->rd_buf[i]);
    if (g->ctx_alive && *g->ctx_alive) {             // stream-ordered: later work on the ctx stream may reuse the memory
        if (g->g) cudaFreeAsync(g->g, g->ctx->stream);
        if (g->gp) cudaFreeAsync(g->gp, g->ctx->stream);
    } else {                                        // the ctx is gone: cudaFree waits for the device
        if (g->g) cudaFree(g->g);
        if (g->gp) cudaFree(g->gp);
    }
    delete g;
}

// ---------------------------------------------------------------------------------------- ligands
struct PackedLig {
    LigHdr h;
    std::vector<float4> f4;
    std::vector<int> ai;
    std::vector<FragRec> fr;
    std::vector<PairRound> rounds;
    std::vector<LaneFrag> lane_frags;   // lane format (internal.h): fragments in pre-order
    std::vector<uint4> lane_stream;     // lane format: the pair instruction stream (header units)
    std::vector<LaneRec> lane_recs;     // lane format: the pair records, in stream order
    long long w_hist[5] = {0, 0, 0, 0, 0};
    std::vector<int> cta_rows;          // CTA format (internal.h): n + 1 row offsets
    std::vector<uint2> cta_recs;        // CTA format: 2 P row records, then P flat records
    std::vector<float> cta_rtab;        // CTA format, n > 64: the round table
    int err = 0;
    const char* msg = "";
};

// Host-side packing of one ligand: validation, depth-first atom order, fragment records, pair schedule.
static void pack_ligand(const tridsk_ligand_batch* b, const tridsk_types* types, int i, bool want_cta, PackedLig& out) {
    const int a0 = b->atom_off[i], n = b->atom_off[i + 1] - a0;
    const int t0 = b->tor_off[i], T = b->tor_off[i + 1] - t0;
    auto bad = [&](int code, const char* m) { out.err = code; out.msg = m; };
    if (n < 1 || T < 0) return bad(TRIDSK_EINVAL, "ligand with no atoms or negative torsion count");
    if (n > TRIDSK_MAX_ATOMS) return bad(TRIDSK_ELIMIT, "ligand has more than 128 atoms");
    if (T > TRIDSK_MAX_TORSIONS) return bad(TRIDSK_ELIMIT, "ligand has more than 31 torsions");
    const float* ref = b->ref_xyz + 3 * (size_t)a0;
    const unsigned char* type = b->atom_type + a0;
    const unsigned char* frag = b->atom_frag + a0;
    const unsigned char* ta = b->tor_a + t0;
    const unsigned char* tb = b->tor_b + t0;
    const signed char* tp = b->tor_parent + t0;
    for (int a = 0; a < n; ++a) {
        if (type[a] >= types->n_types) return bad(TRIDSK_EINVAL, "ligand atom type out of range");
        if (frag[a] > T) return bad(TRIDSK_EINVAL, "atom_frag out of range");
    }
    std::vector<int> parent(T + 1, -1), depth(T + 1, 0);
    for (int k = 0; k < T; ++k) {
        if (tp[k] < -1 || tp[k] >= k) return bad(TRIDSK_EINVAL, "tor_parent must precede its children");
        if (ta[k] >= n || tb[k] >= n || ta[k] == tb[k]) return bad(TRIDSK_EINVAL, "torsion axis atoms out of range");
        if (frag[tb[k]] != k + 1) return bad(TRIDSK_EINVAL, "tor_b[k] must lie in fragment k+1");
        if (frag[ta[k]] != tp[k] + 1) return bad(TRIDSK_EINVAL, "tor_a[k] must lie in the parent fragment");
        parent[k + 1] = tp[k] + 1;
        depth[k + 1] = depth[tp[k] + 1] + 1;
    }
    // depth-first preorder over fragments (children in torsion order)
    std::vector<int> order;
    order.reserve(T + 1);
    {
        int stack[TRIDSK_MAX_TORSIONS + 2], sp = 0;
        stack[sp++] = 0;
        while (sp > 0) {
            const int f = stack[--sp];
            order.push_back(f);
            for (int c = T; c >= 1; --c) if (parent[c] == f) stack[sp++] = c;       // children pushed last-first: popped in torsion order
        }
    }
    std::vector<int> count(T + 1, 0), sub(T + 1, 0), lo(T + 1, 0);
    for (int a = 0; a < n; ++a) count[frag[a]]++;
    for (int f = T; f >= 0; --f) { sub[f] += count[f]; if (f > 0) sub[parent[f]] += sub[f]; }
    std::vector<int> newidx(n), oldidx(n);
    {
        int pos = 0;
        for (int f : order) {
            lo[f] = pos;
            for (int a = 0; a < n; ++a) if (frag[a] == f) { newidx[a] = pos; oldidx[pos] = a; ++pos; }
        }
    }
    const int J = (n + 31) / 32, S = (n + J - 1) / J;
    LigHdr& h = out.h;
    memset(&h, 0, sizeof(h));
    h.n = n; h.T = T; h.J = J; h.S = S;
    h.max_depth = *std::max_element(depth.begin(), depth.end());
    out.f4.resize(n); out.ai.resize(n);
    out.lane_recs.reserve(n * 4); out.lane_stream.reserve(4 * (T + 1) + n); out.rounds.reserve(2 * n);
    for (int p = 0; p < n; ++p) {
        const int a = oldidx[p];
        out.f4[p] = make_float4(ref[3 * a], ref[3 * a + 1], ref[3 * a + 2], types->radius[type[a]]);
        out.ai[p] = (int)type[a] | ((int)frag[a] << 8) | (a << 16);
    }
    out.fr.resize(T + 1);
    for (int f = 0; f <= T; ++f) {
        FragRec& r = out.fr[f];
        memset(&r, 0, sizeof(r));
        r.ux = 1.f;
        r.parent = parent[f]; r.depth = depth[f]; r.lo = lo[f]; r.hi = lo[f] + sub[f];
        r.own_hi = lo[f] + count[f];
        if (f > 0) r.axis = newidx[ta[f - 1]] | (newidx[tb[f - 1]] << 8);
        if (f > 0) {
            const float* A = ref + 3 * ta[f - 1];
            const float* B = ref + 3 * tb[f - 1];
            const double ux = (double)B[0] - A[0], uy = (double)B[1] - A[1], uz = (double)B[2] - A[2];
            const double un = sqrt(ux * ux + uy * uy + uz * uz);
            if (!(un > 1e-6)) return bad(TRIDSK_EINVAL, "torsion axis of zero length");
            r.ux = (float)(ux / un); r.uy = (float)(uy / un); r.uz = (float)(uz / un);   // layout: unit axis, reference frame
            r.ox = B[0]; r.oy = B[1]; r.oz = B[2];
        }
    }
    // intra-ligand pair set (internal indices)
    std::vector<unsigned char> pm((size_t)n * n, 0);
    int P = 0;
    if (b->pair_off) {
        const int p0 = b->pair_off[i], np = b->pair_off[i + 1] - p0;
        for (int k = 0; k < np; ++k) {
            const int a = b->pair_ab[2 * (size_t)(p0 + k)], c = b->pair_ab[2 * (size_t)(p0 + k) + 1];
            if (a >= n || c >= n || a == c) return bad(TRIDSK_EINVAL, "pair index out of range");
            const int x = newidx[a], y = newidx[c];
            if (pm[(size_t)x * n + y]) return bad(TRIDSK_EINVAL, "duplicate intra-ligand pair");
            pm[(size_t)x * n + y] = pm[(size_t)y * n + x] = 1;
            ++P;
        }
    } else {
        if (!b->bond_off || !b->bond_ab) return bad(TRIDSK_EINVAL, "neither pairs nor bonds given");
        const int b0 = b->bond_off[i], nb = b->bond_off[i + 1] - b0;
        // bond graph in CSR form on the stack (n <= 128): no allocation per atom
        int deg[TRIDSK_MAX_ATOMS + 1] = {0};
        for (int k = 0; k < nb; ++k) {
            const int a = b->bond_ab[2 * (size_t)(b0 + k)], c = b->bond_ab[2 * (size_t)(b0 + k) + 1];
            if (a >= n || c >= n || a == c) return bad(TRIDSK_EINVAL, "bond index out of range");
            ++deg[a + 1]; ++deg[c + 1];
        }
        for (int a = 0; a < n; ++a) deg[a + 1] += deg[a];
        std::vector<unsigned char> nbr(2 * (size_t)std::max(nb, 1));
        {
            int fillp[TRIDSK_MAX_ATOMS];
            for (int a = 0; a < n; ++a) fillp[a] = deg[a];
            for (int k = 0; k < nb; ++k) {
                const int a = b->bond_ab[2 * (size_t)(b0 + k)], c = b->bond_ab[2 * (size_t)(b0 + k) + 1];
                nbr[fillp[a]++] = (unsigned char)c; nbr[fillp[c]++] = (unsigned char)a;
            }
        }
        // O6: pairs = {a<b : bond-graph distance >= 4 and different rigid fragment}
        int dist[TRIDSK_MAX_ATOMS], cur[TRIDSK_MAX_ATOMS], nxt[TRIDSK_MAX_ATOMS];
        for (int a = 0; a < n; ++a) {
            for (int c = 0; c < n; ++c) dist[c] = 1 << 20;
            dist[a] = 0;
            int nc = 1;
            cur[0] = a;
            for (int d = 1; d <= 3 && nc > 0; ++d) {
                int nn = 0;
                for (int q = 0; q < nc; ++q) {
                    const int u = cur[q];
                    for (int e = deg[u]; e < deg[u + 1]; ++e) { const int v = nbr[e]; if (dist[v] > d) { dist[v] = d; nxt[nn++] = v; } }
                }
                for (int q = 0; q < nn; ++q) cur[q] = nxt[q];
                nc = nn;
            }
            for (int c = a + 1; c < n; ++c)
                if (dist[c] > 3 && frag[a] != frag[c]) {
                    pm[(size_t)newidx[a] * n + newidx[c]] = pm[(size_t)newidx[c] * n + newidx[a]] = 1;
                    ++P;
                }
        }
    }
    h.n_pairs = P;
    // lane format (internal.h): fragments in depth-first pre-order, pairs as a stream of (tile x partner-run) blocks
    {
        std::vector<int> pre(T + 1);
        for (int g = 0; g <= T; ++g) pre[order[g]] = g;
        out.lane_frags.resize(T + 1);
        for (int g = 0; g <= T; ++g) {
            const int f = order[g];
            const FragRec& r = out.fr[f];
            LaneFrag& q = out.lane_frags[g];
            q.ux = r.ux; q.uy = r.uy; q.uz = r.uz; q.ox = r.ox; q.oy = r.oy; q.oz = r.oz;
            q.lo = r.lo; q.own_hi = r.own_hi; q.parent = f > 0 ? pre[parent[f]] : 0; q.depth = depth[f];
            q.axis = r.axis; q.tor = f - 1;
        }
        auto hbp = [&](int x, int y) {
            const unsigned char rs = types->hb_role[out.ai[x] & 0xff], rt = types->hb_role[out.ai[y] & 0xff];
            return ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
        };
        std::vector<int> gof(n);                 // pre-order fragment of an internal atom
        for (int g = 0; g <= T; ++g) for (int a = out.lane_frags[g].lo; a < out.lane_frags[g].own_hi; ++a) gof[a] = g;
        // which of the two fragments of a pair supplies the 4-slot tiles: the one that needs fewer records (a 5-atom
        // fragment against a 4-atom one is 2 tiles x 4 partners = 8 records one way, 1 tile x 5 partners = 5 the other)
        auto tiles_of = [&](int g, std::vector<std::pair<int, int>>& tl) {
            tl.clear();
            const int lo_g = out.lane_frags[g].lo, cnt = out.lane_frags[g].own_hi - lo_g, nt = (cnt + 3) / 4;
            for (int t = 0, a0 = lo_g; t < nt; ++t) { const int w = cnt / nt + (t < cnt % nt ? 1 : 0); tl.push_back({a0, w}); a0 += w; }
        };
        auto rec_count = [&](int ft, int fp) {
            std::vector<std::pair<int, int>> tl;
            tiles_of(ft, tl);
            int cnt = 0;
            for (auto& t : tl)
                for (int y = out.lane_frags[fp].lo; y < out.lane_frags[fp].own_hi; ++y) {
                    bool any = false;
                    for (int i = 0; i < t.second; ++i) any = any || pm[(size_t)(t.first + i) * n + y];
                    cnt += any;
                }
            return cnt;
        };
        std::vector<unsigned char> tile_side((size_t)(T + 1) * (T + 1), 0);    // [g][fb] = 1: g supplies the tiles of the pair {g, fb}
        for (int g = 0; g <= T; ++g)
            for (int fb = g + 1; fb <= T; ++fb) {
                const bool g_side = rec_count(g, fb) <= rec_count(fb, g);
                tile_side[(size_t)g * (T + 1) + fb] = g_side; tile_side[(size_t)fb * (T + 1) + g] = !g_side;
            }
        int covered2 = 0;
        for (int g = 0; g <= T; ++g) {
            const int lo_g = out.lane_frags[g].lo, cnt = out.lane_frags[g].own_hi - lo_g;
            const size_t hdr_at = out.lane_stream.size();
            out.lane_stream.push_back(make_uint4(0u, 0u, 0u, 0u));
            const int nt = (cnt + 3) / 4;
            unsigned n_tiles = 0;
            for (int tl = 0, a0 = lo_g; tl < nt; ++tl) {
                const int w = cnt / nt + (tl < cnt % nt ? 1 : 0);
                const size_t tile_at = out.lane_stream.size();
                out.lane_stream.push_back(make_uint4((unsigned)a0, (unsigned)w, 0u, 0u));
                unsigned n_runs = 0;
                for (int fb = 0; fb <= T; ++fb) {             // fb == g: only explicit pair lists can pair a fragment with itself
                    if (fb != g && !tile_side[(size_t)g * (T + 1) + fb]) continue;
                    unsigned nb = 0;
                    for (int y = out.lane_frags[fb].lo; y < out.lane_frags[fb].own_hi; ++y) {
                        LaneRec rec;
                        memset(&rec, 0, sizeof(rec));
                        rec.b = (unsigned)y;
                        bool any = false;
                        for (int i = 0; i < 4; ++i) {
                            const int x = a0 + i;
                            rec.dvdw[i] = -1.f;                               // no pair in this slot
                            if (i < w && (fb != g || x < y) && pm[(size_t)x * n + y]) {
                                any = true; ++covered2;
                                rec.dvdw[i] = out.f4[x].w + out.f4[y].w;      // layout: operands of the pair function
                                if (hbp(x, y)) rec.hbmask |= 1u << i;
                            }
                        }
                        if (!any) continue;
                        out.w_hist[w]++;
                        out.lane_recs.push_back(rec);
                        ++nb;
                    }
                    if (nb) { out.lane_stream.push_back(make_uint4((unsigned)fb, nb, 0u, 0u)); ++n_runs; }
                }
                if (n_runs) {
                    // the run headers were pushed after their records were counted: they already follow the tile header
                    out.lane_stream[tile_at].z = n_runs; ++n_tiles;
                } else out.lane_stream.pop_back();
                a0 += w;
            }
            out.lane_stream[hdr_at].x = n_tiles;
        }
        (void)gof;
        if (covered2 != P) return bad(TRIDSK_EINVAL, "internal: lane pair stream does not cover the pair set");
        h.ls_len = (int)out.lane_stream.size();
        h.n_rec = (int)out.lane_recs.size();
    }
    // CTA format (internal.h): row form (every pair from both ends) + flat form (every pair once), internal indices
    if (want_cta) {
        auto hbq = [&](int x, int y) {
            const unsigned char rs = types->hb_role[out.ai[x] & 0xff], rt = types->hb_role[out.ai[y] & 0xff];
            return ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
        };
        auto fbits = [](float v) { unsigned u; memcpy(&u, &v, sizeof(u)); return u; };
        out.cta_rows.assign(n + 1, 0);
        for (int x = 0; x < n; ++x) {
            out.cta_rows[x] = (int)out.cta_recs.size();
            for (int y = 0; y < n; ++y)
                if (y != x && pm[(size_t)x * n + y])
                    out.cta_recs.push_back(make_uint2((unsigned)y | (hbq(x, y) ? 0x100u : 0u), fbits(out.f4[x].w + out.f4[y].w)));
        }
        out.cta_rows[n] = (int)out.cta_recs.size();
        for (int x = 0; x < n; ++x)
            for (int y = x + 1; y < n; ++y)
                if (pm[(size_t)x * n + y])
                    out.cta_recs.push_back(make_uint2((unsigned)x | ((unsigned)y << 8) | (hbq(x, y) ? 0x10000u : 0u),
                                                      fbits(out.f4[x].w + out.f4[y].w)));
        if ((int)out.cta_recs.size() != 3 * P) return bad(TRIDSK_EINVAL, "internal: CTA pair records do not cover the pair set");
        if (n > TRIDSK_CTA_DENSE_MIN) {                       // round table (internal.h): item l of round k = pair (l, (l + k) mod n)
            const int nr = n / 2;
            out.cta_rtab.assign((size_t)nr * n, -1.f);
            int cov = 0;
            for (int k = 1; k <= nr; ++k)
                for (int l = 0; l < n; ++l) {
                    if (n % 2 == 0 && k == nr && l >= nr) continue;          // that half of the last round repeats pairs
                    const int y = (l + k) % n;
                    if (!pm[(size_t)l * n + y]) continue;
                    unsigned bits = fbits(out.f4[l].w + out.f4[y].w);
                    bits = (bits & ~1u) | (hbq(l, y) ? 1u : 0u);              // layout: flag in the lowest mantissa bit
                    float v; memcpy(&v, &bits, sizeof(v));
                    out.cta_rtab[(size_t)(k - 1) * n + l] = v;
                    ++cov;
                }
            if (cov != P) return bad(TRIDSK_EINVAL, "internal: CTA round table does not cover the pair set");
        }
    }
    // conflict-free schedule: round (j1, j2, k): lane l <-> pair (j1*S + l, j2*S + (l+k) mod S)
    auto hb = [&](int x, int y) {
        const unsigned char rs = types->hb_role[out.ai[x] & 0xff], rt = types->hb_role[out.ai[y] & 0xff];
        return ((rs & 1) && (rt & 2)) || ((rs & 2) && (rt & 1));
    };
    int tile = 0, covered = 0;
    for (int j1 = 0; j1 < J; ++j1)
        for (int j2 = j1; j2 < J; ++j2, ++tile) {
            h.tile_off[tile] = (int)out.rounds.size();
            const int k_lo = (j1 == j2) ? 1 : 0, k_hi = (j1 == j2) ? S / 2 : S - 1;
            for (int k = k_lo; k <= k_hi; ++k) {
                PairRound r{0u, 0u, k, 0};
                const bool half = (j1 == j2) && (S % 2 == 0) && (k == S / 2);
                for (int l = 0; l < S; ++l) {
                    if (half && l >= S / 2) break;
                    const int A = j1 * S + l, B = j2 * S + (l + k) % S;
                    if (A >= n || B >= n || !pm[(size_t)A * n + B]) continue;
                    r.mask |= 1u << l;
                    if (hb(A, B)) r.hb |= 1u << l;
                    ++covered;
                }
                if (r.mask) out.rounds.push_back(r);
            }
        }
    for (int t = tile; t <= TRIDSK_MAX_TILES; ++t) h.tile_off[t] = (int)out.rounds.size();
    if (covered != P) return bad(TRIDSK_EINVAL, "internal: pair schedule does not cover the pair set");
}

extern "C" int tridsk_load_ligands(tridsk_ctx* ctx, const tridsk_ligand_batch* b, const tridsk_types* types,
                                   tridsk_ligands** out) {
    if (!ctx || !b || !out) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_load_ligands");
    *out = nullptr;
    int rc = check_types(ctx, types);
    if (rc) return rc;
    if (b->n_lig < 0 || !b->atom_off || !b->tor_off || (b->n_lig && (!b->ref_xyz || !b->atom_type || !b->atom_frag)))
        return fail(ctx, TRIDSK_EINVAL, "bad ligand batch");
    const int L = b->n_lig;
    // offsets must be non-decreasing, and every array an offset table indexes must be there
    auto mono = [&](const int* off) { for (int i = 0; i < L; ++i) if (off[i + 1] < off[i] || off[0] < 0) return false; return true; };
    if (!mono(b->atom_off) || !mono(b->tor_off)) return fail(ctx, TRIDSK_EINVAL, "atom_off / tor_off must be non-decreasing");
    if (L && b->tor_off[L] > b->tor_off[0] && (!b->tor_a || !b->tor_b || !b->tor_parent)) return fail(ctx, TRIDSK_EINVAL, "torsions without tor_a / tor_b / tor_parent");
    if (b->pair_off && (!mono(b->pair_off) || (L && b->pair_off[L] > b->pair_off[0] && !b->pair_ab))) return fail(ctx, TRIDSK_EINVAL, "bad pair_off / pair_ab");
    if (!b->pair_off && L && (!b->bond_off || !mono(b->bond_off) || (b->bond_off[L] > b->bond_off[0] && !b->bond_ab))) return fail(ctx, TRIDSK_EINVAL, "neither pairs nor a valid bond list given");
    std::vector<PackedLig> pk(L);
    // the CTA-per-chain format triples the pair storage: it is the single-dock mapping, so screens do not carry it
    const bool want_cta = L <= TRIDSK_CTA_MAX_LIG;
    const bool dbg = getenv("TRIDSK_DEBUG") != nullptr;
    const double t_a = dbg ? omp_get_wtime() : 0.0;
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < L; ++i) pack_ligand(b, types, i, want_cta, pk[i]);
    const double t_b = dbg ? omp_get_wtime() : 0.0;
    for (int i = 0; i < L; ++i)
        if (pk[i].err) return fail(ctx, pk[i].err, std::string("ligand ") + std::to_string(i) + ": " + pk[i].msg);

    tridsk_ligands* lg = new (std::nothrow) tridsk_ligands();
    if (!lg) return fail(ctx, TRIDSK_ENOMEM, "host alloc");
    lg->ctx = ctx; lg->n_lig = L; lg->has_cta = want_cta;
    size_t na = 0, nf = 0, nr = 0, nls = 0, nrec = 0, ncr = 0, ncc = 0, nrt = 0;
    lg->hdr_h.resize(L); lg->n_pairs.resize(L);
    for (int i = 0; i < L; ++i) {
        LigHdr& h = pk[i].h;
        h.atom_off = (int)na; h.frag_off = (int)nf; h.round_off = (int)nr; h.ls_off = (int)nls; h.rec_off = (int)nrec;
        h.cta_row_off = (int)ncr; h.cta_rec_off = (int)ncc; h.cta_rt_off = pk[i].cta_rtab.empty() ? -1 : (int)nrt;
        na += pk[i].f4.size(); nf += pk[i].fr.size(); nr += pk[i].rounds.size();
        nls += pk[i].lane_stream.size(); nrec += pk[i].lane_recs.size();
        ncr += pk[i].cta_rows.size(); ncc += pk[i].cta_recs.size(); nrt += pk[i].cta_rtab.size();
        lg->hdr_h[i] = h; lg->n_pairs[i] = h.n_pairs;
        lg->max_atoms = std::max(lg->max_atoms, h.n); lg->max_tor = std::max(lg->max_tor, h.T); lg->min_atoms = std::min(lg->min_atoms, h.n);
        lg->bucket[h.J].push_back(i);
        if (want_cta) {
            int th, lpa;
            cta_shape(h.n, &th, &lpa);
            for (int v = 0; v < 2; ++v) {                       // bucket 1: the dense-sweep instance of the kernel
                const int k = h.n > (v ? TRIDSK_CTA_DENSE_MIN : TRIDSK_CTA_ROUNDS_N) ? 1 : 0;
                lg->cta_bucket[v][k].push_back(i);
                lg->cta_smem[v][k] = std::max(lg->cta_smem[v][k], cta_layout(h.n, h.T, h.n_pairs, k == 1).total);
            }
        }
    }
    // One pinned staging block owned by the ctx (grown on demand, reused by later calls) and one device block hold all the
    // packed arrays back to back; the per-ligand pieces are gathered into the staging block in parallel and go up in one copy.
    struct Seg { size_t off, bytes; };
    size_t blob = 0;
    auto seg = [&](size_t bytes) { Seg sg{blob, bytes}; blob = (blob + std::max<size_t>(bytes, 16) + 255) / 256 * 256; return sg; };
    const Seg s_hdr = seg(sizeof(LigHdr) * L), s_f4 = seg(sizeof(float4) * na), s_ai = seg(sizeof(int) * na), s_fr = seg(sizeof(FragRec) * nf),
              s_rd = seg(sizeof(PairRound) * nr), s_lf = seg(sizeof(LaneFrag) * nf), s_ls = seg(sizeof(uint4) * nls),
              s_lr = seg(sizeof(LaneRec) * nrec), s_cr = seg(sizeof(int) * ncr), s_cc = seg(sizeof(uint2) * ncc), s_rt = seg(sizeof(float) * nrt);
    // the staging block is free once the last upload from it is done (an event, not the stream: kernels of an earlier dock may
    // still be running there, and tridsk_screen wants this gather to overlap them)
    if (ctx->pin_ev) cudaEventSynchronize(ctx->pin_ev);
    if (blob > ctx->pin_bytes) {
        if (ctx->pin) { cudaFreeHost(ctx->pin); ctx->pin = nullptr; ctx->pin_bytes = 0; }
        const size_t cap = blob + blob / 8;
        if (cudaHostAlloc(&ctx->pin, cap, cudaHostAllocDefault) != cudaSuccess) { cudaGetLastError(); delete lg; return fail(ctx, TRIDSK_ENOMEM, "pinned staging buffer"); }
        ctx->pin_bytes = cap;
    }
    char* H = (char*)ctx->pin;
    memcpy(H + s_hdr.off, lg->hdr_h.data(), s_hdr.bytes);
#pragma omp parallel for schedule(static, 64)
    for (int i = 0; i < L; ++i) {
        const LigHdr& h = pk[i].h;
        auto put = [&](const Seg& sg, size_t at, const void* src, size_t bytes) { if (bytes) memcpy(H + sg.off + at, src, bytes); };
        put(s_lf, sizeof(LaneFrag) * h.frag_off, pk[i].lane_frags.data(), sizeof(LaneFrag) * pk[i].lane_frags.size());
        put(s_ls, sizeof(uint4) * h.ls_off, pk[i].lane_stream.data(), sizeof(uint4) * pk[i].lane_stream.size());
        put(s_lr, sizeof(LaneRec) * h.rec_off, pk[i].lane_recs.data(), sizeof(LaneRec) * pk[i].lane_recs.size());
        put(s_cr, sizeof(int) * h.cta_row_off, pk[i].cta_rows.data(), sizeof(int) * pk[i].cta_rows.size());
        put(s_cc, sizeof(uint2) * h.cta_rec_off, pk[i].cta_recs.data(), sizeof(uint2) * pk[i].cta_recs.size());
        if (h.cta_rt_off >= 0) put(s_rt, sizeof(float) * h.cta_rt_off, pk[i].cta_rtab.data(), sizeof(float) * pk[i].cta_rtab.size());
        put(s_f4, sizeof(float4) * h.atom_off, pk[i].f4.data(), sizeof(float4) * pk[i].f4.size());
        put(s_ai, sizeof(int) * h.atom_off, pk[i].ai.data(), sizeof(int) * pk[i].ai.size());
        put(s_fr, sizeof(FragRec) * h.frag_off, pk[i].fr.data(), sizeof(FragRec) * pk[i].fr.size());
        put(s_rd, sizeof(PairRound) * h.round_off, pk[i].rounds.data(), sizeof(PairRound) * pk[i].rounds.size());
    }
    if (getenv("TRIDSK_DEBUG")) {
        long long np = 0;
        for (int i = 0; i < L; ++i) np += pk[i].h.n_pairs;
        fprintf(stderr, "tridsk load_ligands: %d ligands, %lld pairs in %zu 4-slot records (slot utilisation %.1f %%)\n", L, np, nrec,
                nrec ? 25.0 * (double)np / (double)nrec : 0.0);
        long long wh[5] = {0, 0, 0, 0, 0};
        for (int i = 0; i < L; ++i) for (int w = 1; w <= 4; ++w) wh[w] += pk[i].w_hist[w];
        fprintf(stderr, "tridsk load_ligands: records by tile width 1..4: %lld %lld %lld %lld\n", wh[1], wh[2], wh[3], wh[4]);
    }
    const double t_c = dbg ? omp_get_wtime() : 0.0;
    cudaError_t e = cudaMalloc(&lg->blob, std::max<size_t>(blob, 256));
    if (e == cudaSuccess && blob) e = cudaMemcpyAsync(lg->blob, H, blob, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess && !ctx->pin_ev) e = cudaEventCreateWithFlags(&ctx->pin_ev, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->pin_ev, ctx->stream);
    char* D = (char*)lg->blob;
    lg->hdr = (LigHdr*)(D + s_hdr.off); lg->atom_f4 = (float4*)(D + s_f4.off); lg->atom_i = (int*)(D + s_ai.off);
    lg->frags = (FragRec*)(D + s_fr.off); lg->rounds = (PairRound*)(D + s_rd.off); lg->lane_frags = (LaneFrag*)(D + s_lf.off);
    lg->lane_stream = (uint4*)(D + s_ls.off); lg->lane_recs = (LaneRec*)(D + s_lr.off); lg->cta_rows = (int*)(D + s_cr.off);
    lg->cta_recs = (uint2*)(D + s_cc.off); lg->cta_rtab = (float*)(D + s_rt.off);
    auto up = [&](void** d, const void* src, size_t bytes) {
        if (e != cudaSuccess) return;
        e = cudaMalloc(d, std::max<size_t>(bytes, 16));
        if (e == cudaSuccess && bytes) e = cudaMemcpyAsync(*d, src, bytes, cudaMemcpyHostToDevice, ctx->stream);
    };
    for (int k = 0; k < 2; ++k)
        for (int v = 0; v < 2; ++v)
            if (!lg->cta_bucket[v][k].empty()) up((void**)&lg->cta_bucket_dev[v][k], lg->cta_bucket[v][k].data(), sizeof(int) * lg->cta_bucket[v][k].size());
    if (e == cudaSuccess) e = cudaMalloc((void**)&lg->all_ids, sizeof(int) * std::max(L, 1));
    for (int j = 1; j <= TRIDSK_MAX_J; ++j)
        if (!lg->bucket[j].empty()) up((void**)&lg->bucket_dev[j], lg->bucket[j].data(), sizeof(int) * lg->bucket[j].size());
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (dbg) fprintf(stderr, "tridsk load_ligands: pack %.1f ms (%d threads), gather %.1f ms, upload %.1f ms\n", (t_b - t_a) * 1e3, omp_get_max_threads(),
                     (t_c - t_b) * 1e3, (omp_get_wtime() - t_c) * 1e3);
    if (e != cudaSuccess) {
        tridsk_free_ligands(lg);
        return fail(ctx, e == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA, std::string("load_ligands: ") + cudaGetErrorString(e));
    }
    // the per-ligand pieces (a dozen small vectors each) are released by all threads, not one after the other by pk's destructor
#pragma omp parallel for schedule(static)
    for (int i = 0; i < L; ++i) pk[i] = PackedLig();
    if (dbg) fprintf(stderr, "tridsk load_ligands: total %.1f ms\n", (omp_get_wtime() - t_a) * 1e3);
    *out = lg;
    return TRIDSK_OK;
}

extern "C" int tridsk_ligand_info(const tridsk_ligands* l, int* n_lig, int* max_atoms, int* max_torsions, int* n_pairs_out) {
    if (!l) return TRIDSK_EINVAL;
    if (n_lig) *n_lig = l->n_lig;
    if (max_atoms) *max_atoms = l->max_atoms;
    if (max_torsions) *max_torsions = l->max_tor;
    if (n_pairs_out) std::copy(l->n_pairs.begin(), l->n_pairs.end(), n_pairs_out);
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- E_MDN (O15)
static void free_mdn(tridsk_ligands* l) {
    for (int i = 0; i < 9; ++i) { if (l->mdn_buf[i]) cudaFree(l->mdn_buf[i]); l->mdn_buf[i] = nullptr; }
    memset(&l->mdn, 0, sizeof(l->mdn));
}

extern "C" int tridsk_load_mdn(tridsk_ctx* ctx, tridsk_ligands* ligs, const tridsk_mdn* m) {
    if (!ctx || !ligs) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_load_mdn");
    CK(cudaStreamSynchronize(ctx->stream));               // earlier work may still read the old term
    free_mdn(ligs);
    if (ctx->graph_exec) { cudaGraphExecDestroy(ctx->graph_exec); ctx->graph_exec = nullptr; ctx->graph_key.clear(); }
    if (!m) return TRIDSK_OK;
    if (m->n_res > 65535) return fail(ctx, TRIDSK_ELIMIT, "more than 65535 residues");
    if (m->n_res < 1 || m->K < 1 || !m->res_off || !m->res_xyz || !m->pi || !m->mu || !m->sigma) return fail(ctx, TRIDSK_EINVAL, "bad mixture-density term");
    if (!(m->d_cut > 0.f) || !std::isfinite(m->d_cut) || !std::isfinite(m->w_mdn)) return fail(ctx, TRIDSK_EINVAL, "bad w_mdn / d_cut");
    for (int i = 0; i < m->n_res; ++i) if (m->res_off[i + 1] < m->res_off[i] || m->res_off[0] != 0) return fail(ctx, TRIDSK_EINVAL, "res_off must start at 0 and be non-decreasing");
    const int L = ligs->n_lig, n_at = m->res_off[m->n_res];
    if (L == 0) return TRIDSK_OK;
    const int K4 = mdn_slot_f4(m->K);
    std::vector<long long> off(2 * (size_t)L);             // [0, L): blocks of the packed records; [L, 2L): blocks of the caller's arrays
    long long total = 0, total_p = 0;
    for (int l = 0; l < L; ++l) {
        off[l] = total_p; off[L + l] = total;
        total += (long long)m->n_res * ligs->hdr_h[l].n * m->K;
        total_p += (long long)m->n_res * ligs->hdr_h[l].n * K4;
    }
    cudaError_t e = cudaMalloc(&ligs->mdn_buf[0], sizeof(float4) * m->n_res);
    if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[1], sizeof(int) * (m->n_res + 1));
    if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[2], sizeof(float4) * std::max(n_at, 1));
    if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[3], sizeof(float4) * (size_t)total_p);
    if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[4], sizeof(long long) * 2 * L);
    // staging: residue coordinates, and the three parameter arrays when they live on the host
    float* d_xyz = nullptr;
    int* d_bad = nullptr;
    float* stage[3] = {nullptr, nullptr, nullptr};
    const float* src[3] = {m->pi, m->mu, m->sigma};
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_xyz, sizeof(float) * 3 * std::max(n_at, 1) + 16);
    if (e == cudaSuccess) e = cudaMalloc((void**)&d_bad, sizeof(int));
    for (int a = 0; a < 3 && e == cudaSuccess; ++a)
        if (!is_device_ptr(src[a])) {
            e = cudaMalloc((void**)&stage[a], sizeof(float) * (size_t)total);
            if (e == cudaSuccess) e = cudaMemcpyAsync(stage[a], src[a], sizeof(float) * (size_t)total, cudaMemcpyHostToDevice, ctx->stream);
            src[a] = stage[a];
        }
    if (e == cudaSuccess) e = cudaMemsetAsync(d_bad, 0, sizeof(int), ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_xyz, m->res_xyz, sizeof(float) * 3 * n_at, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ligs->mdn_buf[1], m->res_off, sizeof(int) * (m->n_res + 1), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ligs->mdn_buf[4], off.data(), sizeof(long long) * 2 * L, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = launch_mdn_spheres(ctx->stream, d_xyz, (const int*)ligs->mdn_buf[1], m->n_res, m->d_cut, (float4*)ligs->mdn_buf[2], (float4*)ligs->mdn_buf[0]);
    if (e == cudaSuccess) e = launch_mdn_pack(ctx->stream, ligs->hdr, ligs->atom_i, L, m->n_res, m->K, (const long long*)ligs->mdn_buf[4], (const long long*)ligs->mdn_buf[4] + L, src[0], src[1], src[2],
                                              m->w_mdn, (float4*)ligs->mdn_buf[3], d_bad);
    int bad = 0;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d_xyz); cudaFree(d_bad);
    for (int a = 0; a < 3; ++a) if (stage[a]) cudaFree(stage[a]);
    ctx->launches += 2;
    if (e != cudaSuccess) {
        free_mdn(ligs);
        return fail(ctx, e == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA, std::string("load_mdn: ") + cudaGetErrorString(e));
    }
    if (bad) { free_mdn(ligs); return fail(ctx, TRIDSK_EINVAL, "mixture parameters: sigma must be > 0 and every value finite"); }
    MdnDev M;
    memset(&M, 0, sizeof(M));
    M.n_res = m->n_res; M.K = m->K; M.K4 = K4; M.d_cut = m->d_cut;
    M.sph = (const float4*)ligs->mdn_buf[0]; M.res_off = (const int*)ligs->mdn_buf[1];
    M.rec = (const float4*)ligs->mdn_buf[2]; M.par = (const float4*)ligs->mdn_buf[3];
    M.lig_off = (const long long*)ligs->mdn_buf[4];
    // cell list (an acceleration structure, not arithmetic of the method): a uniform grid over the residues' bounding box
    // grown by d_cut; the lists are counted and filled on the device, the prefix sum of the counts is taken here
    {
        float lo[3] = {1e30f, 1e30f, 1e30f}, hi[3] = {-1e30f, -1e30f, -1e30f};
        for (int r = 0; r < n_at; ++r)
            for (int c = 0; c < 3; ++c) { lo[c] = std::min(lo[c], m->res_xyz[3 * r + c]); hi[c] = std::max(hi[c], m->res_xyz[3 * r + c]); }
        if (n_at == 0) for (int c = 0; c < 3; ++c) lo[c] = hi[c] = 0.f;
        float cell = 0.6f;                                  // measured on M3: 1.5 A 3.64 s, 1.0 A 2.95 s, 0.75 A 2.61 s, 0.6 A 2.44 s, 0.5 A 2.38 s
        long long ncell = 0;
        for (;; cell *= 1.25f) {                            // at most ~1M cells
            ncell = 1;
            for (int c = 0; c < 3; ++c) { M.nc[c] = std::max(1, (int)std::ceil((hi[c] - lo[c] + 2.f * m->d_cut) / cell)); ncell *= M.nc[c]; }
            if (ncell <= 1048576) break;
        }
        for (int c = 0; c < 3; ++c) M.glo[c] = lo[c] - m->d_cut;
        M.inv_cell = 1.f / cell;
        std::vector<int> cnt((size_t)ncell + 1, 0);
        e = cudaMalloc(&ligs->mdn_buf[5], sizeof(int) * (ncell + 1));
        if (e == cudaSuccess) e = launch_mdn_cells(ctx->stream, M, cell, false, (int*)ligs->mdn_buf[5], nullptr);
        if (e == cudaSuccess) e = cudaMemcpyAsync(cnt.data(), ligs->mdn_buf[5], sizeof(int) * ncell, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        long long run = 0;
        for (long long c = 0; c < ncell; ++c) { const int k = cnt[c]; cnt[c] = (int)run; run += k; }
        cnt[ncell] = (int)run;
        if (e == cudaSuccess && run > 0x7fffffffLL) e = cudaErrorInvalidValue;
        if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[6], sizeof(float4) * std::max<long long>(run, 1));
        if (e == cudaSuccess) e = cudaMemcpyAsync(ligs->mdn_buf[5], cnt.data(), sizeof(int) * (ncell + 1), cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = launch_mdn_cells(ctx->stream, M, cell, true, (int*)ligs->mdn_buf[5], (float4*)ligs->mdn_buf[6]);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        ctx->launches += 2;
        if (e != cudaSuccess) { free_mdn(ligs); return fail(ctx, e == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA, std::string("load_mdn cell list: ") + cudaGetErrorString(e)); }
        M.cell_off = (const int*)ligs->mdn_buf[5]; M.cell_at = (const float4*)ligs->mdn_buf[6];
        // run directory: counted and filled the same way
        e = cudaMalloc(&ligs->mdn_buf[7], sizeof(int) * (ncell + 1));
        if (e == cudaSuccess) e = launch_mdn_dir(ctx->stream, M, false, (int*)ligs->mdn_buf[7], nullptr);
        if (e == cudaSuccess) e = cudaMemcpyAsync(cnt.data(), ligs->mdn_buf[7], sizeof(int) * ncell, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        long long nrun = 0;
        for (long long c = 0; c < ncell; ++c) { const int k = cnt[c]; cnt[c] = (int)nrun; nrun += k; }
        cnt[ncell] = (int)nrun;
        if (e == cudaSuccess && nrun > 0x7fffffffLL) e = cudaErrorInvalidValue;
        if (e == cudaSuccess) e = cudaMalloc(&ligs->mdn_buf[8], sizeof(int2) * std::max<long long>(nrun, 1));
        if (e == cudaSuccess) e = cudaMemcpyAsync(ligs->mdn_buf[7], cnt.data(), sizeof(int) * (ncell + 1), cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = launch_mdn_dir(ctx->stream, M, true, (int*)ligs->mdn_buf[7], (int2*)ligs->mdn_buf[8]);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        ctx->launches += 2;
        if (e != cudaSuccess) { free_mdn(ligs); return fail(ctx, e == cudaErrorMemoryAllocation ? TRIDSK_ENOMEM : TRIDSK_ECUDA, std::string("load_mdn run directory: ") + cudaGetErrorString(e)); }
        M.dir_off = (const int*)ligs->mdn_buf[7]; M.dir = (const int2*)ligs->mdn_buf[8];
        if (getenv("TRIDSK_DEBUG")) fprintf(stderr, "tridsk load_mdn: %d residues, %lld cells of %.2f A, %.1f atoms per cell\n", m->n_res, ncell, cell, (double)run / (double)ncell);
    }
    ligs->mdn = M;
    return TRIDSK_OK;
}

extern "C" void tridsk_free_ligands(tridsk_ligands* l) {
    if (!l) return;                 // cudaFree waits for the device; l->ctx may already be destroyed
    free_mdn(l);
    cudaFree(l->blob); cudaFree(l->all_ids);       // the packed arrays are pieces of one block
    for (int v = 0; v < 2; ++v) for (int k = 0; k < 2; ++k) if (l->cta_bucket_dev[v][k]) cudaFree(l->cta_bucket_dev[v][k]);
    for (int j = 0; j <= TRIDSK_MAX_J; ++j) if (l->bucket_dev[j]) cudaFree(l->bucket_dev[j]);
    delete l;
}

// ---------------------------------------------------------------------------------------- score + gradient
extern "C" int tridsk_score_grad(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs,
                                 const tridsk_params* params, const int* lig_index, const float* poses, int n_pose,
                                 int pose_stride, float* energy, float* grad, int grad_stride, float* coords, int coord_stride) {
    if (!ctx || !grid || !ligs || !params || !lig_index || !poses || !energy || n_pose < 0)
        return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_score_grad");
    if (int prc = check_params(ctx, params)) return prc;
    if (pose_stride < 7 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "pose_stride < 7 + max torsions");
    if (grad && grad_stride < 6 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "grad_stride < 6 + max torsions");
    if (coords && coord_stride < ligs->max_atoms) return fail(ctx, TRIDSK_EINVAL, "coord_stride < max atoms");
    if (n_pose == 0) return TRIDSK_OK;
    // lig_index must be validated on the host: stage a host copy if it lives on the device
    std::vector<int> li(n_pose);
    CK(cudaMemcpyAsync(li.data(), lig_index, sizeof(int) * n_pose, cudaMemcpyDefault, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n_pose; ++i)
        if (li[i] < 0 || li[i] >= ligs->n_lig) return fail(ctx, TRIDSK_EINVAL, "lig_index out of range");
    ScoreLaunch a;
    memset(&a, 0, sizeof(a));
    a.hdr = ligs->hdr; a.atom_f4 = ligs->atom_f4; a.atom_i = ligs->atom_i; a.frags = ligs->frags; a.rounds = ligs->rounds;
    a.lane_frags = ligs->lane_frags; a.lane_stream = ligs->lane_stream; a.lane_recs = ligs->lane_recs;
    a.cta_rows = ligs->cta_rows; a.cta_recs = ligs->cta_recs; a.cta_rtab = ligs->cta_rtab;
    a.grid = grid->d;
    a.mdn = ligs->mdn;
    to_dparams(params, &a.P);
    a.n_pose = n_pose; a.pose_stride = pose_stride; a.grad_stride = grad_stride; a.coord_stride = coord_stride;
    const size_t b_li = sizeof(int) * n_pose, b_po = sizeof(float) * (size_t)n_pose * pose_stride;
    const size_t b_e = sizeof(float) * 3 * n_pose, b_g = grad ? sizeof(float) * (size_t)n_pose * grad_stride : 0;
    const size_t b_c = coords ? sizeof(float) * 3 * (size_t)n_pose * coord_stride : 0;
    // inputs: slot 7 holds [lig_index | poses] when they come from the host
    const bool h_li = !is_device_ptr(lig_index), h_po = !is_device_ptr(poses);
    if (h_po && !host_quats_ok(poses, (size_t)n_pose, pose_stride)) return fail(ctx, TRIDSK_EINVAL, "pose with a zero or non-finite quaternion");
    char* in = nullptr;
    if (h_li || h_po) { int rc = scratch(ctx, 7, b_li + b_po + 64, (void**)&in); if (rc) return rc; }
    const size_t o_po = (b_li + 15) / 16 * 16;
    if (h_li) { CK(cudaMemcpyAsync(in, li.data(), b_li, cudaMemcpyHostToDevice, ctx->stream)); a.lig_index = (const int*)in; }
    else a.lig_index = lig_index;
    if (h_po) { CK(cudaMemcpyAsync(in + o_po, poses, b_po, cudaMemcpyHostToDevice, ctx->stream)); a.poses = (const float*)(in + o_po); }
    else a.poses = poses;
    // outputs: slot 6 holds device temporaries for host outputs
    const bool h_e = !is_device_ptr(energy), h_g = grad && !is_device_ptr(grad), h_c = coords && !is_device_ptr(coords);
    char* ob = nullptr;
    const size_t o_g = (b_e + 15) / 16 * 16, o_c = o_g + (b_g + 15) / 16 * 16;
    if (h_e || h_g || h_c) { int rc = scratch(ctx, 6, o_c + b_c + 64, (void**)&ob); if (rc) return rc; }
    a.energy = h_e ? (float*)ob : energy;
    a.grad = grad ? (h_g ? (float*)(ob + o_g) : grad) : nullptr;
    a.coords = coords ? (h_c ? (float*)(ob + o_c) : coords) : nullptr;
    std::vector<int> seg;                                   // lane form: [seg_lig | seg_start | seg_cnt | perm]
    if (ctx->kernel == 2 || ctx->kernel == 4) {
        // one lane per pose, one 32-lane CTA per run of <= 32 poses of the same ligand
        std::vector<int> perm(n_pose);
        for (int i = 0; i < n_pose; ++i) perm[i] = i;
        std::stable_sort(perm.begin(), perm.end(), [&](int x, int y) { return li[x] < li[y]; });
        std::vector<int> s_lig, s_start, s_cnt;
        size_t smem = 0;
        for (int i = 0; i < n_pose;) {
            int j = i;
            while (j < n_pose && j - i < 32 && li[perm[j]] == li[perm[i]]) ++j;
            s_lig.push_back(li[perm[i]]); s_start.push_back(i); s_cnt.push_back(j - i);
            const LigHdr& h = ligs->hdr_h[li[perm[i]]];
            smem = std::max(smem, lane_topo_bytes(h.n, h.T, h.ls_len, h.n_rec) + 128 * (size_t)lane_chain_slots(h.n, h.T, h.max_depth, 1));
            i = j;
        }
        if (smem > TRIDSK_SMEM_MAX_CTA) return fail(ctx, TRIDSK_ELIMIT, "ligand does not fit the lane kernel's shared memory");
        const int ns = (int)s_lig.size();
        seg.insert(seg.end(), s_lig.begin(), s_lig.end());
        seg.insert(seg.end(), s_start.begin(), s_start.end());
        seg.insert(seg.end(), s_cnt.begin(), s_cnt.end());
        seg.insert(seg.end(), perm.begin(), perm.end());
        int* d_seg;
        { int rc = scratch(ctx, 5, sizeof(int) * seg.size(), (void**)&d_seg); if (rc) return rc; }
        CK(cudaMemcpyAsync(d_seg, seg.data(), sizeof(int) * seg.size(), cudaMemcpyHostToDevice, ctx->stream));
        a.seg_lig = d_seg; a.seg_start = d_seg + ns; a.seg_cnt = d_seg + 2 * ns; a.perm = d_seg + 3 * ns;
        CK(launch_score_lane(ctx->stream, a, ns, smem));
    } else if (ctx->kernel == 3) {
        if (!ligs->has_cta) return fail(ctx, TRIDSK_EINVAL, "the CTA-per-chain mapping needs a ligand batch of at most 1024 ligands");
        const size_t smem = std::max(ligs->cta_smem[0][0], ligs->cta_smem[0][1]);
        if (smem > TRIDSK_SMEM_MAX_CTA) return fail(ctx, TRIDSK_ELIMIT, "ligand does not fit the CTA kernel's shared memory");
        CK(launch_score_cta(ctx->stream, a, smem));
    } else {
        CK(launch_score(ctx->stream, a));
    }
    ctx->launches += 1;
    if (h_e) CK(cudaMemcpyAsync(energy, a.energy, b_e, cudaMemcpyDeviceToHost, ctx->stream));
    if (h_g) CK(cudaMemcpyAsync(grad, a.grad, b_g, cudaMemcpyDeviceToHost, ctx->stream));
    if (h_c) CK(cudaMemcpyAsync(coords, a.coords, b_c, cudaMemcpyDeviceToHost, ctx->stream));
    // li (host vector) was consumed by an async copy: always drain before it goes out of scope
    if (h_e || h_g || h_c || h_li || !seg.empty()) CK(cudaStreamSynchronize(ctx->stream));
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- score, direct receptor sums
extern "C" int tridsk_score_direct(tridsk_ctx* ctx, const float* rec_xyz, const int* rec_type, int n_rec, const tridsk_types* types,
                                   const tridsk_params* params, const tridsk_ligands* ligs, const int* lig_index, const float* poses,
                                   int n_pose, int pose_stride, float* energy, float* grad, int grad_stride) {
    if (!ctx || !rec_xyz || !rec_type || n_rec < 0 || !params || !ligs || !lig_index || !poses || !energy || n_pose < 0)
        return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_score_direct");
    if (int prc = check_params(ctx, params)) return prc;
    int rc = check_types(ctx, types);
    if (rc) return rc;
    if (!ligs->has_cta) return fail(ctx, TRIDSK_EINVAL, "tridsk_score_direct needs a ligand batch of at most 1024 ligands");
    if (pose_stride < 7 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "pose_stride < 7 + max torsions");
    if (grad && grad_stride < 6 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "grad_stride < 6 + max torsions");
    if (n_pose == 0) return TRIDSK_OK;
    const int nt = types->n_types;
    std::vector<int> li(n_pose);
    CK(cudaMemcpyAsync(li.data(), lig_index, sizeof(int) * n_pose, cudaMemcpyDefault, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < n_pose; ++i)
        if (li[i] < 0 || li[i] >= ligs->n_lig) return fail(ctx, TRIDSK_EINVAL, "lig_index out of range");
    // scratch 0: [bad flag (16 B) | float4 rec[n_rec]]; 1: [radius | role]; 4: staged host receptor; 7: inputs; 6: outputs
    char *d_rec0, *d_ty, *stage = nullptr, *in = nullptr, *ob = nullptr;
    if ((rc = scratch(ctx, 0, 16 + sizeof(float4) * std::max(n_rec, 1), (void**)&d_rec0)) ||
        (rc = scratch(ctx, 1, sizeof(float) * nt + nt + 64, (void**)&d_ty))) return rc;
    const size_t b_xyz = (sizeof(float) * 3 * (size_t)n_rec + 15) / 16 * 16;
    const bool h_xyz = n_rec && !is_device_ptr(rec_xyz), h_typ = n_rec && !is_device_ptr(rec_type);
    if ((h_xyz || h_typ) && (rc = scratch(ctx, 4, b_xyz + sizeof(int) * n_rec, (void**)&stage))) return rc;
    const size_t b_li = sizeof(int) * n_pose, b_po = sizeof(float) * (size_t)n_pose * pose_stride, o_po = (b_li + 15) / 16 * 16;
    const bool h_li = !is_device_ptr(lig_index), h_po = !is_device_ptr(poses);
    if (h_po && !host_quats_ok(poses, (size_t)n_pose, pose_stride)) return fail(ctx, TRIDSK_EINVAL, "pose with a zero or non-finite quaternion");
    if ((h_li || h_po) && (rc = scratch(ctx, 7, o_po + b_po + 64, (void**)&in))) return rc;
    const size_t b_e = sizeof(float) * 3 * n_pose, b_g = grad ? sizeof(float) * (size_t)n_pose * grad_stride : 0, o_g = (b_e + 15) / 16 * 16;
    const bool h_e = !is_device_ptr(energy), h_g = grad && !is_device_ptr(grad);
    if ((h_e || h_g) && (rc = scratch(ctx, 6, o_g + b_g + 64, (void**)&ob))) return rc;
    int* d_bad = (int*)d_rec0;
    float4* d_rec = (float4*)(d_rec0 + 16);
    CK(cudaMemsetAsync(d_bad, 0, sizeof(int), ctx->stream));
    if (h_xyz) CK(cudaMemcpyAsync(stage, rec_xyz, sizeof(float) * 3 * n_rec, cudaMemcpyHostToDevice, ctx->stream));
    if (h_typ) CK(cudaMemcpyAsync(stage + b_xyz, rec_type, sizeof(int) * n_rec, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(d_ty, types->radius, sizeof(float) * nt, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(d_ty + sizeof(float) * nt, types->hb_role, nt, cudaMemcpyHostToDevice, ctx->stream));
    CK(launch_rec_pack(ctx->stream, h_xyz ? (const float*)stage : rec_xyz, h_typ ? (const int*)(stage + b_xyz) : rec_type, n_rec, nt, d_rec, d_bad));
    if (h_li) CK(cudaMemcpyAsync(in, li.data(), b_li, cudaMemcpyHostToDevice, ctx->stream));
    if (h_po) CK(cudaMemcpyAsync(in + o_po, poses, b_po, cudaMemcpyHostToDevice, ctx->stream));
    DParams P;
    to_dparams(params, &P);
    float* d_e = h_e ? (float*)ob : energy;
    float* d_g = grad ? (h_g ? (float*)(ob + o_g) : grad) : nullptr;
    CK(launch_score_direct(ctx->stream, ligs->hdr, ligs->atom_f4, ligs->atom_i, ligs->lane_frags, ligs->cta_rows, ligs->cta_recs, d_rec,
                           n_rec, (const float*)d_ty, (const unsigned char*)(d_ty + sizeof(float) * nt), P,
                           h_li ? (const int*)in : lig_index, h_po ? (const float*)(in + o_po) : poses, n_pose, pose_stride, d_e, d_g,
                           grad_stride, ligs->max_atoms));
    ctx->launches += 1 + (n_rec > 0 ? 1 : 0);
    int bad = 0;
    CK(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    if (h_e) CK(cudaMemcpyAsync(energy, d_e, b_e, cudaMemcpyDeviceToHost, ctx->stream));
    if (h_g) CK(cudaMemcpyAsync(grad, d_g, b_g, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));                  // li, bad and the type table are host staging
    if (bad) return fail(ctx, TRIDSK_EINVAL, "receptor atom type out of range");
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- dock
// Lane-per-chain launch plan.  A CTA holds C chains of one ligand (C = n_chains rounded up to a warp, at most 128, fewer
// if a big ligand would not fit) and needs topology + C * chain_slots * 4 bytes of shared memory.  Ligands are grouped
// by (C, resident CTAs per SM) so that small ligands keep their high occupancy; every group is one launch whose dynamic
// shared memory is the group's largest need, the groups run concurrently as parallel branches of the CUDA graph, and
// inside a group the costliest ligands go first (short tail).
static int lane_plan(tridsk_ctx* ctx, tridsk_ligands* lg, int n_chains, int n_refine) {
    const long long key = ((long long)n_chains << 8) | (n_refine > 1 ? 1 : 0) | (ctx->kernel == 4 ? 2 : 0) | (lg->mdn.n_res > 0 ? 4 : 0);
    if (lg->lane_plan_key == key) return TRIDSK_OK;
    const int L = lg->n_lig;
    const int cmax = std::min(128, (n_chains + 31) / 32 * 32);
    const int wmax = lg->mdn.n_res > 0 ? 8 : 12;               // resident warps per SM the register budget allows (mc_lane.cu)
    struct Ent { int cls; long long cost; int lig; size_t need; };
    const bool use_tm = ctx->kernel == 4;
    std::vector<Ent> ent(L);
    for (int i = 0; i < L; ++i) {
        const LigHdr& h = lg->hdr_h[i];
        const size_t topo = lane_topo_bytes(h.n, h.T, h.ls_len, h.n_rec);
        const size_t per_chain = 4 * (size_t)lane_chain_slots(h.n, h.T, h.max_depth, n_refine);
        // chains per CTA: the multiple of a warp that keeps the most warps resident per SM (ties: the larger CTA, which
        // stages the topology fewer times); 168 registers per thread allow 12 warps per SM (255 with E_MDN: 8)
        int c = 0, r = 0;
        size_t need = 0;
        long long best_live = -1;
        for (int cc = cmax; cc >= 32; cc -= 32) {
            const size_t nd = (topo + per_chain * cc + 15) / 16 * 16;
            if (nd > TRIDSK_SMEM_MAX_CTA) continue;
            int rr = (int)(TRIDSK_SMEM_PER_SM / ((nd + 1023) / 1024 * 1024 + TRIDSK_SMEM_RESERVED));   // allocated in KB units
            rr = std::max(1, std::min(std::min(rr, 32), wmax * 32 / cc));
            // live chains resident per SM: a ligand's last CTA may be partly empty (128 chains in CTAs of 96 = 96 + 32)
            const int cpl_ = (n_chains + cc - 1) / cc;
            const long long live = (long long)rr * n_chains / cpl_;
            if (live > best_live) { best_live = live; c = cc; r = rr; need = nd; }
        }
        // tensor-memory form (mc_lane_tm_kernel): coordinates in TMEM columns, the rest of the chain state in shared
        // memory, 4 warps per CTA each with its own topology copy; taken when it keeps more warps resident
        int tm_cols = 0, tm_r = 0;
        size_t region = 0;
        if (use_tm && 3 * h.n + 1 <= 128) {
            tm_cols = 3 * h.n + 1 <= 32 ? 32 : 3 * h.n + 1 <= 64 ? 64 : 128;
            region = (topo + 32 * (per_chain - 12 * (size_t)h.n) + 15) / 16 * 16;
            const size_t cta = (4 * region + 1023) / 1024 * 1024 + TRIDSK_SMEM_RESERVED;
            tm_r = (int)std::min<size_t>(std::min<size_t>(TRIDSK_SMEM_PER_SM / cta, 512 / tm_cols), 3);
            if (4 * region > TRIDSK_SMEM_MAX_CTA - 1024) tm_r = 0;
        }
        if (c == 0 && tm_r == 0) return fail(ctx, TRIDSK_ELIMIT, "ligand does not fit the lane kernel's shared memory");
        const long long cost = (long long)h.n_pairs + 6LL * h.n + 8LL * h.T;
        if (4 * tm_r > r * c / 32) ent[i] = {0x40000000 | (tm_cols << 8) | tm_r, cost, i, region};
        else ent[i] = {(c << 8) | r, cost, i, need};
    }
    std::sort(ent.begin(), ent.end(), [](const Ent& x, const Ent& y) {
        if (x.cls != y.cls) return x.cls < y.cls;
        if (x.cost != y.cost) return x.cost > y.cost;
        return x.lig < y.lig;
    });
    lg->lane_ids_h.resize(L);
    lg->lane_plan.clear();
    for (int i = 0; i < L; ++i) {
        lg->lane_ids_h[i] = ent[i].lig;
        if (i == 0 || ent[i].cls != ent[i - 1].cls) {
            const bool tm = (ent[i].cls & 0x40000000) != 0;
            lg->lane_plan.push_back({tm ? 32 : ent[i].cls >> 8, 0, i, 0, tm ? (ent[i].cls >> 8) & 0xff : 0});
            if (!tm) {                                       // resident warps per SM of this class -> register budget
                const int warps = (ent[i].cls >> 8) * (ent[i].cls & 0xff) / 32;
                lg->lane_plan.back().minb = warps <= 8 ? 2 : 3;     // measured: 12 warps at 168 registers beat 16 at 128
            }
        }
        lg->lane_plan.back().count++;
        lg->lane_plan.back().smem = std::max(lg->lane_plan.back().smem, ent[i].need);
        lg->lane_plan.back().work += ent[i].cost;
    }
    // the buckets run as concurrent graph branches: start the one with the most work first
    std::stable_sort(lg->lane_plan.begin(), lg->lane_plan.end(),
                     [](const tridsk_ligands::LaneBucket& x, const tridsk_ligands::LaneBucket& y) { return x.work > y.work; });
    if (getenv("TRIDSK_DEBUG"))
        for (const auto& b : lg->lane_plan)
            fprintf(stderr, "tridsk lane plan: %d ligands, %s, %d chains per %s, %zu bytes of shared memory\n", b.count,
                    b.tm_cols ? "TMEM" : "smem", b.chains_per_cta, b.tm_cols ? "warp" : "CTA", b.smem);
    CK(cudaStreamSynchronize(ctx->stream));                  // an earlier dock may still read all_ids
    CK(cudaMemcpyAsync(lg->all_ids, lg->lane_ids_h.data(), sizeof(int) * L, cudaMemcpyHostToDevice, ctx->stream));
    lg->lane_plan_key = key;
    return TRIDSK_OK;
}

extern "C" int tridsk_set_kernel(tridsk_ctx* ctx, int kernel) {
    if (!ctx || kernel < 0 || kernel > 4)
        return fail(ctx, TRIDSK_EINVAL, "kernel must be 0 (auto), 1 (warp), 2 (lane), 3 (CTA per chain) or 4 (lane per chain, coordinates in tensor memory)");
    ctx->kernel = kernel;
    return TRIDSK_OK;
}

extern "C" int tridsk_last_kernel(const tridsk_ctx* ctx) { return ctx ? ctx->last_kernel : 0; }

extern "C" int tridsk_dock(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs, const tridsk_params* params,
                           const float box_min[3], const float box_max[3], const float pocket_center[3], float pocket_radius,
                           int n_chains, int n_steps, int top_k, unsigned long long seed, int pose_stride,
                           float* out_energy, float* out_pose, int* out_chain, const tridsk_dock_opts* opts_in) {
    if (!ctx || !grid || !ligs || !params || !box_min || !box_max || !pocket_center)
        return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_dock");
    if (int prc = check_params(ctx, params)) return prc;
    tridsk_dock_opts o;
    memset(&o, 0, sizeof(o));
    if (opts_in) o = *opts_in;
    if (n_chains < 1 || n_steps < 0 || top_k < 0 || top_k > n_chains) return fail(ctx, TRIDSK_EINVAL, "bad n_chains / n_steps / top_k");
    if (top_k > 0 && (!out_energy || !out_pose || !out_chain)) return fail(ctx, TRIDSK_EINVAL, "null output");
    if (pose_stride < 7 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "pose_stride < 7 + max torsions");
    if (params->n_refine < 0 || o.first_step < 0 || o.steps_per_launch < 0) return fail(ctx, TRIDSK_EINVAL, "bad option");
    if (o.resume && !o.chain_state) return fail(ctx, TRIDSK_EINVAL, "resume needs chain_state");
    if (o.resume && o.init_poses) return fail(ctx, TRIDSK_EINVAL, "resume and init_poses are exclusive");
    if (!(o.cluster_rmsd >= 0.f)) return fail(ctx, TRIDSK_EINVAL, "cluster_rmsd must be >= 0");
    if (o.cluster_rmsd > 0.f && (long long)top_k * ligs->max_atoms > 4096)
        return fail(ctx, TRIDSK_ELIMIT, "duplicate-removing top-k needs top_k * max_atoms <= 4096");
    for (int c = 0; c < 3; ++c) if (!(box_min[c] <= box_max[c])) return fail(ctx, TRIDSK_EINVAL, "box_min > box_max");
    const int L = ligs->n_lig;
    if (L == 0) return TRIDSK_OK;
    const size_t nch = (size_t)L * n_chains, n_pose_f = nch * pose_stride;

    // chain state: {pose_cur, pose_best, e_cur, e_best} -- the caller's device buffer, or ctx scratch
    const size_t state_floats = 2 * n_pose_f + 2 * nch;
    float* state = nullptr;
    const bool state_host = o.chain_state && !is_device_ptr(o.chain_state);
    if (o.chain_state && !state_host) state = o.chain_state;
    else { int rc = scratch(ctx, 2, sizeof(float) * state_floats, (void**)&state); if (rc) return rc; }
    if (o.resume && state_host) CK(cudaMemcpyAsync(state, o.chain_state, sizeof(float) * state_floats, cudaMemcpyHostToDevice, ctx->stream));
    const void* d_init = nullptr;
    if (o.init_poses && !is_device_ptr(o.init_poses) && !host_quats_ok(o.init_poses, nch, pose_stride))
        return fail(ctx, TRIDSK_EINVAL, "init pose with a zero or non-finite quaternion");
    if (o.init_poses) { int rc = stage_in(ctx, 8, o.init_poses, sizeof(float) * n_pose_f, &d_init); if (rc) return rc; }
    tridsk_trace_rec* d_trace = nullptr;
    const size_t trace_bytes = sizeof(tridsk_trace_rec) * nch * (size_t)n_steps;
    const bool trace_host = o.trace && !is_device_ptr(o.trace);
    if (o.trace && n_steps > 0) {
        if (trace_host) { int rc = scratch(ctx, 3, trace_bytes, (void**)&d_trace); if (rc) return rc; }
        else d_trace = o.trace;
    }
    // outputs
    const size_t b_oe = sizeof(float) * 2 * (size_t)L * top_k, b_op = sizeof(float) * (size_t)L * top_k * pose_stride;
    const size_t b_oc = sizeof(int) * (size_t)L * top_k;
    const bool h_oe = top_k && !is_device_ptr(out_energy), h_op = top_k && !is_device_ptr(out_pose), h_oc = top_k && !is_device_ptr(out_chain);
    char* ob = nullptr;
    const size_t o_p = (b_oe + 15) / 16 * 16, o_c = o_p + (b_op + 15) / 16 * 16;
    if (h_oe || h_op || h_oc) { int rc = scratch(ctx, 6, o_c + b_oc + 64, (void**)&ob); if (rc) return rc; }

    McLaunch base;
    memset(&base, 0, sizeof(base));
    base.hdr = ligs->hdr; base.atom_f4 = ligs->atom_f4; base.atom_i = ligs->atom_i; base.frags = ligs->frags; base.rounds = ligs->rounds;
    base.lane_frags = ligs->lane_frags; base.lane_stream = ligs->lane_stream; base.lane_recs = ligs->lane_recs;
    base.cta_rows = ligs->cta_rows; base.cta_recs = ligs->cta_recs; base.cta_rtab = ligs->cta_rtab;
    base.grid = grid->d;
    base.mdn = ligs->mdn;
    to_dparams(params, &base.P);
    for (int c = 0; c < 3; ++c) { base.box_min[c] = box_min[c]; base.box_max[c] = box_max[c]; base.centre[c] = pocket_center[c]; }
    base.radius = pocket_radius;
    base.n_chains = n_chains; base.pose_stride = pose_stride; base.seed = seed; base.chain_base = o.chain_base; base.lig_base = o.lig_base;
    base.init_poses = (const float*)d_init;
    base.pose_cur = state; base.pose_best = state + n_pose_f; base.e_cur = state + 2 * n_pose_f; base.e_best = state + 2 * n_pose_f + nch;
    base.trace = d_trace; base.trace_stride = n_steps;

    // Mapping: a CTA per chain when chains are scarce (a single dock: latency of one evaluation), a lane per chain when
    // they outnumber the machine's lanes several times over (screens: throughput), a warp per chain in between.
    // tridsk_set_kernel overrides.
    int mode = ctx->kernel;
    if (mode == 0) {
        // Measured on the final kernels (docks of 384 chains x 500 steps, 1 / 2 / 4 / 8 / 16 at once, ms):
        //   20 atoms: CTA 2.2 / 4.2 / 7.9 / 14.5 / 28.6, warp 2.2 / 2.6 / 3.2 / 6.3 / 11.9, lane 12.6 / 13.1 / 13.1 / 13.1 / 13.3
        //   30 atoms: CTA - / 5.0 / 9.2 / 16.7 / 32.9, warp - / 3.4 / 4.0 / 8.0 / 14.5, lane - / 24 / 24 / 26 / 26  (one C2 dock of 1,000 steps: CTA 5.7, warp 6.4)
        //   48 atoms: CTA 3.5 / 5.8 / 11.1 / 19.0 / 35.7, warp 6.3 / 7.1 / 9.4 / 18.3 / 33.9, lane 51 / 51 / 52 / 52 / 53
        //   64 atoms: CTA 4.5 / 8.3 / 16.3 / 27.1 / 51.8, warp - / 9.2 / 12.7 / 23.7 / 44.3, lane 79 / 79 / 87 / 87 / 91
        //   80 atoms: CTA 10.7 / 12.6 / 24.4 / 40.0 / 76.5, warp 18.0 / 21.5 / 28.2 / 53.2 / 98.9, lane 134 / 134 / 136 / 136 / 136
        // with the mixture-density term (C2-sized ligands, K = 10, 8 / 32 / 128 / 256 docks, M pose evaluations/s): CTA 46.7 / 48.9 /
        // 49.9 / 50.2 (the lanes of an atom split its candidate residues), lane 7.0 / 26.8 / 50.4 / 66.1
        const bool all_dense = ligs->has_cta && ligs->cta_bucket[0][0].empty() && !ligs->cta_bucket[0][1].empty();
        const size_t per_sm = (size_t)ctx->sm_count;
        if (ligs->mdn.n_res > 0 && ligs->has_cta) mode = nch <= per_sm * 330 ? 3 : 2;
        else if (all_dense) mode = nch <= per_sm * 76 ? 3 : 2;       // above 64 atoms (dense sweep): the CTA form beats the warp form at every size
        else if (nch >= per_sm * 64) mode = 2;
        else if (ligs->has_cta && nch <= per_sm * (ligs->min_atoms > 32 ? 5 : 3)) mode = 3;
        else mode = 1;
    }
    if (mode == 3) {
        if (!ligs->has_cta) return fail(ctx, TRIDSK_EINVAL, "the CTA-per-chain mapping needs a ligand batch of at most 1024 ligands");
        for (int v = 0; v < 2; ++v)
            if (std::max(ligs->cta_smem[v][0], ligs->cta_smem[v][1]) > TRIDSK_SMEM_MAX_CTA)
                return fail(ctx, TRIDSK_ELIMIT, "ligand does not fit the CTA kernel's shared memory");
    }
    // CTA form: which ligands take the dense sweep (two warps per chain) -- with more chains than the SMs hold at once (3 record-
    // instance CTAs each) also those of 33 .. 64 atoms
    const int cv = nch > (size_t)ctx->sm_count * 3 ? 1 : 0;
    base.cta_dense_n = cv ? TRIDSK_CTA_DENSE_MIN : TRIDSK_CTA_ROUNDS_N;
    if (o.receptor_direct) {                                        // direct pair sums: the CTA- and the warp-per-chain kernels carry that path
        if (!grid->rd.atoms) return fail(ctx, TRIDSK_EINVAL, "receptor_direct needs tridsk_grid_attach_receptor on this grid");
        if (mode != 3 || ligs->mdn.n_res > 0) mode = 1;             // (the CTA instances with direct sums leave out E_MDN)
        base.rec = grid->rd;
    }
    const bool lane = mode == 2 || mode == 4;
    if (mode == 4 && ligs->mdn.n_res > 0) return fail(ctx, TRIDSK_EINVAL, "the tensor-memory mapping (4) does not evaluate the mixture-density term");
    ctx->last_kernel = mode;
    tridsk_ligands* lg = const_cast<tridsk_ligands*>(ligs);
    if (lane) { int rc = lane_plan(ctx, lg, n_chains, params->n_refine); if (rc) return rc; }

    // launch series: per steps_per_launch slice, one launch per bucket (atoms per lane J, or shared-memory class); then top-k
    struct Item { int kind, arg; size_t smem; int branch; McLaunch a; };
    std::vector<Item> series;
    const int spl = (o.steps_per_launch > 0) ? o.steps_per_launch : std::max(n_steps, 1);
    int done = 0;
    bool first = true;
    do {
        const int ns = std::min(spl, n_steps - done);
        auto fill = [&](McLaunch& a) {
            a.first_step = o.first_step + done; a.n_steps = ns; a.trace_off = done;
            a.init_mode = first ? (o.resume ? 2 : (o.init_poses ? 1 : 0)) : 2;
        };
        if (lane) {
            int br = 0;
            for (const auto& b : lg->lane_plan) {
                McLaunch a = base;
                a.lig_list = lg->all_ids + b.first; a.n_list = b.count;
                fill(a);
                a.lane_region = (int)b.smem; a.tm_cols = b.tm_cols; a.lane_minb = b.minb;
                series.push_back({b.tm_cols ? 4 : 2, b.chains_per_cta, b.smem, br++ % TRIDSK_BRANCHES, a});
            }
        } else if (mode == 3) {
            for (int k = 0; k < 2; ++k) {
                if (ligs->cta_bucket[cv][k].empty()) continue;
                McLaunch a = base;
                a.lig_list = ligs->cta_bucket_dev[cv][k]; a.n_list = (int)ligs->cta_bucket[cv][k].size();
                fill(a);
                series.push_back({3, k, ligs->cta_smem[cv][k], k, a});
            }
        } else {
            for (int j = 1; j <= TRIDSK_MAX_J; ++j) {
                if (ligs->bucket[j].empty()) continue;
                McLaunch a = base;
                a.lig_list = ligs->bucket_dev[j]; a.n_list = (int)ligs->bucket[j].size();
                fill(a);
                series.push_back({1, j, 0, (j - 1) % TRIDSK_BRANCHES, a});
            }
        }
        done += ns; first = false;
    } while (done < n_steps);
    TopkLaunch tk;
    memset(&tk, 0, sizeof(tk));
    tk.hdr = ligs->hdr; tk.e_best = base.e_best; tk.pose_best = base.pose_best;
    tk.n_lig = L; tk.n_chains = n_chains; tk.pose_stride = pose_stride; tk.top_k = top_k; tk.w_tor = params->w_tor;
    tk.atom_f4 = ligs->atom_f4; tk.lane_frags = ligs->lane_frags; tk.cluster_rmsd = o.cluster_rmsd;
    tk.max_atoms = ligs->max_atoms; tk.max_tor = ligs->max_tor;
    tk.out_energy = h_oe ? (float*)ob : out_energy;
    tk.out_pose = h_op ? (float*)(ob + o_p) : out_pose;
    tk.out_chain = h_oc ? (int*)(ob + o_c) : out_chain;
    const int n_launch = (int)series.size() + (top_k > 0 ? 1 : 0);

    for (int i = 0; i < 3; ++i) if (!ctx->ev[i]) CK(cudaEventCreate(&ctx->ev[i]));
    ctx->ev_valid = false;
    // independent launches (size buckets) run as parallel branches: branch 0 is the ctx stream, the others side streams
    int n_branch = 1;
    for (auto& it : series) n_branch = std::max(n_branch, it.branch + 1);
    if (n_branch > 1) {
        if (!ctx->fork_ev) CK(cudaEventCreateWithFlags(&ctx->fork_ev, cudaEventDisableTiming));
        for (int i = 1; i < n_branch; ++i) {
            if (!ctx->side[i]) CK(cudaStreamCreateWithFlags(&ctx->side[i], cudaStreamNonBlocking));
            if (!ctx->join_ev[i]) CK(cudaEventCreateWithFlags(&ctx->join_ev[i], cudaEventDisableTiming));
        }
    }
    // inside a capture the events are recorded with the External flag (event-record nodes that stay queryable);
    // that flag is only legal while capturing
    auto enqueue = [&](cudaStream_t s, bool capturing) -> cudaError_t {
        const unsigned fl = capturing ? cudaEventRecordExternal : cudaEventRecordDefault;
        cudaError_t e = cudaEventRecordWithFlags(ctx->ev[0], s, fl);
        if (e != cudaSuccess) return e;
        if (n_branch > 1) {
            e = cudaEventRecord(ctx->fork_ev, s);
            for (int i = 1; i < n_branch && e == cudaSuccess; ++i) e = cudaStreamWaitEvent(ctx->side[i], ctx->fork_ev, 0);
            if (e != cudaSuccess) return e;
        }
        for (auto& it : series) {
            cudaStream_t bs = it.branch == 0 ? s : ctx->side[it.branch];
            e = it.kind == 4 ? launch_mc_lane_tm(bs, it.a) : it.kind == 2 ? launch_mc_lane(bs, it.a, it.arg, it.smem, it.a.lane_minb)
                : it.kind == 3 ? launch_mc_cta(bs, it.a, it.arg, it.smem) : launch_mc(bs, it.arg, it.a);
            if (e != cudaSuccess) return e;
        }
        for (int i = 1; i < n_branch; ++i) {
            e = cudaEventRecord(ctx->join_ev[i], ctx->side[i]);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ctx->join_ev[i], 0);
            if (e != cudaSuccess) return e;
        }
        e = cudaEventRecordWithFlags(ctx->ev[1], s, fl);
        if (e != cudaSuccess) return e;
        if (top_k > 0) { e = launch_topk(s, tk); if (e != cudaSuccess) return e; }
        return cudaEventRecordWithFlags(ctx->ev[2], s, fl);
    };
    if (o.no_graph) {
        CK(enqueue(ctx->stream, false));
    } else {
        // a10: the whole series as one CUDA graph; re-used while the launch parameters are byte-identical
        std::vector<unsigned char> key;
        for (auto& it : series) {
            const long long hd[4] = {it.kind, it.arg, (long long)it.smem, it.branch};
            key.insert(key.end(), (const unsigned char*)hd, (const unsigned char*)hd + sizeof(hd));
            key.insert(key.end(), (unsigned char*)&it.a, (unsigned char*)&it.a + sizeof(McLaunch));
        }
        key.insert(key.end(), (unsigned char*)&tk, (unsigned char*)&tk + sizeof(tk));
        if (!ctx->graph_exec || key != ctx->graph_key) {
            if (ctx->graph_exec) { cudaGraphExecDestroy(ctx->graph_exec); ctx->graph_exec = nullptr; }
            cudaGraph_t graph = nullptr;
            CK(cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
            cudaError_t e = enqueue(ctx->stream, true);
            cudaError_t e2 = cudaStreamEndCapture(ctx->stream, &graph);
            if (e != cudaSuccess || e2 != cudaSuccess) {
                if (graph) cudaGraphDestroy(graph);
                return fail(ctx, TRIDSK_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e != cudaSuccess ? e : e2));
            }
            e = cudaGraphInstantiate(&ctx->graph_exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { ctx->graph_exec = nullptr; return fail(ctx, TRIDSK_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e)); }
            ctx->graph_key = key;
        }
        CK(cudaGraphLaunch(ctx->graph_exec, ctx->stream));
    }
    ctx->launches += n_launch;
    ctx->ev_valid = true;

    bool need_sync = false;
    if (h_oe) { CK(cudaMemcpyAsync(out_energy, tk.out_energy, b_oe, cudaMemcpyDeviceToHost, ctx->stream)); need_sync = true; }
    if (h_op) { CK(cudaMemcpyAsync(out_pose, tk.out_pose, b_op, cudaMemcpyDeviceToHost, ctx->stream)); need_sync = true; }
    if (h_oc) { CK(cudaMemcpyAsync(out_chain, tk.out_chain, b_oc, cudaMemcpyDeviceToHost, ctx->stream)); need_sync = true; }
    if (state_host) { CK(cudaMemcpyAsync(o.chain_state, state, sizeof(float) * state_floats, cudaMemcpyDeviceToHost, ctx->stream)); need_sync = true; }
    if (trace_host && d_trace) { CK(cudaMemcpyAsync(o.trace, d_trace, trace_bytes, cudaMemcpyDeviceToHost, ctx->stream)); need_sync = true; }
    if (need_sync || (o.init_poses && !is_device_ptr(o.init_poses)) || (o.resume && state_host)) CK(cudaStreamSynchronize(ctx->stream));
    return TRIDSK_OK;
}

extern "C" int tridsk_last_dock_ms(tridsk_ctx* ctx, float ms[2]) {
    if (!ctx || !ms) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    if (!ctx->ev_valid) return fail(ctx, TRIDSK_EINVAL, "no dock has run on this ctx");
    CK(cudaEventSynchronize(ctx->ev[2]));
    CK(cudaEventElapsedTime(&ms[0], ctx->ev[0], ctx->ev[1]));
    CK(cudaEventElapsedTime(&ms[1], ctx->ev[1], ctx->ev[2]));
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- test hook
extern "C" int tridsk_debug_philox(tridsk_ctx* ctx, const unsigned int ctr[4], const unsigned int key[2], unsigned int out[4]) {
    if (!ctx || !ctr || !key || !out) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    unsigned int h[6] = {ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]};
    unsigned int* d;
    int rc = scratch(ctx, 9, 64, (void**)&d);
    if (rc) return rc;
    CK(cudaMemcpyAsync(d, h, sizeof(h), cudaMemcpyHostToDevice, ctx->stream));
    CK(launch_philox_debug(ctx->stream, d, d + 8));
    ctx->launches += 1;
    CK(cudaMemcpyAsync(out, d + 8, 4 * sizeof(unsigned int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return TRIDSK_OK;
}

extern "C" int tridsk_debug_microbench(tridsk_ctx* ctx, int which, unsigned long long bytes, int iters, float* ms, double* work) {
    if (!ctx || !ms || !work || iters < 1) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    const bool mem = which == TRIDSK_MB_L2_READ || which == TRIDSK_MB_GATHER;
    if (which < TRIDSK_MB_FFMA || which > TRIDSK_MB_GATHER || (mem && bytes < 4096)) return fail(ctx, TRIDSK_EINVAL, "bad microbenchmark");
    char* buf = nullptr;
    float* sink;
    int rc = scratch(ctx, 9, 64, (void**)&sink);
    if (rc) return rc;
    if (mem) {
        if ((rc = scratch(ctx, 10, bytes, (void**)&buf))) return rc;
        CK(cudaMemsetAsync(buf, 0, bytes, ctx->stream));
    }
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    double w = 0.0;
    cudaError_t e = launch_microbench(ctx->stream, which, ctx->sm_count, buf, bytes, 1, sink, &w);      // warm-up pass (fills L2)
    if (e == cudaSuccess) e = cudaEventRecord(e0, ctx->stream);
    if (e == cudaSuccess) e = launch_microbench(ctx->stream, which, ctx->sm_count, buf, bytes, iters, sink, &w);
    if (e == cudaSuccess) e = cudaEventRecord(e1, ctx->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) return fail(ctx, TRIDSK_ECUDA, std::string("microbench: ") + cudaGetErrorString(e));
    ctx->launches += 2;
    *work = w;
    return TRIDSK_OK;
}

// ---------------------------------------------------------------------------------------- tridsk_screen
// load + dock + free of a screen given as host arrays, with the host-side packing of most of the batch overlapped with the
// docking of its first part (tridsk.h).  The two parts are sub-batch VIEWS of the caller's arrays (the offset tables hold
// absolute positions); the second part docks with lig_base = size of the first, so every chain draws the Philox streams it
// would draw in one tridsk_dock over the whole batch.
extern "C" int tridsk_screen(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligand_batch* batch, const tridsk_types* types,
                             const tridsk_params* params, const float box_min[3], const float box_max[3],
                             const float pocket_center[3], float pocket_radius, int n_chains, int n_steps, int top_k,
                             unsigned long long seed, int pose_stride, float* out_energy, float* out_pose, int* out_chain) {
    if (!ctx || !grid || !batch || !types || !params) return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_screen");
    const int L = batch->n_lig;
    if (L < 0 || top_k < 0) return fail(ctx, TRIDSK_EINVAL, "bad n_lig / top_k");
    if (L == 0) return TRIDSK_OK;
    if (top_k > 0 && (!out_energy || !out_pose || !out_chain)) return fail(ctx, TRIDSK_EINVAL, "null output");
    // first part: large enough that its docking outlasts the packing of the rest, small enough that its own packing is short
    const int l1 = L >= 8192 ? std::max(2048, L / 16) : L;      // measured on C5 (65,536 ligands): 1/8 1641 ms, 1/12 1630, 1/16 1626, 1/24 1624 per pass
    const size_t per_e = 2 * (size_t)top_k, per_p = (size_t)top_k * pose_stride, per_c = (size_t)top_k;
    const bool h_oe = top_k && !is_device_ptr(out_energy), h_op = top_k && !is_device_ptr(out_pose), h_oc = top_k && !is_device_ptr(out_chain);
    float* d_e = out_energy; float* d_p = out_pose; int* d_c = out_chain;
    if (l1 < L && (h_oe || h_op || h_oc)) {                      // the parts write device memory; one copy back at the end
        char* ob = nullptr;
        const size_t b_e = sizeof(float) * per_e * L, b_p = sizeof(float) * per_p * L, b_c = sizeof(int) * per_c * L;
        const size_t o_p = (b_e + 255) / 256 * 256, o_c = o_p + (b_p + 255) / 256 * 256;
        int rc = scratch(ctx, 11, o_c + b_c + 256, (void**)&ob);
        if (rc) return rc;
        if (h_oe) d_e = (float*)ob;
        if (h_op) d_p = (float*)(ob + o_p);
        if (h_oc) d_c = (int*)(ob + o_c);
    }
    auto view = [&](int a, int b) {
        tridsk_ligand_batch v = *batch;
        v.n_lig = b - a;
        v.atom_off = batch->atom_off + a; v.tor_off = batch->tor_off + a;
        if (batch->pair_off) v.pair_off = batch->pair_off + a;
        if (batch->bond_off) v.bond_off = batch->bond_off + a;
        return v;
    };
    tridsk_ligands* part[2] = {nullptr, nullptr};
    auto cleanup = [&](int rc) { for (auto* p : part) if (p) tridsk_free_ligands(p); return rc; };
    if (!batch->atom_off || !batch->tor_off) return fail(ctx, TRIDSK_EINVAL, "bad ligand batch");
    tridsk_dock_opts o;
    memset(&o, 0, sizeof(o));
    if (l1 == L) {                                               // small batch: nothing to overlap
        int rc = tridsk_load_ligands(ctx, batch, types, &part[0]);
        if (rc) return rc;
        rc = tridsk_dock(ctx, grid, part[0], params, box_min, box_max, pocket_center, pocket_radius, n_chains, n_steps, top_k, seed,
                         pose_stride, out_energy, out_pose, out_chain, &o);
        return cleanup(rc);
    }
    o.no_graph = 1;                                              // two launch series that run once each
    const tridsk_ligand_batch va = view(0, l1), vb = view(l1, L);
    int rc = tridsk_load_ligands(ctx, &va, types, &part[0]);
    if (rc) return cleanup(rc);
    rc = tridsk_dock(ctx, grid, part[0], params, box_min, box_max, pocket_center, pocket_radius, n_chains, n_steps, top_k, seed,
                     pose_stride, d_e, d_p, d_c, &o);            // device outputs: enqueued, not waited for
    if (rc) return cleanup(rc);
    rc = tridsk_load_ligands(ctx, &vb, types, &part[1]);         // packs on the host while the first part docks
    if (rc) return cleanup(rc);
    o.lig_base = l1;
    rc = tridsk_dock(ctx, grid, part[1], params, box_min, box_max, pocket_center, pocket_radius, n_chains, n_steps, top_k, seed,
                     pose_stride, d_e + per_e * l1, d_p + per_p * l1, d_c + per_c * l1, &o);
    if (rc) return cleanup(rc);
    if (h_oe) CK(cudaMemcpyAsync(out_energy, d_e, sizeof(float) * per_e * L, cudaMemcpyDeviceToHost, ctx->stream));
    if (h_op) CK(cudaMemcpyAsync(out_pose, d_p, sizeof(float) * per_p * L, cudaMemcpyDeviceToHost, ctx->stream));
    if (h_oc) CK(cudaMemcpyAsync(out_chain, d_c, sizeof(int) * per_c * L, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));                      // the handles are released below: their kernels must be done
    return cleanup(TRIDSK_OK);
}

// ---------------------------------------------------------------------------------------- tridsk_dock_static
// The docking run for callers that may not allocate (tridsk.h): the chain state lives in a file-scope device array instead
// of ctx scratch.  In host code `g_dock_scratch` is a host-side stand-in for the symbol, NOT a device address; the address
// is taken with cudaGetSymbolAddress once per device, with that device current (tridsk_create), and handed to the kernels.
#define TRIDSK_MAX_DEVICES 64
static __device__ __align__(256) unsigned char g_dock_scratch[TRIDSK_STATIC_SCRATCH_BYTES];
static float* g_dock_scratch_ptr[TRIDSK_MAX_DEVICES] = {};
static std::mutex g_dock_scratch_mu;

static cudaError_t dock_static_prepare(int device) {
    if (device < 0 || device >= TRIDSK_MAX_DEVICES) return cudaSuccess;          // tridsk_dock_static reports it
    std::lock_guard<std::mutex> lk(g_dock_scratch_mu);
    if (g_dock_scratch_ptr[device]) return cudaSuccess;
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_dock_scratch);
    if (e == cudaSuccess) g_dock_scratch_ptr[device] = (float*)ptr;
    return e;
}

extern "C" int tridsk_dock_static(tridsk_ctx* ctx, const tridsk_grid* grid, const tridsk_ligands* ligs, const tridsk_params* params,
                                  const float box_min[3], const float box_max[3], const float pocket_center[3], float pocket_radius,
                                  int n_chains, int n_steps, int top_k, unsigned long long seed, int pose_stride,
                                  float* out_energy, float* out_pose, int* out_chain) {
    if (!ctx || !grid || !ligs || !params || !box_min || !box_max || !pocket_center)
        return fail(ctx, TRIDSK_EINVAL, "null argument");
    ENTER(ctx);
    NvtxRange nvtx_("tridsk_dock_static");
    if (int prc = check_params(ctx, params)) return prc;
    if (n_chains < 1 || n_steps < 0 || top_k < 0 || top_k > n_chains) return fail(ctx, TRIDSK_EINVAL, "bad n_chains / n_steps / top_k");
    if (top_k > 0 && (!out_energy || !out_pose || !out_chain)) return fail(ctx, TRIDSK_EINVAL, "null output");
    if (top_k > 0 && (!is_device_ptr(out_energy) || !is_device_ptr(out_pose) || !is_device_ptr(out_chain)))
        return fail(ctx, TRIDSK_EINVAL, "tridsk_dock_static writes device memory only (a host output would need a staging allocation)");
    if (pose_stride < 7 + ligs->max_tor) return fail(ctx, TRIDSK_EINVAL, "pose_stride < 7 + max torsions");
    for (int c = 0; c < 3; ++c) if (!(box_min[c] <= box_max[c])) return fail(ctx, TRIDSK_EINVAL, "box_min > box_max");
    const int L = ligs->n_lig;
    if (L == 0) return TRIDSK_OK;
    if (!ligs->has_cta) return fail(ctx, TRIDSK_ELIMIT, "tridsk_dock_static needs a ligand batch of at most 1024 ligands (CTA-per-chain pair format)");
    const size_t nch = (size_t)L * n_chains, n_pose_f = nch * pose_stride;
    const int cv = nch > (size_t)ctx->sm_count * 3 ? 1 : 0;          // as tridsk_dock: which ligands take the dense sweep
    if (std::max(ligs->cta_smem[cv][0], ligs->cta_smem[cv][1]) > TRIDSK_SMEM_MAX_CTA)
        return fail(ctx, TRIDSK_ELIMIT, "ligand does not fit the CTA kernel's shared memory");
    const size_t state_bytes = sizeof(float) * (2 * n_pose_f + 2 * nch);
    if (state_bytes > TRIDSK_STATIC_SCRATCH_BYTES)
        return fail(ctx, TRIDSK_ELIMIT, "tridsk_dock_static: the chain state of " + std::to_string(nch) + " chains x pose_stride " +
                    std::to_string(pose_stride) + " needs " + std::to_string(state_bytes) + " bytes, the static scratch array holds " +
                    std::to_string((size_t)TRIDSK_STATIC_SCRATCH_BYTES) + " (use tridsk_dock)");
    float* state = (ctx->device >= 0 && ctx->device < TRIDSK_MAX_DEVICES) ? g_dock_scratch_ptr[ctx->device] : nullptr;
    if (!state) return fail(ctx, TRIDSK_ECUDA, "tridsk_dock_static: no static scratch address for this device");

    McLaunch base;
    memset(&base, 0, sizeof(base));
    base.hdr = ligs->hdr; base.atom_f4 = ligs->atom_f4; base.atom_i = ligs->atom_i; base.frags = ligs->frags; base.rounds = ligs->rounds;
    base.lane_frags = ligs->lane_frags; base.lane_stream = ligs->lane_stream; base.lane_recs = ligs->lane_recs;
    base.cta_rows = ligs->cta_rows; base.cta_recs = ligs->cta_recs; base.cta_rtab = ligs->cta_rtab;
    base.grid = grid->d;
    base.mdn = ligs->mdn;
    to_dparams(params, &base.P);
    for (int c = 0; c < 3; ++c) { base.box_min[c] = box_min[c]; base.box_max[c] = box_max[c]; base.centre[c] = pocket_center[c]; }
    base.radius = pocket_radius;
    base.n_chains = n_chains; base.pose_stride = pose_stride; base.seed = seed;
    base.pose_cur = state; base.pose_best = state + n_pose_f; base.e_cur = state + 2 * n_pose_f; base.e_best = state + 2 * n_pose_f + nch;
    base.cta_dense_n = cv ? TRIDSK_CTA_DENSE_MIN : TRIDSK_CTA_ROUNDS_N;
    base.first_step = 0; base.n_steps = n_steps; base.init_mode = 0;             // a1: Philox initialisation writes every chain's state
    ctx->last_kernel = 3;
    for (int k = 0; k < 2; ++k) {                                                // the two instances of the CTA kernel (internal.h)
        if (ligs->cta_bucket[cv][k].empty()) continue;
        McLaunch a = base;
        a.lig_list = ligs->cta_bucket_dev[cv][k]; a.n_list = (int)ligs->cta_bucket[cv][k].size();
        CK(launch_mc_cta(ctx->stream, a, k, ligs->cta_smem[cv][k]));
        ctx->launches += 1;
    }
    if (top_k > 0) {
        TopkLaunch tk;
        memset(&tk, 0, sizeof(tk));
        tk.hdr = ligs->hdr; tk.e_best = base.e_best; tk.pose_best = base.pose_best;
        tk.n_lig = L; tk.n_chains = n_chains; tk.pose_stride = pose_stride; tk.top_k = top_k; tk.w_tor = params->w_tor;
        tk.atom_f4 = ligs->atom_f4; tk.lane_frags = ligs->lane_frags; tk.cluster_rmsd = 0.f;
        tk.max_atoms = ligs->max_atoms; tk.max_tor = ligs->max_tor;
        tk.out_energy = out_energy; tk.out_pose = out_pose; tk.out_chain = out_chain;
        CK(launch_topk(ctx->stream, tk));
        ctx->launches += 1;
    }
    return TRIDSK_OK;
}
