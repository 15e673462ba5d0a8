// gadep_api.cu -- host side of libgadep.so: the C ABI of include/gadep.h.  Argument marshalling, validation,
// device buffers and kernel launches only; every step of the hot path runs in the kernels.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <new>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include <curand_kernel.h>

#include "../../include/gadep.h"
#include "gadep_build_kernels.cuh"
#include "gadep_transport_kernels.cuh"
#include "gadep_wave_kernels.cuh"
#include "gadep_locate_kernels.cuh"

struct gadep_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int n_sm = 148;
    // materials
    bool have_mat = false;
    int n_mat = 0, n_grid = 0;
    double e_min = 0, e_max = 0;
    float *d_table = nullptr;
    unsigned scoring_mask = 0;
    // mesh
    bool have_mesh = false, have_bvh = false;
    int n_vert = 0, n_tri = 0, n_surf = 0, world = 0;
    float *d_verts = nullptr;
    int *d_tris = nullptr, *d_tri_mats = nullptr, *d_tri_surf = nullptr;
    GdNode *d_nodes = nullptr;
    GdNode4 *d_nodes4 = nullptr;
    GdNode8 *d_nodes8 = nullptr;
    GdNode4q *d_nodes4q = nullptr;
    int bvh_width = 4;             // traversal of the wavefront kernels: 4 = uncompressed 4-wide nodes, 5 = compressed 4-wide
                                   // (64 bytes), 8 = compressed 8-wide
    bool width_set = false;        // gadep_set_bvh_width was called; otherwise the ray cast takes the 64-byte nodes on
                                   // hierarchies far larger than the L2 (14 % faster there), everything else the 4-wide ones
    GdTri *d_leaf_tris = nullptr;
    int bvh_depth = 0;
    int n_ref = 0;                 // leaves of the BVH: facet references after splitting
    // build buffers are kept between builds (no cudaMalloc / cudaFree, and none of their implicit synchronisations,
    // inside a step that rebuilds the BVH every time): [0] counts [1] scene [2] scratch arena [3] nodes [4] leaf
    // triangles [5] 4-wide nodes [13] 8-wide compressed nodes
    // [6..9] the mesh copies (vertices, triangles, side materials, surface ids)
    // [10..12] mesh validation: edge table keys, edge table surfaces, error record + surface sides
    // [14] clearance grid: marks / x distances [15] squared distances after the y pass [16] the grid itself
    void *pool[22] = {};
    size_t pool_cap[22] = {};
    // source
    bool have_src = false;
    GdSource src;
    GdSource *d_src = nullptr;
    // tallies
    unsigned long long *d_tally = nullptr;   // [cap_bins + 1][emitted 64][peak 64]
    int cap_bins = 0;
    GdCounters *d_counters = nullptr;
    unsigned long long *d_next = nullptr;     // history counter of the refill kernel
    int run_width = 4;                        // width used by the current launch (bvh_width, or 8 with GADEP_RUN_BVH8)
    unsigned long long n_stack_overflow = 0;  // rays that ran out of traversal stack since the context was made (must stay 0)
    bool prefer_ws = false;                   // GADEP_WS=1: the warp-specialised kernel instead of the default one (measurement)
    int kernel_variant = 2;                   // 2 = warp-resident wavefront, 1 = persistent lanes, 0 = history per thread
    float *d_pair = nullptr;                  // wavefront kernel: parked annihilation photons, 8 floats per slot
    size_t pair_floats = 0;
    GdWaveTune tune = {16, 16, 2, 6, 16, 1, 6};
    int wave_threads = 0;                     // 0 = by the size of the hierarchy; GADEP_WAVE_THREADS=384|896 forces an instance (measurement)
    float rho[GADEP_MAX_MATERIALS] = {};      // g/cm^3, electron-range mode
    bool have_rho = false;
    // surface-clustered hierarchy: side materials of every surface (host copy), per-material entry table (device)
    std::vector<int> h_sides;                 // [n_surf][2] inside, outside
    int *d_mat_entry = nullptr;               // [GADEP_MAX_MATERIALS][1 + GD_ENTRY_MAX], see GdBvh
    bool have_entries = false;
    // facet-clearance grid: box of all surfaces but the world boundary (host, from gadep_load_mesh), cell budget
    float roi_lo[3] = {0, 0, 0}, roi_hi[3] = {0, 0, 0};
    bool have_roi = false;
    long long grid_cells = 1ll << 22;         // GADEP_GRID_CELLS overrides; 0 = no grid
    double list_reach_cells = 1.0;            // reach of the cells' plane lists in cells; GADEP_GRID_REACH overrides, 0 = no lists
    unsigned long long list_min_hist = 20000000ull;   // GADEP_BUILD default: lists are made by the first run of at least this many
                                              // histories after a build (GADEP_LIST_MIN_HISTORIES overrides)
    int list_policy = 0;                      // build flags of the last gadep_build_bvh: 0 by run size, 1 built with the BVH, 2 never
    bool lists_built = false;
    unsigned char *grid_scalar = nullptr;     // u8 scalar clearance of the last build (input of the list kernel)
    unsigned n_list_cells = 0, n_listed = 0;  // cells below the reach / cells that got a list (last build)
    GdGrid grid = {};
    bool cluster_surfaces = true;             // GADEP_NO_SURFACE_CLUSTERS=1 switches it off (measurement)
    double split_budget = 8.0;                // extra BVH references per facet handed out by the splitting budget
    int n_bins = 0;
    float spec_e_max = 0;
    bool results_stale = false, have_results = false;
    std::vector<unsigned long long> h_spectrum;
    unsigned long long h_emitted[GADEP_MAX_LINES], h_peak[GADEP_MAX_LINES];
    GdCounters h_counters;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, evb0 = nullptr, evb1 = nullptr;
    bool run_timed = false;
    float last_run_ms = 0, last_build_ms = 0;
    int last_run_launches = 0, last_build_launches = 0;
};

static int gd_fail(gadep_ctx *c, int code, const char *fmt, ...) {
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof(buf), fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}

#define GD_CUDA(c, call)                                                                                  \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess)                                                                            \
            return gd_fail((c), GADEP_E_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

static bool gd_is_device_ptr(const void *p) {
    if (!p) return false;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

extern "C" int gadep_create(gadep_ctx **out, int device, void *cuda_stream) {
    if (!out) return GADEP_E_NULL;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0 || device < 0 || device >= n_dev) {
        cudaGetLastError();
        return GADEP_E_CUDA;   // no CPU fallback
    }
    gadep_ctx *c = new (std::nothrow) gadep_ctx();
    if (!c) return GADEP_E_NOMEM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    memset(&c->src, 0, sizeof(c->src));
    memset(&c->h_counters, 0, sizeof(c->h_counters));
    memset(c->h_emitted, 0, sizeof(c->h_emitted));
    memset(c->h_peak, 0, sizeof(c->h_peak));
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_counters, sizeof(GdCounters));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_src, sizeof(GdSource));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_next, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->ev1);
    if (e == cudaSuccess) e = cudaEventCreate(&c->evb0);
    if (e == cudaSuccess) e = cudaEventCreate(&c->evb1);
    if (e != cudaSuccess) { delete c; return GADEP_E_CUDA; }
    if (getenv("GADEP_NO_SURFACE_CLUSTERS")) c->cluster_surfaces = false;
    if (const char *t = getenv("GADEP_WS")) c->prefer_ws = atoi(t) != 0;
    if (const char *t = getenv("GADEP_WAVE_THREADS")) { int v = atoi(t); if (v == GD_W_THREADS || v == GD_W_THREADS_LAT) c->wave_threads = v; }
    if (const char *t = getenv("GADEP_GRID_CELLS")) { long long v = atoll(t); if (v >= 0 && v <= (1ll << 28)) c->grid_cells = v; }
    if (const char *t = getenv("GADEP_GRID_REACH")) { double v = atof(t); if (v >= 0.0 && v <= 8.0) c->list_reach_cells = v; }
    if (const char *t = getenv("GADEP_LIST_MIN_HISTORIES")) { long long v = atoll(t); if (v >= 0) c->list_min_hist = (unsigned long long)v; }
    if (const char *t = getenv("GADEP_TUNE")) {      // "k_fetch,t_keep,n_steps,n_steps_max,p_min,t_help,k_claim" (measurement sweeps)
        int a, b, d, dm = 0, p = c->tune.p_min, ts = c->tune.t_help, kc = c->tune.k_claim;
        if (sscanf(t, "%d,%d,%d,%d,%d,%d,%d", &a, &b, &d, &dm, &p, &ts, &kc) >= 4 && a >= 1 && a <= 32 && b >= 1 && b <= 32 && d >= 1 && d <= 32 && dm >= d && dm <= 32 && p >= 1 && p <= 32 && ts >= 1 && ts <= 1024 && kc >= 1 && kc <= 32)
            c->tune = {a, b, d, dm, p, ts, kc};
    }
    *out = c;
    return GADEP_OK;
}

static cudaError_t gd_pool_get(gadep_ctx *c, int k, size_t bytes, void **out) {
    if (c->pool_cap[k] < bytes) {
        cudaFree(c->pool[k]); c->pool[k] = nullptr; c->pool_cap[k] = 0;
        const size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&c->pool[k], want);
        if (e != cudaSuccess) { *out = nullptr; return e; }
        c->pool_cap[k] = want;
    }
    *out = c->pool[k];
    return cudaSuccess;
}

static void gd_free_mesh(gadep_ctx *c) {
    c->d_nodes4 = nullptr; c->d_nodes8 = nullptr; c->d_nodes4q = nullptr;
    c->d_verts = nullptr; c->d_tris = c->d_tri_mats = c->d_tri_surf = nullptr;
    c->d_nodes = nullptr; c->d_leaf_tris = nullptr;
    c->have_mesh = c->have_bvh = false;
}

extern "C" void gadep_destroy(gadep_ctx *c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    gd_free_mesh(c);
    for (int k = 0; k < 22; ++k) cudaFree(c->pool[k]);
    cudaFree(c->d_table); cudaFree(c->d_src); cudaFree(c->d_tally); cudaFree(c->d_counters); cudaFree(c->d_next); cudaFree(c->d_pair); cudaFree(c->d_mat_entry);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->evb0) cudaEventDestroy(c->evb0);
    if (c->evb1) cudaEventDestroy(c->evb1);
    delete c;
}

extern "C" const char *gadep_last_error(const gadep_ctx *c) { return c ? c->err.c_str() : "null context"; }

extern "C" int gadep_set_materials(gadep_ctx *c, int n_mat, int n_grid, double e_min, double e_max, const float *mu,
                                   const unsigned char *is_scoring) {
    if (!c) return GADEP_E_NULL;
    if (!mu || !is_scoring) return gd_fail(c, GADEP_E_NULL, "mu / is_scoring is null");
    if (n_mat <= 0 || n_mat > GADEP_MAX_MATERIALS || n_grid < 2 || n_grid > 1024 || !(e_min > 0) || !(e_max > e_min))
        return gd_fail(c, GADEP_E_ARG, "bad material table shape or energy range");
    size_t n = (size_t)n_mat * 4 * n_grid;
    std::vector<float> tab(n);
    for (int m = 0; m < n_mat; ++m)
        for (int ch = 0; ch < 4; ++ch)
            for (int g = 0; g < n_grid; ++g) {
                size_t i = ((size_t)m * 4 + ch) * n_grid + g;
                float v = mu[i];
                if (!std::isfinite(v) || v < 0) return gd_fail(c, GADEP_E_ARG, "mu[%d][%d][%d] negative or non-finite", m, ch, g);
                tab[i] = ch < 3 ? (v > 0 ? (float)std::log((double)v) : -1.0e30f) : v;
            }
    GD_CUDA(c, cudaSetDevice(c->device));
    cudaFree(c->d_table); c->d_table = nullptr;
    GD_CUDA(c, cudaMalloc(&c->d_table, n * sizeof(float)));
    GD_CUDA(c, cudaMemcpyAsync(c->d_table, tab.data(), n * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    c->n_mat = n_mat; c->n_grid = n_grid; c->e_min = e_min; c->e_max = e_max;
    c->scoring_mask = 0;
    for (int m = 0; m < n_mat; ++m) if (is_scoring[m]) c->scoring_mask |= 1u << m;
    c->have_mat = true;
    return GADEP_OK;
}

extern "C" int gadep_load_mesh(gadep_ctx *c, const float *vertices, int n_vert, const int *triangles,
                               const int *tri_surface, int n_tri, const int *surf_inside, const int *surf_outside,
                               int n_surf, int world_material) {
    if (!c) return GADEP_E_NULL;
    if (!vertices || !triangles || !tri_surface || !surf_inside || !surf_outside) return gd_fail(c, GADEP_E_NULL, "null mesh array");
    if (n_vert <= 0 || n_tri <= 0 || n_surf <= 0) return gd_fail(c, GADEP_E_ARG, "empty mesh");
    int mat_hi = c->have_mat ? c->n_mat : GADEP_MAX_MATERIALS;
    if (world_material < 0 || world_material >= mat_hi) return gd_fail(c, GADEP_E_INDEX, "world material %d out of range", world_material);
    for (int s = 0; s < n_surf; ++s) {
        if (surf_inside[s] < GADEP_MAT_KILL || surf_inside[s] >= mat_hi || surf_outside[s] < GADEP_MAT_KILL || surf_outside[s] >= mat_hi)
            return gd_fail(c, GADEP_E_INDEX, "surface %d: material id out of range", s);
    }
    // copies first, then the checks on the device (gadep_build_kernels.cuh): O(n) hash-table pass over the directed
    // edges at device rate instead of host rate; one 32-byte read-back carries the verdict
    size_t cap = 16;
    int cap_log2 = 4;
    while (cap < (size_t)n_tri * 6) { cap <<= 1; cap_log2++; }
    GD_CUDA(c, cudaSetDevice(c->device));
    gd_free_mesh(c);
    cudaStream_t st = c->stream;
    unsigned long long *ekey = nullptr;
    int *esurf = nullptr, *sides = nullptr;
    unsigned *err = nullptr;
    GD_CUDA(c, gd_pool_get(c, 6, sizeof(float) * 3 * (size_t)n_vert, (void **)&c->d_verts));
    GD_CUDA(c, gd_pool_get(c, 7, sizeof(int) * 3 * (size_t)n_tri, (void **)&c->d_tris));
    GD_CUDA(c, gd_pool_get(c, 8, sizeof(int) * (size_t)n_tri, (void **)&c->d_tri_mats));
    GD_CUDA(c, gd_pool_get(c, 9, sizeof(int) * (size_t)n_tri, (void **)&c->d_tri_surf));
    GD_CUDA(c, gd_pool_get(c, 10, sizeof(unsigned long long) * cap, (void **)&ekey));
    GD_CUDA(c, gd_pool_get(c, 11, sizeof(int) * cap, (void **)&esurf));
    GD_CUDA(c, gd_pool_get(c, 12, sizeof(int) * 2 * (size_t)n_surf + sizeof(unsigned) * GD_ERR_N, (void **)&err));
    sides = (int *)(err + GD_ERR_N);
    std::vector<int> &h_sides = c->h_sides;
    h_sides.resize(2 * (size_t)n_surf);
    for (int s = 0; s < n_surf; ++s) { h_sides[2 * s] = surf_inside[s]; h_sides[2 * s + 1] = surf_outside[s]; }
    GD_CUDA(c, cudaMemcpyAsync(c->d_verts, vertices, sizeof(float) * 3 * (size_t)n_vert, cudaMemcpyHostToDevice, st));
    GD_CUDA(c, cudaMemcpyAsync(c->d_tris, triangles, sizeof(int) * 3 * (size_t)n_tri, cudaMemcpyHostToDevice, st));
    GD_CUDA(c, cudaMemcpyAsync(c->d_tri_surf, tri_surface, sizeof(int) * (size_t)n_tri, cudaMemcpyHostToDevice, st));
    GD_CUDA(c, cudaMemcpyAsync(sides, h_sides.data(), sizeof(int) * 2 * (size_t)n_surf, cudaMemcpyHostToDevice, st));
    GD_CUDA(c, cudaMemsetAsync(ekey, 0xFF, sizeof(unsigned long long) * cap, st));
    GD_CUDA(c, cudaMemsetAsync(err, 0xFF, sizeof(unsigned) * GD_ERR_N, st));
    const int shift = 64 - cap_log2;
    gd_k_check_verts<<<(unsigned)(((size_t)n_vert * 3 + 255) / 256), 256, 0, st>>>(c->d_verts, (size_t)n_vert * 3, err);
    gd_k_check_tris<<<(n_tri + 255) / 256, 256, 0, st>>>(c->d_verts, c->d_tris, c->d_tri_surf, n_tri, n_vert, n_surf, sides,
                                                         c->d_tri_mats, ekey, esurf, cap - 1, shift, err);
    gd_k_check_closed<<<(unsigned)((cap + 255) / 256), 256, 0, st>>>(ekey, esurf, cap, shift, err);
    unsigned h_err[GD_ERR_N];
    GD_CUDA(c, cudaMemcpyAsync(h_err, err, sizeof(h_err), cudaMemcpyDeviceToHost, st));
    GD_CUDA(c, cudaStreamSynchronize(st));
    GD_CUDA(c, cudaGetLastError());
    const unsigned NONE = 0xFFFFFFFFu;
    if (h_err[GD_ERR_NONFINITE] != NONE) return gd_fail(c, GADEP_E_NONFINITE, "vertex %u is not finite", h_err[GD_ERR_NONFINITE]);
    {   // the first offending triangle decides, classes in the order they are checked within a triangle
        int best = -1;
        for (int k = GD_ERR_SURFACE; k <= GD_ERR_EDGE_TWICE; ++k)
            if (h_err[k] != NONE && (best < 0 || h_err[k] < h_err[best])) best = k;
        if (best == GD_ERR_SURFACE) return gd_fail(c, GADEP_E_INDEX, "triangle %u: surface id out of range", h_err[best]);
        if (best == GD_ERR_VERTEX) return gd_fail(c, GADEP_E_INDEX, "triangle %u: vertex id out of range", h_err[best]);
        if (best == GD_ERR_DEGENERATE) return gd_fail(c, GADEP_E_DEGENERATE, "triangle %u has zero area", h_err[best]);
        if (best == GD_ERR_EDGE_TWICE)
            return gd_fail(c, GADEP_E_NOT_CLOSED, "triangle %u: directed edge used twice (non-manifold or inconsistent winding)", h_err[best]);
    }
    if (h_err[GD_ERR_OPEN] != NONE) return gd_fail(c, GADEP_E_NOT_CLOSED, "surface %u is not closed (open edge)", h_err[GD_ERR_OPEN]);
    c->n_vert = n_vert; c->n_tri = n_tri; c->n_surf = n_surf; c->world = world_material;
    {   // box of every surface that is not a world boundary (outside = KILL): where the clearance grid pays
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        bool any_inner = false;
        for (int s2 = 0; s2 < n_surf; ++s2) any_inner = any_inner || surf_outside[s2] != GADEP_MAT_KILL;
        for (int t = 0; t < n_tri; ++t) {
            if (any_inner && surf_outside[tri_surface[t]] == GADEP_MAT_KILL) continue;
            for (int k = 0; k < 3; ++k) {
                const float *v = vertices + 3 * (size_t)triangles[3 * (size_t)t + k];
                for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], v[a]); hi[a] = std::max(hi[a], v[a]); }
            }
        }
        for (int a = 0; a < 3; ++a) { c->roi_lo[a] = lo[a]; c->roi_hi[a] = hi[a]; }
        c->have_roi = lo[0] <= hi[0];
    }
    c->have_mesh = true;
    return GADEP_OK;
}

// ---------------------------------------------------------------- plane lists of the clearance grid
// For the cells whose scalar clearance is below the reach (GdGrid, gd_k_grid_planes).  Costs 2 - 3 ms on the 40 k-facet
// set-ups and pays on runs whose photons scatter in tiny steps beside walls (volume sources; 10 % of a 1e8-history run),
// not on short point-source runs: so it runs with the build only when asked (GADEP_BUILD_PLANE_LISTS), otherwise before
// the first run of at least list_min_hist histories.  Its time and launches are added to the build's.
static int gd_build_plane_lists(gadep_ctx *c) {
    if (c->lists_built || !c->have_bvh || !c->grid.info || !c->grid_scalar || c->n_ref < 2 || !(c->list_reach_cells > 0.0)) return GADEP_OK;
    GD_CUDA(c, cudaSetDevice(c->device));
    cudaStream_t st = c->stream;
    GdGrid g = c->grid;
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    g.reach = (float)(c->list_reach_cells * (double)g.h);
    const unsigned thr = (unsigned)std::min(255.0, std::ceil((double)g.reach / (double)g.quarter_h));
    unsigned *lc = nullptr;
    float4 *planes = nullptr, *nrm = nullptr;
    GD_CUDA(c, gd_pool_get(c, 17, 16, (void **)&lc));
    GD_CUDA(c, cudaEventRecord(c->evb0, st));
    GD_CUDA(c, cudaMemsetAsync(lc, 0, 16, st));
    gd_k_grid_list_count<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(c->grid_scalar, nc, thr, lc);
    unsigned n_list = 0;
    GD_CUDA(c, cudaMemcpyAsync(&n_list, lc, 4, cudaMemcpyDeviceToHost, st));
    GD_CUDA(c, cudaStreamSynchronize(st));
    c->lists_built = true;
    n_list = std::min(n_list, 1u << 24);
    // a mesh with more references than cells near facets (config 4: 4096 angular segments) has tens of facets around
    // every such cell, hardly any cell gets by with GD_CELL_PLANES planes: no lists
    if (n_list == 0 || (unsigned)c->n_ref > n_list) return GADEP_OK;
    GD_CUDA(c, gd_pool_get(c, 19, sizeof(float4) * GD_CELL_PLANES * (size_t)n_list, (void **)&planes));
    GD_CUDA(c, gd_pool_get(c, 20, sizeof(float4) * (size_t)c->n_ref, (void **)&nrm));
    g.planes = planes;
    gd_k_tri_normals<<<(c->n_ref + 255) / 256, 256, 0, st>>>(c->d_leaf_tris, c->n_ref, nrm);
    gd_k_grid_planes<<<(unsigned)((nc + 127) / 128), 128, 0, st>>>(g, c->grid_scalar, thr, c->d_nodes4, c->d_leaf_tris, nrm,
                                                                   (unsigned *)g.info, planes, lc + 1, n_list);
    GD_CUDA(c, cudaEventRecord(c->evb1, st));
    GD_CUDA(c, cudaGetLastError());
    GD_CUDA(c, cudaMemcpyAsync(&c->n_listed, lc + 1, 4, cudaMemcpyDeviceToHost, st));
    GD_CUDA(c, cudaStreamSynchronize(st));
    float ms = 0.0f;
    cudaEventElapsedTime(&ms, c->evb0, c->evb1);
    c->last_build_ms += ms;
    c->last_build_launches += 3;
    c->n_list_cells = n_list;
    c->grid = g;
    if (getenv("GADEP_GRID_DEBUG"))
        fprintf(stderr, "[gadep] grid %d x %d x %d, h %.4f mm, reach %.4f mm: %u cells below the reach, %u with a plane list, %.2f ms\n",
                g.nx, g.ny, g.nz, g.h, g.reach, c->n_list_cells, c->n_listed, ms);
    return GADEP_OK;
}

// ---------------------------------------------------------------- BVH build
extern "C" int gadep_build_bvh(gadep_ctx *c, int flags) {
    if (!c) return GADEP_E_NULL;
    if (flags != 0 && flags != GADEP_BUILD_PLANE_LISTS && flags != GADEP_BUILD_NO_PLANE_LISTS)
        return gd_fail(c, GADEP_E_ARG, "unknown build flags %d", flags);
    if (!c->have_mesh) return gd_fail(c, GADEP_E_ORDER, "gadep_build_bvh before gadep_load_mesh");
    GD_CUDA(c, cudaSetDevice(c->device));
    const int n_tri = c->n_tri;
    cudaStream_t st = c->stream;
    c->d_nodes = nullptr; c->d_leaf_tris = nullptr; c->d_nodes4 = nullptr; c->d_nodes8 = nullptr; c->d_nodes4q = nullptr; c->have_bvh = false;
    const int tb = 256, nbt = (n_tri + tb - 1) / tb;
    int launches = 0;
    // ---- phase A: how many references (reference splitting) -> one 4-byte read-back sizes the arena
    unsigned *counts = nullptr;
    int *scene = nullptr;
    GD_CUDA(c, gd_pool_get(c, 0, 4 * (size_t)n_tri, (void **)&counts));
    GD_CUDA(c, gd_pool_get(c, 1, 4 * 16, (void **)&scene));
    cudaEventRecord(c->evb0, st);
    gd_k_init_scene<<<1, 32, 0, st>>>(scene);
    gd_k_split_prio<<<nbt, tb, 0, st>>>(c->d_verts, c->d_tris, n_tri, counts, (unsigned long long *)(scene + 10));
    gd_k_ref_count<<<nbt, tb, 0, st>>>(c->d_verts, c->d_tris, n_tri, counts, (const unsigned long long *)(scene + 10),
                                       (unsigned long long)(c->split_budget * (double)n_tri));
    gd_k_scan<<<1, 1024, 0, st>>>(counts, n_tri, (unsigned *)(scene + 8));
    launches += 4;
    unsigned n_ref_u = 0;
    cudaError_t e = cudaMemcpyAsync(&n_ref_u, scene + 8, 4, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess || n_ref_u < (unsigned)n_tri || n_ref_u > (unsigned)n_tri * GD_MAX_SPLITS) {
        return gd_fail(c, GADEP_E_CUDA, "BVH build (reference count) failed: %s", cudaGetErrorString(e));
    }
    const int n = (int)n_ref_u;
    const int nb = (n + tb - 1) / tb;
    const int n_tiles = (n + GD_SORT_TILE - 1) / GD_SORT_TILE;
    // ---- phase B: one scratch arena
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    size_t o_tlo = take(sizeof(float4) * n), o_thi = take(sizeof(float4) * n);
    size_t o_nlo = take(sizeof(float4) * n), o_nhi = take(sizeof(float4) * n);
    size_t o_k0 = take(8 * (size_t)n), o_k1 = take(8 * (size_t)n);
    size_t o_v0 = take(4 * (size_t)n), o_v1 = take(4 * (size_t)n);
    size_t o_hist = take(4 * (size_t)256 * n_tiles);
    size_t o_cl = take(4 * (size_t)n), o_cr = take(4 * (size_t)n), o_pi = take(4 * (size_t)n), o_pl = take(4 * (size_t)n);
    size_t o_vis = take(4 * (size_t)n), o_rt = take(4 * (size_t)n);
    // surface clusters: class bits above the Morton code, one entry node per surface
    int cls_bits = 0;
    if (c->cluster_surfaces && c->n_surf >= 2 && c->n_surf <= 256 && n > 1) while ((1 << cls_bits) < c->n_surf) cls_bits++;
    size_t o_se = take(4 * (size_t)std::max(c->n_surf, 1));
    unsigned char *arena = nullptr;
    if (gd_pool_get(c, 2, off, (void **)&arena) != cudaSuccess) return gd_fail(c, GADEP_E_NOMEM, "BVH scratch (%zu B)", off);
    int rc = GADEP_OK;
    int depth = 0;
    do {
        if ((e = gd_pool_get(c, 3, sizeof(GdNode) * (size_t)std::max(n - 1, 1), (void **)&c->d_nodes)) != cudaSuccess) break;
        if ((e = gd_pool_get(c, 4, sizeof(GdTri) * (size_t)n, (void **)&c->d_leaf_tris)) != cudaSuccess) break;
        if ((e = gd_pool_get(c, 5, sizeof(GdNode4) * (size_t)std::max(n - 1, 1), (void **)&c->d_nodes4)) != cudaSuccess) break;
        if ((e = gd_pool_get(c, 13, sizeof(GdNode8) * (size_t)std::max(n - 1, 1), (void **)&c->d_nodes8)) != cudaSuccess) break;
        if ((e = gd_pool_get(c, 21, sizeof(GdNode4q) * (size_t)std::max(n - 1, 1), (void **)&c->d_nodes4q)) != cudaSuccess) break;
        float4 *ref_lo = (float4 *)(arena + o_tlo), *ref_hi = (float4 *)(arena + o_thi);
        float4 *node_lo = (float4 *)(arena + o_nlo), *node_hi = (float4 *)(arena + o_nhi);
        unsigned long long *keys[2] = {(unsigned long long *)(arena + o_k0), (unsigned long long *)(arena + o_k1)};
        unsigned *vals[2] = {(unsigned *)(arena + o_v0), (unsigned *)(arena + o_v1)};
        unsigned *hist = (unsigned *)(arena + o_hist);
        int *child_l = (int *)(arena + o_cl), *child_r = (int *)(arena + o_cr);
        int *parent_int = (int *)(arena + o_pi), *parent_leaf = (int *)(arena + o_pl);
        int *visits = (int *)(arena + o_vis), *ref_tri = (int *)(arena + o_rt);
        int *surf_entry = (int *)(arena + o_se);
        gd_k_make_refs<<<nbt, tb, 0, st>>>(c->d_verts, c->d_tris, n_tri, counts, (unsigned)n, ref_lo, ref_hi, ref_tri, scene);
        gd_k_morton<<<nb, tb, 0, st>>>(ref_lo, ref_hi, n, scene, keys[0], vals[0], ref_tri, c->d_tri_surf, cls_bits);
        launches += 2;
        int cur = 0;
        for (int shift = 0; shift < 64; shift += 8) {
            gd_k_sort_hist<<<n_tiles, GD_SORT_THREADS, 0, st>>>(keys[cur], n, shift, hist, n_tiles);
            gd_k_scan<<<1, 1024, 0, st>>>(hist, 256 * n_tiles, nullptr);
            gd_k_sort_scatter<<<n_tiles, GD_SORT_THREADS, 0, st>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], n,
                                                                   shift, hist, n_tiles);
            cur ^= 1;
            launches += 3;
        }
        gd_k_leaf_tris<<<nb, tb, 0, st>>>(c->d_verts, c->d_tris, c->d_tri_mats, c->d_tri_surf, ref_tri, vals[cur], n,
                                          c->d_leaf_tris);
        launches += 1;
        if (n > 1) {
            cudaMemsetAsync(visits, 0, 4 * (size_t)n, st);
            cudaMemsetAsync(parent_leaf, 0xFF, 4 * (size_t)n, st);
            cudaMemsetAsync(surf_entry, 0xFF, 4 * (size_t)std::max(c->n_surf, 1), st);        // -1 = no entry node
            gd_k_karras<<<nb, tb, 0, st>>>(keys[cur], n, child_l, child_r, parent_int, parent_leaf, cls_bits, surf_entry);
            gd_k_refit<<<nb, tb, 0, st>>>(n, child_l, child_r, parent_int, parent_leaf, ref_lo, ref_hi, vals[cur], node_lo,
                                          node_hi, visits, c->d_nodes, scene + 6);
            gd_k_collapse4<<<nb, tb, 0, st>>>(n - 1, child_l, child_r, ref_lo, ref_hi, vals[cur], node_lo, node_hi, c->d_nodes4);
            gd_k_collapse8<<<nb, tb, 0, st>>>(n - 1, child_l, child_r, ref_lo, ref_hi, vals[cur], node_lo, node_hi, c->d_nodes8);
            gd_k_collapse4q<<<nb, tb, 0, st>>>(n - 1, child_l, child_r, ref_lo, ref_hi, vals[cur], node_lo, node_hi, c->d_nodes4q);
            launches += 5;
        }
        // ---- facet-clearance grid over the box of the inner surfaces
        c->grid = GdGrid{};
        c->lists_built = false; c->n_list_cells = 0; c->n_listed = 0; c->grid_scalar = nullptr; c->list_policy = flags;
        if (c->grid_cells > 0 && c->have_roi) {
            double ext[3], vol = 1.0;
            for (int a = 0; a < 3; ++a) { ext[a] = std::max((double)c->roi_hi[a] - (double)c->roi_lo[a], 1e-3); vol *= ext[a]; }
            double h = std::cbrt(vol / (double)c->grid_cells);
            int dim[3];
            for (;;) {
                double cells = 1.0;
                for (int a = 0; a < 3; ++a) { dim[a] = (int)std::ceil(ext[a] / h) + 2; cells *= dim[a]; }
                if (cells <= (double)c->grid_cells * 1.05 || cells <= 4096.0) break;
                h *= 1.02;
            }
            GdGrid g;
            g.nx = dim[0]; g.ny = dim[1]; g.nz = dim[2];
            g.lox = (float)(c->roi_lo[0] - h); g.loy = (float)(c->roi_lo[1] - h); g.loz = (float)(c->roi_lo[2] - h);
            g.inv_h = (float)(1.0 / h); g.quarter_h = (float)(0.25 * h * (1.0 - 1e-6));
            g.h = (float)h; g.reach = 0.0f; g.info = nullptr; g.planes = nullptr;
            const size_t nc = (size_t)g.nx * g.ny * g.nz;
            unsigned char *occ = nullptr, *cells = nullptr;
            unsigned short *d2 = nullptr;
            unsigned *info = nullptr;
            if ((e = gd_pool_get(c, 14, nc, (void **)&occ)) != cudaSuccess) break;
            if ((e = gd_pool_get(c, 15, 2 * nc, (void **)&d2)) != cudaSuccess) break;
            if ((e = gd_pool_get(c, 16, nc, (void **)&cells)) != cudaSuccess) break;
            if ((e = gd_pool_get(c, 18, 4 * nc, (void **)&info)) != cudaSuccess) break;
            cudaMemsetAsync(occ, 0, nc, st);
            if (n >= (1 << 16)) gd_k_grid_mark<<<nb, tb, 0, st>>>(ref_lo, ref_hi, n, g, occ, 1);
            else gd_k_grid_mark<<<(unsigned)(((size_t)n * 32 + tb - 1) / tb), tb, 0, st>>>(ref_lo, ref_hi, n, g, occ, 0);
            gd_k_grid_dt_x<<<(g.ny * g.nz + 127) / 128, 128, 0, st>>>(g, occ);
            gd_k_grid_dt_y<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(g, occ, d2);
            gd_k_grid_dt_z<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(g, d2, cells, info);
            launches += 4;
            // so far the cells' words hold scalar bounds only; the plane lists come with the build (GADEP_BUILD_PLANE_LISTS)
            // or with the first large run (gd_build_plane_lists)
            g.info = info;
            c->grid_scalar = cells;
            c->grid = g;
        }
        cudaEventRecord(c->evb1, st);
        if ((e = cudaGetLastError()) != cudaSuccess) break;
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) break;
        if (n > 1 && (e = cudaMemcpy(&depth, scene + 6, sizeof(int), cudaMemcpyDeviceToHost)) != cudaSuccess) break;
        cudaEventElapsedTime(&c->last_build_ms, c->evb0, c->evb1);
        // per-material entry table: the surfaces that have the material on one side.  A surface without an entry node
        // (never for a closed surface of >= 2 references) or too many surfaces around one material -> root for it.
        c->have_entries = false;
        if (cls_bits > 0) {
            std::vector<int> se(c->n_surf);
            if ((e = cudaMemcpy(se.data(), surf_entry, 4 * (size_t)c->n_surf, cudaMemcpyDeviceToHost)) != cudaSuccess) break;
            int table[GADEP_MAX_MATERIALS][1 + GD_ENTRY_MAX];
            memset(table, 0, sizeof(table));
            for (int m = 0; m < GADEP_MAX_MATERIALS; ++m) {
                int cnt = 0;
                bool ok = true;
                for (int s2 = 0; s2 < c->n_surf && ok; ++s2) {
                    if (c->h_sides[2 * s2] != m && c->h_sides[2 * s2 + 1] != m) continue;
                    if (se[s2] < 0 || cnt == GD_ENTRY_MAX) ok = false;
                    else table[m][1 + cnt++] = se[s2];
                }
                table[m][0] = ok ? cnt : 0;
            }
            if (!c->d_mat_entry && (e = cudaMalloc(&c->d_mat_entry, sizeof(table))) != cudaSuccess) break;
            if ((e = cudaMemcpy(c->d_mat_entry, table, sizeof(table), cudaMemcpyHostToDevice)) != cudaSuccess) break;
            c->have_entries = true;
        }
    } while (0);
    if (e != cudaSuccess) rc = gd_fail(c, GADEP_E_CUDA, "BVH build failed: %s", cudaGetErrorString(e));
    else if (depth >= GD_STACK || 3 * depth + 4 + GD_ENTRY_MAX > GD_STACK4) rc = gd_fail(c, GADEP_E_ARG, "BVH depth %d exceeds the traversal stack (%d)", depth, GD_STACK);
    if (rc != GADEP_OK) return rc;
    c->bvh_depth = depth;
    c->n_ref = n;
    c->last_build_launches = launches;
    c->have_bvh = true;
    if (flags == GADEP_BUILD_PLANE_LISTS) return gd_build_plane_lists(c);
    return GADEP_OK;
}

// nodes + triangle records far beyond the 126 MB L2: a node visit is then a fetch from HBM
static bool gd_large_hierarchy(const gadep_ctx *c) { return (size_t)c->n_ref * (sizeof(GdNode4) + sizeof(GdTri)) > ((size_t)256 << 20); }

static GdBvh gd_bvh_view(const gadep_ctx *c) {
    GdBvh b;
    b.grid = c->grid;
    b.nodes = c->d_nodes; b.nodes4 = c->d_nodes4; b.nodes8 = c->d_nodes8; b.nodes4q = c->d_nodes4q; b.tris = c->d_leaf_tris; b.n_tri = c->n_ref; b.root_is_leaf = c->n_ref == 1;
    b.mat_entry = c->have_entries ? c->d_mat_entry : nullptr;
    return b;
}

// ---------------------------------------------------------------- source
extern "C" int gadep_set_source(gadep_ctx *c, const gadep_source *s) {
    if (!c) return GADEP_E_NULL;
    if (!s || !s->line_mev || !s->line_intensity) return gd_fail(c, GADEP_E_NULL, "null source");
    if (!c->have_mat) return gd_fail(c, GADEP_E_ORDER, "gadep_set_source before gadep_set_materials");
    if (s->kind < 0 || s->kind > 2) return gd_fail(c, GADEP_E_ARG, "unknown source kind %d", s->kind);
    if (s->n_lines <= 0 || s->n_lines > GADEP_MAX_LINES) return gd_fail(c, GADEP_E_ARG, "n_lines %d out of range", s->n_lines);
    GdSource g;
    memset(&g, 0, sizeof(g));
    g.kind = s->kind;
    for (int k = 0; k < 3; ++k) { g.pos[k] = s->pos[k]; g.dir[k] = s->dir[k]; }
    g.cyl_r = s->cyl_r; g.cyl_z0 = s->cyl_z0; g.cyl_z1 = s->cyl_z1;
    g.ex_r = s->ex_r; g.ex_z0 = s->ex_z0; g.ex_z1 = s->ex_z1;
    g.n_lines = s->n_lines;
    g.n_copies = 1;
    if (s->kind == GADEP_SRC_VOLUME && !(s->cyl_r > 0 && s->cyl_z1 > s->cyl_z0)) return gd_fail(c, GADEP_E_ARG, "empty source cylinder");
    if (s->kind == GADEP_SRC_BEAM) {
        double n2 = (double)s->dir[0] * s->dir[0] + (double)s->dir[1] * s->dir[1] + (double)s->dir[2] * s->dir[2];
        if (!(std::fabs(n2 - 1.0) < 1e-3)) return gd_fail(c, GADEP_E_ARG, "beam direction is not a unit vector");
    }
    float cum = 0.0f;
    for (int l = 0; l < s->n_lines; ++l) {
        float e = s->line_mev[l], w = s->line_intensity[l];
        if (!(w >= 0) || !std::isfinite(w)) return gd_fail(c, GADEP_E_ARG, "line %d: negative intensity", l);
        if (!((double)e >= c->e_min * (1 - 1e-6) && (double)e <= c->e_max * (1 + 1e-6)))
            return gd_fail(c, GADEP_E_ARG, "line %d: energy %g outside the table range", l, (double)e);
        cum += w;
        g.line_mev[l] = e; g.line_cum[l] = cum;
    }
    if (!(cum > 0)) return gd_fail(c, GADEP_E_ARG, "all line intensities are zero");
    c->src = g;
    c->have_src = true;
    return GADEP_OK;
}

extern "C" int gadep_set_source_copies(gadep_ctx *c, int n_copies, const float *offsets) {
    if (!c) return GADEP_E_NULL;
    if (!c->have_src) return gd_fail(c, GADEP_E_ORDER, "gadep_set_source_copies before gadep_set_source");
    if (n_copies < 1 || n_copies > 8 || (n_copies > 1 && !offsets)) return gd_fail(c, GADEP_E_ARG, "n_copies %d (1..8)", n_copies);
    const int nl = c->src.n_lines;
    if (n_copies * nl > GADEP_MAX_LINES) return gd_fail(c, GADEP_E_ARG, "%d copies x %d lines exceed GADEP_MAX_LINES", n_copies, nl);
    c->src.n_copies = n_copies;
    memset(c->src.copy_off, 0, sizeof(c->src.copy_off));
    for (int k = 0; k < n_copies; ++k)
        for (int a = 0; a < 3; ++a) {
            const float v = n_copies > 1 ? offsets[3 * k + a] : 0.0f;
            if (!std::isfinite(v)) return gd_fail(c, GADEP_E_ARG, "copy %d: offset not finite", k);
            c->src.copy_off[k][a] = v;
        }
    for (int k = 1; k < n_copies; ++k)
        for (int l = 0; l < nl; ++l) c->src.line_mev[k * nl + l] = c->src.line_mev[l];
    return GADEP_OK;
}

// ---------------------------------------------------------------- run
static int gd_ensure_tally(gadep_ctx *c, int n_bins) {
    if (c->d_tally && c->cap_bins >= n_bins) return GADEP_OK;
    cudaFree(c->d_tally); c->d_tally = nullptr;
    GD_CUDA(c, cudaMalloc(&c->d_tally, sizeof(unsigned long long) * ((size_t)n_bins + 1 + 2 * GADEP_MAX_LINES)));
    c->cap_bins = n_bins;
    return GADEP_OK;
}

static int gd_launch_transport(gadep_ctx *c, unsigned long long first, unsigned long long n, unsigned long long seed,
                               int n_bins, float e_max, bool accumulate, float *d_edep, unsigned *d_flags) {
    if (!c->have_mat || !c->have_mesh || !c->have_bvh || !c->have_src)
        return gd_fail(c, GADEP_E_ORDER, "run needs materials, mesh, BVH and source");
    if (n_bins <= 0 || n_bins > (1 << 20) || !(e_max > 0)) return gd_fail(c, GADEP_E_ARG, "bad spectrum shape");
    // materials may have been (re)set after the mesh or the source: every id and line energy is checked against the tables
    // the kernel will index (an id >= n_mat would read past the attenuation table in shared memory)
    if (c->world < 0 || c->world >= c->n_mat) return gd_fail(c, GADEP_E_INDEX, "world material %d outside the %d materials set", c->world, c->n_mat);
    for (size_t k = 0; k < c->h_sides.size(); ++k)
        if (c->h_sides[k] != GADEP_MAT_KILL && (c->h_sides[k] < 0 || c->h_sides[k] >= c->n_mat))
            return gd_fail(c, GADEP_E_INDEX, "surface %zu: side material %d outside the %d materials set", k / 2, c->h_sides[k], c->n_mat);
    for (int l = 0; l < c->src.n_lines; ++l)
        if (!((double)c->src.line_mev[l] >= c->e_min * (1 - 1e-6) && (double)c->src.line_mev[l] <= c->e_max * (1 + 1e-6)))
            return gd_fail(c, GADEP_E_ARG, "line %d: energy %g outside the table range", l, (double)c->src.line_mev[l]);
    GD_CUDA(c, cudaSetDevice(c->device));
    bool same_shape = c->d_tally && c->n_bins == n_bins && c->spec_e_max == e_max;
    int rc = gd_ensure_tally(c, n_bins);
    if (rc) return rc;
    cudaStream_t st = c->stream;
    size_t tally_bytes = sizeof(unsigned long long) * ((size_t)n_bins + 1 + 2 * GADEP_MAX_LINES);
    if (!(accumulate && same_shape)) {
        GD_CUDA(c, cudaMemsetAsync(c->d_tally, 0, tally_bytes, st));
        GD_CUDA(c, cudaMemsetAsync(c->d_counters, 0, sizeof(GdCounters), st));
    }
    c->n_bins = n_bins; c->spec_e_max = e_max;
    double de = (double)e_max / n_bins;
    for (int l = 0; l < c->src.n_lines * c->src.n_copies; ++l) {
        double b = std::floor((double)c->src.line_mev[l] / de);
        c->src.line_bin[l] = b >= n_bins ? n_bins : (int)b;
    }
    GD_CUDA(c, cudaMemcpyAsync(c->d_src, &c->src, sizeof(GdSource), cudaMemcpyHostToDevice, st));
    GdMaterials M;
    M.n_mat = c->n_mat; M.n_grid = c->n_grid;
    M.ln_e0 = (float)std::log(c->e_min);
    M.inv_dln = (float)((c->n_grid - 1) / (std::log(c->e_max) - std::log(c->e_min)));
    M.e_cut = (float)c->e_min;
    M.table = c->d_table; M.scoring_mask = c->scoring_mask; M.world_material = c->world;
    for (int m = 0; m < GADEP_MAX_MATERIALS; ++m) M.rho[m] = c->rho[m];
    GdTally T;
    T.spectrum = c->d_tally; T.emitted = c->d_tally + n_bins + 1; T.peak = T.emitted + GADEP_MAX_LINES;
    T.counters = c->d_counters; T.n_bins = n_bins; T.inv_de = (float)((double)n_bins / (double)e_max);
    if (n > 0xFFFFFFFFull) return gd_fail(c, GADEP_E_ARG, "more than 2^32-1 histories in one launch");
    size_t smem = sizeof(float) * (size_t)c->n_mat * 4 * c->n_grid + sizeof(unsigned) * ((size_t)n_bins + 1);
    const int variant = c->kernel_variant;
    const bool wide8 = c->run_width == 8;
    // a hierarchy far larger than the L2 (126 MB): the 28-warp instance of the wavefront kernel (more rays in flight)
    const bool q4 = c->run_width == GD_WIDTH_4Q;
    const bool lat16 = variant == 2 && !wide8 && c->wave_threads != GD_W_THREADS &&
                       (c->wave_threads == GD_W_THREADS_LAT || gd_large_hierarchy(c));
    const int threads = variant == 2 ? (lat16 ? GD_W_THREADS_LAT : GD_W_THREADS) : (variant == 5 ? GD_WS_THREADS : GD_RUN_THREADS);
    if (variant == 2 || variant == 5) smem += sizeof(float) * (size_t)GD_W_NF * GD_W_NSLOT;
    if (smem > 220 * 1024) return gd_fail(c, GADEP_E_ARG, "tables + spectrum + photon slots (%zu B) do not fit in shared memory", smem);
    const void *kern = variant == 5 ? (wide8 ? (const void *)gd_k_transport_ws<8> : (const void *)gd_k_transport_ws<4>)
                     : variant == 2 ? (wide8 ? (const void *)gd_k_transport_wave<8>
                                      : q4 ? (lat16 ? (const void *)gd_k_transport_wave<GD_WIDTH_4Q, GD_W_THREADS_LAT> : (const void *)gd_k_transport_wave<GD_WIDTH_4Q>)
                                           : (lat16 ? (const void *)gd_k_transport_wave<4, GD_W_THREADS_LAT> : (const void *)gd_k_transport_wave<4>))
                                    : (variant == 1 ? (const void *)gd_k_transport_refill
                                                  : (variant == 3 ? (const void *)gd_k_transport<true, false>
                                                     : (variant == 4 ? (const void *)gd_k_transport<false, true>
                                                        : (variant == 6 ? (const void *)gd_k_transport<false, false, true> : (const void *)gd_k_transport<false, false>))));
    GD_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem));
    if (per_sm < 1) return gd_fail(c, GADEP_E_CUDA, "transport kernel does not fit on an SM (%zu B shared memory)", smem);
    const unsigned long long per_block = (variant == 2 || variant == 5) ? (unsigned long long)GD_W_NSLOT : GD_RUN_THREADS;
    unsigned long long want = (n + per_block - 1) / per_block;
    int grid = (int)std::min<unsigned long long>((unsigned long long)c->n_sm * per_sm, std::max<unsigned long long>(want, 1));
    if (variant == 2 || variant == 5) {
        size_t need = (size_t)grid * GD_W_NSLOT * 8;
        if (need > c->pair_floats) {
            cudaFree(c->d_pair); c->d_pair = nullptr; c->pair_floats = 0;
            GD_CUDA(c, cudaMalloc(&c->d_pair, need * sizeof(float)));
            c->pair_floats = need;
        }
    }
    if ((variant == 2 || variant == 5) && c->list_policy == 0 && !c->lists_built && n >= c->list_min_hist) {
        rc = gd_build_plane_lists(c);
        if (rc) return rc;
    }
    GD_CUDA(c, cudaEventRecord(c->ev0, st));
    c->last_run_launches = 0;
    if (n > 0) {
        unsigned long long warps = (unsigned long long)grid * (threads / 32);
        unsigned chunk = (unsigned)std::min<unsigned long long>(1024, std::max<unsigned long long>(32, n / (warps * 16)));
        if (variant == 2 || variant == 5)     // the wavefront kernels hand out history indices per block
            chunk = (unsigned)std::min<unsigned long long>(8192, std::max<unsigned long long>(256, n / ((unsigned long long)grid * 32)));
        if (variant == 1 || variant == 2 || variant == 5) GD_CUDA(c, cudaMemsetAsync(c->d_next, 0, sizeof(unsigned long long), st));
        if (variant == 5 && wide8) {
            gd_k_transport_ws<8><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags,
                                                              c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 5) {
            gd_k_transport_ws<4><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags,
                                                              c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 2 && wide8) {
            gd_k_transport_wave<8><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags,
                                                                c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 2 && q4 && lat16) {
            gd_k_transport_wave<GD_WIDTH_4Q, GD_W_THREADS_LAT><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep,
                                                                                            d_flags, c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 2 && q4) {
            gd_k_transport_wave<GD_WIDTH_4Q><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags,
                                                                          c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 2 && lat16) {
            gd_k_transport_wave<4, GD_W_THREADS_LAT><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep,
                                                                                  d_flags, c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 2) {
            gd_k_transport_wave<4><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags,
                                                                c->d_next, chunk, c->d_pair, c->tune);
        } else if (variant == 1) {
            gd_k_transport_refill<<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep,
                                                               d_flags, c->d_next, chunk);
        } else if (variant == 3) {
            gd_k_transport<true, false><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags);
        } else if (variant == 4) {
            gd_k_transport<false, true><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags);
        } else if (variant == 6) {
            gd_k_transport<false, false, true><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags);
        } else {
            gd_k_transport<false, false><<<grid, threads, smem, st>>>(gd_bvh_view(c), M, c->d_src, first, n, seed, T, d_edep, d_flags);
        }
        c->last_run_launches = 1;
    }
    GD_CUDA(c, cudaEventRecord(c->ev1, st));
    GD_CUDA(c, cudaGetLastError());
    c->results_stale = true; c->have_results = true; c->run_timed = true;
    return GADEP_OK;
}

static int gd_fetch_results(gadep_ctx *c) {
    if (!c->have_results) return gd_fail(c, GADEP_E_ORDER, "no run yet");
    if (!c->results_stale) return GADEP_OK;
    GD_CUDA(c, cudaSetDevice(c->device));
    GD_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->d_tally && c->n_bins > 0) {
        c->h_spectrum.resize((size_t)c->n_bins + 1);
        GD_CUDA(c, cudaMemcpy(c->h_spectrum.data(), c->d_tally, sizeof(unsigned long long) * ((size_t)c->n_bins + 1), cudaMemcpyDeviceToHost));
        GD_CUDA(c, cudaMemcpy(c->h_emitted, c->d_tally + c->n_bins + 1, sizeof(c->h_emitted), cudaMemcpyDeviceToHost));
        GD_CUDA(c, cudaMemcpy(c->h_peak, c->d_tally + c->n_bins + 1 + GADEP_MAX_LINES, sizeof(c->h_peak), cudaMemcpyDeviceToHost));
    }
    GD_CUDA(c, cudaMemcpy(&c->h_counters, c->d_counters, sizeof(GdCounters), cudaMemcpyDeviceToHost));
    if (c->run_timed) { cudaEventElapsedTime(&c->last_run_ms, c->ev0, c->ev1); c->run_timed = false; }
    c->results_stale = false;
    {
        unsigned ovf = 0;
        GD_CUDA(c, cudaMemcpyFromSymbol(&ovf, gd_stack_overflow, sizeof(ovf)));
        if (ovf) {
            const unsigned zero = 0;
            cudaMemcpyToSymbol(gd_stack_overflow, &zero, sizeof(zero));
            c->n_stack_overflow += ovf;
            return gd_fail(c, GADEP_E_ARG, "%u rays ran out of traversal stack (BVH too deep for GD_STACK8)", ovf);
        }
    }
    return GADEP_OK;
}

static int gd_variant_of(int flags) {
    return (flags & GADEP_RUN_ELECTRON_RANGE) ? 6 : (flags & GADEP_RUN_WARP_SPECIALISED) ? 5 : (flags & GADEP_RUN_PARTIAL_XS) ? 4
           : (flags & GADEP_RUN_PARITY_LOCALISATION) ? 3 : ((flags & GADEP_RUN_HISTORY_PER_THREAD) ? 0 : ((flags & GADEP_RUN_PERSISTENT_LANES) ? 1 : 2));
}

extern "C" int gadep_set_densities(gadep_ctx *c, int n_mat, const float *rho_g_cm3) {
    if (!c) return GADEP_E_NULL;
    if (!rho_g_cm3) return gd_fail(c, GADEP_E_NULL, "null density array");
    if (n_mat <= 0 || n_mat > GADEP_MAX_MATERIALS || (c->have_mat && n_mat != c->n_mat))
        return gd_fail(c, GADEP_E_ARG, "n_mat %d does not match the materials", n_mat);
    for (int m = 0; m < n_mat; ++m)
        if (!(rho_g_cm3[m] >= 0.0f) || !std::isfinite(rho_g_cm3[m])) return gd_fail(c, GADEP_E_ARG, "material %d: bad density", m);
    for (int m = 0; m < GADEP_MAX_MATERIALS; ++m) c->rho[m] = m < n_mat ? rho_g_cm3[m] : 0.0f;
    c->have_rho = true;
    return GADEP_OK;
}

extern "C" int gadep_run(gadep_ctx *c, unsigned long long n_histories, unsigned long long seed, const gadep_run_opts *opts,
                         unsigned long long *spectrum) {
    if (!c) return GADEP_E_NULL;
    if (!opts) return gd_fail(c, GADEP_E_NULL, "null run options");
    bool dev_out = gd_is_device_ptr(spectrum);
    if ((opts->flags & GADEP_RUN_ASYNC) && spectrum && !dev_out)
        return gd_fail(c, GADEP_E_ARG, "GADEP_RUN_ASYNC needs a device spectrum pointer");
    if ((opts->flags & GADEP_RUN_ELECTRON_RANGE) && !c->have_rho)
        return gd_fail(c, GADEP_E_ORDER, "GADEP_RUN_ELECTRON_RANGE needs gadep_set_densities");
    {   // GADEP_RUN_* kernel selectors exclude one another
        const int sel = opts->flags & (GADEP_RUN_HISTORY_PER_THREAD | GADEP_RUN_PERSISTENT_LANES | GADEP_RUN_PARITY_LOCALISATION |
                                       GADEP_RUN_PARTIAL_XS | GADEP_RUN_ELECTRON_RANGE | GADEP_RUN_WARP_SPECIALISED);
        if (sel & (sel - 1)) return gd_fail(c, GADEP_E_ARG, "run flags 0x%x select more than one kernel", opts->flags);
    }
    c->kernel_variant = gd_variant_of(opts->flags);
    if (c->kernel_variant == 2 && c->prefer_ws) c->kernel_variant = 5;
    c->run_width = (opts->flags & GADEP_RUN_BVH8) ? 8 : c->bvh_width;
    int rc = gd_launch_transport(c, opts->first_history, n_histories, seed, opts->n_bins, opts->e_max_mev,
                                 (opts->flags & GADEP_RUN_ACCUMULATE) != 0, nullptr, nullptr);
    if (rc) return rc;
    size_t bytes = sizeof(unsigned long long) * ((size_t)opts->n_bins + 1);
    if (spectrum && dev_out) GD_CUDA(c, cudaMemcpyAsync(spectrum, c->d_tally, bytes, cudaMemcpyDeviceToDevice, c->stream));
    if (opts->flags & GADEP_RUN_ASYNC) return GADEP_OK;
    rc = gd_fetch_results(c);
    if (rc) return rc;
    if (spectrum && !dev_out) memcpy(spectrum, c->h_spectrum.data(), bytes);
    return GADEP_OK;
}

extern "C" int gadep_fepe(const gadep_ctx *cc, int line, int mode, double *fepe, double *std_err) {
    gadep_ctx *c = const_cast<gadep_ctx *>(cc);
    if (!c) return GADEP_E_NULL;
    if (!fepe) return gd_fail(c, GADEP_E_NULL, "null output");
    int rc = gd_fetch_results(c);
    if (rc) return rc;
    if (line < 0 || line >= c->src.n_lines * c->src.n_copies) return gd_fail(c, GADEP_E_ARG, "line %d out of range", line);
    double em = (double)c->h_emitted[line];
    double p = 0.0;
    if (em > 0) {
        if (mode == 0) p = (double)c->h_peak[line] / em;
        else if (mode == 1) {
            int b = c->src.line_bin[line];
            if (b < 1 || b >= c->n_bins - 1) return gd_fail(c, GADEP_E_ARG, "line %d lies outside the spectrum", line);
            p = ((double)c->h_spectrum[b] - 0.5 * ((double)c->h_spectrum[b - 1] + (double)c->h_spectrum[b + 1])) / em;
        } else return gd_fail(c, GADEP_E_ARG, "unknown mode %d", mode);
    }
    *fepe = p;
    if (std_err) *std_err = em > 0 ? std::sqrt(std::max(p * (1.0 - p), 0.0) / em) : 0.0;
    return GADEP_OK;
}

// ---------------------------------------------------------------- hooks
extern "C" int gadep_trace_rays(gadep_ctx *c, const float *org, const float *dir, long long n_rays, int filter_material,
                                float t_min, int *tri_out, float *t_out) {
    if (!c) return GADEP_E_NULL;
    if (!org || !dir || !tri_out || !t_out) return gd_fail(c, GADEP_E_NULL, "null ray array");
    if (!c->have_bvh) return gd_fail(c, GADEP_E_ORDER, "gadep_trace_rays before gadep_build_bvh");
    if (n_rays < 0) return gd_fail(c, GADEP_E_ARG, "negative ray count");
    if (n_rays == 0) return GADEP_OK;
    GD_CUDA(c, cudaSetDevice(c->device));
    bool dev = gd_is_device_ptr(org);
    if (dev != gd_is_device_ptr(dir) || dev != gd_is_device_ptr(tri_out) || dev != gd_is_device_ptr(t_out))
        return gd_fail(c, GADEP_E_ARG, "ray arrays must live in one memory space");
    cudaStream_t st = c->stream;
    const float *d_org = org, *d_dir = dir;
    int *d_tri = tri_out;
    float *d_t = t_out;
    float *stage = nullptr;
    size_t nb3 = sizeof(float) * 3 * (size_t)n_rays, nb1 = sizeof(float) * (size_t)n_rays;
    if (!dev) {
        GD_CUDA(c, cudaMalloc(&stage, 2 * nb3 + 2 * nb1));
        d_org = stage; d_dir = stage + 3 * n_rays; d_tri = (int *)(stage + 6 * n_rays); d_t = stage + 7 * n_rays;
        cudaMemcpyAsync(stage, org, nb3, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(stage + 3 * n_rays, dir, nb3, cudaMemcpyHostToDevice, st);
    }
    cudaMemsetAsync(c->d_counters, 0, sizeof(GdCounters), st);
    int per_sm = 1;
    const bool wide8 = c->bvh_width == 8, q4 = c->bvh_width == GD_WIDTH_4Q || (!c->width_set && gd_large_hierarchy(c));
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, wide8 ? gd_k_trace_wave<8> : (q4 ? gd_k_trace_wave<GD_WIDTH_4Q> : gd_k_trace_wave<4>), 256, 0));
    int grid = (int)std::min<long long>((n_rays + 255) / 256, (long long)c->n_sm * std::max(per_sm, 1));
    unsigned chunk = (unsigned)std::min<long long>(2048, std::max<long long>(32, n_rays / ((long long)grid * 8 * 8)));
    cudaMemsetAsync(c->d_next, 0, sizeof(unsigned long long), st);
    cudaEventRecord(c->ev0, st);
    if (wide8) gd_k_trace_wave<8><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                         c->d_counters, c->d_next, chunk, c->tune);
    else if (q4) gd_k_trace_wave<GD_WIDTH_4Q><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                                   c->d_counters, c->d_next, chunk, c->tune);
    else gd_k_trace_wave<4><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                   c->d_counters, c->d_next, chunk, c->tune);
    cudaEventRecord(c->ev1, st);
    c->last_run_launches = 1;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !dev) {
        cudaMemcpyAsync(tri_out, d_tri, nb1, cudaMemcpyDeviceToHost, st);
        cudaMemcpyAsync(t_out, d_t, nb1, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpy(&c->h_counters, c->d_counters, sizeof(GdCounters), cudaMemcpyDeviceToHost);
    cudaFree(stage);
    if (e != cudaSuccess) return gd_fail(c, GADEP_E_CUDA, "trace failed: %s", cudaGetErrorString(e));
    cudaEventElapsedTime(&c->last_run_ms, c->ev0, c->ev1);
    c->run_timed = false;
    return GADEP_OK;
}

extern "C" int gadep_locate(gadep_ctx *c, const float *org, const float *dir, long long n, int mode, int *material_out) {
    if (!c) return GADEP_E_NULL;
    if (!org || !dir || !material_out) return gd_fail(c, GADEP_E_NULL, "null array");
    if (!c->have_bvh) return gd_fail(c, GADEP_E_ORDER, "gadep_locate before gadep_build_bvh");
    if (n < 0 || (mode != GADEP_LOCATE_SIDE_ID && mode != GADEP_LOCATE_PARITY)) return gd_fail(c, GADEP_E_ARG, "bad count or mode");
    if (n == 0) return GADEP_OK;
    GD_CUDA(c, cudaSetDevice(c->device));
    const bool dev = gd_is_device_ptr(org);
    if (dev != gd_is_device_ptr(dir) || dev != gd_is_device_ptr(material_out))
        return gd_fail(c, GADEP_E_ARG, "arrays must live in one memory space");
    cudaStream_t st = c->stream;
    const float *d_org = org, *d_dir = dir;
    int *d_mat = material_out;
    float *stage = nullptr;
    const size_t nb3 = sizeof(float) * 3 * (size_t)n;
    if (!dev) {
        GD_CUDA(c, cudaMalloc(&stage, 2 * nb3 + sizeof(int) * (size_t)n));
        d_org = stage; d_dir = stage + 3 * n; d_mat = (int *)(stage + 6 * n);
        cudaMemcpyAsync(stage, org, nb3, cudaMemcpyHostToDevice, st);
        cudaMemcpyAsync(stage + 3 * n, dir, nb3, cudaMemcpyHostToDevice, st);
    }
    cudaMemsetAsync(c->d_counters, 0, sizeof(GdCounters), st);
    cudaEventRecord(c->ev0, st);
    gd_k_locate<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n, mode, c->world, d_mat, c->d_counters);
    cudaEventRecord(c->ev1, st);
    c->last_run_launches = 1;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !dev) cudaMemcpyAsync(material_out, d_mat, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpy(&c->h_counters, c->d_counters, sizeof(GdCounters), cudaMemcpyDeviceToHost);
    cudaFree(stage);
    if (e != cudaSuccess) return gd_fail(c, GADEP_E_CUDA, "locate failed: %s", cudaGetErrorString(e));
    cudaEventElapsedTime(&c->last_run_ms, c->ev0, c->ev1);
    c->run_timed = false;
    return GADEP_OK;
}

// ---------------------------------------------------------------- detector-resolution broadening
// out[j] = sum_i S[i] * P(bin j | Gaussian centred on the middle of bin i, FWHM(E)^2 = a + b E + c E^2); bin 0 also takes
// the mass below 0, the overflow slot the mass above e_max (and the unbroadened overflow counts): the total is kept.
__global__ void gd_k_broaden(const unsigned long long *__restrict__ spec, int n_bins, double e_max, double a, double b,
                             double c, double *__restrict__ out) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > n_bins) return;
    const double de = e_max / n_bins;
    const double lo = j == 0 ? -1.0e300 : (j == n_bins ? e_max : j * de);
    const double hi = j == n_bins ? 1.0e300 : (j + 1) * de;
    double acc = j == n_bins ? (double)spec[n_bins] : 0.0;
    for (int i = 0; i < n_bins; ++i) {
        const unsigned long long s = spec[i];
        if (!s) continue;
        const double e = (i + 0.5) * de;
        const double fwhm2 = a + b * e + c * e * e;
        if (!(fwhm2 > 0.0)) { if (i == j) acc += (double)s; continue; }
        const double inv = 2.3548200450309493 / sqrt(2.0 * fwhm2);          // 1 / (sigma sqrt 2)
        acc += (double)s * 0.5 * (erf((hi - e) * inv) - erf((lo - e) * inv));
    }
    out[j] = acc;
}

extern "C" int gadep_broaden(gadep_ctx *c, double fwhm_a, double fwhm_b, double fwhm_c, double *out) {
    if (!c) return GADEP_E_NULL;
    if (!out) return gd_fail(c, GADEP_E_NULL, "null output");
    if (!c->have_results || !c->d_tally || c->n_bins <= 0) return gd_fail(c, GADEP_E_ORDER, "gadep_broaden before gadep_run");
    if (!(fwhm_a >= 0) || !std::isfinite(fwhm_b) || !std::isfinite(fwhm_c)) return gd_fail(c, GADEP_E_ARG, "bad resolution parameters");
    GD_CUDA(c, cudaSetDevice(c->device));
    const bool dev = gd_is_device_ptr(out);
    const size_t bytes = sizeof(double) * ((size_t)c->n_bins + 1);
    double *d_out = out;
    if (!dev) GD_CUDA(c, cudaMalloc(&d_out, bytes));
    gd_k_broaden<<<(c->n_bins + 1 + 127) / 128, 128, 0, c->stream>>>(c->d_tally, c->n_bins, (double)c->spec_e_max, fwhm_a, fwhm_b,
                                                                    fwhm_c, d_out);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !dev) e = cudaMemcpyAsync(out, d_out, bytes, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (!dev) cudaFree(d_out);
    if (e != cudaSuccess) return gd_fail(c, GADEP_E_CUDA, "broaden failed: %s", cudaGetErrorString(e));
    return GADEP_OK;
}

extern "C" int gadep_run_histories_ex(gadep_ctx *c, unsigned long long first, long long n, unsigned long long seed,
                                      int run_flags, float *edep_out, unsigned *flags_out);
extern "C" int gadep_run_histories(gadep_ctx *c, unsigned long long first, long long n, unsigned long long seed,
                                   float *edep_out, unsigned *flags_out) {
    return gadep_run_histories_ex(c, first, n, seed, 0, edep_out, flags_out);
}

extern "C" int gadep_run_histories_ex(gadep_ctx *c, unsigned long long first, long long n, unsigned long long seed,
                                      int run_flags, float *edep_out, unsigned *flags_out) {
    if (!c) return GADEP_E_NULL;
    if (n < 0) return gd_fail(c, GADEP_E_ARG, "negative history count");
    if ((run_flags & GADEP_RUN_ELECTRON_RANGE) && !c->have_rho)
        return gd_fail(c, GADEP_E_ORDER, "GADEP_RUN_ELECTRON_RANGE needs gadep_set_densities");
    GD_CUDA(c, cudaSetDevice(c->device));
    bool dev_e = gd_is_device_ptr(edep_out), dev_f = gd_is_device_ptr(flags_out);
    float *d_e = edep_out;
    unsigned *d_f = flags_out;
    float *stage_e = nullptr;
    unsigned *stage_f = nullptr;
    if (edep_out && !dev_e && n > 0) { GD_CUDA(c, cudaMalloc(&stage_e, sizeof(float) * (size_t)n)); d_e = stage_e; }
    if (flags_out && !dev_f && n > 0) { GD_CUDA(c, cudaMalloc(&stage_f, sizeof(unsigned) * (size_t)n)); d_f = stage_f; }
    int n_bins = c->n_bins > 0 ? c->n_bins : 4096;
    float e_max = c->spec_e_max > 0 ? c->spec_e_max : 2.0f;
    {
        const int sel = run_flags & (GADEP_RUN_HISTORY_PER_THREAD | GADEP_RUN_PERSISTENT_LANES | GADEP_RUN_PARITY_LOCALISATION |
                                     GADEP_RUN_PARTIAL_XS | GADEP_RUN_ELECTRON_RANGE | GADEP_RUN_WARP_SPECIALISED);
        if (sel & (sel - 1)) { cudaFree(stage_e); cudaFree(stage_f); return gd_fail(c, GADEP_E_ARG, "run flags 0x%x select more than one kernel", run_flags); }
    }
    c->kernel_variant = gd_variant_of(run_flags & ~(GADEP_RUN_ASYNC | GADEP_RUN_ACCUMULATE));   // 0: the default kernel
    c->run_width = (run_flags & GADEP_RUN_BVH8) ? 8 : c->bvh_width;
    int rc = gd_launch_transport(c, first, (unsigned long long)n, seed, n_bins, e_max, false, d_e, d_f);
    if (rc == GADEP_OK) rc = gd_fetch_results(c);
    if (rc == GADEP_OK && stage_e) cudaMemcpy(edep_out, stage_e, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost);
    if (rc == GADEP_OK && stage_f) cudaMemcpy(flags_out, stage_f, sizeof(unsigned) * (size_t)n, cudaMemcpyDeviceToHost);
    cudaFree(stage_e); cudaFree(stage_f);
    return rc;
}

extern "C" int gadep_get_counters(const gadep_ctx *cc, gadep_counters *out) {
    gadep_ctx *c = const_cast<gadep_ctx *>(cc);
    if (!c) return GADEP_E_NULL;
    if (!out) return gd_fail(c, GADEP_E_NULL, "null output");
    if (c->have_results && c->results_stale) { int rc = gd_fetch_results(c); if (rc) return rc; }
    memset(out, 0, sizeof(*out));
    const GdCounters &h = c->h_counters;
    out->n_histories = h.n_histories; out->n_queries = h.n_queries; out->n_box_tests = h.n_box_tests;
    out->n_tri_tests = h.n_tri_tests; out->n_crossings = h.n_crossings; out->n_pe = h.n_pe; out->n_compton = h.n_compton;
    out->n_coherent = h.n_coherent; out->n_pair = h.n_pair; out->n_escaped = h.n_escaped; out->n_leak = h.n_leak;
    out->n_cutoff = h.n_cutoff; out->n_stack_overflow = c->n_stack_overflow; out->n_skipped_queries = h.n_skipped;
    out->n_parity_queries = h.n_parity; out->n_parity_mismatch = h.n_parity_mismatch;
    out->n_grid_list_cells = c->n_list_cells; out->n_grid_lists = c->n_listed;
    memcpy(out->emitted, c->h_emitted, sizeof(out->emitted));
    memcpy(out->peak, c->h_peak, sizeof(out->peak));
    out->n_lines = c->src.n_lines * (c->src.n_copies > 0 ? c->src.n_copies : 1);
    out->n_bvh_nodes = c->have_bvh ? std::max(c->n_ref - 1, 0) : 0;
    out->bvh_max_depth = c->bvh_depth;
    out->last_run_ms = c->last_run_ms; out->last_build_ms = c->last_build_ms;
    out->last_run_launches = c->last_run_launches; out->last_build_launches = c->last_build_launches;
    return GADEP_OK;
}

__global__ void gd_k_philox(uint4 ctr, uint2 key, int which, unsigned *out) {
    if (which == 0) {
        uint32_t w[4];
        gd_philox4x32_10(ctr.x, ctr.y, ctr.z, ctr.w, key.x, key.y, w);
        out[0] = w[0]; out[1] = w[1]; out[2] = w[2]; out[3] = w[3];
    } else {
        uint4 r = curand_Philox4x32_10(ctr, key);
        out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
    }
}

extern "C" int gadep_philox_raw(gadep_ctx *c, const unsigned *ctr4, const unsigned *key2, int which, unsigned *out4) {
    if (!c) return GADEP_E_NULL;
    if (!ctr4 || !key2 || !out4) return gd_fail(c, GADEP_E_NULL, "null array");
    GD_CUDA(c, cudaSetDevice(c->device));
    unsigned *d = nullptr;
    GD_CUDA(c, cudaMalloc(&d, 16));
    gd_k_philox<<<1, 1, 0, c->stream>>>(make_uint4(ctr4[0], ctr4[1], ctr4[2], ctr4[3]), make_uint2(key2[0], key2[1]), which, d);
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess) e = cudaMemcpy(out4, d, 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return gd_fail(c, GADEP_E_CUDA, "philox kernel failed: %s", cudaGetErrorString(e));
    return GADEP_OK;
}

// ---------------------------------------------------------------- traversal width, whole-tally exchange
extern "C" int gadep_set_bvh_width(gadep_ctx *c, int width) {
    if (!c) return GADEP_E_NULL;
    if (width != 4 && width != 8 && width != GD_WIDTH_4Q) return gd_fail(c, GADEP_E_ARG, "BVH width %d (4, 5 or 8)", width);
    c->bvh_width = width;
    c->width_set = true;
    return GADEP_OK;
}

extern "C" int gadep_tally_size(const gadep_ctx *c) {
    if (!c) return GADEP_E_NULL;
    return c->n_bins > 0 ? c->n_bins + 1 + 2 * GADEP_MAX_LINES : 0;
}

extern "C" int gadep_get_tallies(gadep_ctx *c, unsigned long long *out) {
    if (!c) return GADEP_E_NULL;
    if (!out) return gd_fail(c, GADEP_E_NULL, "null output");
    if (!c->have_results || !c->d_tally) return gd_fail(c, GADEP_E_ORDER, "no run yet");
    GD_CUDA(c, cudaSetDevice(c->device));
    const size_t bytes = sizeof(unsigned long long) * ((size_t)c->n_bins + 1 + 2 * GADEP_MAX_LINES);
    const bool dev = gd_is_device_ptr(out);
    GD_CUDA(c, cudaMemcpyAsync(out, c->d_tally, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!dev) GD_CUDA(c, cudaStreamSynchronize(c->stream));
    return GADEP_OK;
}

extern "C" int gadep_set_tallies(gadep_ctx *c, const unsigned long long *in) {
    if (!c) return GADEP_E_NULL;
    if (!in) return gd_fail(c, GADEP_E_NULL, "null input");
    if (!c->have_results || !c->d_tally) return gd_fail(c, GADEP_E_ORDER, "no run yet");
    GD_CUDA(c, cudaSetDevice(c->device));
    const size_t bytes = sizeof(unsigned long long) * ((size_t)c->n_bins + 1 + 2 * GADEP_MAX_LINES);
    GD_CUDA(c, cudaMemcpyAsync(c->d_tally, in, bytes, gd_is_device_ptr(in) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    c->results_stale = true;
    return GADEP_OK;
}

// ---------------------------------------------------------------- ray cast without any allocation
// gadep_trace_rays_static (include/gadep.h): gd_k_trace_wave with all of its scratch in one file-scope device array.
//   [0, 256)     ray-fetch counter of the kernel (unsigned long long), must start at zero
//   [256, 512)   GdCounters of the launch, must start at zero
//   [512, ...)   staging for HOST arrays: org float[n][3], dir float[n][3], tri int[n], t float[n] (32 B per ray)
// In host code `gd_static_scratch` names a host-side stand-in, not device memory: the device address comes from
// cudaGetSymbolAddress, once per device with that device current, and that pointer is what the kernel is given.
#define GD_STATIC_HDR 512
static_assert(sizeof(GdCounters) <= 256, "GdCounters must fit its 256-byte cell");
static __device__ __align__(256) unsigned char gd_static_scratch[GD_STATIC_HDR + 32ull * GADEP_STATIC_MAX_RAYS];
#define GD_STATIC_MAX_DEVICES 64
static unsigned char *gd_static_addr[GD_STATIC_MAX_DEVICES] = {};

// device address of the array on `device` (which the caller has made current); resolved on the first call per device
static cudaError_t gd_static_scratch_on(int device, unsigned char **out) {
    if (device < 0 || device >= GD_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    unsigned char *p = __atomic_load_n(&gd_static_addr[device], __ATOMIC_ACQUIRE);
    if (!p) {
        void *sym = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&sym, gd_static_scratch);
        if (e != cudaSuccess) return e;
        if (!sym) return cudaErrorInvalidSymbol;
        p = (unsigned char *)sym;
        __atomic_store_n(&gd_static_addr[device], p, __ATOMIC_RELEASE);    // every thread resolves the same address
    }
    *out = p;
    return cudaSuccess;
}

extern "C" int gadep_trace_rays_static(gadep_ctx *c, const float *org, const float *dir, long long n_rays,
                                       int filter_material, float t_min, int *tri_out, float *t_out) {
    if (!c) return GADEP_E_NULL;
    if (!org || !dir || !tri_out || !t_out) return gd_fail(c, GADEP_E_NULL, "null ray array");
    if (!c->have_bvh) return gd_fail(c, GADEP_E_ORDER, "gadep_trace_rays_static before gadep_build_bvh");
    if (n_rays < 0) return gd_fail(c, GADEP_E_ARG, "negative ray count");
    if (n_rays > (long long)GADEP_STATIC_MAX_RAYS)
        return gd_fail(c, GADEP_E_ARG, "n_rays %lld exceeds GADEP_STATIC_MAX_RAYS (%d): the static scratch array holds no more; "
                       "split the batch or use gadep_trace_rays", n_rays, (int)GADEP_STATIC_MAX_RAYS);
    if (n_rays == 0) return GADEP_OK;
    GD_CUDA(c, cudaSetDevice(c->device));
    const bool dev = gd_is_device_ptr(org);
    if (dev != gd_is_device_ptr(dir) || dev != gd_is_device_ptr(tri_out) || dev != gd_is_device_ptr(t_out))
        return gd_fail(c, GADEP_E_ARG, "ray arrays must live in one memory space");
    unsigned char *scratch = nullptr;
    GD_CUDA(c, gd_static_scratch_on(c->device, &scratch));
    unsigned long long *d_next = (unsigned long long *)scratch;
    GdCounters *d_cnt = (GdCounters *)(scratch + 256);
    float *stage = (float *)(scratch + GD_STATIC_HDR);
    cudaStream_t st = c->stream;
    const float *d_org = org, *d_dir = dir;
    int *d_tri = tri_out;
    float *d_t = t_out;
    const size_t nb3 = sizeof(float) * 3 * (size_t)n_rays, nb1 = sizeof(float) * (size_t)n_rays;
    if (!dev) {
        d_org = stage; d_dir = stage + 3 * n_rays; d_tri = (int *)(stage + 6 * n_rays); d_t = stage + 7 * n_rays;
        GD_CUDA(c, cudaMemcpyAsync(stage, org, nb3, cudaMemcpyHostToDevice, st));
        GD_CUDA(c, cudaMemcpyAsync(stage + 3 * n_rays, dir, nb3, cudaMemcpyHostToDevice, st));
    }
    GD_CUDA(c, cudaMemsetAsync(scratch, 0, GD_STATIC_HDR, st));       // the last call's counter and totals are still there
    int per_sm = 1;
    const bool wide8 = c->bvh_width == 8, q4 = c->bvh_width == GD_WIDTH_4Q || (!c->width_set && gd_large_hierarchy(c));
    GD_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, wide8 ? gd_k_trace_wave<8> : (q4 ? gd_k_trace_wave<GD_WIDTH_4Q> : gd_k_trace_wave<4>), 256, 0));
    const int grid = (int)std::min<long long>((n_rays + 255) / 256, (long long)c->n_sm * std::max(per_sm, 1));
    const unsigned chunk = (unsigned)std::min<long long>(2048, std::max<long long>(32, n_rays / ((long long)grid * 8 * 8)));
    cudaEventRecord(c->ev0, st);
    if (wide8) gd_k_trace_wave<8><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                         d_cnt, d_next, chunk, c->tune);
    else if (q4) gd_k_trace_wave<GD_WIDTH_4Q><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                                   d_cnt, d_next, chunk, c->tune);
    else gd_k_trace_wave<4><<<grid, 256, 0, st>>>(gd_bvh_view(c), d_org, d_dir, n_rays, filter_material, t_min, d_tri, d_t,
                                                   d_cnt, d_next, chunk, c->tune);
    cudaEventRecord(c->ev1, st);
    c->last_run_launches = 1;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && !dev) {
        e = cudaMemcpyAsync(tri_out, d_tri, nb1, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(t_out, d_t, nb1, cudaMemcpyDeviceToHost, st);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpy(&c->h_counters, d_cnt, sizeof(GdCounters), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return gd_fail(c, GADEP_E_CUDA, "static trace failed: %s", cudaGetErrorString(e));
    cudaEventElapsedTime(&c->last_run_ms, c->ev0, c->ev1);
    c->run_timed = false;
    return GADEP_OK;
}

#ifdef GD_PROF
extern "C" int gadep_prof_read(unsigned long long *out16, int reset) {
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out16, gd_prof, sizeof(unsigned long long) * 16);
    if (reset) { unsigned long long z[16] = {}; cudaMemcpyToSymbol(gd_prof, z, sizeof(z)); }
    return 0;
}
#endif
