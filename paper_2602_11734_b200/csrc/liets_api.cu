// liets_api.cu -- the C ABI of libliets.so (include/liets.h).  Argument checking, workspace
// layout, launch sequencing and read-back only: every step of the path runs in the kernels.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/liets.h"
#include "liets_host.h"

using namespace liets;

namespace {

constexpr size_t kAlign = 256;
constexpr uint64_t kSmallGrid = 1ull << 22;     // grids up to this many voxels can finish on the voxel list (its capacity is 2^18 entries)
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t ctl, grid, list0, list1, status2, coff, rowoff, cand, pbits, prow, total;
    size_t g0, g1, stamp, weight;  // STORAGE_TILE (contiguous: G0 | G1 | stamp | weight)
    size_t vox0, vox1, vox_cap;    // STORAGE_TILE: front voxel lists of the small-front steps
    size_t n_tiles, grid_words, list_cap;
    int Wp, ntx, nty, ntz;
};

bool make_layout(int nx, int ny, int nz, int storage, Layout* L) {
    if (nx < 1 || ny < 1 || nz < 1) return false;
    const unsigned long long N = (unsigned long long)nx * (unsigned long long)ny * (unsigned long long)nz;
    if (N >= (1ull << 32)) return false;
    if (storage != LIETS_STORAGE_U8 && storage != LIETS_STORAGE_TILE && storage != LIETS_STORAGE_FULL) return false;
    memset(L, 0, sizeof(*L));
    size_t off = 0;
    L->ctl = off;     off += align_up(sizeof(Control));
    if (storage == LIETS_STORAGE_U8) {
        L->grid = off;    off += align_up((size_t)N + 4);
        L->list_cap = (size_t)N;
    } else {
        L->Wp = (nx + 63) / 64;
        L->ntx = (L->Wp + grow_tile_words() - 1) / grow_tile_words();
        L->nty = (ny + 7) / 8;
        L->ntz = (nz + 7) / 8;
        L->n_tiles = (size_t)L->ntx * L->nty * L->ntz;
        L->grid_words = (size_t)L->Wp * ny * nz;
        L->g0 = off;      off += L->grid_words * 8;
        L->g1 = off;      off += L->grid_words * 8;
        L->stamp = off;   off += L->n_tiles * 4;                // (memset together with G0 | G1 and the weights)
        L->weight = off;  off = align_up(off + L->n_tiles * 4);
        L->list_cap = L->n_tiles;                           // the step stamp admits every tile at most once per list
        L->vox_cap = (size_t)N / 16 < ((size_t)1 << 18) ? ((size_t)1 << 18) : (size_t)N / 16;    // N/16, at least 2^18 entries (1 MiB)
        L->vox0 = off;    off += align_up(L->vox_cap * 4);
        L->vox1 = off;    off += align_up(L->vox_cap * 4);
    }
    L->list0 = off;   off += align_up(L->list_cap * 4);
    L->list1 = off;   off += align_up(L->list_cap * 4);
    L->status2 = off; off += align_up(((size_t)N + 15) / 16 * 4);
    L->coff = off;    off += align_up((((size_t)N + 15) / 16 + 31) / 32 * 32 / 8 * 4 + 64);
    L->rowoff = off;  off += align_up(((size_t)ny * nz + 2) * 4);
    L->cand = off;    off += align_up((size_t)N * 4 < 64 ? 64 : (size_t)N * 4);
    L->pbits = off;   off += align_up(((size_t)N + 7) / 8 + 8);             // liets_set_blocked: N/8 bytes, and the same in row layout
    L->prow = off;    off += align_up(L->grid_words * 8);
    L->total = off;
    return true;
}

// Steps that start with more front voxels than this run on tiles (measured cross-over on B200: one thread per voxel
// with scattered row loads beats the tile kernel's fixed per-tile work up to about one front voxel per 128 cells, and on
// small grids, whose few tiles cannot fill the GPU, up to about 10^5 front voxels).
uint32_t default_vox_threshold(uint64_t N, uint32_t vox_cap) {
    const uint64_t thr = N / 128 < ((uint64_t)1 << 17) ? ((uint64_t)1 << 17) : N / 128;
    return (uint32_t)(thr < vox_cap / 2 ? thr : vox_cap / 2);
}

int fail(liets_ctx* c, int code, const char* msg) {
    if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
    return code;
}

// prob in [0,1] -> floor(p 2^32 + 0.5) in [0, 2^32] (R8)
uint64_t prob_to_threshold(double p) {
    if (p <= 0.0) return 0;
    if (p >= 1.0) return 1ull << 32;
    return (uint64_t)std::floor(p * 4294967296.0 + 0.5);
}

int readback(liets_ctx* c) {
    LIETS_CUDA_TRY(c, cudaMemcpyAsync(c->pinned, c->ctl, kControlScalarBytes, cudaMemcpyDeviceToHost, c->stream));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return 0;
}

int launch_step_kernel(liets_ctx* c) {
    const bool prof = c->profiling && c->prof_n < kProfCap;
    if (c->storage == LIETS_STORAGE_TILE) {                 // exactly one of the two growth kernels acts (Control::mode, pending)
        LIETS_CUDA_TRY(c, launch_tiles_from_grid(c));
        LIETS_CUDA_TRY(c, launch_grow_vox(c));
    }
    if (prof) {                                             // the event pair brackets the dominant kernel (k_grow_tile / k_grow_u8) alone
        if (!c->prof_ev) {
            c->prof_ev = static_cast<cudaEvent_t*>(calloc(2 * kProfCap, sizeof(cudaEvent_t)));
            if (!c->prof_ev) return fail(c, LIETS_E_CUDA, "out of host memory");
        }
        for (int k = 0; k < 2; ++k)
            if (!c->prof_ev[2 * c->prof_n + k]) LIETS_CUDA_TRY(c, cudaEventCreate(&c->prof_ev[2 * c->prof_n + k]));
        LIETS_CUDA_TRY(c, cudaEventRecord(c->prof_ev[2 * c->prof_n], c->stream));
    }
    LIETS_CUDA_TRY(c, c->storage == LIETS_STORAGE_U8 ? launch_grow_u8(c) : c->storage == LIETS_STORAGE_FULL ? launch_grow_full(c) : launch_grow_tile(c));
    if (prof) {
        LIETS_CUDA_TRY(c, cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], c->stream));
        c->prof_n++;
    }
    return 0;
}

// One WHILE node over { growth kernel ; control step }: adds the node to g after `after` (or at the root).
bool add_loop(liets_ctx* c, cudaGraph_t g, const cudaGraphNode_t* after, int which, cudaGraphNode_t* while_node,
              cudaGraphNode_t* grow_node) {
    cudaGraphConditionalHandle loop;
    if (cudaGraphConditionalHandleCreate(&loop, g, 1u, cudaGraphCondAssignDefault) != cudaSuccess) return false;
    cudaGraphNodeParams wp = {};
    wp.type = cudaGraphNodeTypeConditional;
    wp.conditional.handle = loop;
    wp.conditional.type = cudaGraphCondTypeWhile;
    wp.conditional.size = 1;
    if (cudaGraphAddNode(while_node, g, after, after ? 1 : 0, &wp) != cudaSuccess) return false;
    cudaGraph_t body = wp.conditional.phGraph_out[0];
    cudaGraphNode_t ctl_node;
    const cudaError_t e = which == 0 ? grow_u8_node(c, body, nullptr, grow_node)
                        : which == 1 ? grow_full_node(c, body, nullptr, grow_node)
                                     : grow_tile_node(c, body, nullptr, grow_node);
    return e == cudaSuccess && control_loop_node(c, body, *grow_node, loop, &ctl_node) == cudaSuccess;
}

bool ensure_loop_graph(liets_ctx* c) {
    if (c->loop_exec) {
        const bool inter = c->interact && c->has_blocked;
        if (c->loop_seed == c->rng_seed && c->loop_blocked == c->has_blocked && c->loop_interact == inter) return true;
        cudaError_t e = c->storage == LIETS_STORAGE_U8 ? grow_u8_node(c, nullptr, c->loop_exec, &c->loop_grow_node)
                      : c->storage == LIETS_STORAGE_FULL ? grow_full_node(c, nullptr, c->loop_exec, &c->loop_grow_node)
                                                         : grow_tile_node(c, nullptr, c->loop_exec, &c->loop_grow_node);
        if (e == cudaSuccess) { c->loop_seed = c->rng_seed; c->loop_blocked = c->has_blocked; c->loop_interact = inter; return true; }
        cudaGetLastError();
        cudaGraphExecDestroy(c->loop_exec); cudaGraphDestroy(c->loop_graph);        // rebuild below
        c->loop_exec = nullptr; c->loop_graph = nullptr; c->loop_tried = false;
    }
    if (c->loop_tried) return false;
    c->loop_tried = true;
    cudaGraph_t g = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t while1, grow_node, switch_node;
    bool ok = cudaGraphCreate(&g, 0) == cudaSuccess;
    if (ok && c->storage != LIETS_STORAGE_TILE) {
        ok = add_loop(c, g, nullptr, c->storage == LIETS_STORAGE_U8 ? 0 : 1, &while1, &grow_node);
    } else if (ok) {
        // STORAGE_TILE (after the steps on the voxel list, k_grow_vox_loop): k_tiles_from_grid -> WHILE(tiles) { k_grow_tile ; control }
        ok = tiles_from_grid_node(c, g, nullptr, &switch_node) == cudaSuccess &&
             add_loop(c, g, &switch_node, 2, &while1, &grow_node);
    }
    ok = ok && cudaGraphInstantiate(&exec, g, 0) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        if (g) cudaGraphDestroy(g);
        return false;
    }
    c->loop_graph = g; c->loop_exec = exec; c->loop_grow_node = grow_node; c->loop_seed = c->rng_seed; c->loop_blocked = c->has_blocked; c->loop_interact = c->interact && c->has_blocked;
    return true;
}

}  // namespace

extern "C" {

size_t liets_workspace_bytes(int nx, int ny, int nz, int storage) {
    Layout L;
    return make_layout(nx, ny, nz, storage, &L) ? L.total : 0;
}

int liets_create(liets_ctx** out, int nx, int ny, int nz, int boundary, int storage, void* workspace,
                 size_t workspace_bytes, void* cuda_stream) {
    if (!out) return LIETS_E_ARG;
    *out = nullptr;
    Layout L;
    if (!make_layout(nx, ny, nz, storage, &L)) return LIETS_E_ARG;
    if (boundary != LIETS_BOUNDARY_WALL && boundary != LIETS_BOUNDARY_PERIODIC && boundary != LIETS_BOUNDARY_PERIODIC_XY) return LIETS_E_ARG;
    if (workspace && workspace_bytes < L.total) return LIETS_E_CAPACITY;
    if (workspace && (reinterpret_cast<uintptr_t>(workspace) % kAlign)) return LIETS_E_ARG;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) return LIETS_E_CUDA;   // no CPU fallback

    liets_ctx* c = new (std::nothrow) liets_ctx();
    if (!c) return LIETS_E_CUDA;
    memset(c, 0, sizeof(*c));
    c->nx = nx; c->ny = ny; c->nz = nz; c->boundary = boundary; c->storage = storage;
    c->periodic = boundary == LIETS_BOUNDARY_PERIODIC ? 7 : boundary == LIETS_BOUNDARY_PERIODIC_XY ? 3 : 0;
    c->N = (uint64_t)nx * (uint64_t)ny * (uint64_t)nz;
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    c->law = LIETS_LAW_EQ1;
    int dev = 0;
    bool ok = cudaGetDevice(&dev) == cudaSuccess &&
              cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess;
    if (ok && !workspace) {
        ok = cudaMalloc(&c->ws, L.total) == cudaSuccess;
        c->owns_ws = ok;
    } else {
        c->ws = workspace;
    }
    c->ws_bytes = L.total;
    ok = ok && cudaMallocHost(reinterpret_cast<void**>(&c->pinned), sizeof(Control)) == cudaSuccess;
    ok = ok && cudaEventCreate(&c->ev0) == cudaSuccess && cudaEventCreate(&c->ev1) == cudaSuccess;
    if (ok) {
        char* base = static_cast<char*>(c->ws);
        c->ctl = reinterpret_cast<Control*>(base + L.ctl);
        c->grid_u8 = reinterpret_cast<uint8_t*>(base + L.grid);
        c->list[0] = reinterpret_cast<uint32_t*>(base + L.list0);
        c->list[1] = reinterpret_cast<uint32_t*>(base + L.list1);
        c->status2 = reinterpret_cast<uint32_t*>(base + L.status2);
        c->cand = reinterpret_cast<uint32_t*>(base + L.cand);
        c->coff = reinterpret_cast<uint32_t*>(base + L.coff);
        c->rowoff = reinterpret_cast<uint32_t*>(base + L.rowoff);
        c->explicit_idx = reinterpret_cast<uint64_t*>(base + L.cand);
        c->scratch_u8 = reinterpret_cast<uint8_t*>(base + L.cand);
        c->pbits = reinterpret_cast<uint8_t*>(base + L.pbits);
        c->prow = reinterpret_cast<unsigned long long*>(base + L.prow);
        c->list_cap = L.list_cap;
        if (storage != LIETS_STORAGE_U8) {
            c->geom = TileGeom{ nx, ny, nz, L.Wp, L.ntx, L.nty, L.ntz, c->periodic };
            c->n_tiles = L.n_tiles;
            c->grid_words = L.grid_words;
            c->G[0] = reinterpret_cast<unsigned long long*>(base + L.g0);
            c->G[1] = reinterpret_cast<unsigned long long*>(base + L.g1);
            c->stamp = reinterpret_cast<uint32_t*>(base + L.stamp);
            c->weight = reinterpret_cast<uint32_t*>(base + L.weight);
            c->vox[0] = reinterpret_cast<uint32_t*>(base + L.vox0);
            c->vox[1] = reinterpret_cast<uint32_t*>(base + L.vox1);
            c->vox_cap = c->vox_cap_alloc = (uint32_t)L.vox_cap;
            c->vox_thr = default_vox_threshold(c->N, c->vox_cap);
            int coop = 0;                                   // the voxel-list loop is a cooperative launch: without it, tiles from step 0
            if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) { cudaGetLastError(); c->vox_thr = 0; c->no_coop = true; }
            c->grid_u8 = nullptr;
            c->tile_grid = c->sm_count * grow_tile_ctas_per_sm();
        }
        // function attributes are per device: set them for the device of this context (cheap, idempotent)
        ok = seed_kernel_attributes() == cudaSuccess && grow_tile_attributes() == cudaSuccess &&
             cudaMemsetAsync(c->ctl, 0, sizeof(Control), c->stream) == cudaSuccess &&
             launch_set_params(c) == cudaSuccess;
    }
    if (!ok) {
        cudaGetLastError();
        liets_destroy(c);
        return LIETS_E_CUDA;
    }
    *out = c;
    return LIETS_OK;
}

void liets_destroy(liets_ctx* c) {
    if (!c) return;
    if (c->stream || c->ws) cudaStreamSynchronize(c->stream);
    if (c->owns_ws && c->ws) cudaFree(c->ws);
    if (c->pinned) cudaFreeHost(c->pinned);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->loop_exec) cudaGraphExecDestroy(c->loop_exec);
    if (c->loop_graph) cudaGraphDestroy(c->loop_graph);
    if (c->prof_ev) {
        for (uint32_t k = 0; k < 2 * kProfCap; ++k)
            if (c->prof_ev[k]) cudaEventDestroy(c->prof_ev[k]);
        free(c->prof_ev);
    }
    delete c;
}

const char* liets_last_error(const liets_ctx* c) { return c ? c->err : "null ctx"; }

int liets_set_growth(liets_ctx* c, double g_face, double g_edge, double g_corner, int law) {
    if (!c) return LIETS_E_ARG;
    const double g[3] = { g_face, g_edge, g_corner };
    for (double v : g)
        if (!(v >= 0.0 && v <= 1.0)) return fail(c, LIETS_E_ARG, "growth probability outside [0,1]");
    if (law != LIETS_LAW_CONSTANT && law != LIETS_LAW_EQ1) return fail(c, LIETS_E_ARG, "unknown law");
    for (int k = 0; k < 3; ++k) c->R[k] = prob_to_threshold(g[k]);
    c->law = law;
    c->growth_set = true;
    LIETS_CUDA_TRY(c, launch_set_params(c));
    return LIETS_OK;
}

int liets_set_blocked(liets_ctx* c, const void* mask, size_t mask_bytes, int format, int mask_is_device) {
    if (!c) return LIETS_E_ARG;
    c->seeded = false;                                      // takes effect at the next seeding
    if (!mask) {
        c->has_blocked = false;
        c->n_blocked = 0;
        LIETS_CUDA_TRY(c, launch_set_params(c));
        return LIETS_OK;
    }
    if (format != LIETS_FORMAT_U8 && format != LIETS_FORMAT_BITS) return fail(c, LIETS_E_ARG, "unknown mask format");
    const size_t nb = format == LIETS_FORMAT_U8 ? (size_t)c->N : (size_t)((c->N + 7) / 8);
    if (mask_bytes < nb) return fail(c, LIETS_E_CAPACITY, "mask buffer too small for the format");
    const uint8_t* src = static_cast<const uint8_t*>(mask);
    unsigned long long* count_dev = reinterpret_cast<unsigned long long*>(c->status2);       // seeding scratch is idle here
    LIETS_CUDA_TRY(c, cudaMemsetAsync(count_dev, 0, 8, c->stream));
    if (!mask_is_device) {                                  // stage in the seeding scratch (4 N bytes)
        LIETS_CUDA_TRY(c, cudaMemcpyAsync(c->scratch_u8, mask, nb, cudaMemcpyHostToDevice, c->stream));
        src = c->scratch_u8;
    }
    LIETS_CUDA_TRY(c, launch_blocked_set(c, src, format, count_dev));
    unsigned long long n = 0;
    LIETS_CUDA_TRY(c, cudaMemcpyAsync(&n, count_dev, 8, cudaMemcpyDeviceToHost, c->stream));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->has_blocked = true;
    c->n_blocked = n;
    LIETS_CUDA_TRY(c, launch_set_params(c));
    return LIETS_OK;
}

int liets_set_target(liets_ctx* c, double phi) {
    if (!c) return LIETS_E_ARG;
    if (!(phi > 0.0 && phi <= 1.0)) return fail(c, LIETS_E_ARG, "target solid fraction outside (0,1]");
    double x = std::ceil(phi * (double)c->N);               // R7: one IEEE multiply, then ceil
    uint64_t n_t = x < 1.0 ? 1 : (x > (double)c->N ? c->N : (uint64_t)x);
    c->n_t = n_t;
    c->has_target = true;
    LIETS_CUDA_TRY(c, launch_set_params(c));
    return LIETS_OK;
}

int liets_seed(liets_ctx* c, double core_prob, int spacing_s, uint64_t rng_seed, uint64_t* n_seeds_out) {
    if (!c) return LIETS_E_ARG;
    if (!(core_prob >= 0.0 && core_prob <= 1.0)) return fail(c, LIETS_E_ARG, "core probability outside [0,1]");
    if (spacing_s < 0) return fail(c, LIETS_E_ARG, "negative seed spacing");
    c->rng_seed = rng_seed;
    LIETS_CUDA_TRY(c, cudaEventRecord(c->ev0, c->stream));
    LIETS_CUDA_TRY(c, launch_seed_reset(c));
    const int accept_all = spacing_s <= 1;
    LIETS_CUDA_TRY(c, launch_seed_candidates(c, prob_to_threshold(core_prob), accept_all));
    if (!accept_all) {
        if (c->spacing_method == LIETS_SPACING_DENSE) {     // the bit rows go behind the candidate list: its length first
            if (int rc = readback(c)) return rc;
            const uint32_t n_cand = c->pinned->n_cand;
            const size_t need = (((size_t)n_cand * 4u + 255u) & ~(size_t)255u) + 8u * spacing_dense_bytes(c);
            if (need > (size_t)c->N * 4u) return fail(c, LIETS_E_CAPACITY, "dense spacing: the bit rows do not fit the seeding scratch (4 N bytes)");
            LIETS_CUDA_TRY(c, launch_spacing_dense(c, spacing_s, n_cand, nullptr));
        } else if (c->spacing_order == LIETS_ORDER_KEYED) {
            LIETS_CUDA_TRY(c, launch_spacing_keyed(c, spacing_s));
        } else {
            LIETS_CUDA_TRY(c, launch_spacing(c, spacing_s));
        }
    }
    LIETS_CUDA_TRY(c, launch_seed_finalize(c, !accept_all));
    LIETS_CUDA_TRY(c, cudaEventRecord(c->ev1, c->stream));
    if (int rc = readback(c)) return rc;
    LIETS_CUDA_TRY(c, cudaEventElapsedTime(&c->seed_ms, c->ev0, c->ev1));
    c->seeded = true;
    if (n_seeds_out) *n_seeds_out = c->pinned->n_solid;
    return LIETS_OK;
}

int liets_set_interaction(liets_ctx* c, double i_face, double i_edge, double i_corner) {
    if (!c) return LIETS_E_ARG;
    const double I[3] = { i_face, i_edge, i_corner };
    for (int k = 0; k < 3; ++k)
        if (!(I[k] >= 0.0 && I[k] <= 1.0)) return fail(c, LIETS_E_ARG, "interaction probability outside [0,1]");
    const bool on = I[0] > 0.0 || I[1] > 0.0 || I[2] > 0.0;
    if (on && c->storage == LIETS_STORAGE_U8) return fail(c, LIETS_E_ARG, "phase interaction needs a bit-row storage (LIETS_STORAGE_TILE or _FULL)");
    for (int k = 0; k < 3; ++k) c->RI[k] = prob_to_threshold(I[k]);
    c->interact = (c->RI[0] | c->RI[1] | c->RI[2]) != 0;
    LIETS_CUDA_TRY(c, launch_set_interaction(c));
    c->seeded = false;                                      // the sources change: seed again
    return LIETS_OK;
}

int liets_set_spacing(liets_ctx* c, int order, int method) {
    if (!c) return LIETS_E_ARG;
    if ((order != LIETS_ORDER_INDEX && order != LIETS_ORDER_KEYED) || (method != LIETS_SPACING_SPARSE && method != LIETS_SPACING_DENSE))
        return fail(c, LIETS_E_ARG, "unknown spacing order or method");
    if (method == LIETS_SPACING_DENSE && order != LIETS_ORDER_INDEX)
        return fail(c, LIETS_E_ARG, "the dense dilation works in ascending index order only");
    if (method == LIETS_SPACING_DENSE && c->periodic)
        return fail(c, LIETS_E_ARG, "the dense dilation is built for LIETS_BOUNDARY_WALL only");
    c->spacing_order = order;
    c->spacing_method = method;
    return LIETS_OK;
}

int liets_seed_explicit(liets_ctx* c, const uint64_t* idx, uint64_t n, uint64_t rng_seed) {
    if (!c || (n && !idx)) return LIETS_E_ARG;
    // the staging buffer is the 4 N-byte candidate region: at most N/2 (>= 8) indices; n is compared, not n * 8
    if (n > (c->N * 4 < 64 ? 64 : c->N * 4) / 8) return fail(c, LIETS_E_CAPACITY, "too many explicit seeds for the staging buffer (max N/2)");
    for (uint64_t i = 0; i < n; ++i)
        if (idx[i] >= c->N) return fail(c, LIETS_E_ARG, "seed index outside the grid");
    c->rng_seed = rng_seed;
    LIETS_CUDA_TRY(c, launch_seed_reset(c));
    if (n) LIETS_CUDA_TRY(c, cudaMemcpyAsync(c->explicit_idx, idx, n * 8, cudaMemcpyHostToDevice, c->stream));
    LIETS_CUDA_TRY(c, launch_seed_explicit(c, n));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));    // idx may be pageable: do not outlive the call
    c->seeded = true;
    return LIETS_OK;
}

int liets_step(liets_ctx* c, uint64_t* n_solid_out, uint64_t* n_front_out) {
    if (!c) return LIETS_E_ARG;
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_step before liets_seed");
    if (c->law == LIETS_LAW_EQ1 && !c->has_target) return fail(c, LIETS_E_STATE, "Eq. (1) law needs a target");
    c->prof_n = 0;
    LIETS_CUDA_TRY(c, launch_begin(c, 0, 0));
    LIETS_CUDA_TRY(c, launch_control(c, kCtlPrepare | kCtlForce));
    if (int rc = launch_step_kernel(c)) return rc;
    LIETS_CUDA_TRY(c, launch_control(c, kCtlFinish));
    if (n_solid_out || n_front_out) {
        if (int rc = readback(c)) return rc;
        const uint64_t ns = c->pinned->n_solid;
        if (n_solid_out) *n_solid_out = ns;
        const liets::Control* h = c->pinned;
        const uint64_t nf = h->mode == 2u ? 1u : (h->mode == 0u && !h->pending) ? h->vox_count[h->cur] : (uint64_t)h->count[h->cur] + h->count_back[h->cur];
        if (n_front_out) *n_front_out = (ns == 0 || ns == c->N - c->n_blocked) ? 0 : nf;
    }
    return LIETS_OK;
}

int liets_generate(liets_ctx* c, double phi, uint32_t max_steps, uint32_t* steps_out, uint64_t* n_solid_out) {
    if (!c) return LIETS_E_ARG;
    if (int rc = liets_set_target(c, phi)) return rc;
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_generate before liets_seed");
    LIETS_CUDA_TRY(c, cudaEventRecord(c->ev0, c->stream));
    LIETS_CUDA_TRY(c, launch_begin(c, 1, max_steps));
    c->prof_n = 0;
    uint32_t enqueued = 0;
    if (!c->profiling && ensure_loop_graph(c)) {
        // the whole loop on the device: first step prepared here, then WHILE(step armed) { grow ; control } as one graph
        LIETS_CUDA_TRY(c, launch_control(c, kCtlPrepare));
        bool done = false;
        if (c->storage == LIETS_STORAGE_TILE) {
            if (!c->no_coop) LIETS_CUDA_TRY(c, launch_grow_vox_loop(c));     // the steps on the voxel list, one launch
            if (c->N <= kSmallGrid) {                       // a small grid often ends on the voxel list: look before launching the graph
                if (int rc = readback(c)) return rc;
                done = c->pinned->status != kStatusRunning;
            }
        }
        if (!done) {
            LIETS_CUDA_TRY(c, cudaGraphLaunch(c->loop_exec, c->stream));
            if (int rc = readback(c)) return rc;
        }
        c->launches += 2ull * c->pinned->steps_done + (c->storage == LIETS_STORAGE_TILE ? 3 : 2);   // kernels the graph ran (incl. the loop's last, empty round)
    } else for (;;) {
        // a batch of steps back to back; steps after the stop rule fired are no-ops on the device
        uint32_t batch = 32;
        if (max_steps - enqueued < batch) batch = max_steps - enqueued;
        for (uint32_t k = 0; k < batch; ++k) {
            LIETS_CUDA_TRY(c, launch_control(c, k == 0 ? kCtlPrepare : (kCtlFinish | kCtlPrepare)));
            if (int rc = launch_step_kernel(c)) return rc;
        }
        enqueued += batch;
        LIETS_CUDA_TRY(c, launch_control(c, kCtlFinish | kCtlEval));
        if (int rc = readback(c)) return rc;
        if (c->pinned->status != kStatusRunning) break;
    }
    LIETS_CUDA_TRY(c, cudaEventRecord(c->ev1, c->stream));
    LIETS_CUDA_TRY(c, cudaEventSynchronize(c->ev1));
    LIETS_CUDA_TRY(c, cudaEventElapsedTime(&c->gen_ms, c->ev0, c->ev1));
    if (steps_out) *steps_out = c->pinned->steps_done;
    if (n_solid_out) *n_solid_out = c->pinned->n_solid;
    return c->pinned->status;
}

int liets_grid(liets_ctx* c, void* dst, size_t dst_bytes, int format, int dst_is_device) {
    if (!c || !dst) return LIETS_E_ARG;
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_grid before liets_seed");
    const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (format != LIETS_FORMAT_U8 && format != LIETS_FORMAT_BITS) return fail(c, LIETS_E_ARG, "unknown grid format");
    const size_t nb = format == LIETS_FORMAT_U8 ? (size_t)c->N : (size_t)((c->N + 7) / 8);
    if (dst_bytes < nb) return fail(c, LIETS_E_CAPACITY, "dst buffer too small for the requested format");
    const uint8_t* u8 = c->grid_u8;
    if (c->storage != LIETS_STORAGE_U8) {                   // bit rows -> linear uint8 (seeding scratch is idle)
        if (int rc = readback(c)) return rc;                // which grid copy is current
        c->host_step = c->pinned->step;
        if (format == LIETS_FORMAT_BITS && c->nx % 8 == 0) {
            // the x-rows are byte aligned: the packed output is the rows without their padding words
            if (dst_is_device) {
                LIETS_CUDA_TRY(c, launch_rows_to_bits(c, static_cast<uint8_t*>(dst)));
            } else {                                        // gather into the (idle) seeding scratch, then one copy
                LIETS_CUDA_TRY(c, launch_rows_to_bits(c, reinterpret_cast<uint8_t*>(c->status2)));
                LIETS_CUDA_TRY(c, cudaMemcpyAsync(dst, c->status2, nb, kind, c->stream));
                LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
            }
            return LIETS_OK;
        }
        uint8_t* lin = (format == LIETS_FORMAT_U8 && dst_is_device) ? static_cast<uint8_t*>(dst) : c->scratch_u8;
        LIETS_CUDA_TRY(c, launch_unpack_rows_u8(c, lin));
        u8 = lin;
    }
    if (format == LIETS_FORMAT_U8 && c->storage == LIETS_STORAGE_U8 && c->has_blocked) {      // bytes of value 2 are another phase's
        uint8_t* lin = dst_is_device ? static_cast<uint8_t*>(dst) : c->scratch_u8;
        LIETS_CUDA_TRY(c, launch_u8_this_phase(c, lin));
        if (lin != dst) LIETS_CUDA_TRY(c, cudaMemcpyAsync(dst, lin, c->N, kind, c->stream));
    } else if (format == LIETS_FORMAT_U8) {
        if (u8 != dst) LIETS_CUDA_TRY(c, cudaMemcpyAsync(dst, u8, c->N, kind, c->stream));
    } else if (format == LIETS_FORMAT_BITS) {
        if (dst_is_device) {
            LIETS_CUDA_TRY(c, launch_pack_bits_u8(c, u8, static_cast<uint8_t*>(dst)));
        } else {                                            // pack into the (idle) seeding scratch, then copy
            LIETS_CUDA_TRY(c, launch_pack_bits_u8(c, u8, reinterpret_cast<uint8_t*>(c->status2)));
            LIETS_CUDA_TRY(c, cudaMemcpyAsync(dst, c->status2, nb, kind, c->stream));
        }
    } else {
        return fail(c, LIETS_E_ARG, "unknown grid format");
    }
    if (!dst_is_device) LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return LIETS_OK;
}

int liets_s2(liets_ctx* c, int axis, int rmax, uint64_t* pairs, uint64_t* valid) {
    if (!c || !pairs || !valid) return LIETS_E_ARG;
    if (axis < 0 || axis > 2 || rmax < 0 || rmax > 65534) return fail(c, LIETS_E_ARG, "axis must be 0..2 and rmax 0..65534");
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_s2 before liets_seed");
    if (int rc = readback(c)) return rc;                    // which grid copy is current
    c->host_step = c->pinned->step;
    const size_t n_words = (size_t)((c->nx + 63) / 64) * c->ny * c->nz;
    const size_t bytes = (size_t)(rmax + 1) * 8 + (c->storage == LIETS_STORAGE_U8 ? n_words * 8 : 0);
    unsigned long long* dev = nullptr;
    if (cudaMalloc(&dev, bytes) != cudaSuccess) { cudaGetLastError(); return fail(c, LIETS_E_CUDA, "cudaMalloc failed in liets_s2"); }
    bool ok = cudaMemsetAsync(dev, 0, (size_t)(rmax + 1) * 8, c->stream) == cudaSuccess &&
              launch_s2(c, axis, rmax, dev, dev + rmax + 1) == cudaSuccess &&
              cudaMemcpyAsync(pairs, dev, (size_t)(rmax + 1) * 8, cudaMemcpyDeviceToHost, c->stream) == cudaSuccess &&
              cudaStreamSynchronize(c->stream) == cudaSuccess;
    cudaFree(dev);
    if (!ok) { cudaGetLastError(); return fail(c, LIETS_E_CUDA, "liets_s2 failed on the device"); }
    const uint64_t n[3] = { (uint64_t)c->nx, (uint64_t)c->ny, (uint64_t)c->nz };
    for (int r = 0; r <= rmax; ++r)                         // positions counted: all of them if periodic, else those with x + r inside
        valid[r] = ((c->periodic >> axis) & 1) ? c->N : ((uint64_t)r < n[axis] ? c->N / n[axis] * (n[axis] - (uint64_t)r) : 0);
    return LIETS_OK;
}

int liets_step_log(liets_ctx* c, uint64_t* front_in, uint64_t* solid_after, uint64_t* philox_blocks,
                   uint64_t* front_voxels, uint32_t cap) {
    if (!c) return LIETS_E_ARG;
    if (int rc = readback(c)) return rc;
    uint32_t n = c->pinned->step;
    if (n > kLogCap) n = kLogCap;
    if (n > cap) n = cap;
    if (n && front_in)
        LIETS_CUDA_TRY(c, cudaMemcpyAsync(front_in, c->ctl->log_front, n * 8ull, cudaMemcpyDeviceToHost, c->stream));
    if (n && solid_after)
        LIETS_CUDA_TRY(c, cudaMemcpyAsync(solid_after, c->ctl->log_solid, n * 8ull, cudaMemcpyDeviceToHost, c->stream));
    if (n && philox_blocks)
        LIETS_CUDA_TRY(c, cudaMemcpyAsync(philox_blocks, c->ctl->log_items, n * 8ull, cudaMemcpyDeviceToHost, c->stream));
    if (n && front_voxels)
        LIETS_CUDA_TRY(c, cudaMemcpyAsync(front_voxels, c->ctl->log_items0, n * 8ull, cudaMemcpyDeviceToHost, c->stream));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return (int)n;
}

int liets_timings(liets_ctx* c, float* seed_ms, float* generate_ms) {
    if (!c) return LIETS_E_ARG;
    if (seed_ms) *seed_ms = c->seed_ms;
    if (generate_ms) *generate_ms = c->gen_ms;
    return LIETS_OK;
}

int liets_set_profiling(liets_ctx* c, int on) {
    if (!c) return LIETS_E_ARG;
    c->profiling = on != 0;
    return LIETS_OK;
}

int liets_step_times(liets_ctx* c, float* ms, uint32_t cap) {
    if (!c || (cap && !ms)) return LIETS_E_ARG;
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    uint32_t n = c->prof_n < cap ? c->prof_n : cap;
    for (uint32_t k = 0; k < n; ++k)
        LIETS_CUDA_TRY(c, cudaEventElapsedTime(&ms[k], c->prof_ev[2 * k], c->prof_ev[2 * k + 1]));
    return (int)n;
}

uint64_t liets_launch_count(const liets_ctx* c) { return c ? c->launches : 0; }

int liets_seed_info(liets_ctx* c, uint32_t* n_candidates, uint32_t* slow_path) {
    if (!c) return LIETS_E_ARG;
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_seed_info before liets_seed");
    if (int rc = readback(c)) return rc;
    if (n_candidates) *n_candidates = c->pinned->n_cand;
    if (slow_path) *slow_path = c->pinned->spacing_slow;
    return LIETS_OK;
}

int liets_spacing_rounds(liets_ctx* c, uint32_t* rounds) {
    if (!c || !rounds) return LIETS_E_ARG;
    if (!c->seeded) return fail(c, LIETS_E_STATE, "liets_spacing_rounds before liets_seed");
    if (int rc = readback(c)) return rc;
    *rounds = c->pinned->spacing_rounds;
    return LIETS_OK;
}

// ---- batched realisations ---------------------------------------------------
int liets_create_batch(liets_batch** out, int n, int nx, int ny, int nz, int boundary, void* workspace, size_t workspace_bytes,
                       void* cuda_stream) {
    if (!out) return LIETS_E_ARG;
    *out = nullptr;
    if (n < 1 || n > grow_tile_max_batch()) return LIETS_E_ARG;
    const size_t each = liets_workspace_bytes(nx, ny, nz, LIETS_STORAGE_TILE);
    if (each == 0) return LIETS_E_ARG;
    if (workspace && workspace_bytes < each * (size_t)n) return LIETS_E_CAPACITY;
    liets_batch* b = new (std::nothrow) liets_batch();
    if (!b) return LIETS_E_CUDA;
    memset(b, 0, sizeof(*b));
    b->n = n;
    b->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int rc = LIETS_OK;
    for (int i = 0; i < n && rc == LIETS_OK; ++i)
        rc = liets_create(&b->ctx[i], nx, ny, nz, boundary, LIETS_STORAGE_TILE,
                          workspace ? static_cast<char*>(workspace) + each * (size_t)i : nullptr, workspace ? each : 0, cuda_stream);
    if (rc == LIETS_OK && (cudaEventCreate(&b->ev0) != cudaSuccess || cudaEventCreate(&b->ev1) != cudaSuccess)) rc = LIETS_E_CUDA;
    if (rc != LIETS_OK) { cudaGetLastError(); liets_destroy_batch(b); return rc; }
    *out = b;
    return LIETS_OK;
}

void liets_destroy_batch(liets_batch* b) {
    if (!b) return;
    cudaStreamSynchronize(b->stream);
    if (b->exec) cudaGraphExecDestroy(b->exec);
    if (b->graph) cudaGraphDestroy(b->graph);
    if (b->ev0) cudaEventDestroy(b->ev0);
    if (b->ev1) cudaEventDestroy(b->ev1);
    for (int i = 0; i < b->n; ++i) liets_destroy(b->ctx[i]);
    delete b;
}

liets_ctx* liets_batch_ctx(liets_batch* b, int i) { return (b && i >= 0 && i < b->n) ? b->ctx[i] : nullptr; }

const char* liets_batch_last_error(const liets_batch* b) { return b ? b->err : "null batch"; }

// WHILE(any grid live) { k_grow_tile over all grids ; one control step per grid }, built once, keys refreshed after re-seeding
static bool ensure_batch_graph(liets_batch* b) {
    bool same = b->exec != nullptr;
    for (int i = 0; i < b->n && same; ++i) same = b->graph_seed[i] == b->ctx[i]->rng_seed && b->graph_blocked[i] == b->ctx[i]->has_blocked;
    if (same) return true;
    if (b->exec) {
        if (grow_tile_batch_node(b->ctx, b->n, nullptr, b->exec, &b->grow_node) == cudaSuccess) {
            for (int i = 0; i < b->n; ++i) { b->graph_seed[i] = b->ctx[i]->rng_seed; b->graph_blocked[i] = b->ctx[i]->has_blocked; }
            return true;
        }
        cudaGetLastError();
        cudaGraphExecDestroy(b->exec); cudaGraphDestroy(b->graph);
        b->exec = nullptr; b->graph = nullptr;
    }
    cudaGraph_t g = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphConditionalHandle loop;
    cudaGraphNode_t while_node, grow_node, ctl_node;
    bool ok = cudaGraphCreate(&g, 0) == cudaSuccess &&
              cudaGraphConditionalHandleCreate(&loop, g, 1u, cudaGraphCondAssignDefault) == cudaSuccess;
    if (ok) {
        cudaGraphNodeParams wp = {};
        wp.type = cudaGraphNodeTypeConditional;
        wp.conditional.handle = loop;
        wp.conditional.type = cudaGraphCondTypeWhile;
        wp.conditional.size = 1;
        ok = cudaGraphAddNode(&while_node, g, nullptr, 0, &wp) == cudaSuccess;
        if (ok) {
            cudaGraph_t body = wp.conditional.phGraph_out[0];
            ok = grow_tile_batch_node(b->ctx, b->n, body, nullptr, &grow_node) == cudaSuccess &&
                 control_loop_batch_node(b->ctx, b->n, body, grow_node, loop, &ctl_node) == cudaSuccess &&
                 cudaGraphInstantiate(&exec, g, 0) == cudaSuccess;
        }
    }
    if (!ok) {
        cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        if (g) cudaGraphDestroy(g);
        return false;
    }
    b->graph = g; b->exec = exec; b->grow_node = grow_node;
    for (int i = 0; i < b->n; ++i) { b->graph_seed[i] = b->ctx[i]->rng_seed; b->graph_blocked[i] = b->ctx[i]->has_blocked; }
    return true;
}

#define LIETS_BATCH_TRY(b, expr)                                                                       \
    do {                                                                                               \
        cudaError_t e__ = (expr);                                                                      \
        if (e__ != cudaSuccess) {                                                                      \
            snprintf((b)->err, sizeof((b)->err), "%s:%d: %s: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
            return LIETS_E_CUDA;                                                                       \
        }                                                                                              \
    } while (0)

int liets_generate_batch(liets_batch* b, const double* target_solid_fraction, uint32_t max_steps, int* status_out,
                         uint32_t* steps_out, uint64_t* n_solid_out, float* device_ms_out) {
    if (!b || !target_solid_fraction) return LIETS_E_ARG;
    for (int i = 0; i < b->n; ++i) {
        liets_ctx* c = b->ctx[i];
        if (!(target_solid_fraction[i] > 0.0 && target_solid_fraction[i] <= 1.0)) { snprintf(b->err, sizeof(b->err), "target solid fraction of grid %d outside (0,1]", i); return LIETS_E_ARG; }
        if (!c->seeded) { snprintf(b->err, sizeof(b->err), "liets_generate_batch before liets_seed of grid %d", i); return LIETS_E_STATE; }
        if (c->interact && c->has_blocked) { snprintf(b->err, sizeof(b->err), "grid %d: phase interaction (liets_set_interaction) is not provided in batches", i); return LIETS_E_ARG; }
    }
    LIETS_BATCH_TRY(b, cudaEventRecord(b->ev0, b->stream));
    for (int i = 0; i < b->n; ++i) {
        liets_ctx* c = b->ctx[i];
        const uint32_t thr = c->vox_thr;
        c->vox_thr = 0;                                     // the batched loop runs on tiles from its first step
        int rc = liets_set_target(c, target_solid_fraction[i]);             // (also sends vox_thr to the device)
        c->vox_thr = thr;
        if (rc) { snprintf(b->err, sizeof(b->err), "grid %d: %.200s", i, c->err); return rc; }
        LIETS_BATCH_TRY(b, launch_begin(c, 1, max_steps));
        c->prof_n = 0;
        LIETS_BATCH_TRY(b, launch_control(c, kCtlPrepare));
        LIETS_BATCH_TRY(b, launch_tiles_from_grid(c));
    }
    if (!ensure_batch_graph(b)) { snprintf(b->err, sizeof(b->err), "the batch graph could not be built"); return LIETS_E_CUDA; }
    LIETS_BATCH_TRY(b, cudaGraphLaunch(b->exec, b->stream));
    for (int i = 0; i < b->n; ++i) LIETS_BATCH_TRY(b, launch_set_params(b->ctx[i]));      // the contexts' own thresholds again
    LIETS_BATCH_TRY(b, cudaEventRecord(b->ev1, b->stream));
    for (int i = 0; i < b->n; ++i) {
        liets_ctx* c = b->ctx[i];
        if (int rc = readback(c)) { snprintf(b->err, sizeof(b->err), "grid %d: %.200s", i, c->err); return rc; }
        c->launches += 1ull + c->pinned->steps_done;        // its share of the batched loop: one control step per step
        if (status_out) status_out[i] = c->pinned->status;
        if (steps_out) steps_out[i] = c->pinned->steps_done;
        if (n_solid_out) n_solid_out[i] = c->pinned->n_solid;
    }
    LIETS_BATCH_TRY(b, cudaEventSynchronize(b->ev1));
    LIETS_BATCH_TRY(b, cudaEventElapsedTime(&b->gen_ms, b->ev0, b->ev1));
    if (device_ms_out) *device_ms_out = b->gen_ms;
    return LIETS_OK;
}

int liets_debug_thresholds(const uint64_t* R, const uint64_t* n_t, const uint64_t* n_solid, uint64_t* T_out, uint32_t n) {
    if (!R || !n_t || !n_solid || !T_out || n == 0) return LIETS_E_ARG;
    for (uint32_t i = 0; i < n; ++i)
        if (n_t[i] == 0 || n_t[i] > (1ull << 32) || R[i] > (1ull << 32) || n_solid[i] > (1ull << 32)) return LIETS_E_ARG;
    unsigned long long* dev = nullptr;
    if (cudaMalloc(&dev, 4ull * n * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); return LIETS_E_CUDA; }
    bool ok = cudaMemcpy(dev, R, n * 8ull, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(dev + n, n_t, n * 8ull, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(dev + 2ull * n, n_solid, n * 8ull, cudaMemcpyHostToDevice) == cudaSuccess &&
              launch_eq1_thresholds(dev, dev + 3ull * n, n, nullptr) == cudaSuccess &&
              cudaMemcpy(T_out, dev + 3ull * n, n * 8ull, cudaMemcpyDeviceToHost) == cudaSuccess;
    cudaFree(dev);
    if (!ok) { cudaGetLastError(); return LIETS_E_CUDA; }
    return LIETS_OK;
}

int liets_debug_vox_list(liets_ctx* c, uint64_t max_front_voxels, uint32_t capacity) {
    if (!c) return LIETS_E_ARG;
    if (c->storage != LIETS_STORAGE_TILE) return LIETS_OK;
    c->vox_cap = capacity && capacity < c->vox_cap_alloc ? capacity : c->vox_cap_alloc;
    c->vox_thr = max_front_voxels == UINT64_MAX ? default_vox_threshold(c->N, c->vox_cap)
               : (uint32_t)(max_front_voxels > c->vox_cap ? c->vox_cap : max_front_voxels);
    if (c->no_coop) c->vox_thr = 0;
    LIETS_CUDA_TRY(c, launch_set_params(c));
    return LIETS_OK;
}

int liets_debug_spacing_ring(liets_ctx* c, uint32_t ring, uint32_t head) {
    if (!c) return LIETS_E_ARG;
    if (ring == 0) { c->spacing_ring = c->spacing_head = 0; return LIETS_OK; }
    if (ring < 2048u || (ring & (ring - 1u)) || ring > (1u << 17) || head > (1u << 16))
        return fail(c, LIETS_E_ARG, "ring must be a power of two in [2048, 2^17], head <= 2^16");
    c->spacing_ring = ring; c->spacing_head = head;
    return LIETS_OK;
}

}  // extern "C"
