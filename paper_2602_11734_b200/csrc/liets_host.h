// liets_host.h -- host-side context of libliets.so and the launchers each .cu file exports.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#include "liets_device.cuh"

struct HostReadback {                 // pinned; filled by cudaMemcpyAsync from the Control block
    liets::Control head;              // (only the leading scalar part is copied)
};

namespace liets {
struct TileGeom { int nx, ny, nz, Wp, ntx, nty, ntz, periodic; };   // Wp = 64-bit words per x-row; nt* = tiles per axis;
                                                                    // periodic: bit 0 = x wraps, bit 1 = y, bit 2 = z (R5)
}

struct liets_ctx {
    int nx, ny, nz, boundary, storage;
    int periodic;                     // per-axis mask of the boundary mode: bit 0 = x wraps, bit 1 = y, bit 2 = z
    uint64_t N;
    cudaStream_t stream;
    void* ws;
    size_t ws_bytes;
    bool owns_ws;
    int sm_count;
    // device pointers into ws
    liets::Control* ctl;
    uint8_t* grid_u8;                 // STORAGE_U8: N bytes (padded to 4)
    uint32_t* list[2];                // front lists (voxel indices / tile ids)
    uint32_t* status2;                // seeding: 2 bits per voxel (00 none/rejected, 01 pending, 11 accepted)
    uint64_t* explicit_idx;           // staging for liets_seed_explicit (aliases the candidate buffer)
    uint32_t* cand;                   // seeding: candidate voxel indices in ascending order (capacity N) + adjacency
    uint32_t* coff;                   // seeding: candidates before each chunk of 128 voxels
    uint32_t* rowoff;                 // seeding: candidates before each x-row
    // STORAGE_TILE
    liets::TileGeom geom;
    uint64_t n_tiles;
    uint64_t grid_words;              // 64-bit words per grid copy: Wp * ny * nz
    unsigned long long* G[2];         // double-buffered bit grid, x-rows of Wp words
    uint32_t* stamp;                  // per tile: t+1 of the last step whose list holds it
    uint32_t* weight;                 // per tile: front voxels it had when it last ran (orders the list: heavy first)
    uint32_t* vox[2];                 // front VOXEL lists of the small-front steps (grow_vox.cu)
    uint32_t vox_cap;                 // slots per voxel list in use (<= vox_cap_alloc; a test hook shrinks it)
    uint32_t vox_cap_alloc;           // slots per voxel list in the workspace
    uint32_t vox_thr;                 // steps that start with more front voxels run on tiles
    uint8_t* scratch_u8;              // N bytes for format conversion (aliases the candidate buffer)
    uint8_t* pbits;                   // liets_set_blocked: cells of earlier phases, one bit per voxel in linear order
    unsigned long long* prow;         // the same cells in the grid's row layout (bit-row storages)
    bool has_blocked;
    bool no_coop;                     // the device cannot launch cooperative kernels: no voxel-list loop, tiles from step 0
    uint64_t n_blocked;
    uint32_t host_step;               // step counter as of the last read-back (selects the current grid copy)
    int resolve_grid;                 // CTAs of the cooperative spacing kernel (0 = not sized yet)
    int resolve_keyed_grid;           // ... of the keyed-order one
    int spacing_order, spacing_method;   // liets_set_spacing: LIETS_ORDER_*, LIETS_SPACING_*
    uint32_t spacing_ring, spacing_head;  // test hook (liets_debug_spacing_ring): 0 = the built-in sizes
    int tile_grid;                    // CTAs of the tile growth kernel
    int vox_grid;                     // CTAs of the cooperative voxel-list loop (0 = not sized yet)
    uint64_t list_cap;                // slots per front list
    // host state
    liets::Control* pinned;           // pinned host copy of the scalar part of Control
    cudaEvent_t ev0, ev1;
    bool seeded, has_target, growth_set;
    uint64_t rng_seed;
    uint64_t R[3];
    uint64_t RI[3];                   // R20: interaction thresholds per class (all 0: off)
    bool interact;
    int law;
    uint64_t n_t;
    float seed_ms, gen_ms;
    uint64_t launches;                // kernels launched by this ctx
    bool profiling;
    cudaEvent_t* prof_ev;             // 2 * kProfCap events, created on first use
    uint32_t prof_n;                  // growth launches bracketed by the last call
    // liets_generate's device-resident loop: WHILE(step armed) { growth kernel ; control step } as one CUDA graph
    cudaGraph_t loop_graph;
    cudaGraphExec_t loop_exec;
    cudaGraphNode_t loop_grow_node;
    uint64_t loop_seed;               // rng_seed whose Philox key the graph's growth node holds
    bool loop_blocked;                // ... and whether it holds the blocked-cell plane
    bool loop_interact;               // ... and whether its growth node is the interacting variant (R20)
    bool loop_tried;                  // graph creation attempted (on failure generate keeps enqueueing batches)
    char err[256];
};

// liets_create_batch: equally shaped STORAGE_TILE contexts on one stream whose step loops run as ONE graph
struct liets_batch {
    int n;
    liets_ctx* ctx[16];
    cudaStream_t stream;
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    cudaGraphNode_t grow_node;
    uint64_t graph_seed[16];          // rng seeds whose Philox keys the graph's growth node holds
    bool graph_blocked[16];           // ... and whether it holds each grid's blocked-cell plane
    cudaEvent_t ev0, ev1;
    float gen_ms;
    char err[256];
};

#define LIETS_CUDA_TRY(ctx, expr)                                                                 \
    do {                                                                                          \
        cudaError_t e__ = (expr);                                                                 \
        if (e__ != cudaSuccess) {                                                                 \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d: %s: %s", __FILE__, __LINE__, #expr,   \
                     cudaGetErrorString(e__));                                                    \
            return -4;                                                                            \
        }                                                                                         \
    } while (0)

namespace liets {
constexpr uint32_t kProfCap = 4096;
constexpr size_t kControlScalarBytes = offsetof(Control, log_front);

// control.cu
cudaError_t launch_control(liets_ctx* c, uint32_t flags);
cudaError_t launch_begin(liets_ctx* c, int generate, uint32_t max_steps);
cudaError_t launch_set_params(liets_ctx* c);
cudaError_t launch_set_interaction(liets_ctx* c);
cudaError_t launch_eq1_thresholds(const unsigned long long* dev_in, unsigned long long* dev_out, uint32_t n, cudaStream_t stream);
cudaError_t control_loop_node(liets_ctx* c, cudaGraph_t graph, cudaGraphNode_t after, cudaGraphConditionalHandle loop,
                              cudaGraphNode_t* node);
cudaError_t control_loop_batch_node(liets_ctx* const* ctx, int n, cudaGraph_t graph, cudaGraphNode_t after,
                                    cudaGraphConditionalHandle loop, cudaGraphNode_t* node);
// grow_u8.cu
cudaError_t launch_grow_u8(liets_ctx* c);
cudaError_t grow_u8_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node);
// grow_vox.cu
cudaError_t launch_grow_vox(liets_ctx* c);
cudaError_t launch_grow_vox_loop(liets_ctx* c);
cudaError_t launch_tiles_from_grid(liets_ctx* c);
cudaError_t tiles_from_grid_node(liets_ctx* c, cudaGraph_t graph, const cudaGraphNode_t* after, cudaGraphNode_t* node);
// grow_full.cu
cudaError_t launch_grow_full(liets_ctx* c);
cudaError_t grow_full_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node);
// grow_tile.cu
cudaError_t launch_grow_tile(liets_ctx* c);
cudaError_t grow_tile_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node);
cudaError_t grow_tile_batch_node(liets_ctx* const* ctx, int n, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node);
int grow_tile_max_batch();
int grow_tile_words();
int grow_tile_ctas_per_sm();
// seed.cu
cudaError_t launch_seed_reset(liets_ctx* c);
cudaError_t launch_seed_candidates(liets_ctx* c, uint64_t t_core, int accept_all);
cudaError_t launch_spacing(liets_ctx* c, int s);
cudaError_t launch_spacing_keyed(liets_ctx* c, int s);
cudaError_t launch_spacing_dense(liets_ctx* c, int s, uint32_t n_cand, uint32_t* rounds_out);
size_t spacing_dense_bytes(const liets_ctx* c);
cudaError_t launch_seed_finalize(liets_ctx* c, int spaced);
cudaError_t launch_seed_explicit(liets_ctx* c, uint64_t n);
cudaError_t seed_kernel_attributes();
cudaError_t grow_tile_attributes();
// blocked.cu
cudaError_t launch_blocked_set(liets_ctx* c, const uint8_t* src_dev, int format, unsigned long long* count_dev);
cudaError_t launch_blocked_apply(liets_ctx* c);
cudaError_t launch_u8_this_phase(liets_ctx* c, uint8_t* dst);
// s2.cu
cudaError_t launch_s2(liets_ctx* c, int axis, int rmax, unsigned long long* pairs_dev, unsigned long long* rows_scratch);
// export.cu
cudaError_t launch_pack_bits_u8(liets_ctx* c, const uint8_t* src_u8, uint8_t* dst_bits);
cudaError_t launch_unpack_rows_u8(liets_ctx* c, uint8_t* dst_u8);
cudaError_t launch_rows_to_bits(liets_ctx* c, uint8_t* dst_bits);
}  // namespace liets
