// grow_vox.cu -- STORAGE_TILE growth step for SMALL fronts: explicit list of front VOXELS on the bit grid.
//
// While the active set is small (the "very early stages of growth") a tile of 128 x 8 x 8 voxels holds
// a handful of front voxels and the tile kernel spends its time on fixed per-tile work.  Those steps run here
// instead, in the literal list-indexed form of Algorithm 3: one thread per front voxel p of a
// uint32 index list, gather of its 26 neighbours from the bit rows (lines 5-6), the keyed nibble-wise draw (line 8,
// R9), claim by atomicOr (line 9; the thread that flips the bit owns q, "counted once"), and
// A_{t+1} = survivors(A_t) U A_new by one CTA-wide prefix sum per 256 voxels (line 10, :113).  The update is done IN
// PLACE, in both grid copies at once (they stay identical in this mode): a neighbour that another thread claims
// during the same step may be seen solid or void -- seen solid it is solid at the end of the step anyway, seen void
// the atomicOr tells that it was taken -- and draws are keyed, so the grid after the step is exactly the synchronous
// result (the oracle's O-list does the same).  Retirement is lazy as everywhere.
//
// When the list outgrows its threshold (or its capacity: the append then only raises a flag, the grid is still
// exact), the control step hands over to the tile kernel: k_tiles_from_grid lists every tile that holds a solid cell.
#include <cooperative_groups.h>

#include "liets_host.h"

namespace cg = cooperative_groups;

namespace liets {

namespace {

constexpr int kVoxThreads = 256;

// the three cells x-1, x, x+1 of the row that starts at word rb: bit dx+1 = the cell exists and is void
__device__ __forceinline__ uint32_t void3(const unsigned long long* G, unsigned long long rb, int x, int nx, int periodic) {
    const int b = x & 63, w = x >> 6;
    const unsigned long long vm = ~__ldcg(G + rb + w);
    uint32_t r = (uint32_t)(vm >> b) & 1u;
    uint32_t left, right;
    if (b > 0) left = (uint32_t)(vm >> (b - 1)) & 1u;
    else if (x > 0) left = (uint32_t)(~__ldcg(G + rb + w - 1) >> 63) & 1u;
    else left = periodic ? (uint32_t)(~__ldcg(G + rb + ((nx - 1) >> 6)) >> ((nx - 1) & 63)) & 1u : 0u;
    if (x + 1 < nx) right = b < 63 ? (uint32_t)(vm >> (b + 1)) & 1u : (uint32_t)(~__ldcg(G + rb + w + 1)) & 1u;
    else right = periodic ? (uint32_t)(~__ldcg(G + rb)) & 1u : 0u;
    return left | (r << 1) | (right << 2);
}

__device__ __forceinline__ int wrap_coord(int c, int n, int periodic) {       // -1: outside a walled domain
    if (c < 0) return periodic ? n - 1 : -1;
    if (c >= n) return periodic ? 0 : -1;
    return c;
}

// One growth step over the voxel list.  Control fields, list entries and grid words are read from L2 (ld.cg): in the
// persistent loop below other CTAs wrote them in earlier steps of the same launch.
struct VoxShared {
    __align__(16) uint32_t hpat[8][4];
};

__device__ __forceinline__ void vox_step(Control* __restrict__ ctl, const TileGeom& g, unsigned long long* G0,
                                         unsigned long long* G1, uint32_t* vox0, uint32_t* vox1, const PhiloxKey& key,
                                         VoxShared& S) {
    uint32_t (*s_hpat)[4] = S.hpat;
    const uint32_t cur = __ldcg(&ctl->cur);
    const uint32_t n = __ldcg(&ctl->vox_count[cur]), cap = __ldcg(&ctl->vox_cap);
    const uint32_t* in = cur ? vox1 : vox0;
    uint32_t* out = cur ? vox0 : vox1;
    uint32_t* out_count = &ctl->vox_count[cur ^ 1u];
    const uint32_t t = __ldcg(&ctl->step);
    __syncthreads();                                        // the previous step no longer reads S
    if (threadIdx.x < 32) s_hpat[threadIdx.x >> 2][threadIdx.x & 3] = __ldcg(&ctl->hpat[threadIdx.x >> 2][threadIdx.x & 3]);
    const uint32_t en26 = __ldcg(&ctl->en26);
    const PhiloxStep ps = philox_step_uniform(t, key);
    __syncthreads();
    uint32_t my_claims = 0, my_items = 0, my_items0 = 0;

    for (uint64_t base = (uint64_t)blockIdx.x * blockDim.x; base < n; base += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = base + threadIdx.x;
        uint32_t p = 0, mask = 0, won = 0;
        int x = 0, y = 0, z = 0;
        if (i < n) {
            p = __ldcg(in + i);
            x = (int)(p % (uint32_t)g.nx);
            const uint32_t rest = p / (uint32_t)g.nx;
            y = (int)(rest % (uint32_t)g.ny);
            z = (int)(rest / (uint32_t)g.ny);
            uint32_t raw27 = 0;                             // bit 9(dz+1) + 3(dy+1) + (dx+1): that neighbour exists and is void
#pragma unroll
            for (int e = 0; e < 9; ++e) {                   // N_d, C_d (Algorithm 3 lines 5-6), one x-row at a time
                const int Z = wrap_coord(z + e / 3 - 1, g.nz, g.periodic & 4), Y = wrap_coord(y + e % 3 - 1, g.ny, g.periodic & 2);
                if (Z >= 0 && Y >= 0)
                    raw27 |= void3(G0, (unsigned long long)g.Wp * ((unsigned long long)Y + (unsigned long long)g.ny * (unsigned long long)Z),
                                   x, g.nx, g.periodic & 1) << (3 * e);
            }
            mask = (raw27 & 0x1FFFu) | ((raw27 >> 14) << 13);          // the centre (bit 13) is p itself
            if (mask & en26) {
                ++my_items;
                ++my_items0;
                const uint4 B0 = philox_growth_block(p, 0u, ps, key);  // line 8 (rand_num < G_d), nibble level 0 of all 26 draws
                uint32_t le, eq;
                level_compare(B0, s_hpat[0], mask & en26, &le, &eq);
                uint32_t fire = le & ~eq;
                if (eq) fire |= resolve_ties(p, t, eq, s_hpat, key, &my_items);
                while (fire) {                              // two claims in flight: the atomics' return trips overlap
                    uint32_t dd[2] = { 0u, 0u };
                    unsigned long long oo[2] = { ~0ull, ~0ull }, bb[2] = { 0ull, 0ull };
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        if (!fire) break;
                        const uint32_t d = __ffs(fire) - 1u;
                        fire &= fire - 1u;
                        const uint32_t raw = d + (d >= 13u ? 1u : 0u);
                        const int X = wrap_coord(x + (int)(raw % 3u) - 1, g.nx, g.periodic & 1);
                        const int Y = wrap_coord(y + (int)((raw / 3u) % 3u) - 1, g.ny, g.periodic & 2);
                        const int Z = wrap_coord(z + (int)(raw / 9u) - 1, g.nz, g.periodic & 4);
                        const unsigned long long w = (unsigned long long)(X >> 6) + (unsigned long long)g.Wp * ((unsigned long long)Y + (unsigned long long)g.ny * (unsigned long long)Z);
                        bb[k] = 1ull << (X & 63);
                        dd[k] = d;
                        oo[k] = atomicOr(G0 + w, bb[k]);            // line 9: the flipper owns q
                        atomicOr(G1 + w, bb[k]);
                    }
#pragma unroll
                    for (int k = 0; k < 2; ++k)
                        if (bb[k] && !(oo[k] & bb[k])) won |= 1u << dd[k];
                }
            }
        }
        // A_{t+1}: p survives iff it still saw a void neighbour (R13); plus the voxels this thread claimed (line 10)
        const uint32_t keep = mask != 0 ? 1u : 0u;
        const uint32_t cnt = keep + __popc(won);
        my_claims += __popc(won);
        // append: one atomic per warp (no CTA-wide barrier: warps run their list chunks independently)
        uint32_t total;
        uint32_t off = warp_exclusive_scan(cnt, threadIdx.x & 31u, &total);
        uint32_t wbase = 0;
        if ((threadIdx.x & 31u) == 0 && total) wbase = atomicAdd(out_count, total);
        wbase = __shfl_sync(0xffffffffu, wbase, 0);
        off += wbase;
        if (wbase + total > cap) {                          // the list is full: the grid stays exact, the control step switches to tiles
            if ((threadIdx.x & 31u) == 0) ctl->vox_overflow = 1u;
        } else {
            if (keep) out[off++] = p;
            while (won) {
                const uint32_t d = __ffs(won) - 1u;
                won &= won - 1u;
                const uint32_t raw = d + (d >= 13u ? 1u : 0u);
                const int X = wrap_coord(x + (int)(raw % 3u) - 1, g.nx, g.periodic & 1);
                const int Y = wrap_coord(y + (int)((raw / 3u) % 3u) - 1, g.ny, g.periodic & 2);
                const int Z = wrap_coord(z + (int)(raw / 9u) - 1, g.nz, g.periodic & 4);
                out[off++] = (uint32_t)X + (uint32_t)g.nx * ((uint32_t)Y + (uint32_t)g.ny * (uint32_t)Z);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_claims += __shfl_xor_sync(0xffffffffu, my_claims, o);
        my_items += __shfl_xor_sync(0xffffffffu, my_items, o);
        my_items0 += __shfl_xor_sync(0xffffffffu, my_items0, o);
    }
    if ((threadIdx.x & 31u) == 0) {
        if (my_claims) atomicAdd(&ctl->claims, my_claims);
        if (my_items) { atomicAdd(&ctl->items, my_items); atomicAdd(&ctl->items0, my_items0); }
    }
}

__global__ void __launch_bounds__(kVoxThreads) k_grow_vox(Control* __restrict__ ctl, TileGeom g, unsigned long long* G0,
                                                           unsigned long long* G1, uint32_t* vox0, uint32_t* vox1,
                                                           PhiloxKey key) {
    if (!ctl->active || ctl->mode != 0u || ctl->pending) return;
    __shared__ VoxShared S;
    vox_step(ctl, g, G0, G1, vox0, vox1, key, S);
}

// liets_generate: ALL the steps on the voxel list in one cooperative launch -- a grid-wide barrier, the control step
// (thresholds of Eq. (1), stop rule, list swap) on one thread, another barrier, the next step.  Small fronts are bound
// by launch and dependency latency, not by work: this replaces two kernel launches per step by two barriers.
__global__ void __launch_bounds__(kVoxThreads) k_grow_vox_loop(Control* __restrict__ ctl, TileGeom g, unsigned long long* G0,
                                                                unsigned long long* G1, uint32_t* vox0, uint32_t* vox1,
                                                                PhiloxKey key) {
    cg::grid_group grid = cg::this_grid();
    __shared__ VoxShared S;
    for (;;) {
        if (!__ldcg(&ctl->active) || __ldcg(&ctl->mode) != 0u || __ldcg(&ctl->pending)) return;    // the same for every thread
        vox_step(ctl, g, G0, G1, vox0, vox1, key, S);
        grid.sync();
        if (blockIdx.x == 0 && threadIdx.x < 32) control_step(ctl, kCtlFinish | kCtlPrepare);      // one warp
        grid.sync();
    }
}

// The hand-over to the tile kernel: every tile that holds a solid cell enters the tile list of the pending step, once
// (stamp = t + 1, as the tile kernel's own emits use it); a tile without front voxels drops out after one visit.
__global__ void __launch_bounds__(256) k_tiles_from_grid(Control* __restrict__ ctl, TileGeom g, int tile_w,
                                                          const unsigned long long* __restrict__ G0, uint32_t* stamp,
                                                          uint32_t* weight, uint32_t* list0, uint32_t* list1) {
    if (!ctl->active || !ctl->pending || ctl->mode != 0u) return;
    const uint32_t cur = ctl->cur, t = ctl->step, list_cap = ctl->list_cap;
    uint32_t* out = cur ? list1 : list0;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t n_tiles = (uint32_t)g.ntx * (uint32_t)g.nty * (uint32_t)g.ntz;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t tile = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; tile < n_tiles; tile += warps) {
        const uint32_t tx = tile % (uint32_t)g.ntx, rest = tile / (uint32_t)g.ntx;
        const int w0 = (int)tx * tile_w, y0 = 8 * (int)(rest % (uint32_t)g.nty), z0 = 8 * (int)(rest / (uint32_t)g.nty);
        unsigned long long any = 0ull;
        for (int r = (int)lane; r < 64; r += 32) {          // one lane per row of the tile
            const int y = y0 + (r & 7), z = z0 + (r >> 3);
            if (y < g.ny && z < g.nz)
                for (int j = 0; j < tile_w; ++j)
                    if (w0 + j < g.Wp) any |= G0[(unsigned long long)g.Wp * ((unsigned long long)y + (unsigned long long)g.ny * (unsigned long long)z) + (unsigned long long)(w0 + j)];
        }
        const uint32_t have = __ballot_sync(0xffffffffu, any != 0ull);
        if (have && lane == 0) {
            weight[tile] = 0u;
            if (atomicMax(&stamp[tile], t + 1u) < t + 1u) out[list_cap - 1u - atomicAdd(&ctl->count_back[cur], 1u)] = tile;
        }
    }
}

}  // namespace

static void vox_args(liets_ctx* c, PhiloxKey* key, void** a) {
    a[0] = &c->ctl; a[1] = &c->geom; a[2] = &c->G[0]; a[3] = &c->G[1]; a[4] = &c->vox[0]; a[5] = &c->vox[1]; a[6] = key;
}

cudaError_t launch_grow_vox(liets_ctx* c) {
    const PhiloxKey key = philox_make_key(c->rng_seed);
    k_grow_vox<<<c->sm_count * 4, kVoxThreads, 0, c->stream>>>(c->ctl, c->geom, c->G[0], c->G[1], c->vox[0], c->vox[1], key);
    c->launches++;
    return cudaGetLastError();
}

// the whole voxel-list phase of liets_generate as one cooperative launch (the grid must be co-resident)
cudaError_t launch_grow_vox_loop(liets_ctx* c) {
    if (c->vox_grid == 0) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_grow_vox_loop, kVoxThreads, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        c->vox_grid = c->sm_count * (per_sm < 4 ? per_sm : 4);
    }
    PhiloxKey key = philox_make_key(c->rng_seed);
    void* args[7];
    vox_args(c, &key, args);
    c->launches++;
    return cudaLaunchCooperativeKernel((const void*)k_grow_vox_loop, dim3(c->vox_grid), dim3(kVoxThreads), args, 0, c->stream);
}

cudaError_t launch_tiles_from_grid(liets_ctx* c) {
    k_tiles_from_grid<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->geom, grow_tile_words(), c->G[0], c->stamp, c->weight,
                                                              c->list[0], c->list[1]);
    c->launches++;
    return cudaGetLastError();
}

// the hand-over as a kernel node of liets_generate's graph
cudaError_t tiles_from_grid_node(liets_ctx* c, cudaGraph_t graph, const cudaGraphNode_t* after, cudaGraphNode_t* node) {
    int tile_w = grow_tile_words();
    void* args[] = { &c->ctl, &c->geom, &tile_w, &c->G[0], &c->stamp, &c->weight, &c->list[0], &c->list[1] };
    cudaKernelNodeParams p = {};
    p.func = reinterpret_cast<void*>(k_tiles_from_grid);
    p.gridDim = dim3(c->sm_count * 4); p.blockDim = dim3(256); p.sharedMemBytes = 0; p.kernelParams = args;
    return cudaGraphAddKernelNode(node, graph, after, after ? 1 : 0, &p);
}

}  // namespace liets
