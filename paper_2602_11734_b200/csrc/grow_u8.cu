// grow_u8.cu -- STORAGE_U8 growth step: uint8 grid + explicit list of front voxel indices.
//
// This is the list-indexed step of Algorithm 3 with one thread per front
// voxel p: gather the 26 neighbours (line 5-6), draw for the void ones (line 8; nibble-wise draw, R9),
// claim with atomicOr on the 32-bit word holding the target byte (line 9; the thread
// that flips 0 -> 1 owns q, so A_new holds q once -- the paper's "duplicates removed", :113),
// and emit A_{t+1} = survivors(A_t) U A_new with one CTA-wide prefix sum per 256 voxels.
// Retirement is lazy ("cells that no longer have any void neighbors are discarded"):
// p is dropped when this step's gather finds no void neighbour; the grid only grows, so that is
// final.  Reading neighbours that other threads are claiming in the same step is harmless: a
// target seen solid is solid at the end of the step anyway, and draws are keyed, not sequential.
#include "liets_host.h"

namespace liets {

namespace {

struct GridDims { int nx, ny, nz, periodic; };    // periodic: bit 0 = x wraps, bit 1 = y, bit 2 = z (R5)

template <bool PERIODIC>
__device__ __forceinline__ bool neighbour(int d, uint32_t p, int x, int y, int z, const GridDims& g,
                                          uint32_t* q) {
    const int dx = dir_dx(d), dy = dir_dy(d), dz = dir_dz(d);
    int X = x + dx, Y = y + dy, Z = z + dz;
    if (PERIODIC) {                         // some axis wraps: per axis, wrap or stay inside
        if (X < 0) { if (!(g.periodic & 1)) return false; X = g.nx - 1; }
        if (X >= g.nx) { if (!(g.periodic & 1)) return false; X = 0; }
        if (Y < 0) { if (!(g.periodic & 2)) return false; Y = g.ny - 1; }
        if (Y >= g.ny) { if (!(g.periodic & 2)) return false; Y = 0; }
        if (Z < 0) { if (!(g.periodic & 4)) return false; Z = g.nz - 1; }
        if (Z >= g.nz) { if (!(g.periodic & 4)) return false; Z = 0; }
        *q = (uint32_t)X + (uint32_t)g.nx * ((uint32_t)Y + (uint32_t)g.ny * (uint32_t)Z);
        return true;
    } else {
        if ((dx < 0 && X < 0) || (dx > 0 && X >= g.nx) || (dy < 0 && Y < 0) || (dy > 0 && Y >= g.ny) ||
            (dz < 0 && Z < 0) || (dz > 0 && Z >= g.nz))
            return false;
        *q = (uint32_t)((long long)p + dx + (long long)g.nx * (dy + (long long)g.ny * dz));
        return true;
    }
}

template <bool PERIODIC>
__global__ void __launch_bounds__(256) k_grow_u8(Control* __restrict__ ctl, uint8_t* grid,
                                                  uint32_t* list0, uint32_t* list1, GridDims dims,
                                                  PhiloxKey key) {
    if (!ctl->active) return;
    __shared__ uint32_t s_scan[33];
    __shared__ uint32_t s_base;
    const uint32_t cur = ctl->cur;
    const uint32_t n = ctl->count[cur];
    const uint32_t* __restrict__ in = cur ? list1 : list0;
    uint32_t* __restrict__ out = cur ? list0 : list1;
    uint32_t* out_count = &ctl->count[cur ^ 1u];
    const uint32_t t = ctl->step;
    __shared__ __align__(16) uint32_t s_hpat[8][4];
    if (threadIdx.x < 32) s_hpat[threadIdx.x >> 2][threadIdx.x & 3] = ctl->hpat[threadIdx.x >> 2][threadIdx.x & 3];
    const uint32_t en26 = ctl->en26;
    __syncthreads();
    uint32_t my_claims = 0, my_items = 0, my_items0 = 0;

    for (uint64_t base = (uint64_t)blockIdx.x * blockDim.x; base < n; base += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = base + threadIdx.x;
        const bool live = i < n;
        uint32_t p = 0, mask = 0, won = 0;
        int x = 0, y = 0, z = 0;
        if (live) {
            p = in[i];
            x = (int)(p % (uint32_t)dims.nx);
            const uint32_t rest = p / (uint32_t)dims.nx;
            y = (int)(rest % (uint32_t)dims.ny);
            z = (int)(rest / (uint32_t)dims.ny);
#pragma unroll
            for (int d = 0; d < 26; ++d) {                 // N_d, C_d (Algorithm 3 lines 5-6)
                uint32_t q;
                if (neighbour<PERIODIC>(d, p, x, y, z, dims, &q) && grid[q] == 0) mask |= 1u << d;
            }
            if (mask & en26) {
                // line 8 (rand_num < G_d) with the nibble-wise draw (R9): block 0 for all directions at once, the
                // next blocks only for the directions that still tie with the threshold
                ++my_items;
                ++my_items0;
                const uint4 B0 = philox_growth_block(p, 0u, philox_step_uniform(t, key), key);
                uint32_t le, eq;
                level_compare(B0, s_hpat[0], mask & en26, &le, &eq);
                uint32_t fire = le & ~eq;
                if (eq) fire |= resolve_ties(p, t, eq, s_hpat, key, &my_items);
                while (fire) {
                    const uint32_t d = __ffs(fire) - 1u;
                    fire &= fire - 1u;
                    const uint32_t raw = d + (d >= 13u ? 1u : 0u);
                    int X = x + (int)(raw % 3u) - 1, Y = y + (int)((raw / 3u) % 3u) - 1, Z = z + (int)(raw / 9u) - 1;
                    if (PERIODIC) {
                        X = X < 0 ? dims.nx - 1 : (X >= dims.nx ? 0 : X);
                        Y = Y < 0 ? dims.ny - 1 : (Y >= dims.ny ? 0 : Y);
                        Z = Z < 0 ? dims.nz - 1 : (Z >= dims.nz ? 0 : Z);
                    }
                    const uint32_t q = (uint32_t)X + (uint32_t)dims.nx * ((uint32_t)Y + (uint32_t)dims.ny * (uint32_t)Z);
                    const uint32_t sh = (q & 3u) * 8u;
                    const uint32_t old = atomicOr(reinterpret_cast<uint32_t*>(grid) + (q >> 2), 1u << sh);
                    if (((old >> sh) & 0xFFu) == 0) won |= 1u << d;       // line 9-10: owner of q
                }
            }
        }
        // A_{t+1}: p survives iff it still saw a void neighbour; plus the voxels this thread claimed
        const uint32_t keep = mask != 0 ? 1u : 0u;
        const uint32_t cnt = keep + __popc(won);
        my_claims += __popc(won);
        uint32_t total;
        uint32_t off = block_exclusive_scan(cnt, s_scan, &total);
        if (threadIdx.x == 0) s_base = total ? atomicAdd(out_count, total) : 0u;
        __syncthreads();
        off += s_base;
        if (keep) out[off++] = p;
        while (won) {
            const int d = __ffs(won) - 1;
            won &= won - 1;
            // recompute q for direction d (runtime d): offsets from the lexicographic code
            const int raw = d + (d >= 13 ? 1 : 0);
            int X = x + raw % 3 - 1, Y = y + (raw / 3) % 3 - 1, Z = z + raw / 9 - 1;
            if (PERIODIC) {
                X = X < 0 ? dims.nx - 1 : (X >= dims.nx ? 0 : X);
                Y = Y < 0 ? dims.ny - 1 : (Y >= dims.ny ? 0 : Y);
                Z = Z < 0 ? dims.nz - 1 : (Z >= dims.nz ? 0 : Z);
            }
            out[off++] = (uint32_t)X + (uint32_t)dims.nx * ((uint32_t)Y + (uint32_t)dims.ny * (uint32_t)Z);
        }
    }
    // solid count: one atomic per warp at the end of the kernel
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) my_claims += __shfl_xor_sync(0xffffffffu, my_claims, o);
    if ((threadIdx.x & 31u) == 0 && my_claims) atomicAdd(&ctl->claims, my_claims);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) my_items += __shfl_xor_sync(0xffffffffu, my_items, o);
    if ((threadIdx.x & 31u) == 0 && my_items) atomicAdd(&ctl->items, my_items);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) my_items0 += __shfl_xor_sync(0xffffffffu, my_items0, o);
    if ((threadIdx.x & 31u) == 0 && my_items0) atomicAdd(&ctl->items0, my_items0);
}

}  // namespace

cudaError_t launch_grow_u8(liets_ctx* c) {
    const GridDims dims{ c->nx, c->ny, c->nz, c->periodic };
    const PhiloxKey key = philox_make_key(c->rng_seed);
    const int grid = c->sm_count * 8;
    if (c->periodic)
        k_grow_u8<true><<<grid, 256, 0, c->stream>>>(c->ctl, c->grid_u8, c->list[0], c->list[1], dims, key);
    else
        k_grow_u8<false><<<grid, 256, 0, c->stream>>>(c->ctl, c->grid_u8, c->list[0], c->list[1], dims, key);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t grow_u8_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node) {
    GridDims dims{ c->nx, c->ny, c->nz, c->periodic };
    PhiloxKey key = philox_make_key(c->rng_seed);
    void* args[] = { &c->ctl, &c->grid_u8, &c->list[0], &c->list[1], &dims, &key };
    cudaKernelNodeParams p = {};
    p.func = c->periodic ? reinterpret_cast<void*>(k_grow_u8<true>) : reinterpret_cast<void*>(k_grow_u8<false>);
    p.gridDim = dim3(c->sm_count * 8); p.blockDim = dim3(256); p.sharedMemBytes = 0; p.kernelParams = args;
    return exec ? cudaGraphExecKernelNodeSetParams(exec, *node, &p) : cudaGraphAddKernelNode(node, graph, nullptr, 0, &p);
}

}  // namespace liets
