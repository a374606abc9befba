// grow_full.cu -- STORAGE_FULL growth step: Algorithm 2, the vectorised FULL-FIELD sweep, on the bit rows.
//
// No active set at all: every step visits every cell of the grid, as the paper's "vectorized QSGS" does (:66-78; its
// same-hardware comparison with the list-indexed method is :181).  One warp per 32 consecutive cells of an x-row, one lane
// per cell.  The nine rows of the cells' neighbourhood are fetched once per warp (the same words for every lane) as 34-bit
// windows; a lane whose cell is solid and has a void neighbour draws for its void directions (line 8 of Algorithm 3 is
// line 7 of Algorithm 2 per direction) with the SAME keyed draws as the list kernels, so the grid after
// the step is the same grid (made exact) -- only the cost differs: proportional to N instead of N_active
// (PAPER.md:118).  Step t reads G[t&1] and ORs into G[(t+1)&1] (new cells act in the next iteration only, :78); every
// word is carried over, every claim is an atomicOr whose old value tells whether the cell was already taken (:77).
// Segments whose neighbourhood holds no solid cell, or no void cell, are skipped after the nine loads.
#include "liets_host.h"

namespace liets {

namespace {

constexpr int kFullThreads = 256;

__device__ __forceinline__ int full_wrap(int c, int n, int periodic) {      // -1: outside a walled domain
    if (c < 0) return periodic ? n - 1 : -1;
    if (c >= n) return periodic ? 0 : -1;
    return c;
}

// (g_t is immutable during the step, so its rows are read through the read-only L1 path: each is used by nine rows of warps)
// "not void" bits of cells x0-1 .. x0+32 of the row at word offset rb (bit i = cell x0 - 1 + i; cells outside a walled
// domain and cells beyond the row count as not void, a periodic row wraps)
__device__ __forceinline__ unsigned long long window34(const unsigned long long* __restrict__ G, unsigned long long rb, int x0,
                                                       const TileGeom& g) {
    const int w = x0 >> 6, b = x0 & 63;                     // b is 0 or 32
    const int xbase = 64 * w;
    unsigned long long cur = __ldg(G + rb + w);
    if (xbase + 64 > g.nx) cur |= ~0ull << (g.nx - xbase);  // beyond the row: not void
    unsigned long long win = (cur >> b) << 1;               // cells x0 .. x0+31 (and up to x0+62) at bits 1 ..
    // cell x0 - 1
    unsigned long long left;
    if (b) left = (cur >> (b - 1)) & 1ull;
    else if (w > 0) left = __ldg(G + rb + w - 1) >> 63;
    else left = (g.periodic & 1) ? (__ldg(G + rb + ((g.nx - 1) >> 6)) >> ((g.nx - 1) & 63)) & 1ull : 1ull;
    win |= left;
    // cell x0 + 32
    if (b) {                                                // it is in the next word, or across the row end
        unsigned long long right;
        if (xbase + 64 < g.nx) right = __ldg(G + rb + w + 1) & 1ull;
        else right = 1ull;                                  // beyond the row (fixed below if the row ends exactly here)
        win = (win & ~(1ull << 33)) | (right << 33);
    }
    // the cell just beyond the row end, x = nx, is cell 0 of a periodic row
    const int iend = g.nx - (x0 - 1);                       // window bit of cell x = nx
    if (iend >= 0 && iend <= 33) {
        const unsigned long long wrap = (g.periodic & 1) ? __ldg(G + rb) & 1ull : 1ull;
        win = (win & ~(1ull << iend)) | (wrap << iend);
    }
    return win & 0x3FFFFFFFFull;
}

__global__ void __launch_bounds__(kFullThreads) k_grow_full(Control* __restrict__ ctl, TileGeom g, unsigned long long* G0,
                                                             unsigned long long* G1, const unsigned long long* __restrict__ P,
                                                             PhiloxKey key) {
    if (!ctl->active) return;
    __shared__ __align__(16) uint32_t s_hpat[2][8][4];      // [1]: the interaction thresholds (R20), used by sources of earlier phases
    const uint32_t t = ctl->step;
    const unsigned long long* __restrict__ Gc = (t & 1u) ? G1 : G0;
    unsigned long long* Gn = (t & 1u) ? G0 : G1;
    if (threadIdx.x < 32) s_hpat[0][threadIdx.x >> 2][threadIdx.x & 3] = ctl->hpat[threadIdx.x >> 2][threadIdx.x & 3];
    else if (threadIdx.x < 64) s_hpat[1][(threadIdx.x - 32) >> 2][threadIdx.x & 3] = ctl->hpatI[(threadIdx.x - 32) >> 2][threadIdx.x & 3];
    const uint32_t en26 = ctl->en26;
    const bool interact = P != nullptr && ctl->interact != 0u;
    const uint32_t enI26 = ctl->enI26;
    const PhiloxStep ps = philox_step_uniform(t, key);
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t segs_per_row = 2u * (uint32_t)g.Wp;                      // N < 2^32, so the segment count fits 32 bits
    const uint32_t n_seg = segs_per_row * (uint32_t)g.ny * (uint32_t)g.nz;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    uint32_t my_claims = 0, my_items = 0, my_items0 = 0;

    for (uint32_t seg = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; seg < n_seg; seg += warps) {
        const int sx = (int)(seg % segs_per_row);
        const uint32_t rowi = seg / segs_per_row;
        const int y = (int)(rowi % (uint32_t)g.ny), z = (int)(rowi / (uint32_t)g.ny);
        const int x0 = 32 * sx;
        if (x0 >= g.nx) continue;
        // the nine rows (the same for every lane)
        unsigned long long win[9];
        unsigned long long all_or = 0ull, all_and = ~0ull;
#pragma unroll
        for (int e = 0; e < 9; ++e) {
            const int Z = full_wrap(z + e / 3 - 1, g.nz, g.periodic & 4), Y = full_wrap(y + e % 3 - 1, g.ny, g.periodic & 2);
            win[e] = (Z >= 0 && Y >= 0)
                   ? window34(Gc, (unsigned long long)g.Wp * ((unsigned long long)Y + (unsigned long long)g.ny * (unsigned long long)Z), x0, g)
                   : 0x3FFFFFFFFull;
            all_or |= win[e];
            all_and &= win[e];
        }
        const unsigned long long own_word_idx = (unsigned long long)rowi * (unsigned long long)g.Wp + (unsigned long long)(x0 >> 6);
        const uint32_t own32 = (uint32_t)(win[4] >> 1);                     // cells x0 .. x0+31 (not-void = solid or beyond the row)
        uint32_t in_row = 0xFFFFFFFFu;
        if (x0 + 32 > g.nx) in_row = ~(~0u << (g.nx - x0));
        uint32_t solid32 = own32 & in_row;
        // carry g_t into g_{t+1} (one atomic per segment that holds solid cells)
        if (lane == 0 && solid32) atomicOr(Gn + own_word_idx, (unsigned long long)solid32 << (x0 & 63));
        uint32_t other32 = 0;                               // cells of earlier phases: carried; sources only at an interacting interface (R20)
        if (P) { other32 = (uint32_t)(__ldg(P + own_word_idx) >> (x0 & 63)) & solid32; if (!interact) solid32 &= ~other32; }
        // nothing solid in the centre row's cells, or no void cell anywhere around: no attempt can exist here
        if (solid32 == 0u || all_and == 0x3FFFFFFFFull || all_or == 0ull) continue;
        const int x = x0 + (int)lane;
        uint32_t fire = 0;
        if ((solid32 >> lane) & 1u) {
            uint32_t nb27 = 0;                              // bit 9(dz+1) + 3(dy+1) + (dx+1): not void
#pragma unroll
            for (int e = 0; e < 9; ++e) nb27 |= ((uint32_t)(win[e] >> lane) & 7u) << (3 * e);
            const uint32_t v27 = ~nb27;
            const uint32_t kind = (other32 >> lane) & 1u;   // 1: a cell of an earlier phase, it uses I
            const uint32_t mask = ((v27 & 0x1FFFu) | ((v27 >> 14) << 13)) & 0x3FFFFFFu & (kind ? enI26 : en26);     // C_d (Algorithm 2 line 6), the centre skipped
            if (mask) {
                const uint32_t p = (uint32_t)x + (uint32_t)g.nx * ((uint32_t)y + (uint32_t)g.ny * (uint32_t)z);
                ++my_items;
                ++my_items0;
                const uint4 B0 = philox_growth_block(p, 0u, ps, key);      // R_d for all directions (line 7), nibble level 0
                uint32_t le, eq;
                level_compare(B0, s_hpat[kind][0], mask, &le, &eq);
                fire = le & ~eq;
                if (eq) fire |= resolve_ties(p, t, eq, s_hpat[kind], key, &my_items);
            }
        }
        while (fire) {                                      // line 8: phase_new[mask] = 1, "counted once" by the atomic's old value (:77)
            const uint32_t d = __ffs(fire) - 1u;
            fire &= fire - 1u;
            const uint32_t raw = d + (d >= 13u ? 1u : 0u);
            const int X = full_wrap(x + (int)(raw % 3u) - 1, g.nx, g.periodic & 1);
            const int Y = full_wrap(y + (int)((raw / 3u) % 3u) - 1, g.ny, g.periodic & 2);
            const int Z = full_wrap(z + (int)(raw / 9u) - 1, g.nz, g.periodic & 4);
            const unsigned long long w = (unsigned long long)(X >> 6) + (unsigned long long)g.Wp * ((unsigned long long)Y + (unsigned long long)g.ny * (unsigned long long)Z);
            const unsigned long long bit = 1ull << (X & 63);
            const unsigned long long old = atomicOr(Gn + w, bit);
            if (!(old & bit)) ++my_claims;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_claims += __shfl_xor_sync(0xffffffffu, my_claims, o);
        my_items += __shfl_xor_sync(0xffffffffu, my_items, o);
        my_items0 += __shfl_xor_sync(0xffffffffu, my_items0, o);
    }
    if (lane == 0) {
        if (my_claims) atomicAdd(&ctl->claims, my_claims);
        if (my_items) { atomicAdd(&ctl->items, my_items); atomicAdd(&ctl->items0, my_items0); }
    }
}

}  // namespace

cudaError_t launch_grow_full(liets_ctx* c) {
    const PhiloxKey key = philox_make_key(c->rng_seed);
    k_grow_full<<<c->sm_count * 8, kFullThreads, 0, c->stream>>>(c->ctl, c->geom, c->G[0], c->G[1], c->has_blocked ? c->prow : nullptr, key);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t grow_full_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node) {
    PhiloxKey key = philox_make_key(c->rng_seed);
    const unsigned long long* P = c->has_blocked ? c->prow : nullptr;
    void* args[] = { &c->ctl, &c->geom, &c->G[0], &c->G[1], &P, &key };
    cudaKernelNodeParams p = {};
    p.func = reinterpret_cast<void*>(k_grow_full);
    p.gridDim = dim3(c->sm_count * 8); p.blockDim = dim3(kFullThreads); p.sharedMemBytes = 0; p.kernelParams = args;
    return exec ? cudaGraphExecKernelNodeSetParams(exec, *node, &p) : cudaGraphAddKernelNode(node, graph, nullptr, 0, &p);
}

}  // namespace liets
