// seed.cu -- seeding and seed spacing by the L1 "diamond".
//
// Candidates: voxel v is a candidate core iff philox(seed; v>>2)[v&3] < T_core (R9).
// Spacing (R11, R12): the sequential rule "scan candidates in ascending index, accept iff no
// accepted seed within L1 < s" is reproduced exactly by parallel rounds over a 2-bit-per-voxel
// status map (00 = no candidate / rejected, 01 = pending, 11 = accepted):
//   a pending candidate v looks at every LOWER-index voxel within L1 < s (its diamond);
//   - any accepted one  -> v is rejected (final: that seed is accepted in the sequential scan too);
//   - else any pending  -> v waits (its fate depends on them);
//   - else              -> v is accepted (all lower-index candidates in range are rejected).
// Each state change is one atomic on one word, states only move 01 -> {00, 11}, so reading
// neighbours that change during a round is safe, and the fixed point is the sequential result.
#include <cooperative_groups.h>

#include "liets_host.h"

namespace cg = cooperative_groups;

namespace liets {

namespace {

__device__ __forceinline__ uint32_t ld_cg(const uint32_t* p) {
    return __ldcg(p);
}

// --- reset: grid, status map, counters ---------------------------------------------------------
__global__ void k_seed_reset(Control* c) {
    c->n_solid = 0; c->step = 0; c->steps_done = 0; c->active = 0; c->status = 0; c->cur = 0;
    c->count[0] = 0; c->count[1] = 0; c->claims = 0; c->n_cand = 0;
    c->pool_head = 0; c->n_rescan = 0; c->pend3[0] = 0; c->pend3[1] = 0; c->pend3[2] = 0;
}

// --- candidates: one thread per status word = 16 voxels = 4 Philox blocks -----------------------
__global__ void __launch_bounds__(256) k_seed_candidates(Control* ctl, uint32_t* status2, uint32_t* cand,
                                                          unsigned long long N, uint32_t T_core,
                                                          uint32_t always, uint32_t accept_all,
                                                          PhiloxKey key) {
    __shared__ uint32_t s_scan[33];
    __shared__ uint32_t s_base;
    const unsigned long long n_words = (N + 15ull) / 16ull;
    for (unsigned long long base = (unsigned long long)blockIdx.x * blockDim.x; base < n_words;
         base += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long w = base + threadIdx.x;
        uint32_t bits = 0;                                  // bit k: voxel 16w+k is a candidate
        if (w < n_words) {
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const unsigned long long blk = 4ull * w + b;          // = v >> 2
                if (blk * 4ull >= N) break;
                const uint4 r = philox4x32_10((uint32_t)blk, (uint32_t)(blk >> 32), 0u, 0xFFFFFFFFu, key);
                const uint32_t d[4] = { r.x, r.y, r.z, r.w };
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (blk * 4ull + k < N && (always || d[k] < T_core)) bits |= 1u << (4 * b + k);
            }
            uint32_t word = 0;                              // spread: bit k -> field 2k
            for (uint32_t m = bits; m; m &= m - 1) {
                const int k = __ffs(m) - 1;
                word |= (accept_all ? 3u : 1u) << (2 * k);
            }
            status2[w] = word;
        }
        uint32_t total;
        uint32_t off = block_exclusive_scan(__popc(bits), s_scan, &total);
        if (threadIdx.x == 0) s_base = total ? atomicAdd(&ctl->n_cand, total) : 0u;
        __syncthreads();
        off += s_base;
        for (uint32_t m = bits; m; m &= m - 1) cand[off++] = (uint32_t)(16ull * w + (__ffs(m) - 1));
    }
}

// --- seed spacing -------------------------------------------------------------------------------
struct Dims { int nx, ny, nz, periodic; };

constexpr uint32_t kRescan = 0xFFFFFFFFu;       // adjacency of this candidate not stored: rescan its diamond
constexpr int kAdjBuf = 96;                     // neighbours a warp can buffer per candidate

// Warp-cooperative walk over the status words of the LOWER-index voxels within L1 < s of voxel v
// (the candidate's diamond).  on_word(word, lo) gets each status word with the fields
// of out-of-range voxels cleared; lo = linear index of the word's first voxel.
template <class F>
__device__ __forceinline__ void scan_segment(const uint32_t* status2, unsigned long long i0,
                                             unsigned long long i1, unsigned long long limit, F& on_word) {
    if (i0 >= limit) return;
    if (i1 >= limit) i1 = limit - 1;
    for (unsigned long long w = i0 >> 4; w <= (i1 >> 4); ++w) {
        uint32_t word = ld_cg(status2 + w);
        if (!word) continue;
        const unsigned long long lo = w << 4;
        uint32_t field = 0xFFFFFFFFu;                       // keep fields of voxels in [i0, i1]
        if (i0 > lo) field &= 0xFFFFFFFFu << (2 * (uint32_t)(i0 - lo));
        if (i1 < lo + 15) field &= 0xFFFFFFFFu >> (2 * (uint32_t)(lo + 15 - i1));
        word &= field;
        if (word) on_word(word, lo);
    }
}

template <class F>
__device__ __forceinline__ void scan_diamond(const uint32_t* status2, uint32_t v, const Dims& g, int s,
                                             uint32_t lane, F& on_word) {
    const int x = (int)(v % (uint32_t)g.nx);
    const uint32_t rest = v / (uint32_t)g.nx;
    const int y = (int)(rest % (uint32_t)g.ny), z = (int)(rest / (uint32_t)g.ny);
    const int r = s - 1;                                    // diamond radius: L1 <= s-1  <=>  L1 < s
    const int side = 2 * r + 1;
    // without wrap-around, lower-index voxels have dz < 0, or dz = 0 and dy <= 0
    const int n_rows = g.periodic ? side * side : (r + 1) * side;
    for (int j = (int)lane; j < n_rows; j += 32) {
        const int dz = j / side - r, dy = j % side - r;
        const int rem = r - abs(dz) - abs(dy);
        if (rem < 0) continue;
        int Y = y + dy, Z = z + dz;
        if (g.periodic) {
            Y %= g.ny; if (Y < 0) Y += g.ny;
            Z %= g.nz; if (Z < 0) Z += g.nz;
        } else if (Y < 0 || Y >= g.ny || Z < 0 || Z >= g.nz || (dz == 0 && dy > 0)) {
            continue;
        }
        const unsigned long long row = ((unsigned long long)Z * g.ny + Y) * (unsigned long long)g.nx;
        int xa = x - rem, xb = x + rem;
        if (g.periodic && 2 * rem + 1 >= g.nx) {            // the range covers the whole row
            scan_segment(status2, row, row + g.nx - 1, v, on_word);
        } else if (!g.periodic) {                           // clipped at the walls
            xa = xa < 0 ? 0 : xa;
            xb = xb >= g.nx ? g.nx - 1 : xb;
            scan_segment(status2, row + xa, row + xb, v, on_word);
        } else {                                            // wrapped range, at most two segments
            if (xa < 0) {
                scan_segment(status2, row + (xa + g.nx), row + g.nx - 1, v, on_word);
                xa = 0;
            }
            if (xb >= g.nx) {
                scan_segment(status2, row, row + (xb - g.nx), v, on_word);
                xb = g.nx - 1;
            }
            scan_segment(status2, row + xa, row + xb, v, on_word);
        }
    }
}

// layout of the candidate buffer (capacity N words): cand[n] | off[n] | cnt[n] | rescan[n] | pool[N-4n]
struct AdjView {
    bool ok;
    uint32_t *off, *cnt, *rescan, *pool;
    unsigned long long pool_cap;
};
__device__ __forceinline__ AdjView adj_view(uint32_t* cand, uint32_t n, unsigned long long N) {
    AdjView a;
    a.ok = 4ull * n <= N;
    a.off = cand + n; a.cnt = cand + 2ull * n; a.rescan = cand + 3ull * n; a.pool = cand + 4ull * n;
    a.pool_cap = a.ok ? N - 4ull * n : 0ull;
    return a;
}

// Pass 1: one warp per candidate lists the lower-index candidates inside its diamond, once.
__global__ void __launch_bounds__(256) k_spacing_adjacency(Control* ctl, const uint32_t* status2, uint32_t* cand,
                                                            Dims g, int s, unsigned long long N) {
    __shared__ uint32_t s_buf[8][kAdjBuf];
    __shared__ uint32_t s_cnt[8];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t warp_global = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n = ctl->n_cand;
    const AdjView a = adj_view(cand, n, N);
    if (!a.ok) return;
    for (uint32_t i = warp_global; i < n; i += n_warps) {
        const uint32_t v = cand[i];
        if (lane == 0) s_cnt[warp] = 0;
        __syncwarp();
        auto collect = [&](uint32_t word, unsigned long long lo) {
            for (uint32_t m = word & 0x55555555u; m; m &= m - 1) {          // every candidate in the word
                const uint32_t slot = atomicAdd(&s_cnt[warp], 1u);
                if (slot < (uint32_t)kAdjBuf) s_buf[warp][slot] = (uint32_t)lo + ((__ffs(m) - 1) >> 1);
            }
        };
        scan_diamond(status2, v, g, s, lane, collect);
        __syncwarp();
        const uint32_t k = s_cnt[warp];
        uint32_t base = 0;
        bool stored = k <= (uint32_t)kAdjBuf;
        if (stored && k) {
            if (lane == 0) base = atomicAdd(&ctl->pool_head, k);
            base = __shfl_sync(0xffffffffu, base, 0);
            stored = (unsigned long long)base + k <= a.pool_cap;
        }
        if (stored) {
            for (uint32_t e = lane; e < k; e += 32) a.pool[base + e] = s_buf[warp][e];
            if (lane == 0) { a.off[i] = base; a.cnt[i] = k; }
        } else if (lane == 0) {
            a.cnt[i] = kRescan;
            a.rescan[atomicAdd(&ctl->n_rescan, 1u)] = i;
        }
        __syncwarp();
    }
}

__device__ __forceinline__ uint32_t status_of(const uint32_t* status2, uint32_t v) {
    return (ld_cg(status2 + (v >> 4)) >> (2 * (v & 15u))) & 3u;
}

// one look at the stored lower-index neighbours of pending candidate v:
// 0 = still waiting, 1 = resolved now (v's status word updated)
__device__ __forceinline__ uint32_t try_resolve(uint32_t* status2, uint32_t v, const uint32_t* nb, uint32_t k) {
    bool accepted = false, pending = false;
    for (uint32_t e = 0; e < k; ++e) {
        const uint32_t st = status_of(status2, nb[e]);
        accepted = accepted || st == 3u;
        pending = pending || st == 1u;
    }
    if (accepted) { atomicAnd(status2 + (v >> 4), ~(1u << (2 * (v & 15u)))); return 1u; }     // 01 -> 00
    if (!pending) { atomicOr(status2 + (v >> 4), 2u << (2 * (v & 15u))); return 1u; }         // 01 -> 11
    return 0u;
}

// the same look with the neighbour indices in registers (k <= 8): the status loads are independent, so one look
// costs one L2 round trip instead of k
__device__ __forceinline__ uint32_t try_resolve_reg(uint32_t* status2, uint32_t v, const uint32_t (&nbr)[8], uint32_t k) {
    uint32_t w[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) w[e] = (uint32_t)e < k ? ld_cg(status2 + (nbr[e] >> 4)) : 0u;
    bool accepted = false, pending = false;
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        const uint32_t st = (uint32_t)e < k ? (w[e] >> (2 * (nbr[e] & 15u))) & 3u : 0u;
        accepted = accepted || st == 3u;
        pending = pending || st == 1u;
    }
    if (accepted) { atomicAnd(status2 + (v >> 4), ~(1u << (2 * (v & 15u)))); return 1u; }     // 01 -> 00
    if (!pending) { atomicOr(status2 + (v >> 4), 2u << (2 * (v & 15u))); return 1u; }         // 01 -> 11
    return 0u;
}

constexpr int kPolls = 64;      // looks per round before falling back to a grid-wide sync

// Pass 2: all rounds in one cooperative launch.  A pending candidate is rejected as soon as a
// lower-index neighbour is accepted, accepted once none of them is pending, else it waits.  Every
// thread keeps its first candidate in registers and polls its neighbours' status words (L2) a
// bounded number of times per round, so a dependency chain of length L needs about L / kPolls
// grid-wide syncs instead of L.
__global__ void __launch_bounds__(1024) k_spacing_resolve(Control* ctl, uint32_t* status2, uint32_t* cand,
                                                           Dims g, int s, unsigned long long N) {
    cg::grid_group grid = cg::this_grid();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, n_threads = gridDim.x * blockDim.x;
    const uint32_t n = ctl->n_cand;
    const AdjView a = adj_view(cand, n, N);
    const uint32_t n_rescan = a.ok ? ld_cg(&ctl->n_rescan) : n;
    // this thread's own candidate (i = tid), cached
    uint32_t v0 = 0, k0 = 0;
    const uint32_t* nb0 = nullptr;
    bool open0 = false;
    if (a.ok && tid < n) {
        k0 = a.cnt[tid];
        if (k0 != kRescan) { v0 = cand[tid]; nb0 = a.pool + a.off[tid]; open0 = status_of(status2, v0) == 1u; }
    }
    uint32_t nbr[8] = { 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u };
    const bool in_regs = k0 <= 8u;
    if (open0 && in_regs) {
#pragma unroll
        for (int e = 0; e < 8; ++e)
            if ((uint32_t)e < k0) nbr[e] = nb0[e];
    }
    for (uint32_t round = 0;; ++round) {
        uint32_t still = 0;
        for (int poll = 0; poll < kPolls; ++poll) {
            if (!__any_sync(0xffffffffu, open0)) break;
            if (open0 && (in_regs ? try_resolve_reg(status2, v0, nbr, k0) : try_resolve(status2, v0, nb0, k0))) open0 = false;
        }
        if (open0) still++;
        if (a.ok) {
            for (uint32_t i = tid + n_threads; i < n; i += n_threads) {     // more candidates than threads
                const uint32_t k = a.cnt[i];
                if (k == kRescan) continue;
                const uint32_t v = cand[i];
                if (status_of(status2, v) != 1u) continue;
                if (!try_resolve(status2, v, a.pool + a.off[i], k)) still++;
            }
        }
        for (uint32_t q = tid >> 5; q < n_rescan; q += n_threads >> 5) { // one warp per candidate: rescan
            const uint32_t i = a.ok ? a.rescan[q] : q;
            const uint32_t v = cand[i];
            if (status_of(status2, v) != 1u) continue;
            bool accepted = false, pending = false;
            auto look = [&](uint32_t word, unsigned long long) {
                const uint32_t b0 = word & 0x55555555u, b1 = (word >> 1) & 0x55555555u;
                if (b0 & b1) accepted = true;
                if (b0 & ~b1) pending = true;
            };
            scan_diamond(status2, v, g, s, lane, look);
            accepted = __any_sync(0xffffffffu, accepted);
            pending = __any_sync(0xffffffffu, pending);
            if (lane == 0) {
                if (accepted) atomicAnd(status2 + (v >> 4), ~(1u << (2 * (v & 15u))));
                else if (!pending) atomicOr(status2 + (v >> 4), 2u << (2 * (v & 15u)));
                else still++;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) still += __shfl_xor_sync(0xffffffffu, still, o);
        if (lane == 0 && still) atomicAdd(&ctl->pend3[round % 3u], still);
        grid.sync();
        const uint32_t left = ld_cg(&ctl->pend3[round % 3u]);
        if (tid == 0) ctl->pend3[(round + 2u) % 3u] = 0;               // next used in round+2, after another sync
        if (left == 0) break;
    }
}

// --- finalize: accepted candidates -> grid + initial front A_0 = seeds (R3) ---------------------
__global__ void __launch_bounds__(256) k_seed_finalize_u8(Control* ctl, const uint32_t* status2,
                                                           const uint32_t* cand, uint8_t* grid,
                                                           uint32_t* front) {
    __shared__ uint32_t s_scan[33];
    __shared__ uint32_t s_base;
    const uint32_t n = ctl->n_cand;
    for (uint64_t base = (uint64_t)blockIdx.x * blockDim.x; base < n; base += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = base + threadIdx.x;
        uint32_t v = 0, acc = 0;
        if (i < n) {
            v = cand[i];
            acc = ((status2[v >> 4] >> (2 * (v & 15u))) & 3u) == 3u;
        }
        uint32_t total;
        uint32_t off = block_exclusive_scan(acc, s_scan, &total);
        if (threadIdx.x == 0) s_base = total ? atomicAdd(&ctl->count[0], total) : 0u;
        __syncthreads();
        if (acc) { front[s_base + off] = v; grid[v] = 1; }
    }
}

__global__ void k_seed_close(Control* c) { c->n_solid = c->count[0]; c->cur = 0; }

// STORAGE_TILE: set the seed's bit in both grid copies; the tile enters the list of step 0 once
// (stamp = 1).  The 0 -> 1 transition of the bit in G0 dedupes explicit seeds and counts them.
__device__ __forceinline__ void place_seed_tile(Control* ctl, uint32_t v, TileGeom g, int tile_w, unsigned long long* G0,
                                                unsigned long long* G1, uint32_t* stamp, uint32_t* front) {
    const uint32_t x = v % (uint32_t)g.nx, rest = v / (uint32_t)g.nx;
    const uint32_t y = rest % (uint32_t)g.ny, z = rest / (uint32_t)g.ny;
    const unsigned long long w = (unsigned long long)(x >> 6) + (unsigned long long)g.Wp * ((unsigned long long)y + (unsigned long long)g.ny * z);
    const unsigned long long bit = 1ull << (x & 63u);
    const unsigned long long old = atomicOr(G0 + w, bit);
    atomicOr(G1 + w, bit);
    if (!(old & bit)) atomicAdd(&ctl->n_solid, 1ull);
    const uint32_t tile = (x >> 6) / (uint32_t)tile_w + (uint32_t)g.ntx * ((y >> 3) + (uint32_t)g.nty * (z >> 3));
    if (atomicMax(&stamp[tile], 1u) < 1u) front[atomicAdd(&ctl->count[0], 1u)] = tile;
}

__global__ void __launch_bounds__(256) k_seed_finalize_tile(Control* ctl, const uint32_t* status2, const uint32_t* cand,
                                                             TileGeom g, int tile_w, unsigned long long* G0, unsigned long long* G1,
                                                             uint32_t* stamp, uint32_t* front) {
    const uint32_t n = ctl->n_cand;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t v = cand[i];
        if (((status2[v >> 4] >> (2 * (v & 15u))) & 3u) == 3u) place_seed_tile(ctl, v, g, tile_w, G0, G1, stamp, front);
    }
}

__global__ void k_seed_explicit_tile(Control* ctl, const unsigned long long* idx, unsigned long long n, TileGeom g, int tile_w,
                                     unsigned long long* G0, unsigned long long* G1, uint32_t* stamp, uint32_t* front) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x)
        place_seed_tile(ctl, (uint32_t)idx[i], g, tile_w, G0, G1, stamp, front);
}

__global__ void k_seed_close_tile(Control* c) { c->cur = 0; }

// --- explicit seeds: dedupe with the 0 -> 1 transition of the grid byte -------------------------
__global__ void k_seed_explicit_u8(Control* ctl, const unsigned long long* idx, unsigned long long n,
                                   uint8_t* grid, uint32_t* front) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t v = (uint32_t)idx[i];
        const uint32_t sh = (v & 3u) * 8u;
        const uint32_t old = atomicOr(reinterpret_cast<uint32_t*>(grid) + (v >> 2), 1u << sh);
        if (((old >> sh) & 0xFFu) == 0) front[atomicAdd(&ctl->count[0], 1u)] = v;
    }
}

}  // namespace

cudaError_t launch_seed_reset(liets_ctx* c) {
    cudaError_t e;
    if (c->storage == 0) {
        e = cudaMemsetAsync(c->grid_u8, 0, (c->N + 3) & ~3ull, c->stream);
    } else {                                                // G[0], G[1] and the stamps are contiguous
        e = cudaMemsetAsync(c->G[0], 0, c->grid_words * 16 + c->n_tiles * 4, c->stream);
    }
    if (e != cudaSuccess) return e;
    k_seed_reset<<<1, 1, 0, c->stream>>>(c->ctl);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_seed_candidates(liets_ctx* c, uint64_t t_core, int accept_all) {
    const PhiloxKey key = philox_make_key(c->rng_seed);
    const uint32_t always = t_core >= (1ull << 32);
    const uint32_t T = always ? 0xFFFFFFFFu : (uint32_t)t_core;
    k_seed_candidates<<<c->sm_count * 8, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, c->N, T, always,
                                                              (uint32_t)accept_all, key);
    c->launches++;
    return cudaGetLastError();
}

// exact parallel reproduction of the ascending-index greedy (R12): adjacency once, then all rounds
// inside one cooperative kernel (grid-wide syncs on the device, no host round trip)
cudaError_t launch_spacing(liets_ctx* c, int s) {
    Dims g{ c->nx, c->ny, c->nz, c->boundary };
    unsigned long long N = c->N;
    k_spacing_adjacency<<<c->sm_count * 8, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, g, s, N);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (c->resolve_grid == 0) {
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_spacing_resolve, 1024, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1) return cudaErrorLaunchOutOfResources;
        c->resolve_grid = c->sm_count;
    }
    void* args[] = { &c->ctl, &c->status2, &c->cand, &g, &s, &N };
    e = cudaLaunchCooperativeKernel((const void*)k_spacing_resolve, dim3(c->resolve_grid), dim3(1024), args, 0, c->stream);
    c->launches++;
    return e;
}

cudaError_t launch_seed_finalize(liets_ctx* c) {
    if (c->storage == 0)
        k_seed_finalize_u8<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, c->grid_u8, c->list[0]);
    else
        k_seed_finalize_tile<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, c->geom, grow_tile_words(),
                                                                    c->G[0], c->G[1], c->stamp, c->list[0]);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (c->storage == 0) k_seed_close<<<1, 1, 0, c->stream>>>(c->ctl);
    else k_seed_close_tile<<<1, 1, 0, c->stream>>>(c->ctl);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_seed_explicit(liets_ctx* c, uint64_t n) {
    if (n) {
        if (c->storage == 0)
            k_seed_explicit_u8<<<c->sm_count * 2, 256, 0, c->stream>>>(c->ctl, (const unsigned long long*)c->explicit_idx, n,
                                                                      c->grid_u8, c->list[0]);
        else
            k_seed_explicit_tile<<<c->sm_count * 2, 256, 0, c->stream>>>(c->ctl, (const unsigned long long*)c->explicit_idx, n,
                                                                        c->geom, grow_tile_words(), c->G[0], c->G[1], c->stamp, c->list[0]);
        c->launches++;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (c->storage == 0) k_seed_close<<<1, 1, 0, c->stream>>>(c->ctl);
    else k_seed_close_tile<<<1, 1, 0, c->stream>>>(c->ctl);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
