// seed.cu -- seeding and seed spacing by the L1 "diamond".
//
// Candidates: voxel v is a candidate core iff philox(seed; v>>2)[v&3] < T_core (R9).  They are marked in a
// 2-bit-per-voxel status map (00 = no candidate / rejected, 01 = pending, 11 = accepted); prefix sums of the
// per-chunk counts give every candidate its RANK in ascending index order, and the list cand[rank] = voxel.
// Spacing (R11, R12): the sequential rule "scan candidates in ascending index, accept iff no accepted seed
// within L1 < s" is reproduced exactly:
//   a pending candidate looks at every LOWER-index candidate within L1 < s (its neighbours);
//   - any accepted one  -> it is rejected (final: that seed is accepted in the sequential scan too);
//   - else any pending  -> it waits (its fate depends on them);
//   - else              -> it is accepted (all lower-index candidates in range are rejected).
// States only move pending -> {rejected, accepted}, so reading neighbours that change meanwhile is safe, and the
// fixed point is the sequential result.  The dependency chains are long (about 140 links at 400^3: they sweep the
// grid in index order), so the fast path keeps the statuses in ONE CTA's shared memory (a link costs a
// shared-memory round trip, not an L2 one): k_spacing_adjacency lists each candidate's neighbours by rank,
// k_spacing_resolve_cta resolves 1024 ranks per pass.  Lists that do not fit fall back to rescan rounds over
// the global status map (k_spacing_resolve).
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
    c->count[0] = 0; c->count[1] = 0; c->count_back[0] = 0; c->count_back[1] = 0; c->claims = 0; c->n_cand = 0;
    c->pool_head = 0; c->pend3[0] = 0; c->pend3[1] = 0; c->pend3[2] = 0; c->spacing_slow = 0; c->spacing_rounds = 0;
    c->vox_count[0] = 0; c->vox_count[1] = 0; c->vox_overflow = 0; c->pending = 0;
}

// --- candidates: one thread per status word = 16 voxels = 4 Philox blocks -----------------------
// Also counts the candidates of every CHUNK of 8 status words (128 voxels): the prefix sum of these counts
// (k_seed_scan) gives every candidate its rank in ascending index order without sorting.
constexpr int kChunkWords = 8;

__device__ __forceinline__ uint32_t candidate_fields(uint32_t status_word) {      // bit 2k: voxel k of the word is a candidate
    return (status_word | (status_word >> 1)) & 0x55555555u;
}

__global__ void __launch_bounds__(256) k_seed_candidates(uint32_t* status2, uint32_t* ccount,
                                                          unsigned long long N, uint32_t T_core,
                                                          uint32_t always, uint32_t accept_all,
                                                          const uint16_t* __restrict__ blocked16, PhiloxKey key) {
    const unsigned long long n_words = (N + 15ull) / 16ull;
    const unsigned long long n_padded = (n_words + 31ull) / 32ull * 32ull;      // whole warps: the chunk shuffles need every lane
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < n_padded;
         w += (unsigned long long)gridDim.x * blockDim.x) {
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
            if (blocked16) bits &= ~(uint32_t)blocked16[w];  // cells of earlier phases are not unassigned (PAPER.md:40 step 4)
            uint32_t word = 0;                              // spread: bit k -> field 2k
            for (uint32_t m = bits; m; m &= m - 1) {
                const int k = __ffs(m) - 1;
                word |= (accept_all ? 3u : 1u) << (2 * k);
            }
            status2[w] = word;
        }
        uint32_t cnt = __popc(bits);                        // the 8 lanes of a chunk add up their counts
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 1);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 2);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 4);
        if ((threadIdx.x & (kChunkWords - 1)) == 0) ccount[w / kChunkWords] = cnt;
    }
}

// chunk counts -> exclusive prefix sums (in place), total -> ctl->n_cand.  One cooperative launch: per-CTA sums,
// grid-wide sync, then every CTA scans its own contiguous segment tile by tile.
__global__ void __launch_bounds__(1024) k_seed_scan(Control* ctl, uint32_t* ccount, uint32_t* block_sums,
                                                     unsigned long long n_chunks) {
    cg::grid_group grid = cg::this_grid();
    __shared__ uint32_t s_scan[33];
    const unsigned long long per_cta = (n_chunks + gridDim.x - 1) / gridDim.x;
    const unsigned long long lo = min(n_chunks, per_cta * blockIdx.x), hi = min(n_chunks, lo + per_cta);
    uint32_t sum = 0;
    for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x) sum += ccount[i];
    uint32_t total;
    block_exclusive_scan(sum, s_scan, &total);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
    grid.sync();
    uint32_t before = 0, all = 0;                           // candidates in lower CTAs' segments / in all
    for (uint32_t b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
        const uint32_t v = ld_cg(block_sums + b);
        all += v;
        if (b < blockIdx.x) before += v;
    }
    uint32_t t0, t1;
    block_exclusive_scan(before, s_scan, &t0);
    block_exclusive_scan(all, s_scan, &t1);
    if (blockIdx.x == 0 && threadIdx.x == 0) ctl->n_cand = t1;
    uint32_t base = t0;
    for (unsigned long long i0 = lo; i0 < hi; i0 += blockDim.x) {
        const unsigned long long i = i0 + threadIdx.x;
        const uint32_t v = i < hi ? ccount[i] : 0u;
        const uint32_t excl = block_exclusive_scan(v, s_scan, &total);
        if (i < hi) ccount[i] = base + excl;
        base += total;
    }
}

// the candidates in ascending index order: cand[rank] = voxel index
__global__ void __launch_bounds__(256) k_seed_list(const uint32_t* __restrict__ status2, const uint32_t* __restrict__ coff,
                                                    uint32_t* __restrict__ cand, unsigned long long N) {
    const unsigned long long n_words = (N + 15ull) / 16ull;
    const unsigned long long n_padded = (n_words + 31ull) / 32ull * 32ull;      // whole warps: the chunk shuffles need every lane
    for (unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; w < n_padded;
         w += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t f = w < n_words ? candidate_fields(status2[w]) : 0u;
        const uint32_t cnt = __popc(f);
        uint32_t incl = cnt;                                // prefix over the 8 lanes of the chunk
#pragma unroll
        for (int o = 1; o < kChunkWords; o <<= 1) {
            const uint32_t up = __shfl_up_sync(0xffffffffu, incl, o, kChunkWords);
            if ((threadIdx.x & (kChunkWords - 1)) >= (uint32_t)o) incl += up;
        }
        if (cnt) {
            uint32_t r = coff[w / kChunkWords] + incl - cnt;
            for (uint32_t m = f; m; m &= m - 1) cand[r++] = (uint32_t)(16ull * w) + (uint32_t)((__ffs(m) - 1) >> 1);
        }
    }
}

// rank (in ascending index order) of candidate voxel w
__device__ __forceinline__ uint32_t rank_of(const uint32_t* status2, const uint32_t* coff, uint32_t w) {
    const uint32_t word = w >> 4, first = word & ~(uint32_t)(kChunkWords - 1);
    uint32_t r = ld_cg(coff + (word / kChunkWords));
    for (uint32_t k = first; k < word; ++k) r += __popc(candidate_fields(ld_cg(status2 + k)));
    return r + __popc(candidate_fields(ld_cg(status2 + word)) & ((1u << (2 * (w & 15u))) - 1u));
}

// --- seed spacing -------------------------------------------------------------------------------
struct Dims { int nx, ny, nz, periodic; };      // periodic: bit 0 = x wraps, bit 1 = y, bit 2 = z (R5)

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

// whole = true walks every voxel of the diamond (limit = N: no index cut), v itself included
template <class F>
__device__ __forceinline__ void scan_diamond(const uint32_t* status2, uint32_t v, const Dims& g, int s,
                                             uint32_t lane, F& on_word, bool whole = false, unsigned long long n_all = 0ull) {
    const unsigned long long limit = whole ? n_all : (unsigned long long)v;
    const int x = (int)(v % (uint32_t)g.nx);
    const uint32_t rest = v / (uint32_t)g.nx;
    const int y = (int)(rest % (uint32_t)g.ny), z = (int)(rest / (uint32_t)g.ny);
    const int r = s - 1;                                    // diamond radius: L1 <= s-1  <=>  L1 < s
    const int side = 2 * r + 1;
    // without any wrap-around, lower-index voxels have dz < 0, or dz = 0 and dy <= 0; with a periodic axis the whole
    // diamond is walked and `limit` (on_word sees indices below v only) keeps the lower ones
    const int px = g.periodic & 1, py = g.periodic & 2, pz = g.periodic & 4;
    const int n_rows = (g.periodic || whole) ? side * side : (r + 1) * side;
    for (int j = (int)lane; j < n_rows; j += 32) {
        const int dz = j / side - r, dy = j % side - r;
        const int rem = r - abs(dz) - abs(dy);
        if (rem < 0) continue;
        int Y = y + dy, Z = z + dz;
        if (!g.periodic && !whole && dz == 0 && dy > 0) continue;
        if (py) { Y %= g.ny; if (Y < 0) Y += g.ny; } else if (Y < 0 || Y >= g.ny) continue;
        if (pz) { Z %= g.nz; if (Z < 0) Z += g.nz; } else if (Z < 0 || Z >= g.nz) continue;
        const unsigned long long row = ((unsigned long long)Z * g.ny + Y) * (unsigned long long)g.nx;
        int xa = x - rem, xb = x + rem;
        if (px && 2 * rem + 1 >= g.nx) {                    // the range covers the whole row
            scan_segment(status2, row, row + g.nx - 1, limit, on_word);
        } else if (!px) {                                   // clipped at the walls
            xa = xa < 0 ? 0 : xa;
            xb = xb >= g.nx ? g.nx - 1 : xb;
            scan_segment(status2, row + xa, row + xb, limit, on_word);
        } else {                                            // wrapped range, at most two segments
            if (xa < 0) {
                scan_segment(status2, row + (xa + g.nx), row + g.nx - 1, limit, on_word);
                xa = 0;
            }
            if (xb >= g.nx) {
                scan_segment(status2, row, row + (xb - g.nx), limit, on_word);
                xb = g.nx - 1;
            }
            scan_segment(status2, row + xa, row + xb, limit, on_word);
        }
    }
}

// layout of the candidate buffer (capacity N words):
//   cand[n] | off[n] | cnt[n] | st_rank[n] | first8[8][n] | pool[N-12n]
// first8[e][i] = rank of the e-th listed neighbour of candidate i (struct of arrays: a warp's loads are coalesced);
// pool holds every list in full (lists longer than 8 continue there)
struct AdjView {
    bool ok;
    uint32_t *off, *cnt, *st_rank, *first8, *pool;
    unsigned long long pool_cap;
};
__device__ __forceinline__ AdjView adj_view(uint32_t* cand, uint32_t n, unsigned long long N) {
    AdjView a;
    a.ok = 12ull * n <= N;
    a.off = cand + n; a.cnt = cand + 2ull * n; a.st_rank = cand + 3ull * n; a.first8 = cand + 4ull * n; a.pool = cand + 12ull * n;
    a.pool_cap = a.ok ? N - 12ull * n : 0ull;
    return a;
}

// Ranks of the statuses kept in shared memory by k_spacing_resolve_cta: a ring of kRing candidates.  A candidate only
// looks at candidates at most (candidates in s-1 slices) ranks below it; k_spacing_adjacency checks that this fits.
constexpr uint32_t kRing = 1u << 17;             // one status byte per candidate: plain byte stores, no shared-memory atomics
// (kRing / kHead are the defaults; the sizes are kernel arguments so that a test can shrink them until the ring wraps
// after a few thousand candidates: liets_debug_spacing_ring)
// On a periodic grid the candidates of the last slices also look at those of the first slices (ranks near 0): the
// statuses of the first kHead ranks are kept for the whole run, next to the ring.
constexpr uint32_t kHead = 1u << 16;

// rowoff[rho] = number of candidates below row rho = y + ny z (rowoff[ny nz] = all): the candidates of any run of
// consecutive rows are a run of consecutive ranks
__global__ void __launch_bounds__(256) k_seed_rows(const Control* ctl, const uint32_t* status2, const uint32_t* coff,
                                                    uint32_t* rowoff, Dims g) {
    const unsigned long long n_rows = (unsigned long long)g.ny * g.nz;
    for (unsigned long long rho = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; rho <= n_rows;
         rho += (unsigned long long)gridDim.x * blockDim.x)
        rowoff[rho] = rho < n_rows ? rank_of(status2, coff, (uint32_t)(rho * g.nx)) : ctl->n_cand;
}

// key of voxel v in the keyed acceptance order (R19): word v % 4 of Philox at counter (v / 4, 0, 1, 2^32 - 1)
__device__ __forceinline__ uint32_t seed_priority(uint32_t v, const PhiloxKey& key) {
    const uint4 r = philox4x32_10(v >> 2, 0u, 1u, 0xFFFFFFFFu, key);
    const uint32_t w = v & 3u;
    return w == 0u ? r.x : w == 1u ? r.y : w == 2u ? r.z : r.w;
}

// w is tried before v in the keyed order
__device__ __forceinline__ bool keyed_before(uint32_t kw, uint32_t w, uint32_t kv, uint32_t v) {
    return kw < kv || (kw == kv && w < v);
}

// Pass 1: one warp per candidate (rank i, ascending index order) lists the RANKS of the lower-index candidates
// within L1 < s, once: one lane per z-slice of the diamond, which walks the candidates of the slice's rows
// (consecutive ranks) and keeps those in range.  Sets ctl->spacing_slow if a list does not fit or a neighbour is
// too far back in rank for the ring of k_spacing_resolve_cta.
// KEYED (R19): the candidates that come BEFORE i in the keyed order, anywhere in the diamond (no rank window: the
// lists go to k_spacing_resolve_lists).
template <bool KEYED>
__global__ void __launch_bounds__(256) k_spacing_adjacency(Control* ctl, const uint32_t* __restrict__ rowoff, uint32_t* cand,
                                                            Dims g, int s, unsigned long long N, uint32_t ring, uint32_t head,
                                                            PhiloxKey key) {
    __shared__ uint32_t s_buf[8][kAdjBuf];
    __shared__ uint32_t s_cnt[8];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t warp_global = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n = ctl->n_cand;
    const AdjView a = adj_view(cand, n, N);
    if (!a.ok) { if (threadIdx.x == 0 && blockIdx.x == 0) ctl->spacing_slow = 1u; return; }
    const int r = s - 1;                                    // diamond radius: L1 <= s-1  <=>  L1 < s
    // slices to visit: dz = -r..0 between walls (lower index = lower z, or same z and lower row), all slices within r
    // on the torus (each once)
    const int px = g.periodic & 1, py = g.periodic & 2, pz = g.periodic & 4;
    const int n_slices = pz ? min(2 * r + 1, g.nz) : (KEYED ? 2 * r + 1 : r + 1);
    for (uint32_t i = warp_global; i < n; i += n_warps) {
        const uint32_t v = cand[i];
        const uint32_t kv = KEYED ? seed_priority(v, key) : 0u;
        const int x = (int)(v % (uint32_t)g.nx);
        const uint32_t rest = v / (uint32_t)g.nx;
        const int y = (int)(rest % (uint32_t)g.ny), z = (int)(rest / (uint32_t)g.ny);
        if (lane == 0) s_cnt[warp] = 0;
        __syncwarp();
        for (int t = (int)lane; t < n_slices; t += 32) {
            int Z = z - r + t, dz;
            if (pz) {
                if (n_slices == g.nz) Z = t;                // the diamond covers every slice
                Z %= g.nz; if (Z < 0) Z += g.nz;
                dz = abs(Z - z); dz = min(dz, g.nz - dz);
            } else {
                if (Z < 0 || Z >= g.nz) continue;
                dz = abs(z - Z);
            }
            const int rho = r - dz;                         // rows y - rho .. y + rho of slice Z can hold neighbours
            if (rho < 0) continue;
            int ya = y - rho, yb = y + rho;
            int run_lo[2], run_hi[2], n_runs = 1;           // row runs [lo, hi] inside the slice
            if (!py) {
                run_lo[0] = max(ya, 0); run_hi[0] = min(yb, g.ny - 1);
                if (!KEYED && Z == z && !g.periodic) run_hi[0] = min(run_hi[0], y);   // same slice, no wrap anywhere: only rows up to the candidate's own
            } else if (2 * rho + 1 >= g.ny) {
                run_lo[0] = 0; run_hi[0] = g.ny - 1;
            } else {
                ya = (ya % g.ny + g.ny) % g.ny; yb = (yb % g.ny + g.ny) % g.ny;
                if (ya <= yb) { run_lo[0] = ya; run_hi[0] = yb; }
                else { run_lo[0] = 0; run_hi[0] = yb; run_lo[1] = ya; run_hi[1] = g.ny - 1; n_runs = 2; }
            }
            for (int q = 0; q < n_runs; ++q) {
                const uint32_t row0 = (uint32_t)Z * (uint32_t)g.ny;
                const uint32_t r0 = rowoff[row0 + run_lo[q]];
                const uint32_t r1 = KEYED ? rowoff[row0 + run_hi[q] + 1] : min(rowoff[row0 + run_hi[q] + 1], i);   // (index order: ranks below i only)
                for (uint32_t k = r0; k < r1; ++k) {
                    const uint32_t w = cand[k];
                    const int wx = (int)(w % (uint32_t)g.nx);
                    const int wy = (int)((w / (uint32_t)g.nx) % (uint32_t)g.ny);
                    int dx = abs(wx - x), dy = abs(wy - y);
                    if (px) dx = min(dx, g.nx - dx);
                    if (py) dy = min(dy, g.ny - dy);
                    if (dx + dy + dz <= r) {
                        if (KEYED && (k == i || !keyed_before(seed_priority(w, key), w, kv, v))) continue;
                        const uint32_t slot = atomicAdd(&s_cnt[warp], 1u);
                        if (slot < (uint32_t)kAdjBuf) s_buf[warp][slot] = k;
                    }
                }
            }
        }
        __syncwarp();
        const uint32_t k = s_cnt[warp];
        unsigned long long base = 0;
        bool stored = k <= (uint32_t)kAdjBuf;
        if (stored && k) {
            if (lane == 0) base = atomicAdd(&ctl->pool_head, (unsigned long long)k);
            base = __shfl_sync(0xffffffffu, base, 0);
            stored = base + k <= a.pool_cap;
        }
        if (stored) {
            bool far = false;
            for (uint32_t e = lane; e < k; e += 32) {
                const uint32_t rk = s_buf[warp][e];
                a.pool[base + e] = rk;
                if (e < 8u) a.first8[(unsigned long long)e * n + i] = rk;
                // the resolve re-arms the ring slots of a whole pass (1024 ranks) at once: rk's slot must survive until
                // the END of i's pass, not just until i
                if (!KEYED) far = far || ((i | 1023u) - rk >= ring && rk >= head);
            }
            if (far) ctl->spacing_slow = 1u;
            if (lane == 0) { a.off[i] = (uint32_t)base; a.cnt[i] = k; }
        } else if (lane == 0) {
            ctl->spacing_slow = 1u;
        }
        __syncwarp();
    }
}

__device__ __forceinline__ uint32_t status_of(const uint32_t* status2, uint32_t v) {
    return (ld_cg(status2 + (v >> 4)) >> (2 * (v & 15u))) & 3u;
}

// Pass 2: ONE CTA resolves all candidates in ascending rank, 1024 at a time, with the statuses (one byte: 1 pending,
// 3 accepted, 0 rejected) in shared memory, so a link of a dependency chain costs a shared-memory round trip
// instead of an L2 one (the chains are long: ~140 links at 400^3, they sweep the whole grid in index order).
// A pending candidate is rejected as soon as a lower-rank neighbour is accepted, accepted once none of them is
// pending, else it waits; neighbours of lower passes are already final.  The adjacency of the next passes is loaded
// while the current one is resolved.  The final statuses go to st_rank (2 bits per candidate, by rank) for finalize.
__global__ void __launch_bounds__(1024, 1) k_spacing_resolve_cta(Control* ctl, uint32_t* cand, unsigned long long N,
                                                                 uint32_t ring, uint32_t head) {
    extern __shared__ uint8_t s_st_raw[];                   // ring + head status bytes: 1 pending, 3 accepted, 0 rejected
    volatile uint8_t* const s_st = s_st_raw;                // read afresh in every look: other warps write them meanwhile
    if (ctl->spacing_slow) return;
    const uint32_t n = ctl->n_cand;
    const AdjView a = adj_view(cand, n, N);
    uint8_t* const st_rank = reinterpret_cast<uint8_t*>(a.st_rank);    // n bytes of the n-word region
    const uint32_t tid = threadIdx.x;
    const uint32_t kMask = ring - 1u;                       // ring is a power of two >= 2048
    // the next pass's lists (count, offset, first 8 ranks: coalesced) are loaded while this pass is resolved
    uint32_t kB = 0, offB = 0, nbrB[8] = { 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u };
    auto load = [&](uint32_t i) {
        kB = 0; offB = 0;
        if (i < n) {
            kB = a.cnt[i]; offB = a.off[i];
#pragma unroll
            for (int e = 0; e < 8; ++e) nbrB[e] = a.first8[(unsigned long long)e * n + i];
        }
    };
    load(tid);
    for (uint32_t i0 = 0; i0 < n; i0 += 1024u) {
        const uint32_t i = i0 + tid;
        const uint32_t k = kB, off = offB;
        uint32_t slot[8];                                   // ring slot of each neighbour's status
#pragma unroll
        for (int e = 0; e < 8; ++e) slot[e] = nbrB[e] < head ? ring + nbrB[e] : (nbrB[e] & kMask);
        s_st[i & kMask] = 1u;                               // this pass's slots of the ring: all pending
        if (i < head) s_st[ring + i] = 1u;
        load(i + 1024u);                                    // in flight while this pass is resolved
        __syncthreads();
        // every warp keeps looking until its 32 candidates are resolved -- no CTA barrier inside: a link of a chain costs
        // one shared-memory round trip.  Progress: a candidate only waits for lower ranks, all of them resident here.
        bool open = i < n;
        while (__any_sync(0xffffffffu, open)) {
            if (open) {
                uint32_t st[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) st[e] = s_st[slot[e]];         // independent loads (unused slots: any valid byte)
                bool accepted = false, pending = false;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    accepted = accepted || ((uint32_t)e < k && st[e] == 3u);
                    pending = pending || ((uint32_t)e < k && st[e] == 1u);
                }
                if (k > 8u && !accepted && !pending) {      // long lists: the rest from the pool (global memory), only once the
                    for (uint32_t e = 8; e < k; ++e) {      // first 8 are all rejected -- a pending one makes the candidate wait anyway
                        const uint32_t r = a.pool[off + e];
                        const uint32_t sv = s_st[r < head ? ring + r : (r & kMask)];
                        accepted = accepted || sv == 3u;
                        pending = pending || sv == 1u;
                    }
                }
                if (accepted || !pending) {                 // pending -> rejected (0) / accepted (3)
                    const uint8_t fin = accepted ? 0u : 3u;
                    s_st[i & kMask] = fin;
                    if (i < head) s_st[ring + i] = fin;
                    open = false;
                }
            }
        }
        if (i < n) st_rank[i] = s_st[i & kMask];            // final statuses by rank
        __syncthreads();                                    // the pass is final before the next one starts
    }
}

// Slow path (lists that do not fit, extreme densities): every pending candidate rescans its diamond in the global
// status map each round; all rounds in one cooperative launch.  Does nothing unless ctl->spacing_slow is set.
__global__ void __launch_bounds__(1024) k_spacing_resolve(Control* ctl, uint32_t* status2, uint32_t* cand,
                                                           Dims g, int s, unsigned long long N) {
    cg::grid_group grid = cg::this_grid();
    if (!ctl->spacing_slow) return;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, n_threads = gridDim.x * blockDim.x;
    const uint32_t n = ctl->n_cand;
    for (uint32_t round = 0;; ++round) {
        uint32_t still = 0;
        for (uint32_t i = tid >> 5; i < n; i += n_threads >> 5) {      // one warp per candidate
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
        if (lane == 0 && still) atomicAdd(&ctl->pend3[round % 3u], still);
        grid.sync();
        const uint32_t left = ld_cg(&ctl->pend3[round % 3u]);
        if (tid == 0) ctl->pend3[(round + 2u) % 3u] = 0;               // next used in round+2, after another sync
        if (left == 0) break;
    }
}

// --- keyed acceptance order (R19) ---------------------------------------------------------
// The same candidates, tried in ascending (key, index), key(v) = word v % 4 of Philox at counter (v / 4, 0, 1, 2^32 - 1): a
// random order fixed by the seed.  The order has no spatial structure, so there are no rank windows to exploit: every
// pending candidate rescans its WHOLE diamond in the global status map each round and evaluates the key of every
// candidate it meets; the dependency chains are short (a handful of rounds instead of a sweep through the grid).
// Keyed order, fast path: the lists of k_spacing_adjacency<true> hold, for every candidate, the candidates tried before it
// within its diamond.  Rounds over all candidates with the statuses by rank in global memory (1 pending, 3 accepted,
// 0 rejected; the layout seed_accepted reads): the chains are a handful of links long, so a link may cost an L2 round trip.
__global__ void __launch_bounds__(1024) k_spacing_resolve_lists(Control* ctl, uint32_t* cand, unsigned long long N) {
    cg::grid_group grid = cg::this_grid();
    if (ctl->spacing_slow) return;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, n_threads = gridDim.x * blockDim.x;
    const uint32_t n = ctl->n_cand;
    const AdjView a = adj_view(cand, n, N);
    uint8_t* const st = reinterpret_cast<uint8_t*>(a.st_rank);
    for (uint32_t i = tid; i < n; i += n_threads) st[i] = 1u;
    grid.sync();
    for (uint32_t round = 0;; ++round) {
        uint32_t still = 0;
        for (uint32_t i = tid; i < n; i += n_threads) {
            if (__ldcg(st + i) != 1u) continue;
            const uint32_t k = a.cnt[i], off = a.off[i];
            bool accepted = false, pending = false;
            for (uint32_t e = 0; e < k; ++e) {
                const uint32_t sv = __ldcg(st + a.pool[off + e]);
                accepted = accepted || sv == 3u;
                pending = pending || sv == 1u;
            }
            if (accepted) st[i] = 0u;
            else if (!pending) st[i] = 3u;
            else still++;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) still += __shfl_xor_sync(0xffffffffu, still, o);
        if (lane == 0 && still) atomicAdd(&ctl->pend3[round % 3u], still);
        grid.sync();
        const uint32_t left = ld_cg(&ctl->pend3[round % 3u]);
        if (tid == 0) { ctl->pend3[(round + 2u) % 3u] = 0; ctl->spacing_rounds = round + 1u; }
        if (left == 0) break;
    }
}

__global__ void __launch_bounds__(1024) k_spacing_resolve_keyed(Control* ctl, uint32_t* status2, uint32_t* cand,
                                                                 Dims g, int s, unsigned long long N, PhiloxKey key) {
    cg::grid_group grid = cg::this_grid();
    if (!ctl->spacing_slow) return;                         // the lists fitted: k_spacing_resolve_lists has done it
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, n_threads = gridDim.x * blockDim.x;
    const uint32_t n = ctl->n_cand;
    for (uint32_t round = 0;; ++round) {
        uint32_t still = 0;
        for (uint32_t i = tid >> 5; i < n; i += n_threads >> 5) {      // one warp per candidate
            const uint32_t v = cand[i];
            if (status_of(status2, v) != 1u) continue;
            const uint32_t kv = seed_priority(v, key);
            bool accepted = false, pending = false;
            auto look = [&](uint32_t word, unsigned long long lo) {
                uint32_t f = word & 0x55555555u;            // candidates that are pending or accepted
                while (f) {
                    const uint32_t b = (uint32_t)__ffs(f) - 1u;
                    f &= f - 1u;
                    const uint32_t w = (uint32_t)lo + (b >> 1);
                    if (w == v) continue;
                    const uint32_t kw = seed_priority(w, key);
                    if (kw < kv || (kw == kv && w < v)) {   // w is tried before v
                        if ((word >> (b + 1u)) & 1u) accepted = true;
                        else pending = true;
                    }
                }
            };
            scan_diamond(status2, v, g, s, lane, look, true, N);
            accepted = __any_sync(0xffffffffu, accepted);
            pending = __any_sync(0xffffffffu, pending);
            if (lane == 0) {
                if (accepted) atomicAnd(status2 + (v >> 4), ~(1u << (2 * (v & 15u))));
                else if (!pending) atomicOr(status2 + (v >> 4), 2u << (2 * (v & 15u)));
                else still++;
            }
        }
        if (lane == 0 && still) atomicAdd(&ctl->pend3[round % 3u], still);
        grid.sync();
        const uint32_t left = ld_cg(&ctl->pend3[round % 3u]);
        if (tid == 0) { ctl->pend3[(round + 2u) % 3u] = 0; ctl->spacing_rounds = round + 1u; }
        if (left == 0) break;
    }
}

// --- the spacing filter by dense diamond dilation (Fig. 1(D)) ------------------
// The paper's mechanism -- repeated passes of a small kernel over the whole grid -- on bit rows (x-rows of Wp 64-bit
// words), giving exactly the seeds of the ascending-index rule (R12) between walls.  Per round:
//   LB  = the pending cells dilated by the "later half" of the diamond, D+ = { d != 0 : L1(d) <= s-1, d after 0 in index
//         order } = (e_z + (s-2) passes of {0, +-x, +-y, +z}) U (e_y + (s-2) passes of {0, +-x, +y}) U (e_x + (s-2) passes of
//         {0, +x}): a cell of LB has a pending candidate of lower index within its diamond;
//   NEW = pending & ~LB: nothing of lower index can still cover them -- accepted;
//   BL  = NEW dilated by s-1 passes of the full 6-neighbour kernel; pending &= ~BL.
// A round costs 2 (s-1) + 2 sweeps of the bit grid, and the number of rounds is the length of the longest dependency
// chain in index order: this is the cost the candidate-list form (k_spacing_adjacency / k_spacing_resolve_cta) avoids.
struct DenseGeom { int nx, ny, nz, Wp; };
enum : uint32_t { kDilC = 1u, kDilXm = 2u, kDilXp = 4u, kDilYm = 8u, kDilYp = 16u, kDilZm = 32u, kDilZp = 64u };   // out(u) |= in(u), in(u - ex), in(u + ex), ..
struct DensePass { int n; const unsigned long long* in[3]; unsigned long long* out[3]; uint32_t flags[3]; };

__global__ void __launch_bounds__(256) k_dense_pass(DensePass p, DenseGeom g) {
    const unsigned long long n_words = (unsigned long long)g.Wp * g.ny * g.nz;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const int w = (int)(i % (unsigned long long)g.Wp);
        const unsigned long long rowi = i / (unsigned long long)g.Wp;
        const int y = (int)(rowi % (unsigned long long)g.ny), z = (int)(rowi / (unsigned long long)g.ny);
        const int nvalid = min(64, g.nx - 64 * w);
        const unsigned long long valid = nvalid >= 64 ? ~0ull : (nvalid <= 0 ? 0ull : ~(~0ull << nvalid));
        const unsigned long long slice = (unsigned long long)g.Wp * g.ny;
        for (int c = 0; c < p.n; ++c) {
            const unsigned long long* in = p.in[c];
            const uint32_t f = p.flags[c];
            const unsigned long long me = in[i];
            unsigned long long o = (f & kDilC) ? me : 0ull;
            if (f & kDilXm) o |= (me << 1) | (w > 0 ? in[i - 1] >> 63 : 0ull);              // in(u - ex)
            if (f & kDilXp) o |= (me >> 1) | (w + 1 < g.Wp ? in[i + 1] << 63 : 0ull);       // in(u + ex)
            if ((f & kDilYm) && y > 0) o |= in[i - g.Wp];
            if ((f & kDilYp) && y + 1 < g.ny) o |= in[i + g.Wp];
            if ((f & kDilZm) && z > 0) o |= in[i - slice];
            if ((f & kDilZp) && z + 1 < g.nz) o |= in[i + slice];
            p.out[c][i] = o & valid;
        }
    }
}

// pending candidates (status 01) as bit rows; the accepted set starts empty
__global__ void __launch_bounds__(256) k_dense_init(const uint32_t* __restrict__ status2, DenseGeom g, unsigned long long* P,
                                                     unsigned long long* ACC) {
    const unsigned long long n_words = (unsigned long long)g.Wp * g.ny * g.nz;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const int w = (int)(i % (unsigned long long)g.Wp);
        const unsigned long long rowi = i / (unsigned long long)g.Wp;
        const int nvalid = min(64, g.nx - 64 * w);
        unsigned long long bits = 0ull;
        for (int b = 0; b < nvalid; ++b) {
            const unsigned long long v = rowi * (unsigned long long)g.nx + (unsigned long long)(64 * w + b);
            if (((status2[v >> 4] >> (2u * (uint32_t)(v & 15ull))) & 3u) == 1u) bits |= 1ull << b;
        }
        P[i] = bits;
        ACC[i] = 0ull;
    }
}

// NEW = P & ~(LBz | LBy | LBx); ACC |= NEW
__global__ void __launch_bounds__(256) k_dense_accept(const unsigned long long* P, const unsigned long long* LBz,
                                                       const unsigned long long* LBy, const unsigned long long* LBx,
                                                       unsigned long long* NEW, unsigned long long* ACC, unsigned long long n_words) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long nw = P[i] & ~(LBz[i] | LBy[i] | LBx[i]);
        NEW[i] = nw;
        if (nw) ACC[i] |= nw;
    }
}

// P &= ~BL; *left += popc(P)
__global__ void __launch_bounds__(256) k_dense_prune(unsigned long long* P, const unsigned long long* BL, unsigned long long n_words,
                                                      uint32_t* left) {
    uint32_t cnt = 0;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long v = P[i] & ~BL[i];
        P[i] = v;
        cnt += (uint32_t)__popcll(v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31u) == 0u && cnt) atomicAdd(left, cnt);
}

// the accepted set back into the status map (11 accepted, 00 rejected), by candidate
__global__ void __launch_bounds__(256) k_dense_finish(Control* ctl, uint32_t* status2, const uint32_t* cand, DenseGeom g,
                                                       const unsigned long long* ACC, uint32_t rounds) {
    const uint32_t n = ctl->n_cand;
    if (blockIdx.x == 0 && threadIdx.x == 0) { ctl->spacing_slow = 1u; ctl->spacing_rounds = rounds; }
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t v = cand[i];
        const uint32_t x = v % (uint32_t)g.nx;
        const unsigned long long rowi = v / (uint32_t)g.nx;
        const bool acc = (ACC[rowi * (unsigned long long)g.Wp + (x >> 6)] >> (x & 63u)) & 1ull;
        if (acc) atomicOr(status2 + (v >> 4), 2u << (2 * (v & 15u)));
        else atomicAnd(status2 + (v >> 4), ~(3u << (2 * (v & 15u))));
    }
}

// --- finalize: accepted candidates -> grid + initial front A_0 = seeds (R3) ---------------------
// accepted = status 11: by rank in the spacing fast path's st_rank, else by voxel in the global status map
__device__ __forceinline__ bool seed_accepted(const Control* ctl, const uint32_t* status2, const uint32_t* cand,
                                              uint32_t n, unsigned long long N, uint32_t spaced, uint32_t i, uint32_t v) {
    if (spaced && !ctl->spacing_slow) {
        const uint8_t* st_rank = reinterpret_cast<const uint8_t*>(cand + 3ull * n);     // AdjView::st_rank, one byte per rank
        return st_rank[i] == 3u;
    }
    return ((status2[v >> 4] >> (2u * (v & 15u))) & 3u) == 3u;
}

__global__ void __launch_bounds__(256) k_seed_finalize_u8(Control* ctl, const uint32_t* status2,
                                                           const uint32_t* cand, uint8_t* grid,
                                                           uint32_t* front, unsigned long long N, uint32_t spaced) {
    __shared__ uint32_t s_scan[33];
    __shared__ uint32_t s_base;
    const uint32_t n = ctl->n_cand;
    for (uint64_t base = (uint64_t)blockIdx.x * blockDim.x; base < n; base += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = base + threadIdx.x;
        uint32_t v = 0, acc = 0;
        if (i < n) {
            v = cand[i];
            acc = seed_accepted(ctl, status2, cand, n, N, spaced, (uint32_t)i, v);
        }
        uint32_t total;
        uint32_t off = block_exclusive_scan(acc, s_scan, &total);
        if (threadIdx.x == 0) s_base = total ? atomicAdd(&ctl->count[0], total) : 0u;
        __syncthreads();
        if (acc) { front[s_base + off] = v; grid[v] = 1; }
    }
}

__global__ void k_seed_close(Control* c) { c->n_solid = c->count[0]; c->cur = 0; c->mode = 1; c->pending = 0; }

// STORAGE_TILE: set the seed's bit in both grid copies; A_0 = seeds as a voxel list (grow_vox.cu; a list that does
// not fit only raises the overflow flag, and step 0 starts on tiles).  The 0 -> 1 transition of the bit in G0 dedupes
// explicit seeds and counts them.
__device__ __forceinline__ void place_seed_tile(Control* ctl, uint32_t v, TileGeom g, unsigned long long* G0,
                                                unsigned long long* G1, uint32_t* vox, uint32_t vox_cap) {
    const uint32_t x = v % (uint32_t)g.nx, rest = v / (uint32_t)g.nx;
    const uint32_t y = rest % (uint32_t)g.ny, z = rest / (uint32_t)g.ny;
    const unsigned long long w = (unsigned long long)(x >> 6) + (unsigned long long)g.Wp * ((unsigned long long)y + (unsigned long long)g.ny * z);
    const unsigned long long bit = 1ull << (x & 63u);
    const unsigned long long old = atomicOr(G0 + w, bit);
    atomicOr(G1 + w, bit);
    if (old & bit) return;
    atomicAdd(&ctl->n_solid, 1ull);
    const uint32_t slot = atomicAdd(&ctl->vox_count[0], 1u);
    if (slot < vox_cap) vox[slot] = v;
    else ctl->vox_overflow = 1u;
}

__global__ void __launch_bounds__(256) k_seed_finalize_tile(Control* ctl, const uint32_t* status2, const uint32_t* cand,
                                                             TileGeom g, unsigned long long* G0, unsigned long long* G1,
                                                             uint32_t* vox, uint32_t vox_cap, unsigned long long N, uint32_t spaced) {
    const uint32_t n = ctl->n_cand;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t v = cand[i];
        if (seed_accepted(ctl, status2, cand, n, N, spaced, (uint32_t)i, v)) place_seed_tile(ctl, v, g, G0, G1, vox, vox_cap);
    }
}

__global__ void k_seed_explicit_tile(Control* ctl, const unsigned long long* idx, unsigned long long n, TileGeom g,
                                     unsigned long long* G0, unsigned long long* G1, uint32_t* vox, uint32_t vox_cap) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (unsigned long long)gridDim.x * blockDim.x)
        place_seed_tile(ctl, (uint32_t)idx[i], g, G0, G1, vox, vox_cap);
}

__global__ void k_seed_close_tile(Control* c, uint32_t mode) { c->cur = 0; c->mode = mode; c->pending = 0; }

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
    } else {                                                // G[0], G[1], the stamps and the weights are contiguous
        e = cudaMemsetAsync(c->G[0], 0, c->grid_words * 16 + c->n_tiles * 8, c->stream);
    }
    if (e != cudaSuccess) return e;
    if (c->has_blocked && (e = launch_blocked_apply(c)) != cudaSuccess) return e;      // the earlier phases' cells go back in
    k_seed_reset<<<1, 1, 0, c->stream>>>(c->ctl);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_seed_candidates(liets_ctx* c, uint64_t t_core, int accept_all) {
    const PhiloxKey key = philox_make_key(c->rng_seed);
    const uint32_t always = t_core >= (1ull << 32);
    const uint32_t T = always ? 0xFFFFFFFFu : (uint32_t)t_core;
    k_seed_candidates<<<c->sm_count * 8, 256, 0, c->stream>>>(c->status2, c->coff, c->N, T, always, (uint32_t)accept_all,
                                                              c->has_blocked ? reinterpret_cast<const uint16_t*>(c->pbits) : nullptr, key);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // ranks: prefix sums of the chunk counts, then the candidate list in ascending index order
    Control* ctl = c->ctl;
    uint32_t* coff = c->coff;
    uint32_t* sums = c->ctl->scan_sums;
    unsigned long long n_chunks = (((c->N + 15ull) / 16ull + 31ull) / 32ull * 32ull) / (unsigned long long)kChunkWords;
    void* args[] = { &ctl, &coff, &sums, &n_chunks };
    const int scan_grid = c->sm_count < 1024 ? c->sm_count : 1024;
    e = cudaLaunchCooperativeKernel((const void*)k_seed_scan, dim3(scan_grid), dim3(1024), args, 0, c->stream);
    c->launches++;
    if (e != cudaSuccess) return e;
    k_seed_list<<<c->sm_count * 8, 256, 0, c->stream>>>(c->status2, c->coff, c->cand, c->N);
    c->launches++;
    return cudaGetLastError();
}

// exact parallel reproduction of the ascending-index greedy (R12): adjacency lists (ranks) once, then all
// candidates resolved in rank order by one CTA with the statuses in shared memory; a cooperative rescan kernel
// takes over only when the lists do not fit (it returns at once otherwise)
cudaError_t launch_spacing(liets_ctx* c, int s) {
    Dims g{ c->nx, c->ny, c->nz, c->periodic };
    unsigned long long N = c->N;
    k_seed_rows<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->coff, c->rowoff, g);
    c->launches++;
    const uint32_t ring = c->spacing_ring ? c->spacing_ring : kRing, head = c->spacing_ring ? c->spacing_head : kHead;
    k_spacing_adjacency<false><<<c->sm_count * 8, 256, 0, c->stream>>>(c->ctl, c->rowoff, c->cand, g, s, N, ring, head, PhiloxKey{});
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int ring_bytes = (int)(ring + head);
    k_spacing_resolve_cta<<<1, 1024, ring_bytes, c->stream>>>(c->ctl, c->cand, N, ring, head);
    c->launches++;
    e = cudaGetLastError();
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

// R19: the keyed order, all rounds in one cooperative launch
cudaError_t launch_spacing_keyed(liets_ctx* c, int s) {
    Dims g{ c->nx, c->ny, c->nz, c->periodic };
    unsigned long long N = c->N;
    PhiloxKey key = philox_make_key(c->rng_seed);
    if (c->resolve_keyed_grid == 0) {
        int per_sm = 0, per_sm_lists = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_spacing_resolve_keyed, 1024, 0);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_lists, k_spacing_resolve_lists, 1024, 0);
        if (e != cudaSuccess) return e;
        if (per_sm < 1 || per_sm_lists < 1) return cudaErrorLaunchOutOfResources;
        c->resolve_keyed_grid = c->sm_count;
    }
    // the candidates tried before each candidate, listed once; rounds over the lists; the rescan rounds only if they did not fit
    k_seed_rows<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->coff, c->rowoff, g);
    c->launches++;
    k_spacing_adjacency<true><<<c->sm_count * 8, 256, 0, c->stream>>>(c->ctl, c->rowoff, c->cand, g, s, N, 0u, 0u, key);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    void* largs[] = { &c->ctl, &c->cand, &N };
    e = cudaLaunchCooperativeKernel((const void*)k_spacing_resolve_lists, dim3(c->resolve_keyed_grid), dim3(1024), largs, 0, c->stream);
    c->launches++;
    if (e != cudaSuccess) return e;
    void* args[] = { &c->ctl, &c->status2, &c->cand, &g, &s, &N, &key };
    e = cudaLaunchCooperativeKernel((const void*)k_spacing_resolve_keyed, dim3(c->resolve_keyed_grid), dim3(1024), args, 0, c->stream);
    c->launches++;
    return e;
}

// NEXT-1: the dense diamond dilation (walls only, ascending index order).  n_cand: the candidate count (read back by the
// caller); the bit rows live behind the candidate list.  Synchronises once per round (the pending count).
size_t spacing_dense_bytes(const liets_ctx* c) {
    return (size_t)((c->nx + 63) / 64) * 8u * (size_t)c->ny * (size_t)c->nz;
}

cudaError_t launch_spacing_dense(liets_ctx* c, int s, uint32_t n_cand, uint32_t* rounds_out) {
    DenseGeom g{ c->nx, c->ny, c->nz, (c->nx + 63) / 64 };
    const unsigned long long n_words = (unsigned long long)g.Wp * g.ny * g.nz;
    const size_t plane = (size_t)n_words * 8u;
    uint8_t* base = reinterpret_cast<uint8_t*>(c->cand) + (((size_t)n_cand * 4u + 255u) & ~(size_t)255u);
    unsigned long long* B[8];
    for (int k = 0; k < 8; ++k) B[k] = reinterpret_cast<unsigned long long*>(base + (size_t)k * plane);
    unsigned long long *P = B[0], *ACC = B[1];
    const int r = s - 1;
    const int grid = c->sm_count * 8;
    uint32_t* left = &c->ctl->pend3[0];
    k_dense_init<<<grid, 256, 0, c->stream>>>(c->status2, g, P, ACC);
    c->launches++;
    uint32_t rounds = 0;
    for (;;) {
        // the three chains of the later half of the diamond, one sweep per pass: ping-pong between B[2..4] and B[5..7]
        DensePass p;
        p.n = 3;
        p.flags[0] = kDilZm; p.flags[1] = kDilYm; p.flags[2] = kDilXm;                       // the first step of each chain
        for (int k = 0; k < 3; ++k) { p.in[k] = P; p.out[k] = B[2 + k]; }
        k_dense_pass<<<grid, 256, 0, c->stream>>>(p, g);
        c->launches++;
        int cur = 0;                                        // chains now in B[2 + 3 cur ..]
        p.flags[0] = kDilC | kDilXm | kDilXp | kDilYm | kDilYp | kDilZm;
        p.flags[1] = kDilC | kDilXm | kDilXp | kDilYm;
        p.flags[2] = kDilC | kDilXm;
        for (int pass = 1; pass < r; ++pass) {
            for (int k = 0; k < 3; ++k) { p.in[k] = B[2 + 3 * cur + k]; p.out[k] = B[2 + 3 * (cur ^ 1) + k]; }
            k_dense_pass<<<grid, 256, 0, c->stream>>>(p, g);
            c->launches++;
            cur ^= 1;
        }
        unsigned long long* NEW = B[2 + 3 * (cur ^ 1)];
        k_dense_accept<<<grid, 256, 0, c->stream>>>(P, B[2 + 3 * cur], B[2 + 3 * cur + 1], B[2 + 3 * cur + 2], NEW, ACC, n_words);
        c->launches++;
        // the accepted cells cover their diamonds: s-1 passes of the full kernel
        DensePass q;
        q.n = 1;
        q.flags[0] = kDilC | kDilXm | kDilXp | kDilYm | kDilYp | kDilZm | kDilZp;
        unsigned long long* a = NEW;
        unsigned long long* b = B[2 + 3 * cur];
        for (int pass = 0; pass < r; ++pass) {
            q.in[0] = a; q.out[0] = b;
            k_dense_pass<<<grid, 256, 0, c->stream>>>(q, g);
            c->launches++;
            unsigned long long* t = a; a = b; b = t;
        }
        cudaError_t e = cudaMemsetAsync(left, 0, sizeof(uint32_t), c->stream);
        if (e != cudaSuccess) return e;
        k_dense_prune<<<grid, 256, 0, c->stream>>>(P, a, n_words, left);
        c->launches++;
        ++rounds;
        uint32_t h_left = 0;
        e = cudaMemcpyAsync(&h_left, left, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream);
        if (e != cudaSuccess) return e;
        e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return e;
        if (h_left == 0) break;
    }
    k_dense_finish<<<grid, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, g, ACC, rounds);
    c->launches++;
    if (rounds_out) *rounds_out = rounds;
    return cudaGetLastError();
}

// per-device function attributes, set once per context at liets_create (they are per device, not per process)
cudaError_t seed_kernel_attributes() {
    return cudaFuncSetAttribute(k_spacing_resolve_cta, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kRing + kHead));
}

cudaError_t launch_seed_finalize(liets_ctx* c, int spaced) {
    if (c->storage == 0)
        k_seed_finalize_u8<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, c->grid_u8, c->list[0], c->N, (uint32_t)spaced);
    else
        k_seed_finalize_tile<<<c->sm_count * 4, 256, 0, c->stream>>>(c->ctl, c->status2, c->cand, c->geom, c->G[0], c->G[1],
                                                                    c->vox[0], c->vox_cap, c->N, (uint32_t)spaced);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (c->storage == 0) k_seed_close<<<1, 1, 0, c->stream>>>(c->ctl);
    else k_seed_close_tile<<<1, 1, 0, c->stream>>>(c->ctl, c->storage == 2 ? 2u : 0u);
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
                                                                        c->geom, c->G[0], c->G[1], c->vox[0], c->vox_cap);
        c->launches++;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (c->storage == 0) k_seed_close<<<1, 1, 0, c->stream>>>(c->ctl);
    else k_seed_close_tile<<<1, 1, 0, c->stream>>>(c->ctl, c->storage == 2 ? 2u : 0u);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
