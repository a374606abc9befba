// grow_tile.cu -- STORAGE_TILE growth step: bit-packed x-rows + explicit list of active TILES.
//
// Layout in HBM.  The phase array is stored one bit per voxel in x-rows of Wp = ceil(nx/64) 64-bit
// words (bit i of word w of row (y, z) = voxel x = 64 w + i; bits with x >= nx stay 0).  Two copies
// G[0], G[1] are kept: step t reads G[t&1] (immutable during the step, so the update is synchronous
// by construction) and ORs into G[(t+1)&1].  The active set A is kept
// at two levels: in HBM a list of active TILES of kTileW words x 8 x 8 rows (128 x 8 x 8 voxels)
// that hold at least one front voxel, 4 bytes per 8192 voxels; and, per tile and step, the explicit
// list of its front VOXELS, rebuilt from the bits in shared memory.
//
// One CTA owns one tile at a time (tiles are handed out through an atomic cursor):
//   A  gather: the 10 x 10 rows of the tile's one-voxel neighbourhood, kTileW + 2 words each, as "not void"
//      bits (solid, outside the domain, or padding), kept as 18-bit windows at a stride of 16 voxels (window k of a
//      row = tile bits 16k-1 .. 16k+16 in word bits 14..31), so that the three x-neighbours of any voxel come out of
//      ONE word by a left shift of 15 - (x & 15), plus the x part of the front test per row
//   B  front voxels: solid cells with a void neighbour, 64 cells per bit operation;
//      their ids are compacted into a shared-memory list (popc + CTA-wide prefix sum).  A list entry is
//      (15 - (x & 15)) | (8 row + x / 16) << 4: the shift count and the window index, ready to use
//   C  one thread per front voxel, two consecutive list entries per thread in one branch-free block: the voxel's 26
//      void-target bits (Algorithm 3 lines 5-6) from nine window loads, each aligned by one multiply and pushed into the
//      mask by one funnel shift; ONE Philox4x32-10 block = the leading nibble of all 26 draws (R9), one carry-free
//      per-nibble compare (zero test / thresholds below 8 / general, chosen per launch) = the directions that fire or tie
//      with the threshold (line 8); level-0 hits go to a shared-memory claim volume, ties to a per-warp ring
//   D  one lane per ring entry and nibble level: the next block decides all tied directions of the voxel at once; a
//      round runs as soon as 32 entries wait, the few left at the tile's end are resolved two levels per round
//   E  claim + compact: own rows are OR-ed into G[next] together with the carried state, halo hits
//      go to the neighbour tiles' rows with atomicOr (all of a row's atomics in one batch); the returned old word tells
//      who flipped the bit (line 9-10, "counted once" PAPER.md:77) for the solid count; a per-tile step stamp
//      (atomicMax) makes every tile enter the next list exactly once; tiles without front voxels
//      are not re-emitted (lazy retirement).
// With INTERACT (liets_set_interaction, R20) the cells of earlier phases that have a void neighbour are front
// voxels too (bit 15 of their list entry), compared against the interaction thresholds.
#include "liets_host.h"

namespace liets {

namespace {

constexpr int kTileW = 2;                       // 64-bit words per tile row
constexpr int kThreads = 128;
#ifndef LIETS_TILE_CTAS
#define LIETS_TILE_CTAS 10
#endif
constexpr int kCtasPerSm = LIETS_TILE_CTAS;       // resident CTAs per SM the kernel is compiled for (registers) and launched with
constexpr int kWarps = kThreads / 32;
constexpr int kMaxBatch = 16;                   // grids per launch of the batched kernel (kernel parameters: 2.2 KB)
constexpr int kRowWords = kTileW + 2;           // left halo word | tile words | right halo word
constexpr int kWin = 64 * kTileW / 16;          // 18-bit windows per row, one per 16 voxels
#ifndef LIETS_QUEUE_CAP
#define LIETS_QUEUE_CAP 128
#endif
constexpr int kQueueCap = LIETS_QUEUE_CAP;      // tied voxels per warp queue (a ring; power of two, at least 64)
constexpr int kHeavyFront = 64 * 64 * kTileW / 8;  // a tile with at least this many front voxels (1/8 of its cells) is "heavy"
#ifndef LIETS_FRONT_CAP
#define LIETS_FRONT_CAP (32 * 64 * kTileW)
#endif
constexpr int kFrontCap = LIETS_FRONT_CAP;      // front voxels listed at a time (half the tile; more -> several passes)

struct Smem {
    uint32_t win[100 * kWin];                   // row (z'+1)*10 + (y'+1), window k: not-void bits of tile x = 16k-1 .. 16k+16 at bits 14..31
    unsigned long long vx[100][kTileW];         // per tile word: cells with a void cell at x-1, x or x+1 in the same row
    unsigned long long own[64][kTileW];         // the tile's own not-void words (row y + 8 z)
    uint32_t claims[100][2 * kRowWords];        // cells claimed in this step: row as in win, bit 64 + x of the row (32-bit view)
    uint32_t queue[kWarps][2 * kQueueCap];      // ring of (list entry | nibble level << 16, tied directions)
    uint32_t hpat[2][8][4];                     // [1]: the interaction thresholds (R20; only loaded when INTERACT)
    uint32_t dir[28];                           // direction d: claim-word offset 8 (10 dz + dy + 11) | (dx + 1) << 16
    uint32_t ptab[100];                         // voxel index of tile x = 0 of each own row
    uint32_t tile[2], tile_id[2];               // list entry handed to the CTA, double-buffered by tile parity
    uint32_t wsum[2][kWarps];                   // per-warp front-voxel counts, double-buffered
    alignas(4) uint16_t flist[kFrontCap];                  // (15 - (x & 15)) | (8 row + x / 16) << 4 of the tile's front voxels
};

struct TileCoord {
    int w0, y0, z0;                             // first word / row / slice of the tile
    int wcy, wcz;                               // valid rows / slices (< 8 on the high border)
};

// "not void" word of global row (y, z), global word index wg in [-1, Wp]: data inside the domain, the wrap or
// wall value at x = -1 and x = nx, ones beyond.  yz_ok = the row exists (after wrapping).
__device__ __forceinline__ unsigned long long not_void_word(const unsigned long long* __restrict__ G, const TileGeom& g,
                                                            bool yz_ok, unsigned long long row_base, int wg) {
    if (!yz_ok) return ~0ull;
    if (wg < 0) {                               // only bit 63 (x = -1) is ever looked at
        if (!(g.periodic & 1)) return ~0ull;
        const int xl = g.nx - 1;
        return ((__ldcg(G + row_base + (xl >> 6)) >> (xl & 63)) & 1ull) << 63;
    }
    const int xbase = 64 * wg;
    if (xbase > g.nx) return ~0ull;
    unsigned long long v = xbase < g.nx ? __ldcg(G + row_base + wg) : 0ull;
    if (xbase + 64 > g.nx) {                    // the row ends inside this word: halo bit at x = nx, ones above
        const int nvalid = g.nx - xbase;        // 0..63
        const unsigned long long halo = (g.periodic & 1) ? (__ldcg(G + row_base) & 1ull) : 1ull;
        v |= (~0ull << nvalid);
        if (!halo) v &= ~(1ull << nvalid);
    }
    return v;
}

__device__ __forceinline__ TileCoord tile_coord(uint32_t id, const TileGeom& g) {
    TileCoord tc;
    const uint32_t tx = id % (uint32_t)g.ntx, rest = id / (uint32_t)g.ntx;
    tc.w0 = (int)tx * kTileW;
    tc.y0 = 8 * (int)(rest % (uint32_t)g.nty);
    tc.z0 = 8 * (int)(rest / (uint32_t)g.nty);
    tc.wcy = min(8, g.ny - tc.y0);
    tc.wcz = min(8, g.nz - tc.z0);
    return tc;
}

// local row coordinate i in [-1, 8] of a tile that starts at c0 and has wc valid rows -> global coordinate, or -1
__device__ __forceinline__ int row_coord(int i, int c0, int wc, int n, int periodic) {
    if (i > wc) return -1;
    int c = c0 + i;
    if (c < 0) return periodic ? n - 1 : -1;
    if (c >= n) return periodic ? 0 : -1;
    return c;
}

// Shared-memory accesses of the per-voxel loops by 32-bit shared-window address held in a register (see flist_addr).
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
template <int OFF>
__device__ __forceinline__ uint32_t lds_u32_at(uint32_t addr) {            // [addr + OFF], OFF >= 0 an immediate
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(OFF) : "memory");
    return v;
}
__device__ __forceinline__ void lds_u64(uint32_t addr, uint32_t& a, uint32_t& b) {
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(addr) : "memory");
}
__device__ __forceinline__ uint4 lds_u128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u64(uint32_t addr, uint32_t a, uint32_t b) {
    asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(addr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ uint32_t mul_lo_u32(uint32_t a, uint32_t b) {     // a multiply the compiler does not turn into a shift
    uint32_t r;
    asm("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
__device__ __forceinline__ void atoms_or_u32(uint32_t addr, uint32_t v) {
    asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t opaque_shared_addr(const void* p) {     // a register the compiler cannot rematerialise
    uint32_t a;
    asm volatile("mov.u32 %0, %1;" : "=r"(a) : "r"((uint32_t)__cvta_generic_to_shared(p)));
    return a;
}

// The grids of one launch: one for liets_step / liets_generate, up to kMaxBatch equally shaped grids for
// liets_generate_batch (independent realisations).  A CTA starts with grid blockIdx.x mod n and then
// visits the others in turn: each grid hands its tiles out through its own cursor, so CTAs that find a grid's list used
// up move on and the whole GPU works on whatever is left -- small grids, whose few tiles cannot fill it, overlap.
template <int MAXB>
struct TileBatch {
    int n;
    Control* ctl[MAXB];
    unsigned long long* G0[MAXB];
    unsigned long long* G1[MAXB];
    uint32_t* stamp[MAXB];
    uint32_t* weight[MAXB];
    uint32_t* list0[MAXB];
    uint32_t* list1[MAXB];
    const unsigned long long* P[MAXB];      // cells of earlier phases in row layout (liets_set_blocked), or nullptr
    PhiloxKey key[MAXB];
};

// INTERACT (R20): cells of the earlier phases (plane P) that have a void neighbour are sources too, with the thresholds
// Control::hpatI; bit 15 of a list entry says which kind of source the voxel is.
template <int MAXB, bool INTERACT>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) k_grow_tile(const __grid_constant__ TileBatch<MAXB> B, const TileGeom g) {
    __shared__ __align__(16) Smem S;        // static (< 48 KB): shared-memory addresses are immediates, not generic pointers
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t lanes_below = (1u << lane) - 1u;
  for (int bk = 0; bk < (MAXB == 1 ? 1 : B.n); ++bk) {
    const int gi = MAXB == 1 ? 0 : (int)((blockIdx.x + (uint32_t)bk) % (uint32_t)B.n);
    if (MAXB > 1) __syncthreads();          // the previous grid's last tile is no longer read
    Control* __restrict__ ctl = B.ctl[gi];
    if (!ctl->active || (ctl->mode == 0u && !ctl->pending)) continue;   // small fronts run in k_grow_vox
    unsigned long long* const G0 = B.G0[gi];
    unsigned long long* const G1 = B.G1[gi];
    uint32_t* const stamp = B.stamp[gi];
    uint32_t* const weight = B.weight[gi];
    uint32_t* const list0 = B.list0[gi];
    uint32_t* const list1 = B.list1[gi];
    const unsigned long long* const P = B.P[gi];
    const PhiloxKey& key = B.key[gi];

    const uint32_t cur = ctl->cur;
    // the list of step t: heavy tiles in slots [0, n_head), light ones in the last n_back slots; heavy ones are handed
    // out first, so the kernel's tail is made of short tiles
    const uint32_t n_head = ctl->count[cur], n_back = ctl->count_back[cur], list_cap = ctl->list_cap;
    const uint32_t n_list = n_head + n_back;
    const uint32_t* __restrict__ in = cur ? list1 : list0;
    uint32_t* __restrict__ out = cur ? list0 : list1;
    uint32_t* out_count = &ctl->count[cur ^ 1u];
    uint32_t* out_count_back = &ctl->count_back[cur ^ 1u];
    auto list_entry = [&](uint32_t li) { return in[li < n_head ? li : list_cap - 1u - (li - n_head)]; };
    auto emit_tile = [&](uint32_t tile, uint32_t n_front_seen) {        // heavy tiles to the front of the next list, light to its back
        if (n_front_seen >= (uint32_t)kHeavyFront) out[atomicAdd(out_count, 1u)] = tile;
        else out[list_cap - 1u - atomicAdd(out_count_back, 1u)] = tile;
    };
    const uint32_t t = ctl->step;
    const PhiloxStep ps = philox_step_uniform(t, key);
    const unsigned long long* __restrict__ Gc = (t & 1u) ? G1 : G0;     // g_t (read only)
    unsigned long long* Gn = (t & 1u) ? G0 : G1;                        // g_{t+1} (OR target)
    if (tid < 32) S.hpat[0][tid >> 2][tid & 3] = ctl->hpat[tid >> 2][tid & 3];
    else if (INTERACT && tid < 64) S.hpat[1][(tid - 32u) >> 2][tid & 3] = ctl->hpatI[(tid - 32u) >> 2][tid & 3];
    if (tid < 28) {
        const int d = tid < 26 ? (int)tid : 25;
        const int raw = d + (d >= 13 ? 1 : 0);
        const int dx = raw % 3 - 1, dy = (raw / 3) % 3 - 1, dz = raw / 9 - 1;
        S.dir[tid] = (uint32_t)(2 * kRowWords * (dz * 10 + dy + 11)) | ((uint32_t)(dx + 1) << 16);
    }
    const uint32_t en26 = ctl->en26, enI26 = INTERACT ? ctl->enI26 : 0u;
    const bool h0_any = INTERACT || ctl->h0_any != 0u;      // (with two kinds of sources level 0 always takes the general compare)
    const uint32_t h0[4] = { ctl->hpat[0][0], ctl->hpat[0][1], ctl->hpat[0][2], ctl->hpat[0][3] };
    constexpr uint32_t kM8 = 0x88888888u;
    const uint32_t h0m[4] = { h0[0] & kM8, h0[1] & kM8, h0[2] & kM8, h0[3] & kM8 };     // level-0 compare: uniform parts
    const uint32_t h08[4] = { h0[0] | kM8, h0[1] | kM8, h0[2] | kM8, h0[3] | kM8 };
    // every leading nibble below 8 (no class at probability >= 1/2): the three-instruction compares of level0_compare_small
    const bool h0_small = ((h0[0] | h0[1] | h0[2] | h0[3]) & kM8) == 0u;
    uint32_t h0cle[4], h0clt[4], h0nz[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t nz = (((h0[w] & 0x77777777u) + 0x77777777u) | h0[w]) & kM8;      // 0x8 where the nibble is not zero
        h0nz[w] = nz;
        h0cle[w] = 0x77777777u - (h0[w] & 0x77777777u);
        h0clt[w] = 0x77777777u - ((h0[w] - (nz >> 3)) & 0x77777777u);
    }
    uint32_t new_solid = 0;                 // per thread: bits this thread flipped 0 -> 1
    uint32_t n_items = 0, n_items0 = 0;     // per thread: Philox blocks evaluated, front voxels with a void target
    // shared-window address of the voxel list, kept in a register: left to itself the compiler rebuilds it (S2R
    // CgaCtaId, MOV, LEA) at every access inside the per-voxel loops
    const uint32_t flist_addr = opaque_shared_addr(S.flist), win_addr = opaque_shared_addr(S.win);
    const uint32_t claims_addr = opaque_shared_addr(S.claims), queue_addr = opaque_shared_addr(S.queue[warp]);
    const uint32_t hpat_addr = opaque_shared_addr(S.hpat), dir_addr = opaque_shared_addr(S.dir);
    const uint32_t ptab_addr = opaque_shared_addr(S.ptab);

    uint32_t next_li = 0, next_id = 0;      // thread 0: the list entry fetched ahead
    if (tid == 0) {
        next_li = atomicAdd(&ctl->tile_cursor, 1u);
        if (next_li < n_list) next_id = list_entry(next_li);
    }
    if (tid == 0) { S.tile[0] = next_li; S.tile_id[0] = next_id; }
    for (uint32_t kt = 0;; ++kt) {
        __syncthreads();                    // the previous tile's shared memory is no longer read; this tile's slot is written
        const uint32_t li = S.tile[kt & 1u];
        if (li >= n_list) break;
        const uint32_t id = S.tile_id[kt & 1u];
        if (tid == 0) {                     // latency hidden behind this tile's work
            next_li = atomicAdd(&ctl->tile_cursor, 1u);
            if (next_li < n_list) next_id = list_entry(next_li);
        }
        const TileCoord tc = tile_coord(id, g);

        // ---- A: gather ------------------------------------------------------------------------
        const uint32_t p0 = (uint32_t)(64 * tc.w0) + (uint32_t)g.nx * ((uint32_t)tc.y0 + (uint32_t)g.ny * (uint32_t)tc.z0);
        for (int r = (int)tid; r < 100; r += kThreads) {    // one thread per row: the row's address once, its words as independent loads
            const int zl = r / 10 - 1, yl = r % 10 - 1;
            const int zg = row_coord(zl, tc.z0, tc.wcz, g.nz, g.periodic & 4);
            const int yg = row_coord(yl, tc.y0, tc.wcy, g.ny, g.periodic & 2);
            const bool ok = zg >= 0 && yg >= 0;
            const unsigned long long row_base = ok ? (unsigned long long)g.Wp * ((unsigned long long)yg + (unsigned long long)g.ny * (unsigned long long)zg) : 0ull;
            unsigned long long w[kRowWords];
#pragma unroll
            for (int c = 0; c < kRowWords; ++c) w[c] = not_void_word(Gc, g, ok, row_base, tc.w0 + c - 1);
            if (zl >= 0 && zl < 8 && yl >= 0 && yl < 8) {           // an own row: its words for B and E, its first voxel's index
#pragma unroll
                for (int j = 0; j < kTileW; ++j) S.own[zl * 8 + yl][j] = w[1 + j];
                S.ptab[r] = p0 + (uint32_t)g.nx * ((uint32_t)yl + (uint32_t)g.ny * (uint32_t)zl);
            }
#pragma unroll
            for (int j = 0; j < kTileW; ++j) {                      // void at x-1, x or x+1 (the x part of the 3x3x3 dilation)
                const unsigned long long v = ~w[1 + j];
                S.vx[r][j] = v | (v << 1) | (~w[j] >> 63) | (v >> 1) | (~w[2 + j] << 63);
            }
#pragma unroll
            for (int k = 0; k < kWin; k += 4) {                     // window k: row bits 63 + 16 k .. 80 + 16 k (tile x = 16k-1 .. 16k+16) at bits 14..31
                uint32_t wv[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int pos = 63 + 16 * (k + q), wd = pos >> 6, sh = pos & 63;
                    unsigned long long v = w[wd] >> sh;
                    if (sh + 18 > 64) v |= w[wd + 1] << (64 - sh);
                    wv[q] = (uint32_t)v << 14;
                }
                *reinterpret_cast<uint4*>(&S.win[r * kWin + k]) = make_uint4(wv[0], wv[1], wv[2], wv[3]);
            }
        }
        for (int q = (int)tid; q < 100 * 2 * kRowWords / 4; q += kThreads)
            reinterpret_cast<uint4*>(&S.claims[0][0])[q] = make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();
        // ---- B: front voxels of the tile ------------------------------------------------------------
        uint32_t n_front = 0, off0 = 0;
        unsigned long long F = 0ull;        // this thread's word (row tid / kTileW, word tid % kTileW): its front voxels
        unsigned long long Pw = 0ull;       // ... and which of its cells belong to earlier phases
        const int f_row = (int)tid / kTileW, f_j = (int)tid - f_row * kTileW;
        {
            static_assert(64 * kTileW == kThreads, "one tile word per thread");
            const int y = f_row & 7, z = f_row >> 3;
            const int xbase = 64 * (tc.w0 + f_j);
            if (y < tc.wcy && z < tc.wcz && xbase < g.nx) {
                unsigned long long src = S.own[f_row][f_j];
                if (xbase + 64 > g.nx) src &= ~(~0ull << (g.nx - xbase));               // padding is not a source
                if (P) {                                                                // nor is a cell of an earlier phase -- unless it interacts (R20)
                    Pw = __ldg(P + (unsigned long long)g.Wp * ((unsigned long long)(tc.y0 + y) + (unsigned long long)g.ny * (unsigned long long)(tc.z0 + z)) + (unsigned long long)(tc.w0 + f_j));
                    if (!INTERACT) src &= ~Pw;
                }
                if (src) {                                                              // (sparse early steps: most words hold no solid)
                    unsigned long long anyvoid = 0ull;
#pragma unroll
                    for (int k = 0; k < 9; ++k) anyvoid |= S.vx[(z + k / 3) * 10 + (y + k % 3)][f_j];
                    F = src & anyvoid;                                                  // R13
                }
            }
            // CTA prefix sum with one barrier: warp scan, warp totals to shared memory (double-buffered per tile),
            // every thread adds the totals of the warps below its own
            uint32_t wtotal;
            const uint32_t wexcl = warp_exclusive_scan((uint32_t)__popcll(F), lane, &wtotal);
            if (lane == 0) S.wsum[kt & 1u][warp] = wtotal;
            __syncthreads();
            off0 = wexcl;
#pragma unroll
            for (int q = 0; q < kWarps; ++q) {
                const uint32_t v = S.wsum[kt & 1u][q];
                n_front += v;
                if ((uint32_t)q < warp) off0 += v;
            }
        }

        // ---- C + D -----------------------------------------------------------------------------------
        // the hits of voxel (x, row rr): bits of the claim volume
        auto claim = [&](uint32_t fire, uint32_t x, uint32_t rr) {
            const uint32_t cbase = claims_addr + 4u * (2u * kRowWords) * (rr - 11u);
            while (fire) {
                const uint32_t d = 31u - __clz(fire);
                fire ^= 1u << d;
                const uint32_t lut = lds_u32(dir_addr + 4u * d);
                const uint32_t xb = x + 63u + (lut >> 16);          // bit of the row: 64 + x + dx
                atoms_or_u32(cbase + 4u * ((lut & 0xFFFFu) + (xb >> 5)), 1u << (xb & 31u));
            }
        };
        // D: tied voxels wait in a per-warp ring.  resolve() looks at the next nibble level of one entry: the directions that
        // fire are claimed, the ones that tie again are returned.  round() takes the 32 oldest entries of the ring, one lane
        // each, and appends the entries that still tie one level deeper; while the tile is being listed only full rounds run.
        auto resolve = [&](uint32_t vk, uint32_t tie) -> uint32_t {
            const uint32_t x = (vk & 0x7Fu) ^ 15u, rr = (vk >> 7) & 0x7Fu, k = vk >> 16;
            const uint32_t p = lds_u32(ptab_addr + 4u * rr) + x;
            const uint4 B = philox_growth_block(p, k, ps, key);
            ++n_items;
            const uint4 hk = lds_u128(hpat_addr + 16u * k + (INTERACT ? ((vk >> 15) & 1u) * 128u : 0u));
            const uint32_t h[4] = { hk.x, hk.y, hk.z, hk.w };
            uint32_t le, eq;
            level_compare(B, h, tie, &le, &eq);
            const bool last = k == 7u;                                          // last nibble: draw <= U
            claim(last ? le : (le & ~eq), x, rr);
            return last ? 0u : eq;
        };
        // The same for the rounds AFTER the tile's last voxel, when the ring no longer fills: two nibble levels at once.  The
        // blocks k and k + 1 of the entry are evaluated side by side (one latency for both chains), so a direction that ties
        // again is settled in the same round; only a tie at both levels goes back into the ring.  The chain of dependent
        // partial rounds at the end of every tile (it sits on the tile's critical path) shrinks from one round per level to
        // one per two levels.  Only the blocks the draws need are counted.
        auto resolve2 = [&](uint32_t vk, uint32_t tie) -> uint32_t {
            const uint32_t x = (vk & 0x7Fu) ^ 15u, rr = (vk >> 7) & 0x7Fu, k = vk >> 16, k1 = min(k + 1u, 7u);
            const uint32_t p = lds_u32(ptab_addr + 4u * rr) + x;
            const uint4 B = philox_growth_block(p, k, ps, key);
            const uint4 B1 = philox_growth_block(p, k1, ps, key);
            ++n_items;
            const uint32_t hk_addr = hpat_addr + (INTERACT ? ((vk >> 15) & 1u) * 128u : 0u);
            const uint4 hk = lds_u128(hk_addr + 16u * k);
            const uint32_t h[4] = { hk.x, hk.y, hk.z, hk.w };
            uint32_t le, eq, still = 0;
            level_compare(B, h, tie, &le, &eq);
            uint32_t fire = k == 7u ? le : (le & ~eq);                          // last nibble: draw <= U
            if (k < 7u && eq) {
                ++n_items;
                const uint4 hk1 = lds_u128(hk_addr + 16u * k1);
                const uint32_t h1[4] = { hk1.x, hk1.y, hk1.z, hk1.w };
                uint32_t le1, eq1;
                level_compare(B1, h1, eq, &le1, &eq1);
                if (k1 == 7u) fire |= le1;
                else { fire |= le1 & ~eq1; still = eq1; }
            }
            claim(fire, x, rr);
            return still;
        };
        uint32_t qh = 0, qn = 0;            // ring head and fill (warp-uniform)
        auto round = [&](uint32_t n_take) {
            constexpr uint32_t kMask = (uint32_t)kQueueCap - 1u;
            uint32_t vk = 0, tie = 0, still = 0;
            if (lane < n_take) lds_u64(queue_addr + 8u * ((qh + lane) & kMask), vk, tie);
            __syncwarp();                   // this round's entries are read before any slot is written again
            if (tie) still = resolve(vk, tie);
            const uint32_t have = __ballot_sync(0xffffffffu, still != 0u);
            qh = (qh + n_take) & kMask;
            qn -= n_take;
            if (still) sts_u64(queue_addr + 8u * ((qh + qn + __popc(have & ((1u << lane) - 1u))) & kMask), vk + (1u << 16), still);
            qn += __popc(have);
            __syncwarp();
        };
        auto round2 = [&](uint32_t n_take) {
            constexpr uint32_t kMask = (uint32_t)kQueueCap - 1u;
            uint32_t vk = 0, tie = 0, still = 0;
            if (lane < n_take) lds_u64(queue_addr + 8u * ((qh + lane) & kMask), vk, tie);
            __syncwarp();
            if (tie) still = resolve2(vk, tie);
            const uint32_t have = __ballot_sync(0xffffffffu, still != 0u);
            qh = (qh + n_take) & kMask;
            qn -= n_take;
            if (still) sts_u64(queue_addr + 8u * ((qh + qn + __popc(have & ((1u << lane) - 1u))) & kMask), vk + (2u << 16), still);
            qn += __popc(have);
            __syncwarp();
        };
        for (uint32_t pass0 = 0; pass0 < n_front; pass0 += (uint32_t)kFrontCap) {   // almost always a single pass
            if (pass0) __syncthreads();     // the previous pass no longer reads the list
            {
                // entry of bit b of half h of this thread's word: ((8 rr + 4 j + 2 h + b / 16) << 4) | (15 - b % 16) = base_h ^ b
                const uint32_t rr = (uint32_t)((f_row >> 3) + 1) * 10u + (uint32_t)(f_row & 7) + 1u;
                const uint32_t base = ((8u * rr + 4u * (uint32_t)f_j) << 4) | 15u;
                if (n_front <= (uint32_t)kFrontCap) {   // the usual case, one pass: no capacity test, the address just advances
                    uint32_t addr = flist_addr + 2u * off0;
#pragma unroll
                    for (int half = 1; half >= 0; --half) {         // highest bit first: one FLO per voxel
                        const uint32_t hh = base | (uint32_t)(32 * half);
                        for (uint32_t m = (uint32_t)(F >> (32 * half)); m; addr += 2u) {
                            const uint32_t b = 31u - __clz(m);
                            m ^= 1u << b;
                            uint32_t ent = hh ^ b;
                            if (INTERACT) ent |= ((uint32_t)(Pw >> (32 * half)) >> b & 1u) << 15;
                            asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((uint16_t)ent) : "memory");
                        }
                    }
                } else {                    // list the front voxels pass0 .. pass0 + kFrontCap - 1
                    uint32_t off = off0;
#pragma unroll
                    for (int half = 1; half >= 0; --half) {
                        const uint32_t hh = base | (uint32_t)(32 * half);
                        for (uint32_t m = (uint32_t)(F >> (32 * half)); m; ++off) {
                            const uint32_t b = 31u - __clz(m);
                            m ^= 1u << b;
                            if (off - pass0 < (uint32_t)kFrontCap)
                            {
                                uint32_t ent = hh ^ b;
                                if (INTERACT) ent |= ((uint32_t)(Pw >> (32 * half)) >> b & 1u) << 15;
                                asm volatile("st.shared.u16 [%0], %1;" ::"r"(flist_addr + 2u * (off - pass0)), "h"((uint16_t)ent) : "memory");
                            }
                        }
                    }
                }
            }
            __syncthreads();                // flist (and win) complete
            const uint32_t n_pass = min((uint32_t)kFrontCap, n_front - pass0);
            // C: front voxels, two CONSECUTIVE list entries per thread and trip (one 32-bit load), worked without a branch in
            // one basic block: the two Philox chains interleave and share the round keys.  A warp covers 64 entries, so the
            // test that skips a warp beyond the list's end is warp-uniform; a lane beyond the end works on a harmless
            // entry and its result is dropped.  Every listed voxel has a void target unless its directions are disabled
            // (en26), so the block is evaluated unconditionally and the compare masks by void26.
            auto gather26 = [&](uint32_t v) -> uint32_t {
                // the nine rows of the neighbourhood: one window each, aligned so that x+1, x, x-1 are bits 31..29 (a multiply:
                // FMA pipe) and pushed into the mask three bits at a time (row dz = +1, dy = +1 first):
                // bit 9(dz+1) + 3(dy+1) + (dx+1) = not void
                const uint32_t wa = win_addr + ((v >> 2) & 0x0FFCu) - 4u * kWin * 11u;
                const uint32_t mult = 1u << (v & 15u);
                uint32_t nb27 = 0;
#define LIETS_ROW(E) nb27 = __funnelshift_l(mul_lo_u32(lds_u32_at<4 * kWin * (((E) / 3) * 10 + (E) % 3)>(wa), mult), nb27, 3)
                LIETS_ROW(8); LIETS_ROW(7); LIETS_ROW(6); LIETS_ROW(5); LIETS_ROW(4); LIETS_ROW(3); LIETS_ROW(2); LIETS_ROW(1); LIETS_ROW(0);
#undef LIETS_ROW
                // the centre (bit 13) is solid, so ~nb27 has bit 13 clear: closing the gap is (v + (v & 0x1FFF)) >> 1
                const uint32_t lo13 = ~nb27 & 0x1FFFu;
                return (~nb27 + lo13) >> 1;
            };
            constexpr uint32_t kSafeEntry = (8u * 11u) << 4;        // row (0, 0), window 0: a list entry that is always addressable
            auto level0_pair = [&](uint32_t i, uint32_t* v, uint32_t* tie, uint32_t* fire) {
                const uint32_t pair = lds_u32(flist_addr + 2u * i);             // i is even
                const bool live0 = i < n_pass, live1 = i + 1u < n_pass;
                v[0] = live0 ? (pair & 0xFFFFu) : kSafeEntry;
                v[1] = live1 ? (pair >> 16) : kSafeEntry;
                uint32_t void26[2];
                uint4 B0[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) void26[u] = gather26(v[u]) & ((INTERACT && (v[u] >> 15)) ? enI26 : en26);
                void26[0] = live0 ? void26[0] : 0u;
                void26[1] = live1 ? void26[1] : 0u;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const uint32_t p = lds_u32(ptab_addr + ((v[u] >> 5) & 0x1FCu)) + ((v[u] & 0x7Fu) ^ 15u);
                    B0[u] = philox_growth_block(p, 0u, ps, key);
                    n_items0 += void26[u] ? 1u : 0u;
                }
                if (INTERACT) {             // two kinds of sources: the voxel's own thresholds, general compare
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const uint4 hk = lds_u128(hpat_addr + (v[u] >> 15) * 128u);
                        const uint32_t hsel[4] = { hk.x, hk.y, hk.z, hk.w };
                        uint32_t le;
                        level_compare(B0[u], hsel, void26[u], &le, &tie[u]);
                        fire[u] = le & ~tie[u];
                    }
                } else if (h0_any) {        // some leading threshold nibble is non-zero: a draw can fire at level 0
                    if (h0_small) {
#pragma unroll
                        for (int u = 0; u < 2; ++u) level0_compare_small(B0[u], h0cle, h0clt, h0nz, void26[u], &fire[u], &tie[u]);
                    } else {
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            uint32_t le;
                            level0_compare(B0[u], h0, h0m, h08, void26[u], &le, &tie[u]);
                            fire[u] = le & ~tie[u];
                        }
                    }
                } else {                    // all leading nibbles are 0: "<=" and "==" coincide with "== 0"
#pragma unroll
                    for (int u = 0; u < 2; ++u) tie[u] = level_zero(B0[u], void26[u]);
                }
            };
            // level-0 hits to the claim volume, ties to the ring: both entries of the pair behind one capacity test
            auto settle2 = [&](const uint32_t* v, const uint32_t* tie, const uint32_t* fire) {
                if (h0_any) {
#pragma unroll
                    for (int u = 0; u < 2; ++u)
                        if (__ballot_sync(0xffffffffu, fire[u] != 0u)) claim(fire[u], (v[u] & 0x7Fu) ^ 15u, (v[u] >> 7) & 0x7Fu);
                }
                const uint32_t have0 = __ballot_sync(0xffffffffu, tie[0] != 0u), have1 = __ballot_sync(0xffffffffu, tie[1] != 0u);
                if (have0 | have1) {
                    constexpr uint32_t kMask = (uint32_t)kQueueCap - 1u;
                    while (qn >= 32u) round(32u);           // a full round as soon as there is one: little is left at the tile's end
                    const uint32_t n0 = __popc(have0);
                    if (tie[0]) sts_u64(queue_addr + 8u * ((qh + qn + __popc(have0 & lanes_below)) & kMask), v[0] | (1u << 16), tie[0]);
                    if (tie[1]) sts_u64(queue_addr + 8u * ((qh + qn + n0 + __popc(have1 & lanes_below)) & kMask), v[1] | (1u << 16), tie[1]);
                    qn += n0 + __popc(have1);
                }
            };
            for (uint32_t i0 = 0; i0 < n_pass; i0 += 2u * kThreads) {
                uint32_t v[2] = { 0u, 0u }, tie[2] = { 0u, 0u }, fire[2] = { 0u, 0u };
                if (i0 + 64u * warp < n_pass) level0_pair(i0 + 2u * tid, v, tie, fire);     // warp-uniform
                settle2(v, tie, fire);
            }
        }
        while (qn >= 32u) round(32u);
        while (qn) round2(qn);              // fewer than 32 entries left
        if (tid == 0) { S.tile[(kt + 1u) & 1u] = next_li; S.tile_id[(kt + 1u) & 1u] = next_id; }   // read after the next barrier but one
        __syncthreads();                    // all claims are in shared memory

        // ---- E: claim + compact ---------------------------------------------------------------------
        // word (r, c) of the claim volume -> global row, the bits that lie in the row itself (x < nx) and the one
        // bit that may lie across the x border (x = -1, or x = nx on a periodic grid)
        auto halo_word = [&](int r, int c, unsigned long long cw) {
            const int zl = r / 10 - 1, yl = r % 10 - 1;
            const int wg = tc.w0 + c - 1;
            const int zg = row_coord(zl, tc.z0, tc.wcz, g.nz, g.periodic & 4);
            const int yg = row_coord(yl, tc.y0, tc.wcy, g.ny, g.periodic & 2);
            const unsigned long long row_base = (unsigned long long)g.Wp * ((unsigned long long)yg + (unsigned long long)g.ny * (unsigned long long)zg);
            unsigned long long in_row = 0ull, wrap = 0ull;
            int x_wrap = 0;
            if (c == 0) { wrap = cw >> 63; x_wrap = wg >= 0 ? 64 * wg + 63 : g.nx - 1; }
            else if (64 * wg + 64 <= g.nx) in_row = cw;
            else if (64 * wg <= g.nx) {
                const int nvalid = g.nx - 64 * wg;                  // 0..63
                in_row = cw & ~(~0ull << nvalid);
                wrap = (cw >> nvalid) & 1ull;                       // periodic only: the cell at x = nx is x = 0
            }
            if (in_row) {                                           // hits in a neighbour tile's rows
                const unsigned long long old = atomicOr(Gn + row_base + wg, in_row);
                new_solid += __popcll(in_row & ~old);
                const uint32_t nb = (uint32_t)(wg / kTileW) + (uint32_t)g.ntx * ((uint32_t)(yg >> 3) + (uint32_t)g.nty * (uint32_t)(zg >> 3));
                if (nb != id && atomicMax(&stamp[nb], t + 2u) < t + 2u) emit_tile(nb, weight[nb]);          // newly active tile
            }
            if (wrap) {                                             // one cell across the tile's x border
                const unsigned long long bit = 1ull << (x_wrap & 63);
                const unsigned long long old = atomicOr(Gn + row_base + (x_wrap >> 6), bit);
                if (!(old & bit)) new_solid++;
                const uint32_t nb = (uint32_t)((x_wrap >> 6) / kTileW) + (uint32_t)g.ntx * ((uint32_t)(yg >> 3) + (uint32_t)g.nty * (uint32_t)(zg >> 3));
                if (nb != id && atomicMax(&stamp[nb], t + 2u) < t + 2u) emit_tile(nb, weight[nb]);
            }
        };
        // A tile is "x-plain" when no claim of it can cross the x border of the grid: always between walls (cells outside
        // are never void, so they are never claimed), and on a grid that wraps in x when the tile touches neither end of
        // the row.  Its claim words map one to one to words of the grid.
        const bool x_plain = !(g.periodic & 1) || (tc.w0 >= 1 && 64 * (tc.w0 + kTileW) < g.nx);
        // own words first, one per thread: carry g_t and add the hits.  The atomic's old word (who flipped the bit) comes
        // back while the halo rows are worked on and is looked at after them.
        unsigned long long own_hits = 0ull, own_old = ~0ull;
        {
            static_assert(64 * kTileW == kThreads, "one own word per thread");
            const int row = (int)tid / kTileW, j = (int)tid - row * kTileW, y = row & 7, z = row >> 3;
            const int wg = tc.w0 + j, r = (z + 1) * 10 + (y + 1);
            if (y < tc.wcy && z < tc.wcz && 64 * wg < g.nx) {
                const unsigned long long cw = (unsigned long long)S.claims[r][2 * (j + 1)] | ((unsigned long long)S.claims[r][2 * (j + 1) + 1] << 32);
                unsigned long long curw = S.own[row][j], in_row = cw;
                if (64 * wg + 64 > g.nx) {                          // the row ends inside this word
                    const unsigned long long valid = ~(~0ull << (g.nx - 64 * wg));
                    curw &= valid;
                    in_row &= valid;
                    if (!x_plain && (cw & ~valid)) halo_word(r, j + 1, cw & ~valid);       // the cell at x = nx (periodic wrap)
                }
                unsigned long long* dst = Gn + (unsigned long long)g.Wp * ((unsigned long long)(tc.y0 + y) + (unsigned long long)g.ny * (unsigned long long)(tc.z0 + z)) + wg;
                if (in_row) { own_old = atomicOr(dst, curw | in_row); own_hits = in_row; }
                else if (curw) atomicOr(dst, curw);
            }
        }
        // newly active neighbour tile: the first claim of the step into it lists it
        auto wake = [&](uint32_t nb) {
            if (nb != id && atomicMax(&stamp[nb], t + 2u) < t + 2u) emit_tile(nb, weight[nb]);
        };
        for (int r = (int)tid; r < 100; r += kThreads) {    // halo words, one thread per row
            unsigned long long cw[kRowWords], any = 0ull;
#pragma unroll
            for (int c = 0; c < kRowWords; ++c) {
                cw[c] = (unsigned long long)S.claims[r][2 * c] | ((unsigned long long)S.claims[r][2 * c + 1] << 32);
                any |= cw[c];
            }
            const int zl = r / 10 - 1, yl = r % 10 - 1;
            const bool own_row = zl >= 0 && zl < tc.wcz && yl >= 0 && yl < tc.wcy;
            if (own_row) {                                  // the tile words of an own row went out above
#pragma unroll
                for (int c = 1; c <= kTileW; ++c)
                    if (64 * (tc.w0 + c - 1) < g.nx) cw[c] = 0ull;
                any = 0ull;
#pragma unroll
                for (int c = 0; c < kRowWords; ++c) any |= cw[c];
            }
            if (!any) continue;
            if (x_plain) {
                // all atomics of the row go out together, with plain loads of the stamps of the (at most three) tiles they
                // fall into; only a tile whose stamp is still old takes the atomicMax
                const int zg = row_coord(zl, tc.z0, tc.wcz, g.nz, g.periodic & 4);
                const int yg = row_coord(yl, tc.y0, tc.wcy, g.ny, g.periodic & 2);
                unsigned long long* rowp = Gn + (unsigned long long)g.Wp * ((unsigned long long)yg + (unsigned long long)g.ny * (unsigned long long)zg) + (tc.w0 - 1);
                const uint32_t nb_mid = (uint32_t)(tc.w0 / kTileW) + (uint32_t)g.ntx * ((uint32_t)(yg >> 3) + (uint32_t)g.nty * (uint32_t)(zg >> 3));
                cw[0] &= 1ull << 63;                        // (only the cell next to the tile can be claimed in a halo word)
                cw[kRowWords - 1] &= 1ull;
                unsigned long long mid = 0ull;
#pragma unroll
                for (int c = 1; c <= kTileW; ++c) mid |= cw[c];
                unsigned long long old[kRowWords];
                uint32_t st[3] = { ~0u, ~0u, ~0u };
#pragma unroll
                for (int c = 0; c < kRowWords; ++c) {
                    old[c] = ~0ull;
                    if (cw[c]) old[c] = atomicOr(rowp + c, cw[c]);
                }
                if (cw[0]) st[0] = __ldcg(&stamp[nb_mid - 1u]);
                if (mid) st[1] = __ldcg(&stamp[nb_mid]);
                if (cw[kRowWords - 1]) st[2] = __ldcg(&stamp[nb_mid + 1u]);
#pragma unroll
                for (int c = 0; c < kRowWords; ++c) new_solid += __popcll(cw[c] & ~old[c]);
                uint32_t need = (st[0] < t + 2u ? 1u : 0u) | (st[1] < t + 2u ? 2u : 0u) | (st[2] < t + 2u ? 4u : 0u);
                while (need) {                              // rare: at most once per neighbour tile and step
                    const uint32_t k = 31u - __clz(need);
                    need ^= 1u << k;
                    wake(nb_mid + k - 1u);
                }
            } else {
#pragma unroll 1
                for (int c = 0; c < kRowWords; ++c) {       // (the words are read again: no register array indexed at run time)
                    const bool own_word = own_row && c >= 1 && c <= kTileW && 64 * (tc.w0 + c - 1) < g.nx;
                    const unsigned long long cwv = (unsigned long long)S.claims[r][2 * c] | ((unsigned long long)S.claims[r][2 * c + 1] << 32);
                    if (cwv && !own_word) halo_word(r, c, cwv);
                }
            }
        }
        new_solid += __popcll(own_hits & ~own_old);
        if (tid == 0 && n_front) {                                  // this tile still has front voxels
            weight[id] = n_front;                                   // whoever lists the tile for the next step sorts it by this
            if (atomicMax(&stamp[id], t + 2u) < t + 2u) emit_tile(id, n_front);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        new_solid += __shfl_xor_sync(0xffffffffu, new_solid, o);
        n_items += __shfl_xor_sync(0xffffffffu, n_items, o);
        n_items0 += __shfl_xor_sync(0xffffffffu, n_items0, o);
    }
    if (lane == 0 && new_solid) atomicAdd(&ctl->claims, new_solid);
    if (lane == 0 && n_items0) { atomicAdd(&ctl->items, n_items + n_items0); atomicAdd(&ctl->items0, n_items0); }
  }
}

}  // namespace

int grow_tile_words() { return kTileW; }
int grow_tile_ctas_per_sm() { return kCtasPerSm; }
int grow_tile_max_batch() { return kMaxBatch; }

// per-device function attribute, set once per context at liets_create: the SM's shared memory to the CTAs
cudaError_t grow_tile_attributes() {
    static_assert(sizeof(Smem) <= 48 * 1024, "static shared memory");
    cudaError_t e = cudaFuncSetAttribute(k_grow_tile<1, false>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_grow_tile<1, true>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_grow_tile<kMaxBatch, false>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}

template <int MAXB>
static void fill_batch(TileBatch<MAXB>* b, liets_ctx* const* ctx, int n) {
    b->n = n;
    for (int i = 0; i < n; ++i) {
        liets_ctx* c = ctx[i];
        b->ctl[i] = c->ctl; b->G0[i] = c->G[0]; b->G1[i] = c->G[1]; b->stamp[i] = c->stamp; b->weight[i] = c->weight;
        b->list0[i] = c->list[0]; b->list1[i] = c->list[1]; b->P[i] = c->has_blocked ? c->prow : nullptr;
        b->key[i] = philox_make_key(c->rng_seed);
    }
}

cudaError_t launch_grow_tile(liets_ctx* c) {
    TileBatch<1> b;
    fill_batch(&b, &c, 1);
    if (c->interact && c->has_blocked) k_grow_tile<1, true><<<c->tile_grid, kThreads, 0, c->stream>>>(b, c->geom);
    else k_grow_tile<1, false><<<c->tile_grid, kThreads, 0, c->stream>>>(b, c->geom);
    c->launches++;
    return cudaGetLastError();
}

// The same launch as a kernel node of `graph` (exec == nullptr), or its parameters refreshed in an instantiated
// graph (the Philox key changes with every liets_seed).
cudaError_t grow_tile_node(liets_ctx* c, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node) {
    TileBatch<1> b;
    fill_batch(&b, &c, 1);
    void* args[] = { &b, &c->geom };
    cudaKernelNodeParams p = {};
    p.func = (c->interact && c->has_blocked) ? reinterpret_cast<void*>(k_grow_tile<1, true>) : reinterpret_cast<void*>(k_grow_tile<1, false>);
    p.gridDim = dim3(c->tile_grid); p.blockDim = dim3(kThreads); p.sharedMemBytes = 0; p.kernelParams = args;
    return exec ? cudaGraphExecKernelNodeSetParams(exec, *node, &p) : cudaGraphAddKernelNode(node, graph, nullptr, 0, &p);
}

// n equally shaped grids (n <= kMaxBatch) in one kernel node; the launch is the first grid's
cudaError_t grow_tile_batch_node(liets_ctx* const* ctx, int n, cudaGraph_t graph, cudaGraphExec_t exec, cudaGraphNode_t* node) {
    if (n < 1 || n > kMaxBatch) return cudaErrorInvalidValue;
    TileBatch<kMaxBatch> b = {};
    fill_batch(&b, ctx, n);
    void* args[] = { &b, &ctx[0]->geom };
    cudaKernelNodeParams p = {};
    p.func = reinterpret_cast<void*>(k_grow_tile<kMaxBatch, false>);
    p.gridDim = dim3(ctx[0]->tile_grid); p.blockDim = dim3(kThreads); p.sharedMemBytes = 0; p.kernelParams = args;
    return exec ? cudaGraphExecKernelNodeSetParams(exec, *node, &p) : cudaGraphAddKernelNode(node, graph, nullptr, 0, &p);
}

}  // namespace liets
