// liets_device.cuh -- device-side building blocks shared by the kernels of libliets.so.
// (Product code: shares nothing with oracle/.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace liets {

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11) -- the counter-based stream of DESIGN.md reading R9
// ("an independent random number in (0,1) is drawn").
//   growth:  key = (rng_seed lo, hi); the 32-bit draw of (voxel p, step t, direction d) is written nibble by
//            nibble, most significant first, from the voxel's eight blocks B_k = philox(p lo, p hi, t, k):
//            nibble k of draw(d) = nibble d>>2 of word d&3 of B_k.  Block 0 alone decides, for all 26 directions
//            at once, which draws can still fall below the threshold; block k+1 is evaluated only for the
//            directions whose nibbles 0..k all tie with the threshold's
//   seeding: counter = ((v>>2) lo, (v>>2) hi, 0, 0xFFFFFFFF), draw of voxel v = word v&3
// ---------------------------------------------------------------------------------------------
constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

struct PhiloxKey {          // the ten round keys, precomputed once per launch (uniform)
    uint32_t k0[10];
    uint32_t k1[10];
};

__host__ __device__ inline PhiloxKey philox_make_key(uint64_t rng_seed) {
    PhiloxKey k;
    uint32_t a = (uint32_t)rng_seed, b = (uint32_t)(rng_seed >> 32);
    for (int r = 0; r < 10; ++r) {
        k.k0[r] = a; k.k1[r] = b;
        a += kPhiloxW0; b += kPhiloxW1;
    }
    return k;
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKey& key) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)kPhiloxM0 * c0;     // one IMAD.WIDE each
        const unsigned long long p1 = (unsigned long long)kPhiloxM1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[r];
        c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[r];
        c3 = (uint32_t)p0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// The growth blocks B_k = philox(p, 0, t, k) of one step share t and the key: the halves of rounds 1-3 that do not
// depend on the voxel are evaluated once per thread and launch (3 of the 40 multiply / xor pairs of a block).
struct PhiloxStep { uint32_t k10, a, b, c; };

__device__ __forceinline__ PhiloxStep philox_step_uniform(uint32_t t, const PhiloxKey& key) {
    const unsigned long long p1 = (unsigned long long)kPhiloxM1 * t;            // round 1: c2 = t, c1 = 0
    const uint32_t u0 = (uint32_t)(p1 >> 32) ^ key.k0[0], u1 = (uint32_t)p1;    // c0, c1 after round 1
    const unsigned long long q0 = (unsigned long long)kPhiloxM0 * u0;           // round 2: M0 * c0
    PhiloxStep s;
    s.k10 = key.k1[0];                              // round 1: c2 = hi(M0 p) ^ k ^ k10
    s.a = u1 ^ key.k0[1];                           // round 2: c0 = hi(M1 c2) ^ a
    s.b = (uint32_t)(q0 >> 32) ^ key.k1[1];         // round 2: c2 = c3 ^ b
    s.c = (uint32_t)q0 ^ key.k1[2];                 // round 3: c2 = hi(M0 c0) ^ c   (c3 after round 2 is lo(M0 u0))
    return s;
}

__device__ __forceinline__ uint4 philox_growth_block(uint32_t p, uint32_t k, const PhiloxStep& s, const PhiloxKey& key) {
    unsigned long long p0 = (unsigned long long)kPhiloxM0 * p;                  // round 1
    uint32_t c2 = (uint32_t)(p0 >> 32) ^ k ^ s.k10, c3 = (uint32_t)p0;
    unsigned long long p1 = (unsigned long long)kPhiloxM1 * c2;                 // round 2
    uint32_t c0 = (uint32_t)(p1 >> 32) ^ s.a, c1 = (uint32_t)p1;
    c2 = c3 ^ s.b;
    p0 = (unsigned long long)kPhiloxM0 * c0;                                    // round 3
    p1 = (unsigned long long)kPhiloxM1 * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[2];
    c1 = (uint32_t)p1;
    c2 = (uint32_t)(p0 >> 32) ^ s.c;
    c3 = (uint32_t)p0;
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        p0 = (unsigned long long)kPhiloxM0 * c0;
        p1 = (unsigned long long)kPhiloxM1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[r];
        c1 = (uint32_t)p1;
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[r];
        c3 = (uint32_t)p0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// ---------------------------------------------------------------------------------------------
// Control block: all loop state lives in HBM so that the step loop needs no host round trip.
// ---------------------------------------------------------------------------------------------
constexpr int kStatusRunning = -100;
constexpr uint32_t kLogCap = 4096;

struct Control {
    unsigned long long n_solid;      // solid count (phi_a = n_solid / N)
    unsigned long long n_t;          // target count ceil(phi_s N) (R7)
    unsigned long long R[3];         // reference thresholds floor(G_ref 2^32 + .5): face, edge, corner (R8)
    unsigned long long N;
    unsigned long long n_free;       // N minus the cells of earlier phases (liets_set_blocked): the most this phase can hold
    unsigned long long pool_head;    // seeding: entries handed out from the adjacency pool (64-bit: may run far past its size)
    uint32_t U[3];                   // T - 1 of the current step's thresholds T in [1, 2^32] (Eq. (1)):
                                     // a draw fires iff draw <= U
    uint32_t en[3];                  // T >= 1; a class with T == 0 never fires
    uint32_t hpat[8][4];             // [k][w]: nibble k (most significant first) of U of the class of each nibble's direction
    uint32_t en26;                   // directions whose class can fire at all
    uint32_t h0_any;                 // some class has a non-zero leading nibble: level 0 can fire without a tie
    uint32_t tile_cursor;            // STORAGE_TILE: next list entry to hand out (dynamic tile scheduling)
    uint32_t law;
    uint32_t has_target;
    uint32_t step;                   // t, continues across step / generate calls
    uint32_t steps_done;             // by the current generate call
    uint32_t max_steps;
    uint32_t active;                 // the step between two control kernels is live
    int32_t  status;                 // kStatusRunning or a LIETS_* status
    uint32_t cur;                    // which of the two front lists is A_t
    uint32_t count[2];               // entries in each front list (STORAGE_TILE: the heavy tiles, filled from the front)
    uint32_t count_back[2];          // STORAGE_TILE: light tiles of each list, filled from the back of the array
    uint32_t list_cap;               // STORAGE_TILE: slots per list
    uint32_t claims;                 // voxels claimed by the live step (added to n_solid at finish)
    uint32_t n_cand;                 // seeding: candidates
    uint32_t pend3[3];               // seeding: pending candidates after round r, at index r % 3
    uint32_t spacing_slow;           // seeding: the adjacency lists do not fit the fast resolve -> rescan rounds
    uint32_t spacing_rounds;         // seeding: rounds of the keyed-order / dense-dilation spacing (0 for the default path)
    uint32_t interact;               // R20: cells of the earlier phases with a void neighbour are sources, with thresholds I
    uint32_t enI26;                  // ... directions whose interaction class can fire at all
    uint32_t hpatI[8][4];            // ... the interaction thresholds nibble by nibble, laid out like hpat (constant over the run)
    uint32_t items;                  // Philox blocks evaluated by the live step (profiling counter)
    uint32_t items0;                 // front voxels with a void target in the live step (= level-0 blocks)
    // STORAGE_TILE keeps the active set as a voxel list while it is small (grow_vox.cu) and as a tile list afterwards
    uint32_t mode;                   // 0: voxel list (both grid copies identical), 1: tile list (always 1 for STORAGE_U8), 2: no list (STORAGE_FULL)
    uint32_t pending;                // the live step is the first one on tiles: k_tiles_from_grid fills its list
    uint32_t vox_count[2];           // entries of each voxel list
    uint32_t vox_cap;                // slots per voxel list
    uint32_t vox_thr;                // hand over to tiles when a step starts with more front voxels than this
    uint32_t vox_overflow;           // an append did not fit: the list is incomplete (the grid is exact)
    unsigned long long log_front[kLogCap];
    unsigned long long log_solid[kLogCap];
    unsigned long long log_items[kLogCap];
    unsigned long long log_items0[kLogCap];
    uint32_t scan_sums[1024];        // seeding: per-CTA sums of the chunk-count prefix scan
};

// control-kernel flags
enum : uint32_t { kCtlFinish = 1u, kCtlPrepare = 2u, kCtlForce = 4u, kCtlEval = 8u };

__device__ __forceinline__ uint32_t warp_exclusive_scan(uint32_t v, uint32_t lane, uint32_t* total) {
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += n;
    }
    *total = __shfl_sync(0xffffffffu, incl, 31);
    return incl - v;
}

}  // namespace liets

namespace liets {

// CTA-wide exclusive scan of one value per thread (blockDim.x <= 1024, multiple of 32).
// smem: at least 33 uint32.  Returns the exclusive prefix; *total = sum over the CTA.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* smem, uint32_t* total) {
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    uint32_t wtotal;
    uint32_t excl = warp_exclusive_scan(v, lane, &wtotal);
    __syncthreads();                       // protect smem reuse across calls
    if (lane == 0) smem[warp] = wtotal;
    __syncthreads();
    if (warp == 0) {
        uint32_t t = lane < nwarp ? smem[lane] : 0u, tt;
        uint32_t e = warp_exclusive_scan(t, lane, &tt);
        smem[lane] = e;
        if (lane == 0) smem[32] = tt;
    }
    __syncthreads();
    *total = smem[32];
    return excl + smem[warp];
}

// direction d (0..25) -> offsets; R1: lexicographic in (dz, dy, dx), dz slowest, centre skipped.
__host__ __device__ constexpr int dir_raw(int d) { return d + (d >= 13 ? 1 : 0); }
__host__ __device__ constexpr int dir_dx(int d) { return dir_raw(d) % 3 - 1; }
__host__ __device__ constexpr int dir_dy(int d) { return (dir_raw(d) / 3) % 3 - 1; }
__host__ __device__ constexpr int dir_dz(int d) { return dir_raw(d) / 9 - 1; }
__host__ __device__ constexpr int dir_class(int d) {       // 0 face, 1 edge, 2 corner
    return (dir_dx(d) != 0) + (dir_dy(d) != 0) + (dir_dz(d) != 0) - 1;
}

// ---------------------------------------------------------------------------------------------
// The per-step thresholds in the form the two-level draw needs (all warp-uniform).
//   U = T - 1, H = U >> 28 (top nibble), L = U & 0x0FFFFFFF.  draw <= U  <=>  nib < H, or nib == H and low28 <= L.
// Direction d owns nibble d>>2 of word d&3.  A mask that holds one flag per nibble of word w at bit 3 of the
// nibble, shifted right by 3 - w, has the flag of direction d at bit d: the four words interleave into a
// mask in direction order without any bit permutation.
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr uint32_t class_nibble_ones(int w, int cls) {      // 0x1 in every nibble n of word w whose direction 4n+w is of class cls
    uint32_t m = 0;
    for (int n = 0; n < 7; ++n)
        if (4 * n + w < 26 && dir_class(4 * n + w) == cls) m |= 1u << (4 * n);
    return m;
}
__host__ __device__ constexpr uint32_t class_dir_mask(int cls) {                // bit d set iff direction d is of class cls
    uint32_t m = 0;
    for (int d = 0; d < 26; ++d)
        if (dir_class(d) == cls) m |= 1u << d;
    return m;
}

// Per-nibble compares of a Philox word a with a pattern word h, carry-free: the result has bit 3 of nibble n set
// iff the relation holds for nibble n.
__device__ __forceinline__ uint32_t nib_le(uint32_t a, uint32_t h) {            // a <= h
    const uint32_t dd = (h | 0x88888888u) - (a & 0x77777777u);                  // bit 3: low 3 bits of h >= those of a
    return ((h & ~a) | (~(h ^ a) & dd)) & 0x88888888u;
}
__device__ __forceinline__ uint32_t nib_eq(uint32_t a, uint32_t h) {            // a == h
    const uint32_t z = a ^ h;
    return ~(((z & 0x77777777u) + 0x77777777u) | z | 0x77777777u);
}
// four per-word masks (flag of nibble n at bit 4n+3) -> one mask in direction order (flag of direction d at bit d)
__device__ __forceinline__ uint32_t interleave_dirs(uint32_t m0, uint32_t m1, uint32_t m2, uint32_t m3) {
    // the flags do not overlap, so the left shifts and ORs can be multiply-adds (FMA pipe), one right shift at the end
    return (m0 + 2u * m1 + 4u * m2 + 8u * m3) >> 3;
}
// For the directions in `mask`: le = nibble of block B <= the threshold's nibble, eq = they tie.
__device__ __forceinline__ void level_compare(const uint4& B, const uint32_t* h, uint32_t mask, uint32_t* le, uint32_t* eq) {
    const uint32_t l0 = nib_le(B.x, h[0]), l1 = nib_le(B.y, h[1]), l2 = nib_le(B.z, h[2]), l3 = nib_le(B.w, h[3]);
    const uint32_t e0 = nib_eq(B.x, h[0]), e1 = nib_eq(B.y, h[1]), e2 = nib_eq(B.z, h[2]), e3 = nib_eq(B.w, h[3]);
    *le = interleave_dirs(l0, l1, l2, l3) & mask;
    *eq = interleave_dirs(e0, e1, e2, e3) & mask;
}

// Level 0 with the uniform parts of the compare precomputed: hm = h & 0x8888.., h8 = h | 0x8888..
__device__ __forceinline__ void level0_compare(const uint4& B, const uint32_t* h, const uint32_t* hm, const uint32_t* h8,
                                               uint32_t mask, uint32_t* le, uint32_t* eq) {
    const uint32_t a[4] = { B.x, B.y, B.z, B.w };
    uint32_t l[4], e[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t dd = (h8[w] - (a[w] & 0x77777777u)) & 0x88888888u;      // bit 3: low 3 bits of h >= those of a
        l[w] = (hm[w] & ~a[w]) | (~(hm[w] ^ a[w]) & dd);                        // only bit 3 of each nibble survives
        const uint32_t z = a[w] ^ h[w];
        e[w] = ~(((z & 0x77777777u) + 0x77777777u) | z | 0x77777777u);
    }
    *le = interleave_dirs(l[0], l[1], l[2], l[3]) & mask;
    *eq = interleave_dirs(e[0], e[1], e[2], e[3]) & mask;
}

// Level 0 when every leading threshold nibble is below 8 (every class has probability < 1/2 in this step): with the top bit
// of h clear, a <= h  <=>  a's top bit is clear and its low three bits do not exceed h's, i.e. bit 3 of a | ((a & 7) + (7 - h))
// is clear -- three instructions per word, like the zero test.  a < h is the same test against h - 1 in the nibbles
// where h != 0.  cle = 0x777.. - h, clt = 0x777.. - (h - 1 where h != 0), hnz = 0x8 in the nibbles where h != 0: uniform.
__device__ __forceinline__ void level0_compare_small(const uint4& B, const uint32_t* cle, const uint32_t* clt, const uint32_t* hnz,
                                                     uint32_t mask, uint32_t* lt, uint32_t* eq) {
    const uint32_t a[4] = { B.x, B.y, B.z, B.w };
    uint32_t l[4], t[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t al = a[w] & 0x77777777u;
        l[w] = ~(a[w] | (al + cle[w])) & 0x88888888u;                           // a <= h
        t[w] = ~(a[w] | (al + clt[w])) & hnz[w];                                // a < h
    }
    const uint32_t le = interleave_dirs(l[0], l[1], l[2], l[3]);
    *lt = interleave_dirs(t[0], t[1], t[2], t[3]) & mask;
    *eq = le & ~*lt & mask;
}

// all-zero thresholds nibbles (every class has probability < 1/16): "<=" is "== 0"; flag at bit 3 of zero nibbles
__device__ __forceinline__ uint32_t nib_is_zero(uint32_t a) {
#ifdef LIETS_ZERO_MUL
    // bit 3 of a nibble of a | a<<1 | a<<2 | a<<3 is the OR of the nibble's four bits (nothing crosses into bit 3 from the
    // nibble below); the left shifts are multiplies (FMA pipe), two three-input logic ops remain on the ALU pipe
    const uint32_t u = a | (a * 2u);
    return ~(u | (u * 4u)) & 0x88888888u;
#else
    return ~(((a & 0x77777777u) + 0x77777777u) | a | 0x77777777u);
#endif
}
__device__ __forceinline__ uint32_t level_zero(const uint4& B, uint32_t mask) {
    return interleave_dirs(nib_is_zero(B.x), nib_is_zero(B.y), nib_is_zero(B.z), nib_is_zero(B.w)) & mask;
}

// Levels 1..7 for the directions of voxel p that tied at level 0: returns the directions that fire.
__device__ __forceinline__ uint32_t resolve_ties(uint32_t p, uint32_t t, uint32_t tie, const uint32_t (*hpat)[4],
                                                 const PhiloxKey& key, uint32_t* n_blocks) {
    uint32_t fire = 0;
    const PhiloxStep ps = philox_step_uniform(t, key);
    for (uint32_t k = 1; k < 8u && tie; ++k) {
        const uint4 B = philox_growth_block(p, k, ps, key);
        uint32_t le, eq;
        level_compare(B, hpat[k], tie, &le, &eq);
        ++*n_blocks;
        if (k < 7u) { fire |= le & ~eq; tie = eq; }
        else fire |= le;                                                        // last nibble: draw <= U
    }
    return fire;
}


// ---------------------------------------------------------------------------------------------
// The step loop's control logic (control.cu explains the protocol).
// ---------------------------------------------------------------------------------------------
// T = min(2^32, floor(R * max(0, 20 n_t - 19 n_solid) / n_t)) without 128-bit arithmetic:
// a = 20 n_t - 19 n_solid = q n_t + r  =>  floor(R a / n_t) = R q + floor(R r / n_t),
// with q <= 20, R <= 2^32, r < n_t <= 2^32, so every product fits 64 bits.
__device__ __forceinline__ unsigned long long eq1_threshold(unsigned long long R, unsigned long long n_t,
                                            unsigned long long n_solid) {
    unsigned long long a = 20ull * n_t, b = 19ull * n_solid;
    if (b >= a) return 0ull;
    a -= b;
    unsigned long long q = a / n_t, r = a % n_t;
    unsigned long long T = R * q + (R * r) / n_t;
    return T > (1ull << 32) ? (1ull << 32) : T;
}

// One call by ONE WARP (all 32 lanes, converged) between two growth kernels.  All inputs are read up front in one batch of
// L2 loads, the same by every lane (fields that other CTAs update with atomics must not come from L1); the scalar logic
// runs redundantly on registers and lane 0 stores its results; the two parts that cost time on a single thread are spread:
// the three thresholds of Eq. (1) (64-bit divisions) on lanes 0-2, the 32 words of the nibble layout one per lane.  This
// call sits on the critical path of every step (between two growth launches, or between two grid barriers).
static __device__ __noinline__ void control_step(Control* c, uint32_t flags) {
    const uint32_t lane = threadIdx.x & 31u;
    const bool lead = lane == 0u;
    unsigned long long n_solid = __ldcg(&c->n_solid);
    const unsigned long long n_t = __ldcg(&c->n_t), N = __ldcg(&c->n_free);     // (cells this phase can ever hold)
    const unsigned long long R_mine = __ldcg(&c->R[lane < 3u ? lane : 0u]);
    const uint32_t claims = __ldcg(&c->claims), items = __ldcg(&c->items), items0 = __ldcg(&c->items0);
    uint32_t mode = __ldcg(&c->mode), pending = __ldcg(&c->pending);
    const uint32_t vox_thr = __ldcg(&c->vox_thr), vox_overflow = __ldcg(&c->vox_overflow);
    uint32_t count[2];
    const uint32_t interact = __ldcg(&c->interact);
    if (mode == 0u && !pending) { count[0] = __ldcg(&c->vox_count[0]); count[1] = __ldcg(&c->vox_count[1]); }
    else if (mode == 2u) { count[0] = count[1] = (n_solid != 0ull || interact) ? 1u : 0u; }      // the full-field sweep keeps no list
    else { count[0] = __ldcg(&c->count[0]) + __ldcg(&c->count_back[0]); count[1] = __ldcg(&c->count[1]) + __ldcg(&c->count_back[1]); }
    const uint32_t law = __ldcg(&c->law), max_steps = __ldcg(&c->max_steps);
    uint32_t step = __ldcg(&c->step), steps_done = __ldcg(&c->steps_done), cur = __ldcg(&c->cur);
    uint32_t active = __ldcg(&c->active);
    int32_t status = __ldcg(&c->status);
    __syncwarp();                                        // every lane has read the state before lane 0 changes it
    if ((flags & kCtlFinish) && active) {                // close the step that just ran
        n_solid += claims;                               // phi_a update
        if (lead) {
            c->n_solid = n_solid;
            if (step < kLogCap) { c->log_solid[step] = n_solid; c->log_items[step] = items; c->log_items0[step] = items0; }
        }
        cur ^= 1u;                                       // A <- prune(A U A_new) (R4)
        step += 1;
        steps_done += 1;
        active = 0;
        if (lead) { c->cur = cur; c->step = step; c->steps_done = steps_done; c->active = 0; c->claims = 0; }
        if (pending) {                                   // that was the first step on tiles
            mode = 1u; pending = 0u;
            if (lead) { c->mode = 1u; c->pending = 0u; }
        }
    }
    if (!(flags & (kCtlPrepare | kCtlEval))) return;
    if (!(flags & kCtlForce)) {                          // stop rule, between whole steps only
        if (status != kStatusRunning) return;
        if (n_solid >= n_t) status = 0;                                      // LIETS_OK
        else if ((count[cur] == 0 && !(interact && mode == 0u)) || n_solid == N) status = 1;   // FRONT_EMPTY (R20: the interface sources are listed with the tiles)
        else if (steps_done >= max_steps) status = 2;                        // MAX_STEPS
        if (status != kStatusRunning) { if (lead) c->status = status; return; }
    }
    if (!(flags & kCtlPrepare)) return;
    // Eq. (1): lane k < 3 evaluates class k
    uint32_t U_mine = 0, en_mine = 0;
    if (lane < 3u) {
        const unsigned long long T = law ? eq1_threshold(R_mine, n_t, n_solid) : R_mine;
        en_mine = T >= 1ull;                                                 // T in [0, 2^32]
        U_mine = T >= 1ull ? (uint32_t)(T - 1ull) : 0u;                      // draw < T  <=>  draw <= T - 1
        c->en[lane] = en_mine;
        c->U[lane] = U_mine;
    }
    uint32_t U[3], en[3], en26 = 0, h0_any = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        U[k] = __shfl_sync(0xffffffffu, U_mine, k);
        en[k] = __shfl_sync(0xffffffffu, en_mine, k);
        if (en[k]) en26 |= class_dir_mask(k);
        if (en[k] && (U[k] >> 28)) h0_any = 1;
    }
    // the thresholds nibble by nibble, laid out like the draws (direction d: nibble d>>2 of word d&3): lane = 4 level + word
    {
        const uint32_t lv = lane >> 2, w = lane & 3u;
        uint32_t ones[3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
            ones[k] = w == 0u ? class_nibble_ones(0, k) : w == 1u ? class_nibble_ones(1, k) : w == 2u ? class_nibble_ones(2, k) : class_nibble_ones(3, k);
        c->hpat[lv][w] = ((U[0] >> (28u - 4u * lv)) & 15u) * ones[0] + ((U[1] >> (28u - 4u * lv)) & 15u) * ones[1] +
                         ((U[2] >> (28u - 4u * lv)) & 15u) * ones[2];
    }
    if (mode == 0u && (count[cur] > vox_thr || vox_overflow || interact)) pending = 2u;  // the front has outgrown the voxel list: this step
                                                                             // runs on tiles (2: handed over in this very call)
    if (lead) {
        c->en26 = en26;
        c->h0_any = h0_any;
        c->tile_cursor = 0;
        c->count[cur ^ 1u] = 0;
        c->count_back[cur ^ 1u] = 0;
        if (mode == 0u) {
            c->vox_count[cur ^ 1u] = 0;
            if (pending == 2u) {
                c->pending = 1u;
                c->count[cur] = 0;                          // k_tiles_from_grid fills the list of this step
                c->count_back[cur] = 0;
            }
        }
        c->claims = 0;
        c->items = 0;
        c->items0 = 0;
        // entries of the list the step starts from; bit 63: the step runs on tiles (k_grow_tile); bit 62: it is the
        // hand-over step, whose tile list k_tiles_from_grid has yet to fill -- the count is still the voxel list's
        if (step < kLogCap)
            c->log_front[step] = (unsigned long long)count[cur] | ((mode != 0u || pending) ? (1ull << 63) : 0ull) | (pending == 2u ? (1ull << 62) : 0ull);
        c->active = 1;
    }
}

}  // namespace liets
