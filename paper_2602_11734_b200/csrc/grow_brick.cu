// grow_brick.cu -- STORAGE_BRICK growth step: bit-packed 8x8x8 bricks + explicit list of front BRICKS.
//
// Layout in HBM.  The grid is cut into 8x8x8 bricks of 64 bytes: eight 64-bit words, word z holds
// z-slice z of the brick, bit (x + 8y).  Two copies G[0], G[1] are kept: step t reads G[t&1]
// (immutable during the step, so the update is synchronous by construction) and ORs
// into G[(t+1)&1].  The active set A is kept as a list of bricks that hold at least
// one front voxel; which voxels of a brick are front voxels is recomputed from the bits, so the
// list costs 4 bytes per 512 voxels instead of 4 bytes per front voxel.
//
// One warp owns one brick at a time:
//   A  gather: the brick and the needed words of its 26 neighbour bricks -> shared memory, then the
//      10x10x10 neighbourhood as 100 rows of 10 bits ("not void" = solid, outside the domain, or padding)
//   B  masks: per interior row, the 26 void-target masks (Algorithm 3 lines 5-6) as bit operations;
//      every (voxel, Philox block) pair with a void target is one set bit of a flat 3584-bit map in
//      shared memory; the lanes split that map by RANK (lane l takes set bits [l n/32, (l+1) n/32)),
//      so the Philox work is spread evenly over the 32 lanes whatever the shape of the front
//   C  draw + test: one Philox4x32-10 block per item, <= 4 directions tested against the integer
//      thresholds (line 8); hits set bits in a shared-memory claim volume
//   D  claim + compact: own slices are OR-ed into G[next] together with the carried state, halo hits
//      go to the neighbour bricks with atomicOr; the returned old word tells who flipped the bit
//      (line 9-10, "counted once" PAPER.md:77) for the solid count; a per-brick step stamp
//      (atomicMax) makes every brick enter the next list exactly once; bricks without front voxels
//      are not re-emitted (lazy retirement).
#include "liets_host.h"

namespace liets {

namespace {

constexpr int kWarpsPerCta = 8;
constexpr uint32_t kHole = 0xFFFFFFFFu;     // unused slot of a warp's list chunk
constexpr int kChunk = 8;                   // list slots a warp reserves at a time

struct __align__(16) WarpSmem {
    union {
        unsigned long long nbw[27][8];      // phase A: words of the 27 bricks (own = index 13)
        uint2 nz[7 * 64 / 4 + 4];           // phases B-C: the non-zero words of U, in order: (word, word index)
    };
    unsigned long long own[8];              // this brick's words (carried into the next grid copy)
    uint32_t V[7 * 64];                     // [block b][row]: the 4 void-target masks (8 bits each) of block b
    uint32_t U[7 * 64 / 4];                 // [block b][row] bytes: OR of the 4 masks = voxels needing block b
    uint32_t rows[100];                     // 10 bits per row: bit (x'+1), rows (z'+1)*10 + (y'+1)
    uint32_t claims[100];                   // same geometry: cells claimed in this step
    uint32_t rowbase[64];                   // linear voxel index of (x=0, y, z) of the interior rows
    uint4 T4[7];                            // per Philox block: T-1 of its 4 directions (fire iff draw <= T-1)
    uint32_t dir[28];                       // direction d: (row delta + 11) | (dx + 1) << 8 in the 10x10x10 geometry
};

// region index i in [-1, 8] along one axis of brick b -> brick index (or -1: no such cell) and local coordinate
__device__ __forceinline__ void axis_map(int i, int b, int nb, int n, int periodic, int* ob, int* l) {
    const int wc = min(8, n - 8 * b);
    if (i < 0) {
        if (b > 0) { *ob = b - 1; *l = 7; }
        else if (periodic) { *ob = nb - 1; *l = n - 8 * (nb - 1) - 1; }
        else { *ob = -1; *l = 0; }
    } else if (i < wc) {
        *ob = b; *l = i;
    } else if (i == wc) {
        if (b < nb - 1) { *ob = b + 1; *l = 0; }
        else if (periodic) { *ob = 0; *l = 0; }
        else { *ob = -1; *l = 0; }
    } else {
        *ob = -1; *l = 0;
    }
}

struct StepParams {
    uint32_t T[3];
    uint32_t always[3];
    uint32_t t;
};

__global__ void __launch_bounds__(kWarpsPerCta * 32, 4) k_grow_brick(Control* __restrict__ ctl, BrickGeom g,
                                                                    unsigned long long* G0, unsigned long long* G1,
                                                                    uint32_t* stamp, uint32_t* list0, uint32_t* list1,
                                                                    PhiloxKey key) {
    if (!ctl->active) return;
    __shared__ WarpSmem s_ws[kWarpsPerCta];  // static: addresses are compile-time constants + warp offset
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    WarpSmem& S = s_ws[warp];

    const uint32_t cur = ctl->cur;
    const uint32_t n_list = ctl->count[cur];
    const uint32_t* __restrict__ in = cur ? list1 : list0;
    uint32_t* __restrict__ out = cur ? list0 : list1;
    uint32_t* out_count = &ctl->count[cur ^ 1u];
    const uint32_t t = ctl->step;
    const unsigned long long* __restrict__ Gc = (t & 1u) ? G1 : G0;     // g_t (read only)
    unsigned long long* Gn = (t & 1u) ? G0 : G1;                        // g_{t+1} (OR target)
    if (lane < 28) {                        // every warp keeps its own copy: one base register serves all tables
        const int d = lane < 26 ? (int)lane : 25;
        const int raw = d + (d >= 13 ? 1 : 0);
        const int dx = raw % 3 - 1, dy = (raw / 3) % 3 - 1, dz = raw / 9 - 1;
        const int cls = (dx != 0) + (dy != 0) + (dz != 0) - 1;
        // T in [0, 2^32]: "draw < T" == "draw <= T-1" for T >= 1; directions with T = 0 are disabled in phase B
        const uint32_t tm1 = ctl->always[cls] ? 0xFFFFFFFFu : ctl->T[cls] - 1u;
        reinterpret_cast<uint32_t*>(S.T4)[lane] = tm1;
        S.dir[lane] = (uint32_t)(dz * 10 + dy + 11) | ((uint32_t)(dx + 1) << 8);
    }
    __syncwarp();
    // a class whose threshold is 0 never fires: its directions produce no work
    const uint32_t en0 = (ctl->T[0] | ctl->always[0]) ? 0xFFu : 0u;
    const uint32_t en1 = (ctl->T[1] | ctl->always[1]) ? 0xFFu : 0u;
    const uint32_t en2 = (ctl->T[2] | ctl->always[2]) ? 0xFFu : 0u;

    uint32_t new_solid = 0;                 // per lane: bits this lane flipped 0 -> 1
    uint32_t n_items = 0;                   // lane 0: Philox blocks this warp evaluated
    uint32_t chunk_pos = 0, chunk_end = 0;  // lane 0: reserved slots of the next list

    const uint32_t warp_global = blockIdx.x * kWarpsPerCta + warp;
    const uint32_t n_warps = gridDim.x * kWarpsPerCta;
    for (uint32_t li = warp_global; li < n_list; li += n_warps) {
        const uint32_t id = in[li];
        if (id == kHole) continue;
        const int bxi = (int)(id % (uint32_t)g.bx), byi = (int)((id / (uint32_t)g.bx) % (uint32_t)g.by),
                  bzi = (int)(id / ((uint32_t)g.bx * (uint32_t)g.by));
        const int wcx = min(8, g.nx - 8 * bxi), wcy = min(8, g.ny - 8 * byi), wcz = min(8, g.nz - 8 * bzi);

        // ---- A: gather ------------------------------------------------------------------------
        if (lane < 27) {
            const int ox = (int)lane % 3 - 1, oy = ((int)lane / 3) % 3 - 1, oz = (int)lane / 9 - 1;
            int obx, oby, obz, lx, ly, lz;
            axis_map(ox < 0 ? -1 : (ox == 0 ? 0 : wcx), bxi, g.bx, g.nx, g.periodic, &obx, &lx);
            axis_map(oy < 0 ? -1 : (oy == 0 ? 0 : wcy), byi, g.by, g.ny, g.periodic, &oby, &ly);
            axis_map(oz < 0 ? -1 : (oz == 0 ? 0 : wcz), bzi, g.bz, g.nz, g.periodic, &obz, &lz);
            if (obx < 0 || oby < 0 || obz < 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) S.nbw[lane][k] = ~0ull;      // outside the domain: never void
            } else {
                const unsigned long long* src = Gc + 8ull * ((unsigned long long)obx +
                                                             (unsigned long long)g.bx * ((unsigned long long)oby + (unsigned long long)g.by * (unsigned long long)obz));
                if (oz == 0) {
                    const ulonglong2* s2 = reinterpret_cast<const ulonglong2*>(src);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const ulonglong2 v = __ldcg(s2 + k);
                        S.nbw[lane][2 * k] = v.x; S.nbw[lane][2 * k + 1] = v.y;
                    }
                } else {
                    S.nbw[lane][lz] = __ldcg(src + lz);                  // only the touching slice
                }
            }
        }
        __syncwarp();
        if (lane < 8) S.own[lane] = S.nbw[13][lane];
        // local coordinates of the cells just outside the brick on the low side
        const int lxl = bxi > 0 ? 7 : g.nx - 8 * (g.bx - 1) - 1;
        const int lyl = byi > 0 ? 7 : g.ny - 8 * (g.by - 1) - 1;
        const int lzl = bzi > 0 ? 7 : g.nz - 8 * (g.bz - 1) - 1;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int r = (int)lane + 32 * k;
            if (r < 100) {
                const int zp = r / 10 - 1, yp = r % 10 - 1;
                uint32_t row = 0x3FFu;
                if (zp <= wcz && yp <= wcy) {
                    const int ozi = zp < 0 ? 0 : (zp < wcz ? 1 : 2), lz = zp < 0 ? lzl : (zp < wcz ? zp : 0);
                    const int oyi = yp < 0 ? 0 : (yp < wcy ? 1 : 2), ly = yp < 0 ? lyl : (yp < wcy ? yp : 0);
                    const int jc = 1 + 3 * oyi + 9 * ozi;
                    const uint32_t c = (uint32_t)(S.nbw[jc][lz] >> (8 * ly)) & 0xFFu;
                    const uint32_t left = (uint32_t)(S.nbw[jc - 1][lz] >> (8 * ly + lxl)) & 1u;
                    const uint32_t right = (uint32_t)(S.nbw[jc + 1][lz] >> (8 * ly)) & 1u;
                    row = left | ((c & ((1u << wcx) - 1u)) << 1) | (right << (wcx + 1)) | ((0x3FFu << (wcx + 2)) & 0x3FFu);
                }
                S.rows[r] = row;
                S.claims[r] = 0u;
            }
        }
        __syncwarp();

        // ---- B: masks and the flat work map ---------------------------------------------------------
        uint32_t front_bits = 0;            // sources of this lane's rows that have a void neighbour (R13)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int r2 = (int)lane + 32 * h, y = r2 & 7, z = r2 >> 3;
            uint32_t src = 0;
            if (y < wcy && z < wcz) src = (S.rows[(z + 1) * 10 + (y + 1)] >> 1) & ((1u << wcx) - 1u);
            const uint32_t src_c[3] = { src & en0, src & en1, src & en2 };
            uint32_t M[28];
            M[26] = 0; M[27] = 0;
            uint32_t anyvoid = 0;
#pragma unroll
            for (int d = 0; d < 26; ++d) {
                const uint32_t voidrow = ~S.rows[(z + dir_dz(d) + 1) * 10 + (y + dir_dy(d) + 1)];
                M[d] = src_c[dir_class(d)] & (voidrow >> (dir_dx(d) + 1));
                if (dir_dx(d) == 0 || d == 12) anyvoid |= voidrow;          // each of the 9 rows once
            }
            front_bits |= src & (anyvoid | (anyvoid >> 1) | (anyvoid >> 2));
#pragma unroll
            for (int b = 0; b < 7; ++b) {
                const uint32_t v = M[4 * b] | (M[4 * b + 1] << 8) | (M[4 * b + 2] << 16) | (M[4 * b + 3] << 24);
                const uint32_t u = M[4 * b] | M[4 * b + 1] | M[4 * b + 2] | M[4 * b + 3];
                S.V[b * 64 + r2] = v;
                reinterpret_cast<uint8_t*>(S.U)[b * 64 + r2] = (uint8_t)u;
            }
            S.rowbase[r2] = (uint32_t)(8 * bxi) + (uint32_t)g.nx * ((uint32_t)(8 * byi + y) + (uint32_t)g.ny * (uint32_t)(8 * bzi + z));
        }
        __syncwarp();
        // rank partition: lanes 0..27 count 4 words each, scan, every lane takes an equal share of set bits;
        // the non-zero words are also copied to a dense list so that moving to the next word is one load
        uint32_t cnt = 0, nzc = 0;
        uint4 u4 = make_uint4(0u, 0u, 0u, 0u);
        if (lane < 28) {
            u4 = reinterpret_cast<const uint4*>(S.U)[lane];
            cnt = __popc(u4.x) + __popc(u4.y) + __popc(u4.z) + __popc(u4.w);
            nzc = (u4.x != 0u) + (u4.y != 0u) + (u4.z != 0u) + (u4.w != 0u);
        }
        uint32_t total, nz_total;
        const uint32_t excl = warp_exclusive_scan(cnt, lane, &total);
        const uint32_t nz_excl = warp_exclusive_scan(nzc, lane, &nz_total);
        {
            uint32_t k = nz_excl;
            if (u4.x) S.nz[k++] = make_uint2(u4.x, 4u * lane);
            if (u4.y) S.nz[k++] = make_uint2(u4.y, 4u * lane + 1u);
            if (u4.z) S.nz[k++] = make_uint2(u4.z, 4u * lane + 2u);
            if (u4.w) S.nz[k++] = make_uint2(u4.w, 4u * lane + 3u);
            if (lane == 31) S.nz[nz_total] = make_uint2(0xFFFFFFFFu, 0u);      // sentinel: never dereferenced as an item
        }
        __syncwarp();

        // ---- C: draw + test ---------------------------------------------------------------------------
        n_items += total;
        if (total) {
            const uint32_t first = (lane * total) >> 5, last = ((lane + 1u) * total) >> 5;
            // the lane whose 4 words hold item number `first`: largest o with excl[o] <= first
            uint32_t lo = 0, hi = 27;
#pragma unroll
            for (int it = 0; it < 5; ++it) {
                const uint32_t mid = (lo + hi + 1u) >> 1;
                const uint32_t e = __shfl_sync(0xffffffffu, excl, mid);
                if (e <= first) lo = mid; else hi = mid - 1u;
            }
            uint32_t rem = first - __shfl_sync(0xffffffffu, excl, lo);
            uint32_t k = __shfl_sync(0xffffffffu, nz_excl, lo);     // position in the non-zero list
            uint2 w = S.nz[k];
            if (last > first) {                                     // walk to the word that holds item `first`
                uint32_t pc = __popc(w.x);
                while (rem >= pc) { rem -= pc; w = S.nz[++k]; pc = __popc(w.x); }
            }
            uint32_t cur = w.x, wi = w.y;
            for (; rem; --rem) cur &= cur - 1u;                     // skip the set bits that belong to lower lanes
            // flat loop, one item per lane per iteration: the lanes stay in lockstep
            for (uint32_t n_left = last - first; n_left; --n_left) {
                if (cur == 0u) { w = S.nz[++k]; cur = w.x; wi = w.y; }
                const uint32_t bit = __ffs(cur) - 1u;
                cur &= cur - 1u;
                const uint32_t e = (wi << 2) + (bit >> 3), x = bit & 7u;    // e = b*64 + row
                const uint32_t b = e >> 6, r2 = e & 63u;
                const uint32_t p = S.rowbase[r2] + x;
                const uint4 rnd = philox4x32_10(p, 0u, t, b, key);
                const uint4 T4 = S.T4[b];
                if (rnd.x <= T4.x || rnd.y <= T4.y || rnd.z <= T4.z || rnd.w <= T4.w) {
                    // a draw fell below its threshold: claim the target if that direction was a void one
                    uint32_t fire = (rnd.x <= T4.x ? 1u : 0u) | (rnd.y <= T4.y ? 2u : 0u) | (rnd.z <= T4.z ? 4u : 0u) |
                                    (rnd.w <= T4.w ? 8u : 0u);
                    fire &= (((S.V[e] >> x) & 0x01010101u) * 0x10204080u) >> 28;
                    const uint32_t zy = 10u * (r2 >> 3) + (r2 & 7u);
                    while (fire) {
                        const uint32_t j = __ffs(fire) - 1u;
                        fire &= fire - 1u;
                        const uint32_t lut = S.dir[4u * b + j];
                        atomicOr(&S.claims[zy + (lut & 0xFFu)], 1u << (x + (lut >> 8)));
                    }
                }
            }
        }
        __syncwarp();

        // ---- D: claim + compact ---------------------------------------------------------------------
        const unsigned long long own_base = 8ull * id;
        if ((int)lane < wcz) {                                      // own slices: carry g_t and add the hits
            const int z = (int)lane;
            unsigned long long cw = 0;
#pragma unroll
            for (int y = 0; y < 8; ++y)
                if (y < wcy)
                    cw |= (unsigned long long)((S.claims[(z + 1) * 10 + (y + 1)] >> 1) & ((1u << wcx) - 1u)) << (8 * y);
            const unsigned long long val = S.own[z] | cw;
            if (cw) {
                const unsigned long long old = atomicOr(Gn + own_base + z, val);
                new_solid += __popcll(cw & ~old);
            } else if (val) {
                atomicOr(Gn + own_base + z, val);
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {                               // hits outside the brick
            const int r = (int)lane + 32 * k;
            if (r >= 100) continue;
            const int zp = r / 10 - 1, yp = r % 10 - 1;
            uint32_t hb = S.claims[r];
            const bool halo_row = zp < 0 || zp == wcz || yp < 0 || yp == wcy;
            if (!halo_row) hb &= 1u | (1u << (wcx + 1));
            while (hb) {
                const int i = __ffs(hb) - 1;
                hb &= hb - 1;
                int qbx, qby, qbz, qx, qy, qz;
                axis_map(i - 1, bxi, g.bx, g.nx, g.periodic, &qbx, &qx);
                axis_map(yp, byi, g.by, g.ny, g.periodic, &qby, &qy);
                axis_map(zp, bzi, g.bz, g.nz, g.periodic, &qbz, &qz);
                const uint32_t nb = (uint32_t)qbx + (uint32_t)g.bx * ((uint32_t)qby + (uint32_t)g.by * (uint32_t)qbz);
                const unsigned long long bit = 1ull << (qx + 8 * qy);
                const unsigned long long old = atomicOr(Gn + 8ull * nb + qz, bit);
                if (!(old & bit)) new_solid++;
                if (atomicMax(&stamp[nb], t + 2u) < t + 2u) out[atomicAdd(out_count, 1u)] = nb;   // newly active brick
            }
        }
        const bool has_front = __any_sync(0xffffffffu, front_bits != 0u);
        if (lane == 0 && has_front) {                               // this brick still has front voxels
            if (atomicMax(&stamp[id], t + 2u) < t + 2u) {
                if (chunk_pos == chunk_end) {
                    chunk_pos = atomicAdd(out_count, (uint32_t)kChunk);
                    chunk_end = chunk_pos + kChunk;
                }
                out[chunk_pos++] = id;
            }
        }
        __syncwarp();
    }
    if (lane == 0)
        for (; chunk_pos < chunk_end; ++chunk_pos) out[chunk_pos] = kHole;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) new_solid += __shfl_xor_sync(0xffffffffu, new_solid, o);
    if (lane == 0 && new_solid) atomicAdd(&ctl->claims, new_solid);
    if (lane == 0 && n_items) atomicAdd(&ctl->items, n_items);
}

}  // namespace

size_t grow_brick_smem_bytes() { return 0; }   // static shared memory only
int grow_brick_warps_per_cta() { return kWarpsPerCta; }
int grow_brick_chunk() { return kChunk; }

cudaError_t launch_grow_brick(liets_ctx* c) {
    static bool attr_set = false;
    if (!attr_set) {                                        // 4 CTAs x 40 KB of static shared memory per SM
        cudaError_t e = cudaFuncSetAttribute(k_grow_brick, cudaFuncAttributePreferredSharedMemoryCarveout,
                                             (int)cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const size_t smem = 0;
    const PhiloxKey key = philox_make_key(c->rng_seed);
    k_grow_brick<<<c->brick_grid, kWarpsPerCta * 32, smem, c->stream>>>(c->ctl, c->geom, c->G[0], c->G[1], c->stamp,
                                                                       c->list[0], c->list[1], key);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
