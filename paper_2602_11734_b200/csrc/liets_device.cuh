// liets_device.cuh -- device-side building blocks shared by the kernels of libliets.so.
// (Product code: shares nothing with oracle/.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace liets {

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11) -- the counter-based stream of DESIGN.md reading R9
// ("an independent random number in (0,1) is drawn").
//   growth:  key = (rng_seed lo, hi), counter = (p lo, p hi, step t, d>>2), draw of direction d = word d&3
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
    uint32_t T[3];                   // thresholds of the current step (Eq. (1))
    uint32_t always[3];              // T == 2^32: fire regardless of the draw
    uint32_t law;
    uint32_t has_target;
    uint32_t step;                   // t, continues across step / generate calls
    uint32_t steps_done;             // by the current generate call
    uint32_t max_steps;
    uint32_t active;                 // the step between two control kernels is live
    int32_t  status;                 // kStatusRunning or a LIETS_* status
    uint32_t cur;                    // which of the two front lists is A_t
    uint32_t count[2];               // entries in each front list
    uint32_t claims;                 // voxels claimed by the live step (added to n_solid at finish)
    uint32_t n_cand;                 // seeding: candidates
    uint32_t pool_head;              // seeding: used entries of the adjacency pool
    uint32_t n_rescan;               // seeding: candidates whose adjacency was not stored
    uint32_t pend3[3];               // seeding: pending candidates after round r, at index r % 3
    uint32_t items;                  // Philox blocks evaluated by the live step (profiling counter)
    unsigned long long log_front[kLogCap];
    unsigned long long log_solid[kLogCap];
    unsigned long long log_items[kLogCap];
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

}  // namespace liets
