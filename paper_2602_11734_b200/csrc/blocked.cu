// blocked.cu -- cells of earlier growing phases (multi-phase QSGS, PAPER.md:40 step 4, independent phases): "The remaining
// phases are generated on the still unassigned cells ... its cores are placed and grown in the same way as for the first
// phase".  liets_set_blocked hands the library the cells the earlier phases took.  They are NOT VOID -- never cores, never
// claimed, and they close the neighbourhood of a front voxel like solid cells do -- and NOT OF THIS PHASE -- never sources,
// not counted, not in liets_grid's output.
//
// Kept twice: `pbits`, one bit per voxel in linear index order (LSB first: LIETS_FORMAT_BITS, so one phase's packed output
// is the next phase's input as it stands; the seeding reads 16 voxels of it per status word), and for the bit-row
// storages `prow`, the same cells in the grid's row layout.  After every seeding reset the cells are put into the grid:
// OR-ed into both copies of the bit rows (every void test then sees them without any change to the kernels; the tile and
// full-field kernels only mask them out of their SOURCES, one extra word per 64 cells), or written as byte value 2 into the
// uint8 grid (void is 0, this phase is 1; the voxel-list kernels take their sources from the list and need no change).
#include "../../include/liets.h"
#include "liets_host.h"

namespace liets {
namespace {

// uint8 mask (non-zero = taken), N bytes -> pbits
__global__ void __launch_bounds__(256) k_blocked_pack(const uint8_t* __restrict__ src, uint8_t* __restrict__ pbits, unsigned long long N) {
    const unsigned long long n_bytes = (N + 7ull) / 8ull;
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_bytes;
         b += (unsigned long long)gridDim.x * blockDim.x) {
        uint32_t out = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const unsigned long long v = 8ull * b + k;
            if (v < N && src[v]) out |= 1u << k;
        }
        pbits[b] = (uint8_t)out;
    }
}

// packed input: copy, clearing the bits beyond N in the last byte
__global__ void __launch_bounds__(256) k_blocked_copy(const uint8_t* __restrict__ src, uint8_t* __restrict__ pbits, unsigned long long N) {
    const unsigned long long n_bytes = (N + 7ull) / 8ull;
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_bytes;
         b += (unsigned long long)gridDim.x * blockDim.x) {
        uint32_t v = src[b];
        if (8ull * b + 8ull > N) v &= (1u << (uint32_t)(N - 8ull * b)) - 1u;
        pbits[b] = (uint8_t)v;
    }
}

__device__ __forceinline__ uint32_t pbit(const uint8_t* __restrict__ pbits, unsigned long long v) {
    return (pbits[v >> 3] >> (v & 7ull)) & 1u;
}

// pbits -> row layout (one thread per 64-bit row word) and the number of blocked cells
__global__ void __launch_bounds__(256) k_blocked_rows(const uint8_t* __restrict__ pbits, unsigned long long* __restrict__ prow,
                                                       int nx, int Wp, unsigned long long n_rows, unsigned long long* count) {
    unsigned long long mine = 0ull;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_rows * (unsigned long long)Wp;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long row = i / (unsigned long long)Wp;
        const int w = (int)(i - row * (unsigned long long)Wp);
        const int nvalid = min(64, nx - 64 * w);
        unsigned long long word = 0ull;
        const unsigned long long v0 = row * (unsigned long long)nx + 64ull * (unsigned long long)w;
        for (int b = 0; b < nvalid; ++b) word |= (unsigned long long)pbit(pbits, v0 + (unsigned long long)b) << b;
        prow[i] = word;
        mine += (unsigned long long)__popcll(word);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(count, mine);
}

// STORAGE_U8 has no rows: count from pbits (the bits beyond N are clear)
__global__ void __launch_bounds__(256) k_blocked_count(const uint8_t* __restrict__ pbits, unsigned long long n_bytes, unsigned long long* count) {
    unsigned long long mine = 0ull;
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_bytes;
         b += (unsigned long long)gridDim.x * blockDim.x)
        mine += (unsigned long long)__popc((uint32_t)pbits[b]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(count, mine);
}

// after the seeding reset: the earlier phases' cells go into the grid
__global__ void __launch_bounds__(256) k_blocked_apply_rows(const unsigned long long* __restrict__ prow, unsigned long long* G0,
                                                             unsigned long long* G1, unsigned long long n_words) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long p = prow[i];
        if (p) { G0[i] |= p; G1[i] |= p; }
    }
}
__global__ void __launch_bounds__(256) k_blocked_apply_u8(const uint8_t* __restrict__ pbits, uint8_t* grid, unsigned long long N) {
    for (unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; v < N;
         v += (unsigned long long)gridDim.x * blockDim.x)
        if (pbit(pbits, v)) grid[v] = 2;
}

// STORAGE_U8 output: this phase's cells only
__global__ void __launch_bounds__(256) k_u8_this_phase(const uint8_t* __restrict__ grid, uint8_t* __restrict__ dst, unsigned long long N) {
    for (unsigned long long v = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; v < N;
         v += (unsigned long long)gridDim.x * blockDim.x)
        dst[v] = grid[v] == 1 ? 1 : 0;
}

}  // namespace

// src_dev: the mask on the DEVICE in `format`; count_dev: a zeroed 64-bit counter on the device
cudaError_t launch_blocked_set(liets_ctx* c, const uint8_t* src_dev, int format, unsigned long long* count_dev) {
    const int grid = c->sm_count * 8;
    if (format == LIETS_FORMAT_U8) k_blocked_pack<<<grid, 256, 0, c->stream>>>(src_dev, c->pbits, c->N);
    else k_blocked_copy<<<grid, 256, 0, c->stream>>>(src_dev, c->pbits, c->N);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (c->storage == LIETS_STORAGE_U8)
        k_blocked_count<<<grid, 256, 0, c->stream>>>(c->pbits, (c->N + 7ull) / 8ull, count_dev);
    else
        k_blocked_rows<<<grid, 256, 0, c->stream>>>(c->pbits, c->prow, c->nx, c->geom.Wp, (unsigned long long)c->ny * (unsigned long long)c->nz, count_dev);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_blocked_apply(liets_ctx* c) {
    if (c->storage == LIETS_STORAGE_U8) k_blocked_apply_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(c->pbits, c->grid_u8, c->N);
    else k_blocked_apply_rows<<<c->sm_count * 8, 256, 0, c->stream>>>(c->prow, c->G[0], c->G[1], c->grid_words);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_u8_this_phase(liets_ctx* c, uint8_t* dst) {
    k_u8_this_phase<<<c->sm_count * 8, 256, 0, c->stream>>>(c->grid_u8, dst, c->N);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
