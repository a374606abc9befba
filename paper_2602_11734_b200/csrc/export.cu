// export.cu -- liets_grid format conversion on the device.
#include "liets_host.h"

namespace liets {

namespace {
// uint8 {0,1} per voxel -> LSB-first bits; one thread per output byte
__global__ void __launch_bounds__(256) k_pack_bits_u8(const uint8_t* __restrict__ grid, uint8_t* __restrict__ dst,
                                                       unsigned long long N) {
    const unsigned long long n_bytes = (N + 7ull) / 8ull;
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_bytes;
         b += (unsigned long long)gridDim.x * blockDim.x) {
        uint32_t out = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const unsigned long long v = 8ull * b + k;
            if (v < N && grid[v]) out |= 1u << k;
        }
        dst[b] = (uint8_t)out;
    }
}
// bit bricks -> uint8 {0,1} per voxel, x fastest: one thread per brick row (8 voxels)
__global__ void __launch_bounds__(256) k_unpack_bricks_u8(const unsigned long long* __restrict__ G, uint8_t* __restrict__ dst,
                                                           BrickGeom g, unsigned long long n_rows) {
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_rows;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long b = i >> 6;
        const uint32_t ly = (uint32_t)i & 7u, lz = ((uint32_t)i >> 3) & 7u;
        const uint32_t bxi = (uint32_t)(b % (unsigned long long)g.bx);
        const uint32_t byi = (uint32_t)((b / (unsigned long long)g.bx) % (unsigned long long)g.by);
        const uint32_t bzi = (uint32_t)(b / ((unsigned long long)g.bx * (unsigned long long)g.by));
        const uint32_t y = 8u * byi + ly, z = 8u * bzi + lz, x0 = 8u * bxi;
        if (y >= (uint32_t)g.ny || z >= (uint32_t)g.nz) continue;
        const uint32_t bits = (uint32_t)(G[8ull * b + lz] >> (8u * ly)) & 0xFFu;
        const unsigned long long base = (unsigned long long)x0 + (unsigned long long)g.nx * ((unsigned long long)y + (unsigned long long)g.ny * z);
        const uint32_t w = min(8u, (uint32_t)g.nx - x0);
        if (w == 8u && (base & 7ull) == 0) {                 // aligned full row: one 8-byte store
            unsigned long long v = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) v |= (unsigned long long)((bits >> k) & 1u) << (8 * k);
            *reinterpret_cast<unsigned long long*>(dst + base) = v;
        } else {
            for (uint32_t k = 0; k < w; ++k) dst[base + k] = (uint8_t)((bits >> k) & 1u);
        }
    }
}
}  // namespace

cudaError_t launch_pack_bits_u8(liets_ctx* c, const uint8_t* src_u8, uint8_t* dst_bits) {
    k_pack_bits_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(src_u8, dst_bits, c->N);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_unpack_bricks_u8(liets_ctx* c, uint8_t* dst_u8) {
    k_unpack_bricks_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(c->G[c->host_step & 1u], dst_u8, c->geom, c->n_bricks * 64ull);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
