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
            if (v < N && grid[v] == 1) out |= 1u << k;     // (2 = a cell of an earlier phase, liets_set_blocked)
        }
        dst[b] = (uint8_t)out;
    }
}
// bit rows -> uint8 {0,1} per voxel, x fastest: one thread per 8 voxels of a row
__global__ void __launch_bounds__(256) k_unpack_rows_u8(const unsigned long long* __restrict__ G, const unsigned long long* __restrict__ P,
                                                         uint8_t* __restrict__ dst, TileGeom g, unsigned long long n_rows) {
    const unsigned long long per_row = ((unsigned long long)g.nx + 7ull) / 8ull;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_rows * per_row;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long row = i / per_row;
        const uint32_t b = (uint32_t)(i - row * per_row), x0 = 8u * b;
        uint32_t bits = (uint32_t)(G[row * (unsigned long long)g.Wp + (b >> 3)] >> (8u * (b & 7u))) & 0xFFu;
        if (P) bits &= ~(uint32_t)(P[row * (unsigned long long)g.Wp + (b >> 3)] >> (8u * (b & 7u)));      // this phase only
        const unsigned long long base = row * (unsigned long long)g.nx + x0;
        const uint32_t w = min(8u, (uint32_t)g.nx - x0);
        if (w == 8u && (base & 7ull) == 0) {                 // aligned full group: one 8-byte store
            unsigned long long v = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) v |= (unsigned long long)((bits >> k) & 1u) << (8 * k);
            *reinterpret_cast<unsigned long long*>(dst + base) = v;
        } else {
            for (uint32_t k = 0; k < w; ++k) dst[base + k] = (uint8_t)((bits >> k) & 1u);
        }
    }
}
// byte-aligned bit rows (nx % 8 == 0) -> the packed phase array: the rows without their padding words
__global__ void __launch_bounds__(256) k_rows_to_bits(const uint8_t* __restrict__ G, const uint8_t* __restrict__ P, uint8_t* __restrict__ dst,
                                                       unsigned long long n_bytes, uint32_t row_bytes, uint32_t pitch) {
    for (unsigned long long b = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; b < n_bytes;
         b += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long row = b / row_bytes;
        const unsigned long long i = row * pitch + (b - row * row_bytes);
        dst[b] = P ? (uint8_t)(G[i] & ~P[i]) : G[i];
    }
}
}  // namespace

cudaError_t launch_rows_to_bits(liets_ctx* c, uint8_t* dst_bits) {
    k_rows_to_bits<<<c->sm_count * 8, 256, 0, c->stream>>>(reinterpret_cast<const uint8_t*>(c->G[c->host_step & 1u]),
                                                           c->has_blocked ? reinterpret_cast<const uint8_t*>(c->prow) : nullptr, dst_bits,
                                                           c->N / 8, (uint32_t)c->nx / 8, (uint32_t)c->geom.Wp * 8);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_pack_bits_u8(liets_ctx* c, const uint8_t* src_u8, uint8_t* dst_bits) {
    k_pack_bits_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(src_u8, dst_bits, c->N);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_unpack_rows_u8(liets_ctx* c, uint8_t* dst_u8) {
    k_unpack_rows_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(c->G[c->host_step & 1u], c->has_blocked ? c->prow : nullptr, dst_u8, c->geom,
                                                             (unsigned long long)c->ny * (unsigned long long)c->nz);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
