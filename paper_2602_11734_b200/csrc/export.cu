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
}  // namespace

cudaError_t launch_pack_bits_u8(liets_ctx* c, uint8_t* dst_bits) {
    k_pack_bits_u8<<<c->sm_count * 8, 256, 0, c->stream>>>(c->grid_u8, dst_bits, c->N);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
