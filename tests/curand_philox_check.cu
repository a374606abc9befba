// Test helper (not part of the product): prints NVIDIA cuRAND's device curand_Philox4x32_10 for the
// (counter, key) vectors read from stdin, one "c0 c1 c2 c3 k0 k1" line (hex) each -- an independent
// implementation of Philox4x32-10 to pin the oracle's (pin P1).
#include <cstdio>
#include <vector>
#include <curand_philox4x32_x.h>

__global__ void k(const uint4* c, const uint2* key, uint4* out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = curand_Philox4x32_10(c[i], key[i]);
}

int main() {
    std::vector<uint4> c; std::vector<uint2> key;
    unsigned v[6];
    while (scanf("%x %x %x %x %x %x", &v[0], &v[1], &v[2], &v[3], &v[4], &v[5]) == 6) {
        c.push_back(make_uint4(v[0], v[1], v[2], v[3])); key.push_back(make_uint2(v[4], v[5]));
    }
    const int n = (int)c.size();
    uint4 *dc, *dout; uint2* dk;
    if (cudaMalloc(&dc, n * sizeof(uint4)) || cudaMalloc(&dk, n * sizeof(uint2)) || cudaMalloc(&dout, n * sizeof(uint4))) return 1;
    cudaMemcpy(dc, c.data(), n * sizeof(uint4), cudaMemcpyHostToDevice);
    cudaMemcpy(dk, key.data(), n * sizeof(uint2), cudaMemcpyHostToDevice);
    k<<<(n + 255) / 256, 256>>>(dc, dk, dout, n);
    std::vector<uint4> out(n);
    if (cudaMemcpy(out.data(), dout, n * sizeof(uint4), cudaMemcpyDeviceToHost) != cudaSuccess) return 2;
    for (int i = 0; i < n; ++i) printf("%08x %08x %08x %08x\n", out[i].x, out[i].y, out[i].z, out[i].w);
    return 0;
}
