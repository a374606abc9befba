// probe.cu -- measured roofs for the report of bench.py (SURVEY.md 8(d) "Which roofline"):
// the growth path is bound by integer issue and its working set is L2 resident, so the peaks it is held against
// are MEASURED on the box by these kernels instead of being derived from unit counts:
//
//   LIETS_PROBE_PHILOX   Philox4x32-10 blocks back to back, nothing else (the path's irreducible arithmetic,
//                        PAPER.md:112 "an independent random number"; R9): blocks/s
//   LIETS_PROBE_LOP3     three-input logic ops (ALU pipe), 8 independent chains per thread: thread-instructions/s
//   LIETS_PROBE_IMAD     32-bit multiply-adds (FMA pipe), 8 independent chains per thread: thread-instructions/s
//   LIETS_PROBE_MIX      one multiply-add per logic op, interleaved (what Philox alternates): thread-instructions/s
//   LIETS_PROBE_L2_READ  streaming 16-byte loads of an L2-resident buffer, all SMs: bytes/s
//   LIETS_PROBE_HBM_READ the same over a buffer far larger than L2: bytes/s
//
// Every probe runs `reps` launches on the given stream between two CUDA events after one warm-up launch and returns
// the best launch.  Results land in a sink the compiler cannot remove.
#include "../../include/liets.h"
#include "liets_device.cuh"

namespace liets {
namespace {

constexpr int kProbeThreads = 256;

__global__ void __launch_bounds__(kProbeThreads) k_probe_philox(uint32_t* sink, uint32_t iters, PhiloxKey key) {
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    // two independent blocks per iteration (the growth kernel has one per voxel and many warps in flight)
    for (uint32_t i = 0; i < iters; ++i) {
        const uint4 a = philox4x32_10(gid, 0u, i, 0u, key);
        const uint4 b = philox4x32_10(gid, 0u, i, 1u, key);
        acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w;
    }
    if (acc == 0x12345678u) sink[gid & 1023u] = acc;
}

template <int KIND>     // 0 LOP3, 1 IMAD, 2 one IMAD per LOP3
__global__ void __launch_bounds__(kProbeThreads) k_probe_int(uint32_t* sink, uint32_t iters, uint32_t m, uint32_t c) {
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t r[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) r[k] = gid * 2654435761u + (uint32_t)k;
    for (uint32_t i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KIND == 0) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[k]) : "r"(m), "r"(c));
                } else if (KIND == 1) {
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[k]) : "r"(m), "r"(c));
                } else {
                    if (k & 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[k]) : "r"(m), "r"(c));
                    else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[k]) : "r"(m), "r"(c));
                }
            }
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) acc ^= r[k];
    if (acc == 0x12345678u) sink[gid & 1023u] = acc;
}

__global__ void __launch_bounds__(kProbeThreads) k_probe_read(const uint4* __restrict__ buf, unsigned long long n_vec,
                                                               uint32_t passes, uint32_t* sink) {
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    uint32_t acc = 0;
    for (uint32_t p = 0; p < passes; ++p)
        for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) {
            const uint4 v = __ldcg(buf + i);                // L2 (not L1): the growth kernel's grid loads are ld.cg too
            acc ^= v.x ^ v.y ^ v.z ^ v.w;
        }
    if (acc == 0x12345678u) sink[threadIdx.x] = acc;
}

}  // namespace
}  // namespace liets

using namespace liets;

extern "C" int liets_probe(int kind, void* device_scratch, size_t scratch_bytes, void* cuda_stream, int reps,
                           double* units_per_second, double* ms_best) {
    if (!device_scratch || scratch_bytes < (1u << 20) || reps < 1 || !units_per_second) return LIETS_E_ARG;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return LIETS_E_CUDA;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return LIETS_E_CUDA;
    uint32_t* sink = static_cast<uint32_t*>(device_scratch);
    const int grid = sms * 8;                                   // 8 CTAs x 8 warps: every warp slot of the SM
    const PhiloxKey key = philox_make_key(0x0123456789ABCDEFull);
    double units = 0.0;
    auto launch = [&]() -> cudaError_t {
        switch (kind) {
        case LIETS_PROBE_PHILOX: {
            const uint32_t iters = 512;
            k_probe_philox<<<grid, kProbeThreads, 0, stream>>>(sink, iters, key);
            units = 2.0 * iters * (double)grid * kProbeThreads;
            break;
        }
        case LIETS_PROBE_LOP3: case LIETS_PROBE_IMAD: case LIETS_PROBE_MIX: {
            const uint32_t iters = 1024;
            if (kind == LIETS_PROBE_LOP3) k_probe_int<0><<<grid, kProbeThreads, 0, stream>>>(sink, iters, 0x9E3779B9u, 0x7F4A7C15u);
            else if (kind == LIETS_PROBE_IMAD) k_probe_int<1><<<grid, kProbeThreads, 0, stream>>>(sink, iters, 0x9E3779B9u, 0x7F4A7C15u);
            else k_probe_int<2><<<grid, kProbeThreads, 0, stream>>>(sink, iters, 0x9E3779B9u, 0x7F4A7C15u);
            units = 32.0 * iters * (double)grid * kProbeThreads;
            break;
        }
        case LIETS_PROBE_L2_READ: case LIETS_PROBE_HBM_READ: {
            // L2: a 32 MiB window (or the scratch, if smaller) read 16 times; HBM: the whole scratch once
            size_t bytes = scratch_bytes & ~(size_t)255;
            uint32_t passes = 1;
            if (kind == LIETS_PROBE_L2_READ) { if (bytes > ((size_t)32 << 20)) bytes = (size_t)32 << 20; passes = 16; }
            k_probe_read<<<grid, kProbeThreads, 0, stream>>>(reinterpret_cast<const uint4*>(device_scratch), bytes / 16, passes, sink);
            units = (double)bytes * passes;
            break;
        }
        default: return cudaErrorInvalidValue;
        }
        return cudaGetLastError();
    };
    int rc = LIETS_OK;
    float best = 0.f;
    if (kind < LIETS_PROBE_PHILOX || kind > LIETS_PROBE_HBM_READ) rc = LIETS_E_ARG;
    else if (launch() != cudaSuccess) rc = LIETS_E_CUDA;       // warm-up (and, for the L2 probe, the fill of L2)
    for (int r = 0; rc == LIETS_OK && r < reps; ++r) {
        float ms = 0.f;
        if (cudaEventRecord(e0, stream) != cudaSuccess || launch() != cudaSuccess || cudaEventRecord(e1, stream) != cudaSuccess ||
            cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) { rc = LIETS_E_CUDA; break; }
        if (r == 0 || ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (rc != LIETS_OK) { cudaGetLastError(); return rc; }
    *units_per_second = units / (best * 1e-3);
    if (ms_best) *ms_best = best;
    return LIETS_OK;
}
