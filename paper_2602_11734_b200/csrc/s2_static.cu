// s2_static.cu -- liets_s2_static: the two-point correlation of liets_s2 (s2.cu, R16) for callers that cannot
// call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).  liets_s2 takes its per-lag pair
// counters from cudaMalloc on every call; here they live in ONE file-scope device array of LIETS_S2_STATIC_MAX_LAGS
// 64-bit counters (32 KiB, held by every GPU that loads the library until the process exits), and the call makes no
// cudaMalloc, cudaFree or allocating library call.  Same definition, same integers:
//   pairs[r] = #{ x : void(x) and void(x + r e_axis) },  r = 0 .. rmax,  rmax < LIETS_S2_STATIC_MAX_LAGS.
//
// The array is shared by every call on a device and keeps the last call's counts: each call zeroes the rmax + 1
// counters it uses on its stream before the kernel.  Two calls that overlap on the GPU would race on it; the entry
// point holds a host mutex from the zeroing to the end of the copy-out and synchronises its stream, so its own calls
// cannot overlap within a process (another process has its own copy of the array).
//
// g_s2_pairs below is, in HOST code, a stand-in for the symbol and not a device address: the address comes from
// cudaGetSymbolAddress, once per device with that device current, and is handed to the kernel as an argument.
#include <mutex>

#include "../../include/liets.h"
#include "liets_host.h"

namespace liets {
namespace {

constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned long long g_s2_pairs[LIETS_S2_STATIC_MAX_LAGS];

std::mutex g_mutex;                                         // guards g_pairs_addr and the array's use
unsigned long long* g_pairs_addr[kMaxDevices];              // device address of g_s2_pairs on each device (0 = not asked yet)

struct RowGeom { int nx, ny, nz, Wp, periodic; };

// void cells of word w of an x-row as bits (1 = void); positions x >= nx are not cells
__device__ __forceinline__ unsigned long long row_void(const unsigned long long* __restrict__ row, int w, const RowGeom& g) {
    const int x0 = 64 * w;
    if (w >= g.Wp || x0 >= g.nx) return 0ull;
    unsigned long long v = ~row[w];
    if (g.nx - x0 < 64) v &= (1ull << (g.nx - x0)) - 1ull;
    return v;
}

// void bits of the 64 positions s .. s + 63 of a row (0 <= s), no wrap
__device__ __forceinline__ unsigned long long row_void_at(const unsigned long long* __restrict__ row, int s, const RowGeom& g) {
    if (s >= g.nx) return 0ull;
    const int w = s >> 6, b = s & 63;
    unsigned long long v = row_void(row, w, g) >> b;
    if (b) v |= row_void(row, w + 1, g) << (64 - b);
    return v;
}

// void bits of the cells r to the right of the cells of word w (r < nx if periodic)
__device__ __forceinline__ unsigned long long shifted_x(const unsigned long long* __restrict__ row, int w, int r, const RowGeom& g) {
    const int x0 = 64 * w;
    if (!g.periodic) return row_void_at(row, x0 + r, g);
    const int cells = min(64, g.nx - x0);
    unsigned long long out = 0ull;
    int done = 0, s = (x0 + r) % g.nx;
    while (done < cells) {                                  // stretches of the row between wrap-arounds
        const int take = min(cells - done, g.nx - s);
        unsigned long long piece = row_void_at(row, s, g);
        if (take < 64) piece &= (1ull << take) - 1ull;
        out |= piece << done;
        done += take;
        s = 0;
    }
    return out;
}

// blockIdx.y = lag r; the CTAs of a lag stride over the grid's words; one 64-bit atomic per CTA into counters[r]
__global__ void __launch_bounds__(kThreads) k_s2_static(const unsigned long long* __restrict__ G, RowGeom g, int axis,
                                                         unsigned long long* __restrict__ counters) {
    __shared__ unsigned long long s_part[kThreads / 32];
    const int r = (int)blockIdx.y;
    const int extent = axis == 0 ? g.nx : axis == 1 ? g.ny : g.nz;
    const unsigned long long Wp = (unsigned long long)g.Wp, ny = (unsigned long long)g.ny;
    const unsigned long long n_words = Wp * ny * (unsigned long long)g.nz;
    unsigned long long acc = 0ull;
    if (g.periodic || r < extent) {
        const int rr = g.periodic ? r % extent : r;
        for (unsigned long long i = (unsigned long long)blockIdx.x * kThreads + threadIdx.x; i < n_words;
             i += (unsigned long long)gridDim.x * kThreads) {
            const int w = (int)(i % Wp);
            const unsigned long long rowi = i / Wp;
            const unsigned long long* row = G + rowi * Wp;
            const unsigned long long a = row_void(row, w, g);
            if (!a) continue;
            unsigned long long b;
            if (axis == 0) {
                b = shifted_x(row, w, rr, g);
            } else {
                int y = (int)(rowi % ny), z = (int)(rowi / ny);
                if (axis == 1) { y += rr; if (y >= g.ny) { if (!g.periodic) continue; y -= g.ny; } }
                else           { z += rr; if (z >= g.nz) { if (!g.periodic) continue; z -= g.nz; } }
                b = row_void(G + ((unsigned long long)y + ny * (unsigned long long)z) * Wp, w, g);
            }
            acc += (unsigned long long)__popcll(a & b);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0ull;
        for (int k = 0; k < kThreads / 32; ++k) t += s_part[k];
        if (t) atomicAdd(counters + r, t);
    }
}

int fail_static(liets_ctx* c, int code, const char* msg) {
    if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
    return code;
}

}  // namespace
}  // namespace liets

using namespace liets;

extern "C" int liets_s2_static(liets_ctx* c, int axis, int rmax, uint64_t* pairs, uint64_t* valid) {
    if (!c || !pairs || !valid) return LIETS_E_ARG;
    if (axis < 0 || axis > 2 || rmax < 0) return fail_static(c, LIETS_E_ARG, "liets_s2_static: axis must be 0..2 and rmax >= 0");
    if (rmax >= LIETS_S2_STATIC_MAX_LAGS) {
        snprintf(c->err, sizeof(c->err), "liets_s2_static: %lld lags (rmax + 1) exceed the static scratch of %d counters; use liets_s2",
                 (long long)rmax + 1, (int)LIETS_S2_STATIC_MAX_LAGS);
        return LIETS_E_CAPACITY;
    }
    if (c->storage == LIETS_STORAGE_U8)
        return fail_static(c, LIETS_E_ARG, "liets_s2_static: needs a bit-row storage (LIETS_STORAGE_TILE or _FULL); use liets_s2");
    if (!c->seeded) return fail_static(c, LIETS_E_STATE, "liets_s2_static before liets_seed");

    std::lock_guard<std::mutex> lock(g_mutex);
    int dev = -1;
    LIETS_CUDA_TRY(c, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail_static(c, LIETS_E_CUDA, "liets_s2_static: device ordinal out of range");
    if (!g_pairs_addr[dev]) {                               // once per device, with that device current
        void* p = nullptr;
        LIETS_CUDA_TRY(c, cudaGetSymbolAddress(&p, g_s2_pairs));
        if (!p) return fail_static(c, LIETS_E_CUDA, "liets_s2_static: cudaGetSymbolAddress gave no address");
        g_pairs_addr[dev] = static_cast<unsigned long long*>(p);
    }
    unsigned long long* counters = g_pairs_addr[dev];

    // which grid copy is current (the step counter lives on the device)
    LIETS_CUDA_TRY(c, cudaMemcpyAsync(c->pinned, c->ctl, kControlScalarBytes, cudaMemcpyDeviceToHost, c->stream));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->host_step = c->pinned->step;
    const unsigned long long* G = c->G[c->host_step & 1u];

    RowGeom g{ c->nx, c->ny, c->nz, (c->nx + 63) / 64, (c->periodic >> axis) & 1 };   // only the lag axis's boundary matters
    const size_t bytes = (size_t)(rmax + 1) * sizeof(unsigned long long);
    const unsigned long long n_words = (unsigned long long)g.Wp * (unsigned long long)g.ny * (unsigned long long)g.nz;
    unsigned long long bx = (n_words + kThreads - 1) / kThreads;
    const unsigned long long bx_max = (unsigned long long)c->sm_count * 8ull;
    if (bx > bx_max) bx = bx_max;
    if (bx < 1) bx = 1;

    LIETS_CUDA_TRY(c, cudaMemsetAsync(counters, 0, bytes, c->stream));                 // the array keeps the last call's counts
    k_s2_static<<<dim3((unsigned)bx, (unsigned)(rmax + 1)), kThreads, 0, c->stream>>>(G, g, axis, counters);
    c->launches++;
    LIETS_CUDA_TRY(c, cudaGetLastError());
    LIETS_CUDA_TRY(c, cudaMemcpyAsync(pairs, counters, bytes, cudaMemcpyDeviceToHost, c->stream));
    LIETS_CUDA_TRY(c, cudaStreamSynchronize(c->stream));

    const uint64_t n[3] = { (uint64_t)c->nx, (uint64_t)c->ny, (uint64_t)c->nz };
    for (int r = 0; r <= rmax; ++r)                         // positions counted: all if the axis wraps, else those with x + r inside
        valid[r] = g.periodic ? c->N : ((uint64_t)r < n[axis] ? c->N / n[axis] * (n[axis] - (uint64_t)r) : 0);
    return LIETS_OK;
}
