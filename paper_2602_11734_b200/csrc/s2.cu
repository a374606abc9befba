// s2.cu -- two-point correlation of the void phase on the device (R16; BASELINE.json: "outputs checked by
// porosity and two-point correlation").  Exact integer pair counts, as the oracle defines them:
//   pairs[r] = #{ x : void(x) and void(x + r e_axis) },  valid[r] = #{ x : x + r e_axis is counted },  r = 0 .. rmax,
// with pairs inside the domain only on a walled grid and wrapped per coordinate on a periodic one.  S2(r) = pairs / valid.
//
// The phase array is taken as bit rows (x-rows of Wp 64-bit words, as STORAGE_TILE keeps it; a STORAGE_U8 grid is packed
// into such rows first).  One thread per (64-voxel word, lag r): the partner word is the same word of row y + r or z + r,
// or, along x, the 64 row bits that start r cells further on; popc of the AND, one 64-bit atomic per CTA and lag.
#include "../../include/liets.h"
#include "liets_host.h"

namespace liets {
namespace {

constexpr int kS2Threads = 256;

struct S2Geom { int nx, ny, nz, Wp, periodic; };

// void bits of word w of a row (cells x >= nx are not cells)
__device__ __forceinline__ unsigned long long void_word(const unsigned long long* __restrict__ row, int w, int nx) {
    const int xbase = 64 * w;
    if (xbase >= nx) return 0ull;
    unsigned long long v = ~row[w];
    if (xbase + 64 > nx) v &= ~(~0ull << (nx - xbase));
    return v;
}

// 64 void bits of the row starting at cell s (0 <= s), cells beyond nx read as "not void"
__device__ __forceinline__ unsigned long long void_bits_from(const unsigned long long* __restrict__ row, int s, int nx, int Wp) {
    if (s >= nx) return 0ull;
    const int w = s >> 6, b = s & 63;
    unsigned long long v = void_word(row, w, nx) >> b;
    if (b && w + 1 < Wp) v |= void_word(row, w + 1, nx) << (64 - b);
    return v;
}

// the 64 cells that are r cells to the right of the cells of word w, wrapped around the row if periodic
__device__ __forceinline__ unsigned long long partner_x(const unsigned long long* __restrict__ row, int w, int r, const S2Geom& g) {
    const int xbase = 64 * w;
    if (!g.periodic) return void_bits_from(row, xbase + r, g.nx, g.Wp);
    unsigned long long out = 0ull;
    int filled = 0;                                         // cells of the word already paired
    const int n_here = min(64, g.nx - xbase);
    int s = (xbase + r) % g.nx;
    while (filled < n_here) {                               // pieces of the row between wrap-arounds
        const int take = min(n_here - filled, g.nx - s);
        unsigned long long piece = void_bits_from(row, s, g.nx, g.Wp);
        if (take < 64) piece &= ~(~0ull << take);
        out |= piece << filled;
        filled += take;
        s = 0;
    }
    return out;
}

__global__ void __launch_bounds__(kS2Threads) k_s2(const unsigned long long* __restrict__ G, S2Geom g, int axis, int rmax,
                                                    unsigned long long* __restrict__ pairs) {
    __shared__ unsigned long long s_sum[kS2Threads / 32];
    const int r = (int)blockIdx.y;
    const unsigned long long n_words = (unsigned long long)g.Wp * (unsigned long long)g.ny * (unsigned long long)g.nz;
    const int n[3] = { g.nx, g.ny, g.nz };
    unsigned long long acc = 0ull;
    const bool lag_exists = g.periodic || r < n[axis];
    const int rr = g.periodic ? r % n[axis] : r;
    if (lag_exists)
        for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
             i += (unsigned long long)gridDim.x * blockDim.x) {
            const int w = (int)(i % (unsigned long long)g.Wp);
            const unsigned long long rowi = i / (unsigned long long)g.Wp;
            const int y = (int)(rowi % (unsigned long long)g.ny), z = (int)(rowi / (unsigned long long)g.ny);
            const unsigned long long* row = G + rowi * (unsigned long long)g.Wp;
            const unsigned long long a = void_word(row, w, g.nx);
            if (!a) continue;
            unsigned long long b;
            if (axis == 0) {
                b = partner_x(row, w, rr, g);
            } else {
                int y2 = y, z2 = z;
                if (axis == 1) { y2 = y + rr; if (y2 >= g.ny) { if (!g.periodic) continue; y2 -= g.ny; } }
                else { z2 = z + rr; if (z2 >= g.nz) { if (!g.periodic) continue; z2 -= g.nz; } }
                b = void_word(G + ((unsigned long long)y2 + (unsigned long long)g.ny * (unsigned long long)z2) * (unsigned long long)g.Wp, w, g.nx);
            }
            acc += (unsigned long long)__popcll(a & b);
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0ull;
        for (int k = 0; k < kS2Threads / 32; ++k) t += s_sum[k];
        if (t) atomicAdd(pairs + r, t);
    }
}

// STORAGE_U8 -> bit rows (one thread per word)
__global__ void k_u8_to_rows(const uint8_t* __restrict__ grid, S2Geom g, unsigned long long* __restrict__ rows) {
    const unsigned long long n_words = (unsigned long long)g.Wp * (unsigned long long)g.ny * (unsigned long long)g.nz;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const int w = (int)(i % (unsigned long long)g.Wp);
        const unsigned long long rowi = i / (unsigned long long)g.Wp;
        const uint8_t* src = grid + rowi * (unsigned long long)g.nx + 64ull * w;
        const int nvalid = min(64, g.nx - 64 * w);
        unsigned long long v = 0ull;
        for (int b = 0; b < nvalid; ++b) v |= (unsigned long long)(src[b] != 0) << b;
        rows[i] = v;
    }
}

}  // namespace

// pairs_dev: rmax + 1 zeroed 64-bit counters on the device; rows: the bit rows to use (nullptr = the ctx's current grid)
cudaError_t launch_s2(liets_ctx* c, int axis, int rmax, unsigned long long* pairs_dev, unsigned long long* rows_scratch) {
    S2Geom g{ c->nx, c->ny, c->nz, (c->nx + 63) / 64, (c->periodic >> axis) & 1 };      // only the lag axis's boundary matters
    const unsigned long long* G;
    if (c->storage == LIETS_STORAGE_U8) {
        k_u8_to_rows<<<c->sm_count * 8, 256, 0, c->stream>>>(c->grid_u8, g, rows_scratch);
        c->launches++;
        G = rows_scratch;
    } else {
        G = c->G[c->host_step & 1u];
    }
    const unsigned long long n_words = (unsigned long long)g.Wp * (unsigned long long)g.ny * (unsigned long long)g.nz;
    unsigned long long bx = (n_words + kS2Threads - 1) / kS2Threads;
    if (bx > (unsigned long long)c->sm_count * 8ull) bx = (unsigned long long)c->sm_count * 8ull;
    if (bx < 1) bx = 1;
    k_s2<<<dim3((unsigned)bx, (unsigned)(rmax + 1)), kS2Threads, 0, c->stream>>>(G, g, axis, rmax, pairs_dev);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
