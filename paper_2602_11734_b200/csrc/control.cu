// control.cu -- the device-resident step loop: thresholds (Eq. (1)), stop rule, list swap, counters.
//
// One growth step is  control_step(PREPARE) ; grow kernel ; control_step(FINISH ...)  (liets_device.cuh).
// control_step is run by a single warp: it turns the solid count into the three integer thresholds of the
// step (R6/R8), evaluates "while phi_a < phi_s and A not empty" and
// arms or disarms the grow kernel through Control::active, so a batch of steps can be enqueued
// without the host looking at the device in between.  It runs as the one-warp kernel k_control between the
// growth kernels: enqueued ahead, its launch overlaps the previous kernel's tail (folding it into the last CTA of
// the growth kernel was measured slower: the whole GPU idles behind one thread).
#include "liets_host.h"

namespace liets {

__global__ void k_control(Control* c, uint32_t flags) {     // one warp
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    control_step(c, flags);
}

// The control step inside the device-side WHILE loop of liets_generate's CUDA graph: closes the step that just ran,
// prepares the next one and tells the loop whether to go round again.
__global__ void k_control_loop(Control* c, cudaGraphConditionalHandle loop) {      // one warp
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    control_step(c, kCtlFinish | kCtlPrepare);
    __syncwarp();
    if (threadIdx.x == 0) cudaGraphSetConditional(loop, __ldcg(&c->active) ? 1u : 0u);
}

cudaError_t control_loop_node(liets_ctx* c, cudaGraph_t graph, cudaGraphNode_t after, cudaGraphConditionalHandle loop,
                              cudaGraphNode_t* node) {
    void* args[] = { &c->ctl, &loop };
    cudaKernelNodeParams p = {};
    p.func = reinterpret_cast<void*>(k_control_loop);
    p.gridDim = dim3(1); p.blockDim = dim3(32); p.sharedMemBytes = 0; p.kernelParams = args;
    return cudaGraphAddKernelNode(node, graph, &after, 1, &p);
}

// The same for the grids of a batch (liets_generate_batch): warp i steps grid i; the loop goes round while any grid is live.
struct ControlBatch { int n; Control* ctl[32]; };

__global__ void k_control_loop_batch(ControlBatch b, cudaGraphConditionalHandle loop) {
    const int grid_i = (int)(threadIdx.x >> 5);
    int live = 0;
    if (grid_i < b.n) {
        control_step(b.ctl[grid_i], kCtlFinish | kCtlPrepare);
        __syncwarp();
        live = __ldcg(&b.ctl[grid_i]->active) ? 1 : 0;
    }
    live = __syncthreads_or(live);
    if (threadIdx.x == 0) cudaGraphSetConditional(loop, live ? 1u : 0u);
}

cudaError_t control_loop_batch_node(liets_ctx* const* ctx, int n, cudaGraph_t graph, cudaGraphNode_t after,
                                    cudaGraphConditionalHandle loop, cudaGraphNode_t* node) {
    if (n < 1 || n > 32) return cudaErrorInvalidValue;
    ControlBatch b = {};
    b.n = n;
    for (int i = 0; i < n; ++i) b.ctl[i] = ctx[i]->ctl;
    void* args[] = { &b, &loop };
    cudaKernelNodeParams p = {};
    p.func = reinterpret_cast<void*>(k_control_loop_batch);
    p.gridDim = dim3(1); p.blockDim = dim3(32 * n); p.sharedMemBytes = 0; p.kernelParams = args;
    return cudaGraphAddKernelNode(node, graph, &after, 1, &p);
}

__global__ void k_begin(Control* c, int generate, uint32_t max_steps) {
    c->steps_done = 0;
    c->max_steps = max_steps;
    c->status = generate ? kStatusRunning : 0;
    c->active = 0;
}

__global__ void k_set_params(Control* c, unsigned long long R0, unsigned long long R1,
                             unsigned long long R2, uint32_t law, unsigned long long n_t,
                             uint32_t has_target, unsigned long long N, unsigned long long n_free, uint32_t list_cap,
                             uint32_t vox_cap, uint32_t vox_thr) {
    c->R[0] = R0; c->R[1] = R1; c->R[2] = R2;
    c->law = law; c->n_t = n_t; c->has_target = has_target; c->N = N; c->n_free = n_free; c->list_cap = list_cap;
    c->vox_cap = vox_cap; c->vox_thr = vox_thr;
}

// R20: the interaction thresholds RI (floor(I 2^32 + 0.5) per class, constant), laid out nibble by nibble like hpat
__global__ void k_set_interaction(Control* c, unsigned long long RI0, unsigned long long RI1, unsigned long long RI2) {
    const unsigned long long RI[3] = { RI0, RI1, RI2 };
    uint32_t U[3], en26 = 0;
    for (int k = 0; k < 3; ++k) {
        U[k] = RI[k] >= 1ull ? (uint32_t)(RI[k] - 1ull) : 0u;
        if (RI[k] >= 1ull) en26 |= class_dir_mask(k);
    }
    for (uint32_t lv = 0; lv < 8u; ++lv)
        for (int w = 0; w < 4; ++w) {
            uint32_t h = 0;
            for (int k = 0; k < 3; ++k) {
                const uint32_t ones = w == 0 ? class_nibble_ones(0, k) : w == 1 ? class_nibble_ones(1, k) : w == 2 ? class_nibble_ones(2, k) : class_nibble_ones(3, k);
                h += ((U[k] >> (28u - 4u * lv)) & 15u) * ones;
            }
            c->hpatI[lv][w] = h;
        }
    c->enI26 = en26;
    c->interact = en26 != 0u;
}

// test aid: eq1_threshold on the device for n (R, n_t, n_solid) triples (liets_debug_thresholds)
__global__ void k_eq1_thresholds(const unsigned long long* R, const unsigned long long* n_t, const unsigned long long* n_solid,
                                 unsigned long long* T, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) T[i] = eq1_threshold(R[i], n_t[i], n_solid[i]);
}

cudaError_t launch_eq1_thresholds(const unsigned long long* dev_in, unsigned long long* dev_out, uint32_t n, cudaStream_t stream) {
    k_eq1_thresholds<<<(n + 127) / 128, 128, 0, stream>>>(dev_in, dev_in + n, dev_in + 2ull * n, dev_out, n);
    return cudaGetLastError();
}

cudaError_t launch_control(liets_ctx* c, uint32_t flags) {
    k_control<<<1, 32, 0, c->stream>>>(c->ctl, flags);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_begin(liets_ctx* c, int generate, uint32_t max_steps) {
    k_begin<<<1, 1, 0, c->stream>>>(c->ctl, generate, max_steps);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_set_interaction(liets_ctx* c) {
    k_set_interaction<<<1, 1, 0, c->stream>>>(c->ctl, c->RI[0], c->RI[1], c->RI[2]);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_set_params(liets_ctx* c) {
    k_set_params<<<1, 1, 0, c->stream>>>(c->ctl, c->R[0], c->R[1], c->R[2], (uint32_t)c->law, c->n_t,
                                         c->has_target ? 1u : 0u, c->N, c->N - (c->has_blocked ? c->n_blocked : 0), (uint32_t)c->list_cap,
                                         c->vox_cap, c->vox_thr);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
