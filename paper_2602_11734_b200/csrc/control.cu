// control.cu -- the device-resident step loop: thresholds (Eq. (1)), stop rule, list swap, counters.
//
// One growth step is  k_control(PREPARE) ; grow kernel ; k_control(FINISH ...).  The control
// kernel is a single thread: it turns the solid count into the three integer thresholds of the
// step (R6/R8), evaluates "while phi_a < phi_s and A not empty" and
// arms or disarms the grow kernel through Control::active, so a batch of steps can be enqueued
// without the host looking at the device in between.
#include "liets_host.h"

namespace liets {

// T = min(2^32, floor(R * max(0, 20 n_t - 19 n_solid) / n_t)) without 128-bit arithmetic:
// a = 20 n_t - 19 n_solid = q n_t + r  =>  floor(R a / n_t) = R q + floor(R r / n_t),
// with q <= 20, R <= 2^32, r < n_t <= 2^32, so every product fits 64 bits.
__device__ unsigned long long eq1_threshold(unsigned long long R, unsigned long long n_t,
                                            unsigned long long n_solid) {
    unsigned long long a = 20ull * n_t, b = 19ull * n_solid;
    if (b >= a) return 0ull;
    a -= b;
    unsigned long long q = a / n_t, r = a % n_t;
    unsigned long long T = R * q + (R * r) / n_t;
    return T > (1ull << 32) ? (1ull << 32) : T;
}

__global__ void k_control(Control* c, uint32_t flags) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    if ((flags & kCtlFinish) && c->active) {             // close the step that just ran
        c->n_solid += c->claims;                         // phi_a update
        c->claims = 0;
        if (c->step < kLogCap) { c->log_solid[c->step] = c->n_solid; c->log_items[c->step] = c->items; }
        c->cur ^= 1u;                                    // A <- prune(A U A_new) (R4)
        c->step += 1;
        c->steps_done += 1;
        c->active = 0;
    }
    if (flags & (kCtlPrepare | kCtlEval)) {
        const bool force = flags & kCtlForce;
        if (!force) {                                    // stop rule, between whole steps only
            if (c->status != kStatusRunning) return;
            if (c->n_solid >= c->n_t) { c->status = 0; return; }            // LIETS_OK
            if (c->count[c->cur] == 0 || c->n_solid == c->N) { c->status = 1; return; }   // FRONT_EMPTY
            if (c->steps_done >= c->max_steps) { c->status = 2; return; }   // MAX_STEPS
        }
        if (!(flags & kCtlPrepare)) return;
        for (int k = 0; k < 3; ++k) {
            unsigned long long T = c->law ? eq1_threshold(c->R[k], c->n_t, c->n_solid) : c->R[k];
            c->en[k] = T >= 1ull;                                            // T in [0, 2^32]
            c->U[k] = T >= 1ull ? (uint32_t)(T - 1ull) : 0u;                 // draw < T  <=>  draw <= T - 1
        }
        // the thresholds nibble by nibble, laid out like the draws (direction d: nibble d>>2 of word d&3);
        // built in registers: class masks are compile-time constants
        uint32_t en26 = 0, h0_any = 0;
        uint32_t U[3], en[3];
        for (int k = 0; k < 3; ++k) { U[k] = c->U[k]; en[k] = c->en[k]; }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            if (en[k]) en26 |= class_dir_mask(k);
            if (en[k] && (U[k] >> 28)) h0_any = 1;
        }
#pragma unroll
        for (int lv = 0; lv < 8; ++lv)
#pragma unroll
            for (int w = 0; w < 4; ++w)
                c->hpat[lv][w] = ((U[0] >> (28 - 4 * lv)) & 15u) * class_nibble_ones(w, 0) +
                                 ((U[1] >> (28 - 4 * lv)) & 15u) * class_nibble_ones(w, 1) +
                                 ((U[2] >> (28 - 4 * lv)) & 15u) * class_nibble_ones(w, 2);
        c->en26 = en26;
        c->h0_any = h0_any;
        c->tile_cursor = 0;
        c->count[c->cur ^ 1u] = 0;
        c->claims = 0;
        c->items = 0;
        if (c->step < kLogCap) c->log_front[c->step] = c->count[c->cur];
        c->active = 1;
    }
}

__global__ void k_begin(Control* c, int generate, uint32_t max_steps) {
    c->steps_done = 0;
    c->max_steps = max_steps;
    c->status = generate ? kStatusRunning : 0;
    c->active = 0;
}

__global__ void k_set_params(Control* c, unsigned long long R0, unsigned long long R1,
                             unsigned long long R2, uint32_t law, unsigned long long n_t,
                             uint32_t has_target, unsigned long long N) {
    c->R[0] = R0; c->R[1] = R1; c->R[2] = R2;
    c->law = law; c->n_t = n_t; c->has_target = has_target; c->N = N;
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

cudaError_t launch_set_params(liets_ctx* c) {
    k_set_params<<<1, 1, 0, c->stream>>>(c->ctl, c->R[0], c->R[1], c->R[2], (uint32_t)c->law, c->n_t,
                                         c->has_target ? 1u : 0u, c->N);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace liets
