/*
 * liets_oracle.h -- CPU ORACLE for the LIETS-QSGS growth path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, serial C restatement of what the hot path of arxiv/paper_2602_11734 computes.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this.  It shares no code with the CUDA library (paper_2602_11734_b200/),
 * and nothing under the product path may include, link or import it.
 *
 * Citations are PAPER.md:<line> (section / algorithm / equation).  Readings of points where the
 * paper is silent or ambiguous are the ones listed in DESIGN.md ("Readings"), cited as R<n>.
 *
 * Parity pins (tests/test_oracle_*.py): Philox known-answer vectors; closed-form L1 balls /
 * Chebyshev cubes; brute-force dilation greedy for seed spacing; big-integer thresholds; the
 * full-field definition == the list algorithm; binomial acceptance rates; one-step claim
 * probability.  "Parity unpinned" (conventions of this repo that the paper does
 * not fix, so nothing outside the repo can pin them): the Philox counter layout (R9), the
 * rounding of phi_s*N to n_t (R7), the rounding of probabilities to 32-bit thresholds (R8),
 * the ascending-index acceptance order of seed spacing (R12), the key of the optional keyed
 * acceptance order (R19: word v % 4 of the Philox block at counter (v / 4, 0, 1, 2^32 - 1)) and
 * which of the two statements of PAPER.md:40 step 4 about interacting phases is meant (R20: the
 * growing phase takes unassigned cells only, also at its interface with the earlier phases, with
 * the probability I of the direction's class).  Further pins: P5d (seeding by literal dilation
 * passes), P5k (the keyed order against an independent greedy), the closed forms of R20.
 */
#ifndef LIETS_ORACLE_H
#define LIETS_ORACLE_H

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_OK = 0, ORACLE_FRONT_EMPTY = 1, ORACLE_MAX_STEPS = 2 };

typedef struct oracle_state oracle_state;

/* Philox4x32-10 (Salmon et al., SC'11); reading R9. ctr[4], key[2] -> out[4]. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* 32-bit draw for "front voxel p tries direction d at step t" (R9). */
uint32_t oracle_growth_draw(uint64_t rng_seed, uint32_t t, uint64_t p, int d);
/* 32-bit draw deciding whether voxel v is a core (R9). */
uint32_t oracle_seed_draw(uint64_t rng_seed, uint64_t v);

/* direction table (R1): fills dx,dy,dz and class (1 face, 2 edge, 3 corner) of direction d. */
void oracle_direction(int d, int* dx, int* dy, int* dz, int* cls);

/* probability -> integer threshold R = floor(p*2^32 + 0.5) in [0, 2^32] (R8). */
uint64_t oracle_prob_to_threshold(double p);
/* n_t = ceil(phi_s * N) clamped to [1, N] (R7). */
uint64_t oracle_target_count(double phi_s, uint64_t N);
/* Eq. (1) in counts: T = min(2^32, floor(R*max(0,20 n_t - 19 n_solid)/n_t)) (R6,R8);
 * law 0 = constant probability: T = R. */
uint64_t oracle_step_threshold(uint64_t R, int law, uint64_t n_t, uint64_t n_solid);

/* periodic: bit 0 = x wraps, bit 1 = y wraps, bit 2 = z wraps (R5); 0 = walls all round, 7 = torus, 3 = periodic in
 * the x-y plane between walls in z (with nz = 1: the two-dimensional periodic grid of Algorithm 2) */
oracle_state* oracle_new(int nx, int ny, int nz, int periodic);
void oracle_free(oracle_state* o);

int oracle_set_growth(oracle_state* o, double g_face, double g_edge, double g_corner, int law);
int oracle_set_target(oracle_state* o, double phi_s);

/* Seeding + seed spacing (R11, R12). Resets grid, front, step. */
int64_t oracle_seed(oracle_state* o, double core_prob, int spacing_s, uint64_t rng_seed);
/* R19: 0 (default) = candidates are tried in ascending index (R12); 1 = in ascending (oracle_seed_priority, index), a
 * random order fixed by the seed.  Used by the next oracle_seed. */
int oracle_set_spacing_order(oracle_state* o, int order);
uint32_t oracle_seed_priority(uint64_t rng_seed, uint64_t v);
/* The spacing filter by literal diamond dilation (s-1 passes of the 6-neighbour kernel per accepted seed),
 * ascending index order: the same seeds as oracle_seed. */
int64_t oracle_seed_by_dilation(oracle_state* o, double core_prob, int spacing_s, uint64_t rng_seed);
/* Same candidates, but place an explicit list of seeds instead (for closed-form tests). */
int64_t oracle_seed_explicit(oracle_state* o, const uint64_t* idx, uint64_t n, uint64_t rng_seed);

/* One synchronous growth step.
 *   oracle_step_full: the plain definition (Algorithm 2, with keyed draws).
 *   oracle_step_list: Algorithm 3 followed line by line, exact prune.      */
int oracle_step_full(oracle_state* o);
int oracle_step_list(oracle_state* o);

/* while phi_a < phi_s and A not empty, at most max_steps; use_list picks the
 * step function. Returns ORACLE_OK / FRONT_EMPTY / MAX_STEPS; *steps_out = steps done now. */
int oracle_generate(oracle_state* o, double phi_s, uint32_t max_steps, int use_list,
                    uint32_t* steps_out);

int oracle_threads(void);
/* cells of earlier growing phases (N bytes, non-zero = taken; NULL clears): not void, not of this phase (PAPER.md:40 step 4,
 * independent phases).  oracle_grid then holds 2 in those cells.  Takes effect at the next oracle_seed. */
int oracle_set_blocked(oracle_state* o, const uint8_t* mask);
/* R20 (PAPER.md:40 step 4, interacting phases): the cells of the earlier phases that have a void neighbour are sources too,
 * with the phase-interaction probabilities I (face, edge, corner; constant) in place of G.  0, 0, 0 switches it off.
 * Takes effect at the next oracle_seed*. */
int oracle_set_interaction(oracle_state* o, double i_face, double i_edge, double i_corner);
const uint8_t* oracle_grid(const oracle_state* o);          /* N bytes in {0,1}, x fastest */
uint64_t oracle_n_solid(const oracle_state* o);
uint64_t oracle_n_front_exact(const oracle_state* o);       /* #solid cells with a void neighbour */
uint32_t oracle_step_index(const oracle_state* o);
uint64_t oracle_n_target(const oracle_state* o);
/* instrumentation of oracle_step_full: per direction, attempts (source solid, target void at
 * step start) and successes (draw < T). Cumulative since the last oracle_seed*. */
void oracle_rates(const oracle_state* o, uint64_t attempts[26], uint64_t successes[26]);
/* reorder the front list (test of order independence, pin P7): 1 = reverse, 2 = keyed shuffle */
void oracle_permute_front(oracle_state* o, int how, uint64_t key);

/* Two-point correlation of the VOID phase along one axis (R16): for r = 0..rmax,
 * pairs[r] = #{x : void(x) and void(x + r e_axis)}, valid[r] = #{x : x + r e_axis is counted}. */
void oracle_s2(const uint8_t* grid, int nx, int ny, int nz, int periodic, int axis, int rmax,
               uint64_t* pairs, uint64_t* valid);

#ifdef __cplusplus
}
#endif
#endif
