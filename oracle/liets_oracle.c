/*
 * liets_oracle.c -- CPU ORACLE for the LIETS-QSGS growth path.  TEST INFRASTRUCTURE ONLY.
 * See liets_oracle.h for scope, citations and pins.  Plain serial C99 (+ gcc's __int128),
 * no blocking, no fusion, no reordering beyond what the cited passage states.
 */
#include "liets_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (R9).  One round:
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
 * between rounds k0 += W0, k1 += W1; ten rounds.
 * ------------------------------------------------------------------------------------------ */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t prod0 = (uint64_t)M0 * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(prod1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)prod1;
        uint32_t n2 = (uint32_t)(prod0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)prod0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R9: growth draw.  The 32-bit draw of (voxel p, step t, direction d) is written nibble by nibble,
 * most significant first, from eight Philox blocks of the voxel -- block k holds nibble k of the
 * draws of all 26 directions:
 *   key = (seed lo, seed hi);   B_k = philox(counter = (p lo, p hi, step t, k)),  k = 0..7;
 *   nibble k of draw(d) = bits [4 (d / 4), 4 (d / 4) + 4) of word d % 4 of B_k;
 *   draw(d) = sum_k  nibble_k << (28 - 4 k). */
uint32_t oracle_growth_draw(uint64_t rng_seed, uint32_t t, uint64_t p, int d) {
    uint32_t key[2] = { (uint32_t)(rng_seed & 0xFFFFFFFFu), (uint32_t)(rng_seed >> 32) };
    uint32_t draw = 0;
    for (uint32_t k = 0; k < 8; ++k) {
        uint32_t ctr[4] = { (uint32_t)(p & 0xFFFFFFFFu), (uint32_t)(p >> 32), t, k };
        uint32_t B[4];
        oracle_philox4x32_10(ctr, key, B);
        uint32_t nibble = (B[d % 4] >> (4 * (d / 4))) & 0xFu;
        draw |= nibble << (28 - 4 * k);
    }
    return draw;
}

/* R9: seeding draw.  counter = ((v/4) lo, (v/4) hi, 0, 0xFFFFFFFF); draw of voxel v is word v % 4.
 * (c3 = 0xFFFFFFFF never collides with a growth counter, whose c3 is 0..7.) */
uint32_t oracle_seed_draw(uint64_t rng_seed, uint64_t v) {
    uint32_t key[2] = { (uint32_t)(rng_seed & 0xFFFFFFFFu), (uint32_t)(rng_seed >> 32) };
    uint64_t blk = v / 4;
    uint32_t ctr[4] = { (uint32_t)(blk & 0xFFFFFFFFu), (uint32_t)(blk >> 32), 0u, 0xFFFFFFFFu };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[v % 4];
}

/* R19 (the order kept in reserve there): the key of voxel v in the keyed acceptance order of the
 * spacing filter.  The paper does not say in which order candidate cores are tried; with this key the
 * order is a random permutation fixed by the seed.  Counter (v/4, 0, 1, 2^32-1): the core draw uses (v/4, 0, 0, 2^32-1),
 * the growth draws have a last word <= 7, so the three streams never meet. */
uint32_t oracle_seed_priority(uint64_t rng_seed, uint64_t v) {
    uint32_t key[2] = { (uint32_t)(rng_seed & 0xFFFFFFFFu), (uint32_t)(rng_seed >> 32) };
    uint64_t blk = v / 4;
    uint32_t ctr[4] = { (uint32_t)(blk & 0xFFFFFFFFu), (uint32_t)(blk >> 32), 1u, 0xFFFFFFFFu };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[v % 4];
}

/* ------------------------------------------------------------------------------------------
 * R1: the 26 directions.  See DESIGN.md "Readings" R1 for the order; class = |dx|+|dy|+|dz|.
 * ------------------------------------------------------------------------------------------ */
#include "liets_oracle_directions.inc"

void oracle_direction(int d, int* dx, int* dy, int* dz, int* cls) {
    *dx = ORACLE_DIRS[d][0]; *dy = ORACLE_DIRS[d][1]; *dz = ORACLE_DIRS[d][2];
    *cls = abs(*dx) + abs(*dy) + abs(*dz);
}

/* ------------------------------------------------------------------------------------------
 * Integer thresholds (R7, R8) and Eq. (1) (R6).
 * ------------------------------------------------------------------------------------------ */
uint64_t oracle_prob_to_threshold(double p) {
    if (p <= 0.0) return 0;
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)floor(p * 4294967296.0 + 0.5);
}

uint64_t oracle_target_count(double phi_s, uint64_t N) {
    double x = ceil(phi_s * (double)N);
    if (x < 1.0) return 1;
    if (x > (double)N) return N;
    return (uint64_t)x;
}

/* G = G_ref (phi_s - 0.95 phi_a)/(0.05 phi_s) = G_ref (20 n_t - 19 n_solid)/n_t, clamped to [0,1]. */
uint64_t oracle_step_threshold(uint64_t R, int law, uint64_t n_t, uint64_t n_solid) {
    if (law == 0) return R;
    unsigned __int128 a = (unsigned __int128)20 * n_t;
    unsigned __int128 b = (unsigned __int128)19 * n_solid;
    if (b >= a) return 0;
    unsigned __int128 T = ((unsigned __int128)R * (a - b)) / n_t;
    unsigned __int128 one = (unsigned __int128)1 << 32;
    return (uint64_t)(T > one ? one : T);
}

/* ------------------------------------------------------------------------------------------
 * State
 * ------------------------------------------------------------------------------------------ */
struct oracle_state {
    int nx, ny, nz, periodic;
    uint64_t N;
    uint8_t* grid;            /* phase array, 1 = solid, 0 = void; 2 = a cell of an earlier phase (PAPER.md:40 step 4) */
    uint8_t* blocked;         /* NULL, or N bytes: 1 = the cell belongs to an earlier growing phase */
    uint64_t* front;          /* active set A */
    uint64_t n_front, cap_front;
    uint64_t n_solid;
    uint32_t step;            /* t: continues across step/generate calls */
    uint64_t rng_seed;
    int seeded;
    uint64_t R[4];            /* R[class], class 1..3 */
    int law;
    int has_target;
    uint64_t n_t;
    uint64_t attempts[26], successes[26];
    int spacing_order;        /* 0: candidates are tried in ascending index (R12); 1: in ascending (key, index) (R19) */
    int interact;             /* R20: cells of the earlier phases are sources too, with the thresholds RI */
    uint64_t RI[4];           /* RI[class]: floor(I 2^32 + 0.5), constant over the run */
};

oracle_state* oracle_new(int nx, int ny, int nz, int periodic) {
    if (nx < 1 || ny < 1 || nz < 1) return NULL;
    oracle_state* o = (oracle_state*)calloc(1, sizeof(*o));
    o->nx = nx; o->ny = ny; o->nz = nz; o->periodic = periodic & 7;    /* bit 0: x wraps, bit 1: y, bit 2: z (R5) */
    o->N = (uint64_t)nx * (uint64_t)ny * (uint64_t)nz;
    o->grid = (uint8_t*)calloc(o->N, 1);
    o->cap_front = 1024;
    o->front = (uint64_t*)malloc(o->cap_front * sizeof(uint64_t));
    return o;
}

void oracle_free(oracle_state* o) {
    if (!o) return;
    free(o->grid); free(o->blocked); free(o->front); free(o);
}

int oracle_set_growth(oracle_state* o, double g_face, double g_edge, double g_corner, int law) {
    if (g_face < 0 || g_face > 1 || g_edge < 0 || g_edge > 1 || g_corner < 0 || g_corner > 1) return -1;
    if (law != 0 && law != 1) return -1;
    o->R[1] = oracle_prob_to_threshold(g_face);
    o->R[2] = oracle_prob_to_threshold(g_edge);
    o->R[3] = oracle_prob_to_threshold(g_corner);
    o->law = law;
    return 0;
}

int oracle_set_target(oracle_state* o, double phi_s) {
    if (!(phi_s > 0.0) || phi_s > 1.0) return -1;
    o->n_t = oracle_target_count(phi_s, o->N);
    o->has_target = 1;
    return 0;
}

static void front_push(oracle_state* o, uint64_t p) {
    if (o->n_front == o->cap_front) {
        o->cap_front *= 2;
        o->front = (uint64_t*)realloc(o->front, o->cap_front * sizeof(uint64_t));
    }
    o->front[o->n_front++] = p;
}

/* neighbour of p in direction d: returns 1 and *q if it exists (inside a non-periodic domain,
 * PAPER.md:53, :145; or wrapped per coordinate if periodic, "roll"; R5). */
static int neighbour(const oracle_state* o, uint64_t p, int d, uint64_t* q) {
    int64_t x = (int64_t)(p % (uint64_t)o->nx);
    int64_t y = (int64_t)((p / (uint64_t)o->nx) % (uint64_t)o->ny);
    int64_t z = (int64_t)(p / ((uint64_t)o->nx * (uint64_t)o->ny));
    x += ORACLE_DIRS[d][0]; y += ORACLE_DIRS[d][1]; z += ORACLE_DIRS[d][2];
    /* per axis: wrapped if that axis is periodic ("roll"), else the neighbour must lie inside (:53, :145) */
    if (o->periodic & 1) x = (x % o->nx + o->nx) % o->nx; else if (x < 0 || x >= o->nx) return 0;
    if (o->periodic & 2) y = (y % o->ny + o->ny) % o->ny; else if (y < 0 || y >= o->ny) return 0;
    if (o->periodic & 4) z = (z % o->nz + o->nz) % o->nz; else if (z < 0 || z >= o->nz) return 0;
    *q = (uint64_t)x + (uint64_t)o->nx * ((uint64_t)y + (uint64_t)o->ny * (uint64_t)z);
    return 1;
}

/* does solid cell p have at least one void neighbour (R13) */
static int has_void_neighbour(const oracle_state* o, uint64_t p) {
    for (int d = 0; d < 26; ++d) {
        uint64_t q;
        if (neighbour(o, p, d, &q) && o->grid[q] == 0) return 1;
    }
    return 0;
}

/* Multi-phase growth, independent phases (PAPER.md:40 step 4: "The remaining phases are generated on the still
 * unassigned cells ... its cores are placed and grown in the same way as for the first phase"): cells of the phases grown
 * before are given as a mask.  They are not void -- never cores, never claimed -- and not of this phase -- never sources,
 * not counted in n_solid.  mask = NULL clears.  Takes effect at the next seeding. */
int oracle_set_blocked(oracle_state* o, const uint8_t* mask) {
    free(o->blocked);
    o->blocked = NULL;
    if (mask) {
        o->blocked = (uint8_t*)malloc(o->N);
        for (uint64_t v = 0; v < o->N; ++v) o->blocked[v] = mask[v] ? 1 : 0;
    }
    o->seeded = 0;
    return 0;
}

/* Interacting phases (PAPER.md:40 step 4, R20): the growing phase n also grows at its interface with the earlier phases m --
 * a still unassigned cell q next to a cell p of an earlier phase (q = p + e_d) is taken by phase n with the
 * phase-interaction probability I_d^{n,m}, one per direction class, constant over the run.  In the words of the list
 * algorithm: the cells of the earlier phases that have a void neighbour are sources beside the front of phase n, with
 * I in place of G; the draw of (p, t, d) is the same keyed draw.  All three 0 switches it off.  Takes effect at the next
 * seeding. */
int oracle_set_interaction(oracle_state* o, double i_face, double i_edge, double i_corner) {
    if (i_face < 0 || i_face > 1 || i_edge < 0 || i_edge > 1 || i_corner < 0 || i_corner > 1) return -1;
    o->RI[1] = oracle_prob_to_threshold(i_face);
    o->RI[2] = oracle_prob_to_threshold(i_edge);
    o->RI[3] = oracle_prob_to_threshold(i_corner);
    o->interact = (o->RI[1] | o->RI[2] | o->RI[3]) != 0;
    o->seeded = 0;
    return 0;
}

/* R20: after the seeds, the interface cells of the earlier phases join the sources (ascending index) */
static void push_interface_sources(oracle_state* o) {
    if (!o->interact || !o->blocked) return;
    for (uint64_t v = 0; v < o->N; ++v)
        if (o->grid[v] == 2 && has_void_neighbour(o, v)) front_push(o, v);
}

static void reset_run(oracle_state* o, uint64_t rng_seed) {
    memset(o->grid, 0, o->N);
    if (o->blocked)
        for (uint64_t v = 0; v < o->N; ++v)
            if (o->blocked[v]) o->grid[v] = 2;
    o->n_front = 0; o->n_solid = 0; o->step = 0; o->rng_seed = rng_seed; o->seeded = 1;
    memset(o->attempts, 0, sizeof(o->attempts));
    memset(o->successes, 0, sizeof(o->successes));
}

/* ------------------------------------------------------------------------------------------
 * Seeding and seed spacing (R11, R12).
 * Candidates: every voxel v, ascending index, whose draw is below T_core.
 * Spacing: scan candidates in ascending index; accept v iff every already accepted seed w has
 * L1(v,w) >= s (per-axis min(|D|, n-|D|) if periodic).  s <= 1 accepts all.
 * ------------------------------------------------------------------------------------------ */
static int64_t axis_dist(int64_t a, int64_t b, int n, int periodic) {
    int64_t d = a > b ? a - b : b - a;
    if (periodic && n - d < d) d = n - d;
    return d;
}

static int64_t l1_dist(const oracle_state* o, uint64_t v, uint64_t w) {
    int64_t vx = (int64_t)(v % (uint64_t)o->nx), wx = (int64_t)(w % (uint64_t)o->nx);
    int64_t vy = (int64_t)((v / (uint64_t)o->nx) % (uint64_t)o->ny), wy = (int64_t)((w / (uint64_t)o->nx) % (uint64_t)o->ny);
    int64_t vz = (int64_t)(v / ((uint64_t)o->nx * (uint64_t)o->ny)), wz = (int64_t)(w / ((uint64_t)o->nx * (uint64_t)o->ny));
    return axis_dist(vx, wx, o->nx, o->periodic & 1) + axis_dist(vy, wy, o->ny, o->periodic & 2) +
           axis_dist(vz, wz, o->nz, o->periodic & 4);
}

int oracle_set_spacing_order(oracle_state* o, int order) {
    if (order != 0 && order != 1) return -1;
    o->spacing_order = order;
    return 0;
}

typedef struct { uint32_t key; uint64_t v; } keyed_cand;

static int keyed_cmp(const void* a, const void* b) {
    const keyed_cand* p = (const keyed_cand*)a;
    const keyed_cand* q = (const keyed_cand*)b;
    if (p->key != q->key) return p->key < q->key ? -1 : 1;
    return p->v < q->v ? -1 : (p->v > q->v ? 1 : 0);
}

static int u64_cmp(const void* a, const void* b) {
    uint64_t p = *(const uint64_t*)a, q = *(const uint64_t*)b;
    return p < q ? -1 : (p > q ? 1 : 0);
}

int64_t oracle_seed(oracle_state* o, double core_prob, int spacing_s, uint64_t rng_seed) {
    if (core_prob < 0.0 || core_prob > 1.0 || spacing_s < 0) return -1;
    reset_run(o, rng_seed);
    uint64_t T_core = oracle_prob_to_threshold(core_prob);
    if (o->spacing_order == 1 && spacing_s > 1) {
        /* R19: the same candidates, tried in ascending (key, index) instead of ascending index */
        uint64_t n = 0, cap = 1024;
        keyed_cand* c = (keyed_cand*)malloc(cap * sizeof(*c));
        for (uint64_t v = 0; v < o->N; ++v) {
            if (o->grid[v] != 0) continue;
            if ((uint64_t)oracle_seed_draw(rng_seed, v) >= T_core) continue;
            if (n == cap) { cap *= 2; c = (keyed_cand*)realloc(c, cap * sizeof(*c)); }
            c[n].key = oracle_seed_priority(rng_seed, v); c[n].v = v; ++n;
        }
        qsort(c, n, sizeof(*c), keyed_cmp);
        for (uint64_t k = 0; k < n; ++k) {
            int ok = 1;
            for (uint64_t i = 0; i < o->n_front; ++i)                       /* accepted so far */
                if (l1_dist(o, c[k].v, o->front[i]) < (int64_t)spacing_s) { ok = 0; break; }
            if (ok) { o->grid[c[k].v] = 1; front_push(o, c[k].v); }
        }
        free(c);
        qsort(o->front, o->n_front, sizeof(uint64_t), u64_cmp);             /* A_0 listed in ascending index, as always */
        o->n_solid = o->n_front;
        push_interface_sources(o);
        return (int64_t)o->n_solid;
    }
    for (uint64_t v = 0; v < o->N; ++v) {
        if (o->grid[v] != 0) continue;                                     /* an earlier phase's cell: not unassigned */
        if ((uint64_t)oracle_seed_draw(rng_seed, v) >= T_core) continue;   /* not a candidate */
        int ok = 1;
        if (spacing_s > 1) {
            for (uint64_t i = 0; i < o->n_front; ++i) {                    /* accepted so far */
                if (l1_dist(o, v, o->front[i]) < (int64_t)spacing_s) { ok = 0; break; }
            }
        }
        if (ok) { o->grid[v] = 1; front_push(o, v); }
    }
    o->n_solid = o->n_front;       /* A_0 = seeds (R3) */
    push_interface_sources(o);
    return (int64_t)o->n_solid;
}

/* The spacing filter as the paper words it (Fig. 1(D): "diamond dilation is conducted with a small
 * kernel but multiple iterations"): a candidate is accepted iff it is not covered, and every accepted seed covers its
 * diamond, grown literally by s-1 passes of the 6-neighbour kernel (pass: every covered cell covers its face
 * neighbours; walls or wrap per axis as the grid's boundary says).  Ascending index order only.  Same result as
 * oracle_seed (pin P5d); cost O(s^3) per seed, for small cases. */
int64_t oracle_seed_by_dilation(oracle_state* o, double core_prob, int spacing_s, uint64_t rng_seed) {
    static const int FACE[6] = { 4, 10, 12, 13, 15, 21 };                  /* the six directions of class 1 (R1) */
    if (core_prob < 0.0 || core_prob > 1.0 || spacing_s < 0) return -1;
    for (int k = 0; k < 6; ++k)
        if (abs(ORACLE_DIRS[FACE[k]][0]) + abs(ORACLE_DIRS[FACE[k]][1]) + abs(ORACLE_DIRS[FACE[k]][2]) != 1) return -3;
    reset_run(o, rng_seed);
    uint64_t T_core = oracle_prob_to_threshold(core_prob);
    uint8_t* covered = (uint8_t*)calloc(o->N, 1);
    uint64_t* wave = (uint64_t*)malloc(o->N * sizeof(uint64_t));
    for (uint64_t v = 0; v < o->N; ++v) {
        if (o->grid[v] != 0) continue;
        if ((uint64_t)oracle_seed_draw(rng_seed, v) >= T_core) continue;
        if (spacing_s > 1 && covered[v]) continue;
        o->grid[v] = 1; front_push(o, v);
        if (spacing_s > 1) {
            uint8_t* mine = (uint8_t*)calloc(o->N, 1);                     /* this seed's diamond */
            uint64_t n_wave = 1, lo = 0;
            wave[0] = v; mine[v] = 1;
            for (int pass = 1; pass < spacing_s; ++pass) {                 /* s-1 passes */
                uint64_t hi = n_wave;
                for (uint64_t i = lo; i < hi; ++i)
                    for (int k = 0; k < 6; ++k) {
                        uint64_t q;
                        if (neighbour(o, wave[i], FACE[k], &q) && !mine[q]) { mine[q] = 1; wave[n_wave++] = q; }
                    }
                lo = hi;
            }
            for (uint64_t i = 0; i < n_wave; ++i) covered[wave[i]] = 1;
            free(mine);
        }
    }
    free(covered); free(wave);
    o->n_solid = o->n_front;
    push_interface_sources(o);
    return (int64_t)o->n_solid;
}

int64_t oracle_seed_explicit(oracle_state* o, const uint64_t* idx, uint64_t n, uint64_t rng_seed) {
    reset_run(o, rng_seed);
    for (uint64_t i = 0; i < n; ++i) {
        if (idx[i] >= o->N) return -1;
        if (o->grid[idx[i]] == 0) { o->grid[idx[i]] = 1; front_push(o, idx[i]); }
    }
    o->n_solid = o->n_front;
    push_interface_sources(o);
    return (int64_t)o->n_solid;
}

/* per-step thresholds, evaluated once from n_solid at the start of the step (R6) */
static int step_thresholds(const oracle_state* o, uint64_t T[4]) {
    if (!o->seeded) return -2;
    if (o->law == 1 && !o->has_target) return -2;
    for (int c = 1; c <= 3; ++c) T[c] = oracle_step_threshold(o->R[c], o->law, o->n_t, o->n_solid);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * One step, plain definition (Algorithm 2, keyed draws; "counted
 * once"; PAPER.md:78 new cells act only in the next iteration):
 *   for every p with g_t[p] = 1, every direction d, q = p + e_d: if q exists and g_t[q] = 0 and
 *   draw(seed, t, p, d) < T_class(d) then g_{t+1}[q] = 1.
 * ------------------------------------------------------------------------------------------ */
int oracle_step_full(oracle_state* o) {
    uint64_t T[4];
    int rc = step_thresholds(o, T);
    if (rc) return rc;
    uint8_t* next = (uint8_t*)malloc(o->N);
    memcpy(next, o->grid, o->N);
    for (uint64_t p = 0; p < o->N; ++p) {
        if (o->grid[p] != 1 && !(o->interact && o->grid[p] == 2)) continue;     /* sources: phase n, and (R20) the earlier phases */
        const uint64_t* Tp = o->grid[p] == 1 ? T : o->RI;
        for (int d = 0; d < 26; ++d) {
            uint64_t q;
            if (!neighbour(o, p, d, &q)) continue;
            if (o->grid[q] != 0) continue;
            int cls = abs(ORACLE_DIRS[d][0]) + abs(ORACLE_DIRS[d][1]) + abs(ORACLE_DIRS[d][2]);
            o->attempts[d]++;
            if ((uint64_t)oracle_growth_draw(o->rng_seed, o->step, p, d) < Tp[cls]) {
                o->successes[d]++;
                next[q] = 1;
            }
        }
    }
    memcpy(o->grid, next, o->N);
    free(next);
    /* phi_a recomputed from the phase array; the front is rebuilt by definition */
    o->n_solid = 0; o->n_front = 0;
    for (uint64_t p = 0; p < o->N; ++p) o->n_solid += (o->grid[p] == 1);
    for (uint64_t p = 0; p < o->N; ++p)
        if ((o->grid[p] == 1 || (o->interact && o->grid[p] == 2)) && has_void_neighbour(o, p)) front_push(o, p);
    o->step++;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * One step, Algorithm 3 line by line.  A_{t+1} = prune(A_t U A_new) (R4).
 * ------------------------------------------------------------------------------------------ */
int oracle_step_list(oracle_state* o) {
    uint64_t T[4];
    int rc = step_thresholds(o, T);
    if (rc) return rc;
    uint64_t n_old = o->n_front;                       /* sources: A at the start of the step */
#ifndef _OPENMP
    for (int d = 0; d < 26; ++d) {                     /* line 4: for each d in directions   */
        int cls = abs(ORACLE_DIRS[d][0]) + abs(ORACLE_DIRS[d][1]) + abs(ORACLE_DIRS[d][2]);
        for (uint64_t i = 0; i < n_old; ++i) {
            uint64_t p = o->front[i], q;
            if (!neighbour(o, p, d, &q)) continue;     /* line 5: N_d inside domain          */
            if (o->grid[q] != 0) continue;             /* line 6: C_d, still void            */
            const uint64_t* Tp = o->grid[p] == 1 ? T : o->RI;                   /* (R20: a source of an earlier phase uses I) */
            if ((uint64_t)oracle_growth_draw(o->rng_seed, o->step, p, d) < Tp[cls]) { /* line 8 */
                o->grid[q] = 1;                        /* line 9                             */
                front_push(o, q);                      /* line 10: A_new U {q}, once per q   */
                o->n_solid++;
            }
        }
    }
    /* line 14: prune -- drop cells with no void neighbour (duplicates cannot occur: a cell is
     * pushed only at its 0 -> 1 transition) */
    uint64_t kept = 0;
    for (uint64_t i = 0; i < o->n_front; ++i)
        if (has_void_neighbour(o, o->front[i])) o->front[kept++] = o->front[i];
    o->n_front = kept;
#else
    /* The same loops with the front shared among the host's cores (liboracle_omp.so, the all-cores
     * CPU baseline of bench.py).  Legal because draws are keyed by (seed, t, p, d) and
     * the update is an OR: line 6 reads the cell with an atomic load, line 9 is an atomic exchange
     * whose old value says which thread flipped 0 -> 1 -- that thread alone appends q (line 10), to a
     * list of its own; the lists are joined after each direction.  The order of A differs from the
     * serial run, the grid cannot (pin P7).  tests/test_oracle_pins.py proves both libraries equal. */
    int nth = omp_get_max_threads();
    uint64_t** buf = (uint64_t**)calloc((size_t)nth, sizeof(uint64_t*));
    uint64_t* nbuf = (uint64_t*)calloc((size_t)nth, sizeof(uint64_t));
    uint64_t* cbuf = (uint64_t*)calloc((size_t)nth, sizeof(uint64_t));
    for (int d = 0; d < 26; ++d) {                     /* line 4 */
        int cls = abs(ORACLE_DIRS[d][0]) + abs(ORACLE_DIRS[d][1]) + abs(ORACLE_DIRS[d][2]);
#pragma omp parallel
        {
            int me = omp_get_thread_num();
            nbuf[me] = 0;
#pragma omp for schedule(static)
            for (uint64_t i = 0; i < n_old; ++i) {
                uint64_t p = o->front[i], q;
                if (!neighbour(o, p, d, &q)) continue;                                   /* line 5 */
                if (__atomic_load_n(&o->grid[q], __ATOMIC_RELAXED) != 0) continue;       /* line 6 */
                const uint64_t* Tp = o->grid[p] == 1 ? T : o->RI;
                if ((uint64_t)oracle_growth_draw(o->rng_seed, o->step, p, d) < Tp[cls]) { /* line 8 */
                    if (__atomic_exchange_n(&o->grid[q], 1, __ATOMIC_RELAXED) == 0) {    /* line 9 */
                        if (nbuf[me] == cbuf[me]) {                                      /* line 10 */
                            cbuf[me] = cbuf[me] ? 2 * cbuf[me] : 1024;
                            buf[me] = (uint64_t*)realloc(buf[me], cbuf[me] * sizeof(uint64_t));
                        }
                        buf[me][nbuf[me]++] = q;
                    }
                }
            }
        }
        for (int k = 0; k < nth; ++k)
            for (uint64_t j = 0; j < nbuf[k]; ++j) { front_push(o, buf[k][j]); o->n_solid++; }
    }
    for (int k = 0; k < nth; ++k) free(buf[k]);
    free(buf); free(nbuf); free(cbuf);
    /* line 14: prune, the test in parallel, the compaction in order */
    uint8_t* keep = (uint8_t*)malloc(o->n_front ? o->n_front : 1);
#pragma omp parallel for schedule(static)
    for (uint64_t i = 0; i < o->n_front; ++i) keep[i] = (uint8_t)has_void_neighbour(o, o->front[i]);
    uint64_t kept = 0;
    for (uint64_t i = 0; i < o->n_front; ++i)
        if (keep[i]) o->front[kept++] = o->front[i];
    free(keep);
    o->n_front = kept;
#endif
    o->step++;
    return 0;
}

/* while phi_a < phi_s and A not empty (R7: n_solid < n_t; R14: max_steps) */
int oracle_generate(oracle_state* o, double phi_s, uint32_t max_steps, int use_list,
                    uint32_t* steps_out) {
    if (oracle_set_target(o, phi_s)) return -1;
    if (!o->seeded) return -2;
    uint32_t done = 0;
    int status = ORACLE_OK;
    for (;;) {
        if (o->n_solid >= o->n_t) { status = ORACLE_OK; break; }
        if (o->n_front == 0) { status = ORACLE_FRONT_EMPTY; break; }
        if (done >= max_steps) { status = ORACLE_MAX_STEPS; break; }
        int rc = use_list ? oracle_step_list(o) : oracle_step_full(o);
        if (rc) return rc;
        done++;
    }
    if (steps_out) *steps_out = done;
    return status;
}

/* host threads oracle_step_list uses: 1 in liboracle.so, omp_get_max_threads() in liboracle_omp.so */
int oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

const uint8_t* oracle_grid(const oracle_state* o) { return o->grid; }
uint64_t oracle_n_solid(const oracle_state* o) { return o->n_solid; }
uint32_t oracle_step_index(const oracle_state* o) { return o->step; }
uint64_t oracle_n_target(const oracle_state* o) { return o->n_t; }

uint64_t oracle_n_front_exact(const oracle_state* o) {
    uint64_t n = 0;
    for (uint64_t p = 0; p < o->N; ++p)
        if (o->grid[p] == 1 && has_void_neighbour(o, p)) n++;
    return n;
}

void oracle_rates(const oracle_state* o, uint64_t attempts[26], uint64_t successes[26]) {
    memcpy(attempts, o->attempts, sizeof(o->attempts));
    memcpy(successes, o->successes, sizeof(o->successes));
}

void oracle_permute_front(oracle_state* o, int how, uint64_t key) {
    uint64_t n = o->n_front;
    if (how == 1) {
        for (uint64_t i = 0; i < n / 2; ++i) {
            uint64_t tmp = o->front[i]; o->front[i] = o->front[n - 1 - i]; o->front[n - 1 - i] = tmp;
        }
    } else if (how == 2) {                              /* Fisher-Yates with a keyed LCG */
        uint64_t s = key * 6364136223846793005ull + 1442695040888963407ull;
        for (uint64_t i = n; i > 1; --i) {
            s = s * 6364136223846793005ull + 1442695040888963407ull;
            uint64_t j = (s >> 33) % i;
            uint64_t tmp = o->front[i - 1]; o->front[i - 1] = o->front[j]; o->front[j] = tmp;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Two-point correlation of the void phase along one axis, exact pair counts (R16).
 * ------------------------------------------------------------------------------------------ */
void oracle_s2(const uint8_t* grid, int nx, int ny, int nz, int periodic, int axis, int rmax,
               uint64_t* pairs, uint64_t* valid) {
    int n[3] = { nx, ny, nz };
    for (int r = 0; r <= rmax; ++r) {
        uint64_t np = 0, nv = 0;
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    int c[3] = { x, y, z };
                    c[axis] += r;
                    if (c[axis] >= n[axis]) {
                        if (!periodic) continue;
                        c[axis] %= n[axis];
                    }
                    nv++;
                    uint64_t a = (uint64_t)x + (uint64_t)nx * ((uint64_t)y + (uint64_t)ny * (uint64_t)z);
                    uint64_t b = (uint64_t)c[0] + (uint64_t)nx * ((uint64_t)c[1] + (uint64_t)ny * (uint64_t)c[2]);
                    if (grid[a] == 0 && grid[b] == 0) np++;
                }
        pairs[r] = np; valid[r] = nv;
    }
}
