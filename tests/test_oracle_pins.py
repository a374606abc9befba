"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test names the pin of SURVEY.md section 8(c) / DESIGN.md it implements.  Nothing here touches
the CUDA path: the oracle must be trustworthy before any kernel is compared with it.
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def coords(shape):
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return x, y, z


def axis_d(a, b, n, periodic):
    d = np.abs(a - b)
    return np.minimum(d, n - d) if periodic else d


# ------------------------------------------------------------------------------------------ P1
def test_p1_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l[0] not in "#\n"]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_p1_draw_layout_matches_philox_block():
    # R9: hex digit k (most significant first) of the growth draw of direction d = hex digit d//4 (least significant
    # first) of word d%4 of block (p lo, p hi, t, k); seeding counter = (v//4, 0, 0, ~0), word v%4
    seed = 0x0123456789ABCDEF
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for p, t, d in [(0, 0, 0), (12345, 7, 13), (2**32 - 1, 40, 25), (2**31 + 5, 3, 22), (77, 1, 8), (77, 1, 15)]:
        digits = ""
        for k in range(8):
            blk = oracle.philox4x32_10([p & 0xFFFFFFFF, p >> 32, t, k], key)
            digits += ("%08x" % blk[d % 4])[7 - d // 4]
        assert "%08x" % oracle.growth_draw(seed, t, p, d) == digits
    for v in [0, 1, 2, 3, 4, 1000003, 2**32 - 1]:
        blk = oracle.philox4x32_10([(v // 4) & 0xFFFFFFFF, (v // 4) >> 32, 0, 0xFFFFFFFF], key)
        assert oracle.seed_draw(seed, v) == blk[v % 4]


def test_p1_growth_draws_are_uniform_and_independent_across_directions():
    # the 26 draws of one (seed, t, p) must behave as independent uniforms: chi-square of
    # the top byte per direction, and no correlation between the draws of direction pairs
    seed, n = 99, 6000
    draws = np.array([[oracle.growth_draw(seed, t, p, d) for d in range(26)]
                      for t, p in zip(np.arange(n) % 7, np.arange(n) * 977 + 5)], dtype=np.float64) / 2**32
    assert np.all(np.abs(draws.mean(axis=0) - 0.5) < 5 * math.sqrt(1 / 12 / n))
    for d in range(26):
        hist = np.bincount((draws[:, d] * 16).astype(int), minlength=16)
        chi2 = ((hist - n / 16) ** 2 / (n / 16)).sum()
        assert chi2 < 50, (d, chi2)                                # 15 dof: P(chi2 > 50) ~ 1e-5
    c = np.corrcoef(draws.T)
    assert np.abs(c - np.eye(26)).max() < 5 / math.sqrt(n)


def test_direction_table_is_the_26_neighbourhood():
    ds = [oracle.direction(d) for d in range(26)]
    vecs = [d[:3] for d in ds]
    assert len(set(vecs)) == 26 and (0, 0, 0) not in vecs
    assert all(max(map(abs, v)) == 1 for v in vecs)
    cls = [d[3] for d in ds]
    assert (cls.count(1), cls.count(2), cls.count(3)) == (6, 12, 8)       # face / edge / corner
    assert all(c == sum(map(abs, v)) for c, v in zip(cls, vecs))
    # R1: lexicographic in (dz, dy, dx), dz slowest
    assert vecs == [(dx, dy, dz) for dz, dy, dx in itertools.product((-1, 0, 1), repeat=3) if (dx, dy, dz) != (0, 0, 0)]


# ------------------------------------------------------------------------------------------ P8
def test_p8_thresholds_against_big_integers():
    two32 = 1 << 32
    assert oracle.prob_to_threshold(0.0) == 0
    assert oracle.prob_to_threshold(1.0) == two32
    assert oracle.prob_to_threshold(0.5) == 1 << 31
    assert oracle.prob_to_threshold(0.01) == math.floor(0.01 * two32 + 0.5)
    rng = np.random.default_rng(5)
    for _ in range(2000):
        R = int(rng.integers(0, two32 + 1))
        n_t = int(rng.integers(1, 2**32 + 1))
        n = int(rng.integers(0, int(1.2 * n_t) + 1))
        expect = min(two32, (R * max(0, 20 * n_t - 19 * n)) // n_t)
        assert oracle.step_threshold(R, 1, n_t, n) == expect
        assert oracle.step_threshold(R, 0, n_t, n) == R
    for R in (0, 1, 42949673, two32 // 20, two32 // 20 + 1, two32):
        for n_t in (1, 78644, 6_000_000, 858_993_460, 2**32):
            assert oracle.step_threshold(R, 1, n_t, 0) == min(two32, 20 * R)     # 20 G_ref at phi_a = 0
            assert oracle.step_threshold(R, 1, n_t, n_t) == R                    # G_ref at the target
    # Eq. (1) in double precision agrees to one unit of T
    R, n_t = oracle.prob_to_threshold(0.01), 51_200_000
    for n in (0, 1, 999, 25_000_000, 51_199_999):
        phi_s, phi_a = n_t / 64e6, n / 64e6
        G = 0.01 * (phi_s - 0.95 * phi_a) / (0.05 * phi_s)
        assert abs(oracle.step_threshold(R, 1, n_t, n) - G * two32) <= 2.0 + 1e-9 * G * two32


def test_r7_target_count():
    assert oracle.target_count(0.30, 64**3) == 78644
    assert oracle.target_count(0.75, 200**3) == 6_000_000
    assert oracle.target_count(0.8, 2**30) == 858_993_460
    assert oracle.target_count(1.0, 1000) == 1000
    assert oracle.target_count(1e-9, 1000) == 1


# ------------------------------------------------------------------------------------------ P2
def test_p2_zero_growth_leaves_exactly_the_seeds():
    o = oracle.Oracle(40, 36, 28, False)
    o.set_growth(0.0, 0.0, 0.0, 0)
    n = o.seed(0.01, 0, 3)
    g0 = o.grid()
    N = 40 * 36 * 28
    cand = np.array([oracle.seed_draw(3, v) < oracle.prob_to_threshold(0.01) for v in range(N)])
    assert (g0.ravel() == cand).all() and n == cand.sum()
    assert abs(n - 0.01 * N) <= 5 * math.sqrt(N * 0.01 * 0.99)            # binomial bound
    for use_list in (True, False):
        o.step(use_list)
        assert (o.grid() == g0).all() and o.n_solid == n
    rc, steps = o.generate(0.5, 7, True)
    assert rc == oracle.MAX_STEPS and steps == 7 and (o.grid() == g0).all()


# ------------------------------------------------------------------------------------- P3, P4
def _ball_volumes():
    return {int(a): int(b) for a, b in (l.split() for l in open(os.path.join(GOLDEN, "l1_ball_volumes.txt")) if l[0] != "#")}


@pytest.mark.parametrize("use_list", [True, False])
@pytest.mark.parametrize("periodic", [False, True])
def test_p3_face_growth_prob_one_gives_l1_balls(use_list, periodic):
    nx, ny, nz = 23, 19, 21
    vol = _ball_volumes()
    o = oracle.Oracle(nx, ny, nz, periodic)
    o.set_growth(1.0, 0.0, 0.0, 0)
    centre = (11, 9, 10)
    o.seed_explicit([centre[0] + nx * (centre[1] + ny * centre[2])])
    x, y, z = coords((nz, ny, nx))
    for k in range(1, 13):
        o.step(use_list)
        dist = axis_d(x, centre[0], nx, periodic) + axis_d(y, centre[1], ny, periodic) + axis_d(z, centre[2], nz, periodic)
        assert (o.grid() == (dist <= k)).all(), k
        if k <= 9:                                    # ball still clear of walls / of its own images
            assert o.n_solid == vol[k]
    # several seeds, one against a wall / across the seam: union of balls
    seeds = [(0, 0, 0), (22, 18, 20), (5, 17, 3)]
    o.seed_explicit([sx + nx * (sy + ny * sz) for sx, sy, sz in seeds])
    for k in range(1, 6):
        o.step(use_list)
        d = np.min([axis_d(x, sx, nx, periodic) + axis_d(y, sy, ny, periodic) + axis_d(z, sz, nz, periodic)
                    for sx, sy, sz in seeds], axis=0)
        assert (o.grid() == (d <= k)).all()


@pytest.mark.parametrize("periodic", [False, True])
def test_p4_all_directions_prob_one_gives_chebyshev_cubes(periodic):
    nx, ny, nz = 17, 15, 16
    x, y, z = coords((nz, ny, nx))
    c = (3, 7, 12)
    ax, ay, az = axis_d(x, c[0], nx, periodic), axis_d(y, c[1], ny, periodic), axis_d(z, c[2], nz, periodic)
    o = oracle.Oracle(nx, ny, nz, periodic)
    o.set_growth(1.0, 1.0, 1.0, 0)
    o.seed_explicit([c[0] + nx * (c[1] + ny * c[2])])
    for k in range(1, 6):
        o.step(True)
        assert (o.grid() == (np.maximum(np.maximum(ax, ay), az) <= k)).all()
    if not periodic:
        o.seed_explicit([8 + nx * (7 + ny * 8)])
        o.step(True); o.step(True)
        assert o.n_solid == 5 ** 3
    # face + edge at probability 1: {max|D| <= k and sum|D| <= 2k}
    o.set_growth(1.0, 1.0, 0.0, 0)
    o.seed_explicit([c[0] + nx * (c[1] + ny * c[2])])
    for k in range(1, 5):
        o.step(False)
        expect = (np.maximum(np.maximum(ax, ay), az) <= k) & (ax + ay + az <= 2 * k)
        assert (o.grid() == expect).all()
    # corner only: parity-preserving diagonal moves -> after k steps {|Dx|,|Dy|,|Dz| <= k, all same parity as k ... }
    if not periodic:
        o.set_growth(0.0, 0.0, 1.0, 0)
        o.seed_explicit([8 + nx * (7 + ny * 8)])
        o.step(True)
        assert o.n_solid == 1 + 8


# ------------------------------------------------------------------------------------------ P5
def _dilation_greedy(shape, periodic, cand_idx, s):
    """The paper's spacing as literally described: keep a 'blocked' mask that is
    the accepted set dilated s-1 times with the 6-neighbour kernel; accept a candidate iff not blocked."""
    nz, ny, nx = shape
    blocked = np.zeros(shape, bool)
    accepted = []
    for v in cand_idx:
        x, y, z = v % nx, (v // nx) % ny, v // (nx * ny)
        if blocked[z, y, x]:
            continue
        accepted.append(v)
        m = np.zeros(shape, bool)
        m[z, y, x] = True
        for _ in range(max(s - 1, 0)):
            n = m.copy()
            for ax in range(3):
                for sh in (1, -1):
                    r = np.roll(m, sh, axis=ax)
                    if not periodic:
                        sl = [slice(None)] * 3
                        sl[ax] = 0 if sh == 1 else -1
                        r[tuple(sl)] = False
                    n |= r
            m = n
        blocked |= m
    return accepted


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("s", [0, 1, 2, 3, 5, 8])
def test_p5_spacing_equals_dilation_greedy(periodic, s):
    nx, ny, nz = 20, 17, 14
    N = nx * ny * nz
    seed, c = 9 + s, 0.02
    Tc = oracle.prob_to_threshold(c)
    cand = [v for v in range(N) if oracle.seed_draw(seed, v) < Tc]
    expect = _dilation_greedy((nz, ny, nx), periodic, cand, s)
    o = oracle.Oracle(nx, ny, nz, periodic)
    n = o.seed(c, s, seed)
    got = np.flatnonzero(o.grid().ravel())
    assert n == len(expect) and (got == np.array(expect)).all()
    # pairwise distance >= s and maximality (every rejected candidate has an accepted seed with a
    # lower index at L1 < s)
    pts = np.array([(v % nx, (v // nx) % ny, v // (nx * ny)) for v in got])
    dims = np.array([nx, ny, nz])

    def dist(a, b):
        d = np.abs(a - b)
        if periodic:
            d = np.minimum(d, dims - d)
        return d.sum(axis=-1)
    if s > 1 and len(pts) > 1:
        D = dist(pts[:, None, :], pts[None, :, :]) + np.eye(len(pts), dtype=int) * 10**6
        assert D.min() >= s
        for v in set(cand) - set(got.tolist()):
            p = np.array((v % nx, (v // nx) % ny, v // (nx * ny)))
            lower = pts[got < v]
            assert (dist(lower, p) < s).any()
    else:
        assert list(got) == cand


def test_p5_single_seed_dilation_has_closed_form_volume():
    vol = _ball_volumes()
    for s in (2, 4, 6):
        acc = _dilation_greedy((21, 21, 21), False, [10 + 21 * (10 + 21 * 10)], s)
        assert acc == [10 + 21 * (10 + 21 * 10)]
    # the blocked region of one seed is the L1 ball of radius s-1: every point at L1 < s is rejected
    o = oracle.Oracle(21, 21, 21, False)
    x, y, z = coords((21, 21, 21))
    d = np.abs(x - 10) + np.abs(y - 10) + np.abs(z - 10)
    for s in (2, 4, 6):
        assert int((d <= s - 1).sum()) == vol[s - 1]


# ------------------------------------------------------------------------------------- P6, P7
@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("dims", [(32, 32, 32), (45, 31, 38), (5, 4, 3), (1, 9, 2)])
def test_p6_list_algorithm_equals_full_field_definition(periodic, dims):
    nx, ny, nz = dims
    a, b = oracle.Oracle(nx, ny, nz, periodic), oracle.Oracle(nx, ny, nz, periodic)
    for o in (a, b):
        o.set_growth(0.05, 0.02, 0.01, 1)
        o.set_target(0.6)
        o.seed(0.01 if nx * ny * nz > 1000 else 0.2, 3, 77)
    assert (a.grid() == b.grid()).all()
    for t in range(12):
        a.step(True); b.step(False)
        assert (a.grid() == b.grid()).all(), t
        assert a.n_solid == b.n_solid == int(a.grid().sum())
        assert a.n_front_exact == b.n_front_exact
    ra, sa = a.generate(0.6, 1000, True)
    rb, sb = b.generate(0.6, 1000, False)
    assert (ra, sa) == (rb, sb) and (a.grid() == b.grid()).all()


def test_p7_front_order_does_not_matter():
    ref = None
    for how in (0, 1, 2):
        o = oracle.Oracle(36, 36, 36, False)
        o.set_growth(0.04, 0.01, 0.002, 1)
        o.set_target(0.5)
        o.seed(0.004, 4, 21)
        for t in range(10):
            if how:
                o.permute_front(how, 1000 + t)
            o.step(True)
        ref = o.grid() if ref is None else ref
        assert (o.grid() == ref).all()


# ------------------------------------------------------------------------------------------ P9
def test_p9_per_direction_acceptance_rates():
    o = oracle.Oracle(48, 48, 48, False)
    gf, ge, gc = 0.20, 0.10, 0.05
    o.set_growth(gf, ge, gc, 0)
    o.seed(0.02, 0, 5)
    for _ in range(3):
        o.step(False)
    att, suc = o.rates()
    for d in range(26):
        p = {1: gf, 2: ge, 3: gc}[oracle.direction(d)[3]]
        n, k = int(att[d]), int(suc[d])
        assert n > 3000
        assert abs(k - n * p) <= 5 * math.sqrt(n * p * (1 - p)), (d, n, k)


def test_p9_one_step_claim_probability_counts_once():
    # a void cell with m_f/m_e/m_c solid face/edge/corner neighbours is claimed with
    # probability 1 - (1-G_f)^m_f (1-G_e)^m_e (1-G_c)^m_c.  Fixed grid, many rng seeds.
    nx = ny = nz = 7
    solid = [(3, 3, 3), (4, 3, 3), (3, 4, 3), (2, 2, 4)]
    idx = [x + nx * (y + ny * z) for x, y, z in solid]
    gf, ge, gc = 0.3, 0.2, 0.1
    trials = 4000
    hits = np.zeros((nz, ny, nx))
    o = oracle.Oracle(nx, ny, nz, False)
    o.set_growth(gf, ge, gc, 0)
    for s in range(trials):
        o.seed_explicit(idx, rng_seed=1000 + s)
        o.step(s % 2 == 0)
        hits += o.grid()
    g0 = np.zeros((nz, ny, nx), bool)
    for x, y, z in solid:
        g0[z, y, x] = True
    for z, y, x in itertools.product(range(nz), range(ny), range(nx)):
        if g0[z, y, x]:
            assert hits[z, y, x] == trials
            continue
        m = {1: 0, 2: 0, 3: 0}
        for sx, sy, sz in solid:
            dd = (abs(sx - x), abs(sy - y), abs(sz - z))
            if max(dd) == 1:
                m[sum(dd)] += 1
        p = 1 - (1 - gf) ** m[1] * (1 - ge) ** m[2] * (1 - gc) ** m[3]
        k = hits[z, y, x]
        assert abs(k - trials * p) <= 5 * math.sqrt(trials * p * (1 - p)) + 1e-9, ((x, y, z), m, k)


# ------------------------------------------------------------------------------------ P10, P11
def test_p10_p11_monotone_growth_and_stop_rule():
    cfg = dict(dims=(40, 40, 40), c=0.005, s=0, g=(0.02, 0.005, 0.0005), phi=0.30, seed=1)
    o = oracle.Oracle(*cfg["dims"], False)
    o.set_growth(*cfg["g"], 1)
    o.set_target(cfg["phi"])
    o.seed(cfg["c"], cfg["s"], cfg["seed"])
    prev, prev_n, history = o.grid(), o.n_solid, []
    while o.n_solid < o.n_target:
        o.step(True)
        g = o.grid()
        assert (g >= prev).all() and o.n_solid >= prev_n and o.n_solid == int(g.sum())
        history.append(o.n_solid)
        prev, prev_n = g, o.n_solid
    steps_by_hand = len(history)
    assert history[-1] >= o.n_target and (steps_by_hand == 1 or history[-2] < o.n_target)
    # generate == repeated step, bit for bit
    o2 = oracle.Oracle(*cfg["dims"], False)
    o2.set_growth(*cfg["g"], 1)
    o2.seed(cfg["c"], cfg["s"], cfg["seed"])
    rc, steps = o2.generate(cfg["phi"], 10**6, True)
    assert rc == oracle.OK and steps == steps_by_hand and (o2.grid() == prev).all()
    # target already met: no step runs (R15)
    rc, steps = o2.generate(cfg["phi"], 10**6, True)
    assert (rc, steps) == (oracle.OK, 0)
    # resuming with a higher target continues the same stream: t keeps counting
    rc, more = o2.generate(0.5, 10**6, True)
    assert rc == oracle.OK and o2.step_index == steps_by_hand + more and o2.n_solid >= o2.n_target
    # max_steps (R14) and empty front
    o3 = oracle.Oracle(6, 6, 6, False)
    o3.set_growth(1.0, 1.0, 1.0, 0)
    o3.seed_explicit([0])
    rc, steps = o3.generate(1.0, 2, True)
    assert (rc, steps) == (oracle.MAX_STEPS, 2)
    rc, steps = o3.generate(1.0, 100, True)
    assert rc == oracle.OK and o3.n_solid == 216 and o3.n_front_exact == 0
    o4 = oracle.Oracle(6, 6, 6, False)
    o4.set_growth(0.5, 0.5, 0.5, 0)
    o4.seed(0.0, 0, 1)
    assert o4.generate(0.5, 10, True) == (oracle.FRONT_EMPTY, 0)


def test_solid_fraction_reaches_config1_target():
    # BASELINE.json configs[0]; ceil(0.30 * 64^3) = 78644
    o = oracle.Oracle(64, 64, 64, False)
    o.set_growth(0.02, 0.005, 0.0005, 1)
    n_seeds = o.seed(0.005, 0, 1)
    assert abs(n_seeds - 0.005 * 64**3) <= 5 * math.sqrt(64**3 * 0.005)
    rc, steps = o.generate(0.30, 1000, True)
    assert rc == oracle.OK and o.n_target == 78644 and o.n_solid >= 78644 and 2 <= steps <= 20


# ----------------------------------------------------------------------------------------- P12
@pytest.mark.parametrize("periodic", [False, True])
def test_p12_two_point_correlation(periodic):
    rng = np.random.default_rng(3)
    g = (rng.random((16, 14, 12)) < 0.4).astype(np.uint8)          # (nz, ny, nx)
    void = g == 0
    for axis, npax in ((0, 2), (1, 1), (2, 0)):                    # oracle axis 0 = x = numpy axis 2
        pairs, valid = oracle.s2(g, periodic, axis, 6)
        assert pairs[0] == void.sum() and valid[0] == g.size
        for r in range(7):
            if periodic:
                b = np.roll(void, -r, axis=npax)
                exp_pairs, exp_valid = int((void & b).sum()), g.size
            else:
                n = g.shape[npax]
                a = np.take(void, range(0, n - r), axis=npax)
                b = np.take(void, range(r, n), axis=npax)
                exp_pairs, exp_valid = int((a & b).sum()), a.size
            assert (int(pairs[r]), int(valid[r])) == (exp_pairs, exp_valid)
    big = (np.random.default_rng(4).random((40, 40, 40)) < 0.3).astype(np.uint8)
    pairs, valid = oracle.s2(big, True, 0, 5)
    phi = pairs[0] / valid[0]
    for r in range(1, 6):
        assert abs(pairs[r] / valid[r] - phi**2) < 0.01


@pytest.mark.parametrize("dims,periodic,core,s,seed,g,phi", [
    ((64, 64, 64), False, 0.005, 0, 1, (0.02, 0.005, 0.0005), 0.30),
    ((70, 45, 33), True, 0.004, 7, 5, (0.05, 0.02, 0.01), 0.55),
    ((5, 4, 3), True, 0.2, 2, 5, (0.3, 0.2, 0.1), 0.9),
    ((96, 96, 96), False, 0.003, 9, 3, (0.01, 0.0025, 0.00025), 0.6)])
def test_openmp_build_of_the_list_oracle_equals_the_serial_oracle(dims, periodic, core, s, seed, g, phi):
    """liboracle_omp.so (the same source with the front of oracle_step_list shared among the host's cores; the all-cores
    CPU baseline of bench.py) against liboracle.so, the checker of record: seeds, status, steps, solid count and the
    grid after EVERY step are identical, whatever order the threads append the new front in (P7)."""
    a = oracle.Oracle(*dims, periodic)
    b = oracle.Oracle(*dims, periodic, omp=True)
    assert oracle.threads(False) == 1 and oracle.threads(True) >= 1
    for o in (a, b):
        o.set_growth(*g, 1)
        o.set_target(phi)
    assert a.seed(core, s, seed) == b.seed(core, s, seed)
    while a.n_solid < a.n_target and a.n_front_exact:
        a.step(True)
        b.step(True)
        assert a.n_solid == b.n_solid and (a.grid() == b.grid()).all(), a.step_index
    ra, rb = a.generate(min(1.0, phi + 0.2)), b.generate(min(1.0, phi + 0.2))
    assert ra == rb and a.n_solid == b.n_solid and (a.grid() == b.grid()).all()


# ------------------------------------------------------------------------------------------ boundary mode 2 (R5)
def _mask(periodic):
    return {0: (False, False, False), 1: (True, True, True), 2: (True, True, False)}[int(periodic)]


def test_two_dimensional_periodic_grid_uses_the_eight_in_plane_directions():
    """PAPER.md:68 / :76: Algorithm 2 is stated for a two-dimensional grid with "roll" (periodic) shifts.  nz = 1 with
    x and y periodic between walls in z (boundary mode 2) is that grid: the 18 directions with dz != 0 have no target,
    so they are never attempted; face growth at probability 1 gives wrapped 2D diamonds of 2k^2 + 2k + 1 cells, all eight
    in-plane directions give wrapped squares of (2k + 1)^2 cells; edge only (the four diagonals) keeps parity."""
    nx, ny = 31, 27
    x, y, _ = coords((1, ny, nx))
    c = (2, 25)
    ax, ay = axis_d(x, c[0], nx, True), axis_d(y, c[1], ny, True)
    o = oracle.Oracle(nx, ny, 1, 2)
    o.set_growth(1.0, 0.0, 0.0, 0)
    o.seed_explicit([c[0] + nx * c[1]])
    for k in range(1, 12):
        o.step(False)                                   # the full-field definition (it also counts the attempts)
        assert (o.grid() == (ax + ay <= k)).all(), k
        assert o.n_solid == 2 * k * k + 2 * k + 1
    attempts, successes = o.rates()
    for d in range(26):
        dx, dy, dz, cls = oracle.direction(d)
        assert (attempts[d] > 0) == (dz == 0), d        # a void target was only ever seen in the eight in-plane directions
        assert (successes[d] > 0) == (dz == 0 and cls == 1), d   # and only the four faces could fire
    o.set_growth(1.0, 1.0, 1.0, 0)
    o.seed_explicit([c[0] + nx * c[1]])
    for k in range(1, 10):
        o.step(True)
        assert (o.grid() == (np.maximum(ax, ay) <= k)).all() and o.n_solid == (2 * k + 1) ** 2
    o.set_growth(0.0, 1.0, 0.0, 0)
    o.seed_explicit([c[0] + nx * c[1]])
    for k in range(1, 6):
        o.step(True)
    assert (o.grid() == ((ax <= 5) & (ay <= 5) & ((ax + ay) % 2 == 0))).all()
    # the same plane with walls all round (nz = 1, mode 0) clips instead of wrapping
    w = oracle.Oracle(nx, ny, 1, 0)
    w.set_growth(1.0, 0.0, 0.0, 0)
    w.seed_explicit([c[0] + nx * c[1]])
    for k in range(1, 6):
        w.step(True)
    assert (w.grid() == (np.abs(x - c[0]) + np.abs(y - c[1]) <= 5)).all()


@pytest.mark.parametrize("use_list", [True, False])
def test_slab_periodic_in_plane_walls_in_z_against_brute_force_distances(use_list):
    nx, ny, nz = 19, 13, 6
    x, y, z = coords((nz, ny, nx))
    seeds = [(0, 0, 0), (18, 12, 5), (9, 1, 3)]
    for g, metric in (((1.0, 0.0, 0.0), "l1"), ((1.0, 1.0, 1.0), "cheb")):
        o = oracle.Oracle(nx, ny, nz, 2)
        o.set_growth(*g, 0)
        o.seed_explicit([sx + nx * (sy + ny * sz) for sx, sy, sz in seeds])
        for k in range(1, 7):
            o.step(use_list)
            per = []
            for sx, sy, sz in seeds:
                dx, dy, dz = axis_d(x, sx, nx, True), axis_d(y, sy, ny, True), axis_d(z, sz, nz, False)
                per.append(dx + dy + dz if metric == "l1" else np.maximum(np.maximum(dx, dy), dz))
            assert (o.grid() == (np.min(per, axis=0) <= k)).all(), (metric, k)


@pytest.mark.parametrize("s", [2, 4, 7])
def test_spacing_with_in_plane_periodicity_equals_brute_force_greedy(s):
    """Seed spacing when only x and y wrap: the accepted set is the ascending-index greedy under the L1
    distance that wraps in x and y and not in z -- brute force over all pairs."""
    nx, ny, nz = 18, 11, 9
    N = nx * ny * nz
    seed, c = 21 + s, 0.03
    Tc = oracle.prob_to_threshold(c)
    cand = [v for v in range(N) if oracle.seed_draw(seed, v) < Tc]
    dims = np.array([nx, ny, nz])
    wrap = np.array([True, True, False])

    def dist(a, b):
        d = np.abs(np.asarray(a) - np.asarray(b))
        return int(np.where(wrap, np.minimum(d, dims - d), d).sum())
    acc = []
    for v in cand:
        p = (v % nx, (v // nx) % ny, v // (nx * ny))
        if all(dist(p, q) >= s for q in acc):
            acc.append(p)
    o = oracle.Oracle(nx, ny, nz, 2)
    assert o.seed(c, s, seed) == len(acc)
    got = np.flatnonzero(o.grid().ravel())
    assert [(v % nx, (v // nx) % ny, v // (nx * ny)) for v in got] == acc


# ------------------------------------------------------------------------------------------ earlier phases (PAPER.md:40 step 4)
def _bfs_steps(free, starts, neigh):
    """Breadth-first distance (in growth steps) from the start cells through `free` cells with the given neighbour offsets."""
    nz, ny, nx = free.shape
    dist = np.full(free.shape, -1, dtype=np.int64)
    frontier = []
    for (x, y, z) in starts:
        dist[z, y, x] = 0
        frontier.append((x, y, z))
    k = 0
    while frontier:
        k += 1
        nxt = []
        for (x, y, z) in frontier:
            for dx, dy, dz in neigh:
                X, Y, Z = x + dx, y + dy, z + dz
                if 0 <= X < nx and 0 <= Y < ny and 0 <= Z < nz and free[Z, Y, X] and dist[Z, Y, X] < 0:
                    dist[Z, Y, X] = k
                    nxt.append((X, Y, Z))
        frontier = nxt
    return dist


@pytest.mark.parametrize("use_list", [True, False])
def test_cells_of_an_earlier_phase_are_neither_void_nor_sources(use_list):
    """PAPER.md:40 step 4, independent phases: the new phase grows on the still unassigned cells.  With probability 1 the
    cells of the new phase after k steps are exactly the unassigned cells within k moves of a seed along paths that avoid
    the earlier phase (breadth-first search); the earlier phase's cells never change, are never counted, are never cores."""
    nx, ny, nz = 17, 13, 9
    rng = np.random.default_rng(5)
    taken = rng.random((nz, ny, nx)) < 0.3
    taken[:, 6, :] = True                                 # a wall with a hole: the phase has to go round
    taken[4, 6, 8] = False
    seeds = [(2, 2, 2), (15, 11, 7)]
    for s in seeds:
        taken[s[2], s[1], s[0]] = False
    faces = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    alld = [(a, b, c) for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1) if (a, b, c) != (0, 0, 0)]
    for g, neigh in (((1.0, 0.0, 0.0), faces), ((1.0, 1.0, 1.0), alld)):
        o = oracle.Oracle(nx, ny, nz, False)
        o.set_blocked(taken)
        o.set_growth(*g, 0)
        o.seed_explicit([x + nx * (y + ny * z) for x, y, z in seeds] + [8 + nx * (6 + ny * 0)])    # the last one is taken: no seed
        assert o.n_solid == 2
        dist = _bfs_steps(~taken, seeds, neigh)
        for k in range(1, 30):
            o.step(use_list)
            assert (o.grid() == ((dist >= 0) & (dist <= k))).all(), k
            assert ((o.phase_map() == 2) == taken).all() and o.n_solid == int(o.grid().sum())
        if neigh is alld:
            assert o.n_front_exact == 0                    # everything reachable is taken: no solid cell has a void neighbour left
    # keyed cores: the candidates are the unassigned cells whose draw is below the threshold
    o = oracle.Oracle(nx, ny, nz, False)
    o.set_blocked(taken)
    n = o.seed(0.05, 0, 3)
    Tc = oracle.prob_to_threshold(0.05)
    expect = [v for v in range(nx * ny * nz) if not taken.ravel()[v] and oracle.seed_draw(3, v) < Tc]
    assert n == len(expect) and (np.flatnonzero(o.grid().ravel()) == np.array(expect)).all()
    # no earlier phase at all == the plain run
    a, b = oracle.Oracle(nx, ny, nz, True), oracle.Oracle(nx, ny, nz, True)
    b.set_blocked(np.zeros((nz, ny, nx), np.uint8))
    for o in (a, b):
        o.set_growth(0.1, 0.05, 0.02, 1)
        o.seed(0.01, 3, 9)
        o.generate(0.4)
    assert (a.grid() == b.grid()).all() and a.n_solid == b.n_solid


# ------------------------------------------------------------------------- P5d, P5k (NEXT-1: R19)
@pytest.mark.parametrize("periodic", [0, 1, 2])
@pytest.mark.parametrize("s", [0, 2, 4, 7])
def test_p5d_seeding_by_literal_dilation_passes_equals_the_distance_rule(periodic, s):
    """PAPER.md:131 Fig. 1(D): diamond dilation 'with a small kernel but multiple iterations'.  The oracle's literal
    form (every accepted seed covers what s-1 passes of the 6-neighbour kernel reach, walls or wrap per axis) accepts
    exactly the seeds of the distance rule of oracle_seed."""
    nx, ny, nz = 23, 14, 9
    a = oracle.Oracle(nx, ny, nz, periodic)
    b = oracle.Oracle(nx, ny, nz, periodic)
    na, nb = a.seed(0.03, s, 21 + s), b.seed_by_dilation(0.03, s, 21 + s)
    assert na == nb and (a.grid() == b.grid()).all()
    if s > 1:
        assert na < int((np.array([oracle.seed_draw(21 + s, v) for v in range(nx * ny * nz)]) < oracle.prob_to_threshold(0.03)).sum())


def test_p5k_priority_is_a_word_of_its_own_philox_block():
    """R19: key(v) = word v % 4 of Philox4x32-10 at counter (v / 4, 0, 1, 2^32 - 1) -- the block function itself is
    pinned by the known answers (P1); the core draw sits at (v / 4, 0, 0, 2^32 - 1)."""
    for seed in (0, 7, 0x123456789ABCDEF0):
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for v in (0, 1, 2, 3, 4, 1000003, 2**32 + 5, 2**34 + 2):
            blk = v // 4
            ctr = (blk & 0xFFFFFFFF, blk >> 32, 1, 0xFFFFFFFF)
            assert oracle.seed_priority(seed, v) == oracle.philox4x32_10(ctr, key)[v % 4]
            ctr0 = (blk & 0xFFFFFFFF, blk >> 32, 0, 0xFFFFFFFF)
            assert oracle.seed_draw(seed, v) == oracle.philox4x32_10(ctr0, key)[v % 4]


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("s", [0, 1, 2, 3, 5, 8])
def test_p5k_keyed_order_equals_the_greedy_in_key_order(periodic, s):
    """The keyed acceptance order (R19): the same candidates as in index order, tried in ascending (key, index).
    Against the independent dilation greedy fed with the candidates in that order; the result keeps every pair at
    L1 >= s and is maximal: every rejected candidate has an accepted seed EARLIER in the order within L1 < s."""
    nx, ny, nz = 20, 17, 14
    N = nx * ny * nz
    seed, c = 31 + s, 0.02
    Tc = oracle.prob_to_threshold(c)
    cand = [v for v in range(N) if oracle.seed_draw(seed, v) < Tc]
    order = sorted(cand, key=lambda v: (oracle.seed_priority(seed, v), v))
    expect = sorted(_dilation_greedy((nz, ny, nx), periodic, order, s))
    o = oracle.Oracle(nx, ny, nz, periodic)
    o.set_spacing_order(1)
    n = o.seed(c, s, seed)
    got = np.flatnonzero(o.grid().ravel())
    assert n == len(expect) and (got == np.array(expect)).all()
    if s <= 1:
        assert list(got) == cand
        return
    pos = {v: k for k, v in enumerate(order)}
    pts = {v: np.array((v % nx, (v // nx) % ny, v // (nx * ny))) for v in cand}
    dims = np.array([nx, ny, nz])

    def dist(a, b):
        d = np.abs(a - b)
        if periodic:
            d = np.minimum(d, dims - d)
        return int(d.sum())
    acc = [int(v) for v in got]
    for i, v in enumerate(acc):
        for w in acc[:i]:
            assert dist(pts[v], pts[w]) >= s
    for v in set(cand) - set(acc):
        assert any(pos[w] < pos[v] and dist(pts[v], pts[w]) < s for w in acc)
    # the order matters: index order accepts another maximal set (same candidates, another permutation)
    o2 = oracle.Oracle(nx, ny, nz, periodic)
    o2.seed(c, s, seed)
    if s >= 3:
        assert (o2.grid() != o.grid()).any()
    # and growth goes on from the keyed seeds like from any others: list step == full-field step
    for q in (o, o2):
        q.set_growth(0.1, 0.05, 0.02, 0)
    a = oracle.Oracle(nx, ny, nz, periodic)
    a.set_spacing_order(1)
    a.set_growth(0.1, 0.05, 0.02, 0)
    a.seed(c, s, seed)
    o.step(use_list=True)
    a.step(use_list=False)
    assert (o.grid() == a.grid()).all()


# ------------------------------------------------------------------------------- R20: interacting phases
def _dilate26(m, periodic):
    """3x3x3 dilation of a boolean (nz, ny, nx) array: walls (nothing comes in from outside) or wrap."""
    out = m.copy()
    for dz, dy, dx in itertools.product((-1, 0, 1), repeat=3):
        r = np.roll(m, (dz, dy, dx), axis=(0, 1, 2))
        if not periodic:
            for ax, sh in ((0, dz), (1, dy), (2, dx)):
                if sh:
                    sl = [slice(None)] * 3
                    sl[ax] = 0 if sh == 1 else -1
                    r[tuple(sl)] = False
        out |= r
    return out


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("use_list", [True, False])
def test_interaction_with_probability_one_coats_the_earlier_phase(periodic, use_list):
    """PAPER.md:40 step 4, R20: with I = 1 in every direction and G = 0, one step turns exactly the unassigned cells
    that touch the earlier phase (its 3x3x3 dilation minus itself) into the new phase, and a second step adds nothing:
    the interface is covered and the new phase itself does not grow."""
    nx, ny, nz = 19, 14, 11
    rng = np.random.default_rng(5)
    m = np.zeros((nz, ny, nx), bool)
    m[3:6, 4:9, 5:12] = True
    m[8, 2, 1] = True
    m[0, 0, 0] = True                                            # a corner cell: the boundary mode shows
    o = oracle.Oracle(nx, ny, nz, periodic)
    o.set_growth(0.0, 0.0, 0.0, 0)
    o.set_blocked(m.astype(np.uint8))
    o.set_interaction(1.0, 1.0, 1.0)
    o.seed_explicit([], 3)
    o.step(use_list=use_list)
    coat = _dilate26(m, periodic) & ~m
    g = o.phase_map()
    assert ((g == 1) == coat).all() and ((g == 2) == m).all()
    assert o.n_solid == int(coat.sum())
    o.step(use_list=use_list)
    assert ((o.grid() == 1) == coat).all()
    # face probabilities only: the 6-neighbourhood
    o2 = oracle.Oracle(nx, ny, nz, periodic)
    o2.set_growth(0.0, 0.0, 0.0, 0)
    o2.set_blocked(m.astype(np.uint8))
    o2.set_interaction(1.0, 0.0, 0.0)
    o2.seed_explicit([], 3)
    o2.step(use_list=use_list)
    face = m.copy()
    for ax in range(3):
        for sh in (1, -1):
            r = np.roll(m, sh, axis=ax)
            if not periodic:
                sl = [slice(None)] * 3
                sl[ax] = 0 if sh == 1 else -1
                r[tuple(sl)] = False
            face |= r
    assert ((o2.grid() == 1) == (face & ~m)).all()


def test_interaction_zero_is_the_independent_phase_and_list_equals_full():
    nx, ny, nz = 24, 17, 13
    a = oracle.Oracle(nx, ny, nz, False)
    a.set_growth(0.2, 0.1, 0.05, 0)
    a.seed(0.01, 0, 4)
    for _ in range(3):
        a.step()
    m = (a.grid() == 1).astype(np.uint8)
    runs = []
    for inter, use_list in ((None, True), ((0.0, 0.0, 0.0), True), ((0.3, 0.1, 0.02), True), ((0.3, 0.1, 0.02), False)):
        o = oracle.Oracle(nx, ny, nz, False)
        o.set_growth(0.1, 0.05, 0.01, 1)
        o.set_blocked(m)
        if inter is not None:
            o.set_interaction(*inter)
        o.seed(0.005, 3, 8)
        rc, steps = o.generate(0.3, use_list=use_list)
        runs.append((o.grid().copy(), o.n_solid, steps))
    assert (runs[0][0] == runs[1][0]).all() and runs[0][1:] == runs[1][1:]       # I = 0: the independent phase (R18)
    assert (runs[2][0] == runs[3][0]).all() and runs[2][1:] == runs[3][1:]       # list == full field with interface sources
    assert (runs[2][0] != runs[0][0]).any()                                      # and the interface does grow
    assert not (runs[2][0] & m).any()                                            # the earlier phase keeps its cells


def test_interaction_rate_at_the_interface():
    """One step from a flat wall of the earlier phase with I_face = 0.25 and nothing else: every unassigned cell of the
    next plane has exactly one source (the wall cell below it), so the taken fraction is binomial around 0.25."""
    nx, ny, nz = 64, 64, 4
    m = np.zeros((nz, ny, nx), np.uint8)
    m[0] = 1
    o = oracle.Oracle(nx, ny, nz, False)
    o.set_growth(0.0, 0.0, 0.0, 0)
    o.set_blocked(m)
    o.set_interaction(0.25, 0.0, 0.0)
    o.seed_explicit([], 11)
    o.step()
    g = o.grid()
    assert (g[2:] == 0).all()
    k, n = int((g[1] == 1).sum()), nx * ny
    assert abs(k - 0.25 * n) < 5 * math.sqrt(n * 0.25 * 0.75)
