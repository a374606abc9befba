"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit."""
import numpy as np
import pytest

import oracle
from workloads import CONFIGS

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def liets():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_2602_11734_b200 as m
    m.lib()
    return m


STORAGES = [0, 1]
# 2, 3, 4 are STORAGE_TILE with the hand-over from the voxel list to the tile list forced (liets_debug_vox_list):
# 2 = tiles from the first step, 3 = a voxel list of 600 entries used for as long as it fits (the hand-over then happens
# on overflow), 4 = the voxel list for the whole run (small grids fit the allocated 2^18 entries);
# 5 is STORAGE_FULL, the full-field sweep of Algorithm 2 (no active set)
STORAGES_ALL = [0, 1, 2, 3, 4, 5]


def make(liets, dims, periodic, storage, **kw):
    L = liets.Liets(*dims, int(periodic), 2 if storage == 5 else min(storage, 1), **kw)
    if storage == 2:
        L.debug_vox_list(0)
    elif storage == 3:
        L.debug_vox_list(1 << 40, 600)
    elif storage == 4:
        L.debug_vox_list(1 << 40)
    return L


def run_both(liets, dims, periodic, core, s, seed, g, law, target, storage, max_steps=100000):
    nx, ny, nz = dims
    o = oracle.Oracle(nx, ny, nz, periodic)
    o.set_growth(*g, law)
    n_o = o.seed(core, s, seed)
    L = make(liets, dims, periodic, storage)
    L.set_growth(*g, law)
    n_g = L.seed(core, s, seed)
    assert n_g == n_o
    assert (L.grid() == o.grid()).all(), "seeds differ"
    rc_o, st_o = o.generate(target, max_steps, True)
    rc_g, st_g, ns_g = L.generate(target, max_steps)
    assert (rc_g, st_g, ns_g) == (rc_o, st_o, o.n_solid)
    assert (L.grid() == o.grid()).all(), "grids differ"
    return o, L


@pytest.mark.parametrize("storage", STORAGES_ALL)
def test_config1_bit_exact(liets, storage):
    c = CONFIGS["cfg1_64"]
    o, L = run_both(liets, c["dims"], c["periodic"], c["core"], c["s"], c["seeds"][0], c["g"], 1, c["targets"][0], storage)
    # porosity matches exactly; bits format agrees with u8
    assert int(L.grid().sum()) == o.n_solid
    bits = np.unpackbits(L.grid(liets.FORMAT_BITS), bitorder="little")[: L.N]
    assert (bits == o.grid().ravel()).all()
    assert (L.grid_device().cpu().numpy() == o.grid().ravel()).all()
    f, s, blocks = L.step_log()
    assert len(f) == o.step_index and int(s[-1]) == o.n_solid


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [False, True, 2])      # 2 = LIETS_BOUNDARY_PERIODIC_XY: x and y wrap, walls in z
@pytest.mark.parametrize("dims,core,s", [((37, 29, 41), 0.01, 4), ((70, 45, 33), 0.004, 7), ((5, 4, 3), 0.2, 2),
                                          ((1, 9, 2), 0.3, 0), ((96, 96, 96), 0.003, 9), ((17, 130, 9), 0.02, 3),
                                          ((24, 20, 28), 0.5, 8)])    # > 96 lower neighbours per candidate: the rescan path of the spacing
def test_ragged_shapes_bit_exact(liets, storage, periodic, dims, core, s):
    run_both(liets, dims, periodic, core, s, 5, (0.05, 0.02, 0.01), 1, 0.55, storage)


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("s,expect_slow", [(5, 0), (8, 1), (6, None)])
def test_spacing_ring_wrap_and_head_table(liets, periodic, s, expect_slow):
    """The single-CTA spacing resolve keeps one status byte per candidate in a shared-memory ring (2^17 ranks, plus the
    first 2^16 ranks for the periodic wrap).  No BASELINE config below 1024^3 has that many candidates, so the test
    shrinks the ring to 2048 ranks and the head to 1024 (liets_debug_spacing_ring): 8192 candidates wrap it four
    times.  s = 5: every neighbour is < 1024 ranks back -> adjacency-list path; s = 8: neighbours fall in the last 1023
    ranks below the ring size, whose slots the resolve re-arms within the same pass -> must be sent to the rescan path
    (the fit test compares against the END of the pass).  The accepted seeds equal the oracle's either way."""
    dims, core, seed = (96, 96, 48), 0.02, 21                  # 184 candidates per z-slice, about 8800 in all
    o = oracle.Oracle(*dims, periodic)
    n_o = o.seed(core, s, seed)
    L = liets.Liets(*dims, int(periodic), 1)
    L.debug_spacing_ring(2048, 1024)
    assert L.seed(core, s, seed) == n_o
    n_cand, slow = L.seed_info()
    assert n_cand > 3 * 2048
    if expect_slow is not None:
        assert slow == expect_slow
    assert (L.grid() == o.grid()).all()
    L.debug_spacing_ring(0, 0)                                  # built-in sizes: same seeds
    assert L.seed(core, s, seed) == n_o and L.seed_info()[1] == 0
    assert (L.grid() == o.grid()).all()
    L.close()


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [False, True])
def test_dense_front_bit_exact(liets, storage, periodic):
    # 55 % of the cells are seeds, nearly all of them front voxels: more than 4096 front voxels in one 128x8x8 tile,
    # i.e. several passes over the tile's shared-memory voxel list; every class fires at level 0 (large probabilities)
    run_both(liets, (130, 16, 16), periodic, 0.55, 0, 3, (0.3, 0.1, 0.02), 0, 0.97, storage)


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [False, True])
def test_step_by_step_equals_generate(liets, storage, periodic):
    dims, g = (48, 40, 52), (0.03, 0.01, 0.002)
    o = oracle.Oracle(*dims, periodic)
    o.set_growth(*g, 1); o.set_target(0.5); o.seed(0.004, 5, 9)
    A = make(liets, dims, periodic, storage)
    A.set_growth(*g, 1); A.set_target(0.5); A.seed(0.004, 5, 9)
    while o.n_solid < o.n_target:
        o.step(True)
        ns, nf = A.step()
        assert ns == o.n_solid and (nf == 0) == (o.n_front_exact == 0)
        assert (A.grid() == o.grid()).all(), o.step_index
    B = make(liets, dims, periodic, storage)
    B.set_growth(*g, 1); B.seed(0.004, 5, 9)
    rc, steps, ns = B.generate(0.5)
    assert rc == liets.OK and steps == o.step_index and (B.grid() == A.grid()).all()
    # resume with a higher target continues the same stream (P11)
    rc_o, more_o = o.generate(0.7, 10**6, True)
    rc, more, ns = B.generate(0.7)
    assert (rc, more, ns) == (rc_o, more_o, o.n_solid) and (B.grid() == o.grid()).all()
    # target already met: zero steps (R15)
    assert B.generate(0.7)[:2] == (liets.OK, 0)


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [False, True])
def test_closed_forms_on_gpu(liets, storage, periodic):
    nx, ny, nz = 23, 19, 21
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")

    def ad(a, b, n):
        d = np.abs(a - b)
        return np.minimum(d, n - d) if periodic else d
    seeds = [(0, 0, 0), (22, 18, 20), (11, 9, 10)]
    idx = [sx + nx * (sy + ny * sz) for sx, sy, sz in seeds]
    L = make(liets, (nx, ny, nz), periodic, storage)
    L.set_growth(1.0, 0.0, 0.0, liets.LAW_CONSTANT)          # faces only, p = 1: union of L1 balls (P3)
    L.seed_explicit(idx + idx[:1])
    for k in range(1, 6):
        L.step()
        d = np.min([ad(x, sx, nx) + ad(y, sy, ny) + ad(z, sz, nz) for sx, sy, sz in seeds], axis=0)
        assert (L.grid() == (d <= k)).all()
    L.set_growth(1.0, 1.0, 1.0, liets.LAW_CONSTANT)          # all 26, p = 1: Chebyshev cubes (P4)
    L.seed_explicit(idx)
    for k in range(1, 5):
        L.step()
        d = np.min([np.maximum(np.maximum(ad(x, sx, nx), ad(y, sy, ny)), ad(z, sz, nz)) for sx, sy, sz in seeds], axis=0)
        assert (L.grid() == (d <= k)).all()
    L.set_growth(0.0, 0.0, 0.0, liets.LAW_CONSTANT)          # all G = 0: exactly the seeds (P2)
    L.seed(0.01, 0, 3)
    g0 = L.grid()
    rc, steps, ns = L.generate(0.5, 6)
    assert (rc, steps) == (liets.MAX_STEPS, 6) and (L.grid() == g0).all() and ns == g0.sum()


@pytest.mark.parametrize("storage", STORAGES_ALL)
def test_degenerate_cases(liets, storage):
    L = make(liets, (6, 6, 6), 0, storage)
    L.set_growth(0.5, 0.5, 0.5, liets.LAW_CONSTANT)
    assert L.seed(0.0, 0, 1) == 0                             # no seeds: empty front
    assert L.generate(0.5, 10)[:2] == (liets.FRONT_EMPTY, 0)
    L.set_growth(1.0, 1.0, 1.0, liets.LAW_CONSTANT)
    L.seed_explicit([0])
    assert L.generate(1.0, 2)[:2] == (liets.MAX_STEPS, 2)
    rc, steps, ns = L.generate(1.0, 100)
    assert rc == liets.OK and ns == 216
    assert L.step() == (216, 0)                               # full grid: front is empty
    assert L.seed(1.0, 0, 1) == 216                           # every voxel a core
    M = make(liets, (12, 12, 12), 1, storage)
    assert M.seed(1.0, 3, 1) == oracle_seed_count(12, True, 1.0, 3, 1)
    with pytest.raises(liets.LietsError):
        liets.Liets(0, 4, 4)
    N = make(liets, (4, 4, 4), 0, storage)
    with pytest.raises(liets.LietsError):
        N.step()                                              # before seed
    with pytest.raises(liets.LietsError):
        N.set_growth(1.5, 0, 0)
    N.seed(0.5, 0, 1)
    with pytest.raises(liets.LietsError):
        N.step()                                              # Eq. (1) without target


def oracle_seed_count(n, periodic, core, s, seed):
    o = oracle.Oracle(n, n, n, periodic)
    return o.seed(core, s, seed)


@pytest.mark.parametrize("storage", STORAGES)
@pytest.mark.parametrize("seed", CONFIGS["cfg2_200"]["seeds"][:2])
def test_config2_bit_exact(liets, storage, seed):
    c = CONFIGS["cfg2_200"]
    o, L = run_both(liets, c["dims"], c["periodic"], c["core"], c["s"], seed, c["g"], 1, c["targets"][0], storage)
    # two-point correlation of the GPU grid, computed with the oracle, equals that of the oracle grid
    for axis in range(3):
        pg, vg = oracle.s2(L.grid(), False, axis, 16)
        po, vo = oracle.s2(o.grid(), False, axis, 16)
        assert (pg == po).all() and (vg == vo).all()
        assert pg[0] == L.N - o.n_solid
        pd, vd = L.s2(axis, 40)                        # the device's own pair counts (liets_s2)
        po, vo = oracle.s2(o.grid(), False, axis, 40)
        assert (pd == po).all() and (vd == vo).all()


def test_boundary_library_workspace_stream_and_capacity_errors(liets):
    """The C ABI directly: library-owned workspace (NULL), a non-default stream, device-side output, and the
    capacity errors of liets_create / liets_grid."""
    import ctypes
    import torch
    L = liets.lib()
    dims = (40, 24, 33)
    N = dims[0] * dims[1] * dims[2]
    o = oracle.Oracle(*dims, True)
    o.set_growth(0.04, 0.01, 0.002, 1)
    n_o = o.seed(0.01, 4, 21)
    rc_o, st_o = o.generate(0.4, 10**6, True)
    stream = torch.cuda.Stream()
    for storage in STORAGES:
        h = ctypes.c_void_p()
        need = L.liets_workspace_bytes(*dims, storage)
        small = torch.empty(1024, dtype=torch.uint8, device="cuda")
        assert L.liets_create(ctypes.byref(h), *dims, 1, storage, ctypes.c_void_p(small.data_ptr()), 1024,
                              ctypes.c_void_p(stream.cuda_stream)) == liets.E_CAPACITY and need > 1024
        assert L.liets_create(ctypes.byref(h), *dims, 1, storage, None, 0, ctypes.c_void_p(stream.cuda_stream)) == liets.OK
        assert L.liets_set_growth(h, 0.04, 0.01, 0.002, liets.LAW_EQ1) == liets.OK
        n = ctypes.c_uint64(0)
        assert L.liets_seed(h, 0.01, 4, 21, ctypes.byref(n)) == liets.OK and n.value == n_o
        steps, ns = ctypes.c_uint32(0), ctypes.c_uint64(0)
        assert L.liets_generate(h, 0.4, 10**6, ctypes.byref(steps), ctypes.byref(ns)) == rc_o
        assert (steps.value, ns.value) == (st_o, o.n_solid)
        out = torch.empty(N, dtype=torch.uint8, device="cuda")
        assert L.liets_grid(h, ctypes.c_void_p(out.data_ptr()), N - 1, liets.FORMAT_U8, 1) == liets.E_CAPACITY
        assert L.liets_grid(h, ctypes.c_void_p(out.data_ptr()), N, liets.FORMAT_U8, 1) == liets.OK
        stream.synchronize()
        assert (out.cpu().numpy() == o.grid().ravel()).all()
        bits = torch.empty((N + 7) // 8, dtype=torch.uint8, device="cuda")
        assert L.liets_grid(h, ctypes.c_void_p(bits.data_ptr()), (N + 7) // 8, liets.FORMAT_BITS, 1) == liets.OK
        stream.synchronize()
        assert (np.unpackbits(bits.cpu().numpy(), bitorder="little")[:N] == o.grid().ravel()).all()
        assert L.liets_launch_count(h) > 0
        L.liets_destroy(h)


@pytest.mark.parametrize("storage", STORAGES)
def test_concurrent_contexts_on_streams_bit_exact(liets, storage):
    """Independent realisations as contexts on separate CUDA streams, driven from host threads at the same time
    (replicas: SURVEY 8(e) / NEXT-2): each must equal its own oracle run, whatever the interleaving on the GPU."""
    import threading
    import torch
    dims, core, s, g, phi = (72, 56, 64), 0.004, 6, (0.03, 0.01, 0.002), 0.6
    seeds = [11, 12, 13, 14]
    gens, out = [], {}
    for _ in seeds:
        L = liets.Liets(*dims, 0, storage, stream=torch.cuda.Stream())
        L.set_growth(*g, liets.LAW_EQ1)
        gens.append(L)

    def run(L, seed):
        n = L.seed(core, s, seed)
        rc, steps, ns = L.generate(phi)
        out[seed] = (n, rc, steps, ns, L.grid())
    for rep in range(2):                                          # second round: graphs already built, keys refreshed
        th = [threading.Thread(target=run, args=(L, seed + 100 * rep)) for L, seed in zip(gens, seeds)]
        [t.start() for t in th]
        [t.join() for t in th]
        for seed in seeds:
            o = oracle.Oracle(*dims, False)
            o.set_growth(*g, 1)
            n_o = o.seed(core, s, seed + 100 * rep)
            rc_o, st_o = o.generate(phi, 10**6, True)
            n, rc, steps, ns, grid = out[seed + 100 * rep]
            assert (n, rc, steps, ns) == (n_o, rc_o, st_o, o.n_solid)
            assert (grid == o.grid()).all()


def _fuzz_cases(n, seed=2024):
    rng = np.random.default_rng(seed)
    cases = []
    for k in range(n):
        dims = tuple(int(v) for v in rng.choice([1, 2, 3, 7, 8, 9, 15, 16, 17, 31, 33, 63, 64, 65, 70, 129, 140], 3))
        if dims[0] * dims[1] * dims[2] > 300000:
            dims = (dims[0], min(dims[1], 33), min(dims[2], 33))
        cases.append(dict(dims=dims, periodic=int(rng.integers(0, 3)), core=float(rng.choice([0.002, 0.01, 0.05, 0.3])),
                          s=int(rng.choice([0, 1, 2, 3, 5, 9])), seed=int(rng.integers(0, 2**40)),
                          g=tuple(float(v) for v in rng.choice([0.0, 0.003, 0.02, 0.07, 0.2, 0.6, 1.0], 3)),
                          law=int(rng.integers(0, 2)), target=float(rng.choice([0.2, 0.5, 0.9, 1.0])), storage=k % 6))
    return cases


@pytest.mark.parametrize("case", _fuzz_cases(100), ids=lambda c: "%dx%dx%d-%s-s%d-st%d" % (*c["dims"], "per" if c["periodic"] else "wall", c["s"], c["storage"]))
def test_random_parameters_bit_exact(liets, case):
    """Seeded random shapes (1- and 2-cell axes, word and tile boundaries), boundaries, densities, spacings, probabilities
    (0, tiny, above 1/16, 1), laws, targets and 40-bit rng seeds; at most 60 steps each."""
    run_both(liets, case["dims"], case["periodic"], case["core"], case["s"], case["seed"], case["g"], case["law"],
             case["target"], case["storage"], max_steps=60)


def test_oracle_philox_equals_curand_device_philox(liets, tmp_path):
    """Pin P1 on the GPU box: the oracle's Philox4x32-10 against NVIDIA's own device implementation
    (curand_Philox4x32_10 from curand_philox4x32_x.h, compiled here with nvcc) on 2000 random (counter, key) vectors."""
    import os
    import shutil
    import subprocess
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    src = os.path.join(os.path.dirname(__file__), "curand_philox_check.cu")
    exe = str(tmp_path / "curand_philox_check")
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src])
    rng = np.random.default_rng(7)
    vec = rng.integers(0, 2**32, size=(2000, 6), dtype=np.uint64)
    vec[0] = 0
    vec[1] = 2**32 - 1
    text = "\n".join(" ".join("%x" % int(x) for x in row) for row in vec) + "\n"
    out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout.split("\n")
    for row, line in zip(vec, out):
        expect = oracle.philox4x32_10([int(x) for x in row[:4]], [int(x) for x in row[4:]])
        assert tuple(int(t, 16) for t in line.split()) == expect


def test_eq1_thresholds_on_device_against_big_integers(liets):
    """Row 1 of the path (Eq. (1) in counts, R6/R8) directly: the device function the control step uses
    (q, r split, no 128-bit product) against Python big integers, including the extremes n_t = 1 and n_t = 2^32 - 1,
    R = 2^32, n_solid = 0 / n_t - 1 / n_t / beyond 20/19 n_t, and random triples."""
    rng = np.random.default_rng(7)
    big = 1 << 32
    R, n_t, n_s = [], [], []
    for nt in (1, 2, 3, 19, 20, 21, 1000, 6_000_000, 51_200_000, 858_993_460, big - 2, big - 1, big):
        for r in (0, 1, 2, 1 << 16, 42_949_673, 1_073_742, (1 << 31) + 12345, big - 1, big):
            for ns in (0, 1, nt // 2, max(nt - 1, 0), nt, min(nt + 1, big), min(20 * nt // 19, big), min(20 * nt // 19 + 1, big), big):
                R.append(r); n_t.append(nt); n_s.append(ns)
    for _ in range(4000):
        nt = int(rng.integers(1, big + 1))
        R.append(int(rng.integers(0, big + 1))); n_t.append(nt); n_s.append(int(rng.integers(0, min(2 * nt, big) + 1)))
    got = liets.liets.debug_thresholds(R, n_t, n_s)
    for r, nt, ns, T in zip(R, n_t, n_s, got):
        expect = min(big, r * max(0, 20 * nt - 19 * ns) // nt)
        assert T == expect, (r, nt, ns, T, expect)
        assert T == oracle.step_threshold(r, 1, nt, ns)


@pytest.mark.parametrize("storage", STORAGES)
@pytest.mark.parametrize("periodic", [False, True, 2])
@pytest.mark.parametrize("dims", [(70, 45, 33), (130, 9, 17), (5, 4, 3), (1, 9, 2), (64, 64, 8), (191, 3, 2)])
def test_device_two_point_correlation_equals_oracle(liets, storage, periodic, dims):
    """liets_s2 (exact void-void pair counts on the device, R16) against the oracle's plain triple loop, every axis, lags
    beyond the grid size included, on shapes whose rows end inside a word and on axes of 1, 2 and 3 cells."""
    o, L = run_both(liets, dims, periodic, 0.02, 2, 11, (0.08, 0.03, 0.01), 1, 0.45, storage)
    for axis in range(3):
        rmax = 2 * max(dims) + 3
        pd, vd = L.s2(axis, rmax)
        po, vo = oracle.s2(o.grid(), periodic, axis, rmax)
        assert (vd == vo).all(), (axis, vd, vo)
        assert (pd == po).all(), (axis, np.flatnonzero(pd != po)[:5])
        assert pd[0] == L.N - o.n_solid


def _batch_against_singles(liets, name, seeds, spacing=None):
    """n realisations of one BASELINE.json config in ONE batched loop: every grid equals its own oracle run (stored hash
    or live oracle) and its own liets_generate."""
    import hashlib
    import json
    import os
    c = CONFIGS[name]
    s = spacing if spacing is not None else (c["s"] if isinstance(c["s"], int) else c["s"][0])
    gold = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "fullsize_hashes.jsonl")
    for l in open(path):
        r = json.loads(l)
        if r["config"] == name and r.get("kind") is None and r["s"] == s and r["target"] == c["targets"][0]:
            gold[r["rng_seed"]] = r
    B = liets.LietsBatch(len(seeds), *c["dims"], int(c["periodic"]))
    n_seeds = []
    for i, seed in enumerate(seeds):
        B[i].set_growth(*c["g"], liets.LAW_EQ1)
        n_seeds.append(B[i].seed(c["core"], s, seed))
    res = B.generate(c["targets"][0])
    for i, seed in enumerate(seeds):
        rc, steps, n_solid = res[i]
        g = B[i].grid()
        if seed in gold:
            r = gold[seed]
            assert (n_seeds[i], rc, steps, n_solid) == (r["n_seeds"], r["status"], r["steps"], r["n_solid"])
            assert hashlib.sha256(g.tobytes()).hexdigest() == r["sha256"], seed
        else:
            o = oracle.Oracle(*c["dims"], c["periodic"])
            o.set_growth(*c["g"], 1)
            assert o.seed(c["core"], s, seed) == n_seeds[i]
            rc_o, st_o = o.generate(c["targets"][0])
            assert (rc, steps, n_solid) == (rc_o, st_o, o.n_solid) and (g == o.grid()).all(), seed
        f, sol, blocks = B[i].step_log()
        assert len(sol) == steps and int(sol[-1]) == n_solid
    # a second batched run after re-seeding half of the grids (the graph's keys are refreshed), and resuming the others
    for i in range(0, len(seeds), 2):
        B[i].seed(c["core"], s, seeds[i] + 100)
    res2 = B.generate(min(1.0, c["targets"][0] + 0.05))
    L = liets.Liets(*c["dims"], int(c["periodic"]), 1)
    L.set_growth(*c["g"], liets.LAW_EQ1)
    for i in (0, 1):
        L.seed(c["core"], s, seeds[i] + (100 if i % 2 == 0 else 0))
        if i % 2:
            L.generate(c["targets"][0])
        rc, steps, n_solid = L.generate(min(1.0, c["targets"][0] + 0.05))
        assert (rc, n_solid) == (res2[i][0], res2[i][2]) and (L.grid() == B[i].grid()).all()
    B.close()


def test_batched_generate_config1_eight_realisations(liets):
    _batch_against_singles(liets, "cfg1_64", [1, 2, 3, 4, 5, 6, 7, 8])


def test_batched_generate_config2_seeds_1_to_4(liets):
    _batch_against_singles(liets, "cfg2_200", [1, 2, 3, 4])


def test_batch_argument_errors(liets):
    with pytest.raises(liets.LietsError):
        liets.LietsBatch(17, 8, 8, 8)
    B = liets.LietsBatch(2, 8, 8, 8)
    B[0].set_growth(0.1, 0.1, 0.1, 0)
    B[0].seed(0.1, 0, 1)
    with pytest.raises(liets.LietsError):                 # grid 1 is not seeded
        B.generate(0.5)
    B[1].set_growth(0.1, 0.1, 0.1, 0)
    B[1].seed(0.0, 0, 1)                                   # no seeds at all: FRONT_EMPTY at once
    res = B.generate([0.5, 0.5])
    assert res[1][0] == liets.FRONT_EMPTY and res[1][1] == 0 and res[0][0] == liets.OK
    B.close()


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [0, 2])
@pytest.mark.parametrize("dims", [(150, 97, 1), (64, 200, 1), (9, 1, 1)])
def test_two_dimensional_grids_bit_exact(liets, storage, periodic, dims):
    """Two-dimensional grids (Algorithms 1-3 are stated in 2D): nz = 1 between walls (mode 0) or periodic in
    the plane (mode 2, the "roll" of :76), seeding with spacing and growth to the target against the oracle."""
    run_both(liets, dims, periodic, 0.01, 5, 4, (0.08, 0.03, 0.01), 1, 0.6, storage)


@pytest.mark.parametrize("storage", STORAGES_ALL)
@pytest.mark.parametrize("periodic", [False, True])
def test_two_growing_phases_bit_exact(liets, storage, periodic):
    """Multi-phase growth, independent phases (PAPER.md:40 step 4): phase 1 is generated, its cells are handed to a second
    generator (liets_set_blocked: uint8 from the host, packed bits from the device), phase 2 grows on the unassigned cells with
    its own core and growth probabilities.  Seeds, every step's solid count and the final grid equal the oracle's; no cell
    belongs to both phases; re-seeding keeps the mask, clearing it restores the plain run."""
    import torch
    dims = (70, 45, 33)
    nx, ny, nz = dims
    o1, L1 = run_both(liets, dims, periodic, 0.004, 6, 3, (0.05, 0.02, 0.01), 1, 0.35, storage)
    p1 = o1.grid()
    o2 = oracle.Oracle(nx, ny, nz, periodic)
    o2.set_blocked(p1)
    o2.set_growth(0.08, 0.01, 0.0, 1)
    n2 = o2.seed(0.01, 4, 17)
    rc_o, st_o = o2.generate(0.30)
    for how in ("host_u8", "device_bits"):
        L2 = make(liets, dims, periodic, storage)
        L2.set_growth(0.08, 0.01, 0.0, 1)
        if how == "host_u8":
            L2.set_blocked(L1.grid())
        else:
            L2.set_blocked(L1.grid_device(liets.FORMAT_BITS), liets.FORMAT_BITS)
        with pytest.raises(liets.LietsError):
            L2.step()                                      # not seeded since the mask changed
        assert L2.seed(0.01, 4, 17) == n2
        rc, st, ns = L2.generate(0.30)
        assert (rc, ns) == (rc_o, o2.n_solid) and st in (st_o, st_o + (1 if rc == liets.FRONT_EMPTY else 0))
        g2 = L2.grid()
        assert (g2 == o2.grid()).all() and not (g2 & p1).any()
        bits = np.unpackbits(L2.grid(liets.FORMAT_BITS), bitorder="little")[: L2.N]
        assert (bits == o2.grid().ravel()).all()
        f, sol, blocks = L2.step_log()
        assert int(sol[min(st_o, len(sol)) - 1]) == o2.n_solid
        # free cells of the two-phase map, by the device's two-point correlation at lag 0
        pairs, valid = L2.s2(0, 3)
        assert pairs[0] == L2.N - int(p1.sum()) - ns
        L2.close()
    L3 = make(liets, dims, periodic, storage)
    L3.set_growth(0.05, 0.02, 0.01, 1)
    L3.set_blocked(p1)
    L3.set_blocked(None)                                   # cleared: the plain phase-1 run again
    L3.seed(0.004, 6, 3)
    L3.generate(0.35)
    assert (L3.grid() == p1).all()


def test_second_phases_in_a_batch_equal_single_runs(liets):
    """liets_set_blocked on the generators of a batch: two second phases (different earlier phases, different seeds) in one
    batched loop equal their single runs."""
    dims = (64, 40, 24)
    firsts = []
    for seed in (3, 4):
        L = liets.Liets(*dims, 0, 1)
        L.set_growth(0.05, 0.02, 0.01, 1)
        L.seed(0.005, 5, seed)
        L.generate(0.3)
        firsts.append(L.grid())
    singles = []
    for i, p1 in enumerate(firsts):
        L = liets.Liets(*dims, 0, 1)
        L.set_growth(0.06, 0.01, 0.002, 1)
        L.set_blocked(p1)
        n = L.seed(0.01, 3, 20 + i)
        singles.append((n, L.generate(0.25), L.grid()))
    B = liets.LietsBatch(2, *dims, 0)
    for i, p1 in enumerate(firsts):
        B[i].set_growth(0.06, 0.01, 0.002, 1)
        B[i].set_blocked(p1)
        assert B[i].seed(0.01, 3, 20 + i) == singles[i][0]
    res = B.generate(0.25)
    for i in range(2):
        rc, st, ns = singles[i][1]
        assert (res[i][0], res[i][2]) == (rc, ns) and (B[i].grid() == singles[i][2]).all()
        assert not (B[i].grid() & firsts[i]).any()
    B.close()
