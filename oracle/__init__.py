"""CPU oracle for the LIETS-QSGS growth path -- TEST INFRASTRUCTURE ONLY.

ctypes binding of ``oracle/liets_oracle.c`` (plain serial C written from PAPER.md; see the header
for citations and pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2602_11734_b200`` and that package imports nothing from here.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "liets_oracle.c")
_DEPS = [_SRC, os.path.join(_HERE, "liets_oracle.h"), os.path.join(_HERE, "liets_oracle_directions.inc")]
_LIB = os.path.join(_HERE, "liboracle.so")
_LIB_OMP = os.path.join(_HERE, "liboracle_omp.so")

OK, FRONT_EMPTY, MAX_STEPS = 0, 1, 2


def build(force=False):
    """Compile liboracle.so with gcc -O2 (no SIMD intrinsics, no OpenMP: the oracle of record is serial)."""
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in _DEPS):
        return _LIB
    subprocess.check_call(["gcc", "-O2", "-std=gnu99", "-Wall", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def build_omp(force=False):
    """The same source with -fopenmp: oracle_step_list shares the front among the host's cores (the all-cores CPU
    baseline of bench.py).  The serial library stays the checker of record; tests prove the two equal."""
    if not force and os.path.exists(_LIB_OMP) and all(os.path.getmtime(_LIB_OMP) >= os.path.getmtime(d) for d in _DEPS):
        return _LIB_OMP
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=gnu99", "-Wall", "-shared", "-fPIC", "-o", _LIB_OMP, _SRC, "-lm"])
    return _LIB_OMP


_lib = None
_lib_omp = None


def lib(omp=False):
    global _lib, _lib_omp
    if omp and _lib_omp is not None:
        return _lib_omp
    if not omp and _lib is not None:
        return _lib
    L = ctypes.CDLL(build_omp() if omp else build())
    u32, u64, i64, dbl, vp, ci = (ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int64, ctypes.c_double,
                                  ctypes.c_void_p, ctypes.c_int)
    P = ctypes.POINTER
    L.oracle_philox4x32_10.argtypes = [P(u32), P(u32), P(u32)]
    L.oracle_philox4x32_10.restype = None
    L.oracle_growth_draw.argtypes = [u64, u32, u64, ci]
    L.oracle_growth_draw.restype = u32
    L.oracle_seed_draw.argtypes = [u64, u64]
    L.oracle_seed_draw.restype = u32
    L.oracle_direction.argtypes = [ci, P(ci), P(ci), P(ci), P(ci)]
    L.oracle_direction.restype = None
    L.oracle_prob_to_threshold.argtypes = [dbl]
    L.oracle_prob_to_threshold.restype = u64
    L.oracle_target_count.argtypes = [dbl, u64]
    L.oracle_target_count.restype = u64
    L.oracle_step_threshold.argtypes = [u64, ci, u64, u64]
    L.oracle_step_threshold.restype = u64
    L.oracle_new.argtypes = [ci, ci, ci, ci]
    L.oracle_new.restype = vp
    L.oracle_free.argtypes = [vp]
    L.oracle_free.restype = None
    L.oracle_set_growth.argtypes = [vp, dbl, dbl, dbl, ci]
    L.oracle_set_growth.restype = ci
    L.oracle_set_target.argtypes = [vp, dbl]
    L.oracle_set_target.restype = ci
    L.oracle_seed.argtypes = [vp, dbl, ci, u64]
    L.oracle_seed.restype = i64
    L.oracle_set_interaction.argtypes = [vp, dbl, dbl, dbl]
    L.oracle_set_interaction.restype = ci
    L.oracle_seed_by_dilation.argtypes = [vp, dbl, ci, u64]
    L.oracle_seed_by_dilation.restype = i64
    L.oracle_set_spacing_order.argtypes = [vp, ci]
    L.oracle_set_spacing_order.restype = ci
    L.oracle_seed_priority.argtypes = [u64, u64]
    L.oracle_seed_priority.restype = u32
    L.oracle_seed_explicit.argtypes = [vp, P(u64), u64, u64]
    L.oracle_seed_explicit.restype = i64
    L.oracle_step_full.argtypes = [vp]
    L.oracle_step_full.restype = ci
    L.oracle_step_list.argtypes = [vp]
    L.oracle_step_list.restype = ci
    L.oracle_generate.argtypes = [vp, dbl, u32, ci, P(u32)]
    L.oracle_generate.restype = ci
    L.oracle_grid.argtypes = [vp]
    L.oracle_grid.restype = P(ctypes.c_uint8)
    for name in ("oracle_n_solid", "oracle_n_front_exact", "oracle_n_target"):
        getattr(L, name).argtypes = [vp]
        getattr(L, name).restype = u64
    L.oracle_step_index.argtypes = [vp]
    L.oracle_step_index.restype = u32
    L.oracle_rates.argtypes = [vp, P(u64), P(u64)]
    L.oracle_rates.restype = None
    L.oracle_permute_front.argtypes = [vp, ci, u64]
    L.oracle_permute_front.restype = None
    L.oracle_s2.argtypes = [vp, ci, ci, ci, ci, ci, ci, P(u64), P(u64)]
    L.oracle_s2.restype = None
    L.oracle_set_blocked.argtypes = [vp, vp]
    L.oracle_set_blocked.restype = ci
    L.oracle_threads.argtypes = []
    L.oracle_threads.restype = ci
    if omp:
        _lib_omp = L
    else:
        _lib = L
    return L


def threads(omp=False):
    """Host threads oracle_step_list uses in the chosen library."""
    return int(lib(omp).oracle_threads())


def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*ctr)
    k = (ctypes.c_uint32 * 2)(*key)
    o = (ctypes.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def growth_draw(rng_seed, t, p, d):
    return int(lib().oracle_growth_draw(rng_seed, t, p, d))


def seed_draw(rng_seed, v):
    return int(lib().oracle_seed_draw(rng_seed, v))


def seed_priority(rng_seed, v):
    """R19: the key of voxel v in the keyed acceptance order of the spacing filter."""
    return int(lib().oracle_seed_priority(rng_seed, v))


def direction(d):
    a, b, c, k = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    lib().oracle_direction(d, a, b, c, k)
    return a.value, b.value, c.value, k.value


def prob_to_threshold(p):
    return int(lib().oracle_prob_to_threshold(p))


def target_count(phi, N):
    return int(lib().oracle_target_count(phi, N))


def step_threshold(R, law, n_t, n_solid):
    return int(lib().oracle_step_threshold(R, law, n_t, n_solid))


def s2(grid, periodic, axis, rmax):
    """grid: uint8 array of shape (nz, ny, nx); periodic: the boundary mode (0 walls, 1 torus, 2 periodic in x and y).
    Returns (pairs, valid) uint64 arrays of r = 0..rmax."""
    g = np.ascontiguousarray(grid, dtype=np.uint8)
    nz, ny, nx = g.shape
    pairs = np.zeros(rmax + 1, dtype=np.uint64)
    valid = np.zeros(rmax + 1, dtype=np.uint64)
    P64 = ctypes.POINTER(ctypes.c_uint64)
    lib().oracle_s2(g.ctypes.data, nx, ny, nz, (periodic_mask(periodic) >> axis) & 1, axis, rmax,
                    pairs.ctypes.data_as(P64), valid.ctypes.data_as(P64))
    return pairs, valid


def periodic_mask(periodic):
    """Boundary argument of the callers -> the oracle's per-axis mask: False / 0 = walls, True / 1 = torus (7),
    2 = periodic in x and y between walls in z (3)."""
    return {0: 0, 1: 7, 2: 3}[int(periodic)]


class Oracle:
    """One oracle run: create -> set_growth -> seed -> step/generate -> grid()."""

    def __init__(self, nx, ny, nz, periodic=False, omp=False):
        self._L = lib(omp)
        self.nx, self.ny, self.nz, self.periodic = nx, ny, nz, int(periodic)
        self.N = nx * ny * nz
        self._h = self._L.oracle_new(nx, ny, nz, periodic_mask(periodic))
        if not self._h:
            raise ValueError("bad dimensions")

    def close(self):
        if self._h:
            self._L.oracle_free(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def set_growth(self, g_face, g_edge, g_corner, law=1):
        if self._L.oracle_set_growth(self._h, g_face, g_edge, g_corner, law):
            raise ValueError("bad growth parameters")

    def set_target(self, phi):
        if self._L.oracle_set_target(self._h, phi):
            raise ValueError("bad target")

    def seed(self, core_prob, spacing_s, rng_seed):
        n = self._L.oracle_seed(self._h, core_prob, spacing_s, rng_seed)
        if n < 0:
            raise ValueError("bad seed parameters")
        return int(n)

    def set_interaction(self, i_face, i_edge, i_corner):
        """R20: growth of this phase at its interface with the earlier phases (set_blocked), probabilities per class."""
        if self._L.oracle_set_interaction(self._h, i_face, i_edge, i_corner) != 0:
            raise ValueError("bad interaction probabilities")

    def set_spacing_order(self, order):
        """0 = ascending index (R12), 1 = ascending (seed_priority, index) (R19); used by the next seed()."""
        if self._L.oracle_set_spacing_order(self._h, order) != 0:
            raise ValueError("bad spacing order")

    def seed_by_dilation(self, core_prob, spacing_s, rng_seed):
        """seed() with the spacing filter done by literal diamond dilation; ascending index order."""
        n = self._L.oracle_seed_by_dilation(self._h, core_prob, spacing_s, rng_seed)
        if n < 0:
            raise ValueError("bad seed parameters")
        return int(n)

    def seed_explicit(self, idx, rng_seed=0):
        a = np.ascontiguousarray(idx, dtype=np.uint64)
        n = self._L.oracle_seed_explicit(self._h, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)), a.size, rng_seed)
        if n < 0:
            raise ValueError("seed index out of range")
        return int(n)

    def step(self, use_list=True):
        rc = self._L.oracle_step_list(self._h) if use_list else self._L.oracle_step_full(self._h)
        if rc:
            raise RuntimeError("oracle step: state error %d" % rc)

    def generate(self, phi, max_steps=100000, use_list=True):
        steps = ctypes.c_uint32(0)
        rc = self._L.oracle_generate(self._h, phi, max_steps, int(use_list), steps)
        if rc < 0:
            raise RuntimeError("oracle generate: error %d" % rc)
        return rc, int(steps.value)

    def set_blocked(self, mask):
        """Cells of earlier growing phases (array of N entries, non-zero = taken; None clears). Seed again afterwards."""
        if mask is None:
            self._L.oracle_set_blocked(self._h, None)
        else:
            m = np.ascontiguousarray(np.asarray(mask).ravel() != 0, dtype=np.uint8)
            assert m.size == self.N
            self._L.oracle_set_blocked(self._h, m.ctypes.data)

    def phase_map(self):
        """uint8 copy of the raw phase array: 0 void, 1 this phase, 2 an earlier phase (set_blocked)."""
        ptr = self._L.oracle_grid(self._h)
        return np.ctypeslib.as_array(ptr, shape=(self.N,)).reshape(self.nz, self.ny, self.nx).copy()

    def grid(self):
        """uint8 copy of the phase array of THIS phase, shape (nz, ny, nx), 1 = solid."""
        return (self.phase_map() == 1).astype(np.uint8)

    @property
    def n_solid(self):
        return int(self._L.oracle_n_solid(self._h))

    @property
    def n_front_exact(self):
        return int(self._L.oracle_n_front_exact(self._h))

    @property
    def n_target(self):
        return int(self._L.oracle_n_target(self._h))

    @property
    def step_index(self):
        return int(self._L.oracle_step_index(self._h))

    def rates(self):
        a = (ctypes.c_uint64 * 26)()
        s = (ctypes.c_uint64 * 26)()
        self._L.oracle_rates(self._h, a, s)
        return np.array(a[:], dtype=np.uint64), np.array(s[:], dtype=np.uint64)

    def permute_front(self, how, key=0):
        self._L.oracle_permute_front(self._h, how, key)
