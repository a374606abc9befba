"""ctypes binding of libliets.so -- same names as include/liets.h, argument marshalling only."""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libliets.so")

OK, FRONT_EMPTY, MAX_STEPS = 0, 1, 2
E_ARG, E_STATE, E_CAPACITY, E_CUDA = -1, -2, -3, -4
BOUNDARY_WALL, BOUNDARY_PERIODIC, BOUNDARY_PERIODIC_XY = 0, 1, 2
STORAGE_U8, STORAGE_TILE, STORAGE_FULL = 0, 1, 2
LAW_CONSTANT, LAW_EQ1 = 0, 1
FORMAT_U8, FORMAT_BITS = 0, 1
S2_STATIC_MAX_LAGS = 4096
ORDER_INDEX, ORDER_KEYED = 0, 1
SPACING_SPARSE, SPACING_DENSE = 0, 1

# every symbol include/liets.h declares
EXPORTS = ("liets_workspace_bytes", "liets_create", "liets_set_growth", "liets_seed", "liets_seed_explicit",
           "liets_set_target", "liets_set_blocked", "liets_set_interaction", "liets_step", "liets_generate", "liets_grid", "liets_s2", "liets_s2_static", "liets_step_log", "liets_timings",
           "liets_set_profiling", "liets_step_times", "liets_launch_count", "liets_seed_info", "liets_set_spacing", "liets_spacing_rounds",
           "liets_create_batch", "liets_batch_ctx", "liets_generate_batch", "liets_destroy_batch",
           "liets_batch_last_error", "liets_debug_spacing_ring", "liets_debug_vox_list", "liets_debug_thresholds", "liets_probe", "liets_destroy", "liets_last_error")
PROBE_PHILOX, PROBE_LOP3, PROBE_IMAD, PROBE_MIX, PROBE_L2_READ, PROBE_HBM_READ = range(6)


class LietsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("liets error %d: %s" % (code, msg))
        self.code = code


_lib = None


def library_path():
    return _LIB_PATH


def lib():
    """Load libliets.so (built by ``python -m paper_2602_11734_b200.build``). No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("libliets.so is not built: run `python -m paper_2602_11734_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIB_PATH)
    vp, ci, dbl, u32, u64, sz = (ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_uint32,
                                 ctypes.c_uint64, ctypes.c_size_t)
    P = ctypes.POINTER
    L.liets_workspace_bytes.argtypes = [ci, ci, ci, ci]
    L.liets_workspace_bytes.restype = sz
    L.liets_create.argtypes = [P(vp), ci, ci, ci, ci, ci, vp, sz, vp]
    L.liets_create.restype = ci
    L.liets_set_growth.argtypes = [vp, dbl, dbl, dbl, ci]
    L.liets_set_growth.restype = ci
    L.liets_seed.argtypes = [vp, dbl, ci, u64, P(u64)]
    L.liets_seed.restype = ci
    L.liets_seed_explicit.argtypes = [vp, P(u64), u64, u64]
    L.liets_seed_explicit.restype = ci
    L.liets_set_blocked.argtypes = [vp, vp, sz, ci, ci]
    L.liets_set_blocked.restype = ci
    L.liets_set_target.argtypes = [vp, dbl]
    L.liets_set_target.restype = ci
    L.liets_step.argtypes = [vp, P(u64), P(u64)]
    L.liets_step.restype = ci
    L.liets_generate.argtypes = [vp, dbl, u32, P(u32), P(u64)]
    L.liets_generate.restype = ci
    L.liets_grid.argtypes = [vp, vp, sz, ci, ci]
    L.liets_grid.restype = ci
    L.liets_s2.argtypes = [vp, ci, ci, P(u64), P(u64)]
    L.liets_s2.restype = ci
    L.liets_set_interaction.argtypes = [vp, dbl, dbl, dbl]
    L.liets_set_interaction.restype = ci
    L.liets_set_spacing.argtypes = [vp, ci, ci]
    L.liets_set_spacing.restype = ci
    L.liets_spacing_rounds.argtypes = [vp, P(u32)]
    L.liets_spacing_rounds.restype = ci
    L.liets_s2_static.argtypes = [vp, ci, ci, P(u64), P(u64)]
    L.liets_s2_static.restype = ci
    L.liets_step_log.argtypes = [vp, P(u64), P(u64), P(u64), P(u64), u32]
    L.liets_step_log.restype = ci
    L.liets_timings.argtypes = [vp, P(ctypes.c_float), P(ctypes.c_float)]
    L.liets_timings.restype = ci
    L.liets_set_profiling.argtypes = [vp, ci]
    L.liets_set_profiling.restype = ci
    L.liets_step_times.argtypes = [vp, P(ctypes.c_float), u32]
    L.liets_step_times.restype = ci
    L.liets_launch_count.argtypes = [vp]
    L.liets_launch_count.restype = u64
    L.liets_seed_info.argtypes = [vp, P(u32), P(u32)]
    L.liets_seed_info.restype = ci
    L.liets_debug_spacing_ring.argtypes = [vp, u32, u32]
    L.liets_debug_spacing_ring.restype = ci
    L.liets_debug_vox_list.argtypes = [vp, u64, u32]
    L.liets_debug_vox_list.restype = ci
    L.liets_debug_thresholds.argtypes = [P(u64), P(u64), P(u64), P(u64), u32]
    L.liets_debug_thresholds.restype = ci
    L.liets_create_batch.argtypes = [P(vp), ci, ci, ci, ci, ci, vp, sz, vp]
    L.liets_create_batch.restype = ci
    L.liets_batch_ctx.argtypes = [vp, ci]
    L.liets_batch_ctx.restype = vp
    L.liets_generate_batch.argtypes = [vp, P(dbl), u32, P(ci), P(u32), P(u64), P(ctypes.c_float)]
    L.liets_generate_batch.restype = ci
    L.liets_destroy_batch.argtypes = [vp]
    L.liets_destroy_batch.restype = None
    L.liets_batch_last_error.argtypes = [vp]
    L.liets_batch_last_error.restype = ctypes.c_char_p
    L.liets_probe.argtypes = [ci, vp, sz, vp, ci, P(dbl), P(dbl)]
    L.liets_probe.restype = ci
    L.liets_destroy.argtypes = [vp]
    L.liets_destroy.restype = None
    L.liets_last_error.argtypes = [vp]
    L.liets_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


def probe(kind, scratch, reps=5, stream=None):
    """liets_probe on a torch uint8 CUDA tensor `scratch`: (units per second, milliseconds of the best launch)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream(scratch.device)
    ups, ms = ctypes.c_double(0), ctypes.c_double(0)
    rc = lib().liets_probe(kind, ctypes.c_void_p(scratch.data_ptr()), scratch.numel(), ctypes.c_void_p(st.cuda_stream),
                           reps, ctypes.byref(ups), ctypes.byref(ms))
    if rc < 0:
        raise LietsError(rc, "liets_probe failed")
    return float(ups.value), float(ms.value)


def debug_thresholds(R, n_t, n_solid):
    """liets_debug_thresholds on equally long sequences of Python ints: the device's T values as a list of ints."""
    n = len(R)
    arr = [np.ascontiguousarray(a, dtype=np.uint64) for a in (R, n_t, n_solid)]
    out = np.zeros(n, dtype=np.uint64)
    P64 = ctypes.POINTER(ctypes.c_uint64)
    rc = lib().liets_debug_thresholds(arr[0].ctypes.data_as(P64), arr[1].ctypes.data_as(P64), arr[2].ctypes.data_as(P64),
                                          out.ctypes.data_as(P64), n)
    if rc < 0:
        raise LietsError(rc, "liets_debug_thresholds failed")
    return [int(v) for v in out]


class Liets:
    """One generator context.  Mirrors the C ABI: create -> set_growth -> seed -> step / generate -> grid."""

    def __init__(self, nx, ny, nz, boundary=BOUNDARY_WALL, storage=STORAGE_U8, device="cuda:0", stream=None):
        import torch  # device memory and streams only
        self._L = lib()
        self._torch = torch
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.N = self.nx * self.ny * self.nz
        self.boundary, self.storage = int(boundary), int(storage)
        if not torch.cuda.is_available():
            raise LietsError(E_CUDA, "no CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nbytes = self._L.liets_workspace_bytes(self.nx, self.ny, self.nz, self.storage)
        if nbytes == 0:
            raise LietsError(E_ARG, "bad grid dimensions or storage")
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = ctypes.c_void_p()
        rc = self._L.liets_create(ctypes.byref(h), self.nx, self.ny, self.nz, self.boundary, self.storage,
                                  ctypes.c_void_p(base), nbytes, ctypes.c_void_p(self._stream.cuda_stream))
        if rc < 0:
            raise LietsError(rc, "liets_create failed")
        self._h = h

    @classmethod
    def _borrowed(cls, owner, handle, nx, ny, nz, boundary, device):
        """A view of a generator owned by a LietsBatch (never destroyed from here)."""
        import torch
        self = cls.__new__(cls)
        self._L, self._torch, self._owner = lib(), torch, owner
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz
        self.boundary, self.storage, self.device = boundary, STORAGE_TILE, device
        self._ws, self._stream = None, None
        self._h = ctypes.c_void_p(handle)
        self._is_borrowed = True
        return self

    def close(self):
        if getattr(self, "_h", None):
            if not getattr(self, "_is_borrowed", False):
                self._L.liets_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        self.close()

    def _check(self, rc):
        if rc < 0:
            raise LietsError(rc, self._L.liets_last_error(self._h).decode())
        return rc

    def set_growth(self, g_face, g_edge, g_corner, law=LAW_EQ1):
        self._check(self._L.liets_set_growth(self._h, g_face, g_edge, g_corner, law))

    def seed(self, core_prob, spacing_s, rng_seed):
        n = ctypes.c_uint64(0)
        self._check(self._L.liets_seed(self._h, core_prob, spacing_s, rng_seed, ctypes.byref(n)))
        return int(n.value)

    def set_interaction(self, i_face, i_edge, i_corner):
        """Growth at the interface with the earlier phases (set_blocked) with probabilities I per class; seed again afterwards."""
        self._check(self._L.liets_set_interaction(self._h, i_face, i_edge, i_corner))

    def set_spacing(self, order=ORDER_INDEX, method=SPACING_SPARSE):
        """Variant of the spacing filter used by the next seed(): acceptance order and sparse / dense mechanism."""
        self._check(self._L.liets_set_spacing(self._h, order, method))

    def spacing_rounds(self):
        r = ctypes.c_uint32(0)
        self._check(self._L.liets_spacing_rounds(self._h, ctypes.byref(r)))
        return int(r.value)

    def seed_explicit(self, idx, rng_seed=0):
        a = np.ascontiguousarray(idx, dtype=np.uint64)
        self._check(self._L.liets_seed_explicit(self._h, a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)),
                                                a.size, rng_seed))

    def set_blocked(self, mask, format=FORMAT_U8):
        """Cells of earlier growing phases: a numpy array (host) or a torch CUDA uint8 tensor, N bytes (FORMAT_U8, non-zero =
        taken) or ceil(N/8) packed bytes (FORMAT_BITS); None clears.  Seed again afterwards."""
        if mask is None:
            self._check(self._L.liets_set_blocked(self._h, None, 0, format, 0))
            return
        if hasattr(mask, "data_ptr"):                       # torch tensor on the device
            self._check(self._L.liets_set_blocked(self._h, ctypes.c_void_p(mask.data_ptr()), mask.numel(), format, 1))
        else:
            a = np.ascontiguousarray(np.asarray(mask).ravel(), dtype=np.uint8)
            self._check(self._L.liets_set_blocked(self._h, a.ctypes.data, a.size, format, 0))

    def set_target(self, phi):
        self._check(self._L.liets_set_target(self._h, phi))

    def step(self):
        ns, nf = ctypes.c_uint64(0), ctypes.c_uint64(0)
        self._check(self._L.liets_step(self._h, ctypes.byref(ns), ctypes.byref(nf)))
        return int(ns.value), int(nf.value)

    def generate(self, phi, max_steps=100000):
        steps, ns = ctypes.c_uint32(0), ctypes.c_uint64(0)
        rc = self._check(self._L.liets_generate(self._h, phi, max_steps, ctypes.byref(steps), ctypes.byref(ns)))
        return rc, int(steps.value), int(ns.value)

    def grid(self, format=FORMAT_U8):
        """Phase array on the host: uint8 (nz, ny, nx) for FORMAT_U8, flat packed bytes for FORMAT_BITS."""
        n = self.N if format == FORMAT_U8 else (self.N + 7) // 8
        out = np.empty(n, dtype=np.uint8)
        self._check(self._L.liets_grid(self._h, out.ctypes.data, n, format, 0))
        return out.reshape(self.nz, self.ny, self.nx) if format == FORMAT_U8 else out

    def grid_into(self, host_ptr, nbytes, format=FORMAT_U8):
        """Copy the phase array into a caller-owned HOST buffer (e.g. pinned memory)."""
        self._check(self._L.liets_grid(self._h, ctypes.c_void_p(host_ptr), nbytes, format, 0))

    def grid_device(self, format=FORMAT_U8):
        n = self.N if format == FORMAT_U8 else (self.N + 7) // 8
        out = self._torch.empty(n, dtype=self._torch.uint8, device=self.device)
        self._check(self._L.liets_grid(self._h, ctypes.c_void_p(out.data_ptr()), n, format, 1))
        return out

    def s2(self, axis, rmax):
        """Exact void-void pair counts at lags 0..rmax along `axis` (0 = x, 1 = y, 2 = z): (pairs, valid) uint64 arrays."""
        pairs = np.zeros(rmax + 1, dtype=np.uint64)
        valid = np.zeros(rmax + 1, dtype=np.uint64)
        P64 = ctypes.POINTER(ctypes.c_uint64)
        self._check(self._L.liets_s2(self._h, axis, rmax, pairs.ctypes.data_as(P64), valid.ctypes.data_as(P64)))
        return pairs, valid

    def s2_static(self, axis, rmax):
        """s2() through liets_s2_static: no cudaMalloc in the call, counters in a static device array (rmax < S2_STATIC_MAX_LAGS)."""
        pairs = np.zeros(rmax + 1, dtype=np.uint64)
        valid = np.zeros(rmax + 1, dtype=np.uint64)
        P64 = ctypes.POINTER(ctypes.c_uint64)
        self._check(self._L.liets_s2_static(self._h, axis, rmax, pairs.ctypes.data_as(P64), valid.ctypes.data_as(P64)))
        return pairs, valid

    def step_log(self, cap=4096):
        f = np.zeros(cap, dtype=np.uint64)
        s = np.zeros(cap, dtype=np.uint64)
        b = np.zeros(cap, dtype=np.uint64)
        v = np.zeros(cap, dtype=np.uint64)
        P64 = ctypes.POINTER(ctypes.c_uint64)
        n = self._check(self._L.liets_step_log(self._h, f.ctypes.data_as(P64), s.ctypes.data_as(P64),
                                               b.ctypes.data_as(P64), v.ctypes.data_as(P64), cap))
        self.front_voxels = v[:n].copy()      # front voxels with a void target per step
        self.step_on_tiles = (f[:n] >> np.uint64(63)).astype(bool)        # the step ran in the tile kernel
        self.step_handover = ((f[:n] >> np.uint64(62)) & np.uint64(1)).astype(bool)   # ... and its count is still in voxels
        return (f[:n] & np.uint64((1 << 62) - 1)).copy(), s[:n].copy(), b[:n].copy()

    def timings(self):
        a, b = ctypes.c_float(0), ctypes.c_float(0)
        self._check(self._L.liets_timings(self._h, ctypes.byref(a), ctypes.byref(b)))
        return float(a.value), float(b.value)

    def set_profiling(self, on):
        self._check(self._L.liets_set_profiling(self._h, int(on)))

    def step_times(self, cap=4096):
        ms = (ctypes.c_float * cap)()
        n = self._check(self._L.liets_step_times(self._h, ms, cap))
        return np.array(ms[:n], dtype=np.float64)

    def seed_info(self):
        """(keyed candidates before spacing, 1 if the spacing took the rescan slow path)."""
        n, slow = ctypes.c_uint32(0), ctypes.c_uint32(0)
        self._check(self._L.liets_seed_info(self._h, ctypes.byref(n), ctypes.byref(slow)))
        return int(n.value), int(slow.value)

    def debug_spacing_ring(self, ring, head):
        self._check(self._L.liets_debug_spacing_ring(self._h, ring, head))

    def debug_vox_list(self, max_front_voxels=None, capacity=0):
        """max_front_voxels: None = the default, 0 = tiles from the first step; capacity: 0 = as allocated."""
        v = 0xFFFFFFFFFFFFFFFF if max_front_voxels is None else int(max_front_voxels)
        self._check(self._L.liets_debug_vox_list(self._h, v, int(capacity)))

    @property
    def launch_count(self):
        return int(self._L.liets_launch_count(self._h))


class LietsBatch:
    """n equally shaped STORAGE_TILE generators whose step loops run as one device-side loop (liets_create_batch).
    batch[i] is the i-th generator: set_growth / seed / grid / s2 / step_log as usual; generate() runs them all."""

    def __init__(self, n, nx, ny, nz, boundary=BOUNDARY_WALL, device="cuda:0", stream=None):
        import torch
        self._L = lib()
        if not torch.cuda.is_available():
            raise LietsError(E_CUDA, "no CUDA device (there is no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        each = self._L.liets_workspace_bytes(int(nx), int(ny), int(nz), STORAGE_TILE)
        if each == 0 or n < 1:
            raise LietsError(E_ARG, "bad batch size, grid dimensions")
        self._ws = torch.empty(each * n + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = ctypes.c_void_p()
        rc = self._L.liets_create_batch(ctypes.byref(h), n, int(nx), int(ny), int(nz), int(boundary), ctypes.c_void_p(base), each * n,
                                        ctypes.c_void_p(self._stream.cuda_stream))
        if rc < 0:
            raise LietsError(rc, "liets_create_batch failed")
        self._h, self.n = h, n
        self._items = [Liets._borrowed(self, self._L.liets_batch_ctx(h, i), int(nx), int(ny), int(nz), int(boundary), self.device)
                       for i in range(n)]

    def __getitem__(self, i):
        return self._items[i]

    def __len__(self):
        return self.n

    def generate(self, targets, max_steps=100000):
        """targets: one solid fraction per grid (or one for all). Returns [(status, steps, n_solid)] and sets .device_ms."""
        t = [float(targets)] * self.n if np.isscalar(targets) else [float(v) for v in targets]
        arr = (ctypes.c_double * self.n)(*t)
        st, steps, ns = (ctypes.c_int * self.n)(), (ctypes.c_uint32 * self.n)(), (ctypes.c_uint64 * self.n)()
        ms = ctypes.c_float(0)
        rc = self._L.liets_generate_batch(self._h, arr, max_steps, st, steps, ns, ctypes.byref(ms))
        if rc < 0:
            raise LietsError(rc, self._L.liets_batch_last_error(self._h).decode())
        self.device_ms = float(ms.value)
        return [(int(st[i]), int(steps[i]), int(ns[i])) for i in range(self.n)]

    def close(self):
        if getattr(self, "_h", None):
            for it in self._items:
                it._h = None
            self._L.liets_destroy_batch(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        self.close()
