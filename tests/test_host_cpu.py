"""CPU-side checks (no GPU): the C-ABI library loads and exports what include/liets.h declares, the
host-only entry points behave, and the multi-rank reduction of bench.py works over gloo."""
import ctypes
import os
import re
import socket

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def liets():
    from paper_2602_11734_b200 import build
    build.build()
    import paper_2602_11734_b200 as m
    return m


def test_library_exports_every_declared_symbol(liets):
    header = open(os.path.join(ROOT, "include", "liets.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(liets_[a-z0-9_]+)\s*\(", header))
    assert declared == set(liets.EXPORTS), declared ^ set(liets.EXPORTS)
    L = liets.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_sass_is_sm100a_only(liets):
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", liets.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, out


def test_workspace_bytes_host_logic(liets):
    L = liets.lib()
    assert L.liets_workspace_bytes(0, 4, 4, 0) == 0
    assert L.liets_workspace_bytes(4, 4, 4, 7) == 0
    assert L.liets_workspace_bytes(2048, 2048, 2048, 1) == 0          # N >= 2^32
    for storage in (0, 1):
        a = L.liets_workspace_bytes(64, 64, 64, storage)
        b = L.liets_workspace_bytes(128, 128, 128, storage)
        assert 0 < a < b and a % 256 == 0
    # tile storage keeps the grid at about 2 x N/8 bytes: far below the uint8 layout's grid + two voxel lists
    n = 400 ** 3
    assert L.liets_workspace_bytes(400, 400, 400, 0) > 9 * n
    assert L.liets_workspace_bytes(400, 400, 400, 1) < 5.4 * n       # 4 N seeding scratch + bit grids, lists, 2 voxel lists of N/16 entries, 2 planes of earlier-phase cells


def test_bad_arguments_fail_before_touching_the_device(liets):
    L = liets.lib()
    h = ctypes.c_void_p()
    assert L.liets_create(ctypes.byref(h), 0, 4, 4, 0, 0, None, 0, None) == liets.liets.E_ARG
    assert L.liets_create(ctypes.byref(h), 4, 4, 4, 5, 0, None, 0, None) == liets.liets.E_ARG
    assert L.liets_create(None, 4, 4, 4, 0, 0, None, 0, None) == liets.liets.E_ARG
    assert L.liets_set_growth(None, 0.1, 0.1, 0.1, 1) == liets.liets.E_ARG
    assert L.liets_launch_count(None) == 0
    assert L.liets_last_error(None) == b"null ctx"


def test_no_cpu_fallback(liets):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = ctypes.c_void_p()
    assert liets.lib().liets_create(ctypes.byref(h), 8, 8, 8, 0, 0, None, 0, None) == liets.liets.E_CUDA
    with pytest.raises(liets.LietsError):
        liets.Liets(8, 8, 8)


def test_product_does_not_import_the_oracle():
    uses_oracle = re.compile(r"^\s*(import\s+oracle|from\s+oracle|#\s*include.*oracle|.*CDLL.*oracle)", re.M)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2602_11734_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not uses_oracle.search(open(os.path.join(dirpath, f)).read()), os.path.join(dirpath, f)
    uses_product = re.compile(r"^\s*(import\s+paper_2602|from\s+paper_2602|#\s*include.*(liets\.h|liets_device|liets_host))", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h", ".inc")):
            assert not uses_product.search(open(os.path.join(ROOT, "oracle", f)).read()), f


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    t_dev, t_e2e = bench.max_over_ranks([10.0 + rank, 20.0 - rank], dist, "cpu")
    q.put((rank, t_dev, t_e2e, bench.whole_job_throughput(1000, world, 4, t_dev)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t_dev, t_e2e, value in got:
        assert (t_dev, t_e2e) == (11.0, 20.0)                      # max over the two ranks
        assert value == pytest.approx(1000 * 2 * 4 / 11.0e-3)      # whole-job aggregate, not per GPU


def test_algorithmic_bytes_model():
    import bench
    # STORAGE_U8: 4|A_t| + min(27|A_t|, N) + c_t + 4|A_{t+1}|
    b = bench.algorithmic_bytes(0, 1000, [10, 30], [25, 60], 10)
    assert b == [4 * 10 + 270 + 15 + 4 * 30, 4 * 30 + 810 + 35 + 4 * 30]
    b = bench.algorithmic_bytes(0, 100, [10], [25], 10)
    assert b == [40 + 100 + 15 + 40]
    # STORAGE_TILE: 4|L_t| + min(1625|L_t|, N/8) + 1024|L_t| + 4|L_{t+1}|
    assert bench.algorithmic_bytes(1, 10**6, [2, 3], [0, 0], 0)[0] == 8 + 3250 + 2048 + 12
    assert bench.algorithmic_bytes(1, 8000, [2, 3], [0, 0], 0)[0] == 8 + 1000 + 2048 + 12
    # STORAGE_TILE with the first step on the voxel list of the bit grid: 4|A_t| + min(27|A_t|, N)/8 + 2 words per claim + 4|L_{t+1}|
    b = bench.algorithmic_bytes(1, 10**6, [10, 3], [25, 60], 10, on_tiles=[False, True], front_voxels=[10, 999])
    assert b == [40 + 270 // 8 + 16 * 15 + 12, 12 + 3 * 1625 + 3 * 1024 + 12]
