"""Writes the expected values of the full-size parity cases (tests/golden/fullsize_hashes.jsonl).

Calls ONLY the CPU oracle (oracle/): for one BASELINE.json configuration it runs seeding + growth to
the target and records the seed count, step count, final solid count and the SHA-256 of the uint8
phase array (N bytes, x fastest).  The GPU tests compare the CUDA path's outputs with these.

    python tests/golden/make_fullsize_hashes.py cfg3_400 --target 0.80 [--seed 7] [--s 20]

Each run appends one JSON line; runs take minutes to hours of one CPU core (serial oracle).
"""
import argparse
import hashlib
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import CONFIGS  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fullsize_hashes.jsonl")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config")
    ap.add_argument("--target", type=float, required=True)
    ap.add_argument("--seed", type=int, default=None)
    ap.add_argument("--s", type=int, default=None)
    a = ap.parse_args()
    c = CONFIGS[a.config]
    seed = a.seed if a.seed is not None else c["seeds"][0]
    s = a.s if a.s is not None else (c["s"] if isinstance(c["s"], int) else c["s"][0])
    nx, ny, nz = c["dims"]
    t0 = time.time()
    o = oracle.Oracle(nx, ny, nz, c["periodic"])
    o.set_growth(*c["g"], 1)
    n_seeds = o.seed(c["core"], s, seed)
    t_seed = time.time() - t0
    rc, steps = o.generate(a.target, 10**6, True)
    h = hashlib.sha256(o.grid().tobytes()).hexdigest()
    rec = dict(config=a.config, dims=[nx, ny, nz], periodic=c["periodic"], core=c["core"], s=s, rng_seed=seed,
               g=list(c["g"]), target=a.target, n_target=o.n_target, n_seeds=n_seeds, status=rc, steps=steps,
               n_solid=o.n_solid, sha256=h, oracle_seconds=round(time.time() - t0, 1), seed_seconds=round(t_seed, 1))
    with open(OUT, "a") as f:
        f.write(json.dumps(rec) + "\n")
    print(rec)


if __name__ == "__main__":
    main()
