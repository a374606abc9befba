"""Writes the expected values of the full-size parity cases (tests/golden/fullsize_hashes.jsonl).

Calls ONLY the CPU oracle (oracle/): for one BASELINE.json configuration it runs seeding + growth to
the target and records the seed count, step count, final solid count and the SHA-256 of the uint8
phase array (N bytes, x fastest).  The GPU tests compare the CUDA path's outputs with these.

    python tests/golden/make_fullsize_hashes.py cfg3_400 --target 0.80 [--seed 7] [--s 20]
    python tests/golden/make_fullsize_hashes.py cfg5_1024 --seeds-only          # seeding + spacing only
    python tests/golden/make_fullsize_hashes.py cfg3_400 --seeds-only --order keyed   # ... in the keyed acceptance order (R19)
    python tests/golden/make_fullsize_hashes.py cfg5_1024 --target 0.80 --trace --hash-every 4

Each run appends one JSON line to fullsize_hashes.jsonl; runs take minutes to hours of one CPU core
(serial oracle).  --seeds-only records the seed count and the SHA-256 of the grid right after seeding
(kind "seeds").  --trace runs the same generation one step at a time (oracle_generate with max_steps = 1,
which is the loop of PAPER.md:140 cut after every pass) and appends to fullsize_traces.jsonl, after
EVERY step, the step index and solid count, plus the SHA-256 of the phase array every --hash-every
steps: a run that is interrupted still leaves every completed step as an expected value.  Steps that the trace file
already holds for the same run are re-computed, CHECKED against the stored values and not written again, so a run can be
repeated to extend an interrupted trace.  --omp uses liboracle_omp.so (the same oracle source compiled with -fopenmp, the
front of the list step shared among the host's cores; tests/test_oracle_pins.py proves it equal to the serial library
after every step): records made with it carry "oracle": "omp".
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
TRACE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fullsize_traces.jsonl")


def append(path, rec):
    with open(path, "a") as f:
        f.write(json.dumps(rec) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config")
    ap.add_argument("--target", type=float, default=None)
    ap.add_argument("--seeds-only", action="store_true")
    ap.add_argument("--trace", action="store_true")
    ap.add_argument("--hash-every", type=int, default=4)
    ap.add_argument("--seed", type=int, default=None)
    ap.add_argument("--s", type=int, default=None)
    ap.add_argument("--omp", action="store_true")
    ap.add_argument("--order", default="index", choices=["index", "keyed"], help="acceptance order of the spacing filter (R12 / R19)")
    a = ap.parse_args()
    c = CONFIGS[a.config]
    seed = a.seed if a.seed is not None else c["seeds"][0]
    s = a.s if a.s is not None else (c["s"] if isinstance(c["s"], int) else c["s"][0])
    nx, ny, nz = c["dims"]
    t0 = time.time()
    o = oracle.Oracle(nx, ny, nz, c["periodic"], omp=a.omp)
    o.set_growth(*c["g"], 1)
    if a.order == "keyed":
        o.set_spacing_order(1)
    n_seeds = o.seed(c["core"], s, seed)
    t_seed = time.time() - t0
    base = dict(config=a.config, dims=[nx, ny, nz], periodic=c["periodic"], core=c["core"], s=s, rng_seed=seed,
                g=list(c["g"]))
    if a.order == "keyed":
        base["order"] = "keyed"
        if not a.seeds_only:
            ap.error("--order keyed is recorded for --seeds-only runs")
    if a.seeds_only:
        h = hashlib.sha256(o.grid().tobytes()).hexdigest()
        rec = dict(base, kind="seeds", n_seeds=n_seeds, sha256=h, oracle_seconds=round(time.time() - t0, 1))
        append(OUT, rec)
        print(rec)
        return
    if a.target is None:
        ap.error("--target is required unless --seeds-only")
    if a.trace:
        have = {}
        if os.path.exists(TRACE):
            for line in open(TRACE):
                r = json.loads(line)
                if (r["config"], r["s"], r["rng_seed"], r["target"]) == (a.config, s, seed, a.target):
                    have[r["step"]] = r
        steps, rc = 0, oracle.MAX_STEPS
        while rc == oracle.MAX_STEPS:
            rc, done = o.generate(a.target, 1, True)
            steps += done
            if not done:
                break
            rec = dict(base, kind="trace", target=a.target, n_target=o.n_target, n_seeds=n_seeds, step=steps,
                       n_solid=o.n_solid, oracle_seconds=round(time.time() - t0, 1))
            if a.omp:
                rec["oracle"] = "omp"
            old = have.get(steps)
            if steps % a.hash_every == 0 or rc != oracle.MAX_STEPS or (old is not None and "sha256" in old):
                rec["sha256"] = hashlib.sha256(o.grid().tobytes()).hexdigest()
            if old is not None:                        # already recorded: check, do not write again
                assert old["n_solid"] == rec["n_solid"] and old["n_seeds"] == rec["n_seeds"], (old, rec)
                assert "sha256" not in old or old["sha256"] == rec["sha256"], (old, rec)
                print("step %d agrees with the stored record" % steps, flush=True)
                continue
            append(TRACE, rec)
            print(rec, flush=True)
    else:
        rc, steps = o.generate(a.target, 10**6, True)
    h = hashlib.sha256(o.grid().tobytes()).hexdigest()
    rec = dict(config=a.config, dims=[nx, ny, nz], periodic=c["periodic"], core=c["core"], s=s, rng_seed=seed,
               g=list(c["g"]), target=a.target, n_target=o.n_target, n_seeds=n_seeds, status=rc, steps=steps,
               n_solid=o.n_solid, sha256=h, oracle_seconds=round(time.time() - t0, 1), seed_seconds=round(t_seed, 1))
    if a.omp:
        rec["oracle"] = "omp"
    append(OUT, rec)
    print(rec)


if __name__ == "__main__":
    main()
