"""Seeded synthetic workloads: the five BASELINE.json configs as parameters.

The method is a generator, so its "inputs" are parameters and an rng seed; this module holds no
arithmetic of the method and is the only thing the CUDA path's callers and the oracle's callers
share.  Grids stand in for the paper's workloads (400^3 timing case PAPER.md:179; 200^3-1000^3
sweep :189-193; 500^3 Fontainebleau sweep :209) -- same shapes and seed-spacing structure.
"""

CONFIGS = {
    # name: dims, periodic, core probability c, spacing s, rng_seeds, G face/edge/corner, target solid fractions
    "cfg1_64": dict(dims=(64, 64, 64), periodic=False, core=0.005, s=0, seeds=(1,),
                    g=(0.02, 0.005, 0.0005), targets=(0.30,)),
    "cfg2_200": dict(dims=(200, 200, 200), periodic=False, core=0.002, s=10, seeds=(1, 2, 3, 4),
                     g=(0.01, 0.0025, 0.00025), targets=(0.75,)),
    "cfg3_400": dict(dims=(400, 400, 400), periodic=False, core=0.001, s=20, seeds=(7,),
                     g=(0.01, 0.0025, 0.00025), targets=(0.90, 0.80, 0.70)),     # porosity 0.10/0.20/0.30
    "cfg4_500": dict(dims=(500, 500, 500), periodic=False, core=0.0005, s=(10, 20, 30, 40, 50), seeds=(11,),
                     g=(0.01, 0.0025, 0.00025),
                     targets=tuple(round(1.0 - p, 2) for p in (0.08, 0.11, 0.14, 0.17, 0.20, 0.23))),
    "cfg5_1024": dict(dims=(1024, 1024, 1024), periodic=True, core=0.0002, s=30, seeds=(13,),
                      g=(0.01, 0.0025, 0.00025), targets=(0.80,)),
    # config 5 at half the linear size (same parameters, periodic): the serial oracle finishes it in about an hour,
    # the full 1024^3 run needs about ten
    "cfg5_512": dict(dims=(512, 512, 512), periodic=True, core=0.0002, s=30, seeds=(13,),
                     g=(0.01, 0.0025, 0.00025), targets=(0.80,)),
}

# the configuration BASELINE.json's metric is quoted on ("seconds per full 400^3 generation"), porosity 0.20
BENCH = dict(name="cfg3_400", dims=(400, 400, 400), periodic=False, core=0.001, s=20, seed=7,
             g=(0.01, 0.0025, 0.00025), target=0.80)
# bounded CPU-baseline sample: a 160^3 sub-volume of the same workload (same densities, same
# probabilities, same spacing, same target) -- intensive quantities match, ~15-25 s of oracle time on the GPU box host
BENCH_CPU_SAMPLE = dict(BENCH, name="cfg3_400/sample160", dims=(160, 160, 160))
