"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (never the CUDA path).

    python tests/golden/gen_golden.py            # rng_vectors.txt, neglog_vectors.txt, small_configs.json
    python tests/golden/gen_golden.py --full     # additionally full_configs.json (minutes to hours of CPU)
    python tests/golden/gen_golden.py --full-poisson   # additionally full_configs_poisson.json (sampler = 1)
    python tests/golden/gen_golden.py --full-c6 / --full-c7   # big-deme workload / habitat-loss workload
"""
import json
import os
import sys
import hashlib
import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
from oracle import oracle as O                       # noqa: E402
from paper_2108_05815_b200 import inputs as I        # noqa: E402  (input generators only)


def rng_vectors():
    rng = np.random.default_rng(20211)
    with open(os.path.join(HERE, "rng_vectors.txt"), "w") as fh:
        fh.write("# seed lane loc k j r value(hex)   -- oracle outputs, DESIGN.md 2.2 (parity vs the paper's RNG unpinned)\n")
        for lane in ("state", "time", "spec", "disp", "index", "migr"):
            for _ in range(8):
                seed = int(rng.integers(0, 1 << 63)); loc = int(rng.integers(0, 1 << 32)); k = int(rng.integers(0, 1 << 20))
                j = int(rng.integers(1, 40)); r = int(rng.integers(0, 5)) if lane == "disp" else 0
                v = O.batch_draw(seed, lane, np.array([loc], np.uint32), k, j, r=r)[0]
                fh.write("%d %s %d %d %d %d %016x\n" % (seed, lane, loc, k, j, r, int(v)))


def neglog_vectors():
    rng = np.random.default_rng(5)
    xs = [0, 1, 2, 3, (1 << 64) - 1, 1 << 63, (1 << 63) - 1, (1 << 63) + 1, 1 << 32, (1 << 32) - 1]
    xs += [int(v) for v in rng.integers(0, 1 << 64, 30, dtype=np.uint64)]
    with open(os.path.join(HERE, "neglog_vectors.txt"), "w") as fh:
        fh.write("# x(hex) neglog(x) in Q8.56 (decimal)  -- oracle outputs, DESIGN.md 2.3\n")
        for x in xs:
            fh.write("%016x %d\n" % (x, O.neglog(x)))


def result_digest(res):
    ev = res["events"]
    h = hashlib.sha256()
    for name in ("loc", "k", "j", "f", "abundance"):
        h.update(np.ascontiguousarray(ev[name]).tobytes())
    h.update(np.ascontiguousarray(ev["time"]).tobytes())
    h.update(np.ascontiguousarray(res["labels"]).tobytes())
    return h.hexdigest()


def summarise(cfg, res):
    ev = res["events"]
    return dict(name=cfg["name"], n_sampled=int(len(res["labels"])), richness=res["richness"],
                unique_events=res["stats"]["n_events"], digest=result_digest(res),
                first_events=[[int(e["loc"]), int(e["k"]), int(e["j"]), int(e["f"]), int(e["abundance"])] for e in ev[:5]],
                last_events=[[int(e["loc"]), int(e["k"]), int(e["j"]), int(e["f"]), int(e["abundance"])] for e in ev[-5:]],
                labels_head=[int(v) for v in res["labels"][:16]])


def configs(which, fname, epoch_events=0, sampler=0):
    out = []
    for cfg in which:
        sc = O.Scenario(**dict(I.scenario_kwargs(cfg), sampler=sampler))
        res = sc.simulate(cfg["seed"], cfg["nu"], cfg["mask"], dedup=True, epoch_events=epoch_events)
        out.append(summarise(cfg, res))
        print(out[-1]["name"], out[-1]["richness"], out[-1]["unique_events"], flush=True)
        with open(os.path.join(HERE, fname), "w") as fh:
            json.dump(out, fh, indent=1)


if __name__ == "__main__":
    if not any(a.startswith("--full") for a in sys.argv[1:]):
        rng_vectors()
        neglog_vectors()
        configs(I.small_configs(), "small_configs.json")
    if "--full" in sys.argv:
        configs(I.full_configs(), "full_configs.json", epoch_events=50_000_000)
    if "--full-c6" in sys.argv:           # SURVEY NEXT-4 big-deme workload at full size (about 10 minutes of CPU)
        configs([I.c6_bigdeme()], "full_config_c6.json", epoch_events=50_000_000)
    if "--full-c7" in sys.argv:           # temporally varying habitat: the C5 landscape after a habitat loss
        configs([I.c7_habitat_loss()], "full_config_c7.json", epoch_events=50_000_000)
    if "--full-poisson" in sys.argv:      # the Poisson event-time sampler on the same five configs
        configs(I.full_configs(), "full_configs_poisson.json", epoch_events=50_000_000, sampler=1)
