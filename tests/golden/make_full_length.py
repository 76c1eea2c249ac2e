"""Writes tests/golden/full_length.txt: FULL-LENGTH oracle trajectories of BASELINE.json:configs c3 and c4
(and checkpoints on the way) for a stated subset of chains.

Imports ONLY `oracle/` (the CPU oracle) and `paper_2411_18906_b200/workloads.py` (seeded input recipes, no method
arithmetic).  No value in the output comes from the CUDA path.  What is computed is the north-star variant of
PAPER.md Alg. 3 with the incremental pair-count update of Eq. 4, D8-D9, by
`ora_mc_run` with eval_all=False (the oracle's early exit at the first improving k: same trajectory and the same
n_null as eval_all=True -- pinned by tests/test_oracle_pins.py).

    python tests/golden/make_full_length.py [--jobs N] [--configs c3,c4] [--out tests/golden/full_length.txt]

Chains: c4 -> all 16 chains, 1e7 steps each (about 22 core-minutes per chain); c3 -> 16 of the 256 chains
(0, 17, 34, ..., 255), 1e6 steps each (about 70 core-seconds per chain).  Each chain runs as its own process
(chain c is independent of the batch it runs in: RNG keyed by the global chain id, D7).

One record per line, fields separated by blanks:
  config chain steps_done n_accept n_null hash last_accept_step J_bits sha256(occ) counts...
`steps_done` takes every value of CHECKPOINTS (fractions of the configured length) -- the state after a prefix is
the state of a split run (oracle pin: split-run continuation) -- so a divergence can be located.
`J_bits` is the IEEE-754 bit pattern of the fp64 objective, `counts` the S*M*M int32 pair counts, row-major.
"""
import argparse
import hashlib
import os
import sys
import time
from concurrent.futures import ProcessPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CHECKPOINTS = (0.0, 0.001, 0.01, 0.1, 0.5, 1.0)
CHAINS = {"c3": [17 * i for i in range(16)], "c4": list(range(16))}
CONFIG_ID = {"c3": 3, "c4": 4}


def run_chain(job):
    name, chain = job
    from oracle import hea_oracle as ho
    from paper_2411_18906_b200 import workloads
    w = workloads.config(CONFIG_ID[name])
    o = ho.Oracle(*w.create_args())
    occ = o.init_random(1, w.seed, chain0=chain)
    counts = np.stack([o.pair_counts(occ[0])])
    stats = ho.fresh_stats(1)
    stats["J"] = o.objective(counts[0])
    lines, done = [], 0
    for frac in CHECKPOINTS:
        upto = int(round(frac * w.n_steps))
        if upto > done:
            o.mc_run(occ, counts, upto - done, w.K, w.seed, chain0=chain, step0=done, stats=stats,
                     n_threads=1, eval_all=False)
            done = upto
        s = stats[0]
        jbits = np.array([s["J"]], dtype=np.float64).view(np.uint64)[0]
        lines.append(" ".join([name, str(chain), str(done), str(int(s["n_accept"])), str(int(s["n_null"])),
                               f"0x{int(s['hash']):016x}", str(int(s["last_accept_step"])), f"0x{int(jbits):016x}",
                               hashlib.sha256(occ[0].tobytes()).hexdigest(),
                               *[str(int(v)) for v in counts[0].ravel()]]))
    return name, chain, lines


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--jobs", type=int, default=os.cpu_count())
    ap.add_argument("--configs", default="c3,c4")
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "full_length.txt"))
    a = ap.parse_args()
    from oracle import hea_oracle as ho
    ho.build()
    jobs = [(name, c) for name in a.configs.split(",") for c in CHAINS[name]]
    t0 = time.time()
    results = {}
    with ProcessPoolExecutor(max_workers=a.jobs) as ex:
        for name, chain, lines in ex.map(run_chain, jobs):
            results[(name, chain)] = lines
            print(f"[{time.time() - t0:8.1f} s] {name} chain {chain} done", flush=True)
    with open(a.out, "w") as f:
        f.write("# Full-length ORACLE trajectories (oracle/hea_oracle.c only; written by tests/golden/make_full_length.py,\n"
                "# see its docstring for the fields).  PAPER.md Alg. 3 P:242-250 + Eq. 4 P:283-287 in the north-star variant\n"
                "# (DESIGN.md D8-D9) on BASELINE.json:configs c3 (1e6 steps, K=64) and c4 (1e7 steps, K=128).\n"
                "# config chain steps_done n_accept n_null hash last_accept_step J_bits sha256(occ) counts[S*M*M]\n")
        for name in a.configs.split(","):
            for c in CHAINS[name]:
                for ln in results[(name, c)]:
                    f.write(ln + "\n")
    print(f"wrote {a.out} in {time.time() - t0:.0f} s")


if __name__ == "__main__":
    main()
