"""Writes tests/golden/config{3,4,5}_*.json: the ORACLE's result for BASELINE.json configs 3-5 (Orszag-Tang
2044^2 x 200, 4000^2 x 100, 8000^2 x 50 steps, CFL 0.3, periodic, HD on, RK4; PAPER.md:83-95 are these grids)
at their configured step counts, so that the driver-run `-m gpu` suite can compare the CUDA path with them
without re-running the oracle (which needs 10-70 minutes per config on 8-16 cores).

Imports only `oracle/` and `smaug_inputs.py` (never the CUDA path).  Parity is bitwise by contract (DESIGN.md
section 4), so what is stored per checkpoint is a SHA-256 of every field's bytes (float64, C order, interior
[ny, nx]) plus (t, last_dt) and the four reduced maxima as hex floats, and at the final checkpoint the values of
1000 seeded sample cells per field as hex floats (compared to 1e-10 relative as well, so that a hash mismatch
can be told apart from a gross error).

    python tests/golden/make_config_goldens.py [--threads 8] [3 4 5]

The oracle's row-parallel loops are result-neutral (no sum reductions), so the thread count does not change
a bit; `--check N` re-runs an N^2 grid with 1 and `--threads` threads and asserts equal hashes.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                     # noqa: E402
import smaug_inputs as si         # noqa: E402

CONFIGS = {                      # BASELINE.json config number -> (n, checkpoints; the last one is the configured count)
    3: (2044, (1, 50, 100, 200)),
    4: (4000, (1, 25, 50, 100)),
    5: (8000, (1, 10, 25, 50)),
}
CFL = 0.3
N_SAMPLES = 1000
SAMPLE_SEED = 1710


def sample_cells(n: int):
    rng = np.random.default_rng(SAMPLE_SEED + n)
    return rng.integers(0, n, size=N_SAMPLES), rng.integers(0, n, size=N_SAMPLES)     # (j, i)


def field_hashes(w: np.ndarray):
    return [hashlib.sha256(np.ascontiguousarray(w[f]).tobytes()).hexdigest() for f in range(w.shape[0])]


def run(n: int, checkpoints, threads: int, log=print):
    w, bc, gamma = si.orszag_tang(n)
    o = oracle.Oracle(n, n, gamma, bc, threads=threads)
    o.set_state(w)
    out, done, t0 = [], 0, time.time()
    for c in checkpoints:
        o.step(c - done, CFL)
        done = c
        s = o.get_state()
        t, dt = o.time()
        out.append(dict(steps=c, t=float(t).hex(), last_dt=float(dt).hex(),
                        wavespeeds=[float(x).hex() for x in o.wavespeeds()], sha256=field_hashes(s)))
        log(f"  n={n} steps={c} t={t:.12e} ({time.time() - t0:.0f} s)")
    jj, ii = sample_cells(n)
    samples = [[float(x).hex() for x in s[f, jj, ii]] for f in range(6)]
    o.close()
    return out, samples


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("configs", nargs="*", type=int, default=[3, 4, 5])
    ap.add_argument("--threads", type=int, default=8)
    ap.add_argument("--check", type=int, default=0, help="thread-neutrality self check on an N^2 grid, writes nothing")
    a = ap.parse_args()
    oracle.build()
    if a.check:
        r1, _ = run(a.check, (1, 3), 1)
        rt, _ = run(a.check, (1, 3), a.threads)
        assert r1 == rt, "oracle result depends on the thread count"
        print("thread-neutral: ok")
        return
    for c in a.configs:
        n, cps = CONFIGS[c]
        print(f"config {c}: Orszag-Tang {n}^2, checkpoints {cps}, {a.threads} threads", flush=True)
        cps_out, samples = run(n, cps, a.threads, log=lambda s: print(s, flush=True))
        doc = dict(
            cite="BASELINE.json config %d (PAPER.md:83-95 Table 1 grid %d x %d); Orszag-Tang IC of smaug_inputs.orszag_tang, "
                 "periodic, gamma=5/3, CFL 0.3, HD on (defaults), RK4; written by tests/golden/make_config_goldens.py "
                 "from oracle/ only" % (c, n, n),
            config=c, nx=n, ny=n, cfl=CFL, fields=list(si.FIELDS), checkpoints=cps_out,
            sample_seed=SAMPLE_SEED + n, n_samples=N_SAMPLES, samples_at_final=samples)
        path = os.path.join(HERE, f"config{c}_ot{n}.json")
        with open(path, "w") as f:
            json.dump(doc, f, indent=0)
            f.write("\n")
        print("wrote", path, flush=True)


if __name__ == "__main__":
    main()
