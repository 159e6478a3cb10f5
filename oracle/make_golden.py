"""Writes tests/golden/cfg{1,2,3,4}_tally.npz from full-size runs of the CPU ORACLE only (test infrastructure).

north_star asks that, on the same seeded inputs and the same Philox streams, the CUDA path match the oracle with
per-zone counts bit-exact and every spectral bin holding >= 1000 superphotons within 1 % and within 3 Monte Carlo
sigma.  At the full sizes of BASELINE.json the oracle takes minutes, so its result is stored once by this script
and `tests/test_gpu_full_size.py` compares the CUDA path with the stored file.  Nothing here touches the CUDA
path; no stored number comes from it.

  cfg1  scattering sphere, N_s = 1e6
  cfg2  Kerr torus 256x256, N_s = 1e7
  cfg3  3-D perturbed torus on the FULL 192x128x128 grid, N_s = 1e6 (reduced N_s: the oracle's prepare alone
        evaluates 3.1e6 zones x 201 nodes; the zone counts of the full grid are stored too)
  cfg4  torus x1e3 density, analog scattering, N_s = 1e7

Stored per config: the accumulators A = sum wE, Q = sum (wE)^2, W = sum w, n (each [n_th][n_nu]); the run counters;
the integer zone counts (int32) and the number of primaries; the parameter dictionary as JSON (the test refuses to
compare when the generator's parameters have changed); wall time and threads of the oracle run, for the record.

Run:  python oracle/make_golden.py [cfg ...]      (all four: ~25 min on 8 cores; deterministic)
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle_binding import Oracle  # noqa: E402
from paper_2602_13198_b200 import workloads as wl  # noqa: E402

GOLDEN = os.path.join(ROOT, "tests", "golden")
FULL_SIZE = {1: dict(Ns=1e6), 2: dict(Ns=1e7), 3: dict(Ns=1e6), 4: dict(Ns=1e7)}


def params_json(p: dict) -> str:
    return json.dumps({k: (list(v) if isinstance(v, (list, tuple)) else v) for k, v in sorted(p.items())})


def make(cfg: int):
    t0 = time.perf_counter()
    p, prim = wl.CONFIGS[cfg](**FULL_SIZE[cfg])
    t1 = time.perf_counter()
    o = Oracle(p, prim)
    n = o.prepare()
    t2 = time.perf_counter()
    threads = o.run()
    t3 = time.perf_counter()
    A, Q, W, cnt = o.tally()
    st = o.stats()
    Nexp, _ = o.zone_info()
    out = os.path.join(GOLDEN, f"cfg{cfg}_tally.npz")
    np.savez_compressed(out, A=A, Q=Q, W=W, n=cnt, zone_counts=o.zone_counts(), n_primaries=np.int64(n),
                        stats_keys=np.array(list(st.keys())), stats_vals=np.array([float(v) for v in st.values()]),
                        params=np.array(params_json(p)), Nexp_sum=np.float64(Nexp.sum()),
                        timing=np.array([t1 - t0, t2 - t1, t3 - t2, float(threads)]))
    print(f"cfg{cfg}: {n} primaries, {st['n_spawned']} scattered, generate {t1 - t0:.1f} s, prepare {t2 - t1:.1f} s, "
          f"run {t3 - t2:.1f} s on {threads} threads -> {out} ({os.path.getsize(out) / 1e3:.0f} kB)", flush=True)


if __name__ == "__main__":
    for c in ([int(a) for a in sys.argv[1:]] or [1, 4, 3, 2]):
        make(c)
