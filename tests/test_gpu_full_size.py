"""north_star's acceptance criterion at the FULL sizes of BASELINE.json, in the launch configuration bench.py times:

  "per-zone superphoton counts bit-exact, and every spectral bin holding at least 1000 superphotons within 1 %
   relative and within 3 Monte Carlo sigma"  (same seeded inputs, same Philox streams).

The oracle's full-size tallies are stored under tests/golden/ by oracle/make_golden.py (a script that calls only
oracle/); cfg 0 is small enough to run the oracle here.  cfg 3 is compared on its full 192x128x128 grid (201 MB, the
only config whose gather reaches HBM) at the reduced N_s the golden file states.

Per config the test prints (and, when gpurun_out/ exists, appends to gpurun_out/full_size.md): the number of bins
selected, the worst relative deviation, the worst deviation in sigma, the number of bins whose counts differ and by
how much (forked histories), and for the zone counts min_i |frac(N_i) - u_i| / N_i.
"""
import json
import math
import os

import numpy as np
import pytest

from paper_2602_13198_b200 import workloads as wl

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
FULL_SIZE = {1: dict(Ns=1e6), 2: dict(Ns=1e7), 3: dict(Ns=1e6), 4: dict(Ns=1e7)}
MIN_BINS = {0: 20, 1: 20, 2: 100, 3: 100, 4: 100}       # spheres >= 20 bins, 6 x 200 torus tallies >= 100


def _report(line):
    print(line)
    if os.path.isdir("gpurun_out"):
        with open(os.path.join("gpurun_out", "full_size.md"), "a") as f:
            f.write(line + "\n")


def _criterion(cfg, A_o, Q_o, n_o, A_g, n_g, min_count=1000, min_bins=None):
    """Every bin with >= min_count superphotons (oracle count): |A_g/A_o - 1| < 1 % and |A_g - A_o| < 3 sqrt(Q_o).
    nu L_nu and its sigma are A and sqrt(Q) times one common factor per theta bin, so the ratio and the sigma
    distance are those of the spectra."""
    sel = (n_o >= min_count) & (A_o > 0)
    nsel = int(sel.sum())
    rel = np.abs(A_g[sel] / A_o[sel] - 1.0)
    nsig = np.abs(A_g[sel] - A_o[sel]) / np.sqrt(Q_o[sel])
    dn = np.abs(n_g.astype(np.int64) - n_o.astype(np.int64))
    _report(f"| cfg{cfg} | {nsel} | {rel.max():.3e} | {nsig.max():.3e} | {int((dn > 0).sum())} | {int(dn.max())} | "
            f"{int(n_o.sum())} | {int(n_g.sum())} |")
    assert nsel >= (MIN_BINS[cfg] if min_bins is None else min_bins), (cfg, nsel)
    assert np.all(rel < 0.01), rel.max()
    assert np.all(nsig < 3.0), nsig.max()
    # counts per bin equal up to forked histories: a fork moves one superphoton (and its descendants) elsewhere
    assert dn.max() <= max(3, 2e-3 * n_o.max()) and dn.sum() <= max(6, 2e-4 * n_o.sum()), (dn.max(), dn.sum())
    return nsel


def _golden(cfg, p):
    path = os.path.join(GOLDEN, f"cfg{cfg}_tally.npz")
    assert os.path.exists(path), f"{path} missing: run python oracle/make_golden.py {cfg}"
    g = np.load(path)
    gp = json.loads(str(g["params"]))
    for k, v in gp.items():                                  # the generator must not have moved under the file
        if k == "abi_version":
            continue
        assert p[k] == v or (isinstance(v, list) and list(p[k]) == v), (k, p[k], v)
    return g


def _straddle_report(cfg, gm, g, counts_o):
    """counts are floor(N_i) + [u_i < frac(N_i)]; a relative perturbation delta of N_i flips zone i only
    if |frac - u_i| < delta N_i.  Print the closest call of this grid and any mismatch (never masked)."""
    counts_g = g.zone_counts()
    bad = np.nonzero(counts_g != counts_o)[0]
    Nexp = g.table(gm.TABLE_NEXP)
    _report(f"| cfg{cfg} zone counts | zones {len(counts_g)} | emitting {int((Nexp > 0).sum())} | primaries {int(counts_g.sum())} | "
            f"mismatching zones {len(bad)} |")
    assert len(bad) == 0, (bad[:10], counts_g[bad[:10]], counts_o[bad[:10]], Nexp[bad[:10]])


@pytest.fixture(scope="module")
def gm():
    from paper_2602_13198_b200 import binding
    if os.path.isdir("gpurun_out"):
        with open(os.path.join("gpurun_out", "full_size.md"), "a") as f:
            f.write("\n| config | bins with >= 1000 superphotons | worst rel. deviation | worst deviation / sigma | bins whose "
                    "count differs | largest count difference | recorded (oracle) | recorded (CUDA) |\n|---|---|---|---|---|---|---|---|\n")
    return binding


def test_config0_full_size_spectrum(gm):
    """cfg 0 at N_s = 1e5: the oracle runs here.  Its populated band holds ~1000 superphotons per bin, so
    the >= 1000 selection is complemented by the bit-exact per-bin counts of test_gpu_parity."""
    from oracle_binding import Oracle
    p, prim = wl.config0()
    o = Oracle(p, prim); o.prepare(); o.run()
    g = gm.GPUMonty(p); g.set_grid(prim); g.prepare(); g.run()
    assert np.array_equal(o.zone_counts(), g.zone_counts())
    A_o, Q_o, W_o, n_o = o.tally()
    A_g, Q_g, W_g, n_g = g.tally()
    _criterion(0, A_o, Q_o, n_o, A_g, n_g, min_count=1000, min_bins=12)   # the stated bar: 16 bins reach 1000 at this N_s
    _criterion(0, A_o, Q_o, n_o, A_g, n_g, min_count=900)                  # and the whole populated band (33 bins)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_full_size_spectrum_against_the_stored_oracle_tally(gm, cfg):
    p, prim = wl.CONFIGS[cfg](**FULL_SIZE[cfg])
    gold = _golden(cfg, p)
    g = gm.GPUMonty(p)
    if cfg == 3:
        # the stored tally is at N_s = 1e6 (382k primaries), below the size at which the automatic schedule uses the
        # hot / bounded-cold passes: force them, so that the 3.1e6-cell bound table of the full grid is exercised too
        # (cfg 2 at its 3.6e6 primaries gets them by itself)
        g.set_phase_passes(3, 4)
    g.set_grid(prim)
    n = g.prepare()
    assert n == int(gold["n_primaries"])
    _straddle_report(cfg, gm, g, gold["zone_counts"])
    g.run()
    A_g, Q_g, W_g, n_g = g.tally()
    _criterion(cfg, gold["A"], gold["Q"], gold["n"], A_g, n_g)
    # run counters against the oracle's (equal up to forks)
    so = dict(zip([str(k) for k in gold["stats_keys"]], gold["stats_vals"]))
    sg = g.stats()
    assert sg["n_primary"] == so["n_primary"]
    assert sg["n_bound_violations"] == 0          # run-time guard of the cold pass's per-cell bounds (gm_run fails otherwise)
    for k in ("n_spawned", "n_recorded", "n_steps_total", "n_horizon", "n_roulette_killed"):
        assert abs(sg[k] - so[k]) <= max(3, 2e-4 * so[k]), (k, sg[k], so[k])
    for k in ("sum_w_emit", "sum_wE_emit"):
        assert sg[k] == pytest.approx(so[k], rel=1e-10)
    for k in ("sum_w_rec", "sum_wE_rec", "sum_w_absorbed", "sum_w_spawned"):
        assert sg[k] == pytest.approx(so[k], rel=2e-3), k
