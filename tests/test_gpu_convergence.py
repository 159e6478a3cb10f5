"""Monte Carlo convergence of the CUDA path, measured through the C-ABI (Eq. 28-29; Fig. 2 and Fig. 4:
eps_err ~ N_s^-1/2).

1. cfg 0 with sub-zone emission against the ANALYTIC thin-sphere spectrum, Eq. 34, N_s = 1e4...1e8:
   this pins the CUDA path to the mathematics directly, not only to the oracle.
2. configs[4] (torus x1e3 density, analog scattering): N_s swept by decades with batched id ranges; superphotons/s per
   N_s and the convergence of Eq. 29 against a reference run, over the band where the reference is well sampled --
   the paper itself restricts the integral to the well-sampled band ("up to nu = 1e15 Hz").

Why the band of (2) is chosen by EFFECTIVE sample size: with analog scattering a superphoton keeps the Eq. 2 weight
of the frequency it was emitted at, and these weights span 20 decades over the sampled range, so a bin of the
Comptonised spectrum that holds 1e6 superphotons can owe its content to a handful of them.  For a bin with tally
(A = sum wE, Q = sum (wE)^2) the effective sample size is n_eff = A^2 / Q; its relative Monte Carlo error is
n_eff^-1/2 whatever the raw count.  Bins enter Eq. 29 when n_eff at the SMALLEST run of the fit is >= 3 (scaled from
the reference run), i.e. where the error is not yet saturated at ~1 and Eq. 29's N_s^-1/2 law can be seen at all.

Environment: GM_SWEEP_REF (default 4e9) reference N_s of (2); GM_CONV0_MAX (default 1e8).  Tables are printed and,
when gpurun_out/ exists, written to gpurun_out/convergence_cfg0.md and gpurun_out/convergence_cfg4.md.
"""
import math
import os
import time

import numpy as np
import pytest
from scipy import integrate, special

from paper_2602_13198_b200 import workloads as wl

pytestmark = pytest.mark.gpu

EE, CL, ME, HPL = 4.80320680e-10, 2.99792458e10, 9.1093826e-28, 6.6260693e-27


def _write(name, text):
    print("\n" + text)
    if os.path.isdir("gpurun_out"):
        with open(os.path.join("gpurun_out", name), "w") as f:
            f.write(text + "\n")


def _slope(ns, errs):
    return float(np.polyfit(np.log(ns), np.log(errs), 1)[0])


# ---------------------------------------------------------------------------------------------------
# 1. thin sphere against Eq. 34
# ---------------------------------------------------------------------------------------------------
def _thin_nuLnu(nu, R=1e3, ne=1e13, th=10.0, B=1.0, r_in=0.0):
    """PAPER.md Eq. 34 with the Eq. 3 emissivity typed out here: L_nu = V * angle-integrated j_nu (G29)."""
    def j(s):
        nus = (2 / 9) * EE * B / (2 * math.pi * ME * CL) * th * th * s
        X = nu / nus
        return math.sqrt(2) * math.pi * EE ** 2 * ne * nus / (3 * CL * special.kv(2, 1 / th)) * \
            (X ** 0.5 + 2 ** (11 / 12) * X ** (1 / 6)) ** 2 * math.exp(-X ** (1 / 3))
    jint = 4 * math.pi * integrate.quad(lambda t: math.sin(t) * j(math.sin(t)), 0, math.pi / 2, epsrel=1e-10)[0]
    return nu * (4 * math.pi / 3) * (R ** 3 - r_in ** 3) * jint


def test_config0_converges_to_the_analytic_thin_sphere_spectrum():
    from paper_2602_13198_b200 import binding as gm
    ns_max = float(os.environ.get("GM_CONV0_MAX", "1e8"))
    sweep = [n for n in (1e4, 1e5, 1e6, 1e7, 1e8) if n <= ns_max * 1.0001]
    nb, lo, hi = 200, 1e8, 1e24
    db = math.log(hi / lo) / nb
    nub = lo * np.exp((np.arange(nb) + 0.5) * db)
    sel = np.nonzero((nub > 4e10) & (nub < 8e11))[0]          # optically thin band: tau_a(R) < 1e-3
    p0, _ = wl.sphere(1e13, 10.0, 1.0, 1e3, 32, 16, 1e4, 1, False)
    r_in = math.exp(p0["startx"][1])
    ana = np.array([integrate.quad(lambda l: _thin_nuLnu(math.exp(l), r_in=r_in), math.log(nub[j]) - 0.5 * db,
                                   math.log(nub[j]) + 0.5 * db, epsrel=1e-8)[0] / db for j in sel])
    lines = ["| N_s | superphotons | s (gm_run) | superphotons/s | eps_err vs Eq. 34 (mean abs rel. dev.) | max abs rel. dev. | mean sigma/L from Q |",
             "|---|---|---|---|---|---|---|"]
    eps, worst = [], []
    import torch
    for Ns in sweep:
        # several seeds at small N_s: the error of one run is itself noisy
        reps = 8 if Ns <= 1e5 else (3 if Ns <= 1e6 else 1)
        e_acc, w_acc, sig_acc, tracked, secs = [], [], [], 0, 0.0
        for seed in range(1, reps + 1):
            p, prim = wl.sphere(1e13, 10.0, 1.0, 1e3, 32, 16, Ns, seed, False, nu_min=3e10, nu_max=3e12, w_min=0.0,
                                emit_mode=1)
            g = gm.GPUMonty(p)
            g.set_grid(prim)
            n = g.prepare()
            torch.cuda.synchronize(); t0 = time.perf_counter()
            g.run()
            torch.cuda.synchronize(); secs += time.perf_counter() - t0
            spec, sig, cnt = g.spectrum()
            dev = spec[0][sel] / ana - 1.0
            e_acc.append(np.mean(np.abs(dev))); w_acc.append(np.max(np.abs(dev)))
            sig_acc.append(np.mean(sig[0][sel] / np.maximum(spec[0][sel], 1e-300)))
            tracked += n
            g.close()
        eps.append(float(np.mean(e_acc))); worst.append(float(np.max(w_acc)))
        lines.append("| %g | %d | %.3f | %.3e | %.5f | %.5f | %.5f |" % (Ns, tracked // reps, secs / reps, tracked / secs, eps[-1],
                                                                         worst[-1], float(np.mean(sig_acc))))
    fit = [i for i, n in enumerate(sweep) if n <= 1e6]
    slope = _slope([sweep[i] for i in fit], [eps[i] for i in fit])
    lines.append("")
    lines.append("bins: %d (4e10-8e11 Hz); slope d ln eps_err / d ln N_s over N_s <= 1e6: %.3f (Eq. 29 / Fig. 2: -1/2). Above "
                 "1e6 the error approaches the floor set by the log-linear F(K) table (G7: up to 4e-3 at 8e11 Hz)." % (len(sel), slope))
    _write("convergence_cfg0.md", "\n".join(lines))
    assert -0.6 < slope < -0.4, slope
    assert all(eps[i + 1] < eps[i] for i in range(len(eps) - 1)), eps
    if sweep[-1] >= 1e8:
        assert worst[-1] < 0.01, worst                        # < 1 % in every bin at N_s = 1e8


# ---------------------------------------------------------------------------------------------------
# 2. scattering sphere (configs[1]): the paper's own convergence figure with scattering (Fig. 4)
# ---------------------------------------------------------------------------------------------------
def _gpu_tally(gm, make, Ns, seed):
    import torch
    p, prim = make(Ns=Ns, seed=seed)
    g = gm.GPUMonty(p)
    g.set_grid(prim)
    n = g.prepare()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    g.run()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    A, Q, W, cnt = g.tally()
    st = g.stats()
    g.close()
    return {"Ns": Ns, "primaries": n, "tracked": st["n_primary"] + st["n_spawned"], "seconds": dt,
            "A": A.sum(axis=0), "Q": Q.sum(axis=0), "cnt": cnt.sum(axis=0)}


def _neff(r):
    return np.where(r["Q"] > 0, r["A"] ** 2 / np.maximum(r["Q"], 1e-300), 0.0)


def test_config1_scattering_sphere_error_falls_as_inverse_sqrt_Ns():
    """PAPER.md:262-268, Fig. 4: with BIASED scattering (weights of the scattered superphotons kept comparable, Eq. 35)
    the integrated error of the scattering sphere falls as N_s^-1/2; the integral is carried over the well-sampled
    band only (the paper stops at 1e15 Hz; here: bins whose effective sample size A^2/Q is >= 10 in the smallest
    run of the fit, scaled from the reference run at N_s = 1e9)."""
    from paper_2602_13198_b200 import binding as gm
    ref = _gpu_tally(gm, wl.config1, 1e9, 31)
    sweep, reps = [1e5, 1e6, 1e7], {1e5: 8, 1e6: 4, 1e7: 2}
    band = _neff(ref) * (sweep[0] / ref["Ns"]) >= 10.0            # not saturated at the smallest run of the fit
    assert band.sum() >= 8, int(band.sum())
    lines = ["| N_s | runs | superphotons tracked | s (gm_run) | superphotons/s | eps_err (Eq. 29, band) | rms z |", "|---|---|---|---|---|---|---|"]
    eps = []
    for n in sweep:
        rs = [_gpu_tally(gm, wl.config1, n, s) for s in range(1, reps[n] + 1)]
        e = [np.mean(np.abs(r["A"][band] - ref["A"][band]) / ref["A"][band]) for r in rs]
        ok = [(r["Q"][band] > 0) for r in rs]
        z = [np.sqrt(np.mean((r["A"][band][m] - ref["A"][band][m]) ** 2 / (r["Q"][band][m] + ref["Q"][band][m]))) for r, m in zip(rs, ok)]
        eps.append(float(np.mean(e)))
        lines.append("| %g | %d | %d | %.3f | %.3e | %.4f | %.2f |" % (n, len(rs), rs[0]["tracked"], rs[0]["seconds"],
                                                                    rs[0]["tracked"] / rs[0]["seconds"], eps[-1], float(np.mean(z))))
    lines.append("| %g | 1 | %d | %.3f | %.3e | reference | |" % (ref["Ns"], ref["tracked"], ref["seconds"], ref["tracked"] / ref["seconds"]))
    slope = _slope(sweep, eps)
    lines.append("")
    lines.append("band: %d bins with n_eff >= 10 at N_s = 1e5 (scaled from the reference run); slope d ln eps_err / d ln N_s = %.3f (Fig. 4: -1/2)" % (int(band.sum()), slope))
    _write("convergence_cfg1.md", "\n".join(lines))
    assert -0.62 < slope < -0.38, slope


# ---------------------------------------------------------------------------------------------------
# 3. configs[4]: N_s sweep, superphotons/s, convergence
# ---------------------------------------------------------------------------------------------------
def test_config4_sweep_superphotons_per_second_and_convergence():
    """BASELINE configs[4].  The estimator of this workload is heavy-tailed: scattering is
    analog, so an up-scattered superphoton keeps the Eq. 2 weight of its emission frequency (20 decades of weights
    over the sampled range), and absorption leaves weights spread as exp(-tau), tau up to > 30.  In the ORACLE's own
    run at N_s = 1e7 (tests/golden/cfg4_tally.npz) the bins holding >= 1e4 superphotons have a median effective
    sample size n_eff = A^2/Q of 0.4 % of their count (test_oracle_tally_statistics, not gpu).  The mean error of
    Eq. 29 is then carried by a few bins that wait for their rare heavy superphotons, and approaches N_s^-1/2 only
    asymptotically; the MEDIAN over bins and runs of |delta L| (Eq. 28) is reported beside it.  What the test holds the
    path to: the error falls with N_s at a rate between the heavy-tailed and the Gaussian one, the tally's own sigma
    (from Q) predicts the size of the deviations, the oracle's largest run sits on the same curve, and on the same
    streams the two paths agree to rounding."""
    from paper_2602_13198_b200 import binding as gm
    ns_ref = float(os.environ.get("GM_SWEEP_REF", "4e9"))
    _gpu_tally(gm, wl.config4, 1e4, 1)                        # warm-up (context, allocations)
    fit_ns = [1e6, 1e7, 1e8]
    reps = {1e6: 16, 1e7: 8, 1e8: 4}
    runs = {n: [_gpu_tally(gm, wl.config4, n, s) for s in range(1, reps[n] + 1)] for n in fit_ns}
    big = _gpu_tally(gm, wl.config4, 1e9, 11)                 # BASELINE.json: N_s up to 1e9, batched id ranges
    ref = _gpu_tally(gm, wl.config4, ns_ref, 12) if ns_ref > 1e9 else big
    band = _neff(ref) * (fit_ns[0] / ref["Ns"]) >= 3.0
    nbins = int(band.sum())
    assert nbins >= 5, nbins
    lines = ["| N_s | runs | primaries | superphotons tracked | s (gm_run) | superphotons/s | eps_err (Eq. 29, band, mean) | median abs(delta L) | rms z = (A - A_ref)/sqrt(Q + Q_ref) | median n_eff in band |",
             "|---|---|---|---|---|---|---|---|---|---|"]
    eps, med, zs = [], [], []
    for n in fit_ns:
        dev = np.array([np.abs(r["A"][band] - ref["A"][band]) / ref["A"][band] for r in runs[n]])
        z = np.array([(r["A"][band] - ref["A"][band]) / np.sqrt(r["Q"][band] + ref["Q"][band]) for r in runs[n]])
        ne = np.median([np.median(_neff(r)[band]) for r in runs[n]])
        eps.append(float(dev.mean())); med.append(float(np.median(dev))); zs.append(float(np.sqrt(np.mean(z ** 2))))
        r0 = runs[n][0]
        lines.append("| %g | %d | %d | %d | %.3f | %.3e | %.4f | %.4f | %.2f | %.0f |" % (
            n, len(runs[n]), r0["primaries"], r0["tracked"], r0["seconds"], r0["tracked"] / r0["seconds"], eps[-1], med[-1], zs[-1], ne))
    for r in ([big] if ref is big else [big, ref]):
        d = np.abs(r["A"][band] - ref["A"][band]) / ref["A"][band]
        lines.append("| %g | 1 | %d | %d | %.3f | %.3e | %s | %s | | %.0f |" % (
            r["Ns"], r["primaries"], r["tracked"], r["seconds"], r["tracked"] / r["seconds"],
            "reference" if r is ref else "%.4f" % d.mean(), "" if r is ref else "%.4f" % np.median(d), float(np.median(_neff(r)[band]))))
    slope_mean, slope_med = _slope(fit_ns, eps), _slope(fit_ns, med)
    # the oracle's largest run (tests/golden/cfg4_tally.npz, N_s = 1e7, seed 1) against the same reference, and
    # against the CUDA run on the same streams
    gold = np.load(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg4_tally.npz"))
    A_o = gold["A"].sum(axis=0)
    d_o = np.abs(A_o[band] - ref["A"][band]) / ref["A"][band]
    e_same = float(np.max(np.abs(A_o[band] - runs[1e7][0]["A"][band]) / np.maximum(A_o[band], 1e-300)))
    lines.append("")
    lines.append("band: %d bins with n_eff >= 3 at N_s = 1e6 (scaled from the reference run); slope d ln / d ln N_s of the mean "
                 "eps_err %.3f, of the median %.3f (Gaussian limit -1/2; heavy-tailed estimator, see DESIGN.md 4a); oracle run "
                 "(N_s = 1e7, golden) against the same reference: mean %.4f, median %.4f; oracle vs CUDA path on the same streams "
                 "(N_s = 1e7, seed 1): max rel. dev. %.2e" % (nbins, slope_mean, slope_med, d_o.mean(), np.median(d_o), e_same))
    _write("convergence_cfg4.md", "\n".join(lines))
    assert med[0] > med[1] > med[2], med
    assert -0.65 < slope_med < -0.2, slope_med                  # measured -0.30 (profiles/r02_convergence.md)
    assert all(z < 2.5 for z in zs[1:]), zs                      # Q-based sigma predicts the deviations (<= heavy-tail factor)
    assert 0.3 * med[1] < np.median(d_o) < 3.0 * med[1], (np.median(d_o), med[1])
    assert e_same < 1e-9
