"""The parity norm of DESIGN.md reading P20, written once for all GPU tests.

Literal "1e-10 relative per sample" is not attainable in double for samples whose terms cancel
(kappa = S/|value| up to 1e18), whichever implementation computes them, so the bar is:
  (1) every sample:        |gpu - truth| <= 1e-10 * S + FLOOR,  S = sum_t |term_t| from the quad oracle
                           (for kappa ~ 1 this IS the plain relative error);
  (2) kappa <= 1e3 subset: |gpu - truth| <= 1e-10 * |truth| + FLOOR;
  (3) batch mean:          |mean_gpu - mean_truth| <= 1e-10 * mean(S)  and, when the mean itself is
                           well conditioned (mean(S)/|mean| <= 1e3), plain relative <= 1e-10;
  (4) non-finite truth values must be non-finite on the GPU too.
FLOOR = 1e-280 is an absolute allowance tied to the output format, applied to EVERY sample alike (no sample
is exempted from any rule).  The result is complex128 (BASELINE.json: "complex128 output per sample"), whose
normal range ends at 2.2e-308, and the kernels' Fermi/Bose leaves are built with integer exponent arithmetic that
SATURATES at 2^-1021 = 4.5e-308 instead of underflowing (reading P12: no overflow for any beta), so a term whose
true value is 1e-400 can come out as 4.5e-308 times its remaining factors -- reciprocals of denominators down to
1e-8 (the regulator), beta^k of a derivative -- i.e. up to ~1e-280, where the truth reads 0 as a double.  It only
matters where every term underflows (beta |E| of several hundred, test_extreme_temperatures).
kappa is formed from log2 S and log2 |truth| taken in quad precision before the cast to double
(oracle `want_logs`), so samples whose S underflows a double are still classified.
`min_wellcond`: floor on the share of kappa <= 1e3 samples.  S is the denominator of rule (1); an
inflated S would show up as a collapse of that share (S itself is pinned in tests/test_oracle_pins.py).
"""
import numpy as np

TOL = 1e-10
FLOOR = 1e-280

# share of samples with kappa <= 1e3 measured with the quad oracle at the configurations' own parameters
# (cfg1 0.82; cfg2 over its (mu, beta) points 0.73-0.97 / 0.85-0.99 / 0.87-0.99; cfg3 0.45; cfg4 0.28; cfg5 0.41-0.63
# over its four temperatures), less a margin for small batches
WELLCOND_FLOOR = {"cfg1": 0.72, "cfg2_se": 0.65, "cfg2_bubble": 0.75, "cfg2_bubble_doubled": 0.78, "cfg3": 0.38,
                  "cfg4": 0.20, "cfg5": 0.33}


def check_parity(gpu, truth, S, tol=TOL, label="", log2S=None, log2abs=None, min_wellcond=None):
    gpu, truth, S = np.asarray(gpu), np.asarray(truth), np.asarray(S)
    assert gpu.shape == truth.shape == S.shape, (gpu.shape, truth.shape, S.shape)
    fin = np.isfinite(truth.real) & np.isfinite(truth.imag) & np.isfinite(S)
    bad_gpu = ~(np.isfinite(gpu.real) & np.isfinite(gpu.imag))
    assert not (bad_gpu & fin).any(), f"{label}: GPU non-finite where the oracle is finite"
    assert bad_gpu[~fin].all(), f"{label}: oracle non-finite but GPU finite"
    g, t, s = gpu[fin], truth[fin], S[fin]
    err = np.abs(g - t)
    excess = np.maximum(err - FLOOR, 0.0)            # rule (1): err <= tol * S + FLOOR
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(excess > 0.0, excess / s, 0.0)
    worst_S = float(np.max(ratio)) if err.size else 0.0
    assert worst_S <= tol, f"{label}: worst S-relative error {worst_S:.3e}"
    if log2S is not None and log2abs is not None:
        with np.errstate(invalid="ignore", over="ignore"):
            kappa = np.exp2(np.clip(np.asarray(log2S)[fin] - np.asarray(log2abs)[fin], -1000.0, 1000.0))
        kappa = np.where(np.isnan(kappa), 1.0, kappa)          # exact zeros on both sides
    else:
        kappa = s / np.maximum(np.abs(t), 1e-300)
    well = kappa <= 1e3
    rel_excess = np.maximum(err[well] - FLOOR, 0.0)             # rule (2): err <= tol * |t| + FLOOR
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(rel_excess > 0.0, rel_excess / np.abs(t[well]), 0.0)
    worst_rel = float(np.max(rel)) if well.any() else 0.0
    assert worst_rel <= tol, f"{label}: worst relative error on kappa<=1e3: {worst_rel:.3e}"
    stats = {"n": int(err.size), "worst_S_rel": worst_S, "worst_rel_wellcond": worst_rel,
             "frac_wellcond": float(well.mean()) if err.size else 1.0,
             "kappa_median": float(np.median(kappa)) if err.size else 1.0,
             "kappa_max": float(kappa.max()) if err.size else 1.0, "n_nonfinite": int((~fin).sum())}
    if min_wellcond is not None and err.size:
        assert stats["frac_wellcond"] >= min_wellcond, \
            f"{label}: only {stats['frac_wellcond']:.2f} of the samples have kappa <= 1e3 (floor {min_wellcond})"
    if err.size:
        dm = abs(g.mean() - t.mean())
        assert dm <= tol * s.mean() + FLOOR, f"{label}: batch mean off by {dm / s.mean():.3e} of mean(S)"
        if s.mean() <= 1e3 * abs(t.mean()):
            assert dm <= tol * abs(t.mean()) + FLOOR, f"{label}: batch mean relative error {dm / abs(t.mean()):.3e}"
        stats["mean_rel"] = float(dm / max(abs(t.mean()), 1e-300))
    return stats
