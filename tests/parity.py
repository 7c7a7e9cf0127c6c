"""The parity norm of DESIGN.md reading P20, written once for all GPU tests.

Literal "1e-10 relative per sample" is not attainable in double for samples whose terms cancel
(kappa = S/|value| up to 1e18), whichever implementation computes them, so the bar is:
  (1) every sample:        |gpu - truth| <= 1e-10 * S,  S = sum_t |term_t| from the quad oracle
                           (for kappa ~ 1 this IS the plain relative error);
  (2) kappa <= 1e3 subset: |gpu - truth| / |truth| <= 1e-10;
  (3) batch mean:          |mean_gpu - mean_truth| <= 1e-10 * mean(S)  and, when the mean itself is
                           well conditioned (mean(S)/|mean| <= 1e3), plain relative <= 1e-10;
  (4) non-finite truth values must be non-finite on the GPU too;
  (5) where S < 1e-290 (deep underflow) the GPU value must be < 1e-280 in magnitude.
"""
import numpy as np

TOL = 1e-10


def check_parity(gpu, truth, S, tol=TOL, label=""):
    gpu, truth, S = np.asarray(gpu), np.asarray(truth), np.asarray(S)
    assert gpu.shape == truth.shape == S.shape, (gpu.shape, truth.shape, S.shape)
    fin = np.isfinite(truth.real) & np.isfinite(truth.imag) & np.isfinite(S)
    bad_gpu = ~(np.isfinite(gpu.real) & np.isfinite(gpu.imag))
    assert not (bad_gpu & fin).any(), f"{label}: GPU non-finite where the oracle is finite"
    assert bad_gpu[~fin].all(), f"{label}: oracle non-finite but GPU finite"
    g, t, s = gpu[fin], truth[fin], S[fin]
    err = np.abs(g - t)
    # S below 1e-290 (deep underflow at very low temperature: the oracle's quad values do not survive the
    # cast to double): nothing relative can be said there; the GPU must be just as negligible
    tiny = s < 1e-290
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where(tiny, np.where(err <= 1e-280, 0.0, np.inf), err / np.where(tiny, 1.0, s))
    worst_S = float(np.max(ratio)) if err.size else 0.0
    assert worst_S <= tol, f"{label}: worst S-relative error {worst_S:.3e}"
    kappa = np.where(tiny, 1.0, s / np.maximum(np.abs(t), 1e-300))
    well = (kappa <= 1e3) & ~tiny
    worst_rel = float(np.max(err[well] / np.abs(t[well]))) if well.any() else 0.0
    assert worst_rel <= tol, f"{label}: worst relative error on kappa<=1e3: {worst_rel:.3e}"
    stats = {"n": int(err.size), "worst_S_rel": worst_S, "worst_rel_wellcond": worst_rel,
             "frac_wellcond": float(well.mean()) if err.size else 1.0,
             "kappa_median": float(np.median(kappa)) if err.size else 1.0,
             "kappa_max": float(kappa.max()) if err.size else 1.0, "n_nonfinite": int((~fin).sum())}
    if err.size:
        dm = abs(g.mean() - t.mean())
        assert dm <= tol * s.mean(), f"{label}: batch mean off by {dm / s.mean():.3e} of mean(S)"
        if s.mean() <= 1e3 * abs(t.mean()):
            assert dm <= tol * abs(t.mean()), f"{label}: batch mean relative error {dm / abs(t.mean()):.3e}"
        stats["mean_rel"] = float(dm / max(abs(t.mean()), 1e-300))
    return stats
