"""Parity statistics of the CUDA path against the quad-precision oracle, per config (reading P20, item 4):
worst S-relative error, worst plain relative error on the well-conditioned subset, batch-mean error and
the condition-number histogram.  Run on a GPU box:  python tests/parity_report.py  > gpurun_out/parity.md
(test infrastructure: this script may call oracle/)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import ami_inputs as A  # noqa: E402
import oracle  # noqa: E402
import paper_2311_17189_b200 as ami  # noqa: E402
from parity import check_parity  # noqa: E402

CASES = [("cfg1", 10_000, {}), ("cfg2_se", 20_000, {"mu": -0.5, "beta": 10.0}),
         ("cfg2_bubble", 20_000, {"mu": -0.5, "beta": 10.0}), ("cfg2_bubble_doubled", 20_000, {"mu": 0.0, "beta": 5.0}),
         ("cfg3", 20_000, {}), ("cfg4", 4_000, {}), ("cfg5", 300, {})]


def main():
    import torch
    threads = oracle.hardware_threads()
    print("| config | samples x freq x beta | worst \\|err\\|/S | worst rel. err (kappa<=1e3) | share kappa<=1e3 | "
          "kappa median / max | mean rel. err | kappa>1e6 |")
    print("|---|---|---|---|---|---|---|---|")
    for name, n, over in CASES:
        cfg = A.get_config(name, **over)
        tab = ami.AmiTable.from_diagram(cfg.diagram)
        k = tab.generate_momenta(cfg.seed, 0, n)
        out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg).cpu().numpy()
        ot = oracle.OracleTable.from_diagram(cfg.diagram)
        e_rows = ot.dispersion(cfg.momenta(n), [cfg.q], cfg.t, cfg.mu)
        worst_S = worst_rel = mean_rel = kmax = 0.0
        well, kmed, big = [], [], []
        for b, beta in enumerate(cfg.betas):
            truth, S = ot.evaluate(e_rows, cfg.z_ext, beta, e_reg=cfg.e_reg, quad=True, threads=threads, want_S=True)
            st = check_parity(out[b], truth, S, label=name)
            worst_S = max(worst_S, st["worst_S_rel"])
            worst_rel = max(worst_rel, st["worst_rel_wellcond"])
            mean_rel = max(mean_rel, st.get("mean_rel", 0.0))
            kmax = max(kmax, st["kappa_max"])
            well.append(st["frac_wellcond"])
            kmed.append(st["kappa_median"])
            kap = S / np.maximum(np.abs(truth), 1e-300)
            big.append(float((kap > 1e6).mean()))
        print(f"| {name} | {n} x {len(cfg.z_ext)} x {len(cfg.betas)} | {worst_S:.1e} | {worst_rel:.1e} | "
              f"{100 * np.mean(well):.0f} % | {np.median(kmed):.1f} / {kmax:.1e} | {mean_rel:.1e} | {100 * np.mean(big):.1f} % |")
        del tab
        torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
