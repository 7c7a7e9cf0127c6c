"""GPU parity across parameter regimes the fixed configurations do not visit: seeded random draws of the energy
scale (1e-2 .. 30 times the band width), one to five temperatures per launch with beta log-uniform in 1e-3 .. 5e3,
external frequencies on the Matsubara axis, near the real axis, far out and anywhere in the plane, degenerate energy
symbols, real and complex energies (imaginary parts 1e-6 .. 1) -- every (plan, temperature) block against the quad
oracle under the norm of tests/parity.py.  (This is the sweep that found the overflow of the complex-energy leaf at
beta |Re E| of a few hundred; it stays as a regression net for the specialised kernels' leaf arithmetic.)"""
import math

import numpy as np
import pytest

import ami_inputs as A
from parity import check_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ami():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    pkg.lib()
    return pkg


@pytest.mark.parametrize("name", ["cfg1", "cfg2_se", "cfg2_bubble", "cfg2_bubble_doubled", "cfg3", "cfg4", "cfg5"])
def test_random_regimes_against_the_oracle(ami, oracle_mod, name):
    import torch
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    rng = np.random.default_rng(20231117 + sum(map(ord, name)))
    n, n_checks = 96, 0
    fermionic_ext = "bubble" not in name
    for trial in range(12):
        scale = 10.0 ** rng.uniform(-2, 1.5)
        betas = list(10.0 ** rng.uniform(-3, 3.7, size=int(rng.integers(1, 6))))
        e = rng.uniform(-4, 4, size=(n, cfg.diagram.n_eps)) * scale
        if trial % 4 == 1:
            e[:, 1] = e[:, 0]                       # two symbols with the same energy
        kind = trial % 4
        if kind == 0:       # Matsubara points of the first temperature
            z = np.array([[1j * (2 * m + (1 if fermionic_ext else 0)) * math.pi / betas[0]] for m in (0, 1, -3)])
        elif kind == 1:     # continued to just above the real axis
            z = np.array([[w + 1j * g] for w, g in ((0.3, 0.1), (-2.0, 1e-3), (0.0, 1e-6))])
        elif kind == 2:     # far out
            z = np.array([[complex(rng.uniform(-50, 50), rng.uniform(1e-3, 2))] for _ in range(2)])
        else:               # anywhere
            z = np.array([[complex(rng.uniform(-5, 5), rng.uniform(-2, 2))] for _ in range(3)])
        ee = e - 1j * rng.uniform(0, 1, size=e.shape) * 10.0 ** rng.uniform(-6, 0) if trial % 2 else e
        et = torch.from_numpy(np.ascontiguousarray(ee.T)).cuda()
        for plan, pn in ((ami.PLAN_REG, "reg"), (ami.PLAN_FLAT, "flat")):
            out = tab.evaluate(et, z, betas, e_reg=cfg.e_reg, plan=plan).cpu().numpy()
            for b, beta in enumerate(betas):
                truth, S = ot.evaluate(ee, z, beta, e_reg=cfg.e_reg, quad=True, threads=oracle_mod.hardware_threads(),
                                       want_S=True)
                check_parity(out[b], truth, S, label=f"{name} trial {trial} {pn} scale={scale:.2e} beta={beta:.3e} "
                                                     f"n_b={len(betas)} complex={trial % 2}")
                n_checks += 1
    assert n_checks >= 48


@pytest.mark.parametrize("order,seeds", [(2, range(4)), (3, range(6)), (4, range(6)), (5, range(5)), (6, (1, 2))])
def test_random_diagrams_against_the_oracle(ami, oracle_mod, order, seeds):
    """Topologies the fixed configurations do not contain: seeded random 1PI self-energy diagrams (SURVEY 8(d) generator)
    of orders 2-6 -- some with double poles, the largest order-6 tables on the split plan -- constructed by the library
    and by the oracle independently, evaluated by every plan the table supports, against the quad oracle."""
    import torch
    thr = oracle_mod.hardware_threads()
    for seed in seeds:
        d = A.random_self_energy(order, seed)
        tab = ami.AmiTable.from_diagram(d)
        ot = oracle_mod.OracleTable.from_diagram(d)
        n = 128 if order < 6 else 48
        rng = np.random.default_rng(1000 * order + seed)
        k = torch.from_numpy(rng.uniform(-math.pi, math.pi, size=(n, d.n_int, 2))).cuda()
        betas = [float(10 ** rng.uniform(-1, 1.5)), 8.0]
        z = np.array([[1j * math.pi / betas[0]], [0.4 + 0.05j]])
        e = tab.dispersion(k, [[0.5 * math.pi, 0.5 * math.pi]], 1.0, -0.1)
        e_rows = e.cpu().numpy().T.copy()
        truths = [ot.evaluate(e_rows, z, beta, e_reg=1e-8, quad=True, threads=thr, want_S=True) for beta in betas]
        for plan, pn in ((ami.PLAN_AUTO, "auto"), (ami.PLAN_FLAT, "flat"), (ami.PLAN_TREE, "tree")):
            try:
                out = tab.evaluate(e, z, betas, e_reg=1e-8, plan=plan).cpu().numpy()
            except ami.AmiError:
                assert plan == ami.PLAN_TREE        # the only plan a table may be outside of
                continue
            for b, (truth, S) in enumerate(truths):
                check_parity(out[b], truth, S, label=f"order {order} seed {seed} {pn} beta={betas[b]:.3g} "
                                                     f"T={tab.info['n_terms']}")
        # the same table with complex energies (specialised kernels of either kind, and the table-driven one)
        ee = e_rows[:32] - 1j * rng.uniform(0, 0.1, size=e_rows[:32].shape)
        et = torch.from_numpy(np.ascontiguousarray(ee.T)).cuda()
        truth, S = ot.evaluate(ee, z, betas[1], e_reg=1e-8, quad=True, threads=thr, want_S=True)
        for plan, pn in ((ami.PLAN_AUTO, "auto"), (ami.PLAN_FLAT, "flat")):
            out = tab.evaluate(et, z, betas[1:], e_reg=1e-8, plan=plan).cpu().numpy()
            check_parity(out[0], truth, S, label=f"order {order} seed {seed} {pn} complex energies")
