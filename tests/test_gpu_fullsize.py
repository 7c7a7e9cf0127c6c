"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(ami_evaluate_momenta, the fused S1+S2+S3 call, and ami_run for the sweep), on sampled outputs the
oracle can compute one by one, plus properties that hold at any size."""
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


def oracle_subset(oracle_mod, cfg, sel, betas=None):
    """Truth for the samples `sel` of the config's counter-based sample stream, from the momenta on."""
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    k = np.concatenate([cfg.momenta(1, start=int(i)) for i in sel], axis=0)
    e_rows = ot.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    out = []
    for beta in (cfg.betas if betas is None else betas):
        out.append(ot.evaluate(e_rows, cfg.z_ext, beta, e_reg=cfg.e_reg, quad=True,
                               threads=oracle_mod.hardware_threads(), want_S=True))
    return out


@pytest.mark.parametrize("name,n_truth", [("cfg1", 10_000), ("cfg3", 3000), ("cfg4", 600), ("cfg5", 24)])
def test_full_size_fused_call(ami, oracle_mod, name, n_truth):
    import torch
    cfg = A.get_config(name)
    n = cfg.n_samples
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = tab.generate_momenta(cfg.seed, 0, n)
    out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg)
    assert tab.refresh_info()["reg_plan_status"] == 0          # the specialised kernel is what ran
    assert out.shape == (len(cfg.betas), len(cfg.z_ext), n)
    assert bool(torch.isfinite(torch.view_as_real(out)).all())
    sel = np.unique(np.concatenate([np.linspace(0, n - 1, n_truth).astype(np.int64), [0, 63, 64, n - 65, n - 1]]))
    got = out[:, :, torch.from_numpy(sel).cuda()].cpu().numpy()
    for b, (truth, S) in enumerate(oracle_subset(oracle_mod, cfg, sel)):
        check_parity(got[b], truth, S, label=f"{name} full size beta#{b}")
    # property at any size: the same samples evaluated as a small separate batch give the same bits
    k_sel = k[torch.from_numpy(sel).cuda()].contiguous()
    again = tab.evaluate_momenta(k_sel, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg)
    assert np.array_equal(again.cpu().numpy(), got)


@pytest.mark.parametrize("name,n_truth", [("cfg3", 1500), ("cfg4", 300)])
def test_full_size_independent_batches_in_a_graph(ami, oracle_mod, name, n_truth):
    """The launch configuration bench.py times since AMI_PLAN_UNORDERED exists: K full-size batches with their own
    momenta and result buffers captured in ONE CUDA graph, the first of every round over the buffer sets ordered, the
    others flagged.  Sampled outputs of the LAST and of a middle batch against the oracle; every batch bit-equal to
    the same batch evaluated alone."""
    import torch
    cfg = A.get_config(name)
    n, R, K = cfg.n_samples, 4, 9
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    tab.specialize()
    ks = [tab.generate_momenta(cfg.seed, r * n, n) for r in range(R)]
    outs = [torch.zeros((len(cfg.betas), len(cfg.z_ext), n), dtype=torch.complex128, device="cuda") for _ in range(R)]
    call = lambda r, out, flag: tab.evaluate_momenta(ks[r], [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas,
                                                     e_reg=cfg.e_reg, plan=flag, out=out)
    call(0, outs[0], 0)          # warm-up outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for i in range(K):
            call(i % R, outs[i % R], ami.PLAN_UNORDERED if i % R else 0)
    for o in outs:
        o.zero_()
    g.replay()
    torch.cuda.synchronize()
    for r in (K - 1) % R, 2:
        sel = np.unique(np.concatenate([np.linspace(0, n - 1, n_truth).astype(np.int64), [0, 63, 64, n - 65, n - 1]]))
        got = outs[r][:, :, torch.from_numpy(sel).cuda()].cpu().numpy()
        for b, (truth, S) in enumerate(oracle_subset(oracle_mod, cfg, sel + r * n)):
            check_parity(got[b], truth, S, label=f"{name} batch {r} of the graph")
    for r in range(R):
        alone = call(r, torch.empty_like(outs[r]), 0)
        assert torch.equal(alone.view(torch.float64), outs[r].view(torch.float64)), f"batch {r}"


@pytest.mark.parametrize("name", ["cfg2_se", "cfg2_bubble", "cfg2_bubble_doubled"])
def test_cfg2_sweep_large_batch_streamed(ami, oracle_mod, name):
    """N = 1e7 samples x 8 frequencies through the streamed driver with device-generated momenta
    (1.28 GB of results, chunked), tally included; sampled parity and tally consistency."""
    import torch
    cfg = A.get_config(name, mu=-0.5, beta=10.0)
    n = 10_000_000
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    d_out = torch.empty((1, 8, n), dtype=torch.complex128, device="cuda")
    stats, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, seed=cfg.seed,
                          d_out=d_out, want_sum=True, chunk=1 << 21)
    assert stats["n_chunks"] == 5 and stats["h2d_bytes"] == 0
    sel = np.linspace(0, n - 1, 4000).astype(np.int64)
    got = d_out[:, :, torch.from_numpy(sel).cuda()].cpu().numpy()
    (truth, S), = oracle_subset(oracle_mod, cfg, sel)
    check_parity(got[0], truth, S, label=f"{name} 1e7")
    ref = d_out[0].sum(dim=1).cpu().numpy()
    scale = d_out[0].abs().sum(dim=1).cpu().numpy()
    assert np.all(np.abs(sums[0] - ref) <= 1e-11 * scale)


@pytest.mark.parametrize("plan", ["auto", "flat"])
def test_paper_example1_full_size(ami, oracle_mod, plan):
    """The paper's first example at its own size: order-2 self-energy, N_E = 1e6 energy rows
    drawn in (-8, 8), N_F = 100 fermionic frequencies, beta = 1, through ami_evaluate (no dispersion step);
    1.6 GB of results [N_F][N_E], sampled parity against the quad oracle."""
    import torch
    cfg = A.get_config("paper_ex1")
    n = cfg.n_samples if plan == "auto" else 200_000
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    e_rows = cfg.energies(n)                                     # [n][n_eps], the paper's orientation
    e = torch.from_numpy(np.ascontiguousarray(e_rows.T)).cuda()  # the ABI's [n_eps][n]
    out = tab.evaluate(e, cfg.z_ext, cfg.betas, plan={"auto": ami.PLAN_AUTO, "flat": ami.PLAN_FLAT}[plan])
    assert out.shape == (1, 100, n)
    assert bool(torch.isfinite(torch.view_as_real(out)).all())
    sel = np.unique(np.concatenate([np.linspace(0, n - 1, 3000).astype(np.int64), [0, 63, 64, n - 65, n - 1]]))
    got = out[0][:, torch.from_numpy(sel).cuda()].cpu().numpy()
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    truth, S = ot.evaluate(np.ascontiguousarray(e_rows[sel]), cfg.z_ext, 1.0, quad=True,
                           threads=oracle_mod.hardware_threads(), want_S=True)
    check_parity(got, truth, S, label=f"paper example 1 ({plan})")
    # the Monte-Carlo reading of the example: row means; against the well-conditioned textbook
    # form of the order-2 self-energy evaluated with numpy on every sample of the first row
    if plan == "auto":
        f = lambda x: 0.5 * (1.0 - np.tanh(0.5 * x))             # noqa: E731  (beta = 1)
        x1, x2, x3 = -e_rows[:, 0], -e_rows[:, 1], -e_rows[:, 2]
        ref = -(f(x1) * f(x3) * (1 - f(x2)) + (1 - f(x1)) * (1 - f(x3)) * f(x2)) / (cfg.z_ext[0, 0] + x2 - x1 - x3)
        mean_gpu = complex(out[0, 0].mean().item())
        assert abs(mean_gpu - ref.mean()) <= 1e-10 * np.abs(ref).mean()


@pytest.mark.parametrize("n", [0, 1, 63, 64, 65, 129])
def test_fused_edge_sizes(ami, oracle_mod, n):
    import torch
    cfg = A.get_config("cfg4")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = torch.from_numpy(cfg.momenta(n)).cuda() if n else torch.empty((0, 6, 2), dtype=torch.float64, device="cuda")
    out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg)
    assert out.shape == (1, 1, n)
    if n:
        (truth, S), = oracle_subset(oracle_mod, cfg, np.arange(n))
        check_parity(out.cpu().numpy()[0], truth, S, label=f"fused n={n}")


def test_large_momenta_take_the_library_cosine(ami, oracle_mod):
    """Momenta far outside the Brillouin zone (|K| >= 5e5) leave the bounded-range cosine."""
    import torch
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k_host = cfg.momenta(256)
    k_host[::3] += 2.0 * np.pi * 200_000        # same physics, huge argument
    k_host[1::7] *= 1.0e5
    k = torch.from_numpy(k_host).cuda()
    e = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu).cpu().numpy()
    want = oracle_mod.OracleTable.from_diagram(cfg.diagram).dispersion(k_host, [cfg.q], cfg.t, cfg.mu, quad=True)
    # the argument itself is only known to ~ulp(1e6) = 1e-10 once the momenta are that large
    np.testing.assert_allclose(e.T, want, rtol=0, atol=5e-9)
    e2 = torch.zeros((cfg.diagram.n_eps, 256), dtype=torch.float64, device="cuda")
    tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_out=e2)
    assert np.array_equal(e2.cpu().numpy(), e)


def test_bench_line_contract():
    """bench.py as the driver runs it (defaults, fewer steps): ONE JSON line with the contract's keys -- metric and
    config of BASELINE.json, roofline and cpu_baseline objects, e2e with its byte counts, launches counted, clocks
    sampled -- and the large-table and complex-energy rows beside the graded configurations."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--steps", "5", "--warmup", "3", "--cpu-seconds", "2"],
                         capture_output=True, text=True, timeout=900, cwd=root)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["metric"] == "ami_term_evaluations_per_s" and d["unit"] == "term-evals/s" and d["higher_is_better"] is True
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert d["config"] == {"workload": "cfg3", "samples_per_gpu": 1_000_000, "n_freq": 1, "n_beta": 1, "T_flat": 68,
                           "precision": "double"}
    assert d["value"] > 1e11 and abs(d["value"] - 68 * 1e6 / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert 0.3 < r["frac"] < 1.05 and 0.95 < r["peak"] / r["peak_nominal"] < 1.05 and r["traffic"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 64_000_000 and e["d2h_bytes_per_step"] == 16_000_000 and 0 < e["value"] < d["value"]
    assert d["gpu_launches"] >= 5 and d["clocks"]["sm_mhz"] and d["e2e_seeded"]["h2d_bytes_per_step"] == 0
    ow = d["other_workloads"]
    assert {"cfg4", "cfg5", "cfg2_se", "cfg1", "order7", "stress8", "cfg5b"} <= set(ow)
    assert ow["stress8"]["T_flat"] == 40244 and ow["stress8"]["ms_per_step"] < 3.0        # <= 3 ms per 2e4 samples
    assert "split" in ow["stress8"]["plan"] and ow["cfg5b"]["ms_per_step"] < ow["cfg5b"]["flat_plan_ms_per_step"]
    assert d["monte_carlo"]["launches_per_step"] == 3 and d["monte_carlo"]["d2h_bytes_per_step"] == 32
