"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the same seeded
inputs, element by element (norm: tests/parity.py, reading P20)."""
import math

import numpy as np
import pytest

import ami_inputs as A
from parity import WELLCOND_FLOOR, check_parity

pytestmark = pytest.mark.gpu

PLANS = {"flat": 1, "tree": 3, "auto": 0}   # auto = the register plan where the table is eligible, else flat


@pytest.fixture(scope="module")
def ami():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    pkg.lib()  # raises if the extension is missing: no fallback
    return pkg


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    return torch


def gpu_energies(torch, tab, cfg, k_host):
    k = torch.from_numpy(np.ascontiguousarray(k_host)).cuda()
    return tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)


def truth_for(oracle_mod, cfg, e_rows, z, beta, e_reg, quad=True, sum_order=None, want_logs=False):
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram, sum_order=sum_order)
    return ot.evaluate(e_rows, z, beta, e_reg=e_reg, quad=quad, threads=oracle_mod.hardware_threads(), want_S=True,
                       want_logs=want_logs)


# ------------------------------------------------------------------ S1 dispersion
@pytest.mark.parametrize("name,n", [("cfg1", 10_000), ("cfg3", 4133), ("cfg4", 1000), ("cfg5", 777)])
def test_dispersion_parity(ami, torch_mod, oracle_mod, name, n):
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = cfg.momenta(n)
    e = gpu_energies(torch_mod, tab, cfg, k).cpu().numpy()
    want = oracle_mod.OracleTable.from_diagram(cfg.diagram).dispersion(k, [cfg.q], cfg.t, cfg.mu, quad=True)
    assert e.shape == (cfg.diagram.n_eps, n)
    # |e| <= 4t + |mu|; K is a sum of up to m+1 doubles of size pi, so a few ulp of 4*pi in the angle
    np.testing.assert_allclose(e.T, want, rtol=0, atol=2e-14)


def test_dispersion_soa_layout(ami, torch_mod):
    """SoA momenta [2m][N] through the stride arguments of the ABI."""
    import ctypes as C
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = torch_mod.from_numpy(cfg.momenta(1000)).cuda()
    ref = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    ksoa = k.reshape(1000, -1).t().contiguous()
    out = torch_mod.empty_like(ref)
    q = np.array(cfg.q)
    rc = ami.lib().ami_dispersion(tab._h, C.c_void_p(ksoa.data_ptr()), 1, 1000, q.ctypes.data, cfg.t, cfg.mu, 1000,
                                  C.c_void_p(out.data_ptr()), C.c_void_p(torch_mod.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch_mod.cuda.synchronize()
    assert torch_mod.equal(out, ref)


@pytest.mark.parametrize("dim", [1, 2, 3])
@pytest.mark.parametrize("band", [0, 1])
def test_dispersion_lattice_parity(ami, torch_mod, oracle_mod, dim, band):
    """ami_dispersion_lattice (Eq. 14 for d = 1..3, tight-binding and free-particle bands)
    against the oracle in quad precision, then the values of the order-4 diagram from those energies."""
    from ami_inputs.rng import momenta
    cfg = A.get_config("cfg3")
    n = 2048 + 77
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    k = momenta(cfg.seed + 7 * dim + band, n, cfg.diagram.n_int, d=dim)
    q = np.array([0.5 * math.pi, -0.25 * math.pi, 1.0][:dim])
    t, mu = (1.0, -0.2) if band == 0 else (0.5, 1.5)
    e = tab.dispersion(torch_mod.from_numpy(k).cuda(), [q], t, mu, dim=dim, band=band)
    want = ot.dispersion(k, [q], t, mu, quad=True, dim=dim, band=band)
    # tight binding: |e| <= 2 d t + |mu| with a few ulp of (m+1) pi in each angle; free particles:
    # |K_c| <= 5 pi, so e up to 0.5 * 3 * 250 with a few ulp of that
    np.testing.assert_allclose(e.cpu().numpy().T, want, rtol=0, atol=2e-14 if band == 0 else 4e-13)
    if dim == 2 and band == 0:      # the general entry point is the configurations' kernel for d = 2
        assert torch_mod.equal(e, tab.dispersion(torch_mod.from_numpy(k).cuda(), [q], t, mu))
    for plan in (ami.PLAN_REG, ami.PLAN_FLAT):
        got = tab.evaluate(e, cfg.z_ext, cfg.betas, plan=plan).cpu().numpy()
        truth, S = ot.evaluate(np.ascontiguousarray(e.cpu().numpy().T), cfg.z_ext, cfg.betas[0], quad=True,
                               threads=oracle_mod.hardware_threads(), want_S=True)
        ok = np.isfinite(truth[0]) & (S[0] > 1e-290)
        assert ok.mean() > 0.99
        assert np.max(np.abs(got[0, 0] - truth[0])[ok] / S[0][ok]) <= 1e-10


def test_dispersion_lattice_errors(ami, torch_mod):
    import ctypes as C
    cfg = A.get_config("cfg1")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = torch_mod.zeros((8, cfg.diagram.n_int, 3), dtype=torch_mod.float64, device="cuda")
    out = torch_mod.zeros((cfg.diagram.n_eps, 8), dtype=torch_mod.float64, device="cuda")
    q = np.zeros(4)
    st = C.c_void_p(torch_mod.cuda.current_stream().cuda_stream)
    for dim, band in ((0, 0), (4, 0), (2, 2), (2, -1)):
        assert ami.lib().ami_dispersion_lattice(tab._h, C.c_void_p(k.data_ptr()), 6, 1, q.ctypes.data, 1.0, 0.0, dim,
                                                band, 8, C.c_void_p(out.data_ptr()), st) == -1


# ------------------------------------------------------------------ S2 + S3 evaluate
def run_eval_case(ami, torch, oracle_mod, cfg, n, plan, betas=None, z=None, n_truth=None, start=0, sum_order=None):
    tab = ami.AmiTable.from_diagram(cfg.diagram, sum_order=sum_order)
    k = cfg.momenta(n, start=start)
    e_dev = gpu_energies(torch, tab, cfg, k)
    # at the configuration's own temperatures and frequencies the share of well-conditioned samples is known
    floor = WELLCOND_FLOOR.get(cfg.name) if betas is None and z is None else None
    betas = cfg.betas if betas is None else betas
    z = cfg.z_ext if z is None else z
    out = tab.evaluate(e_dev, z, betas, e_reg=cfg.e_reg, plan=plan).cpu().numpy()
    assert out.shape == (len(betas), len(z), n)
    e_rows = e_dev.cpu().numpy().T.copy()
    sel = np.arange(n) if n_truth is None or n_truth >= n else np.linspace(0, n - 1, n_truth).astype(np.int64)
    stats = []
    for b, beta in enumerate(betas):
        truth, S, l2S, l2v = truth_for(oracle_mod, cfg, e_rows[sel], z, beta, cfg.e_reg, sum_order=sum_order,
                                       want_logs=True)
        stats.append(check_parity(out[b][:, sel], truth, S, label=f"{cfg.name} beta={beta}", log2S=l2S, log2abs=l2v,
                                  min_wellcond=floor if len(sel) >= 500 else None))
    return stats


@pytest.mark.parametrize("plan", list(PLANS))
def test_cfg1_order2(ami, torch_mod, oracle_mod, plan):
    run_eval_case(ami, torch_mod, oracle_mod, A.get_config("cfg1"), 10_000, PLANS[plan])


@pytest.mark.parametrize("plan", list(PLANS))
@pytest.mark.parametrize("mu,beta", [(0.0, 2.0), (-0.5, 5.0), (0.0, 10.0)])
@pytest.mark.parametrize("name", ["cfg2_se", "cfg2_bubble", "cfg2_bubble_doubled"])
def test_cfg2_sweep_points(ami, torch_mod, oracle_mod, name, mu, beta, plan):
    """8 frequencies; the bosonic n = 0 case goes through the regulator rule P10(b)."""
    cfg = A.get_config(name, mu=mu, beta=beta)
    run_eval_case(ami, torch_mod, oracle_mod, cfg, 5000 + 37, PLANS[plan])


@pytest.mark.parametrize("plan", list(PLANS))
def test_cfg3_order4(ami, torch_mod, oracle_mod, plan):
    st = run_eval_case(ami, torch_mod, oracle_mod, A.get_config("cfg3"), 20_000 + 11, PLANS[plan])
    assert st[0]["n_nonfinite"] == 0


@pytest.mark.parametrize("plan", list(PLANS))
def test_cfg4_order6(ami, torch_mod, oracle_mod, plan):
    run_eval_case(ami, torch_mod, oracle_mod, A.get_config("cfg4"), 4096 + 5, PLANS[plan], n_truth=1500)


@pytest.mark.parametrize("plan", list(PLANS))
def test_cfg5_grid(ami, torch_mod, oracle_mod, plan):
    """64 continued frequencies x 4 temperatures (launch splitting over frequencies)."""
    run_eval_case(ami, torch_mod, oracle_mod, A.get_config("cfg5"), 600 + 3, PLANS[plan], n_truth=150)


@pytest.mark.parametrize("name", ["cfg5", "cfg3", "cfg2_bubble_doubled"])
@pytest.mark.parametrize("plan", ["flat", "reg", "auto"])
def test_complex_energies_variant_5b(ami, torch_mod, oracle_mod, name, plan):
    """P19: complex energies e_j - i gamma_j (energy_t is complex128) make the Fermi/Bose arguments
    complex.  The specialised kernels have a complex-energy variant (per-symbol exponential 2^n m (cos + i sin),
    exponents still added as integers): AMI_PLAN_REG, which never falls back, must succeed and agree with the quad
    oracle, as must the table-driven flat kernel; cfg3 and the doubled bubble carry derivative leaves."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 500 + 3
    e_real = gpu_energies(torch_mod, tab, cfg, cfg.momenta(n)).cpu().numpy()
    gam = A.uniform01(99, np.arange(e_real.size, dtype=np.uint64)).reshape(e_real.shape) * 0.05
    e_c = e_real - 1j * gam
    z = cfg.z_ext[::8]
    betas = [5.0, 11.0] if name != "cfg2_bubble_doubled" else [4.0]
    pid = {"flat": ami.PLAN_FLAT, "reg": ami.PLAN_REG, "auto": ami.PLAN_AUTO}[plan]
    out = tab.evaluate(torch_mod.from_numpy(e_c).cuda(), z, betas, e_reg=cfg.e_reg, plan=pid).cpu().numpy()
    for b, beta in enumerate(betas):
        truth, S = truth_for(oracle_mod, cfg, e_c.T.copy(), z, beta, cfg.e_reg)
        check_parity(out[b], truth, S, label=f"5b {name} {plan} beta={beta}")
    # one very cold and one very hot temperature alone in a launch (single-temperature body; P12: |d|^2 of the complex
    # leaves must not overflow -- it did in the specialised kernels until the leaf was rescaled by 2^-N)
    for beta in (5000.0, 200.0, 1e-3):
        cold = tab.evaluate(torch_mod.from_numpy(e_c).cuda(), z, [beta], e_reg=cfg.e_reg, plan=pid).cpu().numpy()
        truth, S = truth_for(oracle_mod, cfg, e_c.T.copy(), z, beta, cfg.e_reg)
        check_parity(cold[0], truth, S, label=f"5b {name} {plan} beta={beta}")
    if plan == "reg":      # real energies given as complex numbers: the same values as the real-energy kernels
        e0 = torch_mod.from_numpy(e_real.astype(np.complex128)).cuda()
        a = tab.evaluate(e0, z, betas, e_reg=cfg.e_reg, plan=pid)
        r = tab.evaluate(torch_mod.from_numpy(e_real).cuda(), z, betas, e_reg=cfg.e_reg, plan=pid)
        truth, S = truth_for(oracle_mod, cfg, e_real.T.copy(), z, betas[0], cfg.e_reg)
        check_parity(a.cpu().numpy()[0], truth, S, label="5b zero imaginary part")
        assert np.max(np.abs((a - r).cpu().numpy()[0]) / S) <= 1e-13


@pytest.mark.parametrize("plan", list(PLANS))
def test_stress8_large_table(ami, torch_mod, oracle_mod, plan):
    """Order 8, 4e4 terms: the table is far larger than any on-chip staging tile."""
    cfg = A.get_config("stress8")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 96 + 7
    e_dev = gpu_energies(torch_mod, tab, cfg, cfg.momenta(n))
    out = tab.evaluate(e_dev, cfg.z_ext, cfg.betas, plan=PLANS[plan]).cpu().numpy()
    truth, S = truth_for(oracle_mod, cfg, e_dev.cpu().numpy().T.copy(), cfg.z_ext, cfg.betas[0], 0.0, quad=False)
    # double oracle as truth here (quad is too slow for 4e4 terms): 1e-10 * S still holds
    check_parity(out[0], truth, S, label="stress8")


@pytest.mark.parametrize("n", [0, 1, 31, 32, 33, 257])
def test_edge_sizes(ami, torch_mod, oracle_mod, n):
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    e = torch_mod.zeros((cfg.diagram.n_eps, n), dtype=torch_mod.float64, device="cuda")
    if n:
        e = gpu_energies(torch_mod, tab, cfg, cfg.momenta(n))
    out = tab.evaluate(e, cfg.z_ext, cfg.betas)
    assert out.shape == (1, 1, n)
    if n:
        truth, S = truth_for(oracle_mod, cfg, e.cpu().numpy().T.copy(), cfg.z_ext, cfg.betas[0], 0.0)
        check_parity(out.cpu().numpy()[0], truth, S)


def test_degenerate_samples_nonfinite_agree(ami, torch_mod, oracle_mod):
    """Exactly degenerate bubble at Omega = 0 without regulator: 0/0 on both sides; with the
    regulator both are finite and agree."""
    cfg = A.get_config("cfg2_bubble")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    e_rows = np.array([[0.3, -0.7], [0.5, 0.5], [1.25, 1.25], [-0.2, 0.9]])
    e_dev = torch_mod.from_numpy(e_rows.T.copy()).cuda()
    z = np.array([[0j], [2j * math.pi / 5.0]])
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    for eta in (0.0, 1e-8):
        out = tab.evaluate(e_dev, z, [5.0], e_reg=eta).cpu().numpy()
        truth, S = ot.evaluate(e_rows, z, 5.0, e_reg=eta, quad=True, want_S=True)
        check_parity(out[0], truth, S, label=f"eta={eta}")
        assert np.isfinite(out[0][1]).all()
        assert np.isfinite(out[0][0]).all() == (eta > 0)


# ------------------------------------------------------------------ register plan + fused S1+S2+S3
@pytest.mark.parametrize("name", ["cfg1", "cfg2_bubble_doubled", "cfg3", "cfg4", "cfg5"])
def test_register_plan_is_what_auto_runs(ami, torch_mod, name):
    """AMI_PLAN_AUTO compiles and runs the specialised kernels for every graded config."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.info["reg_plan_status"] == 1          # eligible, not compiled yet
    e = gpu_energies(torch_mod, tab, cfg, cfg.momenta(300))
    a = tab.evaluate(e, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=ami.PLAN_AUTO)
    assert tab.refresh_info()["reg_plan_status"] == 0
    b = tab.evaluate(e, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=ami.PLAN_REG)
    assert torch_mod.equal(a, b)


def test_register_plan_limits(ami, torch_mod):
    """Tables beyond one register-resident kernel (order 8) are specialised as a split plan, for real and for complex
    energies; what no specialised kernel covers (a tally or momenta with the split plan's complex variant) is refused
    by the launcher, not run."""
    cfg = A.get_config("stress8")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.info["reg_plan_status"] == 1 and tab.info["plan_kind"] == 2
    assert ami.AmiTable.from_diagram(A.get_config("cfg4").diagram).info["plan_kind"] == 1
    ec = gpu_energies(torch_mod, tab, cfg, cfg.momenta(40)).to(torch_mod.complex128)
    a = tab.evaluate(ec, cfg.z_ext, cfg.betas, plan=ami.PLAN_REG)       # complex energies, zero imaginary parts ...
    r = tab.evaluate(ec.real.contiguous(), cfg.z_ext, cfg.betas, plan=ami.PLAN_REG)   # ... against the real-energy kernels
    scale = r.abs().max().item()
    assert (a - r).abs().max().item() <= 1e-9 * scale


@pytest.mark.parametrize("name,n", [("cfg1", 10_000), ("cfg3", 50_000 + 3), ("cfg4", 3000 + 1), ("cfg5", 401)])
@pytest.mark.parametrize("plan", ["flat", "tree", "auto"])
def test_fused_momenta_path(ami, torch_mod, oracle_mod, name, n, plan):
    """ami_evaluate_momenta == ami_dispersion followed by ami_evaluate, bit for bit, and the energies
    it stores are those of ami_dispersion; then against the oracle from the momenta on."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k_host = cfg.momenta(n)
    k = torch_mod.from_numpy(k_host).cuda()
    e_ref = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    ref = tab.evaluate(e_ref, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=PLANS[plan])
    e_out = torch_mod.zeros_like(e_ref)
    got = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=PLANS[plan],
                               e_out=e_out)
    assert torch_mod.equal(e_out, e_ref)
    assert torch_mod.equal(got, ref)
    got2 = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=PLANS[plan])
    assert torch_mod.equal(got2, ref)
    sel = np.linspace(0, n - 1, min(n, 300)).astype(np.int64)
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    e_rows = ot.dispersion(k_host[sel], [cfg.q], cfg.t, cfg.mu)
    for b, beta in enumerate(cfg.betas):
        truth, S = ot.evaluate(e_rows, cfg.z_ext, beta, e_reg=cfg.e_reg, quad=True,
                               threads=oracle_mod.hardware_threads(), want_S=True)
        check_parity(got.cpu().numpy()[b][:, sel], truth, S, label=f"fused {name}")


@pytest.mark.parametrize("plan", ["flat", "tree", "auto"])
@pytest.mark.parametrize("fused", [False, True])
def test_grid_larger_than_one_launch(ami, torch_mod, oracle_mod, plan, fused):
    """70 frequencies x 9 temperatures do not fit one launch (64 frequency words, 8 temperatures):
    the call is split into 2 x 2 launches; every (beta, frequency) row must land in its place."""
    cfg = A.get_config("cfg5")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 333
    z = (np.linspace(-3.0, 3.0, 70) + 0.1j).reshape(70, 1)
    z[5, 0] = 1j * math.pi / 5.0                     # one Matsubara point among the continued ones
    betas = [1.0, 2.0, 3.0, 5.0, 8.0, 10.0, 13.0, 20.0, 4.0]
    k_host = cfg.momenta(n)
    k = torch_mod.from_numpy(k_host).cuda()
    e = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    if fused:
        e_out = torch_mod.zeros_like(e) if plan == "auto" else None
        out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, z, betas, plan=PLANS[plan], e_out=e_out)
        if e_out is not None:
            assert torch_mod.equal(e_out, e)
    else:
        out = tab.evaluate(e, z, betas, plan=PLANS[plan])
    assert out.shape == (9, 70, n)
    out = out.cpu().numpy()
    e_rows = e.cpu().numpy().T.copy()
    sel = np.arange(0, n, 11)
    for b in (0, 7, 8):        # first launch, last of the first beta chunk, the second beta chunk
        truth, S = truth_for(oracle_mod, cfg, e_rows[sel], z, betas[b], 0.0)
        check_parity(out[b][:, sel], truth, S, label=f"split grid beta#{b}")
    # rows computed alone equal the rows of the split call, bit for bit
    one = tab.evaluate(e, z[64:], [betas[8]], plan=PLANS[plan]).cpu().numpy()
    # (both are launches of ONE temperature, hence the same body of the register plan: same arithmetic, same bits;
    # a row computed among several temperatures may differ from them in rounding)
    assert np.array_equal(one[0], out[8, 64:])


@pytest.mark.parametrize("n_b", [2, 3, 5, 6, 7, 8])
@pytest.mark.parametrize("name", ["cfg5", "cfg1", "cfg4"])
def test_several_temperatures_per_launch(ami, torch_mod, oracle_mod, name, n_b):
    """The several-temperature body of the register plan for every way n_b splits into blocks of four, two and one
    temperatures (cfg5 and cfg1 take the prefix-product form of the R part, cfg4 keeps the Horner
    form): every (temperature, frequency) row against the oracle, and against the same temperature evaluated alone
    (another summation order: equal to rounding on the scale S of the sample, not bit for bit)."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.specialize()["plan_kind"] == 1
    n = 257
    betas = [1.5, 2.0, 3.0, 5.0, 7.0, 10.0, 14.0, 20.0][:n_b]
    if n_b == 7:       # one launch with a very hot and two very cold temperatures among moderate ones (P12: no overflow)
        betas = [0.01, 5000.0, 1.0, 200.0, 8.0, 1e-4, 50.0]
    z = (np.array([-2.5, -0.3, 0.9, 3.1, 0.0]) + np.array([0.1, 0.1, 0.2, 0.05, math.pi / 5.0]) * 1j).reshape(5, 1)
    k_host = cfg.momenta(n)
    k = torch_mod.from_numpy(k_host).cuda()
    e = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, z, betas, e_reg=cfg.e_reg).cpu().numpy()
    assert out.shape == (n_b, 5, n)
    e_rows = e.cpu().numpy().T.copy()
    for b, beta in enumerate(betas):
        truth, S = truth_for(oracle_mod, cfg, e_rows, z, beta, cfg.e_reg)
        check_parity(out[b], truth, S, label=f"{name} n_b={n_b} beta#{b}")
        alone = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, z, [beta], e_reg=cfg.e_reg).cpu().numpy()[0]
        assert np.all(np.abs(alone - out[b]) <= 1e-12 * S + 1e-280), f"{name} n_b={n_b} beta#{b} against the row computed alone"
    if name != "cfg5":
        return
    # the same with complex energies: complex Q(n) in the prefix-product form
    gam = A.uniform01(7, np.arange(e_rows.size, dtype=np.uint64)).reshape(e_rows.shape) * 0.05
    e_c = e_rows - 1j * gam
    out_c = tab.evaluate(torch_mod.from_numpy(np.ascontiguousarray(e_c.T)).cuda(), z, betas, e_reg=cfg.e_reg).cpu().numpy()
    for b, beta in enumerate(betas):
        truth, S = truth_for(oracle_mod, cfg, e_c, z, beta, cfg.e_reg)
        check_parity(out_c[b], truth, S, label=f"{name} complex energies n_b={n_b} beta#{b}")


@pytest.mark.parametrize("plan", list(PLANS))
@pytest.mark.parametrize("name", ["cfg3", "cfg2_bubble_doubled", "cfg4"])
def test_extreme_temperatures(ami, torch_mod, oracle_mod, name, plan):
    """Reading P12 on the GPU: beta from 0.01 to 5000 (beta |E| up to ~1e5: every exponential would
    overflow if formed naively; the register plan clamps the summed binary exponent instead)."""
    cfg = A.get_config(name)
    z = np.array([[1j * math.pi / 7.0 if cfg.diagram.slot_is_fermionic[-1] else 2j * math.pi / 7.0]])
    sts = run_eval_case(ami, torch_mod, oracle_mod, cfg, 1500 + 3, PLANS[plan], betas=(0.01, 300.0, 5000.0), z=z,
                        n_truth=400)
    assert all(st["n_nonfinite"] == 0 for st in sts)


def split_case(name):
    """Tables beyond one register-resident kernel: the order-8 stress table (T = 40244) and an order-7 one (T = 8598)."""
    cfg = A.get_config("stress8")
    if name == "o7":
        cfg.diagram, cfg.name = A.random_self_energy(7, 0), "o7"
    if name == "o9":      # the largest order the paper benchmarks: T = 137644
        cfg.diagram, cfg.name = A.random_self_energy(9, 0), "o9"
    return cfg


@pytest.mark.parametrize("name", ["o7", "stress8", "o9"])
def test_split_plan_large_tables(ami, torch_mod, oracle_mod, name):
    """AMI_PLAN_AUTO / AMI_PLAN_REG for orders 7-8 (PAPER.md:389-393 runs m = 9): the split plan -- leaf kernel,
    the Horner plan's groups in parts of register-plan size (one launch, grid.y = part), combine kernel.  Values
    against the oracle (double precision as truth: quad is too slow for 4e4 terms; the bar is still 1e-10 S),
    fused == unfused bit for bit, a (beta, frequency) grid, and a batch that spans several sample chunks."""
    cfg = split_case(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.info["plan_kind"] == 2 and tab.info["reg_plan_status"] == 1
    n = 300 + 7 if name != "o9" else 64 + 5
    k = torch_mod.from_numpy(cfg.momenta(n)).cuda()
    e = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    out = tab.evaluate(e, cfg.z_ext, cfg.betas, plan=ami.PLAN_AUTO)
    info = tab.refresh_info()
    assert info["reg_plan_status"] == 0 and info["specialize_ms"] > 0
    fused = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, plan=ami.PLAN_REG)
    assert torch_mod.equal(out, fused)
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    e_rows = e.cpu().numpy().T.copy()
    thr = oracle_mod.hardware_threads()
    truth, S = ot.evaluate(e_rows, cfg.z_ext, cfg.betas[0], quad=False, threads=thr, want_S=True)
    st = check_parity(out.cpu().numpy()[0], truth, S, label=name)
    assert st["n_nonfinite"] == 0
    if name == "o9":
        return
    # the table-driven interpretation of the same Horner plan agrees too
    tree = tab.evaluate(e, cfg.z_ext, cfg.betas, plan=ami.PLAN_TREE).cpu().numpy()
    check_parity(tree[0], truth, S, label=name + " tree")
    # several temperatures and frequencies (one of them continued to the real axis)
    z = np.array([[1j * math.pi / 5.0], [0.3 + 0.1j], [3j * math.pi / 5.0]])
    betas = (5.0, 2.0)
    grid = tab.evaluate(e[:, :96].contiguous(), z, betas).cpu().numpy()
    for b, beta in enumerate(betas):
        truth, S = ot.evaluate(e_rows[:96], z, beta, quad=False, threads=thr, want_S=True)
        check_parity(grid[b], truth, S, label=f"{name} grid beta={beta}")
    # a very cold and a very hot temperature through the leaf kernel and the parts (P12; quad truth on a few samples)
    nq = 24 if name == "o7" else 6
    cold = tab.evaluate(e[:, :nq].contiguous(), z[:2], (5000.0, 1e-3)).cpu().numpy()
    for b, beta in enumerate((5000.0, 1e-3)):
        truth, S = ot.evaluate(e_rows[:nq], z[:2], beta, quad=True, threads=thr, want_S=True)
        check_parity(cold[b], truth, S, label=f"{name} beta={beta}")
    # a batch larger than one chunk of the leaf array: same bits as the small batch on the shared samples,
    # and the streamed driver's tally (unfused here: the parts' results are added before they are summed)
    big = 70_000 + 13
    kb = tab.generate_momenta(cfg.seed, 0, big)
    ob = tab.evaluate_momenta(kb, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas)
    assert torch_mod.equal(ob[:, :, :n], out)
    tail = tab.evaluate_momenta(kb[big - 500:].contiguous(), [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas)
    assert torch_mod.equal(ob[:, :, big - 500:], tail)
    stats, sums = tab.run(5000 + 3, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, want_sum=True)
    ref = ob[:, :, :5003].sum(dim=2).cpu().numpy()
    assert np.max(np.abs(sums - ref)) <= 1e-12 * ob[:, :, :5003].abs().sum().item()


@pytest.mark.parametrize("name", ["o7", "stress8"])
def test_split_plan_complex_energies(ami, torch_mod, oracle_mod, name):
    """Complex energies on tables of split-plan size: leaf kernel, parts and combine kernel with every
    leaf a pair of doubles; a (temperature, frequency) grid with a cold temperature in it, two chunks of the leaf array,
    against the oracle (double precision as truth, as in test_split_plan_large_tables) and the table-driven kernel."""
    cfg = split_case(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.info["plan_kind"] == 2
    n = 96 + 5
    k = torch_mod.from_numpy(cfg.momenta(n)).cuda()
    e_real = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu).cpu().numpy()
    gam = A.uniform01(5, np.arange(e_real.size, dtype=np.uint64)).reshape(e_real.shape) * 0.05
    e_c = torch_mod.from_numpy(e_real - 1j * gam).cuda()
    z = np.array([[1j * math.pi / 5.0], [0.3 + 0.1j]])
    betas = (5.0, 300.0, 0.5)
    out = tab.evaluate(e_c, z, betas, e_reg=cfg.e_reg, plan=ami.PLAN_REG).cpu().numpy()
    assert out.shape == (3, 2, n) and np.isfinite(out).all()
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    e_rows = np.ascontiguousarray(e_c.cpu().numpy().T)
    thr = oracle_mod.hardware_threads()
    for b, beta in enumerate(betas):       # double truth on all samples at the moderate temperatures, quad on a few at all
        if beta < 100.0:
            truth, S = ot.evaluate(e_rows, z, beta, e_reg=cfg.e_reg, quad=False, threads=thr, want_S=True)
            check_parity(out[b], truth, S, label=f"{name} complex beta={beta}")
        nq = 20 if name == "o7" else 5          # quad truth costs 40 ms per sample and row at order 8
        truth, S = ot.evaluate(e_rows[:nq], z, beta, e_reg=cfg.e_reg, quad=True, threads=thr, want_S=True)
        check_parity(out[b][:, :nq], truth, S, label=f"{name} complex beta={beta} (quad)")
    flat = tab.evaluate(e_c[:, :16].contiguous(), z, betas[:1], e_reg=cfg.e_reg, plan=ami.PLAN_FLAT).cpu().numpy()
    truth, S = ot.evaluate(e_rows[:16], z, betas[0], e_reg=cfg.e_reg, quad=False, threads=thr, want_S=True)
    check_parity(flat[0], truth, S, label=f"{name} complex flat")
    # AUTO takes the same kernels; a batch of several leaf-array chunks gives the same bits on the shared samples
    big = 30_000 + 11
    eb = e_c.repeat(1, big // n + 1)[:, :big].contiguous()
    ob = tab.evaluate(eb, z, betas, e_reg=cfg.e_reg).cpu().numpy()
    assert np.array_equal(ob[:, :, :n], out) and np.array_equal(ob[:, :, n:2 * n], out)


def test_kernel_cache_on_disk(ami, torch_mod, tmp_path):
    """The compiled kernels are kept on disk (AMI_JIT_CACHE): a second process on the same diagram loads them
    without compiling -- reported by ami_table_info -- and returns the same bits; AMI_JIT_CACHE=0 compiles."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = """
import sys, numpy as np, torch
import ami_inputs as A, paper_2311_17189_b200 as P
cfg = A.get_config('cfg4'); n = 1000 + 29
tab = P.AmiTable.from_diagram(cfg.diagram)
info = tab.specialize()
k = tab.generate_momenta(cfg.seed, 0, n)
out = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=P.PLAN_REG).cpu().numpy()
np.save(sys.argv[1], out)
print('CACHED', info['specialize_cached'], 'MS', info['specialize_ms'])
"""
    cache = str(tmp_path / "jitcache")
    runs = []
    for i, env in enumerate(({"AMI_JIT_CACHE": cache}, {"AMI_JIT_CACHE": cache}, {"AMI_JIT_CACHE": "0"})):
        path = str(tmp_path / f"out{i}.npy")
        r = subprocess.run([sys.executable, "-c", code, path], capture_output=True, text=True, cwd=root, timeout=600,
                           env=dict(os.environ, **env))
        assert r.returncode == 0, r.stderr[-3000:]
        words = r.stdout.split()
        runs.append((int(words[words.index("CACHED") + 1]), float(words[words.index("MS") + 1]), np.load(path)))
    assert [r[0] for r in runs] == [0, 1, 0]
    assert os.listdir(cache)
    assert runs[1][1] < 250.0 and runs[1][1] < 0.5 * runs[0][1]      # milliseconds instead of an NVRTC compile
    assert np.array_equal(runs[0][2], runs[1][2]) and np.array_equal(runs[0][2], runs[2][2])


@pytest.mark.parametrize("dim,band", [(1, 0), (3, 0), (2, 1), (3, 1)])
def test_fused_lattice_variants(ami, torch_mod, oracle_mod, dim, band):
    """ami_evaluate_momenta_lattice and ami_run(dim, band): other dimensions and the free-particle band (Eq. 14,
    PAPER.md:346; :295) in ONE specialised kernel, bit-identical to ami_dispersion_lattice + ami_evaluate, momenta
    drawn in the kernel included; values against the oracle from the oracle's own quad dispersion."""
    from ami_inputs.rng import momenta
    cfg = A.get_config("cfg3")
    n = 3000 + 5
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    seed = cfg.seed + 11 * dim + band
    k_host = momenta(seed, n, cfg.diagram.n_int, d=dim)
    k = torch_mod.from_numpy(k_host).cuda()
    q = np.array([0.5 * math.pi, -0.25 * math.pi, 1.0][:dim])
    t, mu = (1.0, -0.2) if band == 0 else (0.5, 1.5)
    e = tab.dispersion(k, [q], t, mu, dim=dim, band=band)
    two = tab.evaluate(e, cfg.z_ext, cfg.betas, plan=ami.PLAN_REG)
    e_out = torch_mod.zeros_like(e)
    one = tab.evaluate_momenta(k, [q], t, mu, cfg.z_ext, cfg.betas, plan=ami.PLAN_REG, dim=dim, band=band, e_out=e_out)
    assert tab.refresh_info()["reg_plan_status"] == 0
    assert torch_mod.equal(one, two) and torch_mod.equal(e_out, e)
    gen = tab.generate_momenta(seed, 0, n, dim=dim)
    assert torch_mod.equal(gen, k)
    d_out = torch_mod.zeros_like(one)
    stats, sums = tab.run(n, [q], t, mu, cfg.z_ext, cfg.betas, seed=seed, d_out=d_out, want_sum=True, chunk=1024,
                          dim=dim, band=band)
    assert torch_mod.equal(d_out, one)
    assert np.max(np.abs(sums - one.sum(dim=2).cpu().numpy())) <= 1e-12 * one.abs().sum().item()
    flat = tab.evaluate_momenta(k, [q], t, mu, cfg.z_ext, cfg.betas, plan=ami.PLAN_FLAT, dim=dim, band=band)   # workspace inside
    assert torch_mod.equal(flat, tab.evaluate(e, cfg.z_ext, cfg.betas, plan=ami.PLAN_FLAT))
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    truth, S = ot.evaluate(np.ascontiguousarray(e.cpu().numpy().T), cfg.z_ext, cfg.betas[0], quad=True,
                           threads=oracle_mod.hardware_threads(), want_S=True)
    check_parity(one.cpu().numpy()[0], truth, S, label=f"fused dim={dim} band={band}")


# ------------------------------------------------------------------ S4 streamed driver
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg5"])
def test_run_draws_momenta_in_kernel_bitwise(ami, torch_mod, name):
    """ami_run with a seed and the register plan draws the momenta inside the evaluation kernel (they never exist in
    memory): same bits as feeding the host generator's momenta (P22) through the same driver, across chunk borders
    and a non-zero first sample; the table-driven plan, which generates them with momenta_kernel, agrees too."""
    cfg = A.get_config(name)
    n, first = (3000 + 41, 777) if name != "cfg5" else (600 + 5, 12345)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    nb, nf = len(cfg.betas), len(cfg.z_ext)
    outs = []
    for kw in ({"seed": cfg.seed, "first_sample": first},
               {"h_k": np.ascontiguousarray(cfg.momenta(n, start=first).reshape(n, -1))}):
        d_out = torch_mod.zeros((nb, nf, n), dtype=torch_mod.complex128, device="cuda")
        l0 = ami.kernel_launches()
        stats, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, chunk=1024, d_out=d_out,
                              want_sum=True, **kw)
        outs.append((d_out.cpu().numpy(), sums, ami.kernel_launches() - l0))
    assert tab.refresh_info()["reg_plan_status"] == 0
    assert np.array_equal(outs[0][0], outs[1][0], equal_nan=True)
    assert np.array_equal(outs[0][1], outs[1][1], equal_nan=True)
    assert outs[0][2] == outs[1][2]                  # no generation launches: evaluate + two tally kernels per chunk
    flat = torch_mod.zeros((nb, nf, n), dtype=torch_mod.complex128, device="cuda")
    tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, chunk=1024, d_out=flat, seed=cfg.seed,
            first_sample=first, plan=ami.PLAN_FLAT)
    ref = outs[0][0]
    scale = np.abs(ref).max(axis=-1, keepdims=True)
    assert np.all(np.abs(flat.cpu().numpy() - ref) <= 1e-9 * scale)


def test_generated_momenta_bitwise(ami, torch_mod):
    """P22: device generator == host generator, bit for bit."""
    cfg = A.get_config("cfg4")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    k = tab.generate_momenta(cfg.seed, 12345, 5000).cpu().numpy()
    np.testing.assert_array_equal(k, cfg.momenta(5000, start=12345))


@pytest.mark.parametrize("mode", ["generated", "host", "device"])
def test_run_streamed_matches_stagewise(ami, torch_mod, oracle_mod, mode):
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n, chunk = 10_000 + 77, 3000   # 4 chunks, ragged tail
    k_host = cfg.momenta(n)
    ref = tab.evaluate(gpu_energies(torch_mod, tab, cfg, k_host), cfg.z_ext, cfg.betas)
    h_out = torch_mod.empty((1, 1, n), dtype=torch_mod.complex128).pin_memory()
    kw = {}
    if mode == "host":
        kw["h_k"] = torch_mod.from_numpy(k_host).pin_memory()
    elif mode == "device":
        kw["d_k"] = torch_mod.from_numpy(k_host).cuda()
    stats, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, chunk=chunk,
                          h_out=h_out, want_sum=True, **kw)
    assert stats["n_chunks"] == 4 and stats["kernel_launches"] >= 8
    assert stats["d2h_bytes"] == n * 16 + 32       # results + one row of (sum, sum of squares)
    assert stats["h2d_bytes"] == (n * 8 * 8 if mode == "host" else 0)
    np.testing.assert_array_equal(h_out.numpy(), ref.cpu().numpy())   # same kernels, same inputs
    total = ref.cpu().numpy().sum()
    assert abs(sums[0, 0] - total) <= 1e-12 * np.abs(ref.cpu().numpy()).sum()
    sq = ref.cpu().numpy()[0, 0]
    want_sq = np.array([np.sum(sq.real ** 2), np.sum(sq.imag ** 2)])
    assert np.all(np.abs(tab.last_sumsq[0, 0] - want_sq) <= 1e-12 * want_sq)   # Monte-Carlo error bar input
    # and against the oracle end to end on a subset
    sel = np.arange(0, n, 97)
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    e_rows = ot.dispersion(k_host[sel], [cfg.q], cfg.t, cfg.mu)
    truth, S = ot.evaluate(e_rows, cfg.z_ext, cfg.betas[0], quad=True, want_S=True)
    check_parity(h_out.numpy()[0][:, sel], truth, S, label="run")


@pytest.mark.parametrize("name,n", [("cfg1", 1), ("cfg1", 33), ("cfg3", 5000 + 19), ("cfg2_se", 4096 + 31), ("cfg5", 2500 + 3)])
def test_run_fused_tally(ami, torch_mod, name, n):
    """Register plan (cfg5: a grid of 256 rows): the evaluation kernel leaves per-warp partial sums and nothing else has to be
    stored.  Tally-only call == tally beside stored results == numpy sums of those results (ragged last warp,
    several chunks, several rows); the squares give the error bar.  Deterministic."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    nb, nf = len(cfg.betas), len(cfg.z_ext)
    kw = dict(e_reg=cfg.e_reg, seed=cfg.seed, first_sample=5, chunk=1000, want_sum=True)
    _, only = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, **kw)
    sq_only = tab.last_sumsq.copy()
    d_out = torch_mod.zeros((nb, nf, n), dtype=torch_mod.complex128, device="cuda")
    _, both = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, d_out=d_out, **kw)
    assert tab.refresh_info()["reg_plan_status"] == 0
    assert np.array_equal(only, both) and np.array_equal(sq_only, tab.last_sumsq)
    v = d_out.cpu().numpy()
    assert np.all(np.abs(only - v.sum(axis=-1)) <= 1e-12 * np.abs(v).sum(axis=-1))
    want_sq = np.stack([np.sum(v.real ** 2, axis=-1), np.sum(v.imag ** 2, axis=-1)], axis=-1)
    assert np.all(np.abs(sq_only - want_sq) <= 1e-12 * want_sq + 1e-300)
    _, again = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, **kw)
    assert np.array_equal(only, again)
    # the table-driven plan (results re-read by the tally kernels) agrees to rounding
    _, flat = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, plan=ami.PLAN_FLAT, **kw)
    assert np.all(np.abs(flat - only) <= 1e-9 * np.abs(v).sum(axis=-1))


@pytest.mark.parametrize("name,n,kw", [("cfg1", 20_000 + 7, {}), ("cfg3", 6000 + 1, {}), ("cfg3", 150_000 + 9, {"truth_every": 25}),
                                       ("cfg2_bubble", 9000 + 3, {"chunk": 2048}), ("cfg2_se", 5000, {"plan": "flat"})])
def test_run_tally_against_oracle_mean(ami, torch_mod, oracle_mod, name, n, kw):
    """The Monte-Carlo tally of S4 (the integrator averages the result rows) beside the ORACLE's mean
    and sums of squares of the same seeded samples, under rule (3) of the parity norm: the fused tally (per-warp
    partials, or per-thread sums when there is one row and the batch is large), the chunked one and the
    table-driven plan's.  With truth_every the oracle sees every k-th sample and the GPU the same subset through
    d_out, while the tally of the whole batch is checked against the GPU's own results to rounding."""
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    plan = PLANS[kw.get("plan", "auto")]
    every = kw.get("truth_every", 1)
    d_out = torch_mod.zeros((len(cfg.betas), len(cfg.z_ext), n), dtype=torch_mod.complex128, device="cuda") if every > 1 else None
    stats, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, seed=cfg.seed, want_sum=True,
                          chunk=kw.get("chunk", 0), plan=plan, d_out=d_out)
    sumsq = tab.last_sumsq.copy()
    only_stats, only = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, seed=cfg.seed,
                               want_sum=True, chunk=kw.get("chunk", 0), plan=plan)
    assert np.array_equal(only, sums) or every > 1       # with and without stored results: the same tally
    ot = oracle_mod.OracleTable.from_diagram(cfg.diagram)
    sel = np.arange(0, n, every)
    e_rows = ot.dispersion(cfg.momenta(n)[sel], [cfg.q], cfg.t, cfg.mu)
    for b, beta in enumerate(cfg.betas):
        truth, S = ot.evaluate(e_rows, cfg.z_ext, beta, e_reg=cfg.e_reg, quad=True, threads=oracle_mod.hardware_threads(),
                               want_S=True)
        if every > 1:
            got = d_out[b][:, torch_mod.from_numpy(sel).cuda()].cpu().numpy()
            check_parity(got, truth, S, label=f"{name} run subset")
            ref = d_out[b].sum(dim=1).cpu().numpy()
            assert np.all(np.abs(sums[b] - ref) <= 1e-12 * d_out[b].abs().sum(dim=1).cpu().numpy())
            continue
        mean_gpu, mean_truth = sums[b] / n, truth.mean(axis=1)
        assert np.all(np.abs(mean_gpu - mean_truth) <= 1e-10 * S.mean(axis=1)), (mean_gpu, mean_truth)
        well = S.mean(axis=1) <= 1e3 * np.abs(mean_truth)
        assert np.all(np.abs(mean_gpu - mean_truth)[well] <= 1e-10 * np.abs(mean_truth)[well])
        sq_truth = np.stack([(truth.real ** 2).sum(axis=1), (truth.imag ** 2).sum(axis=1)], axis=-1)
        assert np.all(np.abs(sumsq[b] - sq_truth) <= 1e-10 * (S ** 2).sum(axis=1)[:, None])


def test_run_workspace_across_plans_and_refusals(ami, torch_mod):
    """One table, the table-driven plan with a small chunk first and the specialised kernels with a larger chunk
    afterwards: the driver's workspace (energy buffer of the first call) must not be handed to the second, which
    forms its energies in registers.  A request with no destination at all is refused, not executed."""
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 20_000 + 3
    a = torch_mod.zeros((1, 1, n), dtype=torch_mod.complex128, device="cuda")
    b = torch_mod.zeros_like(a)
    tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, d_out=a, plan=ami.PLAN_FLAT, chunk=512)
    tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, d_out=b, plan=ami.PLAN_REG, chunk=8192)
    torch_mod.cuda.synchronize()
    ref = tab.evaluate_momenta(tab.generate_momenta(cfg.seed, 0, n), [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas)
    assert torch_mod.equal(b, ref)
    assert (a - b).abs().max().item() <= 1e-9 * b.abs().max().item()
    h_k = torch_mod.from_numpy(cfg.momenta(n).reshape(n, -1)).pin_memory()
    h_out = torch_mod.zeros((1, 1, n), dtype=torch_mod.complex128).pin_memory()
    st, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, h_k=h_k, h_out=h_out, chunk=1000)   # pipelined
    assert st["n_chunks"] == 21 and torch_mod.equal(h_out.cuda(), ref)
    with pytest.raises(ami.AmiError) as ei:
        tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed)       # nowhere to put anything
    assert ei.value.code == -1
    with pytest.raises(ami.AmiError):
        tab.run(n, [[0.1, 0.2, 0.3, 0.4]], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, d_out=a, dim=4)


def test_run_device_output_and_determinism(ami, torch_mod):
    cfg = A.get_config("cfg1")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 10_000
    d_out = torch_mod.empty((1, 1, n), dtype=torch_mod.complex128, device="cuda")
    s1, sum1 = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, chunk=1024, d_out=d_out,
                       want_sum=True)
    first = d_out.clone()
    s2, sum2 = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=cfg.seed, chunk=1024, d_out=d_out,
                       want_sum=True)
    assert torch_mod.equal(first, d_out) and sum1[0, 0] == sum2[0, 0]   # deterministic tallies
    assert s1["n_chunks"] == 10


@pytest.mark.parametrize("name,n", [("cfg1", 10_000), ("cfg4", 20_000 + 5), ("cfg5", 3000 + 1)])
def test_unordered_calls_keep_results_and_stream_order(ami, torch_mod, name, n):
    """AMI_PLAN_UNORDERED (include/ami.h): a run of calls declared independent gives bit for bit what the same calls
    give in plain stream order, and what is ordered after the run comes after all of it:
    (a) R batches with their own buffers, the first ordered, the rest flagged, read back by a torch kernel;
    (b) an UNFLAGGED call that overwrites the result buffer of the first flagged one wins (write after write);
    (c) a flagged call whose momenta a torch kernel writes just before it reads the new momenta (read after write
        across work that is not this library's);
    (d) the same inside one CUDA graph, replayed twice.  The energies from memory (ami_evaluate) likewise."""
    torch = torch_mod
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    assert tab.specialize()["plan_kind"] == 1
    R = 6
    U = ami.PLAN_UNORDERED
    ks = [tab.generate_momenta(cfg.seed, r * n, n) for r in range(R)]
    call = lambda k, out, flag: tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg,
                                                     plan=flag, out=out)
    shape = (len(cfg.betas), len(cfg.z_ext), n)
    want = [call(k, torch.empty(shape, dtype=torch.complex128, device="cuda"), 0) for k in ks]
    bits = lambda x: x.view(torch.float64)
    # (a)
    outs = [torch.zeros(shape, dtype=torch.complex128, device="cuda") for _ in range(R)]
    for rep in range(3):
        for r in range(R):
            call(ks[r], outs[r], U if r else 0)
    total = torch.stack([bits(o) for o in outs]).clone()          # a torch kernel right behind the run
    assert torch.equal(total, torch.stack([bits(w) for w in want]))
    # (b)
    for o in outs:
        o.zero_()
    call(ks[0], outs[0], 0)
    call(ks[1], outs[1], U)
    call(ks[2], outs[2], U)
    call(ks[3], outs[1], 0)            # reuse of outs[1]: issued without the flag
    assert torch.equal(bits(outs[1]), bits(want[3])) and torch.equal(bits(outs[2]), bits(want[2]))
    # (c)
    k_var = torch.zeros_like(ks[0])
    for r in (4, 5, 4):
        k_var.copy_(ks[r])                                        # not a kernel of this library: full stream order
        call(k_var, outs[r], U)
    assert torch.equal(bits(outs[4]), bits(want[4])) and torch.equal(bits(outs[5]), bits(want[5]))
    # (d)
    for o in outs:
        o.zero_()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for i in range(2 * R):
            call(ks[i % R], outs[i % R], U if i % R else 0)
    for rep in range(2):
        g.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(bits(o), bits(w)) for o, w in zip(outs, want))
    # energies from memory
    es = [tab.dispersion(k, [cfg.q], cfg.t, cfg.mu) for k in ks[:3]]
    ev = lambda e, out, flag: tab.evaluate(e, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=flag, out=out)
    want_e = [ev(e, torch.empty(shape, dtype=torch.complex128, device="cuda"), 0) for e in es]
    for r in range(3):
        outs[r].zero_()
        ev(es[r], outs[r], U if r else 0)
    assert all(torch.equal(bits(outs[r]), bits(want_e[r])) for r in range(3))
    # the table-driven plans accept the flag and stay ordered; ami_run refuses it
    flat = tab.evaluate_momenta(ks[0], [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=PLANS["flat"] | U,
                                e_out=torch.empty((cfg.diagram.n_eps, n), dtype=torch.float64, device="cuda"))
    ref = tab.evaluate_momenta(ks[0], [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=PLANS["flat"],
                               e_out=torch.empty((cfg.diagram.n_eps, n), dtype=torch.float64, device="cuda"))
    assert torch.equal(bits(flat), bits(ref))
    with pytest.raises(ami.AmiError):
        tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, seed=1, want_sum=True, plan=U)


def test_run_default_chunking_and_workspace_reuse(ami, torch_mod):
    """ami_run with host buffers and the library's default chunk (2^17 samples): several chunks on two
    streams, the cached workspace reused and grown across calls of different sizes and row counts."""
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    for n, z, betas in ((300_000 + 17, cfg.z_ext, cfg.betas), (50_000, np.array([[1j], [0.5 + 0.2j]]), (2.0, 8.0, 9.0)),
                        (400_000, cfg.z_ext, cfg.betas)):
        k_host = cfg.momenta(n)
        h_k = torch_mod.from_numpy(k_host.reshape(n, -1)).pin_memory()
        h_out = torch_mod.empty((len(betas), len(z), n), dtype=torch_mod.complex128).pin_memory()
        stats, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, z, betas, h_k=h_k, h_out=h_out)
        assert stats["n_chunks"] == -(-n // (1 << 17))
        assert stats["h2d_bytes"] == n * 8 * 8 and stats["d2h_bytes"] == n * 16 * len(betas) * len(z)
        ref = tab.evaluate_momenta(torch_mod.from_numpy(k_host).cuda(), [cfg.q], cfg.t, cfg.mu, z, betas)
        assert np.array_equal(h_out.numpy(), ref.cpu().numpy())


@pytest.mark.parametrize("plan", list(PLANS))
def test_two_external_slots_sum_order_and_prefactor(ami, torch_mod, oracle_mod, plan):
    """The ABI beyond the graded configs: two external frequency slots (the external frequency split
    into a fermionic and a bosonic part, one of them exactly zero in one row: regulator rule P10(b) needs
    ALL of a denominator's external values to vanish), a non-default order of the sums, a prefactor."""
    base = A.get_config("cfg3")
    d = base.diagram
    alpha2 = np.concatenate([d.alpha, d.alpha[:, -1:]], axis=1)          # external column twice
    stat2 = np.concatenate([d.slot_is_fermionic, [0]]).astype(np.uint8)  # fermionic + bosonic
    order = [2, 0, 3, 1]
    tab = ami.AmiTable(d.n_int, 2, alpha2, d.eps, stat2, sum_order=order, prefactor=-0.5)
    ot = oracle_mod.OracleTable(d.n_int, 2, alpha2, d.eps, stat2, sum_order=order, prefactor=-0.5)
    n = 2000 + 9
    k_host = base.momenta(n)
    k = torch_mod.from_numpy(k_host).cuda()
    q2 = [base.q, (0.0, 0.0)]                     # the second slot carries no momentum
    beta = 4.0
    z = np.array([[1j * math.pi / beta, 2j * math.pi / beta], [1j * math.pi / beta, 0j], [0.3 + 0.1j, -0.1 + 0.2j]])
    out = tab.evaluate_momenta(k, q2, base.t, base.mu, z, [beta], e_reg=1e-8, plan=PLANS[plan]).cpu().numpy()
    e_rows = ot.dispersion(k_host, q2, base.t, base.mu)
    truth, S = ot.evaluate(e_rows, z, beta, e_reg=1e-8, quad=True, threads=oracle_mod.hardware_threads(), want_S=True)
    check_parity(out[0], truth, S, label="two external slots")
    # same physics as one slot carrying the sum of the two values
    one = ami.AmiTable.from_diagram(d, sum_order=order, prefactor=-0.5)
    ref = one.evaluate_momenta(k, [base.q], base.t, base.mu, z.sum(axis=1, keepdims=True)[[0, 2]], [beta], e_reg=1e-8,
                               plan=PLANS[plan]).cpu().numpy()
    scale = np.abs(ref[0]).max(axis=1, keepdims=True)
    assert np.all(np.abs(out[0][[0, 2]] - ref[0]) <= 1e-9 * scale)


@pytest.mark.parametrize("plan", list(PLANS))
def test_fused_call_with_soa_momenta(ami, torch_mod, plan):
    """ami_evaluate_momenta through the raw ABI with SoA momenta [2m][N] (strides 1, N): same bits as
    the Eq.-8 layout."""
    import ctypes as C
    cfg = A.get_config("cfg3")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n = 3000 + 5
    k = torch_mod.from_numpy(cfg.momenta(n)).cuda()
    ref = tab.evaluate_momenta(k, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, plan=PLANS[plan])
    ksoa = k.reshape(n, -1).t().contiguous()
    out = torch_mod.empty_like(ref)
    e_ws = torch_mod.empty((cfg.diagram.n_eps, n), dtype=torch_mod.float64, device="cuda")
    q = np.array(cfg.q)
    z = np.ascontiguousarray(cfg.z_ext, dtype=np.complex128)
    b = np.array(cfg.betas, dtype=np.float64)
    rc = ami.lib().ami_evaluate_momenta(tab._h, C.c_void_p(ksoa.data_ptr()), 1, n, q.ctypes.data, cfg.t, cfg.mu, n,
                                        z.ctypes.data, len(z), b.ctypes.data, len(b), 0.0, PLANS[plan],
                                        C.c_void_p(e_ws.data_ptr()), C.c_void_p(out.data_ptr()),
                                        C.c_void_p(torch_mod.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch_mod.cuda.synchronize()
    assert torch_mod.equal(out, ref)


def test_argument_errors_and_empty_requests(ami, torch_mod):
    """Error codes instead of crashes: bad plan, missing buffers; empty grids and batches are no-ops."""
    import ctypes as C
    cfg = A.get_config("cfg1")
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    L = ami.lib()
    e = torch_mod.zeros((cfg.diagram.n_eps, 8), dtype=torch_mod.float64, device="cuda")
    out = torch_mod.zeros((1, 1, 8), dtype=torch_mod.complex128, device="cuda")
    z = np.ascontiguousarray(cfg.z_ext, dtype=np.complex128)
    b = np.array(cfg.betas)
    st = C.c_void_p(torch_mod.cuda.current_stream().cuda_stream)

    def call(plan=0, d_e=e.data_ptr(), d_out=out.data_ptr(), n_e=8, n_f=1, n_b=1, zp=z.ctypes.data, bp=b.ctypes.data):
        return L.ami_evaluate(tab._h, C.c_void_p(d_e), 0, n_e, zp, n_f, bp, n_b, 0.0, plan, C.c_void_p(d_out), st)

    assert call() == 0
    assert call(plan=7) == -1 and call(plan=-1) == -1              # AMI_EINVAL
    assert call(d_out=None) == -1 and call(d_e=None) == -1
    assert call(n_e=-1) == -1 and call(n_f=-2) == -1
    assert call(zp=None) == -1 and call(bp=None) == -1
    assert call(n_e=0) == 0 and call(n_f=0, zp=None) == 0 and call(n_b=0, bp=None) == 0   # nothing to do
    assert L.ami_evaluate(None, None, 0, 0, None, 0, None, 0, 0.0, 0, None, st) == -1
    stats, sums = tab.run(0, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, want_sum=True)
    assert stats["n_chunks"] == 0 and sums[0, 0] == 0
    with pytest.raises(ami.AmiError):
        tab.run(10, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, h_k=np.zeros((10, 4)), d_k=torch_mod.zeros((10, 4), dtype=torch_mod.float64, device="cuda"))
    torch_mod.cuda.synchronize()


@pytest.mark.parametrize("plan", list(PLANS))
@pytest.mark.parametrize("name,n,crit", [("cfg3", 20_000 + 7, 0), ("cfg5", 300 + 1, 1), ("cfg3", 5000, 1)])
def test_searched_sum_order(ami, torch_mod, oracle_mod, name, n, crit, plan):
    """Tables built in the order ami_search_sum_order picks: parity against the oracle
    summing in that same order, and the same numbers as the default order within both tolerances."""
    cfg = A.get_config(name)
    order, best, dflt, _ = ami.search_sum_order(cfg.diagram, crit)
    assert best <= dflt
    run_eval_case(ami, torch_mod, oracle_mod, cfg, n, PLANS[plan], sum_order=order, n_truth=150 if name == "cfg5" else None)


@pytest.mark.parametrize("plan", list(PLANS))
def test_diagram_file_to_values(ami, torch_mod, oracle_mod, plan):
    """Fig. 2's diagram file through read_graph -> label_graph -> ami_construct ->
    fused evaluation, against the oracle constructed from the same labels."""
    import os
    import types
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fig2_o2_g0_n0.graph")
    lab = ami.label_graph(ami.read_graph(path))
    base = A.get_config("cfg1")
    n = 6000 + 1
    tab = ami.AmiTable.from_diagram(lab)
    k = base.momenta(n)
    out = tab.evaluate_momenta(torch_mod.from_numpy(k).cuda(), [base.q], base.t, base.mu, base.z_ext, base.betas,
                               plan=PLANS[plan]).cpu().numpy()
    ot = oracle_mod.OracleTable(lab.n_int, lab.n_ext, lab.alpha, lab.eps, lab.slot_is_fermionic)
    e = ot.dispersion(k, [base.q], base.t, base.mu, quad=False)
    truth, S = ot.evaluate(e, base.z_ext, base.betas[0], quad=True, want_S=True)
    check_parity(out[0], truth, S, label="fig2 diagram file")
