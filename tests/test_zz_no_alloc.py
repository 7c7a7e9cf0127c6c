"""ami_tally_static, the allocation-free entry point (include/ami.h): its tally of device-resident results beside
the one ami_run forms for the same seeded samples (the existing path: partial sums in a cudaMalloc'ed workspace, or
inside the evaluation kernel), within the bound the other tally tests use.  Two calls in a row on the same static
workspace, the second smaller than the first so that stale partial sums and counters lie behind it.

The file sorts last on purpose (the suite runs with pytest -x): it passes alone in a fresh process -- the first
call then does the set-up -- and after the other GPU tests."""
import numpy as np
import pytest

import ami_inputs as A

pytestmark = pytest.mark.gpu

TOL = 1e-12      # of sum |v| resp. sum |v|^2, as test_run_tally_against_oracle_mean compares two GPU sums


@pytest.fixture(scope="module")
def ami():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    pkg.lib()  # raises if the extension is missing: no fallback
    return pkg


def run_and_tally(ami, torch, name, n, poison):
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram)
    n_b, n_f = len(cfg.betas), len(cfg.z_ext)
    d_out = torch.zeros((n_b, n_f, n), dtype=torch.complex128, device="cuda")
    _, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, seed=cfg.seed, want_sum=True,
                      d_out=d_out)
    sumsq = tab.last_sumsq.copy()
    tally = torch.full((n_b * n_f, 4), poison, dtype=torch.float64, device="cuda")
    free_before = torch.cuda.mem_get_info()[0]
    ami.tally_static(d_out, tally)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    got = tally.cpu().numpy().reshape(n_b, n_f, 4)
    a = d_out.abs()
    s1 = a.sum(dim=2).cpu().numpy()
    s2 = (a * a).sum(dim=2).cpu().numpy()
    assert np.all(np.isfinite(got)), f"{name}: rows left unwritten"
    assert np.all(np.abs(got[..., 0] - sums.real) <= TOL * s1), (name, got[..., 0], sums.real)
    assert np.all(np.abs(got[..., 1] - sums.imag) <= TOL * s1), (name, got[..., 1], sums.imag)
    assert np.all(np.abs(got[..., 2:] - sumsq) <= TOL * s2[..., None]), (name, got[..., 2:], sumsq)
    return got, d_out, free_before - free_after


def test_tally_static_matches_run_tally_on_two_calls_in_a_row(ami):
    import torch
    # 256 rows (4 temperatures x 64 frequencies) of 20 003 samples, then ONE row of 300 001: the second call uses
    # fewer counters and a different number of partial sums per row than what the first left in the array
    first, d_first, _ = run_and_tally(ami, torch, "cfg5", 20_003, float("nan"))
    second, d_second, grew = run_and_tally(ami, torch, "cfg3", 300_001, float("inf"))
    assert grew == 0, f"device memory in use grew by {grew} bytes across a call that must not allocate"
    # again on the first input: same bits as before (fixed order of the sums, nothing of the call in between is read)
    tally = torch.empty((d_first.shape[0] * d_first.shape[1], 4), dtype=torch.float64, device="cuda")
    ami.tally_static(d_first, tally)
    assert np.array_equal(tally.cpu().numpy().reshape(first.shape), first)
    # an empty batch gives zeros, and set-up alone is a valid call
    ami.tally_static_setup(0)
    empty = torch.zeros((3, 0), dtype=torch.complex128, device="cuda")
    t3 = torch.full((3, 4), 7.0, dtype=torch.float64, device="cuda")
    ami.tally_static(empty, t3)
    assert torch.count_nonzero(t3).item() == 0


def test_tally_static_refuses_sizes_beyond_its_workspace(ami):
    import torch
    rows = ami.TALLY_STATIC_MAX_ROWS + 1
    vals = torch.zeros((rows, 8), dtype=torch.complex128, device="cuda")
    tally = torch.full((rows, 4), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(ami.AmiError) as err:
        ami.tally_static(vals, tally)
    assert err.value.code == -6 and "1024 rows" in str(err.value), err.value
    torch.cuda.synchronize()
    assert torch.all(tally == -1.0).item()            # nothing was launched
    # the limit itself is accepted
    ok = torch.ones((ami.TALLY_STATIC_MAX_ROWS, 8), dtype=torch.complex128, device="cuda")
    t = torch.empty((ami.TALLY_STATIC_MAX_ROWS, 4), dtype=torch.float64, device="cuda")
    ami.tally_static(ok, t)
    want = torch.tensor([8.0, 0.0, 8.0, 0.0], dtype=torch.float64, device="cuda").expand_as(t)
    assert torch.equal(t, want)
