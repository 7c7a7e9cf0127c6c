"""CPU tests of the register plan's generator: the specialised kernels of every graded config are
generated and compiled to an sm_100a cubin with NVRTC (no GPU needed), the plan's instruction counts
are consistent, and tables outside the limits are refused."""
import pytest

import ami_inputs as A


@pytest.fixture(scope="module")
def ami():
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    return pkg


@pytest.mark.parametrize("name", ["cfg1", "cfg2_bubble", "cfg2_bubble_doubled", "cfg3", "cfg4", "cfg5"])
def test_specialised_kernels_compile_for_sm100a(ami, name):
    cfg = A.get_config(name)
    tab = ami.AmiTable.from_diagram(cfg.diagram, device=None)
    info = tab.info
    assert info["reg_plan_status"] == 1
    src = tab.kernel_source()
    assert 'extern "C" __global__' in src and "ami_jit_eval" in src and "ami_jit_fused" in src
    assert "oracle" not in src                       # the product shares nothing with the oracle
    for u in range(info["n_fermi_leaves"]):
        assert f"F{u} = " in src
    try:
        cubin, log = tab.kernel_cubin()
    except ami.AmiError as e:
        if e.code == -6:
            pytest.skip("NVRTC library not available on this machine")
        raise
    assert cubin[:4] == b"\x7fELF" and len(cubin) > 10_000
    assert "ami_jit_fused" in log and "registers" in log
    # counts reported for the roofline: Horner plan far below the flat loop, parts add up
    assert 0 < info["fp64_ops_tree"] < info["fp64_ops_flat"]
    assert 0 <= info["fp64_ops_tree_fermi"] <= info["fp64_ops_tree"]
    assert info["fp64_ops_leaf_fermi"] >= 16 and info["fp64_ops_dispersion"] >= 32 * info["n_eps"]   # >= one exponential; two cosines per symbol


def test_generated_source_is_deterministic(ami):
    cfg = A.get_config("cfg3")
    a = ami.AmiTable.from_diagram(cfg.diagram, device=None).kernel_source()
    b = ami.AmiTable.from_diagram(cfg.diagram, device=None).kernel_source()
    assert a == b


def test_hash_consing_shares_sums_across_groups(ami):
    """Order 6: the FT sums as one DAG need several times fewer instructions than the flat Fermi
    products (688 terms x 6 factors)."""
    info = ami.AmiTable.from_diagram(A.get_config("cfg4").diagram, device=None).info
    assert info["n_terms"] == 688 and info["n_groups"] == 48
    assert info["fp64_ops_tree"] * 20 < info["fp64_ops_flat"]


def test_order8_is_a_split_plan(ami):
    """Order 8 (T = 40244): too large for one register-resident kernel, specialised as a split plan of several
    translation units -- leaf and combine kernels first, then the parts -- each of which compiles in seconds."""
    tab = ami.AmiTable.from_diagram(A.get_config("stress8").diagram, device=None)
    assert tab.info["reg_plan_status"] == 1 and tab.info["plan_kind"] == 2
    assert ami.AmiTable.from_diagram(A.get_config("cfg4").diagram, device=None).info["plan_kind"] == 1
    units = tab.kernel_units()
    assert 2 <= units <= 9
    src = tab.kernel_source()
    for name in ("ami_split_leaves_eval", "ami_split_leaves_fused", "ami_split_parts", "ami_split_combine", "ami_part_0"):
        assert name in src
    assert src.count("translation unit") == units
    try:
        cubin, log = tab.kernel_cubin(unit=units - 1)
    except ami.AmiError as e:
        if e.code == -6:
            pytest.skip("NVRTC library not available on this machine")
        raise
    assert cubin[:4] == b"\x7fELF" and "ami_split_parts" in log
    with pytest.raises(ami.AmiError):      # and no kernel entry point works without a device copy
        tab.specialize()


@pytest.mark.parametrize("kw", [{"complex_energies": True}, {"dim": 1}, {"dim": 3, "band": 1}])
def test_kernel_variants_compile(ami, kw):
    """The kernels are generated per variant -- complex energies, momenta of 1-3 components and either
    band (Eq. 14) -- and each compiles for sm_100a."""
    tab = ami.AmiTable.from_diagram(A.get_config("cfg3").diagram, device=None)
    src = tab.kernel_source(**kw)
    assert src != tab.kernel_source()
    if kw.get("complex_energies"):
        assert "sincos(" in src and "ami_jit_fused" not in src and "Fr0" in src      # momenta give real energies
    else:
        assert ("kz0" in src) == (kw["dim"] == 3) and ("cos_bounded_n" in src.split("ami_jit_fused")[-1]) == (kw.get("band", 0) == 0)
    try:
        cubin, log = tab.kernel_cubin(**kw)
    except ami.AmiError as e:
        if e.code == -6:
            pytest.skip("NVRTC library not available on this machine")
        raise
    assert cubin[:4] == b"\x7fELF" and "ami_jit_eval" in log
    if kw.get("complex_energies"):     # tables of split-plan size: leaf kernel for energies from memory only, leaves in pairs
        big = ami.AmiTable.from_diagram(A.random_self_energy(7, 0), device=None)
        src = big.kernel_source(**kw)
        assert "ami_split_leaves_eval" in src and "ami_split_leaves_fused" not in src and "#define Fi" in src
        cubin, log = big.kernel_cubin(unit=big.kernel_units() - 1, **kw)
        assert cubin[:4] == b"\x7fELF" and "ami_split_parts" in log


def test_register_plan_can_be_switched_off():
    """AMI_DISABLE_JIT=1: every table reports the register plan as unavailable, so AMI_PLAN_AUTO runs
    the table-driven kernels (checked in a fresh process: the switch is read per call)."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = ("import ami_inputs as A, paper_2311_17189_b200 as P;"
            "t = P.AmiTable.from_diagram(A.get_config('cfg3').diagram, device=None);"
            "print(t.info['reg_plan_status'])")
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, cwd=root,
                         env=dict(os.environ, AMI_DISABLE_JIT="1"), timeout=120)
    assert out.returncode == 0, out.stderr
    assert out.stdout.strip() == "-6"


def test_inspect_kernels_reports_register_operands():
    """The inspection tool's operand classes (register-file ceiling) on the smallest table: every FP64
    instruction is classified with 0-3 distinct register operands, most polynomial steps read two."""
    import ami_inputs as A
    import paper_2311_17189_b200 as pkg
    from paper_2311_17189_b200 import inspect_kernels as ik
    tab = pkg.AmiTable.from_diagram(A.get_config("cfg1").diagram, device=None)
    cubin, _ = tab.kernel_cubin()
    hist, classes = ik.histogram(cubin), ik.operand_classes(cubin)
    assert set(hist) == set(classes) and "ami_jit_fused" in classes
    c = classes["ami_jit_fused"]
    n_fp = sum(c["fp64"].values())
    assert n_fp == sum(hist["ami_jit_fused"][o] for o in ("DFMA", "DMUL", "DADD", "DSETP")) > 100
    assert all(0 <= k[2] <= k[1] <= 3 for k in c["fp64"])
    two = sum(v for k, v in c["fp64"].items() if k[1] <= 2)
    assert two > 0.6 * n_fp and c["other"] > 0


def test_instruction_counts_of_the_several_temperature_body():
    """ami_info.fp64_ops_mb_prefix / fp64_ops_mb_sum (the roofline numerator of launches with several temperatures) are
    the multiplications and fused multiply-adds the generator writes: the prefix products once per frequency, and the
    sum of the one-temperature block per (frequency, temperature).  cfg5 takes the prefix-product form, cfg4 keeps the
    Horner form (prefix = 0, sum = the R part of fp64_ops_tree)."""
    import re
    import ami_inputs as A
    import paper_2311_17189_b200 as pkg
    ops = lambda text: text.count("fma(") + len(re.findall(r"= -?\w+ \* \w+;", text))
    tab = pkg.AmiTable.from_diagram(A.get_config("cfg5").diagram, device=None)
    info, src = tab.info, tab.kernel_source()
    body = src[src.index("void ami_body_mb"):]
    prefix = body[body.index("const double P"):body.index("int b0 = 0;")]      # first prefix product .. the blocks
    one = body[body.index("if (b0 < p.n_b)"):body.index("\n}\n", body.index("if (b0 < p.n_b)"))]
    assert info["fp64_ops_mb_prefix"] == ops(prefix) > 0
    # the block of one temperature spreads its terms over four partial sums: three more additions than counted
    assert info["fp64_ops_mb_sum"] == ops(one) > 0
    assert info["fp64_ops_mb_prefix"] + 2 * info["fp64_ops_mb_sum"] <= 2 * (info["fp64_ops_tree"] - info["fp64_ops_tree_fermi"])
    tab4 = pkg.AmiTable.from_diagram(A.get_config("cfg4").diagram, device=None)
    i4 = tab4.info
    assert i4["fp64_ops_mb_prefix"] == 0 and i4["fp64_ops_mb_sum"] == i4["fp64_ops_tree"] - i4["fp64_ops_tree_fermi"]
    assert "int b0 = 0;" not in tab4.kernel_source()
