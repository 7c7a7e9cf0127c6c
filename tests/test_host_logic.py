"""CPU-only tests of the product's host logic: the C-ABI library loads and exports every symbol
include/ami.h declares, ami_construct builds tables whose VALUES (not shape: tables are not
unique, reading P14) agree with the oracle, error codes, and no compute without a device."""
import math
import os
import re

import numpy as np
import pytest

import ami_inputs as A

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ami():
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    return pkg


def test_library_exports_every_declared_symbol(ami):
    header = open(os.path.join(ROOT, "include", "ami.h")).read()
    declared = set(re.findall(r"^\s*(?:int|int64_t|void|const char\*)\s+(ami_\w+)\s*\(", header, flags=re.M))
    assert declared == set(ami.EXPORTS), declared ^ set(ami.EXPORTS)
    L = ami.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert L.ami_version() >= 1


C_CALLER = r"""
/* A caller written in C99: the header must be valid C and the library usable without C++ or Python. */
#include <stdio.h>
#include <string.h>
#include "ami.h"

int main(void) {
  /* order-2 self-energy (PAPER.md:207-231): R0 = three lines, alpha = (1,0,0), (0,1,0), (1,-1,1), external last */
  const int32_t alpha[9] = {1, 0, 0, 0, 1, 0, 1, -1, 1};
  const int32_t eps[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  const uint8_t fermionic[3] = {1, 1, 1};
  ami_table* tab = NULL;
  ami_info info;
  size_t bytes = 0;
  int rc = ami_construct(2, 1, 3, 3, alpha, eps, fermionic, NULL, 1.0, -1, &tab);
  if (rc != AMI_OK) { printf("construct: %s\n", ami_strerror(rc)); return 1; }
  memset(&info, 0, sizeof info);
  rc = ami_table_info(tab, &info);
  if (rc != AMI_OK) return 2;
  if (ami_table_latex(tab, NULL, &bytes) != AMI_OK || bytes == 0) return 3;
  /* a table without a device copy refuses the kernels: no CPU fallback */
  rc = ami_evaluate(tab, NULL, 0, 1, NULL, 0, NULL, 0, 0.0, AMI_PLAN_AUTO | AMI_PLAN_UNORDERED, NULL, NULL);
  printf("version %d terms %lld U_F %d U_D %d has_device_copy %d evaluate_without_device %d max_rows %d\n", ami_version(),
         (long long)info.n_terms, (int)info.n_fermi_leaves, (int)info.n_den_leaves, (int)info.has_device_copy, rc,
         AMI_TALLY_STATIC_MAX_ROWS);
  ami_table_destroy(tab);
  return 0;
}
"""


def test_header_is_c99_and_a_c_program_links(ami, tmp_path):
    """include/ami.h through a C compiler in pedantic C99 mode, and a caller written in C linked against the
    library (host-only table: runs without a GPU)."""
    import subprocess
    src = tmp_path / "caller.c"
    src.write_text(C_CALLER)
    exe = tmp_path / "caller"
    lib_dir = os.path.dirname(ami.LIB_PATH)
    subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"),
                    str(src), "-o", str(exe), "-L", lib_dir, "-l:libami_b200.so", f"-Wl,-rpath,{lib_dir}"],
                   check=True, capture_output=True, text=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    m = re.match(r"version (\d+) terms (\d+) U_F (\d+) U_D (\d+) has_device_copy 0 evaluate_without_device (-?\d+) max_rows 1024", out)
    assert m, out
    tab = ami.AmiTable.from_diagram(A.self_energy_order2(), device=None)
    assert int(m.group(2)) == tab.info["n_terms"] and int(m.group(3)) == tab.info["n_fermi_leaves"]
    assert int(m.group(5)) == -4        # AMI_ECUDA: the table has no device copy


def numpy_eval_export(tab, e, z, beta, prefactor=1.0):
    """Evaluates an exported flat table with numpy (test-side restatement of the layout documented
    in include/ami.h; real energies, derivative order <= 1)."""
    def f_sig(E, sig):
        return 1.0 / (sig * np.exp(beta * E) + 1.0)

    F = []
    for c, sig, k in zip(tab["leafF_c"], tab["leafF_sig"], tab["leafF_k"]):
        E = e @ c
        f = f_sig(E, sig)
        F.append(f if k == 0 else -beta * f * (1 - f))
        assert k <= 1
    D = [1.0 / (e @ c + a @ z) for c, a in zip(tab["leafD_c"], tab["leafD_a"])]
    total = np.zeros(e.shape[0], dtype=complex)
    for fi, di, co in zip(tab["fidx"], tab["didx"], tab["coef"]):
        term = np.full(e.shape[0], co, dtype=complex)
        for u in fi:
            term = term * F[u]
        for u in di:
            if u >= 0:
                term = term * D[u]
        total += term
    return prefactor * total


DIAGRAMS = {
    "order1": A.order1_line, "bubble": A.bubble, "bubble_doubled": A.doubled_line_bubble,
    "se2": A.self_energy_order2, "se2_doubled1": lambda: A.self_energy_order2_doubled(1),
    "se3": lambda: A.random_self_energy(3, 1), "cfg3": lambda: A.get_config("cfg3").diagram,
    "se4_b": lambda: A.random_self_energy(4, 0), "cfg5": lambda: A.get_config("cfg5").diagram,
    "cfg4": lambda: A.get_config("cfg4").diagram,
}


@pytest.mark.parametrize("name", list(DIAGRAMS))
def test_construct_values_match_oracle(ami, oracle_mod, name):
    d = DIAGRAMS[name]()
    tab = ami.AmiTable.from_diagram(d, device=None, prefactor=-2.0)
    ex = tab.export()
    assert ex["fidx"].shape[1] == d.n_int
    rng = np.random.default_rng(3)
    e = rng.uniform(-1.5, 1.5, size=(24, d.n_eps))
    beta = 2.0
    z = np.array([1j * math.pi / beta if d.slot_is_fermionic[-1] else 2j * math.pi / beta])
    got = numpy_eval_export(ex, e, z, beta, prefactor=-2.0)
    want, S = oracle_mod.OracleTable.from_diagram(d, prefactor=-2.0).evaluate(e, [z], beta, quad=True, want_S=True)
    assert np.max(np.abs(got - want[0]) / S[0]) < 1e-12
    info = tab.info
    assert info["n_terms"] == len(ex["coef"]) and info["has_device_copy"] == 0
    assert info["n_terms"] <= info["n_terms_raw"]


def test_construct_sum_order_and_errors(ami, oracle_mod):
    d = A.random_self_energy(4, 1)
    rng = np.random.default_rng(5)
    e = rng.uniform(-1.5, 1.5, size=(16, d.n_eps))
    beta, z = 2.0, np.array([1j * math.pi / 2.0])
    ref = numpy_eval_export(ami.AmiTable.from_diagram(d, device=None).export(), e, z, beta)
    n_ok = 0
    for so in ([3, 2, 1, 0], [1, 3, 0, 2], [2, 0, 3, 1]):
        try:
            t = ami.AmiTable.from_diagram(d, device=None, sum_order=so)
        except ami.AmiError as ex:
            assert ex.code == -2
            with pytest.raises(oracle_mod.OracleError):  # the oracle rejects the same order
                oracle_mod.OracleTable.from_diagram(d, sum_order=so)
            continue
        np.testing.assert_allclose(numpy_eval_export(t.export(), e, z, beta), ref, rtol=1e-9)
        n_ok += 1
    assert n_ok >= 1
    o1 = A.order1_line()
    with pytest.raises(ami.AmiError) as ei:
        ami.AmiTable(1, 1, [[2, 0]], o1.eps, o1.slot_is_fermionic, device=None)
    assert ei.value.code == -2
    with pytest.raises(ami.AmiError) as ei:
        ami.AmiTable(2, 1, [[1, 0, 0]], o1.eps, [1, 1, 1], device=None)
    assert ei.value.code == -3
    with pytest.raises(ami.AmiError) as ei:
        ami.AmiTable(1, 1, [[1, 0]], o1.eps, [0, 1], device=None)  # bosonic internal sum
    assert ei.value.code == -1
    with pytest.raises(ami.AmiError) as ei:
        ami.AmiTable(2, 1, [[1, 0, 0], [0, 1, 0]], np.eye(2, dtype=np.int32), [1, 1, 1], sum_order=[0, 0], device=None)
    assert ei.value.code == -1


def test_search_sum_order(ami, oracle_mod):
    """ami_search_sum_order: the order it returns gives a table of the
    promised size, never larger than the default one, and the same values as the default order."""
    import itertools
    d = A.get_config("cfg3").diagram
    order, best, dflt, tried = ami.search_sum_order(d, ami.ORDER_FEWEST_TERMS)
    assert sorted(order) == list(range(d.n_int)) and 1 <= tried <= math.factorial(d.n_int)
    t_def = ami.AmiTable.from_diagram(d, device=None)
    t_best = ami.AmiTable.from_diagram(d, device=None, sum_order=order)
    assert t_def.info["n_terms"] == dflt and t_best.info["n_terms"] == best and best <= dflt
    sizes = []                                   # brute force over all orders through ami_construct
    for so in itertools.permutations(range(d.n_int)):
        try:
            sizes.append(ami.AmiTable.from_diagram(d, device=None, sum_order=list(so)).info["n_terms"])
        except ami.AmiError:
            pass
    assert len(sizes) == tried and min(sizes) == best
    rng = np.random.default_rng(11)
    e = rng.uniform(-1.5, 1.5, size=(16, d.n_eps))
    beta, z = 2.0, np.array([1j * math.pi / 2.0])
    want, S = oracle_mod.OracleTable.from_diagram(d).evaluate(e, [z], beta, quad=True, want_S=True)
    got = numpy_eval_export(t_best.export(), e, z, beta)
    assert np.max(np.abs(got - want[0]) / S[0]) < 1e-12
    # the operation-count criterion: consistent with ami_table_info of the table it picks
    order2, best2, dflt2, _ = ami.search_sum_order(d, ami.ORDER_FEWEST_OPS)
    i2 = ami.AmiTable.from_diagram(d, device=None, sum_order=order2).info
    assert best2 == i2["fp64_ops_tree"] + i2["fp64_ops_leaf_fermi"] + i2["fp64_ops_leaf_den"] + i2["fp64_ops_combos"]
    assert best2 <= dflt2
    # a cap of one order returns the default; bad arguments are refused
    assert ami.search_sum_order(d, 0, max_orders=1)[:2] == (list(range(d.n_int)), dflt)
    with pytest.raises(ami.AmiError):
        ami.search_sum_order(d, 5)


def test_no_cpu_fallback(ami):
    """A host-only table cannot be evaluated: every kernel entry point refuses (AMI_ECUDA)."""
    import ctypes as C
    tab = ami.AmiTable.from_diagram(A.self_energy_order2(), device=None)
    L = ami.lib()
    buf = np.zeros(64)
    z = np.zeros(2)
    b = np.ones(1)
    rc = L.ami_evaluate(tab._h, buf.ctypes.data, 0, 1, z.ctypes.data, 1, b.ctypes.data, 1, 0.0, 0,
                        buf.ctypes.data, None)
    assert rc == -4
    rc = L.ami_dispersion(tab._h, buf.ctypes.data, 4, 1, z.ctypes.data, 1.0, 0.0, 1, buf.ctypes.data, None)
    assert rc == -4
    assert b"no device copy" in L.ami_last_cuda_error()
    assert L.ami_strerror(-2).startswith(b"|alpha_p|")


def test_denominators_keep_their_orientation(ami):
    """The order-2 self-energy has one denominator up to sign; both orientations are kept as
    separate leaves because the regulator is added to D as it arises (reading P10)."""
    ex = ami.AmiTable.from_diagram(A.self_energy_order2(), device=None).export()
    assert ex["leafD_c"].shape[0] == 2 and len(ex["coef"]) == 4
    np.testing.assert_array_equal(ex["leafD_c"][0], -ex["leafD_c"][1])
    np.testing.assert_array_equal(ex["leafD_a"][0], -ex["leafD_a"][1])


def numpy_run_tree(tab_export, prog, e, z, beta):
    """Interprets the exported tree-plan programs with numpy, all samples at once (test-side restatement
    of the node format documented in DESIGN.md 6.3; derivative order <= 1)."""
    n = e.shape[0]
    UF, UD = len(tab_export["leafF_c"]), len(tab_export["leafD_c"])
    D = [1.0 / (e @ c + a @ z + 0j) for c, a in zip(tab_export["leafD_c"], tab_export["leafD_a"])] + [np.ones(n) + 0j]
    L = []
    for c, sig, k in zip(tab_export["leafF_c"], tab_export["leafF_sig"], tab_export["leafF_k"]):
        f = 1.0 / (sig * np.exp(beta * (e @ c)) + 1.0)
        L.append(f if k == 0 else -beta * f * (1 - f))
        assert k <= 1
    for d in D:                      # L[U_F + 2u] = Re D[u], L[U_F + 2u + 1] = Im D[u]; the last pair is (1, 0)
        L += [d.real, d.imag]
    V = np.zeros((prog["n_slots"] + 2, n))
    for i, cst in enumerate(prog["consts"]):
        V[i] = cst
    result = None
    for code, is_complex in ((prog["code_beta"], False), (prog["code_freq"], True)):
        pos = 0
        while pos < len(code):
            count, dst = int(code[pos]) >> 16, int(code[pos]) & 0xffff
            items = [int(w) for w in code[pos + 1:pos + 1 + count]]
            assert pos // 1024 == (pos + count) // 1024, "a node straddles a tile"
            if not is_complex:
                acc = np.zeros(n)
                for w in items:
                    acc = acc + L[(w >> 16) & 0xfff] * V[w & 0xffff]
                if dst != 0xffff:
                    V[dst] = acc
            else:
                acc = np.zeros(n, dtype=complex)
                for w in items:
                    b = w & 0xffff
                    acc = acc + D[(w >> 16) & 0xfff] * (V[b] + (1j * V[b + 1] if w >> 28 else 0))
                if dst != 0xffff:
                    V[dst], V[dst + 1] = acc.real.copy(), acc.imag.copy()
                else:
                    result = acc
            pos += 1 + count
    return result


@pytest.mark.parametrize("name", list(DIAGRAMS))
def test_tree_program_values_match_oracle(ami, oracle_mod, name):
    """The Horner plan serialised as a program (hash-consed FT sums, frequency-independent sub-sums,
    complex R part) reproduces the oracle's values when interpreted on the CPU."""
    d = DIAGRAMS[name]()
    tab = ami.AmiTable.from_diagram(d, device=None)
    assert tab.info["tree_plan_words"] > 0
    ex, prog = tab.export(), tab.export_tree()
    assert len(prog["code_beta"]) + len(prog["code_freq"]) == tab.info["tree_plan_words"]
    rng = np.random.default_rng(5)
    e = rng.uniform(-1.5, 1.5, size=(16, d.n_eps))
    beta = 2.0
    z = np.array([1j * math.pi / beta if d.slot_is_fermionic[-1] else 2j * math.pi / beta])
    got = numpy_run_tree(ex, prog, e, z, beta)
    want, S = oracle_mod.OracleTable.from_diagram(d).evaluate(e, [z], beta, quad=True, want_S=True)
    assert np.max(np.abs(got - want[0]) / S[0]) < 1e-12
