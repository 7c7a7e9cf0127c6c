"""LaTeX output of the term table.  The pin: the printed expression,
read back by the small evaluator below and evaluated in plain numpy, equals the CPU oracle's value."""
import math
import re

import numpy as np
import pytest

import ami_inputs as A


@pytest.fixture(scope="module")
def ami():
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    pkg.lib()
    return pkg


LIN = re.compile(r"([+-]?)(\d*)(\\epsilon|z)_\{(\d+)\}")


def linear(expr, e, z):
    if expr == "0":
        return 0.0
    tot, pos = 0.0, 0
    for mt in LIN.finditer(expr):
        assert mt.start() == pos, f"cannot read {expr!r}"
        pos = mt.end()
        c = (-1.0 if mt.group(1) == "-" else 1.0) * (float(mt.group(2)) if mt.group(2) else 1.0)
        tot = tot + c * (e[int(mt.group(4))] if mt.group(3) == r"\epsilon" else z[int(mt.group(4))])
    assert pos == len(expr), f"cannot read {expr!r}"
    return tot


def fermi_deriv(sigma, k, E, beta):
    """k-th derivative of 1/(sigma e^{beta E} + 1), by differentiating the polynomial in f (k <= 3)."""
    f = 1.0 / (sigma * np.exp(beta * E) + 1.0)
    P = np.poly1d([1.0, 0.0])                              # P_0(x) = x
    for _ in range(k):
        P = np.polymul(np.polyder(P), np.poly1d([1.0, -1.0, 0.0]))   # P' * (x^2 - x): f' = beta (f^2 - f)
    return beta ** k * np.polyval(P, f)


TERM = re.compile(r"^([+-])(?:\\frac\{(\d+)\}\{(\d+)\}|(\d+))?((?: f_\{[+-]\}(?:\^\{\(\d+\)\})?\([^()]*\))*)"
                  r"((?: \\frac\{1\}\{\([^()]*\)(?:\^\{\d+\})?\})*)$")
FERMI = re.compile(r" f_\{([+-])\}(?:\^\{\((\d+)\)\})?\(([^()]*)\)")
DEN = re.compile(r" \\frac\{1\}\{\(([^()]*)\)(?:\^\{(\d+)\})?\}")


def evaluate_latex(tex, e, z, beta):
    body = tex.strip()
    assert body.startswith("\\begin{aligned}\nI ={}& ") and body.endswith("\n\\end{aligned}")
    body = body[len("\\begin{aligned}\nI ={}& "):-len("\n\\end{aligned}")]
    pref = 1.0
    mt = re.match(r"^(\S+) \\times \\Big\[ \\\\\n& ", body)
    if mt:
        pref = float(mt.group(1))
        assert body.endswith(" \\Big]")
        body = body[mt.end():-len(" \\Big]")]
    total = 0.0
    rows = body.split(" \\\\\n& ")
    for row in rows:
        mt = TERM.match(row)
        assert mt, f"cannot read term {row!r}"
        coef = -1.0 if mt.group(1) == "-" else 1.0
        if mt.group(2):
            coef *= float(mt.group(2)) / float(mt.group(3))
        elif mt.group(4):
            coef *= float(mt.group(4))
        val = coef
        for s, k, arg in FERMI.findall(mt.group(5)):
            val = val * fermi_deriv(1.0 if s == "+" else -1.0, int(k or 0), linear(arg, e, z), beta)
        for arg, p in DEN.findall(mt.group(6)):
            val = val / linear(arg, e, z) ** int(p or 1)
        total = total + val
    return pref * total, len(rows)


DIAGRAMS = {
    "order1": A.order1_line, "bubble": A.bubble, "bubble_doubled": A.doubled_line_bubble,
    "se2": A.self_energy_order2, "se2_doubled1": lambda: A.self_energy_order2_doubled(1),
    "cfg3": lambda: A.get_config("cfg3").diagram, "cfg5": lambda: A.get_config("cfg5").diagram,
}


@pytest.mark.parametrize("name", list(DIAGRAMS))
@pytest.mark.parametrize("prefactor", [1.0, -2.5])
def test_latex_reads_back_to_the_oracle_value(ami, oracle_mod, name, prefactor):
    d = DIAGRAMS[name]()
    tab = ami.AmiTable.from_diagram(d, device=None, prefactor=prefactor)
    tex = tab.latex()
    rng = np.random.default_rng(7)
    e = rng.uniform(-1.5, 1.5, size=(6, d.n_eps))
    beta = 1.7
    z = np.array([0.3 + 1j * math.pi / beta]) if d.slot_is_fermionic[-1] else np.array([-0.2 + 2j * math.pi / beta])
    want, S = oracle_mod.OracleTable.from_diagram(d, prefactor=prefactor).evaluate(e, [z], beta, quad=True, want_S=True)
    for s in range(e.shape[0]):
        got, rows = evaluate_latex(tex, e[s], z, beta)
        assert rows == tab.info["n_terms"]
        assert abs(got - want[0][s]) <= 1e-11 * S[0][s]


def test_latex_of_the_order1_line_and_buffer_protocol(ami):
    """PAPER.md north-star pin in print: one Fermi function of minus the supplied energy."""
    import ctypes as C
    tab = ami.AmiTable.from_diagram(A.order1_line(), device=None)
    assert tab.latex() == "\\begin{aligned}\nI ={}& + f_{+}(-\\epsilon_{0})\n\\end{aligned}\n"
    n = C.c_size_t(3)
    buf = C.create_string_buffer(3)
    assert ami.lib().ami_table_latex(tab._h, buf, C.byref(n)) == -1          # too small
    assert ami.lib().ami_table_latex(None, None, C.byref(n)) == -1


# ---------------------------------------------------------------- factorised form (FT * R)
SROW = re.compile(r"^S_\{(\d+)\} =\{\}&((?: [+-](?:\\frac\{\d+\}\{\d+\}|\d+)? f_\{[+-]\}(?:\^\{\(\d+\)\})?\([^()]*\)(?: S_\{\d+\})?)+)$")
SITEM = re.compile(r" ([+-])(?:\\frac\{(\d+)\}\{(\d+)\}|(\d+))? f_\{([+-])\}(?:\^\{\((\d+)\)\})?\(([^()]*)\)(?: S_\{(\d+)\})?")
GROW = re.compile(r"^(?:\+ S_\{(\d+)\}|([+-])(?:\\frac\{(\d+)\}\{(\d+)\}|(\d+)))((?: \\frac\{1\}\{\([^()]*\)(?:\^\{\d+\})?\})*)$")


def evaluate_latex_factorized(tex, e, z, beta):
    body = tex.strip()
    assert body.startswith("\\begin{aligned}\n") and body.endswith("\n\\end{aligned}")
    body = body[len("\\begin{aligned}\n"):-len("\n\\end{aligned}")]
    head, tail = body.split("I ={}& ")
    S = {}
    for row in [r for r in head.split(" \\\\\n") if r]:
        mt = SROW.match(row)
        assert mt, f"cannot read sum {row!r}"
        tot = 0.0
        for sg, fn, fd, ci, fs, k, arg, child in SITEM.findall(mt.group(2)):
            c = -1.0 if sg == "-" else 1.0
            c *= float(fn) / float(fd) if fn else (float(ci) if ci else 1.0)
            v = c * fermi_deriv(1.0 if fs == "+" else -1.0, int(k or 0), linear(arg, e, z), beta)
            tot = tot + (v * S[int(child)] if child else v)       # children are printed before their parents
        S[int(mt.group(1))] = tot
    pref = 1.0
    mt = re.match(r"^(\S+) \\times \\Big\[ \\\\\n& ", tail)
    if mt:
        pref = float(mt.group(1))
        assert tail.endswith(" \\Big]")
        tail = tail[mt.end():-len(" \\Big]")]
    total = 0.0
    rows = tail.split(" \\\\\n& ")
    for row in rows:
        mt = GROW.match(row)
        assert mt, f"cannot read group {row!r}"
        if mt.group(1):
            val = S[int(mt.group(1))]
        else:
            val = (-1.0 if mt.group(2) == "-" else 1.0) * (float(mt.group(3)) / float(mt.group(4)) if mt.group(3) else float(mt.group(5)))
        for arg, p in DEN.findall(mt.group(6)):
            val = val / linear(arg, e, z) ** int(p or 1)
        total = total + val
    return pref * total, len(rows), len(S)


@pytest.mark.parametrize("name", list(DIAGRAMS))
@pytest.mark.parametrize("prefactor", [1.0, -2.5])
def test_factorized_latex_reads_back_to_the_oracle_value(ami, oracle_mod, name, prefactor):
    """The FT * R form of PAPER.md:100-104 printed from the library's Horner plan: read back and evaluated in numpy
    it equals the oracle's value; it has one row per denominator product and is far shorter than the flat table."""
    d = DIAGRAMS[name]()
    tab = ami.AmiTable.from_diagram(d, device=None, prefactor=prefactor)
    tex = tab.latex(factorized=True)
    rng = np.random.default_rng(11)
    e = rng.uniform(-1.5, 1.5, size=(6, d.n_eps))
    beta = 1.3
    z = np.array([0.3 + 1j * math.pi / beta]) if d.slot_is_fermionic[-1] else np.array([-0.2 + 2j * math.pi / beta])
    want, S = oracle_mod.OracleTable.from_diagram(d, prefactor=prefactor).evaluate(e, [z], beta, quad=True, want_S=True)
    for s in range(e.shape[0]):
        got, rows, sums = evaluate_latex_factorized(tex, e[s], z, beta)
        assert rows == tab.info["n_groups"]
        assert abs(got - want[0][s]) <= 1e-11 * S[0][s]
    if tab.info["n_terms"] >= 60:
        assert len(tex) * 2 < len(tab.latex())


def test_factorized_latex_shows_fig1_shape(ami):
    """Fig. 1: the order-2 self-energy factorises as [f(z1) - f(z2)] [f(z3) + f(z4)] R: one shared sum
    S_0 = f(-e0) - f(e2) multiplies both remaining Fermi/Bose factors."""
    tex = ami.AmiTable.from_diagram(A.self_energy_order2(), device=None).latex(factorized=True)
    assert "S_{0} ={}& + f_{+}(-\\epsilon_{0}) - f_{+}(\\epsilon_{2}) \\\\" in tex
    assert tex.count(" S_{0}") == 2 and tex.count("\\frac{1}{(") == 2
