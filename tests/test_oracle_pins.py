"""Pins of the CPU oracle against what the paper and the mathematics fix (never against
itself): closed forms, brute-force Matsubara sums of Eq. 1, invariances, finite differences.
All CPU-only.  Citations are PAPER.md lines; P-numbers are DESIGN.md readings."""
import itertools
import math
import os

import numpy as np
import pytest
from scipy.special import expit

import ami_inputs as A

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def fermi(x, beta):
    """Textbook Fermi function 1/(e^{beta x}+1) from scipy's logistic sigmoid (independent of
    the oracle and accurate in both tails)."""
    return expit(-beta * np.asarray(x, dtype=float))


def table(oracle_mod, d, **kw):
    return oracle_mod.OracleTable.from_diagram(d, **kw)


RNG = np.random.default_rng(7)


def assert_close_on_scale(got, want, S, tol_S, tol_rel, kappa_max=1e3, min_well=0.3):
    """The parity norm of reading P20: |got-want| <= tol_S * S everywhere (S = sum |term|), and
    plain relative error <= tol_rel where the sum is well conditioned (S/|want| <= kappa_max)."""
    err = np.abs(got - want)
    assert np.max(err / S) <= tol_S, np.max(err / S)
    well = S <= kappa_max * np.abs(want)
    assert well.mean() >= min_well
    assert np.max(err[well] / np.abs(want[well])) <= tol_rel


# ---------------------------------------------------------------- closed forms
@pytest.mark.parametrize("beta", [0.7, 2.0, 9.0])
def test_order1_closed_form(oracle_mod, beta):
    """Eq. 2 + Eq. 3 for one line: I = f(-e1) (reading P3)."""
    t = table(oracle_mod, A.order1_line())
    assert t.info()["T"] == 1
    e = RNG.uniform(-4, 4, size=(50, 1))
    for quad in (False, True):
        got = t.evaluate(e, [[1j * math.pi / beta]], beta, quad=quad)[0]
        np.testing.assert_allclose(got, fermi(-e[:, 0], beta), rtol=1e-13, atol=1e-300)


@pytest.mark.parametrize("beta,n", [(2.0, 1), (5.0, 3), (10.0, 7)])
def test_bubble_closed_form(oracle_mod, beta, n):
    """Bare bubble with bosonic external frequency: (f(a)-f(b))/(i Omega + a - b), a=-e1, b=-e2."""
    t = table(oracle_mod, A.bubble())
    assert t.info()["T"] == 2
    e = RNG.uniform(-4, 4, size=(200, 2))
    Om = 2 * math.pi * n / beta
    a, b = -e[:, 0], -e[:, 1]
    want = (fermi(a, beta) - fermi(b, beta)) / (1j * Om + a - b)
    # the closed form itself cancels in double when f(a) ~ f(b): compare on the scale S (P20)
    got, S = t.evaluate(e, [[1j * Om]], beta, quad=True, want_S=True)
    assert_close_on_scale(got[0], want, S[0], 1e-14, 1e-12)
    got = t.evaluate(e, [[1j * Om]], beta, quad=False)
    assert_close_on_scale(got[0], want, S[0], 1e-13, 1e-11)


def se2_textbook(e, nu, beta):
    """Bose-function-free second-order self-energy with eps_j = -e_j:
    -[f1 f3 (1-f2) + (1-f1)(1-f3) f2] / (i nu + eps2 - eps1 - eps3)."""
    eps = -e
    f1, f2, f3 = (fermi(eps[:, i], beta) for i in range(3))
    g1, g2, g3 = (fermi(-eps[:, i], beta) for i in range(3))  # 1 - f without cancellation
    return -(f1 * f3 * g2 + g1 * g3 * f2) / (1j * nu + eps[:, 1] - eps[:, 0] - eps[:, 2])


@pytest.mark.parametrize("beta,n", [(1.0, 0), (5.0, 0), (5.0, 4), (10.0, 2)])
def test_se2_closed_form(oracle_mod, beta, n):
    """Eq. 7 labels (P1) -> 4 flat terms whose sum is the textbook expression."""
    t = table(oracle_mod, A.self_energy_order2())
    assert t.info()["T"] == 4
    e = RNG.uniform(-4, 4, size=(300, 3))
    nu = (2 * n + 1) * math.pi / beta
    want = se2_textbook(e, nu, beta)
    got, S = t.evaluate(e, [[1j * nu]], beta, quad=True, want_S=True)
    # the AMI form has Bose factors that cancel; compare on the scale S of its terms (P20)
    assert np.max(np.abs(got[0] - want) / S[0]) < 1e-13
    well = S[0] / np.abs(want) < 1e3
    assert well.sum() > 100
    np.testing.assert_allclose(got[0][well], want[well], rtol=1e-11)
    got_d = t.evaluate(e, [[1j * nu]], beta, quad=False)
    assert np.max(np.abs(got_d[0] - want) / S[0]) < 1e-12


def test_se2_fig1_shape(oracle_mod):
    """Fig. 1: the result factorises as [f(z1)-f(z2)][f(z3)+f(z4)] * R:
    [f(-e1) - f(e3)] [f(-e2) - f_{sigma=-1}(-e1-e3)] / (i nu + e1 + e3 - e2)."""
    t = table(oracle_mod, A.self_energy_order2())
    beta, nu = 3.0, math.pi / 3.0
    e = RNG.uniform(-2, 2, size=(100, 3))
    bose_like = 1.0 / (1.0 - np.exp(beta * (-e[:, 0] - e[:, 2])))
    want = ((fermi(-e[:, 0], beta) - fermi(e[:, 2], beta)) * (fermi(-e[:, 1], beta) - bose_like)
            / (1j * nu + e[:, 0] + e[:, 2] - e[:, 1]))
    got = t.evaluate(e, [[1j * nu]], beta, quad=True)[0]
    np.testing.assert_allclose(got, want, rtol=1e-10)


@pytest.mark.parametrize("n", [1, 3])
def test_doubled_bubble_closed_form(oracle_mod, n):
    """G^2 = -dG/de: I = f'(a)/(i Om + a - b) - (f(a)-f(b))/(i Om + a - b)^2, f' = -beta f (1-f).
    Exercises Eq. 5 with M = 2 (P6)."""
    t = table(oracle_mod, A.doubled_line_bubble())
    info = t.info()
    assert info["T"] == 3 and info["max_deriv"] == 1 and info["multipoles"] == 1
    beta = 4.0
    Om = 2 * math.pi * n / beta
    e = RNG.uniform(-3, 3, size=(200, 2))
    a, b = -e[:, 0], -e[:, 1]
    fa, fb = fermi(a, beta), fermi(b, beta)
    den = 1j * Om + a - b
    want = -beta * fa * (1 - fa) / den - (fa - fb) / den ** 2
    got, S = t.evaluate(e, [[1j * Om]], beta, quad=True, want_S=True)
    assert_close_on_scale(got[0], want, S[0], 1e-13, 1e-10)


# ---------------------------------------------------------------- Fermi/Bose functions
@pytest.mark.parametrize("sigma", [1, -1])
@pytest.mark.parametrize("k", [1, 2, 3])
def test_fermi_derivative_finite_difference(oracle_mod, sigma, k):
    """f^{(k)} from the (f,g) recursion (P11) against central differences of f^{(k-1)}."""
    beta = 3.0
    for E in (0.37 + 0.0j, -1.3 + 0.0j, 0.8 - 0.21j):
        h = 1e-5
        fd = (oracle_mod.fermi(E + h, beta, sigma, k - 1) - oracle_mod.fermi(E - h, beta, sigma, k - 1)) / (2 * h)
        got = oracle_mod.fermi(E, beta, sigma, k)
        assert abs(got - fd) <= 1e-8 * max(1.0, abs(got))


def test_fermi_first_derivative_closed_form(oracle_mod):
    beta = 2.5
    for x in (-3.0, -0.2, 0.0, 0.9, 4.0):
        f = fermi(x, beta)
        assert abs(oracle_mod.fermi(x, beta, 1, 1).real - (-beta * f * (1 - f))) < 1e-14
        assert abs(oracle_mod.fermi(x, beta, 1, 0).real - f) < 1e-15


@pytest.mark.parametrize("bx", [1e-9, 1.0, 40.0, 800.0])
def test_fermi_double_vs_quad(oracle_mod, bx):
    """P12: no overflow and no cancellation at beta|E| = 1e-9 ... 800, either sign, both sigma."""
    beta = 10.0
    for sign in (1, -1):
        for sigma in (1, -1):
            for k in (0, 1, 2):
                E = sign * bx / beta
                d = oracle_mod.fermi(E, beta, sigma, k, quad=False)
                q = oracle_mod.fermi(E, beta, sigma, k, quad=True)
                assert np.isfinite(d.real) and np.isfinite(q.real)
                # f'' has a genuine zero at E = 0 (g - f -> 0): allow rounding on the scale
                # beta^k |f g| of the derivative's own factors, which still shrinks in the tails
                fg = abs(oracle_mod.fermi(E, beta, sigma, 1, quad=True)) / beta
                assert abs(d - q) <= 1e-13 * abs(q) + 1e-15 * beta ** k * fg + 1e-300, (bx, sign, sigma, k, d, q)


def test_bose_limits(oracle_mod):
    """sigma = -1: f = 1/(1 - e^{beta E}) = -n_B(E); small-argument limit -1/(beta E) - 1/2... and tails."""
    beta = 2.0
    x = 1e-7
    assert abs(oracle_mod.fermi(x / beta, beta, -1, 0).real - (-1 / x + 0.5)) < 1e-6
    assert abs(oracle_mod.fermi(50.0, beta, -1, 0).real) < 1e-40
    assert abs(oracle_mod.fermi(-50.0, beta, -1, 0).real - 1.0) < 1e-15


# ---------------------------------------------------------------- complex arguments (reading P19)
def mp_fermi(E, beta, sigma, k=0):
    """f_sigma^{(k)}(E) = d^k/dE^k 1/(sigma e^{beta E} + 1) at 40 digits (mpmath), for complex E; the
    derivatives by mpmath's own numerical differentiation of that definition -- independent of the oracle."""
    import mpmath as mp
    mp.mp.dps = 40
    f = lambda x: 1 / (sigma * mp.exp(beta * x) + 1)
    v = f(mp.mpc(E)) if k == 0 else mp.diff(f, mp.mpc(E), k)
    return complex(v)


@pytest.mark.parametrize("sigma", [1, -1])
@pytest.mark.parametrize("k", [0, 1, 2])
def test_fermi_complex_argument(oracle_mod, sigma, k):
    """The complex-argument branch of the oracle's Fermi/Bose function (energy_t is complex128,
    PAPER.md:253-255) against the definition 1/(sigma e^{beta E} + 1) evaluated with mpmath: both
    signs of Re E and Im E, moderate arguments, both tails (Re beta E = -+60, -+700: the branch that
    exponentiates the argument with Re <= 0) and, for sigma = -1, the neighbourhood of the pole
    (expm1 branch).  f(conj E) = conj f(E), so a sign slip in the imaginary part of the complex
    exponential fails the imaginary part here."""
    beta = 2.5
    pts = [0.8 - 0.21j, 0.8 + 0.21j, -0.8 - 0.21j, -0.8 + 0.21j, 0.05 + 1.1j, -0.05 - 1.1j, 3.0 + 0.7j, -3.0 - 0.7j,
           24.0 + 0.3j, -24.0 - 0.3j, 280.0 - 0.4j, -280.0 + 0.4j, 1e-4 + 2e-4j, -1e-4 + 2e-4j, 2e-7 - 1e-7j]
    for E in pts:
        want = mp_fermi(E, beta, sigma, k)
        fg = abs(mp_fermi(E, beta, sigma, 1)) / beta      # |f g|: the scale of the factors of every derivative
        for quad in (True, False):
            got = oracle_mod.fermi(E, beta, sigma, k, quad=quad)
            tol = 1e-13 if quad else 1e-11      # double: beta*E itself is rounded; |f^(k)| ~ 1/|beta E|^(k+1) near the pole
            # f'' = beta^2 f g (g - f) has a genuine zero at E = 0 (sigma = +1): in double, rounding on the
            # scale of its own factors, as in test_fermi_double_vs_quad
            slack = 0.0 if quad else 1e-15 * beta ** k * fg
            assert abs(got - want) <= tol * abs(want) + slack + 1e-300, (E, sigma, k, quad, got, want)
        if abs(want.imag) > 1e-290:
            assert np.sign(got.imag) == np.sign(want.imag), (E, sigma, k)


def test_fermi_complex_closed_forms_numpy(oracle_mod):
    """Same branch against plain numpy complex arithmetic at moderate |beta E| (no mpmath):
    f = 1/(sigma e^x + 1), f' = -beta sigma e^x/(sigma e^x + 1)^2."""
    beta = 1.7
    for sigma in (1, -1):
        for E in (0.31 + 0.52j, 0.31 - 0.52j, -1.4 + 0.9j, -1.4 - 0.9j, 2.2 + 3.0j):
            x = np.exp(beta * E)
            assert abs(oracle_mod.fermi(E, beta, sigma, 0) - 1 / (sigma * x + 1)) < 2e-15
            assert abs(oracle_mod.fermi(E, beta, sigma, 1) - (-beta * sigma * x / (sigma * x + 1) ** 2)) < 1e-14


@pytest.mark.parametrize("beta,n", [(2.0, 1), (5.0, 3)])
def test_bubble_closed_form_complex_energies(oracle_mod, beta, n):
    """A whole diagram with complex energies (variant 5b): the bubble closed form
    (f(a) - f(b))/(i Omega + a - b), a = -e1, b = -e2 complex, f from mpmath."""
    t = table(oracle_mod, A.bubble())
    e = RNG.uniform(-3, 3, size=(40, 2)) + 1j * RNG.uniform(-0.4, 0.4, size=(40, 2))
    Om = 2 * math.pi * n / beta
    a, b = -e[:, 0], -e[:, 1]
    fa = np.array([mp_fermi(x, beta, 1) for x in a])
    fb = np.array([mp_fermi(x, beta, 1) for x in b])
    den = 1j * Om + a - b
    want = (fa - fb) / den
    S_want = (np.abs(fa) + np.abs(fb)) / np.abs(den)
    for quad, tol in ((True, 1e-14), (False, 1e-13)):
        got, S = t.evaluate(e, [[1j * Om]], beta, quad=quad, want_S=True)
        assert np.max(np.abs(got[0] - want) / S_want) <= tol
        np.testing.assert_allclose(S[0], S_want, rtol=1e-13)
    # the conjugate energies give the mirrored result: I(conj e, -Omega) = conj I(e, Omega)
    got_c = t.evaluate(np.conj(e), [[-1j * Om]], beta, quad=True)
    np.testing.assert_allclose(got_c[0], np.conj(want), rtol=0, atol=1e-13 * S_want.max())


# ---------------------------------------------------------------- S = sum_t |term_t|, the scale of the parity norm (P20)
def test_S_closed_forms(oracle_mod):
    """S is the denominator of the parity norm (tests/parity.py), so it is pinned like a value:
    order 1: S = |f(-e1)|;  bubble: S = (|f(a)| + |f(b)|)/|i Om + a - b|;  doubled bubble (3 terms):
    S = beta f_a (1-f_a)/|den| + (f_a + f_b)/|den|^2.  Prefactor A scales it by |A|."""
    beta = 3.0
    e1 = RNG.uniform(-3, 3, size=(30, 1))
    _, S = table(oracle_mod, A.order1_line()).evaluate(e1, [[1j * math.pi / beta]], beta, quad=True, want_S=True)
    np.testing.assert_allclose(S[0], fermi(-e1[:, 0], beta), rtol=1e-14)
    e = RNG.uniform(-3, 3, size=(60, 2))
    Om = 2 * math.pi * 2 / beta
    a, b = -e[:, 0], -e[:, 1]
    fa, fb = fermi(a, beta), fermi(b, beta)
    den = np.abs(1j * Om + a - b)
    for quad in (True, False):
        _, S = table(oracle_mod, A.bubble()).evaluate(e, [[1j * Om]], beta, quad=quad, want_S=True)
        np.testing.assert_allclose(S[0], (fa + fb) / den, rtol=1e-13)
        _, S = table(oracle_mod, A.doubled_line_bubble()).evaluate(e, [[1j * Om]], beta, quad=quad, want_S=True)
        np.testing.assert_allclose(S[0], beta * fa * (1 - fa) / den + (fa + fb) / den ** 2, rtol=1e-12)
    _, S = table(oracle_mod, A.bubble(), prefactor=-2.5).evaluate(e, [[1j * Om]], beta, quad=True, want_S=True)
    np.testing.assert_allclose(S[0], 2.5 * (fa + fb) / den, rtol=1e-13)
    # S >= |value| always, and S = |value| when there is a single term
    v, S = table(oracle_mod, A.self_energy_order2()).evaluate(RNG.uniform(-3, 3, size=(50, 3)), [[1j * math.pi / beta]],
                                                               beta, quad=True, want_S=True)
    assert (S[0] >= np.abs(v[0]) * (1 - 1e-15)).all()


def test_log2_scale_survives_underflow(oracle_mod):
    """log2 S and log2 |value| are taken in quad precision before the cast to double: for one line at
    beta e1 = -1000 the value e^{-1000}/(1 + e^{-1000}) is 0 as a double but its logarithm is exact;
    for ordinary samples they agree with log2 of the double outputs."""
    t = table(oracle_mod, A.order1_line())
    beta = 10.0
    v, S, l2S, l2v = t.evaluate(np.array([[-100.0], [0.3], [-2.0]]), [[1j * math.pi / beta]], beta, quad=True, want_logs=True)
    assert v[0, 0] == 0 and S[0, 0] == 0
    assert abs(l2S[0, 0] - (-1000.0 / math.log(2))) < 1e-9 and l2S[0, 0] == l2v[0, 0]
    np.testing.assert_allclose(l2S[0, 1:], np.log2(S[0, 1:]), rtol=0, atol=1e-12)
    np.testing.assert_allclose(l2v[0, 1:], np.log2(np.abs(v[0, 1:])), rtol=0, atol=1e-12)


# ---------------------------------------------------------------- brute-force Eq. 1
def brute_force(d, e, z_ext, beta, N):
    """beta^-n sum over |n_l| < N (n_l = -N..N-1, symmetric in nu) of prod_j 1/(X^j + E^j),
    Eq. 1 + Eq. 2 written out; internal frequencies fermionic."""
    m = d.n_int
    n = np.arange(-N, N)
    nu = (2 * n + 1) * math.pi / beta
    E = d.eps @ e  # E^j
    total = 0.0 + 0.0j
    grids = np.meshgrid(*([nu] * (m - 1)), indexing="ij") if m > 1 else []
    for nu0 in nu:
        prod = 1.0
        for j in range(d.n_g):
            X = 1j * d.alpha[j, 0] * nu0 + d.alpha[j, m] * z_ext
            for l in range(1, m):
                if d.alpha[j, l]:
                    X = X + 1j * d.alpha[j, l] * grids[l - 1]
            prod = prod * (1.0 / (X + E[j]))
        total += np.sum(prod)
    return total / beta ** m


def richardson2(fn, N):
    """Two Richardson steps in 1/N from N, 2N, 4N."""
    a, b, c = fn(N), fn(2 * N), fn(4 * N)
    r1, r2 = 2 * b - a, 2 * c - b
    return (4 * r2 - r1) / 3


@pytest.mark.parametrize("diagram,N,tol", [
    ("bubble", 20000, 1e-9), ("bubble_doubled", 20000, 1e-10), ("se2", 500, 2e-7),
    ("se2_doubled0", 500, 1e-8), ("se2_doubled1", 500, 1e-8), ("se2_doubled2", 500, 2e-7),
])
def test_brute_force_matsubara(oracle_mod, diagram, N, tol):
    """The definition, Eq. 1, summed directly (every nu_l enters >= 2 lines, so the sum converges
    without a convergence factor; reading P3).  Pins signs, statistics (P4) and structure."""
    d = {"bubble": A.bubble, "bubble_doubled": A.doubled_line_bubble, "se2": A.self_energy_order2,
         "se2_doubled0": lambda: A.self_energy_order2_doubled(0),
         "se2_doubled1": lambda: A.self_energy_order2_doubled(1),
         "se2_doubled2": lambda: A.self_energy_order2_doubled(2)}[diagram]()
    beta = 2.0
    e = np.array([0.45, -0.8, 1.1])[: d.n_eps]
    z = 1j * math.pi / beta if d.slot_is_fermionic[-1] else 1j * 2 * math.pi / beta
    want = richardson2(lambda n: brute_force(d, e, z, beta, n), N)
    got = table(oracle_mod, d).evaluate(e[None, :], [[z]], beta, quad=True)[0, 0]
    assert abs(got - want) <= tol * abs(want), (got, want)


def test_brute_force_order3(oracle_mod):
    """Order-3 random 1PI topology (5 lines, triple sum): N = 24/48/96."""
    d = A.random_self_energy(3, 5)
    beta = 1.5
    e = np.array([0.3, -0.6, 0.9, -1.2, 0.5])[: d.n_eps]
    z = 1j * math.pi / beta
    want = richardson2(lambda n: brute_force(d, e, z, beta, n), 24)
    got = table(oracle_mod, d).evaluate(e[None, :], [[z]], beta, quad=True)[0, 0]
    assert abs(got - want) <= 2e-5 * abs(want), (got, want)


# ---------------------------------------------------------------- invariances (P14)
def random_energies(d, n, lo=-4.0, hi=4.0):
    return RNG.uniform(lo, hi, size=(n, d.n_eps))


@pytest.mark.parametrize("m,seed", [(3, 1), (3, 2), (4, 1), (4, 3), (5, 2)])
def test_integration_order_invariance(oracle_mod, m, seed):
    """Different summation orders give different tables but the same values."""
    d = A.random_self_energy(m, seed)
    beta = 2.0
    e = random_energies(d, 40, -2, 2)
    z = [[1j * math.pi / beta]]
    ref, S = table(oracle_mod, d).evaluate(e, z, beta, quad=True, want_S=True)
    orders = list(itertools.permutations(range(m)))
    picks = orders if m == 3 else [orders[i] for i in RNG.choice(len(orders), 4, replace=False)]
    n_ok = 0
    for so in picks:
        try:
            t = table(oracle_mod, d, sum_order=so)
        except oracle_mod.OracleError as ex:
            assert ex.code == -2  # |alpha_p| = 2 in this order: unsupported (P8), not wrong
            continue
        got, S2 = t.evaluate(e, z, beta, quad=True, want_S=True)
        assert np.max(np.abs(got - ref) / np.maximum(S, S2)) < 1e-14
        n_ok += 1
    assert n_ok >= 1


@pytest.mark.parametrize("m,seed", [(2, 0), (4, 1), (5, 1)])
def test_R0_order_invariance(oracle_mod, m, seed):
    """the ordering of the Green's functions in R0 does not change the result."""
    d = A.self_energy_order2() if m == 2 else A.random_self_energy(m, seed)
    beta = 3.0
    e = random_energies(d, 40, -2, 2)
    z = [[1j * math.pi / beta]]
    ref, S = table(oracle_mod, d).evaluate(e, z, beta, quad=True, want_S=True)
    for _ in range(3):
        got = table(oracle_mod, d.permuted(RNG.permutation(d.n_g))).evaluate(e, z, beta, quad=True)
        assert np.max(np.abs(got - ref) / S) < 1e-14


# ---------------------------------------------------------------- multipoles (P6, P7)
def split_copy(d):
    """Same lines, but every line gets its own energy symbol (no shared symbols)."""
    eps = np.eye(d.n_g, dtype=np.int32)
    return A.Diagram(d.name + "_split", d.n_int, d.n_ext, d.alpha.copy(), eps, d.slot_is_fermionic.copy())


def multipole_diagrams():
    yield A.doubled_line_bubble()
    yield A.self_energy_order2_doubled(0)
    yield A.self_energy_order2_doubled(2)
    yield A.random_self_energy(4, A.configs.TOPOLOGY_SEEDS["cfg3"])


@pytest.mark.parametrize("idx", range(4))
def test_split_energy_limit(oracle_mod, idx):
    """A double pole is the limit of two simple poles at e -+ delta/2: the table built with
    Eq. 5 must agree with the all-simple-pole table of the split diagram as delta -> 0."""
    d = list(multipole_diagrams())[idx]
    t = table(oracle_mod, d)
    assert t.info()["multipoles"] > 0 and t.info()["max_deriv"] >= 1
    ds = split_copy(d)
    ts = table(oracle_mod, ds)
    assert ts.info()["max_deriv"] == 0
    sym = np.argmax(d.eps, axis=1)
    beta = 2.0
    z = [[1j * math.pi / beta if d.slot_is_fermionic[-1] else 2j * math.pi / beta]]
    e = random_energies(d, 10, -1.5, 1.5)
    ref = t.evaluate(e, z, beta, quad=True)

    def split_value(delta):
        es = e[:, sym].copy()
        for s in range(d.n_eps):
            lines = np.nonzero(sym == s)[0]
            if len(lines) > 1:  # symmetric offsets -> error O(delta^2)
                off = (np.arange(len(lines)) - (len(lines) - 1) / 2) * delta
                es[:, lines] += off[None, :]
        return ts.evaluate(es, z, beta, quad=True)

    err1 = np.max(np.abs(split_value(2e-3) - ref) / np.abs(ref))
    err2 = np.max(np.abs(split_value(1e-3) - ref) / np.abs(ref))
    assert err2 < 1e-5 and err2 < 0.3 * err1  # converging quadratically to the Eq. 5 result


def test_doubled_line_is_minus_derivative(oracle_mod):
    """G^2 = -dG/de: the doubled-line order-2 self-energy equals -d/de of the plain one."""
    beta, z = 2.0, [[1j * math.pi / 2.0]]
    e = random_energies(A.self_energy_order2(), 20, -1.5, 1.5)
    plain = table(oracle_mod, A.self_energy_order2())
    for which in range(3):
        got = table(oracle_mod, A.self_energy_order2_doubled(which)).evaluate(e, z, beta, quad=True)

        def cd(h):
            ep, em = e.copy(), e.copy()
            ep[:, which] += h
            em[:, which] -= h
            return -(plain.evaluate(ep, z, beta, quad=True) - plain.evaluate(em, z, beta, quad=True)) / (2 * h)

        want = (4 * cd(1e-3) - cd(2e-3)) / 3  # Richardson, O(h^4)
        np.testing.assert_allclose(got, want, rtol=1e-8)


# ---------------------------------------------------------------- errors (P8, P9)
def test_error_codes(oracle_mod):
    d = A.order1_line()
    with pytest.raises(oracle_mod.OracleError) as ei:
        oracle_mod.OracleTable(1, 1, [[2, 0]], d.eps, d.slot_is_fermionic)
    assert ei.value.code == -2
    with pytest.raises(oracle_mod.OracleError) as ei:
        oracle_mod.OracleTable(2, 1, [[1, 0, 0]], d.eps, [1, 1, 1])  # nothing depends on nu_2
    assert ei.value.code == -3


# ---------------------------------------------------------------- dispersion (Eqs. 8-18)
def load_int_matrix(name):
    rows = [ln.split() for ln in open(os.path.join(GOLD, name)) if ln.strip() and not ln.startswith("#")]
    return np.array(rows, dtype=np.int64)


def test_paper_alpha_and_kron_matrices():
    """Eq. 11 and Eq. 15 as printed in the paper."""
    d = A.self_energy_order2()
    np.testing.assert_array_equal(d.alpha, load_int_matrix("eq11_alpha.txt"))
    np.testing.assert_array_equal(A.kron_identity(d.alpha, 2), load_int_matrix("eq15_A.txt"))


def test_dispersion_matches_eq16(oracle_mod):
    """K = k . A^T (Eq. 16-17, columns as printed) then e_i = 2t(cos Kx + cos Ky) + mu (PAPER.md:84:
    the supplied energy is minus the dispersion), against the oracle's per-symbol loop."""
    d = A.self_energy_order2()
    t = table(oracle_mod, d)
    kint = A.momenta(11, 64, 2)
    q = np.array([0.3, -1.1])
    kfull = np.concatenate([kint.reshape(64, 4), np.tile(q, (64, 1))], axis=1)  # Eq. 9
    K = kfull @ load_int_matrix("eq16_K_columns.txt").T  # Eq. 17
    tt, mu = 1.3, -0.4
    want = np.stack([2 * tt * (np.cos(K[:, 2 * i]) + np.cos(K[:, 2 * i + 1])) + mu for i in range(3)], axis=1)
    for quad in (False, True):
        got = t.dispersion(kint, [q], tt, mu, quad=quad)
        np.testing.assert_allclose(got, want, rtol=0, atol=5e-15)


def test_dispersion_random_topology(oracle_mod):
    d = A.random_self_energy(4, 1)
    t = table(oracle_mod, d)
    kint = A.momenta(5, 32, 4)
    q = np.array([math.pi / 2, math.pi / 2])
    sa = d.symbol_alpha()
    K = np.einsum("sl,nlc->nsc", sa[:, :4], kint) + sa[:, 4][None, :, None] * q[None, None, :]
    want = 2.0 * (np.cos(K[..., 0]) + np.cos(K[..., 1])) + 0.0
    np.testing.assert_allclose(t.dispersion(kint, [q], 1.0, 0.0, quad=True), want, atol=1e-14)


@pytest.mark.parametrize("dim", [1, 2, 3])
def test_dispersion_lattice_special_points(oracle_mod, dim):
    """Other dimensions and bands (Eq. 14 is written for any d): values at points where the
    band is known by inspection.  One line, K = k (order-1 diagram)."""
    t_ = table(oracle_mod, A.order1_line())
    tt, mu = 1.3, -0.4
    pts = {0.0: 2 * tt * dim + mu, math.pi: -2 * tt * dim + mu, math.pi / 3: tt * dim + mu, 2 * math.pi / 3: -tt * dim + mu}
    for x, want in pts.items():
        for quad in (False, True):
            got = t_.dispersion(np.full((1, 1, dim), x), [np.zeros(dim)], tt, mu, quad=quad, dim=dim, band=0)
            assert abs(got[0, 0] - want) < 4e-15 * dim
    got = t_.dispersion(np.full((1, 1, dim), math.pi / 2), [np.zeros(dim)], tt, mu, quad=True, dim=dim)
    assert abs(got[0, 0] - mu) < 1e-15                      # half filling: the band vanishes on the diagonal point
    k = np.array([1.0, 2.0, 2.0])[:dim].reshape(1, 1, dim)   # free particles: e = mu - t |K|^2
    want = mu - tt * float((k ** 2).sum())
    assert t_.dispersion(k, [np.zeros(dim)], tt, mu, dim=dim, band=1)[0, 0] == pytest.approx(want, abs=1e-15)
    with pytest.raises(oracle_mod.OracleError):
        t_.dispersion(np.zeros((1, 1, 4)), [np.zeros(4)], tt, mu, dim=4)


def test_dispersion_lattice_eq14_and_separability(oracle_mod):
    """d = 3: K = k . (alpha (x) I_3)^T (Eq. 14) against the oracle's per-symbol loop; the
    hypercubic band is a sum over components, so the 3D energy is the sum of the 1D energies of the
    components; d = 2, band 0 is the function the configurations use."""
    d = A.self_energy_order2()
    t_ = table(oracle_mod, d)
    n, m = 40, 2
    kint = A.momenta(13, n, m, d=3)
    q = np.array([0.3, -1.1, 2.0])
    kfull = np.concatenate([kint.reshape(n, 3 * m), np.tile(q, (n, 1))], axis=1)
    K = kfull @ A.kron_identity(d.symbol_alpha(), 3).T          # [n][n_eps * 3]
    tt, mu = 0.7, 0.25
    e3 = t_.dispersion(kint, [q], tt, mu, quad=True, dim=3, band=0)
    want = 2 * tt * np.cos(K).reshape(n, d.n_eps, 3).sum(axis=2) + mu
    np.testing.assert_allclose(e3, want, rtol=0, atol=1e-14)
    parts = sum(t_.dispersion(kint[:, :, c:c + 1], [q[c:c + 1]], tt, 0.0, quad=True, dim=1) for c in range(3))
    np.testing.assert_allclose(e3 - mu, parts, rtol=0, atol=1e-14)
    free = t_.dispersion(kint, [q], tt, mu, quad=True, dim=3, band=1)
    np.testing.assert_allclose(free, mu - tt * (K ** 2).reshape(n, d.n_eps, 3).sum(axis=2), rtol=0, atol=1e-13)
    k2 = A.momenta(5, 16, m)
    np.testing.assert_array_equal(t_.dispersion(k2, [q[:2]], tt, mu), t_.dispersion(k2, [q[:2]], tt, mu, dim=2, band=0))


# ---------------------------------------------------------------- layout, regulator, threads
def test_output_layout_and_threads(oracle_mod):
    """[N_F][N_E], energy index fastest; threading changes nothing."""
    d = A.self_energy_order2()
    t = table(oracle_mod, d)
    beta = 2.0
    e = random_energies(d, 37)
    z = np.array([[1j * (2 * n + 1) * math.pi / beta] for n in range(3)])
    full = t.evaluate(e, z, beta)
    assert full.shape == (3, 37)
    for f in range(3):
        np.testing.assert_array_equal(full[f], t.evaluate(e, z[f:f + 1], beta)[0])
    np.testing.assert_array_equal(full, t.evaluate(e, z, beta, threads=4))


def test_regulator_convention(oracle_mod):
    """P10: eta shifts sigma=-1 leaves and frequency-free denominators only.  At Omega = 0 the
    bubble's denominators are purely real; eta = 1e-8 keeps a degenerate sample finite and moves
    ordinary samples by O(eta)."""
    t = table(oracle_mod, A.bubble())
    beta = 5.0
    e = np.array([[0.3, -0.7], [0.5, 0.5]])  # second sample: a = b exactly
    v0 = t.evaluate(e, [[0j]], beta, e_reg=0.0, quad=True)
    v1 = t.evaluate(e, [[0j]], beta, e_reg=1e-8, quad=True)
    assert np.isfinite(v1).all() and not np.isfinite(v0[0, 1])
    assert abs(v1[0, 0] - v0[0, 0]) < 1e-7 * abs(v0[0, 0])
    # with a non-zero frequency the regulator does not touch the bubble at all
    z = [[2j * math.pi / beta]]
    np.testing.assert_array_equal(t.evaluate(e, z, beta, e_reg=1e-8), t.evaluate(e, z, beta, e_reg=0.0))
