"""Diagram files (Fig. 2): ami_graph_parse / ami_graph_label.

What pins the labelling without re-running it: (i) conservation at every vertex, checked here in a
few lines of Python; (ii) a relabelling is a unimodular change of the summed momenta, so the value
of the diagram at momenta k under one set of labels equals its value at the transformed momenta
under the other -- both evaluated by the CPU oracle, which shares nothing with the library."""
import math
import os

import numpy as np
import pytest

import ami_inputs as A

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def ami():
    from paper_2311_17189_b200 import build
    build.build()
    import paper_2311_17189_b200 as pkg
    pkg.lib()
    return pkg


def assert_conserving(edges, alpha_all):
    """sum_in alpha - sum_out alpha = 0 at every vertex that more than one line touches."""
    deg = np.bincount(edges[:, :2].ravel())
    for v in np.nonzero(deg > 1)[0]:
        tot = alpha_all[edges[:, 1] == v].sum(axis=0) - alpha_all[edges[:, 0] == v].sum(axis=0)
        assert not tot.any(), f"not conserved at vertex {v}: {tot}"


def line_momenta(alpha, k, q):
    """K_j = sum_l alpha_jl k_l + alpha_j,ext q for every line j: [N][n_lines][2]."""
    m = k.shape[1]
    K = np.einsum("jl,nlc->njc", alpha[:, :m].astype(float), k)
    if alpha.shape[1] > m:
        K = K + alpha[:, m, None].astype(float)[None] * np.asarray(q, dtype=float)[None, None, :]
    return K


def values_agree(oracle_mod, d_ref, lab, match, seed, n=12):
    """Oracle value of d_ref at momenta k against the oracle value of the library's labelling `lab` at
    the momenta its chords carry under d_ref's labels.  match[g] = line of d_ref that is R0 row g of lab."""
    rng = np.random.default_rng(seed)
    m = d_ref.n_int
    assert lab.n_int == m and lab.n_g == d_ref.alpha.shape[0]
    k = rng.uniform(-math.pi, math.pi, size=(n, m, 2))
    q = np.array([0.7, -1.1])
    K_ref = line_momenta(np.asarray(d_ref.alpha), k, q)              # [n][n_g][2]
    # the chords of the library's labelling carry exactly one unit label each
    k_new = np.zeros_like(k)
    for l in range(m):
        rows = [g for g in range(lab.n_g) if (lab.alpha[g] == np.eye(m + lab.n_ext, dtype=np.int32)[l]).all()]
        assert rows, f"no line carries the bare label {l}"
        k_new[:, l] = K_ref[:, match[rows[0]]]
    K_new = line_momenta(lab.alpha, k_new, q)
    np.testing.assert_allclose(K_new, K_ref[:, match], atol=1e-12)   # every line keeps its momentum
    beta, t, mu = 3.0, 1.0, -0.2
    z = [np.array([1j * math.pi / beta])]
    o_ref = oracle_mod.OracleTable.from_diagram(d_ref)
    o_new = oracle_mod.OracleTable(lab.n_int, lab.n_ext, lab.alpha, lab.eps, lab.slot_is_fermionic)
    e_ref = o_ref.dispersion(k, [q], t, mu, quad=True)
    e_new = o_new.dispersion(k_new, [q], t, mu, quad=True)
    v_ref, S = o_ref.evaluate(e_ref, z, beta, quad=True, want_S=True)
    v_new = o_new.evaluate(e_new, z, beta, quad=True)
    assert np.max(np.abs(v_new[0] - v_ref[0]) / S[0]) < 1e-10


def test_parse_fig2_file(ami):
    edges = ami.read_graph(os.path.join(GOLDEN, "fig2_o2_g0_n0.graph"))
    want = [[0, 2, 1, 0], [2, 3, 0, 0], [3, 4, 1, 0], [4, 3, 1, 0], [4, 5, 0, 0], [2, 5, 1, 0], [5, 1, 1, 0]]
    assert edges.tolist() == want
    assert ami.read_graph("\n\n 1 0 1 7 \n# nothing\n0\t1\t1\t-2").tolist() == [[1, 0, 1, 7], [0, 1, 1, -2]]
    assert ami.read_graph("# empty\n").shape == (0, 4)
    for bad in ("0 1 1\n", "0 1 1 0 5\n", "0 x 1 0\n", "0 1 2 0\n", "-1 1 1 0\n", "0 1 1 0x\n"):
        with pytest.raises(ami.AmiError) as ei:
            ami.read_graph(bad)
        assert ei.value.code == -1


def test_label_fig2_is_the_order2_self_energy(ami, oracle_mod):
    edges = ami.read_graph(os.path.join(GOLDEN, "fig2_o2_g0_n0.graph"))
    lab = ami.label_graph(edges)
    assert (lab.n_int, lab.n_ext, lab.n_g, lab.n_eps) == (2, 1, 3, 3)
    assert lab.row_of_g.tolist() == [2, 3, 5]                      # C, D, F of Fig. 2
    assert lab.slot_is_fermionic.tolist() == [1, 1, 1]
    assert_conserving(edges, lab.alpha_all)
    assert lab.alpha_all[0].tolist() == [0, 0, 1] and lab.alpha_all[6].tolist() == [0, 0, 1]   # the legs carry q
    assert np.abs(lab.alpha_all).max() == 1
    # both interaction lines carry the same transfer (q minus the through-line F)
    assert lab.alpha_all[1].tolist() == lab.alpha_all[4].tolist() == (lab.alpha_all[0] - lab.alpha_all[5]).tolist()
    # Eq. 7 / Eq. 11 (reading P1): G(k1) G(k2) G(q - k1 + k2); C plays the third line, D the second, F the first
    values_agree(oracle_mod, A.self_energy_order2(), lab, match=[2, 1, 0], seed=1)
    tab = ami.AmiTable.from_diagram(lab, device=None)
    assert tab.info["n_terms"] == ami.AmiTable.from_diagram(A.self_energy_order2(), device=None).info["n_terms"]


def graph_of(d, split_vertices):
    """Edge list of a generated contact-interaction topology (ami_inputs meta), legs included; with
    split_vertices every 4-leg vertex becomes two 3-leg vertices joined by a bosonic line."""
    m, meta = d.n_int, d.meta
    lines = [(a, b) for a, b in meta["edges"]]
    rows = [(m, meta["v_in"], 1, 0)] + [(a, b, 1, 0) for a, b in lines] + [(meta["v_out"], m + 1, 1, 0)]
    if not split_vertices:
        return np.array(rows, dtype=np.int32), 1
    ins = {v: [] for v in range(m)}
    outs = {v: [] for v in range(m)}
    for i, (a, b, _, _) in enumerate(rows):
        if a < m:
            outs[a].append(i)
        if b < m:
            ins[b].append(i)
    new = [list(r) for r in rows]
    for v in range(m):
        assert len(ins[v]) == 2 and len(outs[v]) == 2
        for half in range(2):
            new[ins[v][half]][1] = 2 * v + half
            new[outs[v][half]][0] = 2 * v + half
    new[0][0], new[-1][1] = 2 * m, 2 * m + 1
    bosons = [[2 * v, 2 * v + 1, 0, 0] for v in range(m)]
    return np.array(bosons + new, dtype=np.int32), m + 1     # bosons first: R0 rows keep their order


@pytest.mark.parametrize("split", [False, True])
@pytest.mark.parametrize("m,seed", [(2, 0), (3, 1), (3, 4), (4, 0), (4, 7), (5, 2)])
def test_label_random_topologies(ami, oracle_mod, m, seed, split):
    d = A.random_self_energy(m, seed)
    edges, first_line = graph_of(d, split)
    lab = ami.label_graph(edges)
    assert (lab.n_int, lab.n_ext, lab.n_g) == (m, 1, 2 * m - 1)
    assert lab.row_of_g.tolist() == list(range(first_line, first_line + 2 * m - 1))
    assert_conserving(edges, lab.alpha_all)
    # chords carry unit labels, in file order
    units = [g for g in range(lab.n_g) if np.abs(lab.alpha[g]).sum() == 1 and lab.alpha[g, :m].sum() == 1]
    assert [int(np.argmax(lab.alpha[g])) for g in units][:m] == list(range(m))
    # equal labels <=> shared symbol
    for a in range(lab.n_g):
        for b in range(lab.n_g):
            assert (lab.alpha[a] == lab.alpha[b]).all() == (lab.eps[a] == lab.eps[b]).all()
    values_agree(oracle_mod, d, lab, match=list(range(2 * m - 1)), seed=seed)


def test_label_bubble_without_and_with_bosonic_legs(ami):
    """A closed fermion loop has no legs (n_ext = 0); with bosonic legs the external slot is bosonic."""
    lab = ami.label_graph([[0, 1, 1, 0], [1, 0, 1, 0]])
    assert (lab.n_int, lab.n_ext, lab.n_g, lab.n_eps) == (1, 0, 2, 1)     # both lines carry k0: a double pole
    lab = ami.label_graph([[2, 0, 0, 0], [0, 1, 1, 0], [1, 0, 1, 0], [1, 3, 0, 0]])
    assert (lab.n_int, lab.n_ext, lab.n_g, lab.n_eps) == (1, 1, 2, 2)
    assert lab.slot_is_fermionic.tolist() == [1, 0]
    assert_conserving(lab.edges, lab.alpha_all)
    d = A.bubble()
    assert sorted(map(tuple, np.abs(lab.alpha).tolist())) == sorted(map(tuple, np.abs(np.asarray(d.alpha)).tolist()))


def test_label_errors(ami):
    E = ami.AmiError
    for bad, code in [
        ([[0, 1, 1, 0], [1, 2, 1, 0], [2, 1, 1, 0]], -1),                       # one leg only
        ([[0, 1, 1, 0], [1, 0, 1, 0], [2, 3, 1, 0], [3, 2, 1, 0]], -1),         # two pieces
        ([[4, 0, 1, 0], [0, 1, 0, 0], [0, 1, 0, 0], [1, 0, 1, 0], [1, 5, 1, 0]], -6),   # a loop of bosonic lines
        ([[4, 0, 1, 0], [0, 1, 1, 0], [1, 0, 1, 0], [1, 5, 0, 0]], -1),         # legs of different statistics
        ([[0, 1, 1, 0]], -1),                                                   # a line that touches nothing
    ]:
        with pytest.raises(E) as ei:
            ami.label_graph(bad)
        assert ei.value.code == code, bad
    import ctypes as C
    edges = np.array([[0, 1, 1, 0], [1, 0, 1, 0]], dtype=np.int32)
    small = np.zeros(1, dtype=np.int32)
    sz = [C.c_int32(0) for _ in range(4)]
    rc = ami.lib().ami_graph_label(edges.ctypes.data, 2, *[C.byref(x) for x in sz], None, None, small.ctypes.data,
                                   None, None, 1)
    assert rc == -1                                                             # capacity
    assert ami.lib().ami_graph_label(None, 0, *[C.byref(x) for x in sz], None, None, None, None, None, 0) == -1
