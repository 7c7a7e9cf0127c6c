"""Labelled diagrams: the integer ``alpha`` / ``eps`` matrices of R0
(PAPER.md:207-231).  Only integers and graph bookkeeping live here.

Conventions:
* ``alpha[j]`` has length L = n_int + n_ext; internal labels first, the external
  label(s) LAST.
* ``eps[j]`` is a unit vector selecting the energy symbol of line j; lines with
  equal ``alpha`` share one symbol (reading P7).
* ``slot_is_fermionic[l]`` gives the statistics of frequency slot l (reading P5).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Diagram:
    name: str
    n_int: int
    n_ext: int
    alpha: np.ndarray  # int32 [n_g][n_int + n_ext]
    eps: np.ndarray  # int32 [n_g][n_eps]
    slot_is_fermionic: np.ndarray  # uint8 [n_int + n_ext]
    meta: dict = field(default_factory=dict)

    @property
    def n_g(self) -> int:
        return int(self.alpha.shape[0])

    @property
    def n_eps(self) -> int:
        return int(self.eps.shape[1])

    def symbol_alpha(self) -> np.ndarray:
        """alpha row of (any line carrying) each energy symbol: int32 [n_eps][L].
        This is the momentum combination of that symbol, Eq. 13."""
        out = np.zeros((self.n_eps, self.alpha.shape[1]), dtype=np.int32)
        seen = np.zeros(self.n_eps, dtype=bool)
        for j in range(self.n_g):
            (nz,) = np.nonzero(self.eps[j])
            assert len(nz) == 1 and self.eps[j, nz[0]] == 1, "R0 eps rows must be unit vectors"
            s = int(nz[0])
            if seen[s]:
                assert np.array_equal(out[s], self.alpha[j]), "lines sharing a symbol must share alpha"
            out[s] = self.alpha[j]
            seen[s] = True
        assert seen.all()
        return out

    def permuted(self, perm) -> "Diagram":
        """Same diagram with the Green's functions listed in another order
        (the ordering must not change the result)."""
        perm = np.asarray(perm)
        return Diagram(self.name + "_perm", self.n_int, self.n_ext, self.alpha[perm].copy(),
                       self.eps[perm].copy(), self.slot_is_fermionic.copy(), dict(self.meta))


def _mk(name, n_int, alpha, symbols, ext_fermionic, meta=None) -> Diagram:
    alpha = np.asarray(alpha, dtype=np.int32)
    n_eps = max(symbols) + 1
    eps = np.zeros((len(symbols), n_eps), dtype=np.int32)
    for j, s in enumerate(symbols):
        eps[j, s] = 1
    L = alpha.shape[1]
    stat = np.ones(L, dtype=np.uint8)
    stat[n_int:] = 1 if ext_fermionic else 0
    return Diagram(name, n_int, L - n_int, alpha, eps, stat, meta or {})


def order1_line() -> Diagram:
    """One line, one sum: alpha=(1,0).  Closed form I = f(-e1)."""
    return _mk("order1", 1, [[1, 0]], [0], True)


def bubble() -> Diagram:
    """Bare bubble: alpha=(1,0),(1,1), bosonic external frequency."""
    return _mk("bubble", 1, [[1, 0], [1, 1]], [0, 1], False)


def doubled_line_bubble() -> Diagram:
    """Bubble with line 1 doubled (self-energy-insertion shape): a true double pole."""
    return _mk("bubble_doubled", 1, [[1, 0], [1, 0], [1, 1]], [0, 0, 1], False)


def self_energy_order2() -> Diagram:
    """Second-order self-energy, Eq. 7 / Eq. 11; the alpha
    listing at PAPER.md:207-209 is missing and is read off Eq. 11 (reading P1)."""
    return _mk("se2", 2, [[1, 0, 0], [0, 1, 0], [-1, 1, 1]], [0, 1, 2], True)


def self_energy_order2_doubled(which: int = 0) -> Diagram:
    """Order-2 self-energy with line ``which`` doubled (shares its energy symbol)."""
    a = [[1, 0, 0], [0, 1, 0], [-1, 1, 1]]
    sym = [0, 1, 2]
    a.append(list(a[which]))
    sym.append(sym[which])
    return _mk(f"se2_doubled{which}", 2, a, sym, True)


def kron_identity(alpha: np.ndarray, d: int) -> np.ndarray:
    """A = alpha (x) I_d of Eq. 14: pure integer bookkeeping."""
    return np.kron(np.asarray(alpha), np.eye(d, dtype=np.asarray(alpha).dtype))


# --------------------------------------------------------------------------
# Seeded random 1PI Hubbard self-energy topologies (reading P23).
# --------------------------------------------------------------------------

def _connected(n, edges, skip=-1):
    adj = [[] for _ in range(n)]
    for i, (a, b) in enumerate(edges):
        if i == skip:
            continue
        adj[a].append(b)
        adj[b].append(a)
    seen = {0}
    stack = [0]
    while stack:
        v = stack.pop()
        for w in adj[v]:
            if w not in seen:
                seen.add(w)
                stack.append(w)
    return len(seen) == n


def random_self_energy(m: int, seed: int, max_tries: int = 10000) -> Diagram:
    """Order-m self-energy topology with contact interaction: m vertices, each
    with two outgoing and two incoming stubs; one in-stub at v_in and one
    out-stub at v_out are the external legs; the other 2m-1 out-stubs are paired
    with the 2m-1 in-stubs by a seeded permutation.  Rejected and redrawn if a
    line is a self-loop (tadpole), the graph is disconnected, or it has a bridge
    (not 1PI).  Labels: a seeded random spanning tree; the m chords carry the
    independent labels, tree lines follow from conservation at every vertex,
        sum_in alpha - sum_out alpha + [v = v_in] e_ext - [v = v_out] e_ext = 0.
    """
    assert m >= 2
    rng = np.random.Generator(np.random.PCG64(seed))
    for attempt in range(max_tries):
        v_in, v_out = (int(x) for x in rng.choice(m, size=2, replace=False))
        outs = [v for v in range(m) for _ in range(2)]
        ins = [v for v in range(m) for _ in range(2)]
        outs.remove(v_out)
        ins.remove(v_in)
        perm = rng.permutation(2 * m - 1)
        edges = [(outs[i], ins[int(perm[i])]) for i in range(2 * m - 1)]  # (source, target)
        if any(a == b for a, b in edges):
            continue
        if not _connected(m, edges):
            continue
        if any(not _connected(m, edges, skip=i) for i in range(len(edges))):
            continue
        break
    else:
        raise RuntimeError("no 1PI topology found")

    n_g = 2 * m - 1
    # seeded random spanning tree (randomised Kruskal)
    parent = list(range(m))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x

    in_tree = [False] * n_g
    for i in (int(x) for x in rng.permutation(n_g)):
        a, b = find(edges[i][0]), find(edges[i][1])
        if a != b:
            parent[a] = b
            in_tree[i] = True
    chords = [i for i in range(n_g) if not in_tree[i]]
    assert len(chords) == m
    L = m + 1
    alpha = np.zeros((n_g, L), dtype=np.int64)
    solved = [False] * n_g
    for rank, i in enumerate(chords):
        alpha[i, rank] = 1
        solved[i] = True
    # leaf stripping on the tree
    while not all(solved):
        progressed = False
        for v in range(m):
            unsolved = [i for i in range(n_g) if not solved[i] and v in edges[i]]
            if len(unsolved) != 1:
                continue
            i = unsolved[0]
            tot = np.zeros(L, dtype=np.int64)  # sum_in - sum_out of solved lines + external
            for j in range(n_g):
                if solved[j] and v in edges[j]:
                    if edges[j][1] == v:
                        tot += alpha[j]
                    if edges[j][0] == v:
                        tot -= alpha[j]
            if v == v_in:
                tot[m] += 1
            if v == v_out:
                tot[m] -= 1
            # line i enters v (target) -> +alpha_i, leaves v (source) -> -alpha_i
            alpha[i] = -tot if edges[i][1] == v else tot
            solved[i] = True
            progressed = True
        assert progressed
    assert np.abs(alpha).max() <= 1, "spanning-tree labels must be in {-1,0,1}"
    # conservation check at every vertex
    for v in range(m):
        tot = np.zeros(L, dtype=np.int64)
        for j in range(n_g):
            if edges[j][1] == v:
                tot += alpha[j]
            if edges[j][0] == v:
                tot -= alpha[j]
        tot[m] += (v == v_in) - (v == v_out)
        assert not tot.any()
    # lines with equal alpha share one energy symbol (P7)
    symbols, keys = [], {}
    for j in range(n_g):
        key = tuple(int(x) for x in alpha[j])
        if key not in keys:
            keys[key] = len(keys)
        symbols.append(keys[key])
    d = _mk(f"se{m}_seed{seed}", m, alpha.astype(np.int32), symbols, True,
            {"edges": edges, "v_in": v_in, "v_out": v_out, "chords": chords, "seed": seed,
             "attempts": attempt + 1})
    return d
