"""Seeded input generators: determinism, ranges, graph properties (reading P22, P23)."""
import math

import numpy as np
import pytest

import ami_inputs as A


def test_rng_reference_values():
    """splitmix64 finaliser spec, first values written out by hand from the specification in
    ami_inputs/rng.py (pure-Python big-int arithmetic, no numpy)."""
    M = (1 << 64) - 1

    def u(seed, ctr):
        z = (seed + 0x9E3779B97F4A7C15 * (ctr + 1)) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        z ^= z >> 31
        return (z >> 11) * 2.0 ** -53

    ctr = np.array([0, 1, 2, 12345678901, 2 ** 40 + 3], dtype=np.uint64)
    got = A.uniform01(20231118, ctr)
    want = [u(20231118, int(c)) for c in ctr]
    assert got.tolist() == want


def test_momenta_range_and_streaming():
    k = A.momenta(3, 1000, 4)
    assert k.shape == (1000, 4, 2) and k.min() >= -math.pi and k.max() < math.pi
    np.testing.assert_array_equal(A.momenta(3, 100, 4, start=500), k[500:600])  # stateless
    assert abs(k.mean()) < 0.1 and abs(k.std() - 2 * math.pi / math.sqrt(12)) < 0.05


@pytest.mark.parametrize("m", [2, 3, 4, 5, 6, 8])
def test_random_topology_properties(m):
    for seed in range(5):
        d = A.random_self_energy(m, seed)
        assert d.n_g == 2 * m - 1 and d.alpha.shape == (2 * m - 1, m + 1)
        assert np.abs(d.alpha).max() == 1
        # the m chords carry unit labels; the external label is on at least one line
        chords = d.meta["chords"]
        np.testing.assert_array_equal(d.alpha[chords][:, :m], np.eye(m, dtype=np.int32))
        assert np.abs(d.alpha[:, m]).sum() >= 1
        # eps rows are unit vectors, equal alpha <=> same symbol
        assert (d.eps.sum(axis=1) == 1).all()
        sym = d.eps.argmax(axis=1)
        for i in range(d.n_g):
            for j in range(d.n_g):
                assert (sym[i] == sym[j]) == bool((d.alpha[i] == d.alpha[j]).all())
        # deterministic
        np.testing.assert_array_equal(d.alpha, A.random_self_energy(m, seed).alpha)
        # no tadpoles
        assert all(a != b for a, b in d.meta["edges"])


def test_configs_build():
    for name in A.CONFIGS + ("stress8",):
        c = A.get_config(name)
        assert c.z_ext.shape[1] == c.diagram.n_ext
        assert c.momenta(4).shape == (4, c.diagram.n_int, 2)
    c3 = A.get_config("cfg3")
    assert c3.diagram.n_g == 7 and c3.n_samples == 1_000_000 and c3.betas == (8.0,)
    assert A.get_config("cfg4").e_reg == 1e-8 and A.get_config("cfg5").z_ext.shape == (64, 1)


def test_energies_range_and_streaming():
    """Energies of the paper's first example: uniform in [-a, a), stateless."""
    from ami_inputs.rng import energies
    e = energies(5, 4000, 3, 8.0)
    assert e.shape == (4000, 3) and e.min() >= -8.0 and e.max() < 8.0
    np.testing.assert_array_equal(energies(5, 100, 3, 8.0, start=700), e[700:800])
    assert abs(e.mean()) < 0.2 and abs(e.std() - 16 / math.sqrt(12)) < 0.1
    c = A.get_config("paper_ex1")
    assert c.z_ext.shape == (100, 1) and c.betas == (1.0,) and c.n_samples == 1_000_000
    assert c.z_ext[3, 0] == 1j * 7 * math.pi
    np.testing.assert_array_equal(c.energies(10, start=5), energies(c.seed, 10, 3, 8.0, start=5))
