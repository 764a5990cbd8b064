"""Pins of the oracle's general-p couplings (Eq. (2); reading R32)."""
import numpy as np
import pytest

from oracle import ref
import workloads as wl
from tests import helpers as H


def test_p_half_is_the_default_init_bit_for_bit():
    b = wl.betas_linear(0.2, 2.0, 8)
    a = ref.Oracle(8, 2, 4, 8, b, wl.SEED)
    c = ref.Oracle(8, 2, 4, 8, b, wl.SEED, p_ferro=0.5)
    assert np.array_equal(a.get_couplings(), c.get_couplings())
    assert H.crc(c.get_couplings()) == "1cbe91f5"            # the survey's worked example W1 (tests/golden)
    assert np.array_equal(a.get_energy(), c.get_energy())


def test_p_one_is_the_ferromagnet_and_p_zero_the_antiferromagnet():
    L, d, S, T = 6, 3, 2, 3
    b = wl.betas_linear(0.2, 1.0, T)
    f = ref.Oracle(L, d, S, T, b, wl.SEED, p_ferro=1.0)
    assert (f.get_couplings() == 1).all()
    f.set_spins(np.ones((S, 2, T, L ** d), dtype=np.int8))
    assert (f.recompute_energy()[0] == -d * L ** d).all()     # closed form: all bonds satisfied
    a = ref.Oracle(L, d, S, T, b, wl.SEED, p_ferro=0.0)
    assert (a.get_couplings() == -1).all()
    stag = (1 - 2 * H.colours(L, d)).astype(np.int8)          # Neel state satisfies every antiferromagnetic bond (L even)
    a.set_spins(np.broadcast_to(stag, (S, 2, T, L ** d)).copy())
    assert (a.recompute_energy()[0] == -d * L ** d).all()


@pytest.mark.parametrize("p", [0.1, 0.25, 0.7, 0.93])
def test_fraction_of_ferromagnetic_bonds_and_nesting(p):
    o = ref.Oracle(16, 3, 8, 1, np.array([0.5]), wl.SEED, p_ferro=p)
    J = o.get_couplings()
    n = J.size
    assert abs((J == 1).mean() - p) < 5 * np.sqrt(p * (1 - p) / n)       # binomial, 5 sigma
    # the same Philox word decides every p: the +1 bonds at p are a subset of those at any larger p
    J2 = ref.Oracle(16, 3, 8, 1, np.array([0.5]), wl.SEED, p_ferro=min(1.0, p + 0.05)).get_couplings()
    assert ((J == 1) <= (J2 == 1)).all()
    with pytest.raises(ValueError):
        ref.Oracle(4, 2, 1, 1, np.array([0.5]), wl.SEED, p_ferro=1.5)
