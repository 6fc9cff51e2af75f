"""Pins of the oracle's fraction <-> state conversions (Eq. 1): hand values, identities, round trips."""
import numpy as np
import pytest

import mechgen as mg
from mechgen import MechBuilder
from oracle import Oracle

R = 8314.46261815324
CP = lambda a0: [a0, 0, 0, 0, 0, 0.0, 1.0]


def _mech(W):
    mb = MechBuilder()
    for w in W:
        mb.add_species(w, CP(3.5))
    mb.add_reaction({0: 1}, {1: 1}, 1e5, 0.0, 1000.0)
    return mb.build()


def test_hand_values_two_species():
    # X = (1/2, 1/2), W = (2, 32): Y = (2/34, 32/34); T = 1000 K, P = R Pa, V = 2 m^3: n_tot = 2/1000 kmol
    o = Oracle(_mech([2.0, 32.0]))
    phi, par = o.state_from_fractions(mg.CONP, 0, [1000.0], [R], [2.0], [[0.5, 0.5]])
    assert phi.tolist() == [[1000.0, 2.0, 1e-3]] and par.tolist() == [R]
    phi2, par2 = o.state_from_fractions(mg.CONV, 1, [1000.0], [R], [2.0], [[2.0 / 34.0, 32.0 / 34.0]])
    assert phi2[0, 0] == 1000.0 and phi2[0, 1] == R and par2[0] == 2.0
    assert phi2[0, 2] == pytest.approx(1e-3, rel=1e-15)
    assert o.fractions_from_state(mg.CONP, 1, phi, par)[0] == pytest.approx([2.0 / 34.0, 32.0 / 34.0], rel=1e-15)
    assert o.fractions_from_state(mg.CONP, 0, phi, par)[0] == pytest.approx([0.5, 0.5], rel=1e-15)
    # equal molecular weights: mass fractions are mole fractions
    o = Oracle(_mech([30.0, 30.0, 30.0]))
    Y = [[0.2, 0.5, 0.3]]
    a = o.state_from_fractions(mg.CONP, 1, [1500.0], [2e5], [0.1], Y)
    b = o.state_from_fractions(mg.CONP, 0, [1500.0], [2e5], [0.1], Y)
    np.testing.assert_allclose(a[0], b[0], rtol=1e-15)


@pytest.mark.parametrize("c", [1, 3])
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_identities_and_round_trip(c, mode):
    m = mg.config_mechanism(c)
    o = Oracle(m)
    st = mg.config_states(c, 64)
    ns = o.ns
    W = np.asarray(m["mol_weight"])
    phi0, par0 = o.pack(st, mode)                       # mechgen built these from mole fractions with n = X P V / (R T)
    for kind in (0, 1):
        f = o.fractions_from_state(mode, kind, phi0, par0)
        assert f.shape == (64, ns) and np.all(f > -1e-15)
        np.testing.assert_allclose(f.sum(axis=1), 1.0, rtol=1e-13)          # fractions sum to one
        phi1, par1 = o.state_from_fractions(mode, kind, st["T"], st["P"], st["V"], f)
        np.testing.assert_allclose(phi1, phi0, rtol=1e-12)                  # round trip
        assert par1.tobytes() == par0.tobytes()
    X = o.fractions_from_state(mode, 0, phi0, par0); Y = o.fractions_from_state(mode, 1, phi0, par0)
    # the two kinds are related by the mean molecular weight: Y_k / X_k = W_k / W_mean, the same W_mean for every k
    wmean = (X * W).sum(axis=1, keepdims=True)
    np.testing.assert_allclose(Y * wmean, X * W, rtol=1e-13)
    np.testing.assert_allclose(1.0 / (Y / W).sum(axis=1), wmean[:, 0], rtol=1e-13)
    # total moles (incl. the last species) = P V / (R T): the ideal-gas law closes the state
    ntot = st["P"] * st["V"] / (R * st["T"])
    np.testing.assert_allclose(phi0[:, 2:].sum(axis=1) + X[:, -1] * ntot, ntot, rtol=1e-13)
