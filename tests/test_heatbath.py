"""The Wilson-action heat-bath generator (ensembles/heatbath.py; inputs only) against what statistical mechanics fixes:
strong coupling <P> = beta/18 + O(beta^2), weak coupling <1 - P> = (N^2 - 1)/(4 beta) = 2/beta (equipartition over the
8 x 3 physical modes per site), special unitarity, reproducibility from the seed."""
import numpy as np
import pytest

import ensembles as E
from ensembles import heatbath as H

DIMS = (4, 4, 4, 4)


def _mean_plaquette(beta, hot, seeds):
    return float(np.mean([H.average_plaquette(E.wilson(DIMS, beta, 14, s, hot=hot), DIMS) for s in seeds]))


def test_strong_coupling_plaquette():
    beta = 0.6
    p = _mean_plaquette(beta, True, (1, 2, 3, 4, 5, 6))
    assert abs(p - beta / 18.0) < 0.006                      # statistical error ~0.002 on 6 x 1536 plaquettes


def test_weak_coupling_plaquette():
    beta = 30.0
    p = _mean_plaquette(beta, False, (1, 2, 3))
    assert abs((1.0 - p) - 2.0 / beta) < 0.05 * 2.0 / beta


def test_special_unitary_and_seeded():
    U = E.wilson(DIMS, 5.7, 6, 11).numpy()
    assert np.abs(np.einsum("xmij,xmkj->xmik", U, U.conj()) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1.0).max() < 1e-14
    assert np.array_equal(U, E.wilson(DIMS, 5.7, 6, 11).numpy())
    assert not np.array_equal(U, E.wilson(DIMS, 5.7, 6, 12).numpy())
    p = H.average_plaquette(E.wilson(DIMS, 5.7, 6, 11), DIMS)
    assert 0.45 < p < 0.65                                    # between the two limits, where thermalised beta ~ 6 sits


def test_overrelaxation_is_microcanonical():
    """An over-relaxation sweep (ref. [6]) changes every link and leaves the Wilson action -- the average
    plaquette -- unchanged to rounding, and the links special unitary."""
    U = E.wilson(DIMS, 5.8, 8, 21)
    p0 = H.average_plaquette(U, DIMS)
    U1 = H.overrelax_sweep(U, DIMS)
    p1 = H.average_plaquette(U1, DIMS)
    assert abs(p1 - p0) < 1e-13, (p0, p1)
    d = (U1 - U).abs().amax(dim=(1, 2, 3)).numpy()
    assert d.min() > 1e-6                                      # no site was left alone
    V = U1.numpy()
    assert np.abs(np.einsum("xmij,xmkj->xmik", V, V.conj()) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(V) - 1.0).max() < 1e-13
    # two reflections about a fixed staple are the identity; a whole sweep changes the staples, so it is not one: only
    # the action is conserved
    U2 = H.overrelax_sweep(U1, DIMS)
    assert abs(H.average_plaquette(U2, DIMS) - p0) < 1e-13


def test_heatbath_with_overrelaxation_thermalises_to_the_same_plaquette():
    """Mixing over-relaxation sweeps in must not change the equilibrium: same <P> within the statistical error, and the
    plaquette history reaches a plateau (drift between the last two windows no larger than their spread)."""
    beta = 5.7
    hist = []
    E.wilson(DIMS, beta, 24, 5, overrelax=2, history=hist)
    mean, spread, drift = H.plateau(hist, window=6)
    assert len(hist) == 24 and abs(drift) <= max(spread, 0.02)
    p_hb = float(np.mean([H.average_plaquette(E.wilson(DIMS, beta, 14, s), DIMS) for s in (1, 2, 3)]))
    p_or = float(np.mean([H.average_plaquette(E.wilson(DIMS, beta, 10, s, overrelax=2), DIMS) for s in (1, 2, 3)]))
    assert abs(p_hb - p_or) < 0.03, (p_hb, p_or)
