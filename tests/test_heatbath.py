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
