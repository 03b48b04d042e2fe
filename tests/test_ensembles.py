"""Input generators (ensembles/: data, not method).  CPU only."""
import numpy as np

import ensembles as E
import oracle


def test_noisy_device_follows_the_noisy_recipe():
    """ensembles.noisy_device (the torch restatement of `noisy` used for C4, reading A12b): special unitary to rounding,
    reproducible from (seed, stream), and statistically the same ensemble as `noisy` -- average plaquette
    exp(-(8/3) eps^2) (reading A12) and the Haar-start values theta_0 = 128/9, F_0 = 0 of pin P5."""
    dims = (8, 8, 8, 8)
    V = 4096
    for eps in (0.25, 0.35, 0.45):
        U = E.noisy_device(dims, 5, eps, device="cpu").numpy()
        assert U.shape == (V, 4, 3, 3)
        assert np.abs(U @ U.conj().swapaxes(-1, -2) - np.eye(3)).max() < 1e-14
        assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
        o = oracle.Oracle(dims, 18)
        o.load(U)
        o2 = oracle.Oracle(dims, 18)
        o2.load(E.noisy(dims, 5, eps))
        assert abs(o.plaquette() - np.exp(-(8.0 / 3.0) * eps * eps)) < 0.015      # leading order in eps
        assert abs(o.plaquette() - o2.plaquette()) < 0.005
        F, th = o.measure()
        assert abs(th - 128.0 / 9.0) < 0.5 and abs(F) < 0.02
    assert np.array_equal(U, E.noisy_device(dims, 5, 0.45, device="cpu").numpy())
    assert not np.array_equal(U, E.noisy_device(dims, 5, 0.45, stream=1, device="cpu").numpy())
    # pure gauge limit: eps = 0 gives U = h(x) h^dagger(x+mu), plaquette 1
    o.load(E.noisy_device(dims, 5, 0.0, device="cpu").numpy())
    assert abs(o.plaquette() - 1.0) < 1e-13
