"""Slab-decomposed context (include/lgf.h lgf_*_sharded) with P virtual ranks on one B200:
against the CPU oracle at the north-star tolerances, and against the single-context path (same arithmetic: the
difference is summation order only).  No N > 1 GPU run is made anywhere: the ranks are virtual."""
import numpy as np
import pytest

import ensembles as E
import oracle
import paper_1301_3460_b200 as lgf
import slab_maps as slab

pytestmark = pytest.mark.gpu

ALPHA, TOL = 0.08, 1e-15
F_TOL, LINK_TOL = 1e-12, 1e-11


def theta_close(t, ref):
    return abs(t - ref) <= 1e-9 * max(ref, TOL)


@pytest.mark.parametrize("P", [1, 2, 4, 8])
def test_sharded_trajectory_C1_against_the_oracle(P):
    U, cfg = E.make_config("C1")
    dims, storage = cfg["dims"], cfg["storage"]
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    r_ref = o.fix(ALPHA, 0.0, 60, history=True)
    h_ref = np.array(r_ref["history"])
    n_ref = int(np.argmax(h_ref[:, 1] < TOL))
    sg = lgf.ShardedGaugeFixer(dims, P, storage)
    sg.load_links(U)
    assert np.array_equal(sg.get_links()[:, :, :2], U[:, :, :2])           # scatter to the slabs and back: bit exact
    F, th = sg.iterate(10, ALPHA)
    h = sg.get_history()
    assert len(h) == 11 and np.abs(h[:, 0] - h_ref[:11, 0]).max() <= F_TOL
    assert all(theta_close(h[k, 1], h_ref[k, 1]) for k in range(11))
    o2 = oracle.Oracle(dims, storage, fft_mode=1)
    o2.load(U)
    o2.iterate(10, ALPHA)
    assert np.abs(sg.get_links() - o2.get()).max() <= LINK_TOL
    sg.load_links(U)
    r = sg.fix(ALPHA, TOL, 1000)
    assert r["status"] == 0 and r["n_iter"] == n_ref, (r, n_ref)             # the stop iteration: exact (A19)
    assert abs(r["F"] - h_ref[n_ref, 0]) <= F_TOL and theta_close(r["theta"], h_ref[n_ref, 1])
    t = sg.traffic()
    m = slab.traffic_bytes(dims, P, 6 if storage == 12 else 9)
    assert (t["halo_u_bytes"], t["halo_x_bytes"], t["transpose_bytes"]) == (m["halo_u_bytes"], m["halo_x_bytes"], m["transpose_bytes"])
    sg.destroy()


@pytest.mark.parametrize("dims,storage,P", [((16, 16, 16, 32), 12, 4), ((8, 16, 4, 8), 18, 2), ((32, 8, 8, 16), 12, 8), ((64, 4, 4, 4), 12, 2)])
def test_sharded_equals_single_context(dims, storage, P):
    """Anisotropic shapes, both storage modes: F, theta of every iteration and the links after 12 iterations equal the
    single-context path's to rounding (same kernels' arithmetic; the (theta, F) partial sums are grouped differently), and
    lgf_fix stops at the same iteration."""
    U = E.noisy(dims, 31, 0.3)
    g1 = lgf.GaugeFixer(dims, storage)
    g1.load_links(U)
    g1.iterate(12, ALPHA)
    h1 = g1.get_history()
    sg = lgf.ShardedGaugeFixer(dims, P, storage)
    sg.load_links(U)
    sg.iterate(12, ALPHA)
    h = sg.get_history()
    assert np.abs(h[:, 0] - h1[:, 0]).max() <= 1e-14
    assert np.abs(h[:, 1] - h1[:, 1]).max() <= 1e-12 * h1[:, 1].max()
    assert np.abs(sg.get_links() - g1.get_links()).max() <= 1e-13
    g1.load_links(U)
    sg.load_links(U)
    r1, r = g1.fix(ALPHA, TOL, 2000), sg.fix(ALPHA, TOL, 2000)
    assert r1["status"] == 0 and r["status"] == 0 and r["n_iter"] == r1["n_iter"]
    assert abs(r["F"] - r1["F"]) <= F_TOL
    sg.destroy()
    g1.destroy()


def test_sharded_C3_shape_first_iterations():
    """32^3 x 64 (BASELINE.json configs[3] shape) on 4 virtual ranks: three iterations against the single-context
    default path, then the exchange volumes per iteration."""
    dims = (32, 32, 32, 64)
    Ud = E.noisy_device(dims, 4, 0.40)
    U = Ud.cpu().numpy()
    del Ud
    g1 = lgf.GaugeFixer(dims, 12)
    g1.load_links(U)
    F1, th1 = g1.iterate(3, ALPHA)
    sg = lgf.ShardedGaugeFixer(dims, 4, 12)
    sg.load_links(U)
    F, th = sg.iterate(3, ALPHA)
    assert abs(F - F1) <= 1e-14 and abs(th - th1) <= 1e-12 * th1
    assert np.abs(sg.get_links() - g1.get_links()).max() <= 1e-13
    t = sg.traffic()
    assert t["halo_u_bytes"] == 32 ** 3 * 96 and t["halo_x_bytes"] == 32 ** 3 * 64
    assert t["transpose_bytes"] == 2 * (32 ** 3 * 16 * 64) * 3 // 4
    sg.destroy()
    g1.destroy()


def test_sharded_argument_errors():
    with pytest.raises(lgf.LgfError):
        lgf.ShardedGaugeFixer((16, 16, 16, 16), 3)                      # not a power of two
    with pytest.raises(lgf.LgfError):
        lgf.ShardedGaugeFixer((16, 4, 16, 16), 8)                       # more ranks than x1 rows
    sg = lgf.ShardedGaugeFixer((8, 8, 8, 8), 2, 18)
    with pytest.raises(lgf.LgfError):
        sg.iterate(1, ALPHA)                                            # LGF_ERR_NOT_LOADED
    sg.destroy()
