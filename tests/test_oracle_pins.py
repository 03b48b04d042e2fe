"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

Each test names the pin (P1..P17, SURVEY.md section 8(c) / DESIGN.md) and the passage it fixes.
The paper prints no worked example, no F or theta values (PAPER.md:49 is an absent figure), so the
pins are closed forms, invariants, brute force and special cases that reduce to numpy routines.
"""
import numpy as np
import pytest

import ensembles as E
import oracle

ALPHA = 0.08


def shift(A, dims, mu, s=-1):
    """A(x - s*mu_hat) -> with s=-1: A(x+mu_hat), indexed by x."""
    L0, L1, L2, L3 = dims
    return np.roll(A.reshape((L3, L2, L1, L0) + A.shape[1:]), s, axis=3 - mu).reshape(A.shape)


def dag(A):
    return A.conj().swapaxes(-1, -2)


# ------------------------------------------------------------------ DFT (P1, P2, P7 ingredients)
def test_P1_dft_equals_bruteforce_4d_on_4444():
    dims = (4, 4, 4, 4)
    V = 256
    rng = np.random.default_rng(11)
    f = rng.standard_normal(V) + 1j * rng.standard_normal(V)
    # brute force O(V^2): full V x V kernel exp(-2 pi i sum_mu n_mu x_mu / L_mu), x0 fastest
    idx = np.arange(V)
    c = np.stack([(idx // (4 ** k)) % 4 for k in range(4)], axis=1)
    phase = (c[:, None, :] * c[None, :, :] / 4.0).sum(-1)
    K = np.exp(-2j * np.pi * phase)
    brute = K @ f
    for mode in (0, 1):
        got = oracle.dft4(dims, f, -1, mode)
        assert np.abs(got - brute).max() < 1e-13
        gotp = oracle.dft4(dims, f, +1, mode)
        assert np.abs(gotp - K.conj() @ f).max() < 1e-13


def test_P1b_dft_matches_numpy_fftn_anisotropic_and_non_pow2():
    rng = np.random.default_rng(12)
    for dims in [(4, 8, 2, 16), (4, 4, 6, 8), (3, 5, 4, 2)]:
        V = int(np.prod(dims))
        f = rng.standard_normal(V) + 1j * rng.standard_normal(V)
        ref = np.fft.fftn(f.reshape(dims[::-1])).reshape(-1)  # x0 fastest == last numpy axis
        got = oracle.dft4(dims, f, -1, 0)
        assert np.abs(got - ref).max() < 1e-12
        if all((d & (d - 1)) == 0 for d in dims):
            got1 = oracle.dft4(dims, f, -1, 1)
            assert np.abs(got1 - ref).max() < 1e-12


def test_P1c_axis_order_is_x0_fastest():
    # a plane wave along axis mu with wave number k must land on n_mu = k only
    dims = (4, 8, 16, 2)
    V = int(np.prod(dims))
    idx = np.arange(V)
    strides = [1, 4, 32, 512]
    for mu, k in [(0, 1), (1, 3), (2, 5), (3, 1)]:
        x = (idx // strides[mu]) % dims[mu]
        f = np.exp(2j * np.pi * k * x / dims[mu])
        F = oracle.dft4(dims, f, -1, 0)
        peak = int(np.argmax(np.abs(F)))
        assert peak == k * strides[mu]
        assert abs(F[peak] - V) < 1e-10
        F[peak] = 0
        assert np.abs(F).max() < 1e-10


def test_P2_parseval_and_inverse():
    dims = (8, 4, 4, 8)
    V = int(np.prod(dims))
    rng = np.random.default_rng(13)
    f = rng.standard_normal(V) + 1j * rng.standard_normal(V)
    for mode in (0, 1):
        F = oracle.dft4(dims, f, -1, mode)
        assert abs((np.abs(f) ** 2).sum() - (np.abs(F) ** 2).sum() / V) < 1e-10
        back = oracle.dft4(dims, F, +1, mode) / V
        assert np.abs(back - f).max() < 1e-13


def test_filter_weights_closed_form():
    # w(n) = 16 / sum_mu 4 sin^2(pi n_mu / L_mu); w(0) = 0; max momentum (pi,pi,pi,pi) -> p2 = 16 -> w = 1  [NS step 2]
    dims = (4, 8, 4, 16)
    w = oracle.fa_weights(dims)
    assert w[0] == 0.0
    corner = 2 + 4 * (4 + 8 * (2 + 4 * 8))
    assert abs(w[corner] - 1.0) < 1e-15
    # single unit of momentum along axis 1: p2 = 4 sin^2(pi/8)
    assert abs(w[4] - 16.0 / (4 * np.sin(np.pi / 8) ** 2)) < 1e-12
    assert np.all(w[1:] >= 1.0 - 1e-15)
    # even in n
    idx = np.arange(len(w))
    c = [(idx // s) % L for s, L in zip([1, 4, 32, 128], dims)]
    neg = sum(((-ci) % L) * s for ci, s, L in zip(c, [1, 4, 32, 128], dims))
    assert np.abs(w - w[neg]).max() < 1e-12


# ------------------------------------------------------------------ S1: Delta, theta, F (P3, P4, P5)
@pytest.fixture(scope="module")
def haar_links_8():
    dims = (8, 8, 8, 8)
    rng = np.random.Generator(np.random.Philox(key=[99, 0]))
    U = E.haar_su3(rng, 4 * 4096).reshape(4096, 4, 3, 3)
    return dims, U


def test_P18_filter_inverts_the_lattice_laplacian():
    """p^2(n) = sum_mu 4 sin^2(pi n_mu/L_mu) are the eigenvalues of minus the nearest-neighbour lattice Laplacian, so the
    Fourier-accelerated field obeys, site by site and with no transform in sight,
        sum_mu [2 X(x) - X(x+mu) - X(x-mu)] = p2max * (Delta(x) - mean Delta) = 16 Delta(x)       (P4: mean Delta = 0).
    Fixes the filter (every p^2 term, p2max, the zero mode), the 1/V of the inverse transform and the axis/wrap
    handling of S2 together, on an anisotropic lattice, in both FFT modes."""
    dims = (4, 8, 6, 4)
    U = E.noisy(dims, 21, 0.4)
    for mode in ((0, 1) if all((d & (d - 1)) == 0 for d in dims) else (0,)):
        o = oracle.Oracle(dims, 18, fft_mode=mode)
        o.load(U)
        D = o.delta().reshape(dims[::-1] + (3, 3))
        X = o.fa_field().reshape(dims[::-1] + (3, 3))
        lap = np.zeros_like(X)
        for ax in range(4):
            lap += 2.0 * X - np.roll(X, 1, axis=ax) - np.roll(X, -1, axis=ax)
        assert np.abs(lap - 16.0 * D).max() <= 1e-12 * np.abs(X).max()
    dims = (8, 4, 4, 16)
    U = E.noisy(dims, 22, 0.4)
    o = oracle.Oracle(dims, 12, fft_mode=1)
    o.load(U)
    D = o.delta().reshape(dims[::-1] + (3, 3))
    X = o.fa_field().reshape(dims[::-1] + (3, 3))
    lap = sum(2.0 * X - np.roll(X, 1, axis=ax) - np.roll(X, -1, axis=ax) for ax in range(4))
    assert np.abs(lap - 16.0 * D).max() <= 1e-12 * np.abs(X).max()


def test_P3_P4_delta_traceless_antihermitian_zero_sum(haar_links_8):
    dims, U = haar_links_8
    o = oracle.Oracle(dims, 18)
    o.load(U)
    D = o.delta()
    assert np.abs(np.trace(D, axis1=1, axis2=2)).max() < 1e-14
    assert np.abs(D + dag(D)).max() < 1e-14
    assert np.abs(D.sum(0)).max() < 1e-11  # P4: every link enters once with each sign
    # independent numpy restatement of A(x) with explicit shifts (catches a wrong neighbour direction)
    A = sum(shift(U[:, mu], dims, mu, +1) - U[:, mu] for mu in range(4))
    Dn = A - dag(A)
    Dn = Dn - np.trace(Dn, axis1=1, axis2=2)[:, None, None] * np.eye(3) / 3
    assert np.abs(D - Dn).max() < 1e-14
    F, th = o.measure()
    assert abs(th - (np.abs(Dn) ** 2).sum() / (3 * 4096)) < 1e-12
    assert abs(F - np.trace(U, axis1=2, axis2=3).real.sum() / (12 * 4096)) < 1e-14


def test_P5_theta0_normalisation_haar(haar_links_8):
    # independent Haar links: E Tr[Delta Delta^dag] = 48 - 16/3 -> theta_0 = 128/9, F_0 -> 0
    dims, U = haar_links_8
    o = oracle.Oracle(dims, 18)
    o.load(U)
    F, th = o.measure()
    assert abs(th - 128.0 / 9.0) < 0.25
    assert abs(F) < 0.02


# ------------------------------------------------------------------ S2 packing + convention (P6, P7)
def test_P6_packed_transform_equals_nine_separate(haar_links_8):
    """The 4 packed complex fields (D01, D02, D12, Im D00 + i Im D11) carry all of X because the
    filter is real and even in n; this is the identity the CUDA layout relies on."""
    dims, U = haar_links_8
    V = 4096
    o = oracle.Oracle(dims, 18)
    o.load(U)
    D = o.delta()
    X = o.fa_field()
    w = oracle.fa_weights(dims)

    def fa(f):
        return oracle.dft4(dims, oracle.dft4(dims, f, -1, 0) * w, +1, 0) / V

    x01, x02, x12 = fa(D[:, 0, 1]), fa(D[:, 0, 2]), fa(D[:, 1, 2])
    c = fa(D[:, 0, 0].imag + 1j * D[:, 1, 1].imag)
    assert np.abs(X[:, 0, 1] - x01).max() < 1e-13
    assert np.abs(X[:, 1, 0] + x01.conj()).max() < 1e-13
    assert np.abs(X[:, 0, 2] - x02).max() < 1e-13
    assert np.abs(X[:, 2, 0] + x02.conj()).max() < 1e-13
    assert np.abs(X[:, 1, 2] - x12).max() < 1e-13
    assert np.abs(X[:, 2, 1] + x12.conj()).max() < 1e-13
    assert np.abs(X[:, 0, 0] - 1j * c.real).max() < 1e-13
    assert np.abs(X[:, 1, 1] - 1j * c.imag).max() < 1e-13
    assert np.abs(X[:, 2, 2] + 1j * (c.real + c.imag)).max() < 1e-13
    # X traceless anti-Hermitian
    assert np.abs(np.trace(X, axis1=1, axis2=2)).max() < 1e-13
    assert np.abs(X + dag(X)).max() < 1e-13


def test_P7_exponent_sign_convention_immaterial(haar_links_8):
    dims, U = haar_links_8
    o = oracle.Oracle(dims, 18)
    o.load(U)
    X1 = o.fa_field()
    o.set_variant(1, +1)
    X2 = o.fa_field()
    assert np.abs(X1 - X2).max() < 1e-13


# ------------------------------------------------------------------ sign, alpha/2, filter, 1/V (P8, P9)
def test_P8_dF_dalpha_closed_form(haar_links_8):
    """dF/dalpha at 0 = (1/(4 N_d N_c V)) sum_x Tr[X Delta^dag]; without the filter = theta/16."""
    dims, U = haar_links_8
    V = 4096
    for accel in (1, 0):
        o = oracle.Oracle(dims, 18)
        o.set_variant(accel, -1)
        o.load(U)
        F0, th0 = o.measure()
        D, X = o.delta(), o.fa_field()
        pred = np.einsum("xij,xij->", X, D.conj()).real / (4 * 4 * 3 * V)
        if not accel:
            assert abs(pred - th0 / 16.0) < 1e-12
        h = 1e-5
        Fp = o.F_of_g(o.g_field(+h))
        Fm = o.F_of_g(o.g_field(-h))
        fd = (Fp - Fm) / (2 * h)
        assert pred > 0
        assert abs(fd - pred) < 1e-6 * abs(pred) + 1e-8   # sign (A1), alpha/2 (A2), filter and 1/V together


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (4, 8, 4, 16)])
@pytest.mark.parametrize("alpha", [0.08, 0.05])
def test_P9_linearised_rate(dims, alpha):
    """U = h(x) h^dag(x+mu) with h = exp(i s H), s -> 0: every mode contracts by (1 - 16 alpha) per
    iteration, so theta_{k+1}/theta_k = (1 - 16 alpha)^2 -- pins p2max = 16, alpha/2, 1/V, the sign."""
    V = int(np.prod(dims))
    rng = np.random.Generator(np.random.Philox(key=[5, 1]))
    h = E.expi_hermitian(E.gaussian_su3_algebra(rng, V), 1e-5)
    U = np.stack([h @ dag(shift(h, dims, mu)) for mu in range(4)], axis=1)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    _, th0 = o.measure()
    _, th1 = o.iterate(1, alpha)
    _, th2 = o.iterate(1, alpha)
    r = (1 - 16 * alpha) ** 2
    assert abs(th1 / th0 - r) < 2e-4 * r
    assert abs(th2 / th1 - r) < 2e-4 * r


def test_P9b_alpha_one_sixteenth_is_quadratic():
    dims = (4, 4, 4, 4)
    rng = np.random.Generator(np.random.Philox(key=[5, 2]))
    h = E.expi_hermitian(E.gaussian_su3_algebra(rng, 256), 1e-4)
    U = np.stack([h @ dag(shift(h, dims, mu)) for mu in range(4)], axis=1)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    _, th0 = o.measure()
    _, th1 = o.iterate(1, 1.0 / 16.0)
    assert th1 < 1e-6 * th0


# ------------------------------------------------------------------ S3/S4 (P10, P11, P15)
def test_P10_projection_is_special_unitary():
    rng = np.random.default_rng(3)
    n = 2000
    H = rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))
    X = H - dag(H)
    X -= np.trace(X, axis1=1, axis2=2)[:, None, None] * np.eye(3) / 3
    g = oracle.project(X, ALPHA)
    assert np.abs(g @ dag(g) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(g) - 1).max() < 1e-14
    # first row is M0 normalised; second row is in span(M0, M1) with positive coefficient on M1  [NS step 3]
    M = np.eye(3) + 0.5 * ALPHA * X
    assert np.abs(g[:, 0] - M[:, 0] / np.linalg.norm(M[:, 0], axis=1)[:, None]).max() < 1e-15
    coef = np.einsum("nj,nj->n", g[:, 1].conj(), M[:, 1])
    assert np.abs(coef.imag).max() < 1e-14 and coef.real.min() > 0
    # matches numpy QR of M^T up to the standard phase convention: rows of g = Gram-Schmidt of rows of M
    q, r = np.linalg.qr(M.transpose(0, 2, 1))
    ph = np.einsum("nii->ni", r)
    q = q * (ph / np.abs(ph))[:, None, :]
    assert np.abs(g[:, :2] - q.transpose(0, 2, 1)[:, :2]).max() < 1e-13
    # X = 0 -> g = 1
    assert np.abs(oracle.project(np.zeros((1, 3, 3)), ALPHA)[0] - np.eye(3)).max() == 0


@pytest.mark.parametrize("storage", [18, 12])
def test_P10_P11_P16_unitarity_plaquette_monotone_F(storage):
    dims = (8, 8, 8, 8)
    U = E.noisy(dims, 21, 0.35)
    o = oracle.Oracle(dims, storage)
    o.load(U)
    p0 = o.plaquette()
    r = o.fix(ALPHA, 1e-15, 200, history=True)
    assert r["status"] == 0
    hist = r["history"]
    F, th = hist[:, 0], hist[:, 1]
    ok = th[:-1] > 1e-25
    assert np.all((F[1:] - F[:-1])[ok] >= -1e-14)      # P16 (reading A17)
    assert abs(o.plaquette() - p0) < 1e-12             # P11 gauge invariance
    uu, dd = o.unitarity()
    assert uu < 1e-13 and dd < 1e-13                    # P10
    assert th[-1] < 1e-15 and th[-2] >= 1e-15           # strict stop (A6), count = updates applied (A5)
    assert 25 <= r["n_iter"] <= 60                      # P17 ballpark


def test_P15_F_after_update_equals_paper_formula():
    dims = (4, 4, 4, 8)
    U = E.noisy(dims, 22, 0.4)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    g = o.g_field(ALPHA)
    F_paper = o.F_of_g(g)                       # PAPER.md:39 literally, old links + g
    # independent numpy evaluation of the same formula
    V = U.shape[0]
    Fn = sum(np.trace(g @ U[:, mu] @ dag(shift(g, dims, mu)), axis1=1, axis2=2).real.sum() for mu in range(4)) / (12 * V)
    assert abs(F_paper - Fn) < 1e-14
    F1, _ = o.iterate(1, ALPHA)
    assert abs(F1 - F_paper) < 1e-14
    Unew = o.get()
    for mu in range(4):
        assert np.abs(Unew[:, mu] - g @ U[:, mu] @ dag(shift(g, dims, mu))).max() < 1e-14


# ------------------------------------------------------------------ covariance (P12)
def test_P12_translation_and_axis_permutation_covariance():
    dims = (4, 8, 4, 16)
    U = E.noisy(dims, 23, 0.3)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    F, th = o.iterate(3, ALPHA)
    Uout = o.get()
    # translation by (1, 3, 2, 5)
    def roll_all(A, off):
        L0, L1, L2, L3 = dims
        B = A.reshape((L3, L2, L1, L0) + A.shape[1:])
        for mu in range(4):
            B = np.roll(B, off[mu], axis=3 - mu)
        return B.reshape(A.shape)
    off = (1, 3, 2, 5)
    o2 = oracle.Oracle(dims, 18)
    o2.load(roll_all(U, off))
    F2, th2 = o2.iterate(3, ALPHA)
    assert abs(F2 - F) < 1e-14 and abs(th2 - th) < 1e-12 * th
    assert np.abs(o2.get() - roll_all(Uout, off)).max() < 1e-13
    # axis permutation: new axis k = old axis perm[k]; link labels permute with the axes
    perm = (2, 0, 3, 1)
    pdims = tuple(dims[p] for p in perm)
    L0, L1, L2, L3 = dims
    A = U.reshape(L3, L2, L1, L0, 4, 3, 3)
    # numpy axis of old lattice axis m is 3-m; new numpy axis order (slowest..fastest) = new axes 3,2,1,0
    A = A.transpose([3 - perm[3], 3 - perm[2], 3 - perm[1], 3 - perm[0], 4, 5, 6])
    Up = np.ascontiguousarray(A[:, :, :, :, list(perm)]).reshape(-1, 4, 3, 3)
    o3 = oracle.Oracle(pdims, 18)
    o3.load(Up)
    F3, th3 = o3.iterate(3, ALPHA)
    assert abs(F3 - F) < 1e-14 and abs(th3 - th) < 1e-12 * th
    B = Uout.reshape(L3, L2, L1, L0, 4, 3, 3).transpose([3 - perm[3], 3 - perm[2], 3 - perm[1], 3 - perm[0], 4, 5, 6])
    Bp = np.ascontiguousarray(B[:, :, :, :, list(perm)]).reshape(-1, 4, 3, 3)
    assert np.abs(o3.get() - Bp).max() < 1e-13


# ------------------------------------------------------------------ Abelian special case (P13)
def test_P13_abelian_special_case_vs_independent_scalar_code():
    """Diagonal links stay diagonal; each diagonal entry evolves by a scalar recursion that is
    written here independently with numpy.fft (30 lines, no oracle code)."""
    dims = (4, 8, 4, 8)
    V = int(np.prod(dims))
    U = E.abelian(dims, 31, 0.7)
    o = oracle.Oracle(dims, 18)
    o.load(U)
    n_it = 4
    F_o, th_o = o.iterate(n_it, ALPHA)
    Uo = o.get()

    u = np.stack([U[:, :, j, j] for j in range(3)], axis=-1)  # [V,4,3]
    shape = dims[::-1]
    n = np.meshgrid(*[np.arange(L) for L in shape], indexing="ij")
    p2 = sum(4 * np.sin(np.pi * n[k] / shape[k]) ** 2 for k in range(4))
    with np.errstate(divide="ignore"):
        w = np.where(p2 > 0, 16.0 / p2, 0.0)
    for _ in range(n_it):
        a = sum(shift(u[:, mu], dims, mu, +1) - u[:, mu] for mu in range(4))  # [V,3]
        d = 2j * a.imag
        d = d - d.mean(axis=1, keepdims=True)
        x = np.stack([np.fft.ifftn(w * np.fft.fftn(d[:, j].reshape(shape))).reshape(-1) for j in range(3)], axis=1)
        m = 1 + 0.5 * ALPHA * x
        g0 = m[:, 0] / np.abs(m[:, 0])
        g1 = m[:, 1] / np.abs(m[:, 1])
        g = np.stack([g0, g1, (g0 * g1).conj()], axis=1)
        u = np.stack([g * u[:, mu] * shift(g, dims, mu).conj() for mu in range(4)], axis=1)
    for j in range(3):
        assert np.abs(Uo[:, :, j, j] - u[:, :, j]).max() < 1e-13
    off = Uo.copy()
    for j in range(3):
        off[:, :, j, j] = 0
    assert np.abs(off).max() == 0
    assert abs(F_o - u.real.sum() / (12 * V)) < 1e-14


# ------------------------------------------------------------------ fixed point (P14) = config C0
def test_P14_pure_gauge_fixed_point_C0():
    U, cfg = E.make_config("C0")
    o = oracle.Oracle(cfg["dims"], cfg["storage"])
    o.load(U)
    assert abs(o.plaquette() - 1.0) < 1e-13
    r = o.fix(ALPHA, 1e-15, 500)
    assert r["status"] == 0
    assert abs(r["F"] - 1.0) < 1e-13
    assert r["theta"] < 1e-15
    # F = 1 forces every link to the identity
    Ufix = o.get()
    assert np.abs(Ufix - np.eye(3)).max() < 1e-6


# ------------------------------------------------------------------ oracle modes agree
def test_fft_mode_matches_naive_dft_trajectory():
    dims = (8, 8, 8, 8)
    U = E.noisy(dims, 24, 0.35)
    a = oracle.Oracle(dims, 12, fft_mode=0)
    b = oracle.Oracle(dims, 12, fft_mode=1)
    a.load(U)
    b.load(U)
    Fa, ta = a.iterate(10, ALPHA)
    Fb, tb = b.iterate(10, ALPHA)
    assert abs(Fa - Fb) < 1e-14 and abs(ta - tb) < 1e-11 * ta
    assert np.abs(a.get() - b.get()).max() < 1e-13


def test_storage12_drops_third_row_on_load():
    dims = (4, 4, 4, 4)
    U = E.noisy(dims, 25, 0.3)
    bad = U.copy()
    bad[:, :, 2, :] = 0.0       # garbage third row must be ignored in 12-real mode (reading A9)
    o = oracle.Oracle(dims, 12)
    o.load(bad)
    assert np.abs(o.get() - U).max() < 1e-14
    o18 = oracle.Oracle(dims, 18)
    o18.load(bad)
    assert np.abs(o18.get() - bad).max() == 0


def test_thread_count_independence():
    import os, subprocess, sys
    code = ("import ensembles as E, oracle; U=E.noisy((4,4,4,8),26,0.3); o=oracle.Oracle((4,4,4,8),12); o.load(U);"
            "F,t=o.iterate(5,0.08); print(repr(F), repr(t))")
    outs = []
    for nt in ("1", "4"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        outs.append(subprocess.check_output([sys.executable, "-c", code], env=env, cwd=os.path.dirname(os.path.dirname(__file__))))
    assert outs[0] == outs[1]


@pytest.mark.parametrize("name,fft_mode", [("C0", 0), ("C1", 1)])
def test_golden_trajectories_are_what_the_oracle_computes(name, fft_mode):
    """tests/golden/oracle_*_trajectory.txt (written by tests/golden/make_golden.py from the oracle alone) against the
    oracle as it stands: a change of the oracle's arithmetic must show up here.  Rounding-level slack only."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"oracle_{name}_trajectory.txt")
    rows = np.array([[float(v) for v in ln.split()] for ln in open(path) if not ln.startswith("#")])
    U, cfg = E.make_config(name)
    o = oracle.Oracle(cfg["dims"], cfg["storage"], fft_mode=fft_mode)
    o.load(U)
    r = o.fix(0.08, 1e-15, 1000, history=True)
    h = np.array(r["history"])
    assert len(h) == len(rows) and r["n_iter"] == len(rows) - 1
    assert np.abs(h[:, 0] - rows[:, 1]).max() <= 1e-13
    assert np.all(np.abs(h[:, 1] - rows[:, 2]) <= 1e-9 * np.maximum(rows[:, 2], 1e-15))


# ------------------------------------------------------------------ Coulomb-gauge variant of the oracle (nd = 3)
def _coulomb(dims, storage=18, fft_mode=0):
    o = oracle.Oracle(dims, storage, fft_mode=fft_mode)
    o.set_gauge(3)
    return o


@pytest.mark.parametrize("dims,alpha", [((8, 8, 8, 4), 0.08), ((4, 8, 4, 8), 0.05)])
def test_coulomb_linearised_rate(dims, alpha):
    """Coulomb gauge (gauge condition over mu = 0..2): with p2max = 4*3 every mode of non-zero
    spatial momentum contracts by (1 - 12 alpha) per iteration, so theta_{k+1}/theta_k = (1 - 12 alpha)^2; pins
    p2max = 12, the restriction of p^2 to three axes, alpha/2, 1/V and the sign, as P9 does for Landau."""
    V = int(np.prod(dims))
    rng = np.random.Generator(np.random.Philox(key=[6, 1]))
    h = E.expi_hermitian(E.gaussian_su3_algebra(rng, V), 1e-5)
    U = np.stack([h @ dag(shift(h, dims, mu)) for mu in range(4)], axis=1)
    o = _coulomb(dims)
    o.load(U)
    _, th0 = o.measure()
    _, th1 = o.iterate(1, alpha)
    _, th2 = o.iterate(1, alpha)
    r = (1 - 12 * alpha) ** 2
    assert abs(th1 / th0 - r) < 2e-3 * r
    assert abs(th2 / th1 - r) < 2e-3 * r


def test_coulomb_field_is_spatial_and_inverts_the_3d_laplacian():
    """Delta and X of time slice t depend only on the spatial links of that slice; X obeys the 3-D version of P18,
    sum_{mu<3} [2 X(x) - X(x+mu) - X(x-mu)] = 12 Delta(x); F counts three directions (identity links: F = 1)."""
    dims = (4, 6, 4, 4)
    U = E.noisy(dims, 31, 0.4)
    o = _coulomb(dims)
    o.load(U)
    D = o.delta().reshape(dims[::-1] + (3, 3))
    X = o.fa_field().reshape(dims[::-1] + (3, 3))
    lap = sum(2.0 * X - np.roll(X, 1, axis=ax) - np.roll(X, -1, axis=ax) for ax in (1, 2, 3))     # axes x2, x1, x0
    assert np.abs(lap - 12.0 * D).max() <= 1e-12 * np.abs(X).max()
    assert np.abs(D.sum(axis=(1, 2, 3))).max() <= 1e-12                                            # per time slice
    U2 = U.copy().reshape(dims[::-1] + (4, 3, 3))
    U2[1] = E.noisy(dims, 32, 0.4).reshape(dims[::-1] + (4, 3, 3))[1]                              # another slice t = 1
    U2[:, :, :, :, 3] = E.noisy(dims, 33, 0.4).reshape(dims[::-1] + (4, 3, 3))[:, :, :, :, 3]      # all temporal links
    o.load(U2.reshape(-1, 4, 3, 3))
    X2 = o.fa_field().reshape(dims[::-1] + (3, 3))
    assert np.abs(X2[[0, 2, 3]] - X[[0, 2, 3]]).max() <= 1e-13 * np.abs(X).max()
    ident = np.broadcast_to(np.eye(3, dtype=np.complex128), (int(np.prod(dims)), 4, 3, 3)).copy()
    o.load(ident)
    F, th = o.measure()
    assert abs(F - 1.0) < 1e-15 and th == 0.0


def test_coulomb_trajectory_invariants():
    """F_C rises monotonically, the plaquette is invariant, links stay special unitary, theta falls below 1e-15."""
    dims = (8, 8, 8, 4)
    U = E.noisy(dims, 34, 0.3)
    o = _coulomb(dims, storage=12, fft_mode=1)
    o.load(U)
    p0 = o.plaquette()
    r = o.fix(0.08, 1e-15, 500, history=True)
    h = np.array(r["history"])
    assert r["status"] == 0 and h[-1, 1] < 1e-15
    assert np.all(np.diff(h[:, 0]) >= -1e-14)
    assert abs(o.plaquette() - p0) <= 1e-12
    assert max(o.unitarity()) <= 1e-13


# ------------------------------------------------------------------ utility read-outs (plaquette, unitarity)
def test_plaquette_equals_an_independent_numpy_evaluation_and_the_heatbath_measurement():
    """orc_plaquette (the invariant of pin P11 and the number DESIGN.md section 4 reports per ensemble) on non-trivial
    links: (1/18V) sum_x sum_{mu<nu} Re Tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag] written out with explicit
    np.roll shifts on a 4-D array, and the same number from ensembles.heatbath.average_plaquette (torch, written for the
    Wilson action, shares no code with the oracle).  An anisotropic lattice catches swapped directions or shifts."""
    import torch
    from ensembles import heatbath as H
    for dims, eps in [((4, 4, 4, 4), 0.35), ((4, 6, 2, 8), 0.6)]:
        U = E.noisy(dims, 71, eps)
        L0, L1, L2, L3 = dims
        U4 = U.reshape(L3, L2, L1, L0, 4, 3, 3)
        s = 0.0
        for mu in range(4):
            for nu in range(mu + 1, 4):
                Um, Un = U4[..., mu, :, :], U4[..., nu, :, :]
                Un_xmu = np.roll(Un, -1, axis=3 - mu)         # U_nu(x + mu)
                Um_xnu = np.roll(Um, -1, axis=3 - nu)         # U_mu(x + nu)
                P = Um @ Un_xmu @ dag(Um_xnu) @ dag(Un)
                s += np.trace(P, axis1=-2, axis2=-1).real.sum()
        want = s / (18.0 * U.shape[0])
        o = oracle.Oracle(dims, 18)
        o.load(U)
        got = o.plaquette()
        assert abs(got - want) < 1e-14, (dims, got, want)
        assert 0.1 < got < 0.95                                # non-trivial links: neither 1 nor 0
        assert abs(H.average_plaquette(torch.from_numpy(U), dims) - got) < 1e-13
        # a single perturbed link changes exactly the 6 plaquettes through it
        U2 = U.copy()
        U2[5, 2] = U2[5, 2] @ E.expi_hermitian(E.gaussian_su3_algebra(np.random.default_rng(3), 1), 0.4)[0]
        o.load(U2)
        assert abs(o.plaquette() - got) > 1e-6


def test_unitarity_readout_equals_numpy():
    """orc_unitarity = (max |U U^dag - 1|, max |det U - 1|) over all links, against numpy on links that are off the
    group by a known amount."""
    dims = (4, 4, 4, 4)
    U = E.noisy(dims, 72, 0.3)
    rng = np.random.default_rng(5)
    U = U + 1e-3 * (rng.standard_normal(U.shape) + 1j * rng.standard_normal(U.shape))
    o = oracle.Oracle(dims, 18)
    o.load(U)
    uu, dd = o.unitarity()
    want_uu = np.abs(U @ dag(U) - np.eye(3)).max()
    want_dd = np.abs(np.linalg.det(U) - 1.0).max()
    assert abs(uu - want_uu) < 1e-15 and abs(dd - want_dd) < 1e-14
    assert 1e-4 < uu < 1e-1 and 1e-4 < dd < 1e-1
