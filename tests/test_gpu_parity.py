"""GPU parity: the CUDA path (through the C ABI of include/lgf.h) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are the north star's (BASELINE.json) with reading A14 for theta
(DESIGN.md "Readings"): |dF| <= 1e-12, |dtheta| <= 1e-9 * max(theta_ref, 1e-15), links <= 1e-11, iteration
count exact (A19).  Kernel-level stages use the tighter bounds of SURVEY.md section 7 step 4/5.
"""
import numpy as np
import pytest

import ensembles as E
import oracle
import paper_1301_3460_b200 as lgf

pytestmark = pytest.mark.gpu

ALPHA = 0.08
TOL = 1e-15

F_TOL = 1e-12
LINK_TOL = 1e-11


def theta_close(t_gpu, t_ref):
    return abs(t_gpu - t_ref) <= 1e-9 * max(t_ref, TOL)


def all_variants(gf):
    """Every kernel selection the library offers, as (store g, CUDA graph, compile-time-sized FFT passes, PDL)."""
    if gf.V > (1 << 18):
        return [(0, 1, 1, 1), (1, 1, 1, 1), (0, 0, 0, 1), (1, 0, 0, 0), (0, 1, 1, 1, 0)]
    out = [(sg, graph, fast, 1) for fast in (1, 0) for sg in (0, 1) for graph in (1, 0)]
    out += [(0, 1, 1, 0), (1, 0, 0, 0), (0, 1, 1, 1, 0), (0, 0, 1, 0, 0)]      # the last two: pass B with plain loads instead of TMA
    return out


def set_variant(gf, v):
    gf.set_option(lgf.LGF_OPT_STORE_G, v[0])
    gf.set_option(lgf.LGF_OPT_GRAPH, v[1])
    gf.set_option(lgf.LGF_OPT_FAST_FFT, v[2])
    gf.set_option(lgf.LGF_OPT_PDL, v[3] if len(v) > 3 else 1)
    gf.set_option(lgf.LGF_OPT_TMA, v[4] if len(v) > 4 else 1)


# ------------------------------------------------------------------ boundary: load -> get
@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (4, 8, 16, 4)])
def test_load_get_roundtrip(dims):
    U = E.noisy(dims, 41, 0.3)
    g18 = lgf.GaugeFixer(dims, 18)
    g18.load_links(U)
    assert np.array_equal(g18.get_links(), U)                      # 18-real: bit exact
    g12 = lgf.GaugeFixer(dims, 12)
    bad = U.copy()
    bad[:, :, 2, :] = 7.0                                           # row 2 must be ignored on load (A9)
    g12.load_links(bad)
    out = g12.get_links()
    assert np.array_equal(out[:, :, :2], U[:, :, :2])               # rows 0,1 bit exact
    # row 2 rebuilt as conj(row0 x row1): equal to the oracle's rebuild up to FMA contraction (|entries| <= 1,
    # two products per entry -> a few ulp), and to the generator's own row 2 within its unitarity error
    o12 = oracle.Oracle(dims, 12)
    o12.load(bad)
    assert np.abs(out[:, :, 2] - o12.get()[:, :, 2]).max() < 5e-16
    assert np.abs(out[:, :, 2] - U[:, :, 2]).max() < 1e-14
    # two-row host format: rows 0,1 in, rows 0,1 out, bit exact; the same state as the canonical load
    rows = np.ascontiguousarray(U[:, :, :2])
    g12.load_links_12(rows)
    assert np.array_equal(g12.get_links_12(), rows)
    assert np.array_equal(g12.get_links(), out)
    with pytest.raises(lgf.LgfError):
        g18.load_links_12(rows)                                     # LGF_ERR_UNSUPPORTED with full storage
    # float64 [V,4,3,3,2] view is accepted as well
    g18.load_links(E.as_real(U))
    assert np.array_equal(g18.get_links(), U)
    # the library-owned workspace/stream flavour (lgf_create) gives the same bytes
    g3 = lgf.GaugeFixer(dims, 18, use_torch_workspace=False)
    g3.load_links(U)
    assert np.array_equal(g3.get_links(), U)


def test_device_pointer_load_and_get():
    import torch
    dims = (8, 4, 8, 4)
    U = E.noisy(dims, 42, 0.3)
    d_in = torch.from_numpy(E.as_real(U).copy()).cuda()
    d_out = torch.zeros_like(d_in)
    gf = lgf.GaugeFixer(dims, 12)
    gf.load_links_device(d_in.data_ptr())
    gf.get_links_device(d_out.data_ptr())
    torch.cuda.synchronize()
    got = E.as_complex(d_out.cpu().numpy())
    assert np.array_equal(got[:, :, :2], U[:, :, :2])
    assert np.abs(got - U).max() < 1e-14


# ------------------------------------------------------------------ kernel-level stages (S1, S2, S3, S4)
STAGE_CASES = [
    ((8, 8, 8, 8), 18), ((8, 8, 8, 8), 12), ((16, 16, 16, 16), 12),
    # 64 extents (the shapes of C3, C4 on small companions): one-component plane passes, short-chunk pass B
    ((64, 64, 4, 4), 12), ((4, 4, 64, 64), 18), ((32, 64, 4, 8), 12), ((64, 32, 8, 4), 18), ((8, 4, 32, 64), 12), ((4, 8, 64, 32), 12),
    ((8, 8, 16, 32), 12), ((4, 8, 16, 32), 18), ((32, 4, 8, 4), 12), ((4, 4, 4, 4), 12), ((16, 32, 4, 8), 18),
    ((32, 16, 16, 32), 12), ((16, 32, 32, 16), 18), ((32, 32, 16, 16), 12), ((16, 16, 32, 32), 18), ((32, 32, 32, 32), 12),
    # two-row storage with at least two (x2,x3) planes per SM: the TMA-staged pass A on 16 x 32 and 16 x 16 planes
    ((16, 32, 32, 16), 12), ((16, 16, 32, 16), 12),
]


@pytest.mark.parametrize("dims,storage", STAGE_CASES)
def test_stage_parity_delta_X_g_update(dims, storage):
    U = E.noisy(dims, 43, 0.35)
    o = oracle.Oracle(dims, storage)
    o.load(U)
    D_ref, X_ref, g_ref = o.delta(), o.fa_field(), o.g_field(ALPHA)
    F_ref, th_ref = o.measure()
    o.iterate(1, ALPHA)
    U1_ref = o.get()
    F1_ref, th1_ref = o.measure()
    xs = np.abs(X_ref).max()

    gf = lgf.GaugeFixer(dims, storage)
    for v in all_variants(gf):
        gf.load_links(U)
        set_variant(gf, v)
        F, th, _ = gf.measure()
        assert abs(F - F_ref) <= 1e-14, v
        assert abs(th - th_ref) <= 1e-12 * th_ref, v
        D = gf.get_field(lgf.LGF_FIELD_DELTA)
        assert np.abs(D - D_ref).max() <= 1e-14 * max(1.0, np.abs(D_ref).max()), v
        X = gf.get_field(lgf.LGF_FIELD_X)
        assert np.abs(X - X_ref).max() <= 1e-13 * xs, v
        g = gf.get_field(lgf.LGF_FIELD_G, ALPHA)
        assert np.abs(g - g_ref).max() <= 1e-13, v
        assert np.array_equal(gf.get_links()[:, :, :2], U[:, :, :2]), v     # read-outs do not change the links
        F1, th1 = gf.iterate(1, ALPHA)
        assert abs(F1 - F1_ref) <= 1e-13, v
        assert abs(th1 - th1_ref) <= 1e-11 * th1_ref, v
        assert np.abs(gf.get_links() - U1_ref).max() <= 1e-13, v


# ------------------------------------------------------------------ trajectories (configs C0, C1 of BASELINE.json)
def oracle_trajectory(U, dims, storage, checkpoints, fft_mode):
    """F_k, theta_k for k = 0..max(checkpoints) and the links at each checkpoint."""
    o = oracle.Oracle(dims, storage, fft_mode=fft_mode)
    o.load(U)
    hist, links, done = [], {}, 0
    for cp in checkpoints:
        r = o.fix(ALPHA, 0.0, cp - done, history=True)      # theta < 0 never holds: exactly cp-done updates
        assert r["status"] == 100
        h = r["history"]
        hist.extend(h[:-1] if cp != checkpoints[-1] else h)
        links[cp] = o.get()
        done = cp
    return np.array(hist), links


def check_trajectory(name, fft_mode, checkpoints=(10, 100), variants=((0, 1, 1, 1), (1, 1, 1, 1), (0, 0, 0, 1), (1, 0, 0, 0), (0, 1, 1, 1, 0))):
    U, cfg = E.make_config(name)
    dims, storage = cfg["dims"], cfg["storage"]
    hist_ref, links_ref = oracle_trajectory(U, dims, storage, checkpoints, fft_mode)
    n_ref = int(np.argmax(hist_ref[:, 1] < TOL))
    assert hist_ref[n_ref, 1] < TOL, "oracle did not converge inside the trajectory"

    gf = lgf.GaugeFixer(dims, storage)
    _, _, plaq = gf_plaquette(gf, U)
    print(f"{name}: average plaquette {plaq:.6f}, oracle stop iteration {n_ref}, F = {hist_ref[n_ref, 0]:.12f}")
    for v in variants:
        set_variant(gf, v)
        gf.load_links(U)
        done = 0
        hist = []
        for cp in checkpoints:
            F, th = gf.iterate(cp - done, ALPHA)
            h = gf.get_history()
            assert len(h) == cp - done + 1
            assert h[-1, 0] == F and h[-1, 1] == th
            hist.extend(h[:-1] if cp != checkpoints[-1] else h)
            done = cp
            # north star: |dF| <= 1e-12, theta (A14), links <= 1e-11 after 10 and 100 iterations
            assert abs(F - hist_ref[cp, 0]) <= F_TOL, (name, v, cp)
            assert theta_close(th, hist_ref[cp, 1]), (name, v, cp, th, hist_ref[cp, 1])
            assert np.abs(gf.get_links() - links_ref[cp]).max() <= LINK_TOL, (name, v, cp)
        hist = np.array(hist)
        assert np.abs(hist[:, 0] - hist_ref[:, 0]).max() <= F_TOL
        for k in range(len(hist)):
            assert theta_close(hist[k, 1], hist_ref[k, 1]), (name, v, k, hist[k, 1], hist_ref[k, 1])
        # the stop iteration: lgf_fix from the same start
        gf.load_links(U)
        r = gf.fix(ALPHA, TOL, 1000)
        assert r["status"] == lgf.LGF_OK
        assert r["n_iter"] == n_ref, (name, v, r, n_ref)                     # A19: exact
        assert abs(r["F"] - hist_ref[n_ref, 0]) <= F_TOL
        assert theta_close(r["theta"], hist_ref[n_ref, 1])
        assert r["theta"] < TOL
        assert np.abs(gf.get_links() - oracle_links_at(U, dims, storage, n_ref, fft_mode)).max() <= LINK_TOL
    return hist_ref, n_ref


def gf_plaquette(gf, U):
    gf.load_links(U)
    return gf.measure()


_cache = {}


def oracle_links_at(U, dims, storage, n, fft_mode):
    key = (id(U), tuple(dims), storage, n, fft_mode)
    if key not in _cache or _cache[key][0] is not U:          # the array itself is kept: an id can be reused after garbage collection
        o = oracle.Oracle(dims, storage, fft_mode=fft_mode)
        o.load(U)
        o.iterate(n, ALPHA)
        _cache.clear()
        _cache[key] = (U, o.get())
    return _cache[key][1]


def test_trajectory_C0_pure_gauge_fixed_point():
    hist_ref, n_ref = check_trajectory("C0", fft_mode=0)
    assert abs(hist_ref[n_ref, 0] - 1.0) < 1e-13          # closed-form fixed point F = 1 (P14)


def test_trajectory_C1():
    hist_ref, n_ref = check_trajectory("C1", fft_mode=1)
    # the same trajectory as the stored oracle output (tests/golden, written by the oracle alone)
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_C1_trajectory.txt")
    rows = np.array([[float(v) for v in ln.split()] for ln in open(path) if not ln.startswith("#")])
    assert n_ref == len(rows) - 1
    assert np.abs(hist_ref[: len(rows), 0] - rows[:, 1]).max() <= 1e-13


def test_trajectory_C2b_headline_config():
    """BASELINE.json configs[2], eps = 0.35 (the workload bench.py times): F, theta, links after 10 and 100 iterations
    and the stop iteration, against the oracle (radix-2 FFT mode, itself pinned to the naive DFT on CPU)."""
    check_trajectory("C2b", fft_mode=1)


@pytest.mark.parametrize("name", ["C2a", "C2c"])
def test_trajectory_C2a_C2c(name):
    """BASELINE.json configs[2], eps = 0.25 and 0.45: the other two of the three seeded 32^4 ensembles that stand in
    for the paper's three beta values; default path and the store-g path."""
    check_trajectory(name, fft_mode=1, checkpoints=(10, 60), variants=((0, 1, 1, 1), (1, 0, 0, 0)))


def test_trajectory_C3_anisotropic():
    """BASELINE.json configs[3], 32^3 x 64: uneven FFT axes, non-cubic p^2 filter, 64-extent pass B."""
    check_trajectory("C3", fft_mode=1, checkpoints=(10, 100))


# ------------------------------------------------------------------ step-size scan (NEXT-3)
def test_alpha_scan_counts_equal_the_oracle():
    """lgf_scan_alpha on C1: one lgf_fix per alpha from the same start; every count equals the oracle's for that alpha
    (A19: exact), the best alpha is the oracle's best, a diverging alpha is reported as such, and the links in the
    context are the same before and after."""
    U, cfg = E.make_config("C1")
    dims, storage = cfg["dims"], cfg["storage"]
    alphas = [0.05, 0.0625, 0.08, 0.10, 0.2]                   # 0.2 > 1/8: beyond the stability bound of the linearised map
    gf = lgf.GaugeFixer(dims, storage)
    gf.load_links(U)
    before = gf.get_links()
    r = gf.scan_alpha(alphas, TOL, 400)
    assert np.array_equal(gf.get_links(), before)
    ref = []
    for a in alphas[:-1]:
        o = oracle.Oracle(dims, storage, fft_mode=1)
        o.load(U)
        rr = o.fix(a, TOL, 400)
        assert rr["status"] == 0
        ref.append((rr["n_iter"], rr["F"]))
    assert r["counts"][:-1] == [n for n, _ in ref], (r, ref)
    assert max(abs(f - fr) for f, (_, fr) in zip(r["F"][:-1], ref)) <= F_TOL
    assert r["counts"][-1] < 0                                  # alpha = 0.2 does not converge
    assert r["best"] == int(np.argmin([n for n, _ in ref]))
    print("alpha scan C1:", dict(zip(alphas, r["counts"])))
    gf.destroy()


# ------------------------------------------------------------------ C4 as BASELINE.json states it (64^4, eps 0.35, seed 5)
def _c4_inputs():
    """configs[4] on its own ensemble: the configs[1] recipe generated on the device (ensembles.noisy_device, reading
    A12b: the numpy recipe takes minutes at 64^4), copied to the host ONCE; the same array goes to the oracle and to
    lgf_load_links."""
    import torch
    cfg = E.CONFIGS["C4"]
    Ud = E.noisy_device(cfg["dims"], cfg["seed"], cfg["eps"], cfg.get("stream", 0))
    U = Ud.cpu().numpy()
    del Ud
    torch.cuda.empty_cache()
    return U, cfg["dims"], cfg["storage"]


def test_C4_full_lattice_first_iterations_and_full_run():
    """64^4 at full size against the radix-2-FFT-mode oracle (itself pinned to the naive DFT on the CPU): Delta and X of
    the first iteration element by element on all 16.8 M sites, then F, theta and every link after 1, 3 and 10
    iterations, then the whole run to theta < 1e-15 with the stop iteration.  One set of inputs and ONE oracle
    trajectory for all of it (about 7 s of host time per oracle iteration)."""
    U, dims, storage = _c4_inputs()
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    gf = lgf.GaugeFixer(dims, storage)
    gf.load_links(U)
    F0, th0, plaq = gf.measure()
    F0_ref, th0_ref = o.measure()
    print(f"C4: average plaquette {plaq:.6f}, F0 = {F0:.12f}, theta0 = {th0:.6e}")
    assert abs(F0 - F0_ref) <= F_TOL and abs(th0 - th0_ref) <= 1e-12 * th0_ref
    D_ref = o.delta()
    D = gf.get_field(lgf.LGF_FIELD_DELTA)
    assert np.abs(D - D_ref).max() <= 1e-14 * np.abs(D_ref).max()
    del D, D_ref
    X_ref = o.fa_field()
    X = gf.get_field(lgf.LGF_FIELD_X)
    assert np.abs(X - X_ref).max() <= 1e-13 * np.abs(X_ref).max()
    del X, X_ref
    done = 0
    for k in (1, 3):
        F_ref, th_ref = o.iterate(k - done, ALPHA)
        F, th = gf.iterate(k - done, ALPHA)
        done = k
        assert abs(F - F_ref) <= F_TOL, (k, F, F_ref)
        assert theta_close(th, th_ref), (k, th, th_ref)
        assert np.abs(gf.get_links() - o.get()).max() <= 1e-13 * k, k
    # the north star's checkpoint after 10 iterations: F, theta, every link
    F_ref, th_ref = o.iterate(10 - done, ALPHA)
    F, th = gf.iterate(10 - done, ALPHA)
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref), (10, F, F_ref, th, th_ref)
    assert np.abs(gf.get_links() - o.get()).max() <= LINK_TOL
    # the full run to theta < 1e-15 (configs[4]): the oracle goes on from its iteration 10 to its stop, the
    # library runs lgf_fix from the start -- stop iteration exact (A19), F and theta of every iteration from 10 on, every
    # link at the stop.  (C4 stops before 100 iterations, so the stop takes the place of the second checkpoint.)
    r_ref = o.fix(ALPHA, TOL, 1000, history=True)
    assert r_ref["status"] == 0
    n_ref = 10 + r_ref["n_iter"]
    h_ref = np.array(r_ref["history"])                     # h_ref[i] = (F, theta) after 10 + i iterations
    gf.load_links(U)
    r = gf.fix(ALPHA, TOL, 1000)
    h = gf.get_history()
    print(f"C4 full run: n_iter {r['n_iter']} (oracle {n_ref}), F {r['F']:.15f} (oracle {r_ref['F']:.15f}), "
          f"theta {r['theta']:.3e} (oracle {r_ref['theta']:.3e})")
    assert r["status"] == lgf.LGF_OK and r["n_iter"] == n_ref
    assert abs(r["F"] - r_ref["F"]) <= F_TOL and theta_close(r["theta"], r_ref["theta"]) and r["theta"] < TOL
    assert len(h) == n_ref + 1 and len(h_ref) == n_ref - 10 + 1
    assert abs(h[0, 0] - F0_ref) <= F_TOL and theta_close(h[0, 1], th0_ref)
    assert np.abs(h[10:, 0] - h_ref[:, 0]).max() <= F_TOL
    for i in range(len(h_ref)):
        assert theta_close(h[10 + i, 1], h_ref[i, 1]), (10 + i, h[10 + i, 1], h_ref[i, 1])
    dmax = np.abs(gf.get_links() - o.get()).max()
    print(f"C4 full run: max link difference at the stop {dmax:.3e}")
    assert dmax <= LINK_TOL
    gf.destroy()


# ------------------------------------------------------------------ full-size lattices on sampled sites
def _site_coords(x, dims):
    c = []
    for L in dims:
        c.append(x % L)
        x //= L
    return c


def _site_index(c, dims):
    x, m = 0, 1
    for k, L in zip(c, dims):
        x += (k % L) * m
        m *= L
    return x


@pytest.mark.parametrize("dims", [(64, 64, 64, 64), (32, 32, 32, 64)])
def test_full_size_sampled_sites_and_invariants(dims):
    """C4 / C3 shapes at full size, where the oracle cannot run the whole lattice in test time: every stage is checked
    on sampled sites against what the oracle computes site by site, plus properties that hold at any size.
      S1: Delta(x) from the oracle on a 4^4 carrier lattice holding the 8 links of x (the stencil is local);
      S2: -Laplacian X = p2max * Delta, since p2max/p^2 inverts the eigenvalues 4 sin^2(pi n/L) of the lattice Laplacian;
      S3+S4: U' = g(x) U g(x+mu)^dagger with g = oracle.project(X) on the sampled sites;
      theta from the full Delta field; plaquette invariance; F monotone."""
    import torch
    V = int(np.prod(dims))
    Ud = E.device_su3(dims, seed=5, spread=0.15)
    gf = lgf.GaugeFixer(dims, 12)
    gf.load_links_device(Ud.data_ptr())
    F0, th0, plaq0 = gf.measure()
    D = gf.get_field(lgf.LGF_FIELD_DELTA)
    X = gf.get_field(lgf.LGF_FIELD_X)
    assert abs(np.einsum("xij,xij->", D.conj(), D).real / (3.0 * V) - th0) <= 1e-12 * th0      # theta = (1/3V) sum Tr D D^dag
    rng = np.random.default_rng(11)
    sites = [int(v) for v in rng.integers(0, V, 48)] + [0, V - 1, dims[0] - 1, V - dims[0]]      # corners: every wrap
    ident = np.broadcast_to(np.eye(3, dtype=np.complex128), (256, 4, 3, 3)).copy()
    carrier = (4, 4, 4, 4)
    y = _site_index((1, 1, 1, 1), carrier)
    o4 = oracle.Oracle(carrier, 12)
    xs = np.abs(X).max()
    for x in sites:
        c = _site_coords(x, dims)
        nb_f = [_site_index([c[k] + (1 if k == mu else 0) for k in range(4)], dims) for mu in range(4)]
        nb_b = [_site_index([c[k] - (1 if k == mu else 0) for k in range(4)], dims) for mu in range(4)]
        idx = torch.tensor([x] + nb_b, device="cuda")
        Ul = Ud[idx].cpu().numpy()                                  # links of x and of its 4 backward neighbours
        # S1 on the carrier lattice: A(y) = sum_mu [U_mu(y-mu) - U_mu(y)] touches exactly these 8 links
        W = ident.copy()
        W[y] = Ul[0]
        for mu in range(4):
            yb = _site_index([1 - (1 if k == mu else 0) for k in range(4)], carrier)
            W[yb, mu] = Ul[1 + mu, mu]
        o4.load(W)
        assert np.abs(o4.delta()[y] - D[x]).max() <= 1e-14 * max(1.0, np.abs(D[x]).max()), (dims, x)
        # S2: sum_mu [2 X(x) - X(x+mu) - X(x-mu)] = 16 Delta(x)
        lap = sum(2.0 * X[x] - X[nb_f[mu]] - X[nb_b[mu]] for mu in range(4))
        assert np.abs(lap - 16.0 * D[x]).max() <= 1e-11 * max(xs, 1.0), (dims, x)
    # S3 + S4 on the sampled sites
    F1, th1 = gf.iterate(1, ALPHA)
    U1 = torch.empty_like(Ud)
    gf.get_links_device(U1.data_ptr())
    torch.cuda.synchronize()
    for x in sites[:24] + sites[-4:]:
        c = _site_coords(x, dims)
        nb_f = [_site_index([c[k] + (1 if k == mu else 0) for k in range(4)], dims) for mu in range(4)]
        g = oracle.project(np.ascontiguousarray(X[[x] + nb_f]), ALPHA)
        Ux = Ud[x].cpu().numpy()
        got = U1[x].cpu().numpy()
        for mu in range(4):
            want = g[0] @ Ux[mu] @ g[1 + mu].conj().T
            want[2] = np.conj(np.cross(want[0], want[1]))           # 12-real storage (O6)
            assert np.abs(got[mu] - want).max() <= 1e-13, (dims, x, mu)
    assert F1 >= F0 - 1e-14
    F3, th3 = gf.iterate(2, ALPHA)
    assert F3 >= F1 - 1e-14
    _, _, plaq3 = gf.measure()
    assert abs(plaq3 - plaq0) <= 1e-12                              # gauge invariance of the plaquette
    gf.destroy()


@pytest.mark.parametrize("dims,storage", [((8, 8, 8, 8), 18), ((16, 16, 16, 16), 12), ((4, 8, 16, 4), 12)])
def test_plain_steepest_descent_variant(dims, storage):
    """LGF_OPT_FOURIER_ACCEL = 0 (X = Delta) against the oracle's unaccelerated variant:
    trajectory, links, and the first-order rate dF/dalpha = theta/16 of pin P8."""
    U = E.noisy(dims, 51, 0.3)
    o = oracle.Oracle(dims, storage)
    o.set_variant(accel=0)
    o.load(U)
    X_ref = o.fa_field()
    r_ref = o.fix(ALPHA, 0.0, 20, history=True)
    gf = lgf.GaugeFixer(dims, storage)
    for graph in (1, 0):
        gf.set_option(lgf.LGF_OPT_FOURIER_ACCEL, 0)
        gf.set_option(lgf.LGF_OPT_GRAPH, graph)
        assert gf.get_option(lgf.LGF_OPT_FOURIER_ACCEL) == 0
        gf.load_links(U)
        assert np.abs(gf.get_field(lgf.LGF_FIELD_X) - X_ref).max() <= 1e-13 * np.abs(X_ref).max()
        n0 = gf.launch_count()
        F, th = gf.iterate(20, ALPHA)
        assert gf.launch_count() - n0 == 3 * 21
        h = gf.get_history()
        href = np.array(r_ref["history"])
        assert np.abs(h[:, 0] - href[:, 0]).max() <= F_TOL
        assert all(theta_close(a, b) for a, b in zip(h[:, 1], href[:, 1]))
        assert np.abs(gf.get_links() - o.get()).max() <= LINK_TOL
        assert np.all(np.diff(h[:, 0]) >= -1e-14)                       # F rises monotonically for alpha < 1/8
    # pin P8 on the GPU: dF/dalpha at alpha -> 0 equals theta/16 without the filter
    gf.load_links(U)
    F0, th0, _ = gf.measure()
    a = 1e-4
    F1, _ = gf.iterate(1, a)
    assert abs((F1 - F0) / a - th0 / 16.0) <= 2e-3 * th0 / 16.0
    gf.set_option(lgf.LGF_OPT_FOURIER_ACCEL, 1)
    gf.load_links(U)
    F, th = gf.iterate(20, ALPHA)
    assert th < href[-1, 1]                                              # Fourier acceleration converges faster


# ------------------------------------------------------------------ many short runs across the kernel selections
def test_kernel_selections_agree_over_many_configurations():
    """A few hundred lgf_fix runs on seeded device-generated configurations: every kernel selection (generic or sized passes,
    stored g, PDL, graph batching) must stop at the same iteration with the same F, and the mixed-precision run must reach
    the same F.  The stop flag is raised and observed in a different kernel or CTA in each selection; this is the test
    that goes through that transition many times (a per-thread read of the flag once hung an experimental build)."""
    variants = [{}, {"LGF_OPT_FAST_FFT": 0}, {"LGF_OPT_STORE_G": 1}, {"LGF_OPT_PDL": 0}, {"LGF_OPT_BATCH": 1}, {"LGF_OPT_BATCH": 3},
                {"LGF_OPT_GRAPH": 0}]
    for dims, nseeds in [((16, 16, 16, 16), 24), ((32, 32, 16, 16), 8), ((64, 64, 4, 4), 4)]:
        gfs = []
        for opts in variants:
            g = lgf.GaugeFixer(dims, 12)
            for k, v in opts.items():
                g.set_option(getattr(lgf, k), v)
            gfs.append(g)
        gm = lgf.GaugeFixer(dims, 12, precision=lgf.LGF_MIXED)
        for seed in range(nseeds):
            Ud = E.device_su3(dims, 2000 + seed, 0.1 + 0.01 * (seed % 20))
            ref = None
            for opts, g in zip(variants, gfs):
                g.load_links_device(Ud.data_ptr())
                r = g.fix(ALPHA, TOL, 5000)
                assert r["status"] == lgf.LGF_OK, (dims, seed, opts, r)
                ref = ref or r
                assert r["n_iter"] == ref["n_iter"] and abs(r["F"] - ref["F"]) <= 1e-13, (dims, seed, opts, r, ref)
            gm.load_links_device(Ud.data_ptr())
            rm = gm.fix(ALPHA, TOL, 5000)
            assert rm["status"] == lgf.LGF_OK and abs(rm["F"] - ref["F"]) <= 1e-11, (dims, seed, rm, ref)
        for g in gfs + [gm]:
            g.destroy()


# ------------------------------------------------------------------ thermalised Wilson-action inputs
@pytest.mark.parametrize("dims,beta,sweeps,seed", [((8, 8, 8, 8), 5.8, 20, 7), ((16, 16, 16, 16), 6.0, 20, 7),
                                                  ((8, 8, 8, 8), 5.7, 40, 8), ((16, 16, 16, 16), 5.7, 40, 7)])
def test_trajectory_on_thermalised_wilson_configuration(dims, beta, sweeps, seed):
    """The kind of input the paper fixes (Wilson action): a heat-bath configuration (ensembles.wilson,
    generated on the device, fed to both sides as the same host array).  Whole trajectory against the oracle with the
    north-star tolerances -- here theta is far from its rounding floor for the whole run, so the relative theta bound
    bites at every iteration -- the stop iteration exactly, the links at the end; mixed precision reaches the same F.
    The beta = 5.7 cases are rough configurations that need 221 and 383 iterations: the trajectory stays within the
    tolerances over hundreds of iterations (reading A16: the iteration is a well-conditioned map)."""
    from ensembles import heatbath as H
    Ud = E.wilson(dims, beta, sweeps, seed, device="cuda")
    assert 0.53 < H.average_plaquette(Ud, dims) < 0.62          # thermalised around beta = 5.7 .. 6: 0.55 .. 0.60
    U = Ud.cpu().numpy()
    o = oracle.Oracle(dims, 12, fft_mode=1)
    o.load(U)
    r_ref = o.fix(ALPHA, TOL, 5000, history=True)
    href = np.array(r_ref["history"])
    assert r_ref["status"] == 0 and r_ref["n_iter"] > 30
    gf = lgf.GaugeFixer(dims, 12)
    for v in [(0, 1, 1, 1), (1, 1, 1, 1), (0, 0, 0, 1)]:
        set_variant(gf, v)
        gf.load_links(U)
        r = gf.fix(ALPHA, TOL, 5000)
        h = gf.get_history()
        assert r["status"] == lgf.LGF_OK and r["n_iter"] == r_ref["n_iter"], (v, r, r_ref["n_iter"])
        assert len(h) == len(href) and np.abs(h[:, 0] - href[:, 0]).max() <= F_TOL, v
        assert all(theta_close(a, b) for a, b in zip(h[:, 1], href[:, 1])), v
        assert np.abs(gf.get_links() - o.get()).max() <= LINK_TOL, v
    gm = lgf.GaugeFixer(dims, 12, precision=lgf.LGF_MIXED)
    gm.load_links(U)
    rm = gm.fix(ALPHA, TOL, 5000)
    assert rm["status"] == lgf.LGF_OK and rm["theta"] < TOL and abs(rm["F"] - r_ref["F"]) <= 1e-11


# ------------------------------------------------------------------ Coulomb gauge
@pytest.mark.parametrize("dims,storage", [((8, 8, 8, 8), 18), ((16, 16, 16, 8), 12), ((32, 32, 16, 16), 12), ((4, 8, 16, 4), 12)])
def test_coulomb_gauge_against_the_oracle(dims, storage):
    """LGF_OPT_GAUGE_DIRECTIONS = 3: stages, trajectory, stop iteration against the oracle's Coulomb mode (pinned on the
    CPU by the rate (1 - 12 alpha)^2, the 3-D Laplacian identity and slice locality); every kernel selection."""
    U = E.noisy(dims, 61, 0.3)
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.set_gauge(3)
    o.load(U)
    D_ref, X_ref = o.delta(), o.fa_field()
    F_ref, th_ref = o.measure()
    r20 = o.fix(ALPHA, 0.0, 20, history=True)
    href = np.array(r20["history"])
    U20 = o.get()
    o.load(U)
    r_ref = o.fix(ALPHA, TOL, 1000)
    gf = lgf.GaugeFixer(dims, storage)
    gf.set_option(lgf.LGF_OPT_GAUGE_DIRECTIONS, 3)
    assert gf.get_option(lgf.LGF_OPT_GAUGE_DIRECTIONS) == 3
    for v in [(0, 1, 1, 1), (0, 0, 0, 1), (1, 1, 1, 1), (1, 0, 0, 0)]:
        set_variant(gf, v)
        gf.load_links(U)
        F, th, _ = gf.measure()
        assert abs(F - F_ref) <= 1e-14 and abs(th - th_ref) <= 1e-12 * th_ref, v
        assert np.abs(gf.get_field(lgf.LGF_FIELD_DELTA) - D_ref).max() <= 1e-14 * max(1.0, np.abs(D_ref).max()), v
        assert np.abs(gf.get_field(lgf.LGF_FIELD_X) - X_ref).max() <= 1e-13 * np.abs(X_ref).max(), v
        gf.iterate(20, ALPHA)
        h = gf.get_history()
        assert np.abs(h[:, 0] - href[:, 0]).max() <= F_TOL, v
        assert all(theta_close(a, b) for a, b in zip(h[:, 1], href[:, 1])), v
        assert np.abs(gf.get_links() - U20).max() <= LINK_TOL, v
        gf.load_links(U)
        r = gf.fix(ALPHA, TOL, 1000)
        assert r["status"] == lgf.LGF_OK and r["n_iter"] == r_ref["n_iter"] and abs(r["F"] - r_ref["F"]) <= F_TOL, v
    # mixed precision in Coulomb gauge: both phases use the restricted condition
    gm = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_MIXED)
    gm.set_option(lgf.LGF_OPT_GAUGE_DIRECTIONS, 3)
    gm.load_links(U)
    r = gm.fix(ALPHA, TOL, 1000)
    assert r["status"] == lgf.LGF_OK and r["theta"] < TOL and abs(r["F"] - r_ref["F"]) <= 1e-10
    # back to Landau on the same context
    gf.set_option(lgf.LGF_OPT_GAUGE_DIRECTIONS, 4)
    set_variant(gf, (0, 1, 1, 1))
    gf.load_links(U)
    o.set_gauge(4)
    o.load(U)
    F, th = gf.iterate(3, ALPHA)
    F_ref, th_ref = o.iterate(3, ALPHA)
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref)


# ------------------------------------------------------------------ fp32
EPS32 = 2.0 ** -24      # fp32 unit round-off


@pytest.mark.parametrize("dims,storage", [((8, 8, 8, 8), 18), ((16, 16, 16, 16), 12), ((32, 16, 16, 32), 12), ((4, 8, 16, 4), 12),
                                          ((64, 64, 4, 4), 12), ((8, 4, 32, 64), 12)])
def test_fp32_stage_and_trajectory_against_the_fp64_oracle(dims, storage):
    """LGF_FP32: same kernels instantiated for float storage and arithmetic, lattice sums in double.  The oracle stays
    fp64 (it is the definition); the bounds are fp32 round-off times the operation counts of DESIGN.md section 7:
    Delta (16 link terms) 8 eps, X (FFT of log2 V stages, filter <= p2max/p2min) 32 eps, g 32 eps, all relative to the
    field maximum; F (a mean of O(1) terms, summed in double) 16 eps; links after k iterations 64 k eps."""
    U = E.noisy(dims, 43, 0.35)
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    D_ref, X_ref, g_ref = o.delta(), o.fa_field(), o.g_field(ALPHA)
    F_ref, th_ref = o.measure()
    r = o.fix(ALPHA, 0.0, 10, history=True)
    href = np.array(r["history"])
    U10 = o.get()
    gf = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_FP32)
    for v in [(0, 1, 1, 1), (0, 0, 0, 1), (1, 1, 1, 1)]:
        set_variant(gf, v)
        gf.load_links(U)
        F, th, _ = gf.measure()
        assert abs(F - F_ref) <= 16 * EPS32 and abs(th - th_ref) <= 16 * EPS32 * th_ref, v
        assert np.abs(gf.get_field(lgf.LGF_FIELD_DELTA) - D_ref).max() <= 8 * EPS32 * np.abs(D_ref).max(), v
        assert np.abs(gf.get_field(lgf.LGF_FIELD_X) - X_ref).max() <= 32 * EPS32 * np.abs(X_ref).max(), v
        assert np.abs(gf.get_field(lgf.LGF_FIELD_G, ALPHA) - g_ref).max() <= 32 * EPS32, v
        got = gf.get_links()
        assert np.abs(got[:, :, :2] - U[:, :, :2]).max() <= EPS32, v          # stored as float: one rounding
        F10, th10 = gf.iterate(10, ALPHA)
        h = gf.get_history()
        assert np.abs(h[:, 0] - href[:, 0]).max() <= 16 * EPS32, v
        assert np.all(np.abs(h[:, 1] - href[:, 1]) <= 64 * EPS32 * href[:, 1]), v
        assert np.abs(gf.get_links() - U10).max() <= 64 * 10 * EPS32, v


def test_fp32_converges_to_its_rounding_floor_and_keeps_invariants():
    """C1 in fp32: theta < 1e-10 is reached in the oracle's iteration count for that tolerance (+-1: the trajectories
    differ at fp32 round-off), theta < 1e-15 is not reachable (floor ~1e-14: LGF_NOT_CONVERGED), F agrees with the fp64
    fixed point to fp32 accuracy, the plaquette is invariant and the links stay unitary to fp32 accuracy."""
    U, cfg = E.make_config("C1")
    dims, storage = cfg["dims"], cfg["storage"]
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    r_ref = o.fix(ALPHA, 1e-10, 1000)
    gf = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_FP32)
    gf.load_links(U)
    _, _, plaq0 = gf.measure()
    r = gf.fix(ALPHA, 1e-10, 1000)
    assert r["status"] == lgf.LGF_OK and abs(r["n_iter"] - r_ref["n_iter"]) <= 1 and r["theta"] < 1e-10
    assert abs(r["F"] - r_ref["F"]) <= 64 * EPS32
    _, _, plaq1 = gf.measure()
    assert abs(plaq1 - plaq0) <= 64 * EPS32
    L = gf.get_links()
    assert np.abs(np.einsum("xmij,xmkj->xmik", L, L.conj()) - np.eye(3)).max() <= 64 * r["n_iter"] * EPS32
    r = gf.fix(ALPHA, TOL, 200)
    assert r["status"] == lgf.LGF_NOT_CONVERGED and 1e-16 < r["theta"] < 1e-12


@pytest.mark.parametrize("name", ["C0", "C1"])
def test_mixed_precision_fix_is_an_exact_gauge_copy_at_the_same_maximum(name):
    """LGF_MIXED: fp32 phase with accumulated transformation, applied to the fp64 links in one step, fp64 polish.
    The result must (i) reach theta < 1e-15, (ii) be a gauge copy of the input to fp64 accuracy (plaquette, unitarity),
    (iii) sit at the maximum the oracle's fp64 trajectory reaches: same F to 1e-12 (the value of the functional at a
    maximum does not depend on the path; the links themselves agree only up to one global SU(3) rotation, because the
    iteration never fixes the zero mode and fp32 round-off lets it drift, so they are not compared element by element),
    (iv) do most of its iterations in fp32."""
    U, cfg = E.make_config(name)
    dims, storage = cfg["dims"], cfg["storage"]
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    r_ref = o.fix(ALPHA, TOL, 1000)
    gf = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_MIXED)
    gf.load_links(U)
    _, _, plaq0 = gf.measure()
    r = gf.fix(ALPHA, TOL, 1000)
    n32 = gf.get_option(lgf.LGF_OPT_MIXED_FP32_ITERS)
    assert r["status"] == lgf.LGF_OK and r["theta"] < TOL
    assert 0 < n32 < r["n_iter"] <= r_ref["n_iter"] + 8 and r["n_iter"] - n32 <= 10       # most of the work in fp32
    assert abs(r["F"] - r_ref["F"]) <= F_TOL
    F1, th1, plaq1 = gf.measure()
    assert abs(plaq1 - plaq0) <= 1e-12 and F1 == r["F"]
    L = gf.get_links()
    assert np.abs(np.einsum("xmij,xmkj->xmik", L, L.conj()) - np.eye(3)).max() <= 1e-13
    # fp64 lgf_iterate on a mixed context is the plain fp64 path
    gf.load_links(U)
    o.load(U)
    F, th = gf.iterate(3, ALPHA)
    F_ref, th_ref = o.iterate(3, ALPHA)
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref) and np.abs(gf.get_links() - o.get()).max() <= LINK_TOL


def test_mixed_precision_hands_over_when_the_fp32_phase_stalls():
    """the fp32 phase must not eat the max_iter budget when it cannot reach its target.  With the switch
    threshold set to 1e-16 (below the fp32 floor of theta, ~1e-14) the fp32 phase stalls; the stagnation guard (theta
    has not halved within 256 iterations) ends it and the fp64 phase converges with the remaining budget -- where an
    unguarded fp32 phase would have used all of max_iter and returned LGF_NOT_CONVERGED."""
    U, cfg = E.make_config("C1")
    dims, storage = cfg["dims"], cfg["storage"]
    o = oracle.Oracle(dims, storage, fft_mode=1)
    o.load(U)
    r_ref = o.fix(ALPHA, TOL, 1000)
    gf = lgf.GaugeFixer(dims, storage, precision=lgf.LGF_MIXED)
    assert gf.get_option(lgf.LGF_OPT_MIXED_SWITCH) == 12
    gf.set_option(lgf.LGF_OPT_MIXED_SWITCH, 16)
    gf.load_links(U)
    r = gf.fix(ALPHA, TOL, 2000)
    n32 = gf.get_option(lgf.LGF_OPT_MIXED_FP32_ITERS)
    assert r["status"] == lgf.LGF_OK and r["theta"] < TOL, r
    assert r_ref["n_iter"] < n32 <= r_ref["n_iter"] + 256 + 64, (n32, r_ref["n_iter"])     # stalled, then stopped by the guard
    assert r["n_iter"] - n32 <= 12                                                        # a short fp64 polish
    assert abs(r["F"] - r_ref["F"]) <= F_TOL
    with pytest.raises(lgf.LgfError):
        gf.set_option(lgf.LGF_OPT_MIXED_SWITCH, 3)


def test_C1_ten_iterations_against_the_naive_dft_oracle():
    U, cfg = E.make_config("C1")
    o = oracle.Oracle(cfg["dims"], cfg["storage"], fft_mode=0)      # the definition
    o.load(U)
    F_ref, th_ref = o.iterate(10, ALPHA)
    gf = lgf.GaugeFixer(cfg["dims"], cfg["storage"])
    gf.load_links(U)
    F, th = gf.iterate(10, ALPHA)
    assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref)
    assert np.abs(gf.get_links() - o.get()).max() <= LINK_TOL


# ------------------------------------------------------------------ invariants through the GPU path alone
@pytest.mark.parametrize("storage", [12, 18])
def test_gpu_invariants_plaquette_unitarity_monotone(storage):
    dims = (16, 8, 8, 16)
    U = E.noisy(dims, 44, 0.45)
    gf = lgf.GaugeFixer(dims, storage)
    gf.load_links(U)
    _, _, p0 = gf.measure()
    o = oracle.Oracle(dims, storage)
    o.load(U)
    assert abs(p0 - o.plaquette()) < 1e-13
    r = gf.fix(ALPHA, TOL, 500)
    assert r["status"] == lgf.LGF_OK
    h = gf.get_history()
    assert len(h) == r["n_iter"] + 1
    F, th = h[:, 0], h[:, 1]
    assert np.all((F[1:] - F[:-1])[th[:-1] > 1e-25] >= -1e-14)     # monotone F at alpha = 0.08 (NS; A17)
    assert th[-1] < TOL and np.all(th[:-1] >= TOL)                   # strict stop, count = updates applied
    _, _, p1 = gf.measure()
    assert abs(p1 - p0) < 1e-12                                      # gauge invariance of the plaquette (NS)
    Uf = gf.get_links()
    I = np.eye(3)
    assert np.abs(Uf @ Uf.conj().swapaxes(-1, -2) - I).max() < 1e-13
    assert np.abs(np.linalg.det(Uf) - 1).max() < 1e-13


# ------------------------------------------------------------------ edge and degenerate cases
def test_edge_cases():
    dims = (8, 8, 8, 8)
    U = E.noisy(dims, 45, 0.3)
    gf = lgf.GaugeFixer(dims, 12)
    L = lgf.lib()
    import ctypes as C
    F = C.c_double()
    # before load
    assert L.lgf_iterate(gf._h, 1, 0.08, C.byref(F), C.byref(F)) == lgf.LGF_ERR_NOT_LOADED
    assert L.lgf_fix(gf._h, 0.08, 1e-15, 10, None, None, None) == lgf.LGF_ERR_NOT_LOADED
    assert L.lgf_measure(gf._h, None, None, None) == lgf.LGF_ERR_NOT_LOADED
    buf = np.empty(4096 * 72)
    assert L.lgf_get_links(gf._h, buf.ctypes.data) == lgf.LGF_ERR_NOT_LOADED
    gf.load_links(U)
    # bad arguments
    assert L.lgf_iterate(gf._h, -1, 0.08, None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_iterate(gf._h, 1, 0.0, None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_iterate(gf._h, 1, float("nan"), None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_fix(gf._h, 0.08, -1.0, 10, None, None, None) == lgf.LGF_ERR_INVALID_ARG
    assert L.lgf_fix(gf._h, 0.08, 1e-15, -1, None, None, None) == lgf.LGF_ERR_INVALID_ARG
    # n = 0: a pure measurement, links untouched (A5)
    o = oracle.Oracle(dims, 12)
    o.load(U)
    F0, th0 = o.measure()
    Fg, thg = gf.iterate(0, ALPHA)
    assert abs(Fg - F0) <= 1e-14 and abs(thg - th0) <= 1e-12 * th0
    assert np.array_equal(gf.get_links()[:, :, :2], U[:, :, :2])
    # max_iter = 0 -> NOT_CONVERGED with the initial measurement, links untouched
    r = gf.fix(ALPHA, TOL, 0)
    assert r["status"] == lgf.LGF_NOT_CONVERGED and r["n_iter"] == 0 and abs(r["F"] - F0) <= 1e-14
    assert np.array_equal(gf.get_links()[:, :, :2], U[:, :, :2])
    # max_iter smaller than needed, batch boundaries: counts are exact for every batch size
    for batch in (1, 3, 8):
        gf.set_option(lgf.LGF_OPT_BATCH, batch)
        gf.load_links(U)
        r = gf.fix(ALPHA, TOL, 7)
        assert r["status"] == lgf.LGF_NOT_CONVERGED and r["n_iter"] == 7
    o.iterate(7, ALPHA)
    assert np.abs(gf.get_links() - o.get()).max() <= 1e-12
    gf.set_option(lgf.LGF_OPT_BATCH, 8)
    # fix on already fixed links returns 0 updates (A5) and leaves them alone
    r = gf.fix(ALPHA, TOL, 500)
    assert r["status"] == lgf.LGF_OK
    Ufix = gf.get_links()
    r2 = gf.fix(ALPHA, TOL, 500)
    assert r2["status"] == lgf.LGF_OK and r2["n_iter"] == 0
    assert np.array_equal(gf.get_links(), Ufix)
    # a loose tolerance stops earlier, at the oracle's iteration
    gf.load_links(U)
    r3 = gf.fix(ALPHA, 1e-6, 500)
    o2 = oracle.Oracle(dims, 12)
    o2.load(U)
    assert r3["n_iter"] == o2.fix(ALPHA, 1e-6, 500)["n_iter"]


def test_identity_links_are_a_fixed_point():
    dims = (4, 8, 4, 8)
    V = 1024
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (V, 4, 3, 3)).copy()
    for storage in (12, 18):
        gf = lgf.GaugeFixer(dims, storage)
        gf.load_links(U)
        F, th = gf.iterate(3, ALPHA)
        assert F == 1.0 and th == 0.0
        assert np.array_equal(gf.get_links(), U)
        r = gf.fix(ALPHA, TOL, 10)
        assert r["n_iter"] == 0 and r["status"] == lgf.LGF_OK


def test_nonfinite_links_are_reported():
    dims = (4, 4, 4, 4)
    U = E.noisy(dims, 46, 0.3)
    U[17, 2, 0, 1] = np.nan
    gf = lgf.GaugeFixer(dims, 18)
    gf.load_links(U)
    with pytest.raises(lgf.LgfError) as ei:
        gf.iterate(2, ALPHA)
    assert ei.value.status == lgf.LGF_ERR_NUMERIC


def test_largest_axis_and_smallest_lattice():
    # L = 128 on one axis (the library's maximum) and the 4^4 minimum; oracle in FFT mode for the long axis
    for dims in [(128, 4, 4, 4), (4, 4, 4, 128), (4, 128, 4, 4), (4, 4, 128, 4)]:
        U = E.noisy(dims, 47, 0.3)
        o = oracle.Oracle(dims, 12, fft_mode=1)
        o.load(U)
        F_ref, th_ref = o.iterate(3, ALPHA)
        gf = lgf.GaugeFixer(dims, 12)
        gf.load_links(U)
        F, th = gf.iterate(3, ALPHA)
        assert abs(F - F_ref) <= F_TOL and theta_close(th, th_ref), dims
        assert np.abs(gf.get_links() - o.get()).max() <= LINK_TOL, dims


def test_launch_count_and_profile():
    dims = (8, 8, 8, 8)
    U = E.noisy(dims, 48, 0.3)
    gf = lgf.GaugeFixer(dims, 12)
    gf.load_links(U)
    n0 = gf.launch_count()
    gf.iterate(8, ALPHA)
    assert gf.launch_count() - n0 == 9 * 5       # generic passes at 8^4: S1+A, S5, B, C, S3+S4
    gf.set_profiling(True)
    gf.iterate(4, ALPHA)
    prof = gf.get_profile()
    gf.set_profiling(False)
    assert prof["k_fft23_mid"]["launches"] == 5 and prof["k_update_quad"]["launches"] == 5
    assert all(v["ms"] > 0 for v in prof.values())
    assert lgf.copy_peak_gbs(1 << 28, 3) > 500.0
    assert lgf.stream_peak_gbs(1 << 18, False, 3) > 500.0 and lgf.stream_peak_gbs(1 << 18, True, 3) > 500.0


def test_option_changes_between_calls_never_replay_a_stale_graph():
    """The CUDA-graph cache is keyed by the full selection tuple and alpha (a hashed key collided): after any
    change of option or alpha on one context, the next call must give what a fresh context with those settings gives."""
    dims, storage = (16, 16, 16, 16), 12
    U = E.noisy(dims, 49, 0.35)
    gf = lgf.GaugeFixer(dims, storage)
    seq = [({}, 0.08), ({"LGF_OPT_STORE_G": 1}, 0.08), ({"LGF_OPT_STORE_G": 0}, 0.05), ({"LGF_OPT_FAST_FFT": 0}, 0.05),
           ({"LGF_OPT_FAST_FFT": 1, "LGF_OPT_PDL": 0}, 0.08), ({"LGF_OPT_FOURIER_ACCEL": 0}, 0.08),
           ({"LGF_OPT_FOURIER_ACCEL": 1, "LGF_OPT_GAUGE_DIRECTIONS": 3}, 0.08), ({"LGF_OPT_GAUGE_DIRECTIONS": 4, "LGF_OPT_PDL": 1}, 0.0625)]
    state = {}
    for opts, alpha in seq:
        state.update(opts)
        for k, v in opts.items():
            gf.set_option(getattr(lgf, k), v)
        fresh = lgf.GaugeFixer(dims, storage)
        for k, v in state.items():
            fresh.set_option(getattr(lgf, k), v)
        gf.load_links(U)
        fresh.load_links(U)
        a = gf.iterate(16, alpha)
        b = fresh.iterate(16, alpha)
        assert a == b, (state, alpha, a, b)
        assert np.array_equal(gf.get_links(), fresh.get_links()), (state, alpha)
        fresh.destroy()


def test_fast_fft_pass_selection_64_extents():
    """64 extents: plane passes with one component per CTA (bits 1 and 4), pass B with a short x0 chunk (bit 2)."""
    for dims, mask in [((64, 64, 4, 4), 5), ((4, 4, 64, 64), 2), ((32, 64, 32, 64), 7), ((8, 8, 64, 32), 2), ((64, 32, 16, 16), 7)]:
        gf = lgf.GaugeFixer(dims, 12)
        assert gf.get_option(lgf.LGF_OPT_FAST_FFT) == mask, dims
        gf.destroy()


def test_fast_fft_pass_selection():
    """Which lattices run the compile-time-sized passes (bit mask: 1 pass A, 2 pass B, 4 pass C)."""
    for dims, mask in [((32, 32, 32, 32), 7), ((16, 16, 16, 16), 7), ((16, 32, 32, 16), 7), ((8, 8, 16, 32), 2),
                       ((16, 32, 4, 8), 5), ((4, 8, 16, 32), 0), ((8, 8, 8, 8), 0)]:
        gf = lgf.GaugeFixer(dims, 12)
        assert gf.get_option(lgf.LGF_OPT_FAST_FFT) == mask, dims
        # TMA-staged passes: bit 1 pass B (wherever the compile-time-sized pass B runs), bit 2 pass A (16/32-extent planes,
        # from two planes per SM on: 32^4 has 1024, 16^4 256)
        tma_a = 2 if ((mask & 1) and dims[2] * dims[3] >= 512) else 0
        assert gf.get_option(lgf.LGF_OPT_TMA) == ((1 if (mask & 2) else 0) | tma_a), dims
        gf.set_option(lgf.LGF_OPT_FAST_FFT, 0)
        assert gf.get_option(lgf.LGF_OPT_TMA) == 0
        assert gf.get_option(lgf.LGF_OPT_FAST_FFT) == 0
