"""Seeded synthetic SU(3) gauge-link ensembles (inputs only).

This module is DATA, not method: it holds none of the gauge-fixing arithmetic
(no Delta, no FFT, no filter, no projection, no link update).  It serves both
the CPU oracle (``oracle/``) and the CUDA path (``paper_1301_3460_b200/``),
which otherwise share nothing.

The paper's inputs were Wilson-action configurations on 32^4 at three
unstated beta values; they are not available, so the ensembles
below stand in for them, as prescribed by BASELINE.json ``configs``:

* ``pure_gauge``: U_mu(x) = h(x) h^dagger(x+mu), h Haar-random SU(3)
  (BASELINE.json configs[0]); a gauge copy of the trivial configuration, so the
  closed-form maximum is F = 1.
* ``noisy``: U_mu(x) = h(x) exp(i eps H_mu(x)) h^dagger(x+mu), with
  H = sum_a c_a lambda_a / 2, c_a ~ N(0,1) (BASELINE.json configs[1];
  normalisation reading A12 of SURVEY.md section 8(c)).

Array convention (the canonical host layout of include/lgf.h):
``links[x, mu, i, j]`` complex128, site index
``x = x0 + L0*(x1 + L1*(x2 + L2*x3))`` (x0 fastest), periodic boundaries;
viewed as float64 this is ``[V][4][3][3][2]``.

RNG: numpy's counter-based Philox bit generator keyed by (seed, stream); all
draws are made serially in a fixed order, so an ensemble depends only on
(dims, seed, stream, eps).
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "CONFIGS",
    "volume",
    "haar_su3",
    "gaussian_su3_algebra",
    "expi_hermitian",
    "pure_gauge",
    "noisy",
    "make_config",
    "abelian",
    "as_real",
    "as_complex",
    "device_su3",
    "noisy_device",
    "wilson",
]

# Gell-Mann matrices lambda_1..lambda_8
_GM = np.zeros((8, 3, 3), dtype=np.complex128)
_GM[0, 0, 1] = _GM[0, 1, 0] = 1
_GM[1, 0, 1] = -1j
_GM[1, 1, 0] = 1j
_GM[2, 0, 0] = 1
_GM[2, 1, 1] = -1
_GM[3, 0, 2] = _GM[3, 2, 0] = 1
_GM[4, 0, 2] = -1j
_GM[4, 2, 0] = 1j
_GM[5, 1, 2] = _GM[5, 2, 1] = 1
_GM[6, 1, 2] = -1j
_GM[6, 2, 1] = 1j
_GM[7] = np.diag([1, 1, -2]) / np.sqrt(3.0)


def volume(dims) -> int:
    d = tuple(int(v) for v in dims)
    assert len(d) == 4
    return d[0] * d[1] * d[2] * d[3]


def _rng(seed: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def haar_su3(rng: np.random.Generator, n: int) -> np.ndarray:
    """n Haar-random SU(3) matrices: QR of a complex Ginibre matrix, the phases of
    diag(R) moved into Q (Haar on U(3)), then divided by det^(1/3)."""
    z = rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))
    q, r = np.linalg.qr(z)
    d = np.einsum("nii->ni", r)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    q = q * np.exp(-1j * np.angle(det) / 3.0)[:, None, None]
    return np.ascontiguousarray(q)


def gaussian_su3_algebra(rng: np.random.Generator, n: int) -> np.ndarray:
    """n traceless Hermitian H = sum_a c_a lambda_a/2, c_a ~ N(0,1) ("unit variance per generator")."""
    c = rng.standard_normal((n, 8))
    return np.einsum("na,aij->nij", c, _GM) * 0.5


def expi_hermitian(H: np.ndarray, eps: float) -> np.ndarray:
    """exp(i eps H) for stacked Hermitian H by eigendecomposition."""
    w, v = np.linalg.eigh(H)
    return np.einsum("nik,nk,njk->nij", v, np.exp(1j * eps * w), v.conj())


def _shift_fwd(h: np.ndarray, dims, mu: int) -> np.ndarray:
    """h(x + mu_hat) as an array indexed by x (periodic)."""
    L0, L1, L2, L3 = dims
    h4 = h.reshape(L3, L2, L1, L0, 3, 3)
    return np.roll(h4, -1, axis=3 - mu).reshape(-1, 3, 3)


def _dress(h: np.ndarray, dims, middle=None) -> np.ndarray:
    V = h.shape[0]
    U = np.empty((V, 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        hf = _shift_fwd(h, dims, mu).conj().transpose(0, 2, 1)
        if middle is None:
            U[:, mu] = h @ hf
        else:
            U[:, mu] = h @ middle[mu] @ hf
    return U


def pure_gauge(dims, seed: int, stream: int = 0) -> np.ndarray:
    """U_mu(x) = h(x) h^dagger(x+mu), h Haar (BASELINE.json configs[0])."""
    dims = tuple(int(v) for v in dims)
    rng = _rng(seed, stream)
    h = haar_su3(rng, volume(dims))
    return _dress(h, dims)


def noisy(dims, seed: int, eps: float, stream: int = 0, chunk: int = 1 << 20) -> np.ndarray:
    """U_mu(x) = h(x) exp(i eps H_mu(x)) h^dagger(x+mu) (BASELINE.json configs[1])."""
    dims = tuple(int(v) for v in dims)
    V = volume(dims)
    rng = _rng(seed, stream)
    h = haar_su3(rng, V)
    U = np.empty((V, 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        hf = _shift_fwd(h, dims, mu).conj().transpose(0, 2, 1)
        for a in range(0, V, chunk):
            b = min(V, a + chunk)
            E = expi_hermitian(gaussian_su3_algebra(rng, b - a), eps)
            U[a:b, mu] = h[a:b] @ E @ hf[a:b]
    return U


def abelian(dims, seed: int, scale: float = 1.0) -> np.ndarray:
    """Diagonal links diag(e^{ia}, e^{ib}, e^{-i(a+b)}), a,b ~ scale*N(0,1)
    (inputs of the Abelian special-case pin P13)."""
    dims = tuple(int(v) for v in dims)
    V = volume(dims)
    rng = _rng(seed, 77)
    ab = scale * rng.standard_normal((V, 4, 2))
    ph = np.stack([ab[..., 0], ab[..., 1], -(ab[..., 0] + ab[..., 1])], axis=-1)
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    for j in range(3):
        U[:, :, j, j] = np.exp(1j * ph[..., j])
    return U


# name -> (dims, storage, builder kwargs); BASELINE.json configs[0..4] (0-based, reading A11).
CONFIGS = {
    "C0": dict(dims=(8, 8, 8, 8), storage=18, kind="pure_gauge", seed=1),
    "C1": dict(dims=(16, 16, 16, 16), storage=12, kind="noisy", seed=2, eps=0.35),
    "C2a": dict(dims=(32, 32, 32, 32), storage=12, kind="noisy", seed=3, stream=0, eps=0.25),
    "C2b": dict(dims=(32, 32, 32, 32), storage=12, kind="noisy", seed=3, stream=1, eps=0.35),
    "C2c": dict(dims=(32, 32, 32, 32), storage=12, kind="noisy", seed=3, stream=2, eps=0.45),
    "C3": dict(dims=(32, 32, 32, 64), storage=12, kind="noisy", seed=4, eps=0.40),
    "C4": dict(dims=(64, 64, 64, 64), storage=12, kind="noisy", seed=5, eps=0.35),
}


def make_config(name: str) -> tuple[np.ndarray, dict]:
    cfg = dict(CONFIGS[name])
    if cfg["kind"] == "pure_gauge":
        U = pure_gauge(cfg["dims"], cfg["seed"], cfg.get("stream", 0))
    else:
        U = noisy(cfg["dims"], cfg["seed"], cfg["eps"], cfg.get("stream", 0))
    return U, cfg


def as_real(U: np.ndarray) -> np.ndarray:
    """complex [V,4,3,3] -> float64 [V,4,3,3,2] (no copy when contiguous)."""
    U = np.ascontiguousarray(U, dtype=np.complex128)
    return U.view(np.float64).reshape(U.shape + (2,))


def as_complex(R: np.ndarray) -> np.ndarray:
    R = np.ascontiguousarray(R, dtype=np.float64)
    return R.view(np.complex128).reshape(R.shape[:-1])


def device_su3(dims, seed: int, spread: float = 0.15):
    """Seeded random SU(3) links generated ON THE CUDA DEVICE (torch), for lattices too large to build with numpy
    in test time (64^4: 67 M links).  U = rows of GramSchmidt(1 + spread * G), G complex Gaussian, third row the
    conjugate cross product -- smooth-ish links near the identity, no gauge structure.  Returns a torch complex128
    tensor [V, 4, 3, 3] in the canonical order of include/lgf.h.  Inputs only: nothing of the method is here.
    These are not the BASELINE.json ensembles (those are `noisy`/`pure_gauge`); they serve property and
    sampled-site parity tests and kernel timing at sizes where the host generator takes minutes."""
    import torch
    V = volume(dims)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(int(seed))
    n = V * 4
    U = torch.empty(n, 3, 3, dtype=torch.complex128, device="cuda")
    chunk = 1 << 22
    for o in range(0, n, chunk):
        m = min(chunk, n - o)
        A = torch.randn(m, 2, 3, 2, dtype=torch.float64, device="cuda", generator=gen)
        A = torch.view_as_complex(A) * spread
        A[:, 0, 0] += 1
        A[:, 1, 1] += 1
        u = A[:, 0]
        u = u / u.abs().pow(2).sum(-1, keepdim=True).sqrt()
        v = A[:, 1] - (u.conj() * A[:, 1]).sum(-1, keepdim=True) * u
        v = v / v.abs().pow(2).sum(-1, keepdim=True).sqrt()
        U[o:o + m, 0] = u
        U[o:o + m, 1] = v
        U[o:o + m, 2] = torch.linalg.cross(u, v).conj()
    return U.reshape(V, 4, 3, 3)


def noisy_device(dims, seed: int, eps: float, stream: int = 0, device: str = "cuda", chunk: int = 1 << 22):
    """The `noisy` recipe of BASELINE.json configs[1] -- U_mu(x) = h(x) exp(i eps H_mu(x)) h^dagger(x+mu), h Haar-random
    SU(3), H = sum_a c_a lambda_a / 2 with c_a ~ N(0,1) (reading A12) -- generated with torch on `device`, for the
    lattices whose numpy build takes minutes (C4: 64^4, 67 M links).  Same distribution as `noisy`, different random
    stream (torch's Philox generator seeded with (seed, stream) instead of numpy's), and the two linear-algebra steps
    are written as their closed forms so that they run as plain tensor ops: the QR of the Ginibre matrix with a
    positive R diagonal IS column Gram-Schmidt, and exp(i eps H) is torch.linalg.matrix_exp.  Returns a torch
    complex128 tensor [V, 4, 3, 3] in the canonical order of include/lgf.h; the caller copies it to the host once and
    feeds the same array to the oracle and to lgf_load_links (reading A12b).  Inputs only."""
    import torch
    dims = tuple(int(v) for v in dims)
    V = volume(dims)
    gen = torch.Generator(device=device)
    gen.manual_seed((int(seed) << 20) + int(stream))
    gm = torch.from_numpy(_GM).to(device)
    h = torch.empty(V, 3, 3, dtype=torch.complex128, device=device)
    for a in range(0, V, chunk):
        b = min(V, a + chunk)
        z = torch.view_as_complex(torch.randn(b - a, 3, 3, 2, dtype=torch.float64, device=device, generator=gen))
        # column Gram-Schmidt = QR with positive diag(R): Haar on U(3) (the phase fix of haar_su3); a second pass
        # restores orthogonality to rounding where two Gaussian columns were nearly parallel
        q = z
        for _ in range(2):
            q0 = q[:, :, 0] / q[:, :, 0].abs().pow(2).sum(-1, keepdim=True).sqrt()
            v1 = q[:, :, 1] - (q0.conj() * q[:, :, 1]).sum(-1, keepdim=True) * q0
            q1 = v1 / v1.abs().pow(2).sum(-1, keepdim=True).sqrt()
            v2 = q[:, :, 2] - (q0.conj() * q[:, :, 2]).sum(-1, keepdim=True) * q0 - (q1.conj() * q[:, :, 2]).sum(-1, keepdim=True) * q1
            q2 = v2 / v2.abs().pow(2).sum(-1, keepdim=True).sqrt()
            q = torch.stack([q0, q1, q2], dim=-1)
        det = torch.linalg.det(q)
        h[a:b] = q * torch.exp(-1j * torch.angle(det) / 3.0)[:, None, None]
    L0, L1, L2, L3 = dims
    h4 = h.view(L3, L2, L1, L0, 3, 3)
    U = torch.empty(V, 4, 3, 3, dtype=torch.complex128, device=device)
    for mu in range(4):
        hf = torch.roll(h4, -1, dims=3 - mu).reshape(V, 3, 3).conj().transpose(1, 2)      # h^dagger(x + mu)
        for a in range(0, V, chunk):
            b = min(V, a + chunk)
            c = torch.randn(b - a, 8, dtype=torch.float64, device=device, generator=gen)
            H = torch.einsum("na,aij->nij", c.to(torch.complex128), gm) * 0.5
            Ex = torch.linalg.matrix_exp(1j * eps * H)
            # one Gram-Schmidt clean-up of the rows (A12): matrix_exp leaves ~1e-14 of non-unitarity
            u = Ex[:, 0] / Ex[:, 0].abs().pow(2).sum(-1, keepdim=True).sqrt()
            v = Ex[:, 1] - (u.conj() * Ex[:, 1]).sum(-1, keepdim=True) * u
            v = v / v.abs().pow(2).sum(-1, keepdim=True).sqrt()
            Ex = torch.stack([u, v, torch.linalg.cross(u, v).conj()], dim=1)
            U[a:b, mu] = h[a:b] @ Ex @ hf[a:b]
    return U


def wilson(dims, beta: float, sweeps: int, seed: int, device: str = "cpu", hot: bool = False, overrelax: int = 0, history=None):
    """Thermalised Wilson-action configuration (ensembles/heatbath.py: Cabibbo-Marinari heat bath, Kennedy-Pendleton
    SU(2) updates, `overrelax` over-relaxation sweeps after each heat-bath sweep) -- the kind of input the paper fixes
    (generated as in its ref. [6]), at a beta of the caller's choice.  `history` (a list)
    receives the average plaquette after every sweep (thermalisation check: heatbath.plateau).  Returns a torch
    complex128 tensor [V, 4, 3, 3] on `device` (use .cpu().numpy() for the host entry points)."""
    from .heatbath import thermalise
    return thermalise(dims, beta, sweeps, seed, device=device, hot=hot, overrelax=overrelax, history=history)
