"""Thermalised SU(3) gauge configurations for the Wilson action (inputs only).

The paper fixes the gauge of Wilson-action configurations at three beta values; those ensembles are not
available.  This module generates configurations of the same kind: Cabibbo-Marinari pseudo heat bath over the three
SU(2) subgroups of SU(3), each subgroup update drawn with the Kennedy-Pendleton algorithm, links visited direction by
direction on the two checkerboard parities (links of one direction and one parity share no plaquette), rows
re-orthonormalised after every sweep.  It is written with torch tensor operations so that it runs on the GPU for the
32^4 workloads (seconds) and on the CPU for small test lattices.  Nothing of the gauge-fixing method is in here.

    S = beta * sum_plaquettes (1 - (1/3) Re Tr U_P)

Array convention as everywhere (include/lgf.h): links[x, mu, i, j], x = x0 + L0*(x1 + L1*(x2 + L2*x3)).
Seeded: torch.Generator(seed) on the chosen device; a configuration depends on (dims, beta, sweeps, seed, device type).
"""
from __future__ import annotations

import math

__all__ = ["thermalise", "average_plaquette", "overrelax_sweep", "plateau"]


def _axis(mu: int) -> int:
    return 3 - mu            # lattice view [L3, L2, L1, L0, 4, 3, 3]: direction mu lives on tensor axis 3 - mu


def _fwd(f, mu):             # f(x + mu)
    return f.roll(-1, dims=_axis(mu))


def _bwd(f, mu):             # f(x - mu)
    return f.roll(1, dims=_axis(mu))


def _dag(m):
    return m.conj().transpose(-1, -2)


def _staples(U, mu):
    """A_mu(x) = sum_{nu != mu} [U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)],
    so that the plaquettes through U_mu(x) contribute Re Tr[U_mu(x) A_mu(x)]."""
    Um = U[..., mu, :, :]
    A = None
    for nu in range(4):
        if nu == mu:
            continue
        Un = U[..., nu, :, :]
        up = _fwd(Un, mu) @ _dag(_fwd(Um, nu)) @ _dag(Un)
        Un_b = _bwd(Un, nu)
        dn = _dag(_fwd(Un_b, mu)) @ _dag(_bwd(Um, nu)) @ Un_b
        A = up + dn if A is None else A + up + dn
    return A


def _kennedy_pendleton(gamma, gen):
    """x0 in [-1, 1] with density sqrt(1 - x0^2) exp(gamma x0), elementwise (gamma > 0), by rejection."""
    import torch
    x0 = torch.empty_like(gamma)
    todo = torch.ones_like(gamma, dtype=torch.bool)
    for _ in range(200):
        n = int(todo.sum())
        if n == 0:
            break
        g = gamma[todo]
        r = torch.rand(4, n, dtype=gamma.dtype, device=gamma.device, generator=gen).clamp_min(1e-300)
        lam2 = -(torch.log(r[0]) + torch.cos(2.0 * math.pi * r[1]) ** 2 * torch.log(r[2])) / (2.0 * g)
        ok = r[3] ** 2 <= 1.0 - lam2
        idx = todo.nonzero(as_tuple=True)[0][ok]
        x0[idx] = 1.0 - 2.0 * lam2[ok]
        todo[idx] = False
    x0[todo] = 1.0          # not reached in practice (acceptance > 0.5 per trial)
    return x0


def _su2_heatbath(W, i, j, beta, gen):
    """New SU(2) element alpha (as 4 real quaternion components embedded on rows/cols i, j) for the subgroup (i, j),
    given W = U A restricted to the sites being updated.  Returns the 3x3 matrices alpha."""
    import torch
    w00, w01, w10, w11 = W[:, i, i], W[:, i, j], W[:, j, i], W[:, j, j]
    a0 = 0.5 * (w00.real + w11.real)
    a1 = 0.5 * (w01.imag + w10.imag)
    a2 = 0.5 * (w01.real - w10.real)
    a3 = 0.5 * (w00.imag - w11.imag)
    k = torch.sqrt(a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3).clamp_min(1e-300)
    v0, v1, v2, v3 = a0 / k, a1 / k, a2 / k, a3 / k               # V = v0 + i v.sigma in SU(2)
    gamma = (2.0 * beta / 3.0) * k                                   # weight exp(gamma * x0), x0 = (1/2) tr(alpha V)
    x0 = _kennedy_pendleton(gamma, gen)
    n = x0.numel()
    rad = torch.sqrt((1.0 - x0 * x0).clamp_min(0.0))
    ct = 2.0 * torch.rand(n, dtype=x0.dtype, device=x0.device, generator=gen) - 1.0
    st = torch.sqrt((1.0 - ct * ct).clamp_min(0.0))
    ph = 2.0 * math.pi * torch.rand(n, dtype=x0.dtype, device=x0.device, generator=gen)
    x1, x2, x3 = rad * st * torch.cos(ph), rad * st * torch.sin(ph), rad * ct
    # alpha = X V^dag with quaternions: (x0 + i x.sigma)(v0 - i v.sigma)
    b0 = x0 * v0 + x1 * v1 + x2 * v2 + x3 * v3
    b1 = -x0 * v1 + x1 * v0 + x2 * v3 - x3 * v2
    b2 = -x0 * v2 + x2 * v0 + x3 * v1 - x1 * v3
    b3 = -x0 * v3 + x3 * v0 + x1 * v2 - x2 * v1
    return _embed_su2(b0, b1, b2, b3, i, j, W.dtype, W.device)


def _embed_su2(b0, b1, b2, b3, i, j, dtype, device):
    """The SU(2) element b0 + i b.sigma on rows/columns i, j of a 3x3 identity."""
    import torch
    n = b0.numel()
    al = torch.zeros(n, 3, 3, dtype=dtype, device=device)
    for d in range(3):
        al[:, d, d] = 1.0
    al[:, i, i] = torch.complex(b0, b3)
    al[:, i, j] = torch.complex(b2, b1)
    al[:, j, i] = torch.complex(-b2, b1)
    al[:, j, j] = torch.complex(b0, -b3)
    return al


def _su2_overrelax(W, i, j):
    """Micro-canonical (over-relaxation) update of the subgroup (i, j): with the SU(2) part of W = U A written as k V,
    alpha = (V^dagger)^2 reflects U about the minimum of the local action; tr(alpha k V) = k tr(V^dagger) = k tr(V), so
    Re Tr[U A] -- and with it the Wilson action -- is unchanged (ref. [6]: heat bath + over-relaxation)."""
    import torch
    w00, w01, w10, w11 = W[:, i, i], W[:, i, j], W[:, j, i], W[:, j, j]
    a0 = 0.5 * (w00.real + w11.real)
    a1 = 0.5 * (w01.imag + w10.imag)
    a2 = 0.5 * (w01.real - w10.real)
    a3 = 0.5 * (w00.imag - w11.imag)
    k = torch.sqrt(a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3).clamp_min(1e-300)
    v0, v1, v2, v3 = a0 / k, a1 / k, a2 / k, a3 / k
    return _embed_su2(2.0 * v0 * v0 - 1.0, -2.0 * v0 * v1, -2.0 * v0 * v2, -2.0 * v0 * v3, i, j, W.dtype, W.device)


def _reunitarise(U):
    import torch
    u = U[..., 0, :]
    u = u / torch.linalg.vector_norm(u, dim=-1, keepdim=True)
    v = U[..., 1, :] - (u.conj() * U[..., 1, :]).sum(-1, keepdim=True) * u
    v = v / torch.linalg.vector_norm(v, dim=-1, keepdim=True)
    w = torch.linalg.cross(u, v).conj()
    return torch.stack([u, v, w], dim=-2)


def average_plaquette(links, dims):
    """(1/(6 V)) sum_x sum_{mu<nu} (1/3) Re Tr U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag  for links [V,4,3,3] (torch)."""
    U = links.reshape(dims[3], dims[2], dims[1], dims[0], 4, 3, 3)
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Um, Un = U[..., mu, :, :], U[..., nu, :, :]
            P = Um @ _fwd(Un, mu) @ _dag(_fwd(Um, nu)) @ _dag(Un)
            tot = tot + P.diagonal(dim1=-2, dim2=-1).sum(-1).real.mean()
    return float(tot) / 18.0


def _parity_masks(shape, device):
    import torch
    ar = [torch.arange(n, device=device) for n in shape]
    parity = (ar[0][:, None, None, None] + ar[1][None, :, None, None] + ar[2][None, None, :, None] + ar[3][None, None, None, :]) % 2
    return [(parity == p).reshape(-1) for p in (0, 1)]


def _sweep(U, shape, masks, update):
    """One sweep over all links: direction by direction, parity by parity; `update(W, i, j)` gives the SU(2) factor."""
    for mu in range(4):
        for p in (0, 1):
            A = _staples(U, mu).reshape(-1, 3, 3)[masks[p]]
            Ul = U[..., mu, :, :].reshape(-1, 3, 3)[masks[p]]
            for (i, j) in ((0, 1), (0, 2), (1, 2)):
                Ul = update(Ul @ A, i, j) @ Ul
            flat = U[..., mu, :, :].reshape(-1, 3, 3).clone()
            flat[masks[p]] = Ul
            U[..., mu, :, :] = flat.reshape(*shape, 3, 3)
    return U


def overrelax_sweep(links, dims):
    """One micro-canonical over-relaxation sweep of links [V,4,3,3] (torch): every link reflected in each SU(2) subgroup.
    Deterministic; leaves the Wilson action unchanged up to rounding (no re-orthonormalisation here, so that the
    conservation can be checked to rounding; thermalise() re-orthonormalises after its sweeps)."""
    L0, L1, L2, L3 = (int(d) for d in dims)
    shape = (L3, L2, L1, L0)
    U = links.reshape(*shape, 4, 3, 3).clone()
    U = _sweep(U, shape, _parity_masks(shape, U.device), _su2_overrelax)
    return U.reshape(-1, 4, 3, 3)


def plateau(history, window: int = 5):
    """Thermalisation check on a plaquette history (one value per sweep): (mean of the last `window` values, their
    spread max - min, the drift between the means of the two last windows).  A thermalised run shows a drift no larger
    than the spread."""
    import numpy as np
    h = np.asarray(history, dtype=float)
    if len(h) < 2 * window:
        return float(h[-window:].mean()), float(np.ptp(h[-window:])), float("nan")
    return float(h[-window:].mean()), float(np.ptp(h[-window:])), float(h[-window:].mean() - h[-2 * window:-window].mean())


def thermalise(dims, beta: float, sweeps: int, seed: int, device: str = "cpu", hot: bool = False, overrelax: int = 0, history=None):
    """`sweeps` compound sweeps at coupling beta from a cold (identity) or hot (random) start, each one heat-bath sweep
    followed by `overrelax` over-relaxation sweeps (the usual mix, PAPER.md:72 ref. [6]).  `history`: a list that
    receives the average plaquette after every compound sweep (for the thermalisation check, plateau()).
    Returns a torch complex128 tensor [V, 4, 3, 3] on `device`."""
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(int(seed))
    L0, L1, L2, L3 = (int(d) for d in dims)
    shape = (L3, L2, L1, L0)
    U = torch.zeros(*shape, 4, 3, 3, dtype=torch.complex128, device=device)
    for d in range(3):
        U[..., d, d] = 1.0
    if hot:
        A = torch.view_as_complex(torch.randn(*shape, 4, 3, 3, 2, dtype=torch.float64, device=device, generator=gen))
        U = _reunitarise(A)
    masks = _parity_masks(shape, device)
    for _ in range(int(sweeps)):
        U = _sweep(U, shape, masks, lambda W, i, j: _su2_heatbath(W, i, j, float(beta), gen))
        for _ in range(int(overrelax)):
            U = _sweep(U, shape, masks, _su2_overrelax)
        U = _reunitarise(U)
        if history is not None:
            history.append(average_plaquette(U.reshape(-1, 4, 3, 3), dims))
    return U.reshape(-1, 4, 3, 3)
