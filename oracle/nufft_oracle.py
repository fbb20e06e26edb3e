"""fp64 oracle of the NUFFT force path (TEST INFRASTRUCTURE, see package docstring).

Two independent things live here:

* ``nudft_force_bruteforce`` -- the DEFINITION: Eq. 2.18 (:254) followed by the Poisson
  solve / spectral gradient (:264) and Eq. 2.19 (:268), as plain O(N * modes) sums.  Usable
  for N <~ 2000, modes <~ 16^3.  It is what pins everything else in this file.
* ``nufft_force`` and its stages ``es_spread`` / ``nufft_kspace`` / ``es_interp`` -- the
  algorithm of Sec. 2.5 (:258-262) step by step: spread with the exponential-of-semicircle
  kernel onto the sigma-upsampled grid, FFT, keep the modes below the particle Nyquist
  (:260, reading R8), divide by the kernel's Fourier transform once per transform (:262,
  reading R10), Poisson + i k gradient, zero-pad, inverse FFT, interpolate with the same kernel.

Readings: R8 symmetric mode set |n_a| < m/2; R10 kernel parameters
w = ceil(log10(1/eps)) + 1, beta = 2.30 w at sigma = 2 and 0.97 pi w (1 - 1/(2 sigma)) otherwise
(tunables validated against the brute force, PAPER.md gives none); R13 phi' = 0 at |z| >= 1.
Parity unpinned: VJP for particles within 1e-6 cells of the kernel's support edge (R13).
"""
from __future__ import annotations

import numpy as np


# ---------------------------------------------------------------------------------------
# Definition: Eq. 2.18 -> Poisson/gradient -> Eq. 2.19, brute force
# ---------------------------------------------------------------------------------------
def mode_set(m: int):
    """Integer wave vectors with |n_a| < m/2 (reading R8), shape [K, 3]."""
    r = np.arange(-(m // 2) + 1, (m + 1) // 2) if m % 2 == 0 else np.arange(-(m // 2), m // 2 + 1)
    return np.stack(np.meshgrid(r, r, r, indexing="ij"), axis=-1).reshape(-1, 3)


def nudft_density_bruteforce(pos, m: int, box: float):
    """delta_hat_n = sum_l exp(-2 pi i n.X_l / L), M_l = 1 (Eq. 2.18 :254); returns (modes, values)."""
    X = np.asarray(pos).astype(np.float64)
    n = mode_set(m)
    ph = (2.0 * np.pi / box) * (n.astype(np.float64) @ X.T)  # [K, N]
    return n, np.exp(-1j * ph).sum(axis=1)


def nudft_force_bruteforce(pos, m: int, box: float, coeff: float = 1.0):
    """g_i = (coeff/N) sum_{n != 0} (i k/|k|^2) delta_hat_n exp(i k.X_i), k = 2 pi n / L
    (Eq. 2.19 :268 applied to g_hat = -(i k) * coeff * delta_hat / (-k^2), :264)."""
    X = np.asarray(pos).astype(np.float64)
    npart = X.shape[0]
    n, dh = nudft_density_bruteforce(X, m, box)
    k = (2.0 * np.pi / box) * n.astype(np.float64)
    k2 = (k * k).sum(axis=1)
    nz = k2 > 0.0
    ghat = np.zeros((n.shape[0], 3), dtype=np.complex128)
    ghat[nz] = (1j * k[nz] / k2[nz, None]) * (coeff / npart) * dh[nz, None]
    ph = np.exp(1j * (k @ X.T))  # [K, N]
    return np.real(ph.T @ ghat)  # imaginary part cancels over +-n


# ---------------------------------------------------------------------------------------
# Exponential-of-semicircle kernel (:260, refs [82, 83]) and its parameters (reading R10)
# ---------------------------------------------------------------------------------------
def es_params(eps: float, sigma: float, width: int = 0):
    """(w, beta) from the tolerance, or from an explicit width (:260 'either ... or')."""
    w = int(width) if width else int(np.ceil(np.log10(1.0 / eps))) + 1
    if abs(sigma - 2.0) < 1e-12:
        beta = 2.30 * w
    else:
        beta = 0.97 * np.pi * w * (1.0 - 1.0 / (2.0 * sigma))
    return w, float(beta)


def es_kernel(z, beta: float):
    """phi(z) = exp(beta (sqrt(1 - z^2) - 1)) for |z| <= 1, else 0."""
    z = np.asarray(z, dtype=np.float64)
    inside = np.abs(z) <= 1.0
    s = np.sqrt(np.where(inside, 1.0 - z * z, 0.0))
    return np.where(inside, np.exp(beta * (s - 1.0)), 0.0)


def es_kernel_dz(z, beta: float):
    """phi'(z) = -beta z phi(z)/sqrt(1 - z^2), set to 0 for |z| >= 1 (reading R13)."""
    z = np.asarray(z, dtype=np.float64)
    inside = np.abs(z) < 1.0
    s = np.sqrt(np.where(inside, 1.0 - z * z, 1.0))
    return np.where(inside, -beta * z * np.exp(beta * (s - 1.0)) / s, 0.0)


def es_kernel_ft(n, m_fine: int, w: int, beta: float, nodes: int = 400):
    """phi_hat(n) = int_{-w/2}^{w/2} phi(2x/w) cos(2 pi n x / m_fine) dx by Gauss-Legendre."""
    xg, wg = np.polynomial.legendre.leggauss(nodes)
    x = 0.5 * w * xg
    f = es_kernel(xg, beta) * (0.5 * w) * wg
    n = np.asarray(n, dtype=np.float64)
    return (np.cos(2.0 * np.pi * n[..., None] * x / m_fine) * f).sum(axis=-1)


def es_nodes(u, w: int):
    """First node j0 = ceil(u - w/2) and offsets z = 2 (j - u)/w for the w nodes of one axis."""
    j0 = np.ceil(u - 0.5 * w).astype(np.int64)
    z = 2.0 * ((j0[:, None] + np.arange(w)[None, :]).astype(np.float64) - u[:, None]) / w
    return j0, z


# ---------------------------------------------------------------------------------------
# Stages
# ---------------------------------------------------------------------------------------
def es_spread(pos, m_fine: int, box: float, w: int, beta: float, weights=None, mesh=None):
    """fine_j += sum_i c_i prod_a phi(2 (j_a - u_a)/w), u = X/(box/m_fine)  (:258-260)."""
    X = np.asarray(pos).astype(np.float64)
    u = X / (box / m_fine)
    c = np.ones(X.shape[0]) if weights is None else np.asarray(weights).astype(np.float64)
    if mesh is None:
        mesh = np.zeros((m_fine,) * 3, dtype=np.float64)
    jx, zx = es_nodes(u[:, 0], w)
    jy, zy = es_nodes(u[:, 1], w)
    jz, zz = es_nodes(u[:, 2], w)
    px, py, pz = es_kernel(zx, beta), es_kernel(zy, beta), es_kernel(zz, beta)
    flat = mesh.reshape(-1)
    G = m_fine ** 3
    for a in range(w):
        ia = np.mod(jx + a, m_fine)
        for b in range(w):
            ib = np.mod(jy + b, m_fine)
            wab = c * px[:, a] * py[:, b]
            for d in range(w):
                ic = np.mod(jz + d, m_fine)
                flat += np.bincount((ia * m_fine + ib) * m_fine + ic, weights=wab * pz[:, d], minlength=G)
    return mesh


def es_interp(mesh, pos, box: float, w: int, beta: float, deriv_axis: int | None = None):
    """v_i = sum_j mesh_j prod_a phi(2 (j_a - u_a)/w)  (Eq. 2.19 evaluated through the grid).
    deriv_axis = a: derivative w.r.t. X_i^a (length units)."""
    mesh = np.asarray(mesh, dtype=np.float64)
    m_fine = mesh.shape[0]
    X = np.asarray(pos).astype(np.float64)
    u = X / (box / m_fine)
    js, ps = [], []
    for a in range(3):
        j0, z = es_nodes(u[:, a], w)
        js.append(j0)
        if deriv_axis == a:  # d/du phi(2 (j-u)/w) = -(2/w) phi'(z)
            ps.append(-(2.0 / w) * es_kernel_dz(z, beta))
        else:
            ps.append(es_kernel(z, beta))
    out = np.zeros(X.shape[0])
    for a in range(w):
        ia = np.mod(js[0] + a, m_fine)
        for b in range(w):
            ib = np.mod(js[1] + b, m_fine)
            wab = ps[0][:, a] * ps[1][:, b]
            for d in range(w):
                ic = np.mod(js[2] + d, m_fine)
                out += mesh[ia, ib, ic] * wab * ps[2][:, d]
    if deriv_axis is not None:
        out *= m_fine / box
    return out


def _kspace_multiplier(m_fine: int, m: int, box: float, n_particles: int, w: int, beta: float,
                       coeff: float):
    """M_a(n) on the fine half-complex grid: (i k_a/|k|^2) (coeff/N) / phi_hat(n)^2 for
    0 < |n|, |n_a| < m/2 (reading R8), zero elsewhere.  phi_hat enters squared: once for the
    type-1 and once for the type-2 transform (:262)."""
    h = m_fine // 2 + 1
    nf = np.fft.fftfreq(m_fine, 1.0 / m_fine)
    keep = np.abs(nf) < 0.5 * m
    ph1 = es_kernel_ft(nf, m_fine, w, beta)
    k1 = (2.0 * np.pi / box) * nf
    kx, ky, kz = k1[:, None, None], k1[None, :, None], k1[None, None, :h]
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    mask = keep[:, None, None] & keep[None, :, None] & keep[None, None, :h]
    phat = ph1[:, None, None] * ph1[None, :, None] * ph1[None, None, :h]
    base = np.where(mask, (coeff / n_particles) / (k2 * phat * phat), 0.0)
    base[0, 0, 0] = 0.0
    return [1j * ka * base for ka in (kx, ky, kz)]


def kspace_multiplier_at(idx, m_fine: int, m: int, box: float, n_particles: int, w: int, beta: float,
                         coeff: float):
    """M_a(n) of :func:`_kspace_multiplier` for single modes idx = (ix, iy, iz) (FFT indices on the fine
    grid, arrays allowed); complex [3, ...].  For fine grids too large for the 3-D arrays; pinned against
    _kspace_multiplier element by element."""
    ix, iy, iz = (np.asarray(v, dtype=np.int64) for v in idx)
    nf = np.fft.fftfreq(m_fine, 1.0 / m_fine)
    keep = np.abs(nf) < 0.5 * m
    ph1 = es_kernel_ft(nf, m_fine, w, beta)
    k1 = (2.0 * np.pi / box) * nf
    k2 = k1[ix] ** 2 + k1[iy] ** 2 + k1[iz] ** 2
    ok = keep[ix] & keep[iy] & keep[iz] & (k2 > 0.0)
    phat = ph1[ix] * ph1[iy] * ph1[iz]
    base = np.where(ok, (coeff / n_particles) / (np.where(ok, k2, 1.0) * phat * phat), 0.0)
    return np.stack([1j * k1[i] * base for i in (ix, iy, iz)])


def nufft_kspace(fine, m: int, box: float, n_particles: int, w: int, beta: float, coeff: float = 1.0):
    """Spread grid -> three fine force grids ready for ``es_interp`` (:260-264)."""
    fine = np.asarray(fine, dtype=np.float64)
    m_fine = fine.shape[0]
    F = np.fft.rfftn(fine)
    M = _kspace_multiplier(m_fine, m, box, n_particles, w, beta, coeff)
    return [np.fft.irfftn(Ma * F, s=(m_fine,) * 3, axes=(0, 1, 2)) * float(m_fine) ** 3 for Ma in M]


def nufft_kspace_potential(fine, m: int, box: float, n_particles: int, w: int, beta: float, coeff: float = 1.0):
    """Spread grid -> fine POTENTIAL grid phi, ready for interpolation with the ES kernel or its gradient:
    phi_hat = coeff * delta_hat / (-k^2) (Eq. 2.2 :84) on the retained modes, divided by phi_ES_hat twice
    (:262).  The force of the 'kernel gradient' option (:264) is -grad of its interpolant."""
    fine = np.asarray(fine, dtype=np.float64)
    m_fine = fine.shape[0]
    h = m_fine // 2 + 1
    nf = np.fft.fftfreq(m_fine, 1.0 / m_fine)
    keep = np.abs(nf) < 0.5 * m
    ph1 = es_kernel_ft(nf, m_fine, w, beta)
    k1 = (2.0 * np.pi / box) * nf
    k2 = (k1 * k1)[:, None, None] + (k1 * k1)[None, :, None] + (k1 * k1)[None, None, :h]
    k2[0, 0, 0] = 1.0
    mask = keep[:, None, None] & keep[None, :, None] & keep[None, None, :h]
    phat = ph1[:, None, None] * ph1[None, :, None] * ph1[None, None, :h]
    P = np.where(mask, -(coeff / n_particles) / (k2 * phat * phat), 0.0)
    P[0, 0, 0] = 0.0
    return np.fft.irfftn(P * np.fft.rfftn(fine), s=(m_fine,) * 3, axes=(0, 1, 2)) * float(m_fine) ** 3


def nufft_kspace_vjp(fine_cot, m: int, box: float, n_particles: int, w: int, beta: float, coeff: float = 1.0):
    """Transpose of ``nufft_kspace``: sum_a F^H conj(M_a) F fine_cot_a."""
    m_fine = np.asarray(fine_cot[0]).shape[0]
    M = _kspace_multiplier(m_fine, m, box, n_particles, w, beta, coeff)
    q = sum(np.conj(Ma) * np.fft.rfftn(np.asarray(g, dtype=np.float64)) for Ma, g in zip(M, fine_cot))
    return np.fft.irfftn(q, s=(m_fine,) * 3, axes=(0, 1, 2)) * float(m_fine) ** 3


def nufft_force(pos, m: int, box: float, sigma: float = 2.0, eps: float = 1e-6, width: int = 0,
                coeff: float = 1.0, beta: float | None = None, kernel_grad: bool = False):
    """Per-particle acceleration [N, 3] through the ES-kernel NUFFT (Sec. 2.5).  kernel_grad: the
    gradient is taken of the interpolation kernel ("similarly to ... smoothed-particle hydrodynamics",
    :264) instead of multiplying by i k: g_i = -grad_X sum_j phi_j prod_a phi_ES(2 (j_a - u_a)/w)."""
    w, b = es_params(eps, sigma, width)
    if beta is not None:
        b = beta
    m_fine = int(round(sigma * m))
    n = np.asarray(pos).shape[0]
    fine = es_spread(pos, m_fine, box, w, b)
    if kernel_grad:
        phi = nufft_kspace_potential(fine, m, box, n, w, b, coeff)
        return np.stack([-es_interp(phi, pos, box, w, b, deriv_axis=a) for a in range(3)], axis=1)
    g = nufft_kspace(fine, m, box, n, w, b, coeff)
    return np.stack([es_interp(g[a], pos, box, w, b) for a in range(3)], axis=1)


def nufft_force_vjp(pos, lam, m: int, box: float, sigma: float = 2.0, eps: float = 1e-6,
                    width: int = 0, coeff: float = 1.0):
    """X_bar = lam^T dg/dX for ``nufft_force`` (App. C rules hold for any compact
    differentiable W, :858)."""
    w, b = es_params(eps, sigma, width)
    m_fine = int(round(sigma * m))
    lam = np.asarray(lam).astype(np.float64)
    n = np.asarray(pos).shape[0]
    fine = es_spread(pos, m_fine, box, w, b)
    g = nufft_kspace(fine, m, box, n, w, b, coeff)
    xbar = np.zeros((n, 3))
    for a in range(3):
        for c in range(3):
            xbar[:, c] += lam[:, a] * es_interp(g[a], pos, box, w, b, deriv_axis=c)
    gbar = [es_spread(pos, m_fine, box, w, b, weights=lam[:, a]) for a in range(3)]
    fbar = nufft_kspace_vjp(gbar, m, box, n, w, b, coeff)
    for c in range(3):
        xbar[:, c] += es_interp(fbar, pos, box, w, b, deriv_axis=c)
    return xbar
