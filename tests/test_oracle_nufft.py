"""Pins of the NUFFT oracle: the brute-force definition (Eq. 2.18-2.19) against closed forms, and
the ES-kernel algorithm against the brute force (no GPU)."""
import numpy as np
import pytest

from oracle import nufft_oracle as no
from pm_inputs import uniform_random
from pm_inputs.generators import uniform_lattice


def test_nudft_on_lattice_is_the_standard_dft():
    """:256 'for uniformly spaced particles on a grid, [Eq. 2.18] reduces to the standard forward
    DFT': with weights = a field sampled on the lattice the sums equal numpy's FFT of that field."""
    n_p, box = 6, 12.0
    pos = uniform_lattice(n_p, box).astype(np.float64)
    f = np.random.default_rng(0).standard_normal((n_p, n_p, n_p))
    n = no.mode_set(n_p)  # |n_a| < n_p/2
    ph = (2 * np.pi / box) * (n.astype(float) @ pos.T)
    direct = (np.exp(-1j * ph) * f.reshape(-1)[None, :]).sum(1)
    F = np.fft.fftn(f)
    assert np.abs(direct - F[n[:, 0] % n_p, n[:, 1] % n_p, n[:, 2] % n_p]).max() < 1e-11
    # unit masses: only n = 0 (mod n_p) survives => no force on the lattice
    assert np.abs(no.nudft_force_bruteforce(pos, n_p, box)).max() < 1e-12


def test_bruteforce_two_particles_closed_form():
    """Two particles separated along x by d: g on particle 0 is
    -(coeff/N) sum_n (k_x/k^2) sin(k_x d) summed over the kept modes (pairwise antisymmetric)."""
    m, box, coeff, d = 8, 10.0, 1.3, 1.7
    pos = np.array([[2.0, 3.0, 4.0], [2.0 + d, 3.0, 4.0]])
    g = no.nudft_force_bruteforce(pos, m, box, coeff)
    n = no.mode_set(m).astype(float)
    k = 2 * np.pi / box * n
    k2 = (k * k).sum(1)
    ok = k2 > 0
    # force on particle 0 from particle 1: X_0 - X_1 = -d x^
    expect = (coeff / 2) * (-(k[ok, 0] / k2[ok]) * np.sin(k[ok, 0] * (-d))).sum()
    assert abs(g[0, 0] - expect) < 1e-13 * abs(expect)
    assert np.abs(g[0] + g[1]).max() < 1e-14 * abs(expect) and np.abs(g[:, 1:]).max() < 1e-14 * abs(expect)
    assert g[0, 0] > 0  # attraction towards the neighbour at +x (coeff > 0)


def test_bruteforce_plane_wave_sheet_force():
    """Same sheet-model pin as the PM oracle, without assignment-window error: g = coeff Psi."""
    n_p, box, A, coeff = 12, 24.0, 0.2, 0.8
    k0 = 2 * np.pi / box
    q = uniform_lattice(n_p, box).astype(np.float64)
    psi = (A / k0) * np.sin(k0 * q[:, 0])
    pos = q.copy()
    pos[:, 0] = np.mod(q[:, 0] + psi, box)
    g = no.nudft_force_bruteforce(pos, n_p, box, coeff)
    assert np.linalg.norm(g[:, 0] - coeff * psi) / np.linalg.norm(coeff * psi) < 0.02
    assert np.abs(g[:, 1:]).max() < 1e-12


def test_momentum_conservation_bruteforce():
    pos = uniform_random(150, 9.0, 2)
    g = no.nudft_force_bruteforce(pos, 8, 9.0)
    assert np.abs(g.sum(0)).max() < 1e-13 * np.abs(g).sum()


def test_es_kernel_ft_quadrature():
    """phi_hat by Gauss-Legendre equals a fine trapezoid rule of the same integral."""
    w, beta, mf = 7, 16.1, 32
    x = np.linspace(-w / 2, w / 2, 2_000_001)
    phi = no.es_kernel(2 * x / w, beta)
    for n in (0, 1, 5, 8):
        ref = np.trapezoid(phi * np.cos(2 * np.pi * n * x / mf), x)
        assert abs(no.es_kernel_ft(np.array([n]), mf, w, beta)[0] - ref) < 1e-8 * abs(ref) + 1e-10
    # derivative of the kernel against a difference quotient
    z = np.linspace(-0.95, 0.95, 101)
    fd = (no.es_kernel(z + 1e-6, beta) - no.es_kernel(z - 1e-6, beta)) / 2e-6
    assert np.abs(fd - no.es_kernel_dz(z, beta)).max() < 1e-6


def test_es_params_rule():
    assert no.es_params(1e-6, 2.0) == (7, pytest.approx(16.1))
    assert no.es_params(1e-6, 2.0, width=13)[0] == 13
    w, b = no.es_params(1e-4, 1.25)
    assert w == 5 and b == pytest.approx(0.97 * np.pi * 5 * 0.6)


@pytest.mark.parametrize("sigma,width,tol", ((2.0, 7, 1e-5), (2.0, 13, 1e-10), (2.0, 6, 1e-4), (1.25, 10, 1e-5)))
def test_nufft_vs_bruteforce(sigma, width, tol):
    """ES-kernel NUFFT within 10*eps of the exact sums (north_star tolerance), w from eps=1e-6 -> 7."""
    m, box = 8, 10.0
    pos = uniform_random(300, box, 17)
    gb = no.nudft_force_bruteforce(pos, m, box, coeff=1.4)
    g = no.nufft_force(pos, m, box, sigma=sigma, width=width, coeff=1.4)
    assert np.linalg.norm(g - gb) / np.linalg.norm(gb) < tol


def test_spread_interp_adjoint_and_mass():
    mf, box, w, beta = 16, 10.0, 7, 16.1
    pos = uniform_random(200, box, 4)
    rng = np.random.default_rng(1)
    c, mesh = rng.standard_normal(200), rng.standard_normal((mf, mf, mf))
    lhs = (no.es_spread(pos, mf, box, w, beta, weights=c) * mesh).sum()
    assert abs(lhs - (c * no.es_interp(mesh, pos, box, w, beta)).sum()) < 1e-12 * abs(lhs)


def test_nufft_force_vjp_vs_finite_differences():
    m, box = 6, 9.0
    rng = np.random.default_rng(3)
    pos = rng.random((40, 3)) * box
    lam = rng.standard_normal((40, 3))
    kw = dict(sigma=2.0, width=9, coeff=1.1)
    xbar = no.nufft_force_vjp(pos, lam, m, box, **kw)
    h = 1e-5
    for (i, a) in ((0, 0), (11, 1), (39, 2)):
        e = np.zeros_like(pos)
        e[i, a] = h
        fd = ((no.nufft_force(pos + e, m, box, **kw) * lam).sum() - (no.nufft_force(pos - e, m, box, **kw) * lam).sum()) / (2 * h)
        assert abs(fd - xbar[i, a]) < 1e-6 * max(1.0, np.abs(xbar).max()), (fd, xbar[i, a])


def test_nufft_kspace_vjp_is_transpose():
    m, mf, box = 6, 12, 9.0
    rng = np.random.default_rng(9)
    f = rng.standard_normal((mf, mf, mf))
    gb = rng.standard_normal((3, mf, mf, mf))
    g = no.nufft_kspace(f, m, box, 100, 7, 16.1)
    lhs = sum((g[a] * gb[a]).sum() for a in range(3))
    assert abs(lhs - (no.nufft_kspace_vjp(gb, m, box, 100, 7, 16.1) * f).sum()) < 1e-11 * abs(lhs)


@pytest.mark.parametrize("sigma,width,tol", ((2.0, 7, 1e-5), (2.0, 8, 1e-6), (2.0, 5, 1e-3), (2.0, 13, 1e-9)))
def test_kernel_gradient_force_vs_bruteforce(sigma, width, tol):
    """The 'SPH-like' gradient option (:264: "the gradient of the exponential-of-semicircle kernel ... we found
    little difference between the two"): -grad of the ES interpolant of the potential, against the exact
    sums of Eq. 2.18-2.19 -- same 10*eps bar as the i k gradient (its error is ~7x larger at sigma = 2)."""
    m, box = 8, 10.0
    pos = uniform_random(300, box, 17)
    gb = no.nudft_force_bruteforce(pos, m, box, coeff=1.4)
    g = no.nufft_force(pos, m, box, sigma=sigma, width=width, coeff=1.4, kernel_grad=True)
    assert np.linalg.norm(g - gb) / np.linalg.norm(gb) < tol
    # the potential grid differentiated spectrally IS the i k force grid: -i k phi_hat = M_a delta_hat
    w, b = no.es_params(1e-6, sigma, width)
    mf = int(round(sigma * m))
    fine = no.es_spread(pos, mf, box, w, b)
    phi = no.nufft_kspace_potential(fine, m, box, 300, w, b, coeff=1.4)
    gx = no.nufft_kspace(fine, m, box, 300, w, b, coeff=1.4)[0]
    k = (2 * np.pi / box) * np.fft.fftfreq(mf, 1.0 / mf)
    k[np.abs(np.fft.fftfreq(mf, 1.0 / mf)) >= 0.5 * m] = 0.0
    spec = np.fft.ifft(-1j * k[:, None, None] * np.fft.fft(phi, axis=0), axis=0).real
    assert np.abs(spec - gx).max() < 1e-10 * np.abs(gx).max()


def test_kspace_multiplier_at_matches_the_arrays():
    mf, m, box, n, w, beta = 16, 8, 10.0, 300, 7, 16.1
    M = no._kspace_multiplier(mf, m, box, n, w, beta, 1.4)
    rng = np.random.default_rng(80)
    idx = (rng.integers(0, mf, 300), rng.integers(0, mf, 300), rng.integers(0, mf // 2 + 1, 300))
    idx[0][:2] = idx[1][:2] = idx[2][:2] = 0
    Ma = no.kspace_multiplier_at(idx, mf, m, box, n, w, beta, 1.4)
    for a in range(3):
        assert np.allclose(M[a][idx], Ma[a], rtol=1e-14, atol=0)
