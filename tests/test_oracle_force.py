"""Pins of the oracle's full force and VJP: invariants north_star names (no GPU)."""
import numpy as np
import pytest

from oracle import pm_oracle as po
from pm_inputs import lattice_displaced, uniform_random
from pm_inputs.generators import uniform_lattice


@pytest.mark.parametrize("worder", (2, 3, 4))
@pytest.mark.parametrize("ratio", (1, 2))
@pytest.mark.parametrize("grad_order,deconv", ((0, 2), (4, 0)))
def test_zero_force_on_uniform_lattice(worder, ratio, grad_order, deconv):
    """R7 / Eq. 2.3: a uniform lattice has delta = const => zero force (m = n_p and 2 n_p)."""
    n_p, box = 8, 16.0  # lattice + offset exactly representable in fp32
    pos = uniform_lattice(n_p, box, offset=0.25)
    F = po.force(pos, ratio * n_p, box, worder=worder, grad_order=grad_order, deconv_pow=deconv)
    assert np.abs(F).max() < 1e-12


@pytest.mark.parametrize("worder", (2, 3, 4))
@pytest.mark.parametrize("interlace", (0, 2))
def test_momentum_conservation(worder, interlace):
    """Same W for assign and gather + odd gradient symbol => sum_i F_i = 0 (interlace 0, 2; R1)."""
    m, box = 16, 50.0
    pos = uniform_random(2000, box, 21)
    F = po.force(pos, m, box, worder=worder, interlace=interlace, grad_order=4, deconv_pow=2)
    assert np.abs(F.sum(0)).max() < 1e-12 * np.abs(F).sum()


@pytest.mark.parametrize("worder,tol", ((2, 0.08), (3, 0.03), (4, 0.01)))
def test_plane_wave_sheet_force(worder, tol):
    """Pre-shell-crossing plane wave X = q + Psi(q) x^, Psi = (A/k0) sin(k0 q_x): the 1-D sheet
    model gives g = coeff * Psi (Eq. 2.1-2.2); PM reproduces it up to its window errors."""
    n_p, box, A, coeff = 32, 64.0, 0.3, 1.7
    k0 = 2 * np.pi / box
    q = uniform_lattice(n_p, box).astype(np.float64)
    psi = (A / k0) * np.sin(k0 * q[:, 0])
    pos = q.copy()
    pos[:, 0] = np.mod(q[:, 0] + psi, box)
    F = po.force(pos.astype(np.float32), n_p, box, worder=worder, grad_order=0, deconv_pow=2, coeff=coeff)
    assert np.abs(F[:, 1:]).max() < 1e-9 * np.abs(F[:, 0]).max()  # transverse components vanish
    err = np.linalg.norm(F[:, 0] - coeff * psi) / np.linalg.norm(coeff * psi)
    assert err < tol, err
    # sign and scale: correlation with +coeff*Psi must be ~1 (a flipped sign gives -1)
    assert np.dot(F[:, 0], psi) / (coeff * np.dot(psi, psi)) > 0.9


def test_force_scales_linearly_with_coeff():
    pos = uniform_random(500, 10.0, 3)
    F1 = po.force(pos, 8, 10.0, coeff=1.0)
    F3 = po.force(pos, 8, 10.0, coeff=3.0)
    assert np.abs(F3 - 3 * F1).max() < 1e-13 * np.abs(F3).max()


def test_interlace_mode1_translation_covariance():
    """R1/R9: C(X) = 1/2 [A(X) + P A(X - s)] obeys C(X + s) = P C(X) off the Nyquist planes."""
    m, box, wo = 12, 24.0, 3
    s = np.full(3, 0.5 * box / m)
    pos = uniform_random(700, box, 31).astype(np.float64)
    P = po.interlace_phase_3d(m)

    def comb(x):
        a = np.fft.rfftn(po.scatter(x, m, box, wo))
        b = np.fft.rfftn(po.scatter(x, m, box, wo, shift=s))
        return 0.5 * (a + P * b)

    lhs, rhs = comb(np.mod(pos + s, box)), P * comb(pos)
    n = po.mode_numbers(m)
    ok = (np.abs(n)[:, None, None] < m // 2) & (np.abs(n)[None, :, None] < m // 2) & \
         (np.abs(n[: m // 2 + 1])[None, None, :] < m // 2)
    assert np.abs(lhs - rhs)[ok].max() < 1e-11
    # and the combined field is real after a COMPLEX inverse transform (Hermitian phase, R9)
    p1 = po.interlace_phase(m)
    Pfull = p1[:, None, None] * p1[None, :, None] * p1[None, None, :]
    cube = 0.5 * (np.fft.fftn(po.scatter(pos, m, box, wo)) + Pfull * np.fft.fftn(po.scatter(pos, m, box, wo, shift=s)))
    back = np.fft.ifftn(cube)
    assert np.abs(back.imag).max() < 1e-13 * np.abs(back.real).max()
    # without R9 (raw e^{-i pi n/m} on the Nyquist index) it is not
    raw = np.exp(-1j * np.pi * po.mode_numbers(m) / m)
    Praw = raw[:, None, None] * raw[None, :, None] * raw[None, None, :]
    bad = np.fft.ifftn(0.5 * (np.fft.fftn(po.scatter(pos, m, box, wo)) + Praw * np.fft.fftn(po.scatter(pos, m, box, wo, shift=s))))
    assert np.abs(bad.imag).max() > 1e-6 * np.abs(bad.real).max()


def test_interlace_cancels_odd_alias_images():
    """Two-grid interlacing removes the odd alias images (:367, ref. [95]): for particles that
    sample a single mode n0 with n0 + m a (|a| odd) aliasing onto n1, the interlaced density at
    n1 is far smaller than the single-grid one."""
    m, box = 8, 8.0
    rng = np.random.default_rng(5)
    pos = (rng.random((4000, 3)) * box).astype(np.float32)
    d1 = po.density_contrast(po.scatter(pos, m, box, 2), 4000)
    d2 = po.density_contrast(po.scatter(pos, m, box, 2, shift=np.full(3, 0.5)), 4000)
    single = np.fft.rfftn(d1)
    inter = 0.5 * (single + po.interlace_phase_3d(m) * np.fft.rfftn(d2))
    # shot noise power at high k is dominated by aliases; interlacing must lower it
    hi = np.zeros(single.shape, bool)
    hi[3, 3, 3] = hi[3, 2, 3] = hi[2, 3, 3] = True
    assert (np.abs(inter[hi]) ** 2).sum() < 0.8 * (np.abs(single[hi]) ** 2).sum()


@pytest.mark.parametrize("worder,interlace,grad_order,deconv", (
    (3, 0, 4, 2), (4, 0, 0, 2), (3, 1, 4, 2), (3, 2, 0, 0), (4, 1, 6, 1)))
def test_force_vjp_vs_finite_differences(worder, interlace, grad_order, deconv):
    """App. C rule table (:949-955) composed as step V, against central differences of
    sum lam.F(X) -- the paper's own validation method (:435)."""
    m, box = 8, 16.0
    rng = np.random.default_rng(77)
    pos = (rng.random((60, 3)) * box)
    lam = rng.standard_normal((60, 3))
    kw = dict(worder=worder, interlace=interlace, grad_order=grad_order, deconv_pow=deconv, coeff=1.3)
    xbar = po.force_vjp(pos, lam, m, box, **kw)
    h = 1e-5
    for (i, a) in ((0, 0), (7, 1), (13, 2), (59, 0), (31, 2)):
        e = np.zeros_like(pos)
        e[i, a] = h
        fd = ((po.force(pos + e, m, box, **kw) * lam).sum() - (po.force(pos - e, m, box, **kw) * lam).sum()) / (2 * h)
        assert abs(fd - xbar[i, a]) < 2e-7 * max(1.0, np.abs(xbar).max()), (i, a, fd, xbar[i, a])


def test_poisson_force_vjp_is_transpose():
    """<g, A d> = <A^T g, d> for the k-space operator, single and interlaced."""
    m, box = 8, 8.0
    rng = np.random.default_rng(4)
    d1, d2 = rng.standard_normal((2, m, m, m))
    gb = rng.standard_normal((3, m, m, m))
    kw = dict(box=box, worder=3, grad_order=4, lap_order=2, deconv_pow=2, coeff=0.9)
    g = po.poisson_force(d1, **kw)
    lhs = sum((g[a] * gb[a]).sum() for a in range(3))
    assert abs(lhs - (po.poisson_force_vjp(gb, **kw) * d1).sum()) < 1e-11 * abs(lhs)
    g = po.poisson_force(d1, delta_mesh2=d2, **kw)
    lhs = sum((g[a] * gb[a]).sum() for a in range(3))
    c1, c2 = po.poisson_force_vjp(gb, interlace=True, **kw)
    assert abs(lhs - (c1 * d1).sum() - (c2 * d2).sum()) < 1e-11 * abs(lhs)
