"""Pins of oracle/analysis_oracle.py (power spectrum, sheet resampling) against closed forms (no GPU)."""
import numpy as np
import pytest

from oracle import analysis_oracle as ao
from oracle import pm_oracle as po
from pm_inputs import uniform_random
from pm_inputs.generators import uniform_lattice


def test_power_spectrum_parseval():
    """sum over ALL modes of |delta_hat|^2 = G sum_j delta_j^2: pins the mode multiplicities of the stored half
    and the V / G^2 normalisation."""
    m, box = 12, 30.0
    pos = uniform_random(900, box, 71)
    d = po.density_contrast(po.scatter(pos, m, box, 3), 900)
    k, P, cnt = ao.power_spectrum(pos, m, box, nbins=12, worder=3, deconvolve=False)
    G = m ** 3
    assert cnt.sum() == G - 1  # every mode but n = 0 (|n| <= sqrt(3) m/2 < 12.5)
    assert abs((P * cnt).sum() * G ** 2 / box ** 3 - G * np.sum(d * d)) < 1e-9 * G * np.sum(d * d)
    n1 = po.mode_numbers(m)
    kn = np.sqrt(n1[:, None, None] ** 2 + n1[None, :, None] ** 2 + n1[None, None, :] ** 2)
    for b in (0, 3, 7):  # bin b holds b + 1/2 <= |n| < b + 3/2, full cube
        sel = (kn >= b + 0.5) & (kn < b + 1.5)
        assert cnt[b] == sel.sum()
        assert abs(k[b] - (2 * np.pi / box) * kn[sel].mean()) < 1e-12


@pytest.mark.parametrize("interlace", (0, 1))
def test_power_spectrum_of_a_plane_wave(interlace):
    """X = q + (eps A / k0) sin(k0 q_x): delta = -eps A cos(k0 x) + O(eps^2), so the bin of |n0| holds
    P = V (eps A)^2 / (2 n_modes) and every other bin is ~0; a copy translated by d along x has the cross
    spectrum P cos(k0 d) (translation by whole cells is exact)."""
    n_p, box, n0, epsA = 16, 32.0, 2, 1e-3
    k0 = 2 * np.pi * n0 / box
    q = uniform_lattice(n_p, box).astype(np.float64)
    pos = q.copy()
    pos[:, 0] = np.mod(q[:, 0] + (epsA / k0) * np.sin(k0 * q[:, 0]), box)
    k, P, cnt = ao.power_spectrum(pos, n_p, box, nbins=8, worder=4, interlace=interlace)
    b = n0 - 1
    expect = box ** 3 * epsA ** 2 / (2 * cnt[b])
    assert abs(P[b] - expect) < 1e-2 * expect
    others = np.delete(P, b)
    assert np.abs(others).max() < 1e-4 * expect
    d = 3 * box / n_p
    pos2 = pos.copy()
    pos2[:, 0] = np.mod(pos2[:, 0] + d, box)
    _, Pc, _ = ao.power_spectrum(pos, n_p, box, nbins=8, worder=4, interlace=interlace, pos2=pos2)
    assert abs(Pc[b] - P[b] * np.cos(k0 * d)) < 1e-6 * abs(P[b])
    _, Pa, _ = ao.power_spectrum(pos, n_p, box, nbins=8, worder=4, interlace=interlace, pos2=pos)
    assert np.array_equal(Pa, P)


def test_power_spectrum_shot_noise():
    """Uniform random points: <P(k)> = V / N at every k (Poisson noise), seen after deconvolution + interlacing."""
    m, box, n = 16, 40.0, 20000
    pos = uniform_random(n, box, 72)
    k, P, cnt = ao.power_spectrum(pos, m, box, nbins=6, worder=3, interlace=1)
    sel = cnt > 200
    assert sel.sum() >= 3
    assert np.abs(P[sel] / (box ** 3 / n) - 1.0).max() < 0.15


def test_deconvolution_is_by_one_power_of_the_window():
    m, box = 8, 8.0
    pos = uniform_random(300, box, 73)
    a = ao.density_modes(pos, m, box, worder=3, deconvolve=False)
    b = ao.density_modes(pos, m, box, worder=3, deconvolve=True)
    W1 = po.window_1d(m, 3)
    assert np.allclose(a[1, 2, 3], b[1, 2, 3] * W1[1] * W1[2] * W1[3], rtol=1e-13)


# ---------------------------------------------------------------- sheet resampling
def test_resample_identity_and_lattice():
    n_p, box = 8, 16.0  # spacings exactly representable in fp32
    pos = uniform_random(n_p ** 3, box, 74)
    assert np.abs(ao.sheet_resample(pos, n_p, box, 1) - pos.astype(np.float64)).max() < 1e-12
    lat = uniform_lattice(n_p, box)
    fine = ao.sheet_resample(lat, n_p, box, 4)
    assert np.abs(fine - uniform_lattice(4 * n_p, box).astype(np.float64)).max() < 1e-12


def test_resample_is_trilinear_in_the_displacement():
    """Copies sit on the trilinear interpolant of Psi between the 8 Lagrangian neighbours (:371): checked on the
    cell of particle (1, 2, 3) by hand, on a displaced lattice that crosses the periodic boundary."""
    n_p, box, r = 4, 8.0, 2
    rng = np.random.default_rng(75)
    q = uniform_lattice(n_p, box).astype(np.float64).reshape(n_p, n_p, n_p, 3)
    psi = rng.standard_normal((n_p, n_p, n_p, 3)) * 0.9
    pos = np.mod(q + psi, box).reshape(-1, 3)
    out = ao.sheet_resample(pos, n_p, box, r).reshape(r * n_p, r * n_p, r * n_p, 3)
    i, j, k = 1, 2, 3  # k + 1 wraps to 0
    want = np.zeros(3)
    for dx in (0, 1):
        for dy in (0, 1):
            for dz in (0, 1):
                want += 0.125 * psi[(i + dx) % n_p, (j + dy) % n_p, (k + dz) % n_p]
    want += (np.array([2 * i + 1, 2 * j + 1, 2 * k + 1]) * box / (r * n_p))
    got = out[2 * i + 1, 2 * j + 1, 2 * k + 1]
    d = np.abs(got - np.mod(want, box))
    assert np.minimum(d, box - d).max() < 1e-12
    # the original particles are among the copies (t = 0)
    assert np.abs(out[::r, ::r, ::r].reshape(-1, 3) - pos).max() < 1e-12
    # a displacement field that is linear inside a cell is reproduced exactly: Psi = eps sin(k q_x) sampled
    # at r = 1 vs the same plane wave: second-order accurate, error ~ (k h)^2 / 8
    n_p = 16
    q = uniform_lattice(n_p, box).astype(np.float64)
    k0 = 2 * np.pi / box
    pos = q.copy()
    pos[:, 0] = q[:, 0] + 0.1 * np.sin(k0 * q[:, 0])
    fine = ao.sheet_resample(pos, n_p, box, 4)
    qf = uniform_lattice(4 * n_p, box).astype(np.float64)
    err = np.abs(fine[:, 0] - np.mod(qf[:, 0] + 0.1 * np.sin(k0 * qf[:, 0]), box))
    err = np.minimum(err, box - err)
    assert err.max() < 0.1 * (k0 * box / n_p) ** 2 / 8 * 1.05
