"""Oracle of the two NEXT-4 rows (TEST INFRASTRUCTURE): the binned (cross-)power spectrum of the interlaced,
deconvolved PM density ("(cross-)power spectrum routine") and the sheet-based particle
resampling by trilinear interpolation of the displacement field in Lagrangian space (:369-371, Table 5
``n_resample`` :411).  The paper gives neither algorithm in detail; the readings are listed in DESIGN.md
(R20, R21) and restated in the docstrings.  Built on pm_oracle's scatter / symbols; NumPy fp64.

Pins (tests/test_oracle_analysis.py): Parseval; a single plane-wave density lands in one bin with the
closed-form amplitude; shot noise V/N of uniform random points; cross spectrum of a set with itself = auto
spectrum, with a translated copy = auto spectrum times cos(k.d) on a single mode; resampling: r = 1 is the
identity, an undisplaced lattice gives the finer lattice, a linear-in-cell displacement is reproduced
exactly, copies sit on the trilinear interpolant between their 8 Lagrangian neighbours.
"""
from __future__ import annotations

import numpy as np

from . import pm_oracle as po


def density_modes(pos, m, box, worder=2, interlace=0, deconvolve=True):
    """delta_hat(n) on the half-complex grid: assignment (Eq. C.1), density contrast (Eq. 2.3), forward FFT,
    optional two-grid interlacing 1/2 [d1 + e^{-ik.s} d2] (R1, R9) and division by the assignment window
    W~(n) ONCE (R20: one assignment and no gather, unlike the force's W~^2, :262)."""
    n = np.asarray(pos).shape[0]
    d = po.density_contrast(po.scatter(pos, m, box, worder), n)
    dh = np.fft.rfftn(d)
    if interlace:
        s = np.full(3, 0.5 * box / m)
        d2 = po.density_contrast(po.scatter(pos, m, box, worder, shift=s), n)
        dh = 0.5 * (dh + po.interlace_phase_3d(m) * np.fft.rfftn(d2))
    if deconvolve:
        W1 = po.window_1d(m, worder)
        h = m // 2 + 1
        dh = dh / (W1[:, None, None] * W1[None, :, None] * W1[None, None, :h])
    return dh


def power_spectrum(pos, m, box, nbins, worder=2, interlace=0, deconvolve=True, pos2=None):
    """Shell-averaged P(k) (R20).  Bin b = 0..nbins-1 holds the modes with b + 1/2 <= |n| < b + 3/2 (integer
    wave vector n, k = 2 pi n / L; the n = 0 mode belongs to no bin); every mode of the FULL Fourier cube counts
    once (the stored half counts twice off the n_z = 0 and n_z = m/2 planes).
    Returns (k_mean [nbins], P [nbins], n_modes [nbins]); P = V <Re(d1_hat conj d2_hat)> / G^2, V = L^3,
    G = m^3, no shot-noise subtraction; empty bins give 0."""
    dh1 = density_modes(pos, m, box, worder, interlace, deconvolve)
    dh2 = dh1 if pos2 is None else density_modes(pos2, m, box, worder, interlace, deconvolve)
    h = m // 2 + 1
    n1 = po.mode_numbers(m)
    nz = n1[:h].copy()
    nz[-1] = abs(nz[-1]) if m % 2 == 0 else nz[-1]
    kn = np.sqrt(n1[:, None, None] ** 2 + n1[None, :, None] ** 2 + nz[None, None, :] ** 2)
    mult = np.full(h, 2.0)
    mult[0] = 1.0
    if m % 2 == 0:
        mult[-1] = 1.0
    wgt = np.broadcast_to(mult[None, None, :], kn.shape)
    b = np.floor(kn - 0.5).astype(np.int64)
    ok = (b >= 0) & (b < nbins)
    pw = (dh1 * np.conj(dh2)).real
    cnt = np.bincount(b[ok], weights=wgt[ok], minlength=nbins)
    ksum = np.bincount(b[ok], weights=(wgt * kn)[ok], minlength=nbins)
    psum = np.bincount(b[ok], weights=(wgt * pw)[ok], minlength=nbins)
    G = float(m) ** 3
    safe = np.maximum(cnt, 1.0)
    return (2.0 * np.pi / box) * ksum / safe, (box ** 3 / G ** 2) * psum / safe, cnt


def sheet_resample(pos, n_p, box, r):
    """Sheet-based resampling, trilinear variant (R21).  ``pos`` [n_p^3, 3] in Lagrangian (C, k fastest) order:
    particle (i, j, k) started at q = (i, j, k) L / n_p.  Its displacement Psi = X - q is taken with the minimum
    image convention.  The refined sheet has (r n_p)^3 points q' = (i', j', k') L / (r n_p); each gets
    X' = q' + trilinear interpolation of Psi between its 8 Lagrangian neighbours, wrapped into [0, L).
    Returns fp64 [(r n_p)^3, 3] in the same (C) order; r = 1 returns the wrapped input."""
    X = np.asarray(pos).astype(np.float64).reshape(n_p, n_p, n_p, 3)
    q1 = np.arange(n_p) * (box / n_p)
    q = np.stack(np.meshgrid(q1, q1, q1, indexing="ij"), axis=-1)
    psi = X - q
    psi -= box * np.round(psi / box)
    nf = r * n_p
    idx = np.arange(nf)
    i0 = idx // r
    t = (idx % r) / float(r)
    out = np.zeros((nf, nf, nf, 3))
    for dx in (0, 1):
        wx = np.where(dx, t, 1.0 - t)[:, None, None, None]
        ix = (i0 + dx) % n_p
        for dy in (0, 1):
            wy = np.where(dy, t, 1.0 - t)[None, :, None, None]
            iy = (i0 + dy) % n_p
            for dz in (0, 1):
                wz = np.where(dz, t, 1.0 - t)[None, None, :, None]
                iz = (i0 + dz) % n_p
                out += wx * wy * wz * psi[np.ix_(ix, iy, iz)]
    qf1 = idx * (box / nf)
    out += np.stack(np.meshgrid(qf1, qf1, qf1, indexing="ij"), axis=-1)
    return np.mod(out, box).reshape(-1, 3)
