"""Seeded input generators (see package docstring; recipe in DESIGN.md "Input recipe").

Everything here is plain NumPy (SciPy's pocketfft when present, only to use
several host threads).  Nothing here knows about mass-assignment kernels,
Green's functions or NUFFT kernels.
"""
from __future__ import annotations

import numpy as np

try:  # scipy.fft only buys host threads; numpy.fft gives identical inputs to ~1e-16
    import scipy.fft as _fft

    def _rfftn(a):
        return _fft.rfftn(a, workers=-1)

    def _irfftn(a, s):
        return _fft.irfftn(a, s=s, workers=-1)

except Exception:  # pragma: no cover
    def _rfftn(a):
        return np.fft.rfftn(a)

    def _irfftn(a, s):
        return np.fft.irfftn(a, s=s)


# The workloads named by BASELINE.json "configs" (+ the north_star headline).
# Fields: n_p particles per dim, m mesh cells per dim, box L, rms displacement in
# MESH cells, assignment order, interlace mode, gradient / Laplacian order,
# deconvolution power, seed.  SURVEY.md 8(d) fixes what BASELINE leaves open.
CONFIGS = {
    "cfg0": dict(n_p=32, m=32, box=256.0, rms=0.5, worder=2, interlace=0, grad_order=0,
                 lap_order=0, deconv_pow=2, seed=1000),
    "cfg1": dict(n_p=128, m=128, box=500.0, rms=1.0, worder=3, interlace=1, grad_order=4,
                 lap_order=0, deconv_pow=2, seed=1001, cot_seed=2001),
    "cfg2": dict(n_p=256, m=512, box=640.0, rms=1.5, worder=2, interlace=0, grad_order=4,
                 lap_order=0, deconv_pow=0, seed=1002),
    "cfg3": dict(n_p=512, m=512, box=1000.0, rms=2.0, nufft=True, sigma=2.0, eps=1e-6,
                 grad_order=0, lap_order=0, seed=1003),
    "cfg4": dict(n_p=512, m=1024, box=1000.0, rms=2.0, worder=2, interlace=0, grad_order=4,
                 lap_order=0, deconv_pow=0, seed=1004, cot_seed=2004, clustered=True),
    "headline": dict(n_p=512, m=512, box=1000.0, rms=1.0, worder=2, interlace=0, grad_order=4,
                     lap_order=0, deconv_pow=2, seed=1005),
    # cfg3 with the paper's own NUFFT setting (upsampling 5/4, kernel of 5^3 cells): fine grid 640^3
    "cfg3_paper": dict(n_p=512, m=512, box=1000.0, rms=2.0, nufft=True, sigma=1.25, eps=1e-4, width=5,
                       grad_order=0, lap_order=0, seed=1006),
}


def _wrap_fp32(x64: np.ndarray, box: float) -> np.ndarray:
    """Periodic wrap into [0, box) and cast to fp32; values that round to box become 0."""
    x64 = np.mod(x64, box)
    x32 = x64.astype(np.float32)
    x32[x32 >= np.float32(box)] = np.float32(0.0)
    return x32


def _power_law_displacement(shape, seed: int) -> np.ndarray:
    """Curl-free Gaussian displacement field on a lattice of ``shape`` points.

    White noise -> FFT -> amplitude |n|^-1 (a density spectrum P ~ k^-2), zero at
    n = 0 and on every Nyquist plane -> psi_hat = i n / |n|^2 delta_hat -> inverse FFT.
    Returns psi with shape ``shape + (3,)`` in arbitrary units (the caller rescales).
    """
    rng = np.random.default_rng(seed)
    white = rng.standard_normal(shape)
    wh = _rfftn(white)
    del white
    nx = np.fft.fftfreq(shape[0], 1.0 / shape[0])[:, None, None]
    ny = np.fft.fftfreq(shape[1], 1.0 / shape[1])[None, :, None]
    nz = np.fft.rfftfreq(shape[2], 1.0 / shape[2])[None, None, :]
    # use wave numbers per unit lattice LENGTH so anisotropic lattices stay isotropic in k
    n2 = nx * nx + ny * ny + nz * nz
    n2[0, 0, 0] = 1.0
    amp = 1.0 / np.sqrt(n2)
    amp[0, 0, 0] = 0.0
    for ax, n in enumerate(shape):
        if n % 2 == 0:
            idx = [slice(None)] * 3
            idx[ax] = n // 2
            amp[tuple(idx)] = 0.0
    wh *= amp
    del amp
    psi = np.empty(tuple(shape) + (3,), dtype=np.float64)
    for a, na in enumerate((nx, ny, nz)):
        psi[..., a] = _irfftn(1j * (na / n2) * wh, tuple(shape))
    return psi


def lattice_displaced(n_p, m: int, box: float, rms_cells: float, seed: int,
                      return_lattice: bool = False):
    """Lattice + Gaussian displacement particle set (configs 0-3, headline).

    ``n_p`` is an int (cubic lattice) or a 3-tuple.  Lattice points q = (i,j,k) * box/n_p
    in C order (k fastest) -- the Lagrangian particle order of a real run.  The
    displacement is rescaled so that sqrt(<|psi|^2>) (3-D norm) = rms_cells * box / m.
    Returns fp32 positions [N, 3] in [0, box).
    """
    shape = (n_p,) * 3 if np.isscalar(n_p) else tuple(int(v) for v in n_p)
    psi = _power_law_displacement(shape, seed)
    norm = np.sqrt(np.mean(np.sum(psi * psi, axis=-1)))
    psi *= (rms_cells * box / m) / norm
    for a in range(3):
        q = np.arange(shape[a], dtype=np.float64) * (box / shape[a])
        sh = [1, 1, 1]
        sh[a] = shape[a]
        psi[..., a] += q.reshape(sh)
    pos = _wrap_fp32(psi.reshape(-1, 3), box)
    if return_lattice:
        return pos, shape
    return pos


def uniform_lattice(n_p: int, box: float, offset: float = 0.0) -> np.ndarray:
    """Undisplaced lattice (zero-force invariant), fp32 [N,3]."""
    q = (np.arange(n_p, dtype=np.float64) * (box / n_p) + offset)
    g = np.stack(np.meshgrid(q, q, q, indexing="ij"), axis=-1).reshape(-1, 3)
    return _wrap_fp32(g, box)


def uniform_random(n: int, box: float, seed: int) -> np.ndarray:
    """Uniform random positions, fp32 [n,3] (incoherent order: stresses binning)."""
    rng = np.random.default_rng(seed)
    return _wrap_fp32(rng.random((n, 3)) * box, box)


def clustered_halos(n_total: int, m: int, box: float, seed: int, n_halos: int = 10_000,
                    scale_radius: float = 1.0, slope: float = -1.9, mass_range=(1.0, 1.0e3),
                    lattice_shape=None, rms_cells: float = 2.0, shuffle: bool = False) -> np.ndarray:
    """Config 4: half Plummer-profile halos, half displaced lattice (BASELINE.json configs[4]).

    Halo half: ``n_halos`` centres uniform in the box; masses from dn/dM ~ M^slope on
    ``mass_range`` by inverse CDF; particle counts proportional to mass (largest-remainder
    rounding); Plummer radii r = a / sqrt(u^(-2/3) - 1), u ~ U(0, 0.999); isotropic
    directions.  Lattice half: ``lattice_shape`` points (default n x n x n/2 with
    n = round((2*n_half)^(1/3))) displaced with ``rms_cells`` mesh cells.
    Order: halo particles grouped by halo, then the lattice half; ``shuffle`` applies a
    seeded global permutation.
    """
    rng = np.random.default_rng(seed)
    n_half = n_total // 2
    n_lat = n_total - n_half
    # halo masses, inverse CDF of a power law
    a1 = slope + 1.0
    lo, hi = mass_range
    u = rng.random(n_halos)
    mass = (lo ** a1 + u * (hi ** a1 - lo ** a1)) ** (1.0 / a1)
    share = mass / mass.sum() * n_half
    counts = np.floor(share).astype(np.int64)
    rem = n_half - counts.sum()
    if rem > 0:
        order = np.argsort(-(share - counts), kind="stable")
        counts[order[:rem]] += 1
    centres = rng.random((n_halos, 3)) * box
    halo_id = np.repeat(np.arange(n_halos), counts)
    uu = rng.random(n_half) * 0.999
    uu = np.maximum(uu, 1e-12)
    r = scale_radius / np.sqrt(uu ** (-2.0 / 3.0) - 1.0)
    cth = rng.random(n_half) * 2.0 - 1.0
    sth = np.sqrt(1.0 - cth * cth)
    ph = rng.random(n_half) * (2.0 * np.pi)
    xh = np.empty((n_half, 3), dtype=np.float64)
    xh[:, 0] = r * sth * np.cos(ph)
    xh[:, 1] = r * sth * np.sin(ph)
    xh[:, 2] = r * cth
    xh += centres[halo_id]
    pos_h = _wrap_fp32(xh, box)
    del xh
    if lattice_shape is None:
        n = int(round((2.0 * n_lat) ** (1.0 / 3.0)))
        lattice_shape = (n, n, n // 2)
    assert int(np.prod(lattice_shape)) == n_lat, (lattice_shape, n_lat)
    pos_l = lattice_displaced(lattice_shape, m, box, rms_cells, seed + 7919)
    pos = np.concatenate([pos_h, pos_l], axis=0)
    if shuffle:
        pos = pos[rng.permutation(pos.shape[0])]
    return np.ascontiguousarray(pos)


def gaussian_cotangent(n: int, seed: int, ncomp: int = 3) -> np.ndarray:
    """Seeded N(0,1) cotangent on per-particle forces, fp32 [n, ncomp]."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, ncomp)).astype(np.float32)


def random_mesh(m: int, seed: int, ncomp: int = 1) -> np.ndarray:
    """Seeded N(0,1) mesh values, fp32 [ncomp, m, m, m] (inputs for gather-only parity)."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((ncomp, m, m, m)).astype(np.float32)


def make_config_positions(name: str, n_p: int | None = None, m: int | None = None,
                          shuffle: bool = False) -> tuple[np.ndarray, dict]:
    """Positions for a named BASELINE config, optionally at reduced (n_p, m).

    Reduced sizes keep the config's ratio m/n_p, box/m (cell size), kernel settings and
    rms displacement in cells; the parity tests use them where the fp64 oracle would not
    finish in seconds at full size.
    """
    c = dict(CONFIGS[name])
    if n_p is not None:
        ratio = c["m"] / c["n_p"]
        cell = c["box"] / c["m"]
        c["n_p"] = int(n_p)
        c["m"] = int(m) if m is not None else int(round(n_p * ratio))
        c["box"] = cell * c["m"]
    if c.get("clustered"):
        n_total = c["n_p"] ** 3
        n_halos = max(4, int(round(10_000 * n_total / 512 ** 3)))
        pos = clustered_halos(n_total, c["m"], c["box"], c["seed"], n_halos=n_halos,
                              lattice_shape=(c["n_p"], c["n_p"], c["n_p"] // 2),
                              rms_cells=c["rms"], shuffle=shuffle)
    else:
        pos = lattice_displaced(c["n_p"], c["m"], c["box"], c["rms"], c["seed"])
        if shuffle:
            pos = pos[np.random.default_rng(c["seed"] + 1).permutation(pos.shape[0])]
    return pos, c


def plane_wave_modes(m: int, n_waves: int, seed: int):
    """Seeded set of distinct Fourier modes and complex amplitudes for a synthetic mesh field
    f(j) = Re sum_w c_w exp(2 pi i n_w . j / m): integer FFT indices idx [W, 3] in [0, m) and c [W].
    Mixes low wave numbers, modes on the Nyquist planes and modes with zero components with random ones;
    no mode is its own conjugate and no two modes are conjugates of each other."""
    rng = np.random.default_rng(seed)
    idx = rng.integers(0, m, size=(n_waves, 3))
    k = n_waves // 8
    idx[:k] = rng.integers(-3, 4, size=(k, 3)) % m                      # low |n|
    idx[k:2 * k, rng.integers(0, 3)] = m // 2                           # a Nyquist plane
    idx[2 * k:3 * k, 0] = 0                                             # n_x = 0 plane
    idx[3 * k:4 * k, 2] = rng.integers(0, 2, size=k) * (m // 2)         # n_z in {0, Nyquist}
    seen, keep = set(), []
    for w in range(n_waves):
        t = tuple(int(v) for v in idx[w])
        neg = tuple((-v) % m for v in t)
        if t == neg or t in seen or neg in seen:
            continue
        seen.add(t)
        keep.append(w)
    idx = idx[keep]
    coef = rng.standard_normal(len(keep)) + 1j * rng.standard_normal(len(keep))
    return idx, coef


def plane_wave_values(m: int, idx, coef, nodes):
    """f at integer node triples ``nodes`` [K, 3] for the field of :func:`plane_wave_modes`, fp64."""
    nodes = np.asarray(nodes, dtype=np.int64)
    out = np.zeros(nodes.shape[0])
    for w0 in range(0, idx.shape[0], 64):  # chunks keep the phase table small
        ph = (nodes @ idx[w0:w0 + 64].T.astype(np.int64)) % m
        out += (np.exp(2j * np.pi * ph / m) * coef[None, w0:w0 + 64]).real.sum(axis=1)
    return out
