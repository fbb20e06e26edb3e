"""Pins of the fp64 PM oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage (PAPER.md line / equation / table) it pins.
"""
import os

import numpy as np
import pytest

from oracle import pm_oracle as po
from pm_inputs import lattice_displaced, uniform_random
from pm_inputs.generators import uniform_lattice

ORDERS = (2, 3, 4)


def _load_table(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


# ---------------------------------------------------------------- Table 1 kernels
def test_table1_hand_values(golden_dir):
    for wo, x, val in _load_table(os.path.join(golden_dir, "table1_kernels.txt")):
        assert abs(po.kernel_W(float(x), int(wo)) - float(val)) < 1e-15
        assert abs(po.kernel_W(-float(x), int(wo)) - float(val)) < 1e-15


@pytest.mark.parametrize("worder", ORDERS)
def test_partition_of_unity_and_moments(worder):
    """Sum_j W(j-u) = 1 (mass conservation, Eq. C.1), sum_j j W(j-u) = u, sum_j dW = 0."""
    u = np.random.default_rng(1).random(1000) * 7.0 + 3.0
    j0, W = po.node_weights(u, worder)
    _, dW = po.node_weights(u, worder, deriv=True)
    nodes = j0[:, None] + np.arange(po.SUPPORT[worder])[None, :]
    assert np.abs(W.sum(1) - 1.0).max() < 1e-14
    assert np.abs((nodes * W).sum(1) - u).max() < 1e-13
    assert np.abs(dW.sum(1)).max() < 1e-14
    assert np.abs((nodes * dW).sum(1) - 1.0).max() < 1e-13  # d/du of the first moment
    assert (W >= 0).all()


@pytest.mark.parametrize("worder", (3, 4))
def test_kernel_derivative_matches_difference_quotient(worder):
    x = np.linspace(-2.2, 2.2, 4001)
    h = 1e-6
    fd = (po.kernel_W(x + h, worder) - po.kernel_W(x - h, worder)) / (2 * h)
    assert np.abs(fd - po.kernel_dW(x, worder)).max() < 1e-5


@pytest.mark.parametrize("worder", ORDERS)
def test_window_is_fourier_transform_of_kernel(worder):
    """Table 1 Fourier column: int W(x) cos(theta x) dx = sinc(n/m)^p with theta = 2 pi n/m."""
    m = 16
    x = np.linspace(-2.0, 2.0, 400001)
    Wx = po.kernel_W(x, worder)
    n = po.mode_numbers(m)
    num = np.array([np.trapezoid(Wx * np.cos(2 * np.pi * nn / m * x), x) for nn in n])
    assert np.abs(num - po.window_1d(m, worder)).max() < 1e-9


# ---------------------------------------------------------------- scatter / gather
@pytest.mark.parametrize("worder", ORDERS)
@pytest.mark.parametrize("shifted", (False, True))
def test_scatter_gather_vs_bruteforce(worder, shifted):
    """Eq. C.1 (:864) and C.2 (:872) summed over every (particle, node) pair."""
    m, box = 10, 25.0
    pos = uniform_random(300, box, 11)
    w = np.random.default_rng(2).standard_normal(300)
    shift = np.array([0.3, -1.7, 0.5 * box / m]) if shifted else None
    rho = po.scatter(pos, m, box, worder, weights=w, shift=shift)
    assert np.abs(rho - po.scatter_bruteforce(pos, m, box, worder, w, shift)).max() < 1e-13
    mesh = np.random.default_rng(3).standard_normal((m, m, m))
    v = po.gather(mesh, pos, box, worder, shift=shift)
    assert np.abs(v - po.gather_bruteforce(mesh, pos, box, worder, shift)).max() < 1e-13


@pytest.mark.parametrize("worder", ORDERS)
def test_mass_conservation_and_accumulate(worder):
    m, box = 12, 30.0
    pos = uniform_random(500, box, 5)
    w = np.random.default_rng(6).random(500)
    pre = np.full((m, m, m), 0.25)
    rho = po.scatter(pos, m, box, worder, weights=w, mesh=pre.copy())
    assert abs((rho - pre).sum() - w.sum()) < 1e-11  # exact up to summation rounding
    assert np.abs(rho - pre - po.scatter(pos, m, box, worder, weights=w)).max() < 1e-14  # adds (:884)


@pytest.mark.parametrize("worder", ORDERS)
def test_adjointness(worder):
    """<scatter(w), rho>_mesh = <w, gather(rho)>_particles, Eq. C.14 (:966)."""
    m, box = 12, 30.0
    pos = uniform_random(400, box, 7)
    rng = np.random.default_rng(8)
    w, mesh = rng.standard_normal(400), rng.standard_normal((m, m, m))
    lhs = (po.scatter(pos, m, box, worder, weights=w) * mesh).sum()
    rhs = (w * po.gather(mesh, pos, box, worder)).sum()
    assert abs(lhs - rhs) < 1e-12


@pytest.mark.parametrize("worder", (3, 4))
def test_gradW_gather_vs_finite_difference(worder):
    """Eq. C.11/C.12: d gather / dX by central differences (smooth kernels only, R12)."""
    m, box = 12, 30.0
    pos = uniform_random(50, box, 9).astype(np.float64)
    mesh = np.random.default_rng(10).standard_normal((m, m, m))
    h = 1e-5
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        fd = (po.gather(mesh, pos + e, box, worder) - po.gather(mesh, pos - e, box, worder)) / (2 * h)
        an = po.gather(mesh, pos, box, worder, deriv_axis=a)
        assert np.abs(fd - an).max() < 1e-7 * np.abs(an).max() + 1e-8


# ---------------------------------------------------------------- Table 2 symbols
def test_fft_convention_bruteforce():
    """O4: numpy.fft.rfftn is the unnormalised forward sum_j f_j exp(-i k.r_j)."""
    m = 4
    f = np.random.default_rng(0).standard_normal((m, m, m))
    j = np.arange(m)
    F = np.zeros((m, m, m), dtype=complex)
    for a in range(m):
        for b in range(m):
            for c in range(m):
                ph = np.exp(-2j * np.pi * (a * j[:, None, None] + b * j[None, :, None] + c * j[None, None, :]) / m)
                F[a, b, c] = (f * ph).sum()
    assert np.abs(F[:, :, : m // 2 + 1] - np.fft.rfftn(f)).max() < 1e-12


def test_symbols_are_dft_of_printed_stencils(golden_dir):
    """Table 2 (:231-242): Fourier column = DFT of the Real column (R4 fixes the order-2 sign)."""
    m = 32
    th = 2 * np.pi * po.mode_numbers(m) / m
    for kind, order, den, *coef in _load_table(os.path.join(golden_dir, "table2_stencils.txt")):
        c = np.array([float(v) for v in coef]) / float(den)
        r = (len(c) - 1) // 2
        s = np.arange(-r, r + 1)
        sym = (c[None, :] * np.exp(1j * th[:, None] * s[None, :])).sum(1)
        if kind == "grad":
            assert np.abs(sym - 1j * po.grad_symbol_1d(m, int(order))).max() < 1e-14
        else:
            assert np.abs(sym - po.lap_symbol_1d(m, int(order))).max() < 1e-13


def test_symbol_small_k_limits():
    """Table 2: every order tends to i k resp. -k^2 as k -> 0; exact rows are i k, -k^2."""
    m = 4096
    th = 2 * np.pi * po.mode_numbers(m) / m
    lo = slice(1, 6)
    for o in (2, 4, 6):
        assert np.abs(po.grad_symbol_1d(m, o)[lo] / th[lo] - 1).max() < 1e-4
        assert np.abs(po.lap_symbol_1d(m, o)[lo] / (-th[lo] ** 2) - 1).max() < 1e-4
    assert np.abs(po.grad_symbol_1d(m, 0)[1 : m // 2] - th[1 : m // 2]).max() == 0
    assert po.grad_symbol_1d(m, 0)[m // 2] == 0.0  # R5
    assert np.abs(po.lap_symbol_1d(m, 0) + th ** 2).max() == 0


@pytest.mark.parametrize("grad_order", (0, 2, 4, 6))
@pytest.mark.parametrize("lap_order", (0, 2, 4, 6))
def test_mesh_injection_closed_form(grad_order, lap_order):
    """delta_j = A cos(k0.r_j) => g_a = coeff A [D(th_a)/Delta]/[sum_b l(th_b)/Delta^2] sin(k0.r_j)
    (Eq. 2.1-2.2 with Table 2 symbols; R6: gradient along its own axis, Laplacian summed)."""
    m, box, A, coeff = 16, 40.0, 0.7, 2.5
    n0 = np.array([2, -3, 1])
    d = box / m
    j = np.arange(m)
    phase = 2 * np.pi * (n0[0] * j[:, None, None] + n0[1] * j[None, :, None] + n0[2] * j[None, None, :]) / m
    g = po.poisson_force(A * np.cos(phase), box, 2, grad_order, lap_order, 0, coeff)
    th = 2 * np.pi * n0 / m
    D = {0: lambda t: t, 2: np.sin, 4: lambda t: (8 * np.sin(t) - np.sin(2 * t)) / 6,
         6: lambda t: (45 * np.sin(t) - 9 * np.sin(2 * t) + np.sin(3 * t)) / 30}[grad_order]
    # Laplacian symbols retyped from the printed stencils of Table 2 (not from the oracle)
    L = {0: lambda t: -t * t, 2: lambda t: 2 * np.cos(t) - 2,
         4: lambda t: (-2 * np.cos(2 * t) + 32 * np.cos(t) - 30) / 12,
         6: lambda t: (4 * np.cos(3 * t) - 54 * np.cos(2 * t) + 540 * np.cos(t) - 490) / 180}[lap_order]
    lap = sum(L(t) for t in th) / d ** 2
    for a in range(3):
        expect = coeff * A * (D(th[a]) / d) / lap * np.sin(phase)
        assert np.abs(g[a] - expect).max() < 1e-13 * max(1.0, np.abs(expect).max())


def test_deconvolution_divides_by_window_power():
    """:262 'division by the squared Fourier kernel': injection amplitude scales by 1/W~^p."""
    m, box = 16, 16.0
    n0 = np.array([3, 0, -2])
    j = np.arange(m)
    phase = 2 * np.pi * (n0[0] * j[:, None, None] + n0[1] * j[None, :, None] + n0[2] * j[None, None, :]) / m
    base = po.poisson_force(np.cos(phase), box, 3, 4, 0, 0)[0]
    for p in (1, 2):
        win = np.prod(np.sinc(n0 / m) ** 3)
        assert np.abs(po.poisson_force(np.cos(phase), box, 3, 4, 0, p)[0] - base / win ** p).max() < 1e-12


# ---------------------------------------------------------------- forward-mode rules, Eq. C.13
@pytest.mark.parametrize("worder", (3, 4))
@pytest.mark.parametrize("shifted", (False, True))
def test_jvp_rules_match_central_differences(worder, shifted):
    """Eq. C.13a/b (:943-945): tangents of scatter and gather w.r.t. positions, weights and mesh against
    central differences of Eq. C.1 / C.2 (TSC / PCS: continuous derivatives)."""
    m, box, n = 10, 25.0, 200
    rng = np.random.default_rng(40 + worder)
    pos = uniform_random(n, box, 41).astype(np.float64)
    w = rng.standard_normal(n)
    tX, tw = rng.standard_normal((n, 3)), rng.standard_normal(n)
    mesh, tmesh = rng.standard_normal((m, m, m)), rng.standard_normal((m, m, m))
    rho_in_tan = rng.standard_normal((m, m, m))
    shift = np.array([0.3, -1.7, 0.5 * box / m]) if shifted else None
    h = 1e-6
    fd = (po.scatter(pos + h * tX, m, box, worder, weights=w + h * tw, shift=shift)
          - po.scatter(pos - h * tX, m, box, worder, weights=w - h * tw, shift=shift)) / (2 * h) + rho_in_tan
    jvp = po.scatter_jvp(pos, m, box, worder, weights=w, pos_tan=tX, w_tan=tw, shift=shift, mesh_tan=rho_in_tan)
    assert np.abs(fd - jvp).max() < 1e-7 * np.abs(jvp).max()
    fdg = (po.gather(mesh + h * tmesh, pos + h * tX, box, worder, shift=shift)
           - po.gather(mesh - h * tmesh, pos - h * tX, box, worder, shift=shift)) / (2 * h)
    jg = po.gather_jvp(mesh, pos, box, worder, pos_tan=tX, mesh_tan=tmesh, shift=shift)
    assert np.abs(fdg - jg).max() < 1e-7 * np.abs(jg).max()


@pytest.mark.parametrize("worder", ORDERS)
def test_jvp_vjp_duality(worder):
    """<JVP(tangent), cotangent> = <tangent, VJP(cotangent)> for scatter and gather (rule table :949-960);
    also pins the CIC rules, whose derivative is piecewise constant (R12)."""
    m, box, n = 9, 18.0, 150
    rng = np.random.default_rng(50 + worder)
    pos = uniform_random(n, box, 51)
    w = rng.standard_normal(n)
    tX, tw = rng.standard_normal((n, 3)), rng.standard_normal(n)
    cot_mesh = rng.standard_normal((m, m, m))
    lhs = np.sum(po.scatter_jvp(pos, m, box, worder, weights=w, pos_tan=tX, w_tan=tw) * cot_mesh)
    xbar = np.stack([w * po.gather(cot_mesh, pos, box, worder, deriv_axis=a) for a in range(3)], axis=1)  # Eq. C.6
    wbar = po.gather(cot_mesh, pos, box, worder)                                                          # Eq. C.8
    assert abs(lhs - (np.sum(tX * xbar) + np.sum(tw * wbar))) < 1e-11 * max(1.0, abs(lhs))
    mesh, tmesh = rng.standard_normal((m, m, m)), rng.standard_normal((m, m, m))
    cot_v = rng.standard_normal(n)
    lhs = np.sum(po.gather_jvp(mesh, pos, box, worder, pos_tan=tX, mesh_tan=tmesh) * cot_v)
    mbar = po.scatter(pos, m, box, worder, weights=cot_v)                                                 # Eq. C.10
    xbar = np.stack([cot_v * po.gather(mesh, pos, box, worder, deriv_axis=a) for a in range(3)], axis=1)  # Eq. C.12
    assert abs(lhs - (np.sum(tmesh * mbar) + np.sum(tX * xbar))) < 1e-11 * max(1.0, abs(lhs))


# ---------------------------------------------------------------- Table 2, "Real" column
def test_real_space_stencils_are_the_printed_ones(golden_dir):
    for kind, order, den, *coef in _load_table(os.path.join(golden_dir, "table2_stencils.txt")):
        if kind != "grad":
            continue
        d, c = po.GRAD_STENCIL[int(order)]
        r = len(c)
        printed = [float(v) for v in coef]
        assert d == float(den) and printed[r] == 0.0
        assert printed[r + 1:] == list(c) and printed[:r] == [-v for v in reversed(c)]


@pytest.mark.parametrize("order", (2, 4, 6))
@pytest.mark.parametrize("interlaced", (False, True))
def test_real_space_gradient_equals_fourier_symbol(order, interlaced):
    """g = -stencil(IFFT(phi_hat)) is the same operator as IFFT(-i D(theta)/Delta phi_hat) (Table 2: the
    Fourier entries are the DFTs of the stencils): one inverse FFT instead of three."""
    m, box = 12, 30.0
    d = np.random.default_rng(60).standard_normal((2, m, m, m))
    d2 = d[1] if interlaced else None
    a = po.poisson_force(d[0], box, 3, order, 0, 2, coeff=1.3, delta_mesh2=d2)
    b = po.poisson_force_real_gradient(d[0], box, 3, order, 0, 2, coeff=1.3, delta_mesh2=d2)
    for x, y in zip(a, b):
        assert np.abs(x - y).max() < 1e-13 * np.abs(x).max()
    # the stencil differentiates a resolved plane wave to its order of accuracy
    x = np.arange(m) * (box / m)
    f = np.broadcast_to(np.sin(2 * np.pi * x / box)[:, None, None], (m, m, m))
    exact = np.broadcast_to((2 * np.pi / box) * np.cos(2 * np.pi * x / box)[:, None, None], (m, m, m))
    err = np.abs(po.fd_gradient_real(f, box, order, 0) - exact).max() / (2 * np.pi / box)
    assert err < {2: 0.05, 4: 4e-3, 6: 4e-4}[order]
    assert np.abs(po.fd_gradient_real(f, box, order, 1)).max() < 1e-14


def test_force_symbol_at_matches_the_symbol_arrays():
    m, box = 12, 30.0
    rng = np.random.default_rng(70)
    idx = tuple(rng.integers(0, m, 200) for _ in range(2)) + (rng.integers(0, m // 2 + 1, 200),)
    idx[0][:3] = idx[1][:3] = idx[2][:3] = 0          # the n = 0 mode
    idx[0][3:6] = m // 2                              # Nyquist planes
    idx[2][6:9] = m // 2
    for go, lo, dp, wo in ((0, 0, 2, 2), (4, 0, 2, 3), (6, 6, 1, 4), (2, 2, 0, 2)):
        S = po.force_symbols(m, box, wo, go, lo, dp, 1.7)
        Sa = po.force_symbol_at(idx, m, box, wo, go, lo, dp, 1.7)
        for a in range(3):
            assert np.array_equal(S[a][idx], Sa[a])
