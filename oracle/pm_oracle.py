"""Plain fp64 oracle of the particle-mesh force path (TEST INFRASTRUCTURE, see package docstring).

Every function follows the paper step by step (citations are PAPER.md line numbers and the
section / equation / table they fall in) with the readings R1..R15 of DESIGN.md.  NumPy only;
``numpy.bincount`` (a weighted histogram) and ``numpy.fft`` serve as library steps, nothing is
blocked, fused or reordered.  Inputs are the fp32 arrays the GPU path receives, cast exactly
to fp64.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): brute-force Eq. C.1 / C.2 over all (i, j)
with W taken from the piecewise definition; partition of unity and first moment of Table 1;
adjointness Eq. C.14; mesh-injection closed form for every (grad, lap) order of Table 2; DFT of
the printed stencils equals the printed symbols; zero force on a lattice; momentum
conservation; plane-wave sheet force; central finite differences for the VJP and the JVPs
(Eq. C.13), JVP/VJP duality; the real-space stencils of Table 2 against their Fourier symbols.
Parity unpinned (GPU-vs-oracle only): the CIC position-VJP for particles that sit exactly on
a mesh node (R12: the derivative of W is discontinuous there).
"""
from __future__ import annotations

import numpy as np

SUPPORT = {2: 2, 3: 3, 4: 4}  # worder -> nodes per axis (Table 1 :223-229, "Discrete support")

# The FFT is a library step (:244).  FFT_WORKERS = 1: numpy.fft.  FFT_WORKERS != 1: the same transforms
# through scipy.fft (pocketfft as well) with that many host threads (-1 = all) -- set by the full-size
# parity tests (1024^3 meshes) and by bench.py's all-cores timing; the arithmetic is unchanged.
FFT_WORKERS = 1


def _rfftn(a):
    if FFT_WORKERS == 1:
        return np.fft.rfftn(a)
    import scipy.fft as sfft
    return sfft.rfftn(a, workers=FFT_WORKERS)


def _irfftn(a, m):
    if FFT_WORKERS == 1:
        return np.fft.irfftn(a, s=(m, m, m), axes=(0, 1, 2))
    import scipy.fft as sfft
    return sfft.irfftn(a, s=(m, m, m), axes=(0, 1, 2), workers=FFT_WORKERS)


# --------------------------------------------------------------------------------------
# Table 1 (:223-229): 1-D assignment kernels W(x), x in grid cells (reading R2)
# --------------------------------------------------------------------------------------
def kernel_W(x, worder: int):
    """W(x) of Table 1: CIC (worder 2), TSC (3), PCS (4); x in cells, any sign."""
    a = np.abs(np.asarray(x, dtype=np.float64))
    if worder == 2:
        return np.where(a <= 1.0, 1.0 - a, 0.0)
    if worder == 3:
        return np.where(a <= 0.5, 0.75 - a * a,
                        np.where(a <= 1.5, 0.5 * (1.5 - a) ** 2, 0.0))
    if worder == 4:
        return np.where(a <= 1.0, (4.0 - 6.0 * a * a + 3.0 * a ** 3) / 6.0,
                        np.where(a <= 2.0, (2.0 - a) ** 3 / 6.0, 0.0))
    raise ValueError("worder must be 2, 3 or 4")


def kernel_dW(x, worder: int):
    """dW/dx of Table 1's kernels.  CIC is one-sided at x = 0 and |x| = 1 (reading R12):
    the slope is that of the cell [i0, i0+1) which contains the particle."""
    x = np.asarray(x, dtype=np.float64)
    a = np.abs(x)
    sgn = np.where(x >= 0.0, 1.0, -1.0)
    if worder == 2:
        return np.where(a <= 1.0, -sgn, 0.0)
    if worder == 3:
        return np.where(a <= 0.5, -2.0 * x, np.where(a <= 1.5, -(1.5 - a) * sgn, 0.0))
    if worder == 4:
        return np.where(a <= 1.0, (-12.0 * a + 9.0 * a * a) / 6.0 * sgn,
                        np.where(a <= 2.0, -0.5 * (2.0 - a) ** 2 * sgn, 0.0))
    raise ValueError("worder must be 2, 3 or 4")


# --------------------------------------------------------------------------------------
# O1/O2: cell coordinates and the node set each particle touches (readings R3)
# --------------------------------------------------------------------------------------
def cell_coords(pos, m: int, box: float, shift=None):
    """u = (X - s)/Delta in fp64, Delta = box/m; mesh nodes sit at r_j = j*Delta (:854-860)."""
    X = np.asarray(pos).astype(np.float64)
    if shift is not None:
        X = X - np.asarray(shift, dtype=np.float64)[None, :]
    return X / (box / m)


def first_node(u, worder: int):
    """Index of the lowest node with non-zero weight: floor(u) for CIC, floor(u+1/2)-1 for
    TSC, floor(u)-1 for PCS (unwrapped, int64)."""
    if worder == 2:
        return np.floor(u).astype(np.int64)
    if worder == 3:
        return np.floor(u + 0.5).astype(np.int64) - 1
    if worder == 4:
        return np.floor(u).astype(np.int64) - 1
    raise ValueError("worder must be 2, 3 or 4")


def node_weights(u, worder: int, deriv: bool = False):
    """(j0 [N], W [N, p]) for one axis: nodes j0..j0+p-1 and W(j - u) (or d/du W(j - u))."""
    p = SUPPORT[worder]
    j0 = first_node(u, worder)
    x = (j0[:, None] + np.arange(p)[None, :]).astype(np.float64) - u[:, None]  # r_j - X_i in cells
    if deriv:
        # d/du W(j - u) = -W'(j - u).  CIC one-sided (R12): particle in [j0, j0+1) sees slope
        # -1 on node j0 and +1 on node j0+1, also when it sits exactly on node j0.
        if worder == 2:
            return j0, np.tile(np.array([-1.0, 1.0]), (u.shape[0], 1))
        return j0, -kernel_dW(x, worder)
    return j0, kernel_W(x, worder)


# --------------------------------------------------------------------------------------
# O3: scatter, Eq. C.1 (:864); adds onto the caller's mesh (:884)
# --------------------------------------------------------------------------------------
def scatter(pos, m: int, box: float, worder: int, weights=None, shift=None, mesh=None,
            deriv_axis: int | None = None):
    """rho_j += sum_i w_i W(r_j - X_i + s); returns the fp64 mesh [m, m, m].  With deriv_axis = a the
    kernel is replaced by dW_j(X_i)/dX_i^a = -grad_a W(r_j - X_i) (length units; the scatter of the
    JVP rule Eq. C.6 / C.13a)."""
    u = cell_coords(pos, m, box, shift)
    n = u.shape[0]
    w = np.ones(n) if weights is None else np.asarray(weights).astype(np.float64)
    if deriv_axis is not None:
        w = w * (m / box)
    if mesh is None:
        mesh = np.zeros((m, m, m), dtype=np.float64)
    p = SUPPORT[worder]
    jx, Wx = node_weights(u[:, 0], worder, deriv=(deriv_axis == 0))
    jy, Wy = node_weights(u[:, 1], worder, deriv=(deriv_axis == 1))
    jz, Wz = node_weights(u[:, 2], worder, deriv=(deriv_axis == 2))
    flat = mesh.reshape(-1)
    for a in range(p):
        ia = np.mod(jx + a, m)
        for b in range(p):
            ib = np.mod(jy + b, m)
            for c in range(p):
                ic = np.mod(jz + c, m)
                val = w * Wx[:, a] * Wy[:, b] * Wz[:, c]
                flat += np.bincount((ia * m + ib) * m + ic, weights=val, minlength=m ** 3)
    return mesh


# --------------------------------------------------------------------------------------
# O8: gather, Eq. C.2 (:872); deriv_axis selects the grad-W gather of Eq. C.6 / C.12
# --------------------------------------------------------------------------------------
def gather(mesh, pos, box: float, worder: int, shift=None, deriv_axis: int | None = None):
    """v_i = sum_j mesh_j W(r_j - X_i + s).  With deriv_axis = a it returns
    sum_j mesh_j dW_j(X_i)/dX_i^a (length units: the 1/Delta is included)."""
    mesh = np.asarray(mesh, dtype=np.float64)
    m = mesh.shape[0]
    u = cell_coords(pos, m, box, shift)
    p = SUPPORT[worder]
    js, Ws = [], []
    for a in range(3):
        j0, W = node_weights(u[:, a], worder, deriv=(deriv_axis == a))
        js.append(j0)
        Ws.append(W)
    out = np.zeros(u.shape[0], dtype=np.float64)
    for a in range(p):
        ia = np.mod(js[0] + a, m)
        for b in range(p):
            ib = np.mod(js[1] + b, m)
            for c in range(p):
                ic = np.mod(js[2] + c, m)
                out += mesh[ia, ib, ic] * Ws[0][:, a] * Ws[1][:, b] * Ws[2][:, c]
    if deriv_axis is not None:
        out *= m / box
    return out


# --------------------------------------------------------------------------------------
# Brute force straight from Eq. C.1 / C.2: every (particle, node) pair, minimum image
# --------------------------------------------------------------------------------------
def _min_image(d, m):
    return d - m * np.round(d / m)


def scatter_bruteforce(pos, m, box, worder, weights=None, shift=None):
    u = cell_coords(pos, m, box, shift)
    w = np.ones(u.shape[0]) if weights is None else np.asarray(weights, dtype=np.float64)
    j = np.arange(m, dtype=np.float64)
    Wx = kernel_W(_min_image(j[None, :] - u[:, 0:1], m), worder)  # [N, m]
    Wy = kernel_W(_min_image(j[None, :] - u[:, 1:2], m), worder)
    Wz = kernel_W(_min_image(j[None, :] - u[:, 2:3], m), worder)
    return np.einsum("i,ia,ib,ic->abc", w, Wx, Wy, Wz)


def gather_bruteforce(mesh, pos, box, worder, shift=None):
    mesh = np.asarray(mesh, dtype=np.float64)
    m = mesh.shape[0]
    u = cell_coords(pos, m, box, shift)
    j = np.arange(m, dtype=np.float64)
    Wx = kernel_W(_min_image(j[None, :] - u[:, 0:1], m), worder)
    Wy = kernel_W(_min_image(j[None, :] - u[:, 1:2], m), worder)
    Wz = kernel_W(_min_image(j[None, :] - u[:, 2:3], m), worder)
    return np.einsum("abc,ia,ib,ic->i", mesh, Wx, Wy, Wz)


# --------------------------------------------------------------------------------------
# Forward-mode rules, Eq. C.13 (:943-945), rule table :956-960
# --------------------------------------------------------------------------------------
def scatter_jvp(pos, m: int, box: float, worder: int, weights=None, pos_tan=None, w_tan=None,
                shift=None, mesh_tan=None):
    """Eq. C.13a: rho~_j = rho~_in,j + sum_i [ w~_i W_j(X_i) - w_i X~_i . grad W_j(X_i) ].
    -grad W_j(X_i) = dW_j/dX_i (:860), so the second term is a scatter with the derivative kernel of
    each axis weighted by w_i X~_i^a.  Adds onto ``mesh_tan`` (= rho~_in, Eq. C.4)."""
    n = np.asarray(pos).shape[0]
    w = np.ones(n) if weights is None else np.asarray(weights).astype(np.float64)
    out = np.zeros((m, m, m)) if mesh_tan is None else np.array(mesh_tan, dtype=np.float64)
    if w_tan is not None:
        scatter(pos, m, box, worder, weights=np.asarray(w_tan).astype(np.float64), shift=shift, mesh=out)
    if pos_tan is not None:
        t = np.asarray(pos_tan).astype(np.float64)
        for a in range(3):
            scatter(pos, m, box, worder, weights=w * t[:, a], shift=shift, mesh=out, deriv_axis=a)
    return out


def gather_jvp(mesh, pos, box: float, worder: int, pos_tan=None, mesh_tan=None, shift=None):
    """Eq. C.13b: v~_i = sum_j [ rho~_j W_j(X_i) - rho_j X~_i . grad W_j(X_i) ]."""
    n = np.asarray(pos).shape[0]
    out = np.zeros(n)
    if mesh_tan is not None:
        out += gather(mesh_tan, pos, box, worder, shift=shift)
    if pos_tan is not None:
        t = np.asarray(pos_tan).astype(np.float64)
        for a in range(3):
            out += t[:, a] * gather(mesh, pos, box, worder, shift=shift, deriv_axis=a)
    return out


# --------------------------------------------------------------------------------------
# O5: Fourier symbols, Table 2 (:231-242) and Table 1's Fourier column (:225-229)
# --------------------------------------------------------------------------------------
def mode_numbers(m: int):
    """Integer wave numbers n_a in FFT order, n in {0..m/2-1, -m/2..-1}."""
    return np.fft.fftfreq(m, 1.0 / m)


def grad_symbol_1d(m: int, order: int):
    """D(theta) with Grad = i*D/Delta, theta = 2*pi*n/m = k*Delta.  Table 2 gradient rows with
    k in Nyquist units (theta = pi*k): exact i*k -> theta; order 2 -> sin(theta);
    4 -> (8 sin(theta) - sin(2 theta))/6; 6 -> (45 sin - 9 sin 2 + sin 3)/30.
    Reading R5: the exact symbol is set to 0 at the Nyquist index n = -m/2 (even m)."""
    n = mode_numbers(m)
    th = 2.0 * np.pi * n / m
    if order == 0:
        d = th.copy()
        if m % 2 == 0:
            d[m // 2] = 0.0
    elif order == 2:
        d = np.sin(th)
    elif order == 4:
        d = (8.0 * np.sin(th) - np.sin(2.0 * th)) / 6.0
    elif order == 6:
        d = (45.0 * np.sin(th) - 9.0 * np.sin(2.0 * th) + np.sin(3.0 * th)) / 30.0
    else:
        raise ValueError("grad_order must be 0, 2, 4 or 6")
    return d


def lap_symbol_1d(m: int, order: int):
    """l(theta) with Lap = sum_a l(theta_a)/Delta^2.  Table 2 Laplacian rows: exact -k^2 ->
    -theta^2; order 2 -> 2 cos(theta) - 2 (reading R4: the printed sign is a typo);
    4 -> -(cos 2 theta - 16 cos theta + 15)/6; 6 -> -(-2 cos 3 + 27 cos 2 - 270 cos + 245)/90."""
    n = mode_numbers(m)
    th = 2.0 * np.pi * n / m
    if order == 0:
        return -th * th
    if order == 2:
        return 2.0 * np.cos(th) - 2.0
    if order == 4:
        return -(np.cos(2.0 * th) - 16.0 * np.cos(th) + 15.0) / 6.0
    if order == 6:
        return -(-2.0 * np.cos(3.0 * th) + 27.0 * np.cos(2.0 * th) - 270.0 * np.cos(th) + 245.0) / 90.0
    raise ValueError("lap_order must be 0, 2, 4 or 6")


def window_1d(m: int, worder: int):
    """Table 1 Fourier column: sinc^p(k/2) with k in Nyquist units = sinc(n/m)^p,
    sinc(x) = sin(pi x)/(pi x) (numpy.sinc has exactly this convention)."""
    return np.sinc(mode_numbers(m) / m) ** SUPPORT[worder]


def force_symbols(m: int, box: float, worder: int, grad_order: int, lap_order: int,
                  deconv_pow: int, coeff: float):
    """S_a(n) = -Grad_a * coeff / Lap / W~^deconv_pow on the half-complex grid
    [m, m, m/2+1] (O6; :262-264; Eq. 2.1 g = -grad phi; Eq. 2.2 Lap phi = coeff*delta).
    S_a(0) = 0 (reading R7).  Gradient: the 1-D symbol of its own axis; Laplacian: sum over
    axes (reading R6)."""
    delta = box / m
    h = m // 2 + 1
    D = grad_symbol_1d(m, grad_order)
    l1 = lap_symbol_1d(m, lap_order)
    W1 = window_1d(m, worder)
    lap = (l1[:, None, None] + l1[None, :, None] + l1[None, None, :h]) / delta ** 2
    lap[0, 0, 0] = 1.0
    green = coeff / lap
    green[0, 0, 0] = 0.0
    if deconv_pow:
        win = W1[:, None, None] * W1[None, :, None] * W1[None, None, :h]
        green = green / win ** deconv_pow
    Dz = D[:h].copy()
    if grad_order == 0 and m % 2 == 0:
        Dz[m // 2] = 0.0  # the rfft half keeps n_z = +m/2, the same Nyquist plane (R5)
    S = []
    for a, Da in enumerate((D[:, None, None], D[None, :, None], Dz[None, None, :])):
        S.append(-(1j * Da / delta) * green)
    return S


def force_symbol_at(idx, m: int, box: float, worder: int, grad_order: int, lap_order: int,
                    deconv_pow: int, coeff: float):
    """S_a(n) of :func:`force_symbols` for single modes: idx = (ix, iy, iz) integer FFT indices in [0, m)
    (arrays allowed); returns complex [3, ...].  For meshes too large to hold the 3-D symbol arrays
    (m = 1024); pinned against force_symbols element by element."""
    ix, iy, iz = (np.asarray(v, dtype=np.int64) for v in idx)
    delta = box / m
    D = grad_symbol_1d(m, grad_order)
    l1 = lap_symbol_1d(m, lap_order)
    W1 = window_1d(m, worder)
    lap = (l1[ix] + l1[iy] + l1[iz]) / delta ** 2
    zero = (ix == 0) & (iy == 0) & (iz == 0)
    green = np.where(zero, 0.0, coeff / np.where(zero, 1.0, lap))
    if deconv_pow:
        green = green / (W1[ix] * W1[iy] * W1[iz]) ** deconv_pow
    return np.stack([-(1j * D[i] / delta) * green for i in (ix, iy, iz)])


def interlace_phase(m: int):
    """Per-axis factor of e^{-i k.s} for s = (Delta/2)(1,1,1): exp(-i pi n_a/m); reading R9:
    real part only (= 0) on the Nyquist index so the combined field stays Hermitian."""
    n = mode_numbers(m)
    ph = np.exp(-1j * np.pi * n / m)
    if m % 2 == 0:
        ph[m // 2] = ph[m // 2].real
    return ph


def interlace_phase_3d(m: int):
    p = interlace_phase(m)
    h = m // 2 + 1
    return p[:, None, None] * p[None, :, None] * p[None, None, :h]


# --------------------------------------------------------------------------------------
# O4, O6, O7: delta mesh(es) -> three force meshes
# --------------------------------------------------------------------------------------
def poisson_force(delta_mesh, box: float, worder: int, grad_order: int, lap_order: int,
                  deconv_pow: int, coeff: float = 1.0, delta_mesh2=None):
    """g_a = IFFT(S_a * FFT(delta)).  With delta_mesh2 (second, half-cell shifted grid) the
    two spectra are first combined as 1/2 [d1 + e^{-ik.s} d2] (O9 mode 1, reading R1)."""
    d = np.asarray(delta_mesh, dtype=np.float64)
    m = d.shape[0]
    dh = _rfftn(d)
    if delta_mesh2 is not None:
        dh = 0.5 * (dh + interlace_phase_3d(m) * _rfftn(np.asarray(delta_mesh2, dtype=np.float64)))
    S = force_symbols(m, box, worder, grad_order, lap_order, deconv_pow, coeff)
    return [_irfftn(Sa * dh, m) for Sa in S]


def poisson_force_vjp(force_cot, box, worder, grad_order, lap_order, deconv_pow, coeff=1.0,
                      interlace: bool = False):
    """Transpose of poisson_force: delta_cot = IFFT(sum_a conj(S_a) FFT(gbar_a)) (step V(iii));
    for the interlaced combination returns (cot of grid 1, cot of grid 2)."""
    m = np.asarray(force_cot[0]).shape[0]
    S = force_symbols(m, box, worder, grad_order, lap_order, deconv_pow, coeff)
    q = sum(np.conj(Sa) * _rfftn(np.asarray(g, dtype=np.float64)) for Sa, g in zip(S, force_cot))
    if not interlace:
        return _irfftn(q, m)
    return (_irfftn(0.5 * q, m), _irfftn(0.5 * np.conj(interlace_phase_3d(m)) * q, m))


# --------------------------------------------------------------------------------------
# Table 2, "Real" column (:231-242): the finite-difference gradient as a real-space stencil
# --------------------------------------------------------------------------------------
GRAD_STENCIL = {2: (2.0, (1.0,)), 4: (12.0, (8.0, -1.0)), 6: (60.0, (45.0, -9.0, 1.0))}
# order -> (denominator, coefficients of offsets +1, +2, ...; antisymmetric: offset -s carries -c_s)
# Table 2: 1/2 [-1 0 1], 1/12 [1 -8 0 8 -1], 1/60 [-1 9 -45 0 45 -9 1]


def fd_gradient_real(phi, box: float, order: int, axis: int):
    """d phi / d x_axis with the stencil printed in Table 2 for this order, periodic mesh."""
    phi = np.asarray(phi, dtype=np.float64)
    m = phi.shape[0]
    den, coef = GRAD_STENCIL[order]
    out = np.zeros_like(phi)
    for s_, c in enumerate(coef, start=1):
        out += c * (np.roll(phi, -s_, axis=axis) - np.roll(phi, s_, axis=axis))
    return out / (den * (box / m))


def poisson_potential(delta_mesh, box: float, worder: int, lap_order: int, deconv_pow: int,
                      coeff: float = 1.0, delta_mesh2=None):
    """phi = IFFT(coeff * delta_hat / Lap / W~^deconv_pow), phi_hat(0) = 0 (O6 without the gradient)."""
    d = np.asarray(delta_mesh, dtype=np.float64)
    m = d.shape[0]
    dh = _rfftn(d)
    if delta_mesh2 is not None:
        dh = 0.5 * (dh + interlace_phase_3d(m) * _rfftn(np.asarray(delta_mesh2, dtype=np.float64)))
    delta = box / m
    h = m // 2 + 1
    l1 = lap_symbol_1d(m, lap_order)
    lap = (l1[:, None, None] + l1[None, :, None] + l1[None, None, :h]) / delta ** 2
    lap[0, 0, 0] = 1.0
    green = coeff / lap
    green[0, 0, 0] = 0.0
    if deconv_pow:
        W1 = window_1d(m, worder)
        green = green / (W1[:, None, None] * W1[None, :, None] * W1[None, None, :h]) ** deconv_pow
    return _irfftn(green * dh, m)


def poisson_force_real_gradient(delta_mesh, box, worder, grad_order, lap_order, deconv_pow, coeff=1.0,
                                delta_mesh2=None):
    """g_a = -stencil_a(phi): the same operator as poisson_force for grad_order 2, 4, 6 (the Fourier
    symbols of Table 2 are the DFTs of these stencils), evaluated with ONE inverse FFT."""
    phi = poisson_potential(delta_mesh, box, worder, lap_order, deconv_pow, coeff, delta_mesh2)
    return [-fd_gradient_real(phi, box, grad_order, a) for a in range(3)]


# --------------------------------------------------------------------------------------
# Full force (O1-O9) and its reverse-mode VJP (step V; App. C rule table :949-955)
# --------------------------------------------------------------------------------------
def _half_cell(m, box):
    return np.full(3, 0.5 * box / m)


def density_contrast(rho, n_particles):
    """delta_j = (G/N) rho_j - 1 (Eq. 2.3 :92, equal masses :256)."""
    return rho * (rho.size / float(n_particles)) - 1.0


def force(pos, m, box, worder=2, interlace=0, grad_order=0, lap_order=0, deconv_pow=2,
          coeff=1.0, return_meshes=False):
    """Per-particle acceleration g_i = A(X_i), [N, 3] fp64.  interlace: 0 none, 1 Fourier-space
    combination of two grids (gather from the unshifted mesh), 2 average of two complete
    evaluations, the second on the half-cell shifted grid (reading R1)."""
    n = np.asarray(pos).shape[0]
    kw = dict(box=box, worder=worder, grad_order=grad_order, lap_order=lap_order,
              deconv_pow=deconv_pow, coeff=coeff)
    if interlace == 2:
        s = _half_cell(m, box)
        out = np.zeros((n, 3))
        for sh in (None, s):
            d = density_contrast(scatter(pos, m, box, worder, shift=sh), n)
            g = poisson_force(d, **kw)
            for a in range(3):
                out[:, a] += 0.5 * gather(g[a], pos, box, worder, shift=sh)
        return out
    d1 = density_contrast(scatter(pos, m, box, worder), n)
    d2 = None
    if interlace == 1:
        d2 = density_contrast(scatter(pos, m, box, worder, shift=_half_cell(m, box)), n)
    g = poisson_force(d1, delta_mesh2=d2, **kw)
    out = np.stack([gather(g[a], pos, box, worder) for a in range(3)], axis=1)
    if return_meshes:
        return out, d1, d2, g
    return out


def _force_vjp_single(pos, lam, m, box, worder, grad_order, lap_order, deconv_pow, coeff,
                      interlace, shift):
    n = pos.shape[0]
    kw = dict(box=box, worder=worder, grad_order=grad_order, lap_order=lap_order,
              deconv_pow=deconv_pow, coeff=coeff)
    d1 = density_contrast(scatter(pos, m, box, worder, shift=shift), n)
    d2 = None
    if interlace:
        d2 = density_contrast(scatter(pos, m, box, worder, shift=_half_cell(m, box)), n)
    g = poisson_force(d1, delta_mesh2=d2, **kw)
    xbar = np.zeros((n, 3))
    # (i) gather w.r.t. positions: grad-W gather weighted by the cotangent (Eq. C.12 :937)
    for a in range(3):
        for b in range(3):
            xbar[:, b] += lam[:, a] * gather(g[a], pos, box, worder, shift=shift, deriv_axis=b)
    # (ii) gather w.r.t. mesh: scatter of the cotangent values (Eq. C.10 :925)
    gbar = [scatter(pos, m, box, worder, weights=lam[:, a], shift=shift) for a in range(3)]
    # (iii) transposed k-space operator, then d(delta)/d(rho) = G/N
    dbar = poisson_force_vjp(gbar, interlace=bool(interlace), **kw)
    scale = m ** 3 / float(n)
    # (iv) scatter w.r.t. positions: grad-W gather of the cotangent mesh, w_i = 1 (Eq. C.6 :901)
    if interlace:
        for b in range(3):
            xbar[:, b] += scale * gather(dbar[0], pos, box, worder, deriv_axis=b)
            xbar[:, b] += scale * gather(dbar[1], pos, box, worder, shift=_half_cell(m, box), deriv_axis=b)
    else:
        for b in range(3):
            xbar[:, b] += scale * gather(dbar, pos, box, worder, shift=shift, deriv_axis=b)
    return xbar


def force_vjp(pos, lam, m, box, worder=2, interlace=0, grad_order=0, lap_order=0, deconv_pow=2,
              coeff=1.0):
    """X_bar = lam^T dF/dX, [N, 3] fp64, for the force of :func:`force`."""
    pos = np.asarray(pos)
    lam = np.asarray(lam).astype(np.float64)
    args = (m, box, worder, grad_order, lap_order, deconv_pow, coeff)
    if interlace == 2:
        return 0.5 * (_force_vjp_single(pos, lam, *args, 0, None)
                      + _force_vjp_single(pos, lam, *args, 0, _half_cell(m, box)))
    return _force_vjp_single(pos, lam, *args, interlace, None)
