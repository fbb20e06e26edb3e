"""Pins of the DKD-step oracle (oracle/dkd_oracle.py) against what the paper and the mathematics fix (no GPU)."""
import numpy as np
import pytest

from oracle import dkd_oracle as dk
from oracle import pm_oracle as po
from pm_inputs import uniform_random


def test_harmonic_oscillator_verlet_recurrence():
    """Eq. 2.14 with alpha = 1, beta = tau, tau_1 = tau_2 = tau/2 is the textbook leapfrog; for A(x) = -w^2 x its
    positions obey the three-term Verlet recurrence x_{n+1} - (2 - w^2 tau^2) x_n + x_{n-1} = 0 and the
    discrete frequency cos(theta) = 1 - w^2 tau^2 / 2."""
    w2, tau = 1.7, 0.05
    X = np.array([[0.3, -1.0, 2.0]])
    V = np.array([[1.0, 0.5, -0.25]])
    xs = [X.copy()]
    for _ in range(60):
        X, V = dk.dkd_step(X, V, tau / 2, tau / 2, 1.0, tau, lambda x: -w2 * x, None, state_dtype=np.float64)
        xs.append(X.copy())
    xs = np.array(xs)[:, 0, :]
    rec = xs[2:] - (2.0 - w2 * tau * tau) * xs[1:-1] + xs[:-2]
    assert np.abs(rec).max() < 1e-13
    # closed form: x_n = x_0 cos(n theta) + c sin(n theta); c from x_1
    th = np.arccos(1.0 - 0.5 * w2 * tau * tau)
    n = np.arange(xs.shape[0])[:, None]
    c = (xs[1] - xs[0] * np.cos(th)) / np.sin(th)
    assert np.abs(xs - (xs[0] * np.cos(n * th) + c * np.sin(n * th))).max() < 1e-11


def test_kick_coefficients_enter_as_eq_2_14b():
    """V^{n+1} = alpha V^n + beta A(X^{n+1/2}) with the acceleration taken AFTER the first drift (:185)."""
    X = np.array([[1.0, 2.0, 3.0]])
    V = np.array([[0.5, -0.5, 0.25]])
    seen = []

    def acc(x):
        seen.append(np.array(x))
        return np.full_like(x, 2.0)

    Xn, Vn = dk.dkd_step(X, V, 0.1, 0.3, 0.9, 0.4, acc, None, state_dtype=np.float64)
    assert np.allclose(seen[0], [[1.05, 1.95, 3.025]], atol=1e-15)
    assert np.allclose(Vn, [[0.45 + 0.8, -0.45 + 0.8, 0.225 + 0.8]], atol=1e-15)
    assert np.allclose(Xn, seen[0] + 0.3 * Vn, atol=1e-15)


def _pm_callables(m, box, worder):
    kw = dict(worder=worder, interlace=0, grad_order=4, lap_order=0, deconv_pow=2, coeff=0.8)
    return (lambda x: po.force(x, m, box, **kw)), (lambda x, lam: po.force_vjp(x, lam, m, box, **kw))


def test_time_reversibility():
    """Table 3's primal rows undo Eq. 2.14 ("propagate backwards on the exact same trajectory", :309)."""
    m, box = 8, 8.0
    acc, vjp = _pm_callables(m, box, 3)
    X0 = uniform_random(60, box, 5).astype(np.float64)
    V0 = np.random.default_rng(6).standard_normal((60, 3)) * 0.3
    X, V = X0, V0
    coefs = [(0.11, 0.09, 0.93, 0.21), (0.07, 0.13, 1.04, 0.17)]
    for c in coefs:
        X, V = dk.dkd_step(X, V, *c, acc, box, state_dtype=np.float64)
    z = np.zeros_like(X)
    for c in reversed(coefs):
        X, V, _, _, _ = dk.dkd_step_adjoint(X, V, z, z, *c, acc, vjp, box, state_dtype=np.float64)
    assert np.abs(X - X0).max() < 1e-12 and np.abs(V - V0).max() < 1e-12


@pytest.mark.parametrize("worder", (3, 4))
def test_adjoint_matches_finite_differences(worder):
    """The paper's own check (:425-445): gradient of a scalar loss through the time integration from the
    adjoint method vs an independent derivative (here central differences), w.r.t. initial positions and
    velocities and w.r.t. the temporal coefficients tau_1, tau_2, alpha, beta of every step (Table 3)."""
    m, box, n = 8, 8.0, 40
    acc, vjp = _pm_callables(m, box, worder)
    rng = np.random.default_rng(10 + worder)
    X0 = uniform_random(n, box, 7).astype(np.float64)
    V0 = rng.standard_normal((n, 3)) * 0.3
    cX, cV = rng.standard_normal((n, 3)), rng.standard_normal((n, 3))
    coefs = [[0.11, 0.09, 0.93, 0.21], [0.07, 0.13, 1.04, 0.17], [0.10, 0.10, 0.97, 0.19]]

    def loss(X, V, cf):
        for c in cf:
            X, V = dk.dkd_step(X, V, *c, acc, box, state_dtype=np.float64)
        return float(np.sum(cX * X) + np.sum(cV * V))

    X, V = X0, V0
    for c in coefs:
        X, V = dk.dkd_step(X, V, *c, acc, box, state_dtype=np.float64)
    Xs, Vs = cX.copy(), cV.copy()
    adjs = []
    for c in reversed(coefs):
        X, V, Xs, Vs, a = dk.dkd_step_adjoint(X, V, Xs, Vs, *c, acc, vjp, box, state_dtype=np.float64)
        adjs.append(a)
    adjs = adjs[::-1]
    h = 1e-6
    for (i, a) in ((0, 0), (3, 1), (17, 2), (31, 0)):
        for arr, grad in ((X0, Xs), (V0, Vs)):
            ap, am = arr.copy(), arr.copy()
            ap[i, a] += h
            am[i, a] -= h
            fd = (loss(ap, V0, coefs) - loss(am, V0, coefs)) / (2 * h) if arr is X0 else \
                 (loss(X0, ap, coefs) - loss(X0, am, coefs)) / (2 * h)
            assert abs(fd - grad[i, a]) < 2e-7 * max(1.0, abs(fd)), (i, a, fd, grad[i, a])
    for s in range(len(coefs)):
        for k, name in enumerate(("tau1", "tau2", "alpha", "beta")):
            cp = [list(c) for c in coefs]
            cm = [list(c) for c in coefs]
            cp[s][k] += h
            cm[s][k] -= h
            fd = (loss(X0, V0, cp) - loss(X0, V0, cm)) / (2 * h)
            assert abs(fd - adjs[s][name]) < 2e-7 * max(1.0, abs(fd)), (s, name, fd, adjs[s][name])


def test_fp32_state_drift_arithmetic():
    """Reading R18: the fp32 drift wraps into [0, L) and keeps fp32 bits; a value that rounds to L becomes 0."""
    box = 1000.0
    X = np.array([[999.99994, 0.0, 500.0], [1e-6, 999.0, 3.0]], dtype=np.float32)
    V = np.array([[1.0, -1.0, 0.0], [-1.0, 2.0, 1.9e3]], dtype=np.float32)
    Y = dk.drift(X, V, 0.5, box, np.float32)
    assert Y.dtype == np.float32 and (Y >= 0).all() and (Y < np.float32(box)).all()
    ref = np.mod(X.astype(np.float64) + 0.5 * V.astype(np.float64), box)
    d = np.abs(Y - ref)
    d = np.minimum(d, box - d)
    assert d.max() < 2e-4  # a few fp32 ulps of L
