"""Oracle of the drift-kick-drift step and of its backward-in-time adjoint step (TEST INFRASTRUCTURE).

Follows PAPER.md Sec. 2.4 Eq. 2.14a-c (:179-183) for the forward step and Sec. 2.7 Table 3 (:344-358) row by
row, in the table's order, for the backward step.  The acceleration A(X) and its VJP lam^T dA/dX are passed
in as callables (``pm_oracle.force`` / ``pm_oracle.force_vjp`` in the tests); alpha, beta, tau_1, tau_2 are
plain scalars (the cosmology that produces them, Eq. 2.15-2.17, is out of scope).

Reading R18 -- precision of the state.  The paper's arrays are single precision by default
(:445 "single precision ... is the default").  ``state_dtype = numpy.float32`` stores X, V, X*, V* in fp32
between operations exactly like the CUDA path does, with this arithmetic for a drift (every operation
rounded to fp32, no fused multiply-add, so that both sides produce the same bits):

    x' = x + (tau * v);   if x' < 0: x' = x' + L;   if x' >= L: x' = x' - L

(a particle moves less than one box length per drift; a value that the addition rounds up to L is taken to 0 by
the subtraction), so the acceleration is evaluated at identical fp32 positions on both sides (a force evaluated at positions
that differ by one fp32 ulp of L differs by ~1e-5 relative).  Kicks and the adjoint
updates are evaluated in fp64 from the fp32 state and rounded once.  ``state_dtype = numpy.float64`` keeps
everything in fp64 and does not wrap (used by the pins: time reversibility, finite differences).

Pins (tests/test_oracle_dkd.py): the three-term Verlet recurrence of a harmonic oscillator; time
reversibility (Table 3's primal rows invert Eq. 2.14 to rounding, :309); the adjoint state and the four
scalar adjoints against central finite differences of a scalar loss through three steps (the paper's own
check of its adjoint method, :425-445).
"""
from __future__ import annotations

import numpy as np


def wrap_fp32(x, box):
    """Periodic wrap of an fp32 array into [0, L) with fp32 operations only (see module docstring)."""
    L = np.float32(box)
    y = np.asarray(x, dtype=np.float32)
    y = np.where(y < np.float32(0), y + L, y)
    y = np.where(y >= L, y - L, y)
    return y.astype(np.float32)


def drift(X, V, tau, box, state_dtype):
    """X + tau V (Eq. 2.14a / 2.14c; Table 3 'Primal drift' with -tau)."""
    if state_dtype == np.float32:
        X = np.asarray(X, dtype=np.float32)
        V = np.asarray(V, dtype=np.float32)
        t = np.float32(tau)
        return wrap_fp32(X + t * V, box)
    return np.asarray(X, dtype=np.float64) + float(tau) * np.asarray(V, dtype=np.float64)


def _store(a, state_dtype):
    return np.asarray(a, dtype=np.float64).astype(state_dtype)


def dkd_step(X, V, tau1, tau2, alpha, beta, accel, box, state_dtype=np.float32):
    """One step of Eq. 2.14: returns (X^{n+1}, V^{n+1})."""
    Xh = drift(X, V, tau1, box, state_dtype)                                   # (2.14a)
    A = np.asarray(accel(Xh), dtype=np.float64)
    Vn = _store(float(alpha) * np.asarray(V, dtype=np.float64) + float(beta) * A, state_dtype)  # (2.14b)
    Xn = drift(Xh, Vn, tau2, box, state_dtype)                                 # (2.14c)
    return Xn, Vn


def dkd_step_adjoint(X, V, Xs, Vs, tau1, tau2, alpha, beta, accel, accel_vjp, box,
                     state_dtype=np.float32):
    """One backward-in-time step, Table 3 (:344-358), rows in the table's order.

    In: (X^n, V^n, X*^n, V*^n).  Out: (X^{n-1}, V^{n-1}, X*^{n-1}, V*^{n-1}) and the scalar adjoints
    {tau1, tau2, alpha, beta} of this step.  accel_vjp(X, lam) = lam^T dA/dX (:338 'jax.vjp')."""
    f64 = lambda a: np.asarray(a, dtype=np.float64)  # noqa: E731
    adj = {}
    # Primal drift            X^{n-1/2} = X^n - tau_2 V^n
    Xh = drift(X, V, -tau2, box, state_dtype)
    # Adjoint drift           V*^{n-1/2} = V*^n + tau_2 X*^n
    Vsh = _store(f64(Vs) + float(tau2) * f64(Xs), state_dtype)
    # Adjoint for tau_2       tau_2* = X*^n . V^n
    adj["tau2"] = float(np.sum(f64(Xs) * f64(V)))
    # Primal kick             V^{n-1} = (V^n - beta A(X^{n-1/2})) / alpha
    A = f64(accel(Xh))
    Vp = _store((f64(V) - float(beta) * A) / float(alpha), state_dtype)
    # Adjoint kick            X*^{n-1} = X*^n + beta V*^{n-1/2} . grad_X A(X^{n-1/2})
    Xsp = _store(f64(Xs) + float(beta) * f64(accel_vjp(Xh, f64(Vsh))), state_dtype)
    # Rescale adjoint velocity V*^{n-1/2,K} = alpha V*^{n-1/2}
    VsK = _store(float(alpha) * f64(Vsh), state_dtype)
    # Adjoint for alpha       alpha* = V*^{n-1/2} . V^{n-1}
    #   (Table 3 prints V^n here; d V^n / d alpha = V^{n-1} by Eq. 2.14b, and the finite-difference pin
    #    decides for V^{n-1}: reading R19)
    adj["alpha"] = float(np.sum(f64(Vsh) * f64(Vp)))
    # Adjoint for beta        beta* = V*^{n-1/2} . A(X^{n-1/2})
    adj["beta"] = float(np.sum(f64(Vsh) * A))
    # Primal drift            X^{n-1} = X^{n-1/2} - tau_1 V^{n-1}
    Xp = drift(Xh, Vp, -tau1, box, state_dtype)
    # Adjoint drift           V*^{n-1} = V*^{n-1/2,K} + tau_1 X*^{n-1}
    Vsp = _store(f64(VsK) + float(tau1) * f64(Xsp), state_dtype)
    # Adjoint for tau_1       tau_1* = X*^{n-1} . V^{n-1}
    adj["tau1"] = float(np.sum(f64(Xsp) * f64(Vp)))
    return Xp, Vp, Xsp, Vsp, adj
