"""Helpers shared by the GPU parity tests: error norms, the max-abs guard, records of the measured errors."""
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# A relative L2 norm hides a handful of wrong entries (one bad edge tile among 1e8 particles is invisible at
# 1e-5), so every comparison also bounds the largest single deviation against the rms of the reference.  fp32
# rounding gives max|d| / rms(ref) of a few 1e-6 for fields with a wide dynamic range; 1e-4 leaves room for the
# tails of 1e8 samples and still catches a wrong halo node (error ~ rms) by four orders of magnitude.
MAXABS_OVER_RMS = 1e-4


# The scatter of signed weights accumulates in 32-bit fixed point whose quantum is 2^-30 of the work item's bound
# B = sum_i |w_i| W_max^3 (up to 4096 particles): q ~ 4e-6 for unit-variance weights.  A node that receives n deposits
# carries a rounding error of q sqrt(n / 12); in a clump where hundreds of random-sign cotangents land on one node
# (the stage tests build one on purpose) that is ~3e-5 and up to ~3e-4 of the mesh rms over 1e5 nodes -- ten times
# what fp32 atomics would give there, invisible in L2 (measured 1.2e-6 .. 2.7e-6) and far below the 1e-5 VJP bar.
MAXABS_SIGNED_SCATTER = 1e-3


def es_edge_guard(beta: float) -> float:
    """The ES kernel jumps from e^-beta to 0 at the edge of its support, so whether a node exactly at the edge is
    touched depends on the rounding of the coordinate: a deviation of e^-beta of one mesh value is legitimate
    (R13; 1e-4 at w = 4, 1e-7 at w = 7)."""
    return MAXABS_OVER_RMS + 3.0 * float(np.exp(-beta))


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def max_over_rms(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    rms = float(np.sqrt(np.mean(b * b)))
    return float(np.abs(a - b).max() / max(rms, 1e-300))


def record_error(name: str, value: float, tol: float, maxabs: float = float("nan")):
    """Append a measured parity error to gpurun_out/parity_errors.tsv (kept beside the GPU test log):
    name, relative L2, its bar, max|d| / rms(ref)."""
    out = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_errors.tsv"), "a") as f:
            f.write(f"{name}\t{value:.3e}\t{tol:.1e}\t{maxabs:.3e}\n")
    except OSError:
        pass


def _test_id() -> str:
    cur = os.environ.get("PYTEST_CURRENT_TEST", "")
    return cur.split("::")[-1].split(" ")[0] if cur else "?"


def check(tag: str, got, ref, tol: float, maxabs_tol: float = MAXABS_OVER_RMS):
    """Assert relative L2 <= tol and max|got - ref| <= maxabs_tol * rms(ref); record both under the id of the
    running test + tag.  `got` may be a torch tensor."""
    if hasattr(got, "detach"):
        got = got.detach().cpu().numpy()
    name = f"{_test_id()}/{tag}" if tag else _test_id()
    e, mx = rel_l2(got, ref), max_over_rms(got, ref)
    record_error(name, e, tol, mx)
    assert e <= tol, f"{name}: relative L2 {e:.3e} > {tol:.1e}"
    assert mx <= maxabs_tol, f"{name}: max|d|/rms(ref) {mx:.3e} > {maxabs_tol:.1e}"
    return e
