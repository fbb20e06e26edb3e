"""ctypes binding of include/pmforce.h.  Argument marshalling only: every step runs in libpmforce.so."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))

EXPORTED_SYMBOLS = (
    "pm_create", "pm_destroy", "pm_strerror", "pm_last_error", "pm_mesh_dim", "pm_fine_dim", "pm_nufft_width",
    "pm_nufft_beta", "pm_bin", "pm_assign", "pm_assign_vjp", "pm_poisson_force", "pm_poisson_force_vjp",
    "pm_interp", "pm_interp_vjp", "nufft_spread", "nufft_spread_vjp", "nufft_poisson_force",
    "nufft_poisson_force_vjp", "nufft_interp", "nufft_interp_vjp", "pm_force", "pm_force_vjp", "pm_force_host",
    "pm_set_profiling", "pm_get_stage_ms", "pm_assign_jvp", "pm_interp_jvp", "pm_dkd_step", "pm_dkd_step_adjoint",
    "pm_power_spectrum", "pm_sheet_resample", "pm_smem_peak", "pm_mesh_power_noalloc", "pm_force_host_async",
)

STAGE_NAMES = ("bin", "assign", "fft_fwd", "kspace", "fft_inv", "interp", "vjp_scatter", "vjp_kspace", "vjp_gather",
               "gradient", "step")


FLAG_BIN_TWOPASS, FLAG_NO_XFUSE, FLAG_GRAD_REAL, FLAG_KERNEL_GRAD = 1, 2, 4, 8  # pm_params.flags


class PMError(RuntimeError):
    """A libpmforce call returned a negative pm_status."""


class _CParams(C.Structure):
    _fields_ = [
        ("m", C.c_int32), ("worder", C.c_int32), ("interlace", C.c_int32), ("deconv_pow", C.c_int32),
        ("grad_order", C.c_int32), ("lap_order", C.c_int32), ("method", C.c_int32), ("nufft_width", C.c_int32),
        ("box", C.c_double), ("coeff", C.c_double), ("nufft_sigma", C.c_double), ("nufft_eps", C.c_double),
        ("max_particles", C.c_int64), ("flags", C.c_int32), ("reserved", C.c_int32),
    ]


@dataclass
class PMParams:
    """Mirror of ``pm_params`` (names of Table 5)."""
    m: int
    box: float
    max_particles: int
    worder: int = 2
    interlace: int = 0
    deconv_pow: int = 2
    grad_order: int = 4
    lap_order: int = 0
    coeff: float = 1.0
    method: int = 0
    nufft_sigma: float = 2.0
    nufft_eps: float = 1e-6
    nufft_width: int = 0
    flags: int = 0  # FLAG_* bits (PM_FLAG_* of pmforce.h)

    def _c(self) -> _CParams:
        return _CParams(self.m, self.worder, self.interlace, self.deconv_pow, self.grad_order, self.lap_order,
                        self.method, self.nufft_width, self.box, self.coeff, self.nufft_sigma, self.nufft_eps,
                        self.max_particles, self.flags, 0)


_lib = None


def library_path() -> str:
    return os.path.join(_PKG, "libpmforce.so")


def load_library(build_if_missing: bool = False):
    """dlopen libpmforce.so and declare the prototypes.  Raises if it is absent: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        if not build_if_missing:
            raise RuntimeError(
                f"{path} not found: build it with `python -m paper_2510_05206_b200.build` "
                "(there is no CPU / PyTorch fallback for the force path)")
        from . import build as _build
        _build.build()
    lib = C.CDLL(path)
    vp, i64, f64p = C.c_void_p, C.c_int64, C.POINTER(C.c_double)
    sig = {
        "pm_create": (C.c_int, [C.POINTER(vp), C.POINTER(_CParams)]),
        "pm_destroy": (C.c_int, [vp]),
        "pm_strerror": (C.c_char_p, [C.c_int]),
        "pm_last_error": (C.c_char_p, [vp]),
        "pm_mesh_dim": (C.c_int32, [vp]),
        "pm_fine_dim": (C.c_int32, [vp]),
        "pm_nufft_width": (C.c_int32, [vp]),
        "pm_nufft_beta": (C.c_double, [vp]),
        "pm_bin": (C.c_int, [vp, vp, i64, vp]),
        "pm_assign": (C.c_int, [vp, vp, vp, i64, f64p, vp, vp]),
        "pm_assign_vjp": (C.c_int, [vp, vp, vp, i64, f64p, vp, vp, vp, vp]),
        "pm_poisson_force": (C.c_int, [vp, vp, vp, C.POINTER(vp), vp]),
        "pm_poisson_force_vjp": (C.c_int, [vp, C.POINTER(vp), vp, vp, vp]),
        "pm_interp": (C.c_int, [vp, C.POINTER(vp), C.c_int, vp, i64, f64p, vp, vp]),
        "pm_interp_vjp": (C.c_int, [vp, C.POINTER(vp), C.c_int, vp, i64, f64p, vp, C.POINTER(vp), vp, vp]),
        "nufft_spread": (C.c_int, [vp, vp, vp, i64, vp, vp]),
        "nufft_spread_vjp": (C.c_int, [vp, vp, vp, i64, vp, vp, vp, vp]),
        "nufft_poisson_force": (C.c_int, [vp, vp, i64, C.POINTER(vp), vp]),
        "nufft_poisson_force_vjp": (C.c_int, [vp, C.POINTER(vp), i64, vp, vp]),
        "nufft_interp": (C.c_int, [vp, C.POINTER(vp), C.c_int, vp, i64, vp, vp]),
        "nufft_interp_vjp": (C.c_int, [vp, C.POINTER(vp), C.c_int, vp, i64, vp, C.POINTER(vp), vp, vp]),
        "pm_force": (C.c_int, [vp, vp, i64, vp, vp]),
        "pm_force_vjp": (C.c_int, [vp, vp, i64, vp, vp, vp]),
        "pm_force_host": (C.c_int, [vp, vp, i64, vp, vp]),
        "pm_force_host_async": (C.c_int, [vp, vp, i64, vp, vp]),
        "pm_assign_jvp": (C.c_int, [vp, vp, vp, i64, f64p, vp, vp, vp, vp]),
        "pm_interp_jvp": (C.c_int, [vp, C.POINTER(vp), C.c_int, vp, i64, f64p, vp, C.POINTER(vp), vp, vp]),
        "pm_dkd_step": (C.c_int, [vp, vp, vp, i64, C.c_double, C.c_double, C.c_double, C.c_double, vp]),
        "pm_dkd_step_adjoint": (C.c_int, [vp, vp, vp, vp, vp, i64, C.c_double, C.c_double, C.c_double, C.c_double,
                                          vp, vp]),
        "pm_power_spectrum": (C.c_int, [vp, vp, i64, vp, i64, C.c_int, C.c_int, vp, vp, vp, vp]),
        "pm_sheet_resample": (C.c_int, [vp, vp, C.c_int32, C.c_int32, vp, vp]),
        "pm_mesh_power_noalloc": (C.c_int, [vp, vp, C.c_int32, C.c_double, C.c_double, C.c_int32, vp, vp, vp,
                                            C.c_char_p, C.c_int32, vp]),
        "pm_smem_peak": (C.c_int, [vp, C.c_int, C.POINTER(C.c_double), vp]),
        "pm_set_profiling": (C.c_int, [vp, C.c_int]),
        "pm_get_stage_ms": (C.c_int, [vp, C.POINTER(C.c_float), C.c_int, C.POINTER(i64)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


# ---- marshalling helpers -------------------------------------------------------------------------------
def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _dev(t, name: str, numel: int | None = None):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def _ptr_array(tensors, name: str, numel: int):
    if tensors is None:
        return None
    arr = (C.c_void_p * len(tensors))()
    for k, t in enumerate(tensors):
        arr[k] = _dev(t, f"{name}[{k}]", numel)
    return arr


def _shift(shift):
    if shift is None:
        return None
    return (C.c_double * 3)(*[float(s) for s in shift])


class PMContext:
    """Owns one ``pm_ctx*``."""

    def __init__(self, params: PMParams):
        lib = load_library()
        self.params = params
        self._h = C.c_void_p()
        cp = params._c()
        rc = lib.pm_create(C.byref(self._h), C.byref(cp))
        if rc != 0:
            why = lib.pm_last_error(None).decode()
            raise PMError(f"pm_create: {lib.pm_strerror(rc).decode()}: {why}")
        self.m = params.m
        self.mg = lib.pm_fine_dim(self._h) if params.method == 1 else params.m  # grid of the scatter / gather calls
        self.G = self.mg ** 3

    def check(self, rc: int, what: str):
        if rc != 0:
            lib = load_library()
            raise PMError(f"{what}: {lib.pm_strerror(rc).decode()}: {lib.pm_last_error(self._h).decode()}")

    @property
    def handle(self):
        if not self._h:
            raise PMError("context already destroyed")
        return self._h

    def close(self):
        if self._h:
            load_library().pm_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def nufft_width(self) -> int:
        return load_library().pm_nufft_width(self.handle)

    @property
    def nufft_beta(self) -> float:
        return load_library().pm_nufft_beta(self.handle)


def pm_create(params: PMParams) -> PMContext:
    return PMContext(params)


def pm_destroy(ctx: PMContext) -> None:
    ctx.close()


def _n(pos) -> int:
    if pos.dim() != 2 or pos.shape[1] != 3:
        raise ValueError("pos must have shape [N, 3]")
    return pos.shape[0]


def pm_bin(ctx, pos):
    ctx.check(load_library().pm_bin(ctx.handle, _dev(pos, "pos"), _n(pos), _stream()), "pm_bin")


def pm_assign(ctx, pos, w, mesh, shift=None):
    n = _n(pos)
    ctx.check(load_library().pm_assign(ctx.handle, _dev(pos, "pos"), _dev(w, "w", n), n, _shift(shift),
                                       _dev(mesh, "mesh", ctx.G), _stream()), "pm_assign")


def pm_assign_vjp(ctx, pos, w, mesh_cot, pos_cot=None, w_cot=None, shift=None):
    n = _n(pos)
    ctx.check(load_library().pm_assign_vjp(ctx.handle, _dev(pos, "pos"), _dev(w, "w", n), n, _shift(shift),
                                           _dev(mesh_cot, "mesh_cot", ctx.G), _dev(pos_cot, "pos_cot", 3 * n),
                                           _dev(w_cot, "w_cot", n), _stream()), "pm_assign_vjp")


def pm_poisson_force(ctx, delta_mesh, force_mesh, delta_mesh2=None):
    ctx.check(load_library().pm_poisson_force(ctx.handle, _dev(delta_mesh, "delta_mesh", ctx.G),
                                              _dev(delta_mesh2, "delta_mesh2", ctx.G),
                                              _ptr_array(force_mesh, "force_mesh", ctx.G), _stream()),
              "pm_poisson_force")


def pm_poisson_force_vjp(ctx, force_cot, delta_cot, delta_cot2=None):
    ctx.check(load_library().pm_poisson_force_vjp(ctx.handle, _ptr_array(force_cot, "force_cot", ctx.G),
                                                  _dev(delta_cot, "delta_cot", ctx.G),
                                                  _dev(delta_cot2, "delta_cot2", ctx.G), _stream()),
              "pm_poisson_force_vjp")


def pm_interp(ctx, mesh, pos, out, shift=None):
    n, ncomp = _n(pos), len(mesh)
    ctx.check(load_library().pm_interp(ctx.handle, _ptr_array(mesh, "mesh", ctx.G), ncomp, _dev(pos, "pos"), n,
                                       _shift(shift), _dev(out, "out", n * ncomp), _stream()), "pm_interp")


def pm_interp_vjp(ctx, mesh, pos, out_cot, mesh_cot=None, pos_cot=None, shift=None):
    n = _n(pos)
    ncomp = out_cot.shape[1] if out_cot.dim() == 2 else 1
    ctx.check(load_library().pm_interp_vjp(ctx.handle, _ptr_array(mesh, "mesh", ctx.G), ncomp, _dev(pos, "pos"), n,
                                           _shift(shift), _dev(out_cot, "out_cot", n * ncomp),
                                           _ptr_array(mesh_cot, "mesh_cot", ctx.G), _dev(pos_cot, "pos_cot", 3 * n),
                                           _stream()), "pm_interp_vjp")


def nufft_spread(ctx, pos, c, fine):
    n = _n(pos)
    ctx.check(load_library().nufft_spread(ctx.handle, _dev(pos, "pos"), _dev(c, "c", n), n,
                                          _dev(fine, "fine", ctx.G), _stream()), "nufft_spread")


def nufft_spread_vjp(ctx, pos, c, fine_cot, pos_cot=None, c_cot=None):
    n = _n(pos)
    ctx.check(load_library().nufft_spread_vjp(ctx.handle, _dev(pos, "pos"), _dev(c, "c", n), n,
                                              _dev(fine_cot, "fine_cot", ctx.G), _dev(pos_cot, "pos_cot", 3 * n),
                                              _dev(c_cot, "c_cot", n), _stream()), "nufft_spread_vjp")


def nufft_poisson_force(ctx, fine, n_particles, force_fine):
    ctx.check(load_library().nufft_poisson_force(ctx.handle, _dev(fine, "fine", ctx.G), int(n_particles),
                                                 _ptr_array(force_fine, "force_fine", ctx.G), _stream()),
              "nufft_poisson_force")


def nufft_poisson_force_vjp(ctx, force_cot, n_particles, fine_cot):
    ctx.check(load_library().nufft_poisson_force_vjp(ctx.handle, _ptr_array(force_cot, "force_cot", ctx.G),
                                                     int(n_particles), _dev(fine_cot, "fine_cot", ctx.G),
                                                     _stream()), "nufft_poisson_force_vjp")


def nufft_interp(ctx, fine, pos, out):
    n, ncomp = _n(pos), len(fine)
    ctx.check(load_library().nufft_interp(ctx.handle, _ptr_array(fine, "fine", ctx.G), ncomp, _dev(pos, "pos"), n,
                                          _dev(out, "out", n * ncomp), _stream()), "nufft_interp")


def nufft_interp_vjp(ctx, fine, pos, out_cot, fine_cot=None, pos_cot=None):
    n = _n(pos)
    ncomp = out_cot.shape[1] if out_cot.dim() == 2 else 1
    ctx.check(load_library().nufft_interp_vjp(ctx.handle, _ptr_array(fine, "fine", ctx.G), ncomp, _dev(pos, "pos"),
                                              n, _dev(out_cot, "out_cot", n * ncomp),
                                              _ptr_array(fine_cot, "fine_cot", ctx.G),
                                              _dev(pos_cot, "pos_cot", 3 * n), _stream()), "nufft_interp_vjp")


def pm_force(ctx, pos, force):
    n = _n(pos)
    ctx.check(load_library().pm_force(ctx.handle, _dev(pos, "pos"), n, _dev(force, "force", 3 * n), _stream()),
              "pm_force")


def pm_force_vjp(ctx, pos, force_cot, pos_cot):
    n = _n(pos)
    ctx.check(load_library().pm_force_vjp(ctx.handle, _dev(pos, "pos"), n, _dev(force_cot, "force_cot", 3 * n),
                                          _dev(pos_cot, "pos_cot", 3 * n), _stream()), "pm_force_vjp")


def pm_assign_jvp(ctx, pos, w, mesh_tan, pos_tan=None, w_tan=None, shift=None):
    n = _n(pos)
    ctx.check(load_library().pm_assign_jvp(ctx.handle, _dev(pos, "pos"), _dev(w, "w", n), n, _shift(shift),
                                           _dev(pos_tan, "pos_tan", 3 * n), _dev(w_tan, "w_tan", n),
                                           _dev(mesh_tan, "mesh_tan", ctx.G), _stream()), "pm_assign_jvp")


def pm_interp_jvp(ctx, mesh, pos, out_tan, pos_tan=None, mesh_tan=None, shift=None):
    n, ncomp = _n(pos), len(mesh)
    ctx.check(load_library().pm_interp_jvp(ctx.handle, _ptr_array(mesh, "mesh", ctx.G), ncomp, _dev(pos, "pos"), n,
                                           _shift(shift), _dev(pos_tan, "pos_tan", 3 * n),
                                           _ptr_array(mesh_tan, "mesh_tan", ctx.G),
                                           _dev(out_tan, "out_tan", n * ncomp), _stream()), "pm_interp_jvp")


def _dev64(t, name: str, numel: int):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float64 CUDA tensor")
    if t.numel() != numel:
        raise ValueError(f"{name} has {t.numel()} elements, expected {numel}")
    return t.data_ptr()


def pm_dkd_step(ctx, pos, vel, tau1, tau2, alpha, beta):
    """In place: pos, vel [N,3] (Eq. 2.14a-c)."""
    n = _n(pos)
    ctx.check(load_library().pm_dkd_step(ctx.handle, _dev(pos, "pos"), _dev(vel, "vel", 3 * n), n, float(tau1),
                                         float(tau2), float(alpha), float(beta), _stream()), "pm_dkd_step")


def pm_dkd_step_adjoint(ctx, pos, vel, pos_adj, vel_adj, tau1, tau2, alpha, beta, scalar_adj=None):
    """In place: pos, vel, pos_adj, vel_adj [N,3] (Table 3); scalar_adj: float64 CUDA tensor [4] or None."""
    n = _n(pos)
    ctx.check(load_library().pm_dkd_step_adjoint(ctx.handle, _dev(pos, "pos"), _dev(vel, "vel", 3 * n),
                                                 _dev(pos_adj, "pos_adj", 3 * n), _dev(vel_adj, "vel_adj", 3 * n), n,
                                                 float(tau1), float(tau2), float(alpha), float(beta),
                                                 _dev64(scalar_adj, "scalar_adj", 4), _stream()),
              "pm_dkd_step_adjoint")


def pm_power_spectrum(ctx, pos, k_mean, power, n_modes, pos2=None, deconvolve=True):
    """k_mean, power, n_modes: float64 CUDA tensors [nbins]."""
    nbins = k_mean.numel()
    ctx.check(load_library().pm_power_spectrum(ctx.handle, _dev(pos, "pos"), _n(pos), _dev(pos2, "pos2"),
                                               _n(pos2) if pos2 is not None else 0, int(bool(deconvolve)), nbins,
                                               _dev64(k_mean, "k_mean", nbins), _dev64(power, "power", nbins),
                                               _dev64(n_modes, "n_modes", nbins), _stream()), "pm_power_spectrum")


NOALLOC_MAX_BINS = 1024  # PM_NOALLOC_MAX_BINS of include/pmforce.h


def pm_mesh_power_noalloc(spec_a, m, box, norm, k_mean, power, n_modes, spec_b=None):
    """Shell-binned (cross-)power of half-complex spectra the caller holds; allocates nothing (no ctx).

    spec_a / spec_b: contiguous float32 CUDA tensors [m, m, m//2 + 1, 2] (``torch.view_as_real`` of a complex64
    ``rfftn``); k_mean, power, n_modes: float64 CUDA tensors [nbins], nbins <= NOALLOC_MAX_BINS."""
    nbins = k_mean.numel()
    ncomplex = m * m * (m // 2 + 1)
    err = C.create_string_buffer(256)
    rc = load_library().pm_mesh_power_noalloc(
        _dev(spec_a, "spec_a", 2 * ncomplex), _dev(spec_b, "spec_b", 2 * ncomplex), int(m), float(box), float(norm),
        nbins, _dev64(k_mean, "k_mean", nbins), _dev64(power, "power", nbins), _dev64(n_modes, "n_modes", nbins),
        err, len(err), _stream())
    if rc != 0:
        raise PMError(f"pm_mesh_power_noalloc: {err.value.decode() or rc}")


def pm_sheet_resample(ctx, pos, n_p, r, pos_out):
    if _n(pos) != n_p ** 3 or _n(pos_out) != (n_p * r) ** 3:
        raise ValueError("pos must hold n_p^3 and pos_out (r n_p)^3 particles")
    ctx.check(load_library().pm_sheet_resample(ctx.handle, _dev(pos, "pos"), int(n_p), int(r),
                                               _dev(pos_out, "pos_out"), _stream()), "pm_sheet_resample")


def pm_force_host(ctx, pos_host, force_host):
    """pos_host / force_host: contiguous float32 CPU tensors [N,3] (pinned for asynchronous copies)."""
    for t, name in ((pos_host, "pos_host"), (force_host, "force_host")):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
            raise TypeError(f"{name} must be a contiguous float32 CPU tensor")
    n = _n(pos_host)
    if force_host.numel() != 3 * n:
        raise ValueError("force_host must have 3*N elements")
    ctx.check(load_library().pm_force_host(ctx.handle, pos_host.data_ptr(), n, force_host.data_ptr(), _stream()),
              "pm_force_host")


def pm_force_host_async(ctx, pos_host, force_host):
    """pm_force_host without the final synchronisation (enqueued on torch's current stream): the pinned host tensors
    must stay alive and untouched until that stream has been synchronised."""
    for t, name in ((pos_host, "pos_host"), (force_host, "force_host")):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
            raise TypeError(f"{name} must be a contiguous float32 CPU tensor")
    n = _n(pos_host)
    if force_host.numel() != 3 * n:
        raise ValueError("force_host must have 3*N elements")
    ctx.check(load_library().pm_force_host_async(ctx.handle, pos_host.data_ptr(), n, force_host.data_ptr(), _stream()),
              "pm_force_host_async")


def pm_smem_peak(ctx, kind: int) -> float:
    """Measured shared-memory lane operations per second (0 loads, 1 integer atomics, 2 128-bit loads)."""
    v = C.c_double(0.0)
    ctx.check(load_library().pm_smem_peak(ctx.handle, int(kind), C.byref(v), _stream()), "pm_smem_peak")
    return float(v.value)


def pm_set_profiling(ctx, enable: bool):
    ctx.check(load_library().pm_set_profiling(ctx.handle, int(bool(enable))), "pm_set_profiling")


def pm_get_stage_ms(ctx):
    """(dict stage -> ms, kernel launches of libpmforce in the last profiled call)."""
    ms = (C.c_float * len(STAGE_NAMES))()
    nl = C.c_int64(0)
    ctx.check(load_library().pm_get_stage_ms(ctx.handle, ms, len(STAGE_NAMES), C.byref(nl)), "pm_get_stage_ms")
    return {k: float(ms[i]) for i, k in enumerate(STAGE_NAMES)}, int(nl.value)
