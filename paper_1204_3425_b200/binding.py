"""Thin ctypes binding of libhubbard_b200 (include/hubbard.h).  Argument
marshalling only: every step of the path runs in the library's CUDA kernels.
Function names are those of the C ABI.  There is no fallback: if the library
cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

HUBBARD_F32, HUBBARD_F64 = 0, 1
VARIANT_AUTO, VARIANT_PAPER, VARIANT_TWOSWEEP, VARIANT_GATHER, VARIANT_PERSIST = 0, 1, 2, 3, 4
ERR_TOO_LARGE = -7
NOALLOC_CHUNK, NOALLOC_MAX_N = 32768, 8192 * 32768          # include/hubbard.h: lanczos_shard_update_noalloc
N_KCLASS = 6
KCLASS_NAMES = ("hv_paper", "row_sweep", "col_sweep", "vec_sweep", "scalar", "setup")

ABI_SYMBOLS = (
    "hubbard_create", "hubbard_create_host", "hubbard_destroy", "hubbard_dims", "hubbard_set_U",
    "hubbard_set_variant", "hubbard_apply", "lanczos_run", "lanczos_run_until", "lanczos_ground_state",
    "lanczos_ground_vector", "lanczos_propagate", "lanczos_propagate_complex", "lanczos_expm_e1", "lanczos_set_tau", "hubbard_apply_host",
    "lanczos_run_host", "hubbard_get_basis", "hubbard_get_hops", "hubbard_get_gather_table", "lanczos_ground_energy",
    "hubbard_profile", "hubbard_kernel_times", "hubbard_launch_count", "hubbard_last_cuda_error",
    "hubbard_strerror", "hubbard_debug_set", "hubbard_debug_get", "hubbard_apply_rows", "lanczos_shard_update",
    "lanczos_shard_update_noalloc",
)


def _load() -> C.CDLL:
    path: Path = _build.LIB
    try:
        path = _build.build()            # no-op when the library is newer than its sources
    except Exception:
        if not path.exists():            # no usable library and no compiler: there is no fallback
            raise
    lib = C.CDLL(str(path))
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    P = C.POINTER
    lib.hubbard_create.argtypes = [P(vp), i32, i32, i32, P(C.c_int32), i32, dbl, dbl, i32]
    lib.hubbard_create_host.argtypes = lib.hubbard_create.argtypes
    lib.hubbard_destroy.argtypes = [vp]
    lib.hubbard_destroy.restype = None
    lib.hubbard_dims.argtypes = [vp, P(i64), P(i64)]
    lib.hubbard_set_U.argtypes = [vp, dbl]
    lib.hubbard_set_variant.argtypes = [vp, i32]
    lib.hubbard_apply.argtypes = [vp, vp, vp, vp]
    lib.lanczos_run.argtypes = [vp, vp, i32, P(dbl), P(dbl), P(i32), vp]
    lib.lanczos_set_tau.argtypes = [vp, dbl]
    lib.lanczos_run_until.argtypes = [vp, vp, i32, i32, dbl, P(dbl), P(dbl), P(i32), P(dbl), vp]
    lib.lanczos_ground_state.argtypes = [vp, vp, i32, vp, P(dbl), P(i32), vp]
    lib.lanczos_ground_vector.argtypes = [P(dbl), P(dbl), i32, P(dbl), P(dbl)]
    lib.lanczos_propagate.argtypes = [vp, vp, i32, dbl, dbl, vp, vp, P(i32), vp]
    lib.lanczos_propagate_complex.argtypes = [vp, vp, vp, i32, dbl, dbl, vp, vp, P(i32), vp]
    lib.lanczos_expm_e1.argtypes = [P(dbl), P(dbl), i32, dbl, dbl, P(dbl), P(dbl)]
    lib.hubbard_apply_host.argtypes = [vp, vp, vp, vp]
    lib.lanczos_run_host.argtypes = [vp, vp, i32, P(dbl), P(dbl), P(i32), vp]
    lib.hubbard_get_basis.argtypes = [vp, i32, P(C.c_uint32)]
    lib.hubbard_get_hops.argtypes = [vp, i32, P(i32), P(C.c_int32), P(dbl)]
    lib.hubbard_get_gather_table.argtypes = [vp, i32, i32, i32, i32, P(i32), P(i64), P(C.c_uint32), P(C.c_int32),
                                             P(C.c_uint16), P(C.c_int32), P(i64), P(i64)]
    lib.lanczos_ground_energy.argtypes = [P(dbl), P(dbl), i32, P(dbl)]
    lib.hubbard_profile.argtypes = [vp, i32]
    lib.hubbard_kernel_times.argtypes = [vp, P(i64), P(dbl)]
    lib.hubbard_launch_count.argtypes = [vp]
    lib.hubbard_launch_count.restype = i64
    lib.hubbard_last_cuda_error.argtypes = [vp]
    lib.hubbard_apply_rows.argtypes = [vp, vp, vp, i64, i64, vp]
    lib.lanczos_shard_update.argtypes = [vp, i32, vp, vp, vp, i64, dbl, vp, vp]
    lib.lanczos_shard_update_noalloc.argtypes = lib.lanczos_shard_update.argtypes
    lib.hubbard_debug_set.argtypes = [vp, C.c_char_p, i32]
    lib.hubbard_debug_get.argtypes = [vp, C.c_char_p, P(i32)]
    lib.hubbard_strerror.argtypes = [i32]
    lib.hubbard_strerror.restype = C.c_char_p
    return lib


lib = _load()
LIB_PATH = str(_build.LIB)


class HubbardError(RuntimeError):
    def __init__(self, code: int, what: str, cuda: int = 0):
        self.code = code
        msg = f"{what}: {lib.hubbard_strerror(code).decode()} ({code})"
        if cuda:
            msg += f" [cudaError {cuda}]"
        super().__init__(msg)


def _check(code: int, what: str, handle=None):
    if code != 0:
        raise HubbardError(code, what, lib.hubbard_last_cuda_error(handle) if handle else 0)


def _bonds_array(bonds) -> np.ndarray:
    return np.ascontiguousarray(np.array(list(bonds), dtype=np.int32).reshape(-1, 2))


def _dtype_code(dtype) -> int:
    s = str(dtype)
    if s in ("f32", "float32", "torch.float32", "0"):
        return HUBBARD_F32
    if s in ("f64", "float64", "torch.float64", "1"):
        return HUBBARD_F64
    raise ValueError(f"dtype {dtype!r}: use 'f32' or 'f64'")


def _dptr(t) -> int:
    """Device pointer of a contiguous CUDA torch tensor."""
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


class Model:
    """Owner of a `hubbard_model*`; methods are the ABI calls of the same name."""

    def __init__(self, n_sites, n_up, n_dn, bonds, t, U, dtype="f64", host_only=False):
        self._h = C.c_void_p()
        b = _bonds_array(bonds)
        fn = lib.hubbard_create_host if host_only else lib.hubbard_create
        code = fn(C.byref(self._h), n_sites, n_up, n_dn, b.ctypes.data_as(C.POINTER(C.c_int32)), len(b),
                  float(t), float(U), _dtype_code(dtype))
        _check(code, "hubbard_create_host" if host_only else "hubbard_create")
        self.dtype_code = _dtype_code(dtype)
        du, dd = C.c_int64(), C.c_int64()
        _check(lib.hubbard_dims(self._h, C.byref(du), C.byref(dd)), "hubbard_dims")
        self.dim_up, self.dim_dn = du.value, dd.value
        self.dim = self.dim_up * self.dim_dn

    # -- lifetime
    def hubbard_destroy(self):
        if self._h:
            lib.hubbard_destroy(self._h)
            self._h = C.c_void_p()

    close = hubbard_destroy

    def __del__(self):
        try:
            self.hubbard_destroy()
        except Exception:
            pass

    # -- configuration
    def hubbard_set_U(self, U):
        _check(lib.hubbard_set_U(self._h, float(U)), "hubbard_set_U")

    def hubbard_set_variant(self, variant):
        _check(lib.hubbard_set_variant(self._h, int(variant)), "hubbard_set_variant")

    def lanczos_set_tau(self, tau):
        _check(lib.lanczos_set_tau(self._h, float(tau)), "lanczos_set_tau")

    def hubbard_debug_set(self, key, value):
        _check(lib.hubbard_debug_set(self._h, key.encode(), int(value)), f"hubbard_debug_set({key})", self._h)

    def hubbard_debug_get(self, key):
        v = C.c_int(0)
        _check(lib.hubbard_debug_get(self._h, key.encode(), C.byref(v)), f"hubbard_debug_get({key})")
        return v.value

    # -- hot path, device buffers (torch CUDA tensors)
    def hubbard_apply(self, x, y, stream=None):
        _check(lib.hubbard_apply(self._h, _dptr(x), _dptr(y), _stream(stream)), "hubbard_apply", self._h)
        return y

    def lanczos_run(self, v0, iters, stream=None):
        alpha = np.zeros(max(iters, 1))
        beta = np.zeros(max(iters, 1))
        done = C.c_int(0)
        dp = C.POINTER(C.c_double)
        _check(lib.lanczos_run(self._h, _dptr(v0), iters, alpha.ctypes.data_as(dp), beta.ctypes.data_as(dp),
                               C.byref(done), _stream(stream)), "lanczos_run", self._h)
        return alpha[:done.value].copy(), beta[:done.value].copy()

    def lanczos_run_until(self, v0, max_iters, check_every=10, tol=1e-12, stream=None):
        """(alpha, beta, e0): stops when E_0 moved by <= tol * max(1, |E_0|) over `check_every` iterations."""
        alpha = np.zeros(max(max_iters, 1))
        beta = np.zeros(max(max_iters, 1))
        done, e0 = C.c_int(0), C.c_double(0.0)
        dp = C.POINTER(C.c_double)
        _check(lib.lanczos_run_until(self._h, _dptr(v0), max_iters, check_every, float(tol), alpha.ctypes.data_as(dp),
                                     beta.ctypes.data_as(dp), C.byref(done), C.byref(e0), _stream(stream)),
               "lanczos_run_until", self._h)
        return alpha[:done.value].copy(), beta[:done.value].copy(), e0.value

    def lanczos_ground_state(self, v0, iters, psi, stream=None):
        """Fills psi (device tensor, dim elements) with the normalised ground-state vector; returns (e0, iters_done)."""
        done, e0 = C.c_int(0), C.c_double(0.0)
        _check(lib.lanczos_ground_state(self._h, _dptr(v0), iters, _dptr(psi), C.byref(e0), C.byref(done), _stream(stream)),
               "lanczos_ground_state", self._h)
        return e0.value, done.value

    def lanczos_propagate(self, v0, iters, tau, t, out_re, out_im=None, stream=None):
        """out = exp(-(tau + i t) H) v0 by Krylov propagation (real v0); returns the iterations done."""
        done = C.c_int(0)
        _check(lib.lanczos_propagate(self._h, _dptr(v0), iters, float(tau), float(t), _dptr(out_re),
                                     _dptr(out_im) if out_im is not None else None, C.byref(done), _stream(stream)),
               "lanczos_propagate", self._h)
        return done.value

    def lanczos_propagate_complex(self, re_in, im_in, iters, tau, t, out_re, out_im, stream=None):
        """(out_re + i out_im) = exp(-(tau + i t) H) (re_in + i im_in); im_in may be None; returns the iterations done."""
        done = C.c_int(0)
        _check(lib.lanczos_propagate_complex(self._h, _dptr(re_in), _dptr(im_in) if im_in is not None else None, iters,
                                             float(tau), float(t), _dptr(out_re), _dptr(out_im), C.byref(done), _stream(stream)),
               "lanczos_propagate_complex", self._h)
        return done.value

    # -- row-sharded pieces (see sharded.py)
    def hubbard_apply_rows(self, x_full, y_rows, row0, row1, stream=None):
        _check(lib.hubbard_apply_rows(self._h, _dptr(x_full), _dptr(y_rows), int(row0), int(row1), _stream(stream)),
               "hubbard_apply_rows", self._h)
        return y_rows

    def lanczos_shard_update(self, mode, inout, other, f, coef, result, stream=None):
        _check(lib.lanczos_shard_update(self._h, int(mode), _dptr(inout), _dptr(other) if other is not None else None,
                                        _dptr(f) if f is not None else None, inout.numel(), float(coef),
                                        _dptr(result) if result is not None else None, _stream(stream)),
               "lanczos_shard_update", self._h)

    def lanczos_shard_update_noalloc(self, mode, inout, other, f, coef, result, stream=None, n=None):
        """lanczos_shard_update with the library's fixed scratch array: no allocation, n <= NOALLOC_MAX_N
        (include/hubbard.h).  `n` overrides the element count (default: all of `inout`)."""
        _check(lib.lanczos_shard_update_noalloc(self._h, int(mode), _dptr(inout), _dptr(other) if other is not None else None,
                                                _dptr(f) if f is not None else None, inout.numel() if n is None else int(n),
                                                float(coef), _dptr(result) if result is not None else None, _stream(stream)),
               "lanczos_shard_update_noalloc", self._h)

    # -- hot path, host buffers (numpy arrays or CPU torch tensors)
    @staticmethod
    def _hptr(a) -> int:
        if isinstance(a, np.ndarray):
            if not a.flags.c_contiguous:
                raise ValueError("expected a C-contiguous array")
            return a.ctypes.data
        return a.data_ptr()

    def hubbard_apply_host(self, x, y, stream=None):
        _check(lib.hubbard_apply_host(self._h, self._hptr(x), self._hptr(y), _stream(stream)),
               "hubbard_apply_host", self._h)
        return y

    def lanczos_run_host(self, v0, iters, stream=None):
        alpha = np.zeros(max(iters, 1))
        beta = np.zeros(max(iters, 1))
        done = C.c_int(0)
        dp = C.POINTER(C.c_double)
        _check(lib.lanczos_run_host(self._h, self._hptr(v0), iters, alpha.ctypes.data_as(dp),
                                    beta.ctypes.data_as(dp), C.byref(done), _stream(stream)),
               "lanczos_run_host", self._h)
        return alpha[:done.value].copy(), beta[:done.value].copy()

    # -- introspection
    def hubbard_get_basis(self, spin):
        n = self.dim_up if spin == 0 else self.dim_dn
        out = np.empty(n, dtype=np.uint32)
        _check(lib.hubbard_get_basis(self._h, spin, out.ctypes.data_as(C.POINTER(C.c_uint32))), "hubbard_get_basis")
        return out

    def hubbard_get_hops(self, spin):
        n = self.dim_up if spin == 0 else self.dim_dn
        w = C.c_int(0)
        _check(lib.hubbard_get_hops(self._h, spin, C.byref(w), None, None), "hubbard_get_hops")
        cols = np.empty((n, w.value), dtype=np.int32)
        vals = np.empty((n, w.value), dtype=np.float64)
        _check(lib.hubbard_get_hops(self._h, spin, C.byref(w), cols.ctypes.data_as(C.POINTER(C.c_int32)),
                                    vals.ctypes.data_as(C.POINTER(C.c_double))), "hubbard_get_hops")
        return w.value, cols, vals

    def hubbard_get_gather_table(self, spin, lanes, R=1, sorted=False):
        """Variant GATHER's table: dict(slots, ld, entries[slots/8, ld, 8], counts[ld], warp_slots[ld/32], perm[ld],
        conflicts, wavefronts)."""
        w, ld, cf, wf = C.c_int(0), C.c_int64(0), C.c_int64(0), C.c_int64(0)
        _check(lib.hubbard_get_gather_table(self._h, spin, lanes, R, int(sorted), C.byref(w), C.byref(ld), None, None,
                                            None, None, C.byref(cf), C.byref(wf)), "hubbard_get_gather_table")
        ent = np.empty((w.value // 8, ld.value, 8), dtype=np.uint32)
        cnt = np.empty(ld.value, dtype=np.int32)
        wsl = np.empty(ld.value // 32, dtype=np.uint16)
        perm = np.empty(ld.value, dtype=np.int32)
        _check(lib.hubbard_get_gather_table(self._h, spin, lanes, R, int(sorted), C.byref(w), C.byref(ld),
                                            ent.ctypes.data_as(C.POINTER(C.c_uint32)),
                                            cnt.ctypes.data_as(C.POINTER(C.c_int32)),
                                            wsl.ctypes.data_as(C.POINTER(C.c_uint16)),
                                            perm.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(cf), C.byref(wf)),
               "hubbard_get_gather_table")
        return {"slots": w.value, "ld": ld.value, "entries": ent, "counts": cnt, "warp_slots": wsl, "perm": perm,
                "conflicts": cf.value, "wavefronts": wf.value}

    # -- measurement hooks
    def hubbard_profile(self, enable=True):
        _check(lib.hubbard_profile(self._h, int(bool(enable))), "hubbard_profile")

    def hubbard_kernel_times(self):
        n = (C.c_int64 * N_KCLASS)()
        ms = (C.c_double * N_KCLASS)()
        _check(lib.hubbard_kernel_times(self._h, n, ms), "hubbard_kernel_times", self._h)
        return {KCLASS_NAMES[k]: (int(n[k]), float(ms[k])) for k in range(N_KCLASS)}

    def hubbard_launch_count(self):
        return int(lib.hubbard_launch_count(self._h))


def hubbard_create(n_sites, n_up, n_dn, bonds, t, U, dtype="f64") -> Model:
    return Model(n_sites, n_up, n_dn, bonds, t, U, dtype)


def hubbard_create_host(n_sites, n_up, n_dn, bonds, t, U, dtype="f64") -> Model:
    return Model(n_sites, n_up, n_dn, bonds, t, U, dtype, host_only=True)


def lanczos_ground_energy(alpha, beta, m=None) -> float:
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    b = np.ascontiguousarray(beta, dtype=np.float64)
    m = len(a) if m is None else int(m)
    if len(b) < max(m - 1, 0) or len(a) < m:
        raise ValueError("alpha/beta shorter than m")
    if len(b) == 0:
        b = np.zeros(1)
    e0 = C.c_double(0.0)
    dp = C.POINTER(C.c_double)
    _check(lib.lanczos_ground_energy(a.ctypes.data_as(dp), b.ctypes.data_as(dp), m, C.byref(e0)),
           "lanczos_ground_energy")
    return e0.value


def lanczos_ground_vector(alpha, beta, m=None):
    """(e0, y): smallest eigenvalue of T_m and its unit eigenvector (host utility)."""
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    b = np.ascontiguousarray(beta, dtype=np.float64)
    m = len(a) if m is None else int(m)
    if len(b) < max(m - 1, 0) or len(a) < m:
        raise ValueError("alpha/beta shorter than m")
    if len(b) == 0:
        b = np.zeros(1)
    e0 = C.c_double(0.0)
    y = np.zeros(m)
    dp = C.POINTER(C.c_double)
    _check(lib.lanczos_ground_vector(a.ctypes.data_as(dp), b.ctypes.data_as(dp), m, C.byref(e0), y.ctypes.data_as(dp)),
           "lanczos_ground_vector")
    return e0.value, y


def lanczos_expm_e1(alpha, beta, tau, t, m=None):
    """exp(-(tau + i t) T_m) e_1 as a complex numpy vector (host utility)."""
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    b = np.ascontiguousarray(beta, dtype=np.float64)
    m = len(a) if m is None else int(m)
    if len(b) == 0:
        b = np.zeros(1)
    yr, yi = np.zeros(m), np.zeros(m)
    dp = C.POINTER(C.c_double)
    _check(lib.lanczos_expm_e1(a.ctypes.data_as(dp), b.ctypes.data_as(dp), m, float(tau), float(t), yr.ctypes.data_as(dp),
                               yi.ctypes.data_as(dp)), "lanczos_expm_e1")
    return yr + 1j * yi
