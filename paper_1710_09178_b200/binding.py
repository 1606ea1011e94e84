"""ctypes binding of include/qcd.h -- argument marshalling only.

Module-level functions carry the C names (`qcd_create`, `qcd_dslash`, ...) and take raw
pointers (ints) exactly like the C ABI.  `Context` is a convenience wrapper that accepts
torch CUDA tensors (device entry points) or numpy arrays (host entry points) and passes
their addresses; it holds no arithmetic.  There is no fallback of any kind: a missing
library, a missing GPU or a failing call raises.
"""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np

QCD_EVEN, QCD_ODD = 0, 1
QCD_OPT_PDL, QCD_OPT_CG_GRAPH, QCD_OPT_CG_BATCH, QCD_OPT_LINK_ROWS, QCD_OPT_TGROUP = 0, 1, 2, 3, 4
QCD_OPT_L2_PERSIST_MB, QCD_OPT_Y_ONLY, QCD_OPT_DSLASH_KERNEL, QCD_OPT_DSLASH_PERSIST = 5, 6, 7, 8
QCD_OPT_MIXED, QCD_OPT_MIXED_SWITCH_EXP, QCD_OPT_OPERATOR_LINKS32, QCD_OPT_SWEEP_ALTERNATE, QCD_OPT_CG_DEFER, QCD_OPT_SWEEP_KEEP_MB, QCD_OPT_CG_FUSE = 9, 10, 11, 12, 13, 14, 15
QCD_OK, QCD_EINVAL, QCD_ENOMEM, QCD_ECUDA, QCD_ENOTCONV, QCD_ESTATE = range(6)
_STATUS_NAMES = ["QCD_OK", "QCD_EINVAL", "QCD_ENOMEM", "QCD_ECUDA", "QCD_ENOTCONV", "QCD_ESTATE"]

_HERE = os.path.dirname(os.path.abspath(__file__))
# QCD_B200_LIB: load another build of the same library (tuning aid: builds with different QCD_NVCC_EXTRA macros)
_LIB_PATH = os.environ.get("QCD_B200_LIB") or os.path.join(_HERE, "libqcd_b200.so")
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "qcd.h")

_vp, _ci, _cd, _cl = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_long
_SIGNATURES = {
    "qcd_version": (ctypes.c_char_p, []),
    "qcd_create": (_ci, [ctypes.POINTER(_ci), _cd, _vp, ctypes.POINTER(_vp)]),
    "qcd_destroy": (_ci, [_vp]),
    "qcd_set_mass": (_ci, [_vp, _cd]),
    "qcd_set_stream": (_ci, [_vp, _vp]),
    "qcd_set_option": (_ci, [_vp, _ci, _cl]),
    "qcd_vector_doubles": (_cl, [_vp]),
    "qcd_load_gauge": (_ci, [_vp, _vp]),
    "qcd_load_gauge_host": (_ci, [_vp, _vp]),
    "qcd_pack": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_unpack": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_dslash": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_dslash_range": (_ci, [_vp, _ci, _vp, _vp, _ci, _ci, _vp, _cd]),
    "qcd_set_slab": (_ci, [_vp, _ci, _vp, _vp, _vp]),
    "qcd_mdagm": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_multishift_cg": (_ci, [_vp, _ci, _vp, _ci, _vp, _vp, _cd, _ci, _vp, _vp,
                                ctypes.POINTER(_ci), _vp]),
    "qcd_inv_sqrt_coeffs": (_ci, [_ci, _cd, _cd, _vp, _vp, _vp, _vp]),
    "qcd_inv_sqrt": (_ci, [_vp, _ci, _vp, _ci, _cd, _cd, _cd, _ci, _vp, ctypes.POINTER(_ci), _vp, _vp]),
    "qcd_pow_coeffs": (_ci, [_ci, _ci, _ci, _cd, _cd, _vp, _vp, _vp, _vp]),
    "qcd_apply_pow": (_ci, [_vp, _ci, _vp, _ci, _ci, _ci, _cd, _cd, _cd, _ci, _vp, ctypes.POINTER(_ci), _vp, _vp]),
    "qcd_dslash_host": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_mdagm_host": (_ci, [_vp, _ci, _vp, _vp]),
    "qcd_multishift_cg_host": (_ci, [_vp, _ci, _vp, _ci, _vp, _vp, _cd, _ci, _vp, _vp,
                                     ctypes.POINTER(_ci), _vp]),
    "qcd_launch_count": (_cl, [_vp]),
    "qcd_last_error": (ctypes.c_char_p, [_vp]),
}


class QcdError(RuntimeError):
    def __init__(self, status: int, where: str, text: str):
        self.status = status
        name = _STATUS_NAMES[status] if 0 <= status < len(_STATUS_NAMES) else str(status)
        super().__init__(f"{where}: {name}: {text}")


def library_path() -> str:
    return _LIB_PATH


def exported_symbols():
    """Every function include/qcd.h declares (parsed from the header)."""
    with open(_HEADER) as fh:
        text = fh.read()
    return sorted(set(re.findall(r"QCD_API[^;(]*?\b(qcd_\w+)\s*\(", text)))


_lib = None


def load_library():
    """dlopen the in-tree libqcd_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise FileNotFoundError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_1710_09178_b200.build` "
            "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(_LIB_PATH)
    for name, (res, args) in _SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _make_raw(name):
    def call(*args):
        return getattr(load_library(), name)(*args)
    call.__name__ = name
    call.__doc__ = f"Raw C-ABI call {name} (see include/qcd.h); pointers are ints."
    return call


for _n in _SIGNATURES:
    globals()[_n] = _make_raw(_n)


def _dev_ptr(t, doubles: int | None = None) -> int:
    """Address of a contiguous float64 CUDA tensor (holding at least `doubles` elements)."""
    if not (t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float64"):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    if doubles is not None and t.numel() < doubles:
        raise ValueError(f"device buffer holds {t.numel()} doubles, the call needs {doubles}")
    return t.data_ptr()


def _host_ptr(a: np.ndarray, doubles: int | None = None) -> int:
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous):
        raise TypeError("expected a C-contiguous float64 numpy array")
    if doubles is not None and a.size < doubles:
        raise ValueError(f"host buffer holds {a.size} doubles, the call needs {doubles}")
    return a.ctypes.data


def inv_sqrt_coeffs(n: int, xmin: float, xmax: float):
    """qcd_inv_sqrt_coeffs (host only): returns (c0, c[n], d[n], delta)."""
    lib = load_library()
    c0, delta = np.zeros(1), np.zeros(1)
    c, d = np.zeros(max(int(n), 1)), np.zeros(max(int(n), 1))
    st = lib.qcd_inv_sqrt_coeffs(int(n), float(xmin), float(xmax), _host_ptr(c0), _host_ptr(c),
                                 _host_ptr(d), _host_ptr(delta))
    if st != QCD_OK:
        raise QcdError(st, "qcd_inv_sqrt_coeffs", lib.qcd_last_error(None).decode())
    return float(c0[0]), c, d, float(delta[0])


def pow_coeffs(num: int, den: int, n: int, xmin: float, xmax: float):
    """qcd_pow_coeffs (host only): x^(num/den) ~= c0 + sum c[k]/(x + d[k]); returns (c0, c, d, delta)."""
    lib = load_library()
    c0, delta = np.zeros(1), np.zeros(1)
    c, d = np.zeros(max(int(n), 1)), np.zeros(max(int(n), 1))
    st = lib.qcd_pow_coeffs(int(num), int(den), int(n), float(xmin), float(xmax), _host_ptr(c0),
                            _host_ptr(c), _host_ptr(d), _host_ptr(delta))
    if st != QCD_OK:
        raise QcdError(st, "qcd_pow_coeffs", lib.qcd_last_error(None).decode())
    return float(c0[0]), c, d, float(delta[0])


class Context:
    """Owns one qcd_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, dims, mass: float, stream=None):
        self._lib = load_library()
        self._h = _vp(None)
        self.dims = tuple(int(d) for d in dims)
        self.volume = int(np.prod(self.dims))
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        cd = (_ci * 4)(*self.dims)
        st = self._lib.qcd_create(cd, float(mass), _vp(stream), ctypes.byref(self._h))
        if st != QCD_OK:
            raise QcdError(st, "qcd_create", self._lib.qcd_last_error(None).decode())
        self.vector_doubles = int(self._lib.qcd_vector_doubles(self._h))

    def close(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._lib.qcd_destroy(h)

    __del__ = close

    def _check(self, st: int, where: str, allow=()):
        exc, self._slab_exc = getattr(self, "_slab_exc", None), None
        if exc is not None:
            raise exc
        if st != QCD_OK and st not in allow:
            raise QcdError(st, where, self._lib.qcd_last_error(self._h).decode())
        return st

    # -- helpers that only allocate device memory (torch is plumbing) --
    def new_vector(self, n: int | None = None):
        import torch
        shape = (self.vector_doubles,) if n is None else (n, self.vector_doubles)
        return torch.empty(shape, dtype=torch.float64, device="cuda")

    @property
    def launch_count(self) -> int:
        return int(self._lib.qcd_launch_count(self._h))

    def set_mass(self, mass: float):
        self._check(self._lib.qcd_set_mass(self._h, float(mass)), "qcd_set_mass")

    def set_option(self, option: int, value: int):
        self._check(self._lib.qcd_set_option(self._h, int(option), int(value)), "qcd_set_option")

    def set_stream(self, stream: int):
        self._check(self._lib.qcd_set_stream(self._h, _vp(stream)), "qcd_set_stream")

    # -- device entry points --
    def load_gauge(self, d_links):
        self._check(self._lib.qcd_load_gauge(self._h, _dev_ptr(d_links, 72 * self.volume)), "qcd_load_gauge")

    def pack(self, parity: int, d_canonical, d_internal):
        self._check(self._lib.qcd_pack(self._h, parity, _dev_ptr(d_canonical, self.vector_doubles), _dev_ptr(d_internal, self.vector_doubles)),
                    "qcd_pack")

    def unpack(self, parity: int, d_internal, d_canonical):
        self._check(self._lib.qcd_unpack(self._h, parity, _dev_ptr(d_internal, self.vector_doubles), _dev_ptr(d_canonical, self.vector_doubles)),
                    "qcd_unpack")

    def dslash(self, out_parity: int, d_in, d_out):
        self._check(self._lib.qcd_dslash(self._h, out_parity, _dev_ptr(d_in, self.vector_doubles), _dev_ptr(d_out, self.vector_doubles)),
                    "qcd_dslash")

    def dslash_range(self, out_parity: int, d_in, d_out, t0: int, nt: int, d_src=None, coeff: float = 0.0):
        vd = self.vector_doubles
        self._check(self._lib.qcd_dslash_range(self._h, out_parity, _dev_ptr(d_in, vd), _dev_ptr(d_out, vd),
                                               int(t0), int(nt), None if d_src is None else _dev_ptr(d_src, vd),
                                               float(coeff)), "qcd_dslash_range")

    def set_slab(self, halo=None, allreduce=None):
        """qcd_set_slab.  halo(ptr: int, stream: int) fills the two halo t-slices of the internal vector at
        device address ptr; allreduce(ptr: int, count: int, stream: int) sums count doubles at device address
        ptr over the ranks, in place.  Both None: leave slab mode.  The ctypes trampolines are kept alive here."""
        if halo is None and allreduce is None:
            self._slab_cbs = None
            self._check(self._lib.qcd_set_slab(self._h, 0, None, None, None), "qcd_set_slab")
            return
        halo_t = ctypes.CFUNCTYPE(None, _vp, _vp, _vp)
        red_t = ctypes.CFUNCTYPE(None, _vp, _vp, _ci, _vp)
        self._slab_exc = None

        def guard(fn, *a):          # an exception must not unwind through the C frames: keep it for _check
            try:
                fn(*a)
            except BaseException as e:  # noqa: BLE001
                if self._slab_exc is None:
                    self._slab_exc = e

        h = halo_t(lambda user, ptr, stream: guard(halo, int(ptr or 0), int(stream or 0)))
        r = red_t(lambda user, ptr, count, stream: guard(allreduce, int(ptr or 0), int(count), int(stream or 0)))
        self._slab_cbs = (h, r)
        self._check(self._lib.qcd_set_slab(self._h, 1, ctypes.cast(h, _vp), ctypes.cast(r, _vp), None), "qcd_set_slab")

    def mdagm(self, parity: int, d_in, d_out):
        self._check(self._lib.qcd_mdagm(self._h, parity, _dev_ptr(d_in, self.vector_doubles), _dev_ptr(d_out, self.vector_doubles)), "qcd_mdagm")

    def multishift_cg(self, parity: int, d_b, shifts, residues, tol: float, max_iter: int,
                      d_x=None, d_y=None):
        """Returns (status, iterations, true_res[nshift]); status is QCD_OK or QCD_ENOTCONV."""
        shifts = np.ascontiguousarray(shifts, dtype=np.float64)
        residues = np.ascontiguousarray(residues, dtype=np.float64)
        n = int(shifts.size)
        if residues.size != n:
            raise ValueError("shifts and residues must have the same length")
        true_res = np.full(n, np.nan)
        it = _ci(0)
        st = self._lib.qcd_multishift_cg(
            self._h, parity, _dev_ptr(d_b, self.vector_doubles), n, _host_ptr(shifts), _host_ptr(residues), float(tol),
            int(max_iter), None if d_x is None else _dev_ptr(d_x, n * self.vector_doubles),
            None if d_y is None else _dev_ptr(d_y, self.vector_doubles), ctypes.byref(it), _host_ptr(true_res))
        self._check(st, "qcd_multishift_cg", allow=(QCD_ENOTCONV,))
        return st, it.value, true_res

    def inv_sqrt(self, parity: int, d_phi, n: int, xmin: float, xmax: float, tol: float,
                 max_iter: int, d_out):
        """Returns (status, iterations, true_res[n], delta)."""
        true_res = np.full(int(n), np.nan)
        delta = np.zeros(1)
        it = _ci(0)
        st = self._lib.qcd_inv_sqrt(self._h, parity, _dev_ptr(d_phi, self.vector_doubles), int(n), float(xmin), float(xmax),
                                    float(tol), int(max_iter), _dev_ptr(d_out, self.vector_doubles), ctypes.byref(it),
                                    _host_ptr(true_res), _host_ptr(delta))
        self._check(st, "qcd_inv_sqrt", allow=(QCD_ENOTCONV,))
        return st, it.value, true_res, float(delta[0])

    def apply_pow(self, parity: int, d_phi, num: int, den: int, n: int, xmin: float, xmax: float,
                  tol: float, max_iter: int, d_out):
        """Returns (status, iterations, true_res[n], delta)."""
        true_res = np.full(int(n), np.nan)
        delta = np.zeros(1)
        it = _ci(0)
        st = self._lib.qcd_apply_pow(self._h, parity, _dev_ptr(d_phi, self.vector_doubles), int(num), int(den), int(n),
                                     float(xmin), float(xmax), float(tol), int(max_iter),
                                     _dev_ptr(d_out, self.vector_doubles), ctypes.byref(it), _host_ptr(true_res),
                                     _host_ptr(delta))
        self._check(st, "qcd_apply_pow", allow=(QCD_ENOTCONV,))
        return st, it.value, true_res, float(delta[0])

    # -- host entry points (canonical numpy arrays; copies happen inside the C call) --
    def load_gauge_host(self, h_links: np.ndarray):
        self._check(self._lib.qcd_load_gauge_host(self._h, _host_ptr(h_links, 72 * self.volume)), "qcd_load_gauge_host")

    def dslash_host(self, out_parity: int, h_in: np.ndarray, h_out: np.ndarray):
        self._check(self._lib.qcd_dslash_host(self._h, out_parity, _host_ptr(h_in, self.vector_doubles), _host_ptr(h_out, self.vector_doubles)),
                    "qcd_dslash_host")

    def mdagm_host(self, parity: int, h_in: np.ndarray, h_out: np.ndarray):
        self._check(self._lib.qcd_mdagm_host(self._h, parity, _host_ptr(h_in, self.vector_doubles), _host_ptr(h_out, self.vector_doubles)),
                    "qcd_mdagm_host")

    def multishift_cg_host(self, parity: int, h_b: np.ndarray, shifts, residues, tol: float,
                           max_iter: int, h_x: np.ndarray | None = None,
                           h_y: np.ndarray | None = None):
        shifts = np.ascontiguousarray(shifts, dtype=np.float64)
        residues = np.ascontiguousarray(residues, dtype=np.float64)
        n = int(shifts.size)
        if residues.size != n:
            raise ValueError("shifts and residues must have the same length")
        true_res = np.full(n, np.nan)
        it = _ci(0)
        st = self._lib.qcd_multishift_cg_host(
            self._h, parity, _host_ptr(h_b, self.vector_doubles), n, _host_ptr(shifts), _host_ptr(residues), float(tol),
            int(max_iter), None if h_x is None else _host_ptr(h_x, n * self.vector_doubles),
            None if h_y is None else _host_ptr(h_y, self.vector_doubles), ctypes.byref(it), _host_ptr(true_res))
        self._check(st, "qcd_multishift_cg_host", allow=(QCD_ENOTCONV,))
        return st, it.value, true_res
