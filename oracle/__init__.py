"""ctypes loader for the CPU oracle (``oracle/ami_oracle.cpp``).

TEST INFRASTRUCTURE.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product package
``paper_2311_17189_b200`` never does, and this package never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ami_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

ERRORS = {-1: "EINVAL", -2: "EUNSUPPORTED_ALPHA (|alpha_p| != 1 at a summation)", -3: "ENOPOLE"}


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle error {code}: {ERRORS.get(code, '?')}")
        self.code = code


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (seconds).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-o", tmp, _SRC,
                               "-lquadmath", "-lpthread"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.oracle_construct.restype = C.c_void_p
        L.oracle_construct.argtypes = [C.c_int] * 4 + [C.c_void_p] * 4 + [C.c_double, C.POINTER(C.c_int)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_info.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_describe.restype = C.c_long
        L.oracle_describe.argtypes = [C.c_void_p, C.c_char_p, C.c_long]
        L.oracle_evaluate.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_long, C.c_void_p, C.c_int,
                                      C.c_double, C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_evaluate_ex.argtypes = L.oracle_evaluate.argtypes + [C.c_void_p, C.c_void_p]
        L.oracle_dispersion.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                        C.c_long, C.c_int, C.c_int, C.c_void_p]
        L.oracle_dispersion_lattice.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                                C.c_long, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.oracle_fermi.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_void_p]
        _lib = L
    return _lib


def hardware_threads() -> int:
    return int(lib().oracle_hardware_threads())


def fermi(E: complex, beta: float, sigma: int, k: int, quad: bool = True) -> complex:
    out = np.zeros(2)
    lib().oracle_fermi(float(np.real(E)), float(np.imag(E)), float(beta), int(sigma), int(k),
                       1 if quad else 0, out.ctypes.data)
    return complex(out[0], out[1])


class OracleTable:
    """The symbolic AMI result of one diagram (``construct``)."""

    def __init__(self, n_int, n_ext, alpha, eps, slot_is_fermionic, sum_order=None, prefactor=1.0):
        alpha = np.ascontiguousarray(alpha, dtype=np.int32)
        eps = np.ascontiguousarray(eps, dtype=np.int32)
        stat = np.ascontiguousarray(slot_is_fermionic, dtype=np.uint8)
        assert alpha.shape[1] == n_int + n_ext and alpha.shape[0] == eps.shape[0]
        so = None if sum_order is None else np.ascontiguousarray(sum_order, dtype=np.int32)
        err = C.c_int(0)
        self.n_int, self.n_ext, self.n_g, self.n_eps = n_int, n_ext, alpha.shape[0], eps.shape[1]
        self._h = lib().oracle_construct(n_int, n_ext, self.n_g, self.n_eps, alpha.ctypes.data,
                                         eps.ctypes.data, stat.ctypes.data,
                                         None if so is None else so.ctypes.data, float(prefactor),
                                         C.byref(err))
        if not self._h:
            raise OracleError(err.value)

    @classmethod
    def from_diagram(cls, d, sum_order=None, prefactor=1.0):
        return cls(d.n_int, d.n_ext, d.alpha, d.eps, d.slot_is_fermionic, sum_order, prefactor)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:   # _lib is gone at interpreter shutdown
            _lib.oracle_destroy(self._h)
            self._h = None

    def info(self) -> dict:
        a = np.zeros(4, dtype=np.int64)
        lib().oracle_info(self._h, a.ctypes.data)
        return {"T": int(a[0]), "max_deriv": int(a[1]), "multipoles": int(a[2]), "deriv_terms": int(a[3])}

    def describe(self) -> str:
        n = lib().oracle_describe(self._h, None, 0)
        buf = C.create_string_buffer(n)
        lib().oracle_describe(self._h, buf, n)
        return buf.value.decode()

    def evaluate(self, e, z_ext, beta, e_reg=0.0, quad=False, threads=1, want_S=False, want_logs=False):
        """e: [n_e][n_eps] float64 or complex128 (paper's energy_t);
        z_ext: complex [n_f][n_ext].  Returns complex128 [n_f][n_e] and,
        if want_S, S = sum_t |term_t| with the same shape; if want_logs also log2 S and log2 |value|
        taken before the cast to double (they survive where S itself underflows a double)."""
        e = np.ascontiguousarray(e)
        is_c = np.iscomplexobj(e)
        e = e.astype(np.complex128 if is_c else np.float64)
        assert e.ndim == 2 and e.shape[1] == self.n_eps
        z = np.ascontiguousarray(np.asarray(z_ext, dtype=np.complex128).reshape(-1, self.n_ext))
        n_e, n_f = e.shape[0], z.shape[0]
        out = np.zeros((n_f, n_e), dtype=np.complex128)
        S = np.zeros((n_f, n_e), dtype=np.float64)
        l2S = np.zeros((n_f, n_e)) if want_logs else None
        l2v = np.zeros((n_f, n_e)) if want_logs else None
        rc = lib().oracle_evaluate_ex(self._h, e.ctypes.data, int(is_c), n_e, z.ctypes.data, n_f, float(beta),
                                      float(e_reg), 1 if quad else 0, int(threads), out.ctypes.data,
                                      S.ctypes.data, None if l2S is None else l2S.ctypes.data,
                                      None if l2v is None else l2v.ctypes.data)
        if rc:
            raise OracleError(rc)
        if want_logs:
            return out, S, l2S, l2v
        return (out, S) if want_S else out

    def dispersion(self, k, q, t, mu, quad=False, threads=1, dim=2, band=0):
        """k: [n_e][n_int][dim] (Eq. 8), q: [n_ext][dim] -> e [n_e][n_eps], e_i = -eps(K_i); band 0 =
        hypercubic tight binding -2t sum cos K_c - mu, band 1 = free particles t |K|^2 - mu."""
        k = np.ascontiguousarray(k, dtype=np.float64).reshape(-1, self.n_int, dim)
        q = np.ascontiguousarray(np.asarray(q, dtype=np.float64).reshape(self.n_ext, dim))
        out = np.zeros((k.shape[0], self.n_eps))
        rc = lib().oracle_dispersion_lattice(self._h, k.ctypes.data, q.ctypes.data, float(t), float(mu),
                                             k.shape[0], int(dim), int(band), 1 if quad else 0, int(threads),
                                             out.ctypes.data)
        if rc:
            raise OracleError(rc)
        return out
