"""Thin ctypes binding of include/ami.h: argument marshalling only.  Every step of the path
runs in the CUDA kernels of libami_b200.so; PyTorch supplies device memory and streams.
There is no CPU fallback: without the built library, or without a device copy of the table,
every call raises."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libami_b200.so")

PLAN_AUTO, PLAN_FLAT, PLAN_REG, PLAN_TREE = 0, 1, 2, 3
PLAN_UNORDERED = 0x100   # AMI_PLAN_UNORDERED: OR into `plan` (see include/ami.h)
BAND_TIGHT_BINDING, BAND_FREE = 0, 1

EXPORTS = [
    "ami_construct", "ami_table_info", "ami_table_export", "ami_table_export_tree", "ami_table_destroy", "ami_dispersion",
    "ami_dispersion_lattice",
    "ami_evaluate", "ami_evaluate_momenta", "ami_table_specialize", "ami_table_kernel_source",
    "ami_table_kernel_cubin", "ami_run", "ami_generate_momenta", "ami_fp64_peak_probe", "ami_strerror",
    "ami_last_cuda_error", "ami_version", "ami_kernel_launches", "ami_search_sum_order", "ami_graph_parse",
    "ami_graph_label", "ami_table_latex", "ami_evaluate_momenta_lattice", "ami_generate_momenta_lattice",
    "ami_table_kernel_units", "ami_table_kernel_cubin_unit", "ami_table_kernel_source_variant",
    "ami_table_kernel_cubin_variant", "ami_table_latex_factorized", "ami_tally_static",
]


class AmiError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ami error {code}: {msg}")
        self.code = code


class ami_info(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_int", "n_ext", "n_g", "n_eps", "n_fermi_leaves", "n_den_leaves",
                                         "max_deriv", "max_den_per_term")] + \
               [(n, C.c_int64) for n in ("n_terms", "n_terms_raw", "n_multipoles", "n_groups", "n_tree_nodes",
                                         "n_den_nodes", "table_bytes", "fp64_ops_flat", "fp64_ops_tree",
                                         "fp64_ops_tree_fermi", "fp64_ops_leaf_fermi", "fp64_ops_leaf_den",
                                         "fp64_ops_dispersion", "fp64_ops_combos", "tree_plan_words", "tree_plan_slots")] + \
               [("has_device_copy", C.c_int32), ("reg_plan_status", C.c_int32), ("plan_kind", C.c_int32),
                ("specialize_cached", C.c_int32), ("specialize_ms", C.c_double), ("fp64_ops_mb_prefix", C.c_int64),
                ("fp64_ops_mb_sum", C.c_int64)]


class ami_run_cfg(C.Structure):
    _fields_ = [("n", C.c_int64), ("chunk", C.c_int64), ("seed", C.c_uint64), ("first_sample", C.c_int64),
                ("h_k", C.c_void_p), ("d_k", C.c_void_p), ("q", C.c_void_p), ("t", C.c_double),
                ("mu", C.c_double), ("z_ext", C.c_void_p), ("n_f", C.c_int32), ("beta", C.c_void_p),
                ("n_b", C.c_int32), ("e_reg", C.c_double), ("plan", C.c_int32), ("want_sum", C.c_int32),
                ("h_out", C.c_void_p), ("d_out", C.c_void_p), ("h_sum", C.c_void_p), ("stream", C.c_void_p),
                ("h_sumsq", C.c_void_p), ("dim", C.c_int32), ("band", C.c_int32)]


class ami_run_stats(C.Structure):
    _fields_ = [("n_chunks", C.c_int64), ("kernel_launches", C.c_int64), ("h2d_bytes", C.c_int64),
                ("d2h_bytes", C.c_int64), ("gpu_ms", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run __graft_entry__.build() "
                               "(python -m paper_2311_17189_b200.build); there is no fallback path")
        L = C.CDLL(LIB_PATH)
        L.ami_construct.argtypes = [C.c_int] * 4 + [C.c_void_p] * 4 + [C.c_double, C.c_int, C.POINTER(C.c_void_p)]
        L.ami_table_info.argtypes = [C.c_void_p, C.POINTER(ami_info)]
        L.ami_graph_parse.argtypes = [C.c_char_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.ami_graph_label.argtypes = [C.c_void_p, C.c_int32] + [C.POINTER(C.c_int32)] * 4 + [C.c_void_p] * 5 + [C.c_int64]
        L.ami_search_sum_order.argtypes = [C.c_int] * 4 + [C.c_void_p] * 3 + [C.c_int, C.c_int64, C.c_void_p] + \
            [C.POINTER(C.c_int64)] * 3
        L.ami_table_export.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_export_tree.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_destroy.argtypes = [C.c_void_p]
        L.ami_table_latex.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_latex_factorized.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_destroy.restype = None
        L.ami_dispersion.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double,
                                     C.c_double, C.c_int64, C.c_void_p, C.c_void_p]
        L.ami_dispersion_lattice.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double,
                                             C.c_double, C.c_int, C.c_int, C.c_int64, C.c_void_p, C.c_void_p]
        L.ami_evaluate.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_int, C.c_void_p,
                                   C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
        L.ami_evaluate_momenta.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double,
                                           C.c_double, C.c_int64, C.c_void_p, C.c_int, C.c_void_p, C.c_int,
                                           C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.ami_evaluate_momenta_lattice.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_double,
                                                   C.c_double, C.c_int, C.c_int, C.c_int64, C.c_void_p, C.c_int,
                                                   C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_void_p, C.c_void_p,
                                                   C.c_void_p]
        L.ami_generate_momenta_lattice.argtypes = [C.c_void_p, C.c_uint64, C.c_int64, C.c_int64, C.c_int, C.c_void_p,
                                                   C.c_void_p]
        L.ami_table_specialize.argtypes = [C.c_void_p]
        L.ami_table_kernel_source.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_kernel_cubin.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t), C.c_void_p, C.c_size_t]
        L.ami_table_kernel_units.argtypes = [C.c_void_p, C.POINTER(C.c_int)]
        L.ami_table_kernel_cubin_unit.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_size_t), C.c_void_p,
                                                  C.c_size_t]
        L.ami_table_kernel_source_variant.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_size_t)]
        L.ami_table_kernel_cubin_variant.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                                     C.POINTER(C.c_size_t), C.c_void_p, C.c_size_t]
        L.ami_run.argtypes = [C.c_void_p, C.POINTER(ami_run_cfg), C.POINTER(ami_run_stats)]
        L.ami_generate_momenta.argtypes = [C.c_void_p, C.c_uint64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        L.ami_fp64_peak_probe.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ami_tally_static.argtypes = [C.c_int, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        L.ami_strerror.restype = C.c_char_p
        L.ami_strerror.argtypes = [C.c_int]
        L.ami_last_cuda_error.restype = C.c_char_p
        L.ami_kernel_launches.restype = C.c_int64
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        msg = lib().ami_strerror(rc).decode()
        if rc in (-1, -4, -5, -6) and lib().ami_last_cuda_error():
            msg += " [" + lib().ami_last_cuda_error().decode() + "]"
        raise AmiError(rc, msg)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream))


def _host(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _z_host(z_ext, n_ext):
    return np.ascontiguousarray(np.asarray(z_ext, dtype=np.complex128).reshape(-1, max(n_ext, 1)))


class AmiTable:
    """ami_construct: the symbolic result of one labelled diagram, resident on
    ``device`` (a CUDA ordinal) or host-only when ``device`` is None."""

    def __init__(self, n_int, n_ext, alpha, eps, slot_is_fermionic, sum_order=None, prefactor=1.0, device=0):
        alpha = _host(alpha, np.int32)
        eps = _host(eps, np.int32)
        stat = _host(slot_is_fermionic, np.uint8)
        so = None if sum_order is None else _host(sum_order, np.int32)
        if alpha.ndim != 2 or eps.ndim != 2 or alpha.shape[0] != eps.shape[0] or alpha.shape[1] != n_int + n_ext \
                or stat.shape != (n_int + n_ext,):
            raise AmiError(-1, "shape mismatch")
        h = C.c_void_p()
        _check(lib().ami_construct(n_int, n_ext, alpha.shape[0], eps.shape[1], alpha.ctypes.data, eps.ctypes.data,
                                   stat.ctypes.data, None if so is None else so.ctypes.data, float(prefactor),
                                   -1 if device is None else int(device), C.byref(h)))
        self._h = h
        self.device = device
        self.info = self._info()
        self.n_int, self.n_ext, self.n_eps = n_int, n_ext, eps.shape[1]

    @classmethod
    def from_diagram(cls, d, **kw):
        return cls(d.n_int, d.n_ext, d.alpha, d.eps, d.slot_is_fermionic, **kw)

    def close(self):
        if getattr(self, "_h", None):
            lib().ami_table_destroy(self._h)
            self._h = None

    __del__ = close

    def latex(self, factorized=False) -> str:
        """ami_table_latex: the flat term table as LaTeX, or (factorized) the FT * R form with
        the Fermi/Bose sums in Horner form, shared sums named once (ami_table_latex_factorized)."""
        fn = lib().ami_table_latex_factorized if factorized else lib().ami_table_latex
        n = C.c_size_t(0)
        _check(fn(self._h, None, C.byref(n)))
        buf = C.create_string_buffer(n.value)
        _check(fn(self._h, buf, C.byref(n)))
        return buf.value.decode()

    def _info(self) -> dict:
        s = ami_info()
        _check(lib().ami_table_info(self._h, C.byref(s)))
        return {n: getattr(s, n) for n, _ in ami_info._fields_}

    def refresh_info(self) -> dict:
        self.info = self._info()
        return self.info

    # ---- register plan ----------------------------------------------------------------------
    def specialize(self):
        """ami_table_specialize: compile and load the specialised kernels now."""
        _check(lib().ami_table_specialize(self._h))
        return self.refresh_info()

    def kernel_source(self, dim=2, band=BAND_TIGHT_BINDING, complex_energies=False) -> str:
        n = C.c_size_t(0)
        args = (self._h, int(dim), int(band), int(bool(complex_energies)))
        _check(lib().ami_table_kernel_source_variant(*args, None, C.byref(n)))
        buf = C.create_string_buffer(n.value)
        _check(lib().ami_table_kernel_source_variant(*args, buf, C.byref(n)))
        return buf.value.decode()

    def kernel_units(self) -> int:
        """Translation units of the specialised kernels (1 for the register plan, 1 + M for a split plan)."""
        n = C.c_int(0)
        _check(lib().ami_table_kernel_units(self._h, C.byref(n)))
        return n.value

    def kernel_cubin(self, cap=64 << 20, unit=0, dim=2, band=BAND_TIGHT_BINDING, complex_energies=False):
        """(cubin bytes, compiler log) of translation unit ``unit`` of a variant; needs NVRTC but no GPU."""
        buf = C.create_string_buffer(cap)
        log = C.create_string_buffer(1 << 18)
        n = C.c_size_t(cap)
        _check(lib().ami_table_kernel_cubin_variant(self._h, int(dim), int(band), int(bool(complex_energies)), int(unit),
                                                    buf, C.byref(n), log, len(log)))
        return buf.raw[: n.value], log.value.decode()

    def export(self) -> dict:
        """ami_table_export parsed into numpy arrays (layout documented in include/ami.h)."""
        n = C.c_size_t(0)
        _check(lib().ami_table_export(self._h, None, C.byref(n)))
        buf = np.zeros(n.value, dtype=np.uint8)
        _check(lib().ami_table_export(self._h, buf.ctypes.data, C.byref(n)))
        w = buf[: (n.value // 4) * 4].view(np.int32)
        assert w[0] == 0x31494D41
        n_int, n_ext, n_eps, UF, UD, T, mf, nd = (int(x) for x in w[1:9])
        pos = 9

        def take(*shape):
            nonlocal pos
            cnt = int(np.prod(shape)) if shape else 1
            a = w[pos:pos + cnt].reshape(shape).copy()
            pos += cnt
            return a

        out = {"n_int": n_int, "n_ext": n_ext, "n_eps": n_eps,
               "leafF_c": take(UF, n_eps), "leafF_sig": take(UF), "leafF_k": take(UF),
               "leafD_c": take(UD, n_eps), "leafD_a": take(UD, n_ext),
               "fidx": take(T, mf), "didx": take(T, nd)}
        off = (pos * 4 + 7) // 8 * 8
        out["coef"] = buf[off:off + 8 * T].view(np.float64).copy()
        return out

    def export_tree(self) -> dict:
        """ami_table_export_tree parsed: the two programs (uint32 words), the constants, the slot count."""
        n = C.c_size_t(0)
        _check(lib().ami_table_export_tree(self._h, None, C.byref(n)))
        buf = np.zeros(n.value, dtype=np.uint8)
        _check(lib().ami_table_export_tree(self._h, buf.ctypes.data, C.byref(n)))
        w = buf[: (n.value // 4) * 4].view(np.uint32)
        assert w[0] == 0x31544D41
        nb, nf, nc, ns = (int(x) for x in w[1:5])
        off = ((5 + nb + nf) * 4 + 7) // 8 * 8
        return {"code_beta": w[5:5 + nb].copy(), "code_freq": w[5 + nb:5 + nb + nf].copy(),
                "consts": buf[off:off + 8 * nc].view(np.float64).copy(), "n_slots": ns}

    # ---- kernels -------------------------------------------------------------------------
    def dispersion(self, k, q, t, mu, out=None, stream=None, dim=2, band=BAND_TIGHT_BINDING):
        """ami_dispersion (dim = 2, tight binding) / ami_dispersion_lattice.  k: CUDA float64 tensor
        [n][n_int][dim] (Eq. 8 layout) -> e [n_eps][n]."""
        import torch
        assert k.is_cuda and k.dtype == torch.float64 and k.is_contiguous()
        n = k.shape[0]
        if out is None:
            out = torch.empty((self.n_eps, n), dtype=torch.float64, device=k.device)
        qh = _host(np.asarray(q, dtype=np.float64).reshape(max(self.n_ext, 1), dim), np.float64)
        if dim == 2 and band == BAND_TIGHT_BINDING:
            _check(lib().ami_dispersion(self._h, C.c_void_p(k.data_ptr()), 2 * self.n_int, 1, qh.ctypes.data, float(t),
                                        float(mu), n, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        else:
            _check(lib().ami_dispersion_lattice(self._h, C.c_void_p(k.data_ptr()), dim * self.n_int, 1, qh.ctypes.data,
                                                float(t), float(mu), int(dim), int(band), n,
                                                C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def evaluate(self, e, z_ext, beta, e_reg=0.0, plan=PLAN_AUTO, out=None, stream=None):
        """ami_evaluate.  e: CUDA tensor [n_eps][n_e], float64 or complex128 -> complex128
        [n_b][n_f][n_e]."""
        import torch
        assert e.is_cuda and e.is_contiguous() and e.shape[0] == self.n_eps
        is_c = e.dtype == torch.complex128
        assert is_c or e.dtype == torch.float64
        z = _z_host(z_ext, self.n_ext)
        b = _host(np.atleast_1d(beta), np.float64)
        n_e, n_f, n_b = e.shape[1], z.shape[0], b.shape[0]
        if out is None:
            out = torch.empty((n_b, n_f, n_e), dtype=torch.complex128, device=e.device)
        assert out.is_contiguous() and out.dtype == torch.complex128 and out.numel() == n_b * n_f * n_e
        _check(lib().ami_evaluate(self._h, C.c_void_p(e.data_ptr()), int(is_c), n_e, z.ctypes.data, n_f,
                                  b.ctypes.data, n_b, float(e_reg), int(plan), C.c_void_p(out.data_ptr()),
                                  _stream_ptr(stream)))
        return out

    def evaluate_momenta(self, k, q, t, mu, z_ext, beta, e_reg=0.0, plan=PLAN_AUTO, e_out=None, out=None,
                         stream=None, dim=2, band=BAND_TIGHT_BINDING):
        """ami_evaluate_momenta (dim = 2, tight binding) / ami_evaluate_momenta_lattice: S1+S2+S3 for momenta
        k [n][n_int][dim] -> complex128 [n_b][n_f][n].  ``e_out`` ([n_eps][n] float64) receives the energies
        when given (a table-driven plan that needs them as workspace allocates its own otherwise)."""
        import torch
        assert k.is_cuda and k.dtype == torch.float64 and k.is_contiguous()
        n = k.shape[0]
        z = _z_host(z_ext, self.n_ext)
        b = _host(np.atleast_1d(beta), np.float64)
        n_f, n_b = z.shape[0], b.shape[0]
        if out is None:
            out = torch.empty((n_b, n_f, n), dtype=torch.complex128, device=k.device)
        assert out.is_contiguous() and out.dtype == torch.complex128 and out.numel() == n_b * n_f * n
        qh = _host(np.asarray(q, dtype=np.float64).reshape(max(self.n_ext, 1), dim), np.float64)
        e_ptr = None if e_out is None else C.c_void_p(e_out.data_ptr())
        if dim == 2 and band == BAND_TIGHT_BINDING:
            _check(lib().ami_evaluate_momenta(self._h, C.c_void_p(k.data_ptr()), 2 * self.n_int, 1, qh.ctypes.data,
                                              float(t), float(mu), n, z.ctypes.data, n_f, b.ctypes.data, n_b,
                                              float(e_reg), int(plan), e_ptr, C.c_void_p(out.data_ptr()),
                                              _stream_ptr(stream)))
        else:
            _check(lib().ami_evaluate_momenta_lattice(self._h, C.c_void_p(k.data_ptr()), dim * self.n_int, 1,
                                                      qh.ctypes.data, float(t), float(mu), int(dim), int(band), n,
                                                      z.ctypes.data, n_f, b.ctypes.data, n_b, float(e_reg), int(plan),
                                                      e_ptr, C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def generate_momenta(self, seed, first_sample, n, stream=None, dim=2):
        import torch
        k = torch.empty((n, self.n_int, dim), dtype=torch.float64, device=f"cuda:{self.device}")
        _check(lib().ami_generate_momenta_lattice(self._h, int(seed), int(first_sample), n, int(dim),
                                                  C.c_void_p(k.data_ptr()), _stream_ptr(stream)))
        return k

    def run(self, n, q, t, mu, z_ext, beta, e_reg=0.0, plan=PLAN_AUTO, seed=0, first_sample=0, chunk=0,
            h_k=None, d_k=None, h_out=None, d_out=None, want_sum=False, stream=None, dim=2, band=BAND_TIGHT_BINDING):
        """ami_run, the streamed driver.  h_k / h_out are (preferably pinned) CPU tensors or numpy
        arrays; d_k / d_out CUDA tensors.  Returns (stats dict, sums or None)."""
        z = _z_host(z_ext, self.n_ext)
        b = _host(np.atleast_1d(beta), np.float64)
        qh = _host(np.asarray(q, dtype=np.float64).reshape(max(self.n_ext, 1), dim), np.float64)
        cfg = ami_run_cfg()
        cfg.dim, cfg.band = int(dim), int(band)
        cfg.n, cfg.chunk, cfg.seed, cfg.first_sample = int(n), int(chunk), int(seed), int(first_sample)
        ptr = lambda x: None if x is None else (x.ctypes.data if isinstance(x, np.ndarray) else x.data_ptr())
        cfg.h_k, cfg.d_k, cfg.h_out, cfg.d_out = ptr(h_k), ptr(d_k), ptr(h_out), ptr(d_out)
        cfg.q, cfg.t, cfg.mu = qh.ctypes.data, float(t), float(mu)
        cfg.z_ext, cfg.n_f, cfg.beta, cfg.n_b = z.ctypes.data, z.shape[0], b.ctypes.data, b.shape[0]
        cfg.e_reg, cfg.plan, cfg.want_sum = float(e_reg), int(plan), int(bool(want_sum))
        sums = np.zeros((b.shape[0], z.shape[0]), dtype=np.complex128) if want_sum else None
        cfg.h_sum = None if sums is None else sums.ctypes.data
        self.last_sumsq = np.zeros((b.shape[0], z.shape[0], 2)) if want_sum else None   # sums of re^2, im^2
        cfg.h_sumsq = None if self.last_sumsq is None else self.last_sumsq.ctypes.data
        cfg.stream = _stream_ptr(stream)
        st = ami_run_stats()
        _check(lib().ami_run(self._h, C.byref(cfg), C.byref(st)))
        return {n_: getattr(st, n_) for n_, _ in ami_run_stats._fields_}, sums


def read_graph(text_or_path):
    """ami_graph_parse (read_graph): rows ``source target is_fermion spin`` of a diagram
    file, or of its text, as an int32 array [n_edges][4]."""
    text = text_or_path
    if "\n" not in text and os.path.exists(text):
        with open(text) as f:
            text = f.read()
    raw = text.encode()
    n = C.c_int32(0)
    _check(lib().ami_graph_parse(raw, None, 0, C.byref(n)))
    edges = np.zeros((n.value, 4), dtype=np.int32)
    _check(lib().ami_graph_parse(raw, edges.ctypes.data, n.value, C.byref(n)))
    return edges


def label_graph(edges):
    """ami_graph_label (label_graph + graph_to_R0): conserving labels of every line
    and the inputs of ami_construct.  Returns a namespace that AmiTable.from_diagram accepts
    (n_int, n_ext, alpha, eps, slot_is_fermionic) plus alpha_all [n_edges][L] and row_of_g [n_g]."""
    import types
    edges = _host(edges, np.int32).reshape(-1, 4)
    sz = [C.c_int32(0) for _ in range(4)]
    ne = edges.shape[0]
    _check(lib().ami_graph_label(edges.ctypes.data, ne, *[C.byref(x) for x in sz], None, None, None, None, None, 0))
    m, n_ext, n_g, n_eps = (x.value for x in sz)
    L = m + n_ext
    alpha_all = np.zeros((ne, L), dtype=np.int32)
    row_of_g = np.zeros(n_g, dtype=np.int32)
    alpha = np.zeros((n_g, L), dtype=np.int32)
    eps = np.zeros((n_g, n_eps), dtype=np.int32)
    stat = np.zeros(L, dtype=np.uint8)
    cap = max(alpha_all.size, alpha.size, eps.size)
    alpha_all, alpha, eps = (np.zeros(cap, dtype=np.int32) for _ in range(3))
    _check(lib().ami_graph_label(edges.ctypes.data, ne, *[C.byref(x) for x in sz], alpha_all.ctypes.data,
                                 row_of_g.ctypes.data, alpha.ctypes.data, eps.ctypes.data, stat.ctypes.data, cap))
    return types.SimpleNamespace(n_int=m, n_ext=n_ext, n_g=n_g, n_eps=n_eps,
                                 alpha=alpha[:n_g * L].reshape(n_g, L).copy(),
                                 eps=eps[:n_g * n_eps].reshape(n_g, n_eps).copy(), slot_is_fermionic=stat,
                                 alpha_all=alpha_all[:ne * L].reshape(ne, L).copy(), row_of_g=row_of_g, edges=edges)


ORDER_FEWEST_TERMS, ORDER_FEWEST_OPS = 0, 1


def search_sum_order(d, criterion=ORDER_FEWEST_TERMS, max_orders=0):
    """ami_search_sum_order: the order of the sums of diagram ``d`` with the smallest table
    (criterion 0) or the fewest FP64 operations per sample of the factorised form (1).
    Returns (order, cost, cost of the default order or -1, orders accepted)."""
    alpha, eps = _host(d.alpha, np.int32), _host(d.eps, np.int32)
    stat = _host(d.slot_is_fermionic, np.uint8)
    order = np.zeros(d.n_int, dtype=np.int32)
    best, dflt, tried = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    _check(lib().ami_search_sum_order(d.n_int, d.n_ext, alpha.shape[0], eps.shape[1], alpha.ctypes.data,
                                      eps.ctypes.data, stat.ctypes.data, int(criterion), int(max_orders),
                                      order.ctypes.data, C.byref(best), C.byref(dflt), C.byref(tried)))
    return order.tolist(), best.value, dflt.value, tried.value


def kernel_launches() -> int:
    """Kernels launched by the library in this process so far."""
    return int(lib().ami_kernel_launches())


def fp64_peak_probe(device=0, distinct_sources=2):
    """Measured DFMA lane-operations per second of ``device`` (register-only chains): 2 = two distinct register
    sources per DFMA (the pipe's issue rate), 3 = three of which two repeat (operand reuse), 4 = three that change
    from one DFMA to the next (register-file bandwidth), 5 = 4 with integer instructions in between, 6 / 7 = two changing
    register operands and an immediate addend without / with that integer work (include/ami.h)."""
    r, ms = C.c_double(0), C.c_double(0)
    _check(lib().ami_fp64_peak_probe(int(device), int(distinct_sources), C.byref(r), C.byref(ms)))
    return r.value, ms.value


TALLY_STATIC_MAX_ROWS = 1024   # AMI_TALLY_STATIC_MAX_ROWS


def tally_static(vals, tally, stream=None):
    """ami_tally_static, the allocation-free tally: ``vals`` a contiguous complex128 CUDA tensor [..., n] (every
    leading index a row), ``tally`` a contiguous float64 CUDA tensor [rows][4] that receives (sum re, sum im,
    sum re^2, sum im^2) of each row.  Nothing is allocated, by the library or here; at most 1024 rows per call; calls
    that overlap on the GPU race on the library's static workspace."""
    n = int(vals.shape[-1]) if vals.dim() else 1
    rows = int(vals.numel() // n) if n else int(tally.shape[0])
    if not (vals.is_cuda and tally.is_cuda and vals.is_contiguous() and tally.is_contiguous()) or \
            vals.element_size() != 16 or tally.element_size() != 8 or tally.numel() != 4 * rows:
        raise AmiError(-1, "tally_static: vals complex128 [..., n] and tally float64 [rows][4], contiguous CUDA tensors")
    _check(lib().ami_tally_static(int(vals.device.index or 0), C.c_void_p(vals.data_ptr()), rows, n, n,
                                  C.c_void_p(tally.data_ptr()), _stream_ptr(stream)))


def tally_static_setup(device=0):
    """The set-up half of ami_tally_static alone (n_rows = 0): looks up the static workspace of ``device``; call it
    before a stream capture."""
    _check(lib().ami_tally_static(int(device), None, 0, 0, 0, None, None))
