"""Thin ctypes binding of include/lqcd.h (argument marshalling only).

Every function has the name of the C entry point it calls; every step of the path runs in
the CUDA kernels of liblqcd_b200.so.  There is no CPU fallback: if the library is missing
or a call fails, an exception is raised.

Device fields are torch tensors (torch supplies device memory and streams only).
"""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# LQCD_B200_LIB selects another build of the same library (e.g. the index-checked debug build)
LIB_PATH = os.environ.get("LQCD_B200_LIB") or os.path.join(_HERE, "liblqcd_b200.so")

PREC_DOUBLE, PREC_SINGLE, PREC_HALF = 0, 1, 2
RECON_18, RECON_12, RECON_8 = 18, 12, 8
SOLVER_BICGSTAB, SOLVER_GCR_DD, SOLVER_CGNR, SOLVER_CGNE = 0, 1, 2, 3
MATPC_ASYMMETRIC, MATPC_SYMMETRIC = 0, 1
SCHWARZ_ADDITIVE, SCHWARZ_MULTIPLICATIVE = 0, 1
FIELD_SPINOR_PARITY, FIELD_STAGGERED_PARITY = 0, 1
OK, EINVAL, ESTATE, ENOMEM, ECUDA, ENOCONV, EBREAKDOWN = 0, -1, -2, -3, -4, -5, -6

EXPORTS = [
    "lqcd_create", "lqcd_destroy", "lqcd_last_error", "lqcd_release_workspace", "lqcd_load_gauge", "lqcd_build_clover",
    "lqcd_field_bytes", "lqcd_pack_spinor", "lqcd_unpack_spinor", "lqcd_dslash", "lqcd_clover",
    "lqcd_matpc", "lqcd_matpc_sym", "lqcd_dslash_mrhs", "lqcd_matpc_mrhs", "lqcd_schwarz", "lqcd_schwarz_sap", "lqcd_set_schwarz_group", "lqcd_set_schwarz_overlap", "lqcd_invert", "lqcd_invert_mrhs", "lqcd_apply_host", "lqcd_apply_host_c64", "lqcd_invert_host",
    "lqcd_axpy_norm", "lqcd_cdot", "lqcd_cdot_static", "lqcd_launch_count",
    "lqcd_load_staggered_links", "lqcd_pack_staggered", "lqcd_unpack_staggered", "lqcd_staggered_dslash", "lqcd_staggered_mdagm", "lqcd_staggered_multishift",
]


class InvertParams(ctypes.Structure):
    _fields_ = [
        ("kappa", ctypes.c_double), ("c_sw", ctypes.c_double), ("tol", ctypes.c_double), ("delta", ctypes.c_double),
        ("max_iter", ctypes.c_int), ("solver", ctypes.c_int),
        ("prec_outer", ctypes.c_int), ("prec_sloppy", ctypes.c_int), ("prec_precond", ctypes.c_int),
        ("recon_outer", ctypes.c_int), ("recon_sloppy", ctypes.c_int), ("recon_precond", ctypes.c_int),
        ("parity", ctypes.c_int), ("gcr_kmax", ctypes.c_int), ("schwarz_block", ctypes.c_int * 4),
        ("mr_steps", ctypes.c_int), ("mr_omega", ctypes.c_double),
        ("use_initial_guess", ctypes.c_int), ("precondition", ctypes.c_int), ("matpc_type", ctypes.c_int),
        ("schwarz_group", ctypes.c_int), ("schwarz_type", ctypes.c_int), ("sap_cycles", ctypes.c_int), ("history_len", ctypes.c_int),
        ("residual_history", ctypes.POINTER(ctypes.c_double)), ("schwarz_overlap", ctypes.c_int),
    ]


class InvertResult(ctypes.Structure):
    _fields_ = [
        ("status", ctypes.c_int), ("iterations", ctypes.c_int), ("restarts", ctypes.c_int),
        ("matpc_sloppy", ctypes.c_int), ("matpc_outer", ctypes.c_int), ("matpc_precond", ctypes.c_int),
        ("true_residual", ctypes.c_double), ("iterated_residual", ctypes.c_double),
        ("seconds", ctypes.c_double), ("gflop", ctypes.c_double), ("history_count", ctypes.c_int),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class LqcdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("lqcd error %d: %s" % (code, text))
        self.code = code


_lib = None


def load_library():
    """dlopen liblqcd_b200.so; raises if it is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("CUDA extension missing: %s (run __graft_entry__.build())" % LIB_PATH)
        lib = ctypes.CDLL(LIB_PATH)
        vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        sig = {
            "lqcd_create": (i, [ctypes.POINTER(vp), ctypes.POINTER(i), ctypes.POINTER(i), i]),
            "lqcd_destroy": (i, [vp]),
            "lqcd_release_workspace": (i, [vp]),
            "lqcd_last_error": (ctypes.c_char_p, [vp]),
            "lqcd_load_gauge": (i, [vp, vp, vp]),
            "lqcd_build_clover": (i, [vp, d, vp]),
            "lqcd_field_bytes": (ctypes.c_size_t, [vp, i, i]),
            "lqcd_pack_spinor": (i, [vp, vp, vp, i, i, vp]),
            "lqcd_unpack_spinor": (i, [vp, vp, vp, i, i, vp]),
            "lqcd_dslash": (i, [vp, vp, vp, i, i, i, i, vp]),
            "lqcd_clover": (i, [vp, vp, vp, i, i, d, i, vp]),
            "lqcd_matpc": (i, [vp, vp, vp, i, i, d, i, i, vp]),
            "lqcd_matpc_sym": (i, [vp, vp, vp, i, i, d, i, i, vp]),
            "lqcd_dslash_mrhs": (i, [vp, vp, vp, i, i, i, i, i, vp]),
            "lqcd_matpc_mrhs": (i, [vp, vp, vp, i, i, i, d, i, i, vp]),
            "lqcd_schwarz": (i, [vp, vp, vp, i, d, ctypes.POINTER(i), i, d, i, i, i, vp]),
            "lqcd_set_schwarz_group": (i, [vp, i]),
            "lqcd_set_schwarz_overlap": (i, [vp, i]),
            "lqcd_schwarz_sap": (i, [vp, vp, vp, i, d, ctypes.POINTER(i), i, d, i, i, i, i, i, vp]),
            "lqcd_invert": (i, [vp, vp, vp, ctypes.POINTER(InvertParams), ctypes.POINTER(InvertResult), vp]),
            "lqcd_invert_mrhs": (i, [vp, vp, vp, i, ctypes.POINTER(InvertParams), ctypes.POINTER(InvertResult), vp]),
            "lqcd_apply_host": (i, [vp, vp, vp, i, i, i, d, i, i, vp]),
            "lqcd_apply_host_c64": (i, [vp, vp, vp, i, i, i, d, i, i, vp]),
            "lqcd_invert_host": (i, [vp, vp, vp, ctypes.POINTER(InvertParams), ctypes.POINTER(InvertResult), vp]),
            "lqcd_axpy_norm": (i, [vp, d, vp, vp, i, ctypes.POINTER(d), vp]),
            "lqcd_cdot": (i, [vp, vp, vp, i, ctypes.POINTER(d), vp]),
            "lqcd_cdot_static": (i, [vp, vp, vp, i, vp, vp]),
            "lqcd_launch_count": (ctypes.c_longlong, [vp]),
            "lqcd_load_staggered_links": (i, [vp, vp, vp, d, vp]),
            "lqcd_pack_staggered": (i, [vp, vp, vp, i, i, vp]),
            "lqcd_unpack_staggered": (i, [vp, vp, vp, i, i, vp]),
            "lqcd_staggered_dslash": (i, [vp, vp, vp, i, i, vp]),
            "lqcd_staggered_mdagm": (i, [vp, vp, vp, i, d, d, i, vp]),
            "lqcd_staggered_multishift": (i, [vp, vp, vp, i, d, ctypes.POINTER(d), i, d, i, i, ctypes.POINTER(InvertResult), vp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(lib, name)
            f.restype, f.argtypes = res, args
        _lib = lib
    return _lib


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr())


def _i4(v):
    return (ctypes.c_int * 4)(*[int(x) for x in v])


class Context:
    """Owns one lqcd_ctx.  Methods are named after the C entry points they call."""

    def __init__(self, dims, boundary, device=0):
        self.lib = load_library()
        self.dims = tuple(int(x) for x in dims)
        self.device = torch.device("cuda", device)
        h = ctypes.c_void_p()
        rc = self.lib.lqcd_create(ctypes.byref(h), _i4(dims), _i4(boundary), device)
        if rc != OK:
            raise LqcdError(rc, "lqcd_create failed")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.lqcd_destroy(self.h)
            self.h = None

    def release_workspace(self):
        self._check(self.lib.lqcd_release_workspace(self.h))

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise LqcdError(rc, self.lib.lqcd_last_error(self.h).decode())
        return rc

    # -- fields ---------------------------------------------------------------------------------
    def field_bytes(self, prec):
        return self.lib.lqcd_field_bytes(self.h, FIELD_SPINOR_PARITY, prec)

    def new_field(self, prec):
        return torch.empty(self.field_bytes(prec), dtype=torch.uint8, device=self.device)

    def load_gauge(self, U):
        assert U.is_cuda and U.dtype == torch.complex128 and U.is_contiguous()
        self._check(self.lib.lqcd_load_gauge(self.h, _ptr(U), _stream()))

    def build_clover(self, c_sw):
        self._check(self.lib.lqcd_build_clover(self.h, c_sw, _stream()))

    def pack_spinor(self, canonical, parity, prec, out=None):
        assert canonical.is_cuda and canonical.dtype == torch.complex128 and canonical.is_contiguous()
        out = self.new_field(prec) if out is None else out
        self._check(self.lib.lqcd_pack_spinor(self.h, _ptr(out), _ptr(canonical), parity, prec, _stream()))
        return out

    def unpack_spinor(self, canonical, packed, parity, prec):
        assert canonical.is_cuda and canonical.dtype == torch.complex128 and canonical.is_contiguous()
        self._check(self.lib.lqcd_unpack_spinor(self.h, _ptr(canonical), _ptr(packed), parity, prec, _stream()))
        return canonical

    # -- operators ------------------------------------------------------------------------------
    def dslash(self, out, inp, parity_out, dagger, prec, recon):
        self._check(self.lib.lqcd_dslash(self.h, _ptr(out), _ptr(inp), parity_out, int(dagger), prec, recon, _stream()))
        return out

    def clover(self, out, inp, parity, inverse, kappa, prec):
        self._check(self.lib.lqcd_clover(self.h, _ptr(out), _ptr(inp), parity, int(inverse), kappa, prec, _stream()))
        return out

    def matpc(self, out, inp, parity, dagger, kappa, prec, recon):
        self._check(self.lib.lqcd_matpc(self.h, _ptr(out), _ptr(inp), parity, int(dagger), kappa, prec, recon, _stream()))
        return out

    def matpc_sym(self, out, inp, parity, dagger, kappa, prec, recon):
        self._check(self.lib.lqcd_matpc_sym(self.h, _ptr(out), _ptr(inp), parity, int(dagger), kappa, prec, recon, _stream()))
        return out

    def new_fields(self, prec, nrhs):
        """nrhs packed fields back to back (the layout of the *_mrhs calls); row r is field r."""
        return torch.empty((nrhs, self.field_bytes(prec)), dtype=torch.uint8, device=self.device)

    def dslash_mrhs(self, out, inp, nrhs, parity_out, dagger, prec, recon):
        self._check(self.lib.lqcd_dslash_mrhs(self.h, _ptr(out), _ptr(inp), nrhs, parity_out, int(dagger), prec, recon, _stream()))
        return out

    def matpc_mrhs(self, out, inp, nrhs, parity, dagger, kappa, prec, recon):
        self._check(self.lib.lqcd_matpc_mrhs(self.h, _ptr(out), _ptr(inp), nrhs, parity, int(dagger), kappa, prec, recon, _stream()))
        return out

    def schwarz_sap(self, out, inp, parity, kappa, block, n_mr, omega_mr, n_cycle, prec, recon, prec_io, recon_io):
        self._check(self.lib.lqcd_schwarz_sap(self.h, _ptr(out), _ptr(inp), parity, kappa, _i4(block), n_mr, omega_mr, n_cycle,
                                              prec, recon, prec_io, recon_io, _stream()))
        return out

    def set_schwarz_group(self, blocks_per_group):
        self._check(self.lib.lqcd_set_schwarz_group(self.h, int(blocks_per_group)))

    def set_schwarz_overlap(self, overlap):
        self._check(self.lib.lqcd_set_schwarz_overlap(self.h, int(overlap)))

    def schwarz(self, out, inp, parity, kappa, block, n_mr, omega_mr, prec, recon, prec_io):
        self._check(self.lib.lqcd_schwarz(self.h, _ptr(out), _ptr(inp), parity, kappa, _i4(block), n_mr, omega_mr,
                                          prec, recon, prec_io, _stream()))
        return out

    # -- improved staggered ------------------------------------------------------------------------
    def load_staggered_links(self, fat, lng, long_scale=0.0):
        """long_scale != 0: every long link is long_scale x SU(3) (checked) and is stored as 12 reals."""
        for t in (fat, lng):
            assert t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()
        self._check(self.lib.lqcd_load_staggered_links(self.h, _ptr(fat), _ptr(lng), float(long_scale), _stream()))

    def new_staggered_field(self, prec):
        return torch.empty(self.lib.lqcd_field_bytes(self.h, FIELD_STAGGERED_PARITY, prec), dtype=torch.uint8, device=self.device)

    def pack_staggered(self, canonical, parity, prec, out=None):
        assert canonical.is_cuda and canonical.dtype == torch.complex128 and canonical.is_contiguous()
        out = self.new_staggered_field(prec) if out is None else out
        self._check(self.lib.lqcd_pack_staggered(self.h, _ptr(out), _ptr(canonical), parity, prec, _stream()))
        return out

    def unpack_staggered(self, canonical, packed, parity, prec):
        assert canonical.is_cuda and canonical.dtype == torch.complex128 and canonical.is_contiguous()
        self._check(self.lib.lqcd_unpack_staggered(self.h, _ptr(canonical), _ptr(packed), parity, prec, _stream()))
        return canonical

    def staggered_dslash(self, out, inp, parity_out, prec):
        self._check(self.lib.lqcd_staggered_dslash(self.h, _ptr(out), _ptr(inp), parity_out, prec, _stream()))
        return out

    def staggered_mdagm(self, out, inp, parity, mass, sigma, prec):
        self._check(self.lib.lqcd_staggered_mdagm(self.h, _ptr(out), _ptr(inp), parity, mass, sigma, prec, _stream()))
        return out

    def staggered_multishift(self, x, b, parity, mass, sigmas, tol, max_iter=10000, allow_fail=False, multishift_prec=PREC_SINGLE):
        """x: [nshift, T, Z, Y, X, 3], b: [T, Z, Y, X, 3] complex128 device tensors.  One result dict per shift."""
        n = len(sigmas)
        assert x.is_cuda and b.is_cuda and x.dtype == b.dtype == torch.complex128 and x.is_contiguous() and x.shape[0] == n
        sg = (ctypes.c_double * n)(*[float(v) for v in sigmas])
        r = (InvertResult * n)()
        rc = self.lib.lqcd_staggered_multishift(self.h, _ptr(x), _ptr(b), parity, mass, sg, n, tol, max_iter, multishift_prec, r, _stream())
        self._check(rc, allow=(ENOCONV, EBREAKDOWN) if allow_fail else ())
        return [r[k].as_dict() for k in range(n)]

    # -- BLAS-1 ---------------------------------------------------------------------------------
    def axpy_norm(self, a, x, y, prec):
        n = ctypes.c_double(0)
        self._check(self.lib.lqcd_axpy_norm(self.h, a, _ptr(x), _ptr(y), prec, ctypes.byref(n), _stream()))
        return n.value

    def cdot(self, x, y, prec):
        d = (ctypes.c_double * 2)()
        self._check(self.lib.lqcd_cdot(self.h, _ptr(x), _ptr(y), prec, d, _stream()))
        return complex(d[0], d[1])

    def cdot_static(self, x, y, prec, out):
        """lqcd_cdot_static: (re <x,y>, im <x,y>, ||y||^2) into the caller's CUDA float64 tensor `out` (3 elements);
        nothing is allocated, copied or synchronised."""
        assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 3 and out.is_contiguous()
        self._check(self.lib.lqcd_cdot_static(self.h, _ptr(x), _ptr(y), prec, _ptr(out), _stream()))

    # -- solvers --------------------------------------------------------------------------------
    @staticmethod
    def make_params(kappa, c_sw, tol, solver=SOLVER_BICGSTAB, prec=(PREC_DOUBLE, PREC_SINGLE, PREC_HALF),
                    recon=(RECON_18, RECON_12, RECON_12), delta=0.1, max_iter=5000, parity=0, gcr_kmax=16,
                    schwarz_block=(0, 0, 0, 0), mr_steps=10, mr_omega=1.0, use_initial_guess=False, precondition=True,
                    matpc_type=MATPC_ASYMMETRIC, schwarz_group=0, history_len=0, schwarz_type=0, sap_cycles=1, schwarz_overlap=0):
        p = InvertParams()
        p.kappa, p.c_sw, p.tol, p.delta = kappa, c_sw, tol, delta
        p.max_iter, p.solver = max_iter, solver
        p.prec_outer, p.prec_sloppy, p.prec_precond = prec
        p.recon_outer, p.recon_sloppy, p.recon_precond = recon
        p.parity, p.gcr_kmax = parity, gcr_kmax
        for k in range(4):
            p.schwarz_block[k] = int(schwarz_block[k])
        p.mr_steps, p.mr_omega = mr_steps, mr_omega
        p.use_initial_guess, p.precondition = int(use_initial_guess), int(precondition)
        p.matpc_type = int(matpc_type)
        p.schwarz_group = int(schwarz_group)
        p.schwarz_type, p.sap_cycles = int(schwarz_type), int(sap_cycles)
        p.schwarz_overlap = int(schwarz_overlap)
        if history_len > 0:                       # host buffer owned by the params object
            p._history = (ctypes.c_double * int(history_len))()
            p.history_len = int(history_len)
            p.residual_history = ctypes.cast(p._history, ctypes.POINTER(ctypes.c_double))
        return p

    def invert(self, x, b, params, allow_fail=False):
        """x, b: canonical full-lattice complex128 device tensors.  Returns the result dict."""
        assert x.is_cuda and b.is_cuda and x.dtype == b.dtype == torch.complex128
        r = InvertResult()
        rc = self.lib.lqcd_invert(self.h, _ptr(x), _ptr(b), ctypes.byref(params), ctypes.byref(r), _stream())
        self._check(rc, allow=(ENOCONV, EBREAKDOWN) if allow_fail else ())
        d = r.as_dict()
        if params.history_len > 0:
            d["residual_history"] = [params._history[k] for k in range(r.history_count)]
        return d

    def invert_mrhs(self, x, b, params, allow_fail=False):
        """x, b: [nrhs, T, Z, Y, X, 4, 3] complex128 device tensors.  Returns one result dict per source."""
        assert x.is_cuda and b.is_cuda and x.dtype == b.dtype == torch.complex128 and x.is_contiguous() and b.is_contiguous()
        nrhs = b.shape[0]
        r = (InvertResult * nrhs)()
        rc = self.lib.lqcd_invert_mrhs(self.h, _ptr(x), _ptr(b), nrhs, ctypes.byref(params), r, _stream())
        self._check(rc, allow=(ENOCONV, EBREAKDOWN) if allow_fail else ())
        return [r[k].as_dict() for k in range(nrhs)]

    def apply_host(self, out_host, in_host, op, parity, dagger, kappa, prec, recon):
        """out_host, in_host: canonical complex128 (or, for fp32 / half compute, complex64) HOST tensors (pinned for
        full-speed copies); the dtype selects lqcd_apply_host / lqcd_apply_host_c64."""
        assert not out_host.is_cuda and not in_host.is_cuda and out_host.dtype == in_host.dtype
        fn = self.lib.lqcd_apply_host_c64 if in_host.dtype == torch.complex64 else self.lib.lqcd_apply_host
        self._check(fn(self.h, _ptr(out_host), _ptr(in_host), op, parity, int(dagger), kappa, prec, recon, _stream()))
        return out_host

    def invert_host(self, x_host, b_host, params, allow_fail=False):
        assert not x_host.is_cuda and not b_host.is_cuda
        r = InvertResult()
        rc = self.lib.lqcd_invert_host(self.h, _ptr(x_host), _ptr(b_host), ctypes.byref(params), ctypes.byref(r), _stream())
        self._check(rc, allow=(ENOCONV, EBREAKDOWN) if allow_fail else ())
        return r.as_dict()

    def launch_count(self):
        return int(self.lib.lqcd_launch_count(self.h))
