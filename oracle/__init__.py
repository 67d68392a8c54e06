"""CPU oracle (TEST INFRASTRUCTURE ONLY) -- ctypes face of wilson_clover_oracle.cpp.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1109_2935_b200 and shares no
code with the CUDA path.  All arrays are numpy complex128, C-contiguous, in the
canonical layouts of include/lqcd.h:

    gauge   U[mu][t][z][y][x][3][3]      spinor  psi[t][z][y][x][4][3]
    clover  T[t][z][y][x][12][12]        (row = spin*3 + colour)

What each function computes and the passage of the paper it follows is stated in
wilson_clover_oracle.cpp.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wilson_clover_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_SRC_S = os.path.join(_HERE, "staggered_oracle.cpp")
_LIB_S = os.path.join(_HERE, "liboracle_staggered.so")
_lib = None
_lib_s = None

BICGSTAB, GCR_DD, CGNR, CGNE = 0, 1, 2, 3


def build(force=False):
    """Compile the oracle with g++ (OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC])
    if force or not os.path.exists(_LIB_S) or os.path.getmtime(_LIB_S) < os.path.getmtime(_SRC_S):
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _LIB_S, _SRC_S])
    return _LIB


def lib_s():
    """The improved staggered oracle (staggered_oracle.cpp)."""
    global _lib_s
    if _lib_s is None:
        build()
        _lib_s = ctypes.CDLL(_LIB_S)
        _lib_s.ors_cg.restype = ctypes.c_int
    return _lib_s


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_num_threads.restype = ctypes.c_int
        for name in ("orc_bicgstab_pc", "orc_gcr_pc", "orc_gcr_sap_pc", "orc_cgnr_pc", "orc_invert", "orc_invert_sym"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _i4(v):
    return (ctypes.c_int * 4)(*[int(t) for t in v])


def _blk(block):
    return None if block is None else _i4(block)


def num_threads():
    return lib().orc_num_threads()


def dims_of(psi):
    """(X,Y,Z,T) of a canonical spinor psi[t][z][y][x][4][3]."""
    T, Z, Y, X = psi.shape[:4]
    return (X, Y, Z, T)


def gamma(mu):
    """gamma_mu for mu=0..3 (x,y,z,t), gamma5 for mu=4, as a 4x4 complex array."""
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().orc_gamma(ctypes.c_int(mu), _p(out))
    return out


def dslash(psi, U, bc, dagger=False, block=None):
    psi, U = _c(psi), _c(U)
    out = np.empty_like(psi)
    lib().orc_dslash(_p(out), _p(psi), _p(U), _i4(dims_of(psi)), _i4(bc), ctypes.c_int(int(dagger)), _blk(block))
    return out


def clover_term(U, c_sw):
    U = _c(U)
    _, T, Z, Y, X = U.shape[:5]
    out = np.empty((T, Z, Y, X, 12, 12), dtype=np.complex128)
    lib().orc_clover_term(_p(out), _p(U), _i4((X, Y, Z, T)), ctypes.c_double(c_sw))
    return out


def clover_apply(psi, Tcl, kappa, inverse=False, parity=-1):
    psi, Tcl = _c(psi), _c(Tcl)
    out = np.empty_like(psi)
    lib().orc_clover_apply(_p(out), _p(psi), _p(Tcl), _i4(dims_of(psi)), ctypes.c_double(kappa),
                           ctypes.c_int(int(inverse)), ctypes.c_int(parity))
    return out


def M(psi, U, Tcl, bc, kappa, dagger=False, block=None):
    psi, U, Tcl = _c(psi), _c(U), _c(Tcl)
    out = np.empty_like(psi)
    lib().orc_M(_p(out), _p(psi), _p(U), _p(Tcl), _i4(dims_of(psi)), _i4(bc), ctypes.c_double(kappa),
                ctypes.c_int(int(dagger)), _blk(block))
    return out


def matpc(psi, U, Tcl, bc, kappa, parity, dagger=False, block=None):
    psi, U, Tcl = _c(psi), _c(U), _c(Tcl)
    out = np.empty_like(psi)
    lib().orc_matpc(_p(out), _p(psi), _p(U), _p(Tcl), _i4(dims_of(psi)), _i4(bc), ctypes.c_double(kappa),
                    ctypes.c_int(parity), ctypes.c_int(int(dagger)), _blk(block))
    return out


def matpc_sym(psi, U, Tcl, bc, kappa, parity, dagger=False):
    """Symmetric even-odd form: Mhat_s = 1 - kappa^2 A_pp^-1 D A_pbar^-1 D  (= A_pp^-1 Mhat)."""
    psi, U, Tcl = _c(psi), _c(U), _c(Tcl)
    out = np.empty_like(psi)
    lib().orc_matpc_sym(_p(out), _p(psi), _p(U), _p(Tcl), _i4(dims_of(psi)), _i4(bc), ctypes.c_double(kappa),
                        ctypes.c_int(parity), ctypes.c_int(int(dagger)))
    return out


def invert_sym(b, U, Tcl, bc, kappa, parity=0, tol=1e-12, maxit=10000, solver=BICGSTAB):
    """Full-lattice solve of M x = b through the symmetric Schur system.  Returns (x, info)."""
    b, U, Tcl = _c(b), _c(U), _c(Tcl)
    x = np.zeros_like(b)
    it, tr = ctypes.c_int(0), ctypes.c_double(0)
    st = lib().orc_invert_sym(_p(x), _p(b), _p(U), _p(Tcl), _i4(dims_of(b)), _i4(bc), ctypes.c_double(kappa),
                              ctypes.c_int(parity), ctypes.c_double(tol), ctypes.c_int(maxit), ctypes.c_int(solver),
                              ctypes.byref(it), ctypes.byref(tr))
    return x, dict(status=st, iterations=it.value, true_residual=tr.value)


def prepare_source(b, U, Tcl, bc, kappa, parity):
    b, U, Tcl = _c(b), _c(U), _c(Tcl)
    out = np.empty_like(b)
    lib().orc_prepare_source(_p(out), _p(b), _p(U), _p(Tcl), _i4(dims_of(b)), _i4(bc), ctypes.c_double(kappa),
                             ctypes.c_int(parity))
    return out


def reconstruct(xp, b, U, Tcl, bc, kappa, parity):
    x = _c(xp).copy()
    b, U, Tcl = _c(b), _c(U), _c(Tcl)
    lib().orc_reconstruct(_p(x), _p(b), _p(U), _p(Tcl), _i4(dims_of(b)), _i4(bc), ctypes.c_double(kappa),
                          ctypes.c_int(parity))
    return x


def schwarz(r, U, Tcl, bc, kappa, parity, block, n_mr=10, omega_mr=1.0):
    r, U, Tcl = _c(r), _c(U), _c(Tcl)
    out = np.empty_like(r)
    lib().orc_schwarz(_p(out), _p(r), _p(U), _p(Tcl), _i4(dims_of(r)), _i4(bc), ctypes.c_double(kappa),
                      ctypes.c_int(parity), _blk(block), ctypes.c_int(n_mr), ctypes.c_double(omega_mr))
    return out


def schwarz_ras(r, U, Tcl, bc, kappa, parity, block, overlap, n_mr=10, omega_mr=1.0, only_block=-1):
    """Overlapping (restricted) additive Schwarz: every block's domain grown by `overlap` sites, block by block
    (wilson_clover_oracle.cpp schwarz_ras).  only_block >= 0: the contribution of that block alone."""
    r, U, Tcl = _c(r), _c(U), _c(Tcl)
    out = np.empty_like(r)
    rc = lib().orc_schwarz_ras(_p(out), _p(r), _p(U), _p(Tcl), _i4(dims_of(r)), _i4(bc), ctypes.c_double(kappa),
                               ctypes.c_int(parity), _blk(block), ctypes.c_int(overlap), ctypes.c_int(n_mr),
                               ctypes.c_double(omega_mr), ctypes.c_int(only_block))
    if rc:
        raise ValueError("schwarz_ras: a domain would reach around the lattice")
    return out


def schwarz_sap(r, U, Tcl, bc, kappa, parity, block, n_mr=4, omega_mr=1.0, n_cycle=1):
    """Multiplicative Schwarz (SAP) preconditioner: n_cycle cycles over the two block colours (wilson_clover_oracle.cpp)."""
    r, U, Tcl = _c(r), _c(U), _c(Tcl)
    out = np.empty_like(r)
    lib().orc_schwarz_sap(_p(out), _p(r), _p(U), _p(Tcl), _i4(dims_of(r)), _i4(bc), ctypes.c_double(kappa),
                          ctypes.c_int(parity), _blk(block), ctypes.c_int(n_mr), ctypes.c_double(omega_mr), ctypes.c_int(n_cycle))
    return out


def gcr_sap_pc(bhat, U, Tcl, bc, kappa, parity, stop, block, maxit=10000, kmax=16, delta=0.1, n_mr=4, omega_mr=1.0, n_cycle=1):
    """GCR preconditioned by the multiplicative Schwarz procedure on one parity.  Returns (x, info)."""
    bhat, U, Tcl = _c(bhat), _c(U), _c(Tcl)
    x = np.zeros_like(bhat)
    it, rs, rn = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_double(0)
    st = lib().orc_gcr_sap_pc(_p(x), _p(bhat), _p(U), _p(Tcl), _i4(dims_of(bhat)), _i4(bc), ctypes.c_double(kappa),
                              ctypes.c_int(parity), ctypes.c_double(stop), ctypes.c_int(maxit), ctypes.c_int(kmax),
                              ctypes.c_double(delta), _blk(block), ctypes.c_int(n_mr), ctypes.c_double(omega_mr),
                              ctypes.c_int(n_cycle), ctypes.byref(it), ctypes.byref(rs), ctypes.byref(rn))
    return x, dict(status=st, iterations=it.value, restarts=rs.value, residual_norm=rn.value)


def bicgstab_pc(bhat, U, Tcl, bc, kappa, parity, stop, maxit=10000, x0=None):
    """Solve Mhat x = bhat on one parity; stop = absolute residual norm.  Returns (x, info)."""
    bhat, U, Tcl = _c(bhat), _c(U), _c(Tcl)
    x = np.zeros_like(bhat) if x0 is None else _c(x0).copy()
    it, rn = ctypes.c_int(0), ctypes.c_double(0)
    st = lib().orc_bicgstab_pc(_p(x), _p(bhat), _p(U), _p(Tcl), _i4(dims_of(bhat)), _i4(bc), ctypes.c_double(kappa),
                               ctypes.c_int(parity), ctypes.c_double(stop), ctypes.c_int(maxit),
                               ctypes.byref(it), ctypes.byref(rn))
    return x, dict(status=st, iterations=it.value, residual_norm=rn.value)


def gcr_pc(bhat, U, Tcl, bc, kappa, parity, stop, maxit=10000, kmax=16, delta=0.1, precond=True,
           block=None, n_mr=10, omega_mr=1.0, x0=None):
    bhat, U, Tcl = _c(bhat), _c(U), _c(Tcl)
    x = np.zeros_like(bhat) if x0 is None else _c(x0).copy()
    it, rs, rn = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_double(0)
    st = lib().orc_gcr_pc(_p(x), _p(bhat), _p(U), _p(Tcl), _i4(dims_of(bhat)), _i4(bc), ctypes.c_double(kappa),
                          ctypes.c_int(parity), ctypes.c_double(stop), ctypes.c_int(maxit), ctypes.c_int(kmax),
                          ctypes.c_double(delta), ctypes.c_int(int(precond)), _blk(block), ctypes.c_int(n_mr),
                          ctypes.c_double(omega_mr), ctypes.byref(it), ctypes.byref(rs), ctypes.byref(rn))
    return x, dict(status=st, iterations=it.value, restarts=rs.value, residual_norm=rn.value)


def invert(b, U, Tcl, bc, kappa, parity=0, tol=1e-12, maxit=10000, solver=BICGSTAB, kmax=16, delta=0.1,
           block=None, n_mr=10, omega_mr=1.0):
    """Full-lattice solve of M x = b (Eq. 1).  Returns (x, info)."""
    b, U, Tcl = _c(b), _c(U), _c(Tcl)
    x = np.zeros_like(b)
    it, tr = ctypes.c_int(0), ctypes.c_double(0)
    st = lib().orc_invert(_p(x), _p(b), _p(U), _p(Tcl), _i4(dims_of(b)), _i4(bc), ctypes.c_double(kappa),
                          ctypes.c_int(parity), ctypes.c_double(tol), ctypes.c_int(maxit), ctypes.c_int(solver),
                          ctypes.c_int(kmax), ctypes.c_double(delta), _blk(block), ctypes.c_int(n_mr),
                          ctypes.c_double(omega_mr), ctypes.byref(it), ctypes.byref(tr))
    return x, dict(status=st, iterations=it.value, true_residual=tr.value)


# ---------------------------------------------------------------- improved staggered (staggered_oracle.cpp)
def _sdims(chi):
    T, Z, Y, X = chi.shape[:4]
    return (X, Y, Z, T)


def stag_dslash(chi, fat, lng, bc):
    """D chi of PAPER.md Eq. 3 in the reading R13 (anti-Hermitian, staggered phases explicit)."""
    chi, fat, lng = _c(chi), _c(fat), _c(lng)
    out = np.empty_like(chi)
    lib_s().ors_dslash(_p(out), _p(chi), _p(fat), _p(lng), _i4(_sdims(chi)), _i4(bc))
    return out


def stag_M(chi, fat, lng, bc, mass, dagger=False):
    chi, fat, lng = _c(chi), _c(fat), _c(lng)
    out = np.empty_like(chi)
    lib_s().ors_M(_p(out), _p(chi), _p(fat), _p(lng), _i4(_sdims(chi)), _i4(bc), ctypes.c_double(mass), ctypes.c_int(int(dagger)))
    return out


def stag_MdagM(chi, fat, lng, bc, mass, sigma=0.0):
    chi, fat, lng = _c(chi), _c(fat), _c(lng)
    out = np.empty_like(chi)
    lib_s().ors_MdagM(_p(out), _p(chi), _p(fat), _p(lng), _i4(_sdims(chi)), _i4(bc), ctypes.c_double(mass), ctypes.c_double(sigma))
    return out


def stag_cg(b, fat, lng, bc, mass, sigma=0.0, tol=1e-12, maxit=100000):
    """x = (M^dag M + sigma)^-1 b by plain CG (Eq. 4, one shift).  Returns (x, info)."""
    b, fat, lng = _c(b), _c(fat), _c(lng)
    x = np.empty_like(b)
    it, rr = ctypes.c_int(0), ctypes.c_double(0)
    st = lib_s().ors_cg(_p(x), _p(b), _p(fat), _p(lng), _i4(_sdims(b)), _i4(bc), ctypes.c_double(mass), ctypes.c_double(sigma),
                        ctypes.c_double(tol), ctypes.c_int(maxit), ctypes.byref(it), ctypes.byref(rr))
    return x, dict(status=st, iterations=it.value, true_residual=rr.value)
