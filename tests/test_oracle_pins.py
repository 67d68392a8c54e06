"""Pins for the CPU oracle: what the paper and the mathematics fix, independent of the oracle.

Every check here compares oracle/ against a closed form, an invariant or dense linear
algebra (numpy) -- never against the CUDA path and never against the oracle itself.
Citations are PAPER.md lines (arXiv:1109.2935); readings R1..R8 are listed in DESIGN.md.
"""
import numpy as np
import pytest

import oracle
from paper_1109_2935_b200 import inputs

BC = (1, 1, 1, -1)          # periodic x,y,z, antiperiodic t (BASELINE.json config 1)


def _dot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def _gammas():
    return [oracle.gamma(mu) for mu in range(5)]


def _spin_mul(g, psi):
    return np.einsum("ab,...bc->...ac", g, psi)


# ---------------------------------------------------------------- gamma algebra (R2)
def test_gamma_algebra():
    g = _gammas()
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)                       # Hermitian
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2 * np.eye(4) * (mu == nu))        # Clifford
        for s in (+1, -1):                                              # (1 +- g)/2: rank-2 projector
            P = (np.eye(4) + s * g[mu]) / 2
            assert np.allclose(P @ P, P)
            assert np.isclose(np.trace(P).real, 2.0)
    assert np.allclose(g[4], g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g[4], np.diag([1, 1, -1, -1]))                    # chiral basis
    for mu in range(4):
        for nu in range(mu + 1, 4):                                      # sigma_munu block-diagonal
            sig = 0.5j * (g[mu] @ g[nu] - g[nu] @ g[mu])
            assert np.allclose(sig[:2, 2:], 0) and np.allclose(sig[2:, :2], 0)
            assert np.allclose(sig, sig.conj().T)


# ------------------------------------------------ free field: closed form M(p) (Eq. 2; BASELINE.json)
@pytest.mark.parametrize("dims,bc,n", [
    ((4, 6, 2, 8), (1, 1, 1, -1), (1, 2, 1, 3)),
    ((6, 4, 4, 4), (-1, 1, -1, 1), (2, 3, 0, 1)),
    ((4, 4, 4, 4), (1, 1, 1, 1), (0, 0, 0, 0)),
])
def test_plane_wave_closed_form(dims, bc, n):
    X, Y, Z, T = dims
    kappa, c_sw = 0.12, 1.0
    U = inputs.unit_gauge(dims)
    Tcl = oracle.clover_term(U, c_sw)
    assert np.max(np.abs(Tcl)) == 0.0                                   # A = 1 at U = 1
    L = np.array(dims, dtype=float)
    p = 2 * np.pi * (np.array(n) + np.where(np.array(bc) < 0, 0.5, 0.0)) / L
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    rng = np.random.default_rng(5)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = phase[..., None, None] * u
    g = _gammas()
    Mp = np.eye(4, dtype=complex)
    Dp = np.zeros((4, 4), dtype=complex)
    for mu in range(4):
        Dp += (np.eye(4) - g[mu]) * np.exp(1j * p[mu]) + (np.eye(4) + g[mu]) * np.exp(-1j * p[mu])
    Mp = Mp - kappa * Dp
    want = phase[..., None, None] * (Mp @ u)
    got = oracle.M(psi, U, Tcl, bc, kappa)
    assert _rel(got, want) < 1e-14
    # D alone and D^dagger alone
    got_d = oracle.dslash(psi, U, bc)
    assert _rel(got_d, phase[..., None, None] * (Dp @ u)) < 1e-14 or np.allclose(Dp @ u, 0)
    Dpd = Dp.conj().T
    got_dd = oracle.dslash(psi, U, bc, dagger=True)
    assert _rel(got_dd, phase[..., None, None] * (Dpd @ u)) < 1e-14


# --------------------------------------------- gamma5-hermiticity and the dagger flag
@pytest.fixture(scope="module")
def small():
    dims = (4, 2, 6, 4)
    U = inputs.random_gauge(dims, 0.5, 1)
    Tcl = oracle.clover_term(U, 1.0)
    x = inputs.gaussian_spinor(dims, 2)
    y = inputs.gaussian_spinor(dims, 3)
    return dims, U, Tcl, x, y


def test_links_are_su3(small):
    _, U, _, _, _ = small
    UU = np.einsum("...ij,...kj->...ik", U, U.conj())
    assert np.allclose(UU, np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(U), 1.0, atol=1e-13)


def test_gamma5_hermiticity(small):
    dims, U, Tcl, x, y = small
    g5 = oracle.gamma(4)
    kappa = 0.12
    # <x, D y> = <D^dag x, y> with D^dag from the dagger flag, and D^dag = g5 D g5
    Dy = oracle.dslash(y, U, BC)
    Ddx = oracle.dslash(x, U, BC, dagger=True)
    assert abs(_dot(x, Dy) - _dot(Ddx, y)) < 1e-11 * abs(_dot(x, Dy))
    g5Dg5x = _spin_mul(g5, oracle.dslash(_spin_mul(g5, x), U, BC))
    assert _rel(g5Dg5x, Ddx) < 1e-14
    # full M
    My = oracle.M(y, U, Tcl, BC, kappa)
    Mdx = oracle.M(x, U, Tcl, BC, kappa, dagger=True)
    assert abs(_dot(x, My) - _dot(Mdx, y)) < 1e-11 * abs(_dot(x, My))
    assert _rel(_spin_mul(g5, oracle.M(_spin_mul(g5, x), U, Tcl, BC, kappa)), Mdx) < 1e-14
    # even-odd preconditioned operator, both parities
    for p in (0, 1):
        Mh = oracle.matpc(y, U, Tcl, BC, kappa, p)
        Mhd = oracle.matpc(x, U, Tcl, BC, kappa, p, dagger=True)
        mask = (inputs.parity_mask(dims) == p)[..., None, None]
        assert abs(_dot(x * mask, Mh) - _dot(Mhd, y * mask)) < 1e-11 * abs(_dot(x * mask, Mh))
        assert _rel(_spin_mul(g5, oracle.matpc(_spin_mul(g5, x), U, Tcl, BC, kappa, p)), Mhd) < 1e-13


def test_dslash_couples_opposite_parities_only(small):
    dims, U, _, x, _ = small
    par = inputs.parity_mask(dims)
    for p in (0, 1):
        xin = x * (par == p)[..., None, None]
        out = oracle.dslash(xin, U, BC)
        assert np.max(np.abs(out[par == p])) == 0.0                     # PAPER.md:112 (Fig. 1)


# --------------------------------------------- gauge covariance
def test_gauge_covariance(small):
    dims, U, Tcl, x, _ = small
    kappa = 0.12
    g = inputs.random_su3_field(dims, 3)
    Ug = np.empty_like(U)
    for mu in range(4):
        axis = 3 - mu                                                   # U[mu][t][z][y][x]: x is axis 3
        g_fwd = np.roll(g, -1, axis=axis)                               # g(x + mu)
        Ug[mu] = np.einsum("...ij,...jk,...lk->...il", g, U[mu], g_fwd.conj())
    xg = np.einsum("...ij,...sj->...si", g, x)
    Tg = oracle.clover_term(Ug, 1.0)
    lhs = oracle.M(xg, Ug, Tg, BC, kappa)
    rhs = np.einsum("...ij,...sj->...si", g, oracle.M(x, U, Tcl, BC, kappa))
    assert _rel(lhs, rhs) < 1e-13
    # the clover term itself: A'_x = g A_x g^dag in colour
    T6 = Tcl.reshape(Tcl.shape[:4] + (4, 3, 4, 3))
    want = np.einsum("...ab,...sbtc,...dc->...satd", g, T6, g.conj()).reshape(Tcl.shape)
    assert _rel(Tg, want) < 1e-13


# --------------------------------------------- clover term: magnitude AND sign (R4)
def test_clover_abelian_closed_form():
    dims = (4, 6, 2, 2)
    X, Y, Z, T = dims
    k, c_sw, kappa = 1, 1.3, 0.11
    B = 2 * np.pi * k / (X * Y)
    H = np.array([1.0, -1.0, 0.0])
    U = inputs.unit_gauge(dims)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    for c in range(3):
        U[0][..., c, c] = np.exp(-1j * B * y * H[c])
        U[1][..., c, c] = np.where(y == Y - 1, np.exp(1j * B * Y * x * H[c]), 1.0)
    Tcl = oracle.clover_term(U, c_sw)
    g = _gammas()
    sig_xy = 0.5j * (g[0] @ g[1] - g[1] @ g[0])
    assert np.allclose(sig_xy, np.diag([1, -1, 1, -1]))
    want_T = -c_sw * np.kron(sig_xy, np.diag(np.sin(B * H)))           # A = 1 - kappa c_sw sigma_xy (x) sin(BH)
    assert np.max(np.abs(Tcl - want_T)) < 1e-14
    psi = inputs.gaussian_spinor(dims, 7)
    A = np.eye(12) + kappa * want_T
    got = oracle.clover_apply(psi, Tcl, kappa)
    want = np.einsum("ij,...j->...i", A, psi.reshape(psi.shape[:4] + (12,))).reshape(psi.shape)
    assert _rel(got, want) < 1e-14
    got_inv = oracle.clover_apply(got, Tcl, kappa, inverse=True)
    assert _rel(got_inv, psi) < 1e-13


def test_clover_structure(small):
    dims, U, Tcl, x, _ = small
    assert np.allclose(Tcl, np.conj(np.swapaxes(Tcl, -1, -2)), atol=1e-14)       # Hermitian
    assert np.max(np.abs(Tcl[..., :6, 6:])) == 0.0 and np.max(np.abs(Tcl[..., 6:, :6])) == 0.0
    assert np.max(np.abs(oracle.clover_term(U, 0.0))) == 0.0                     # c_sw = 0 => A = 1
    ev = np.linalg.eigvalsh(Tcl.reshape(-1, 12, 12))
    assert np.max(np.abs(ev)) <= 6.0 + 1e-12                                      # ||F|| <= 1 => ||T|| <= 6 c_sw
    assert abs(np.trace(Tcl, axis1=-2, axis2=-1)).max() < 1e-12                  # sigma traceless
    # linear in c_sw
    assert _rel(oracle.clover_term(U, 0.7), 0.7 * Tcl) < 1e-14
    # inverse really inverts, parity masks
    y = oracle.clover_apply(oracle.clover_apply(x, Tcl, 0.12), Tcl, 0.12, inverse=True)
    assert _rel(y, x) < 1e-13
    par = inputs.parity_mask(dims)
    y0 = oracle.clover_apply(x, Tcl, 0.12, parity=0)
    assert np.max(np.abs(y0[par == 1])) == 0.0
    assert _rel(y0[par == 0], oracle.clover_apply(x, Tcl, 0.12)[par == 0]) < 1e-15


# --------------------------------------------- dense linear algebra on 2^4 and 4^4 (c.5, c.7, c.9)
def _dense(apply, shape, cols=None):
    """Dense matrix of a linear map, column by column (only the columns `cols` if given; the others stay 0)."""
    n = int(np.prod(shape))
    Mat = np.empty((n, n), dtype=np.complex128) if cols is None else np.zeros((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for j in (range(n) if cols is None else cols):
        e[j] = 1.0
        Mat[:, j] = apply(e.reshape(shape)).ravel()
        e[j] = 0.0
    return Mat


@pytest.fixture(scope="module")
def tiny():
    dims = (2, 2, 2, 2)
    U = inputs.random_gauge(dims, 0.5, 1)
    Tcl = oracle.clover_term(U, 1.0)
    b = inputs.gaussian_spinor(dims, 2)
    kappa = 0.12
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    return dims, U, Tcl, b, kappa, Md


def test_dense_lu_2to4_bicgstab(tiny):
    dims, U, Tcl, b, kappa, Md = tiny
    assert Md.shape == (192, 192)
    x_lu = np.linalg.solve(Md, b.ravel()).reshape(b.shape)
    for parity in (0, 1):
        x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=parity, tol=1e-13, solver=oracle.BICGSTAB)
        assert info["status"] == 0
        assert info["true_residual"] < 1e-12
        assert _rel(x, x_lu) < 1e-11


def test_dense_schur_complement(tiny):
    dims, U, Tcl, b, kappa, Md = tiny
    par = np.repeat(inputs.parity_mask(dims).ravel(), 12)
    for p in (0, 1):
        ip, iq = np.where(par == p)[0], np.where(par != p)[0]
        Mpp, Mpq, Mqp, Mqq = Md[np.ix_(ip, ip)], Md[np.ix_(ip, iq)], Md[np.ix_(iq, ip)], Md[np.ix_(iq, iq)]
        S = Mpp - Mpq @ np.linalg.solve(Mqq, Mqp)
        got = oracle.matpc(b, U, Tcl, BC, kappa, p).ravel()
        assert np.max(np.abs(got[iq])) == 0.0
        assert _rel(got[ip], S @ b.ravel()[ip]) < 1e-13
        # source preparation and reconstruction
        bh = oracle.prepare_source(b, U, Tcl, BC, kappa, p).ravel()
        want_bh = b.ravel()[ip] - Mpq @ np.linalg.solve(Mqq, b.ravel()[iq])
        assert _rel(bh[ip], want_bh) < 1e-13
        xp = np.zeros_like(b).ravel()
        xp[ip] = np.linalg.solve(S, want_bh)
        xfull = oracle.reconstruct(xp.reshape(b.shape), b, U, Tcl, BC, kappa, p)
        assert _rel(xfull, np.linalg.solve(Md, b.ravel()).reshape(b.shape)) < 1e-12
        # dagger
        Sd = S.conj().T
        gotd = oracle.matpc(b, U, Tcl, BC, kappa, p, dagger=True).ravel()
        assert _rel(gotd[ip], Sd @ b.ravel()[ip]) < 1e-13


@pytest.fixture(scope="module")
def four():
    dims = (4, 4, 4, 4)
    U = inputs.random_gauge(dims, 0.5, 1)
    Tcl = oracle.clover_term(U, 1.0)
    b = inputs.gaussian_spinor(dims, 2)
    kappa = 0.12
    return dims, U, Tcl, b, kappa


def test_dense_lu_4to4_both_solvers(four):
    dims, U, Tcl, b, kappa = four
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    x_lu = np.linalg.solve(Md, b.ravel()).reshape(b.shape)
    x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=0, tol=1e-12, solver=oracle.BICGSTAB)
    assert info["status"] == 0 and info["true_residual"] < 2e-12
    assert _rel(x, x_lu) < 1e-10
    x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=1, tol=1e-12, solver=oracle.GCR_DD,
                            kmax=8, delta=0.1, block=(2, 2, 2, 4), n_mr=4)
    assert info["status"] == 0 and info["true_residual"] < 2e-12
    assert _rel(x, x_lu) < 1e-10
    # kappa-normalisation vs Eq. 2: 2 kappa M^WC = A - kappa D with m = 1/(2 kappa) - 4, A_paper = T/2
    m = 1 / (2 * kappa) - 4
    v = inputs.gaussian_spinor(dims, 9)
    Mwc = -0.5 * oracle.dslash(v, U, BC) + (4 + m) * v + \
        0.5 * (oracle.clover_apply(v, Tcl, 1.0) - v)
    assert _rel(2 * kappa * Mwc, oracle.M(v, U, Tcl, BC, kappa)) < 1e-14


def test_dense_lu_cgnr(four):
    """CGNR: the solution equals the dense LU solution of M x = b on both parities; on
    the dense normal equations A = Mhat^dag Mhat the method is plain CG, whose A-norm error decreases
    monotonically and which ends (in exact arithmetic) after at most dim steps -- checked through the
    iteration count bound and a dense restatement of the first steps."""
    dims, U, Tcl, b, kappa = four
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    x_lu = np.linalg.solve(Md, b.ravel()).reshape(b.shape)
    for parity in (0, 1):
        x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=parity, tol=1e-12, solver=oracle.CGNR)
        assert info["status"] == 0 and info["true_residual"] < 2e-12
        assert _rel(x, x_lu) < 1e-10
    # BiCGstab needs fewer operator applications than CGNR (cond(Mhat^dag Mhat) = cond(Mhat)^2) but both agree
    xb, ib = oracle.invert(b, U, Tcl, BC, kappa, parity=0, tol=1e-12, solver=oracle.BICGSTAB)
    assert _rel(x, xb) < 1e-10
    # dense restatement on the parity-0 Schur system: 3 CG steps on A y = Mhat^dag bhat from y = 0
    par = inputs.parity_mask(dims)
    mask = (par == 0)[..., None, None]
    idx = np.flatnonzero(np.broadcast_to(mask, b.shape).ravel())
    Mh = _dense(lambda v: oracle.matpc(v, U, Tcl, BC, kappa, 0), b.shape)[np.ix_(idx, idx)]
    bhat = oracle.prepare_source(b, U, Tcl, BC, kappa, 0).ravel()[idx]
    A, rhs = Mh.conj().T @ Mh, Mh.conj().T @ bhat
    y = np.zeros_like(rhs); r = rhs.copy(); pvec = r.copy()
    for _ in range(3):
        Ap = A @ pvec
        al = np.vdot(r, r) / np.vdot(pvec, Ap)
        y = y + al * pvec
        rn = r - al * Ap
        pvec = rn + (np.vdot(rn, rn) / np.vdot(r, r)) * pvec
        r = rn
    stop3 = np.linalg.norm(bhat - Mh @ y)
    xo = np.zeros(b.shape, dtype=np.complex128)
    lib = oracle.lib()
    import ctypes
    it, rnorm = ctypes.c_int(0), ctypes.c_double(0)
    bh_full = np.zeros(b.size, dtype=np.complex128); bh_full[idx] = bhat
    st = lib.orc_cgnr_pc(xo.ctypes.data_as(ctypes.c_void_p), bh_full.ctypes.data_as(ctypes.c_void_p),
                         U.ctypes.data_as(ctypes.c_void_p), Tcl.ctypes.data_as(ctypes.c_void_p),
                         (ctypes.c_int * 4)(*dims), (ctypes.c_int * 4)(*BC), ctypes.c_double(kappa), ctypes.c_int(0),
                         ctypes.c_double(0.0), ctypes.c_int(3), ctypes.byref(it), ctypes.byref(rnorm))
    assert st == 1 and it.value == 3                      # stopped by the iteration cap after exactly 3 steps
    assert np.linalg.norm(xo.ravel()[idx] - y) <= 1e-12 * np.linalg.norm(y)
    assert abs(rnorm.value - stop3) <= 1e-12 * stop3


def test_dense_lu_cgne(four):
    """CGNE / Craig's method: dense-LU solution on both parities; its iterates minimise the
    ERROR over the Krylov space of Mhat^dag (Mhat Mhat^dag)^k r0, so the error norm against the dense solution
    decreases monotonically (the residual need not) -- checked on the first 12 iterations."""
    dims, U, Tcl, b, kappa = four
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    x_lu = np.linalg.solve(Md, b.ravel()).reshape(b.shape)
    for parity in (0, 1):
        x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=parity, tol=1e-12, solver=oracle.CGNE)
        assert info["status"] == 0 and info["true_residual"] < 2e-12
        assert _rel(x, x_lu) < 1e-10
    errs = []
    for k in range(1, 13):
        x, info = oracle.invert(b, U, Tcl, BC, kappa, parity=0, tol=1e-30, maxit=k, solver=oracle.CGNE)
        assert info["iterations"] == k
        errs.append(np.linalg.norm((x - x_lu)[inputs.parity_mask(dims) == 0]))
    assert all(e1 < e0 for e0, e1 in zip(errs, errs[1:]))


def test_symmetric_even_odd_form(four):
    """Mhat_s = A_pp^-1 Mhat as dense matrices; the dagger flag is the true adjoint; solving through the
    symmetric system gives the dense-LU solution of M x = b with the full-system criterion met."""
    dims, U, Tcl, b, kappa = four
    par = inputs.parity_mask(dims)
    for p in (0, 1):
        mask = (par == p)[..., None, None]
        idx = np.flatnonzero(np.broadcast_to(mask, b.shape).ravel())
        Mh = _dense(lambda v: oracle.matpc(v, U, Tcl, BC, kappa, p), b.shape, idx)[np.ix_(idx, idx)]
        Ms = _dense(lambda v: oracle.matpc_sym(v, U, Tcl, BC, kappa, p), b.shape, idx)[np.ix_(idx, idx)]
        Msd = _dense(lambda v: oracle.matpc_sym(v, U, Tcl, BC, kappa, p, dagger=True), b.shape, idx)[np.ix_(idx, idx)]
        A = _dense(lambda v: oracle.clover_apply(v, Tcl, kappa, parity=p), b.shape, idx)[np.ix_(idx, idx)]
        assert np.linalg.norm(A @ Ms - Mh) <= 1e-13 * np.linalg.norm(Mh)
        assert np.linalg.norm(Msd - Ms.conj().T) <= 1e-13 * np.linalg.norm(Ms)
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    x_lu = np.linalg.solve(Md, b.ravel()).reshape(b.shape)
    for solver in (oracle.BICGSTAB, oracle.CGNR):
        x, info = oracle.invert_sym(b, U, Tcl, BC, kappa, parity=0, tol=1e-12, solver=solver)
        assert info["status"] == 0 and info["true_residual"] <= 1e-12
        assert _rel(x, x_lu) < 1e-10


# --------------------------------------------- Schwarz preconditioner (c.8)
def test_schwarz_structure(four):
    dims, U, Tcl, b, kappa = four
    blk = (2, 2, 4, 2)
    p = 0
    par = inputs.parity_mask(dims)
    T_, Z_, Y_, X_ = b.shape[:4]
    t, z, y, x = np.meshgrid(np.arange(T_), np.arange(Z_), np.arange(Y_), np.arange(X_), indexing="ij")
    bid = (x // blk[0]) + 2 * ((y // blk[1]) + 2 * ((z // blk[2]) + 1 * (t // blk[3])))
    # (1) Mhat_D equals the dense Schur complement of the block-masked M
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    site_b = np.repeat(bid.ravel(), 12)
    Mcut = np.where(site_b[:, None] == site_b[None, :], Md, 0.0)
    sp = np.repeat(par.ravel(), 12)
    ip, iq = np.where(sp == p)[0], np.where(sp != p)[0]
    S = Mcut[np.ix_(ip, ip)] - Mcut[np.ix_(ip, iq)] @ np.linalg.solve(Mcut[np.ix_(iq, iq)], Mcut[np.ix_(iq, ip)])
    got = oracle.matpc(b, U, Tcl, BC, kappa, p, block=blk).ravel()
    assert _rel(got[ip], S @ b.ravel()[ip]) < 1e-13
    # (2) support on one block stays exactly inside it, for Mhat_D and for K
    src = b * ((bid == 3) & (par == p))[..., None, None]
    out = oracle.matpc(src, U, Tcl, BC, kappa, p, block=blk)
    assert np.max(np.abs(out[bid != 3])) == 0.0
    Kout = oracle.schwarz(src, U, Tcl, BC, kappa, p, blk, n_mr=5)
    assert np.max(np.abs(Kout[bid != 3])) == 0.0 and np.max(np.abs(Kout[par != p])) == 0.0
    # (3) K follows MR step by step: dense restatement with per-block alpha
    rho = (b.ravel() * (sp == p)).copy()
    xk = np.zeros_like(rho)
    Sfull = np.zeros((rho.size, rho.size), dtype=complex)
    Sfull[np.ix_(ip, ip)] = S
    norms = []
    for _ in range(5):
        w = Sfull @ rho
        for bb in np.unique(bid):
            sel = site_b == bb
            ww = np.vdot(w[sel], w[sel]).real
            a = np.vdot(w[sel], rho[sel]) / ww if ww > 0 else 0.0
            xk[sel] += a * rho[sel]
            rho[sel] -= a * w[sel]
        norms.append(np.linalg.norm(rho))
    Kb = oracle.schwarz(b, U, Tcl, BC, kappa, p, blk, n_mr=5).ravel()
    assert _rel(Kb, xk) < 1e-12
    assert all(n2 <= n1 * (1 + 1e-14) for n1, n2 in zip(norms, norms[1:]))       # MR: residual non-increasing
    # (4) K is a useful approximate inverse of Mhat: ||r - Mhat K r|| < ||r||
    r = b * (par == p)[..., None, None]
    res = r - oracle.matpc(oracle.schwarz(r, U, Tcl, BC, kappa, p, blk, n_mr=10), U, Tcl, BC, kappa, p)
    assert np.linalg.norm(res) < 0.5 * np.linalg.norm(r)
    # (5) one block == whole lattice keeps the (anti)periodic wrap: Mhat_D == Mhat
    assert _rel(oracle.matpc(b, U, Tcl, BC, kappa, p, block=dims), oracle.matpc(b, U, Tcl, BC, kappa, p)) < 1e-15


def test_gcr_identities(four):
    """Algorithm 1: plain GCR (K = 1) must reach the dense solution of the
    parity system, and with k_max >= iterations needed there is exactly one restart cycle."""
    dims, U, Tcl, b, kappa = four
    p = 0
    bh = oracle.prepare_source(b, U, Tcl, BC, kappa, p)
    stop = 1e-12 * np.linalg.norm(bh)
    x1, i1 = oracle.gcr_pc(bh, U, Tcl, BC, kappa, p, stop, kmax=64, delta=0.0, precond=False)
    x2, i2 = oracle.gcr_pc(bh, U, Tcl, BC, kappa, p, stop, kmax=5, delta=0.1, precond=False)
    x3, i3 = oracle.bicgstab_pc(bh, U, Tcl, BC, kappa, p, stop)
    assert i1["status"] == 0 and i2["status"] == 0 and i3["status"] == 0
    assert i1["restarts"] == 1
    assert _rel(x1, x3) < 1e-10 and _rel(x2, x3) < 1e-10
    r = bh - oracle.matpc(x2, U, Tcl, BC, kappa, p)
    assert np.linalg.norm(r) <= 1.01 * stop
    # preconditioned converges in fewer outer iterations than unpreconditioned at the same k_max
    x4, i4 = oracle.gcr_pc(bh, U, Tcl, BC, kappa, p, stop, kmax=16, delta=0.1, precond=True, block=(2, 2, 2, 2), n_mr=6)
    x5, i5 = oracle.gcr_pc(bh, U, Tcl, BC, kappa, p, stop, kmax=16, delta=0.1, precond=False)
    assert _rel(x4, x3) < 1e-10
    assert i4["iterations"] < i5["iterations"]


# --------------------------------------------- multiplicative Schwarz, SAP (R16)
def test_schwarz_sap_pins(four):
    """K_sap against what fixes it: (1) with accurate block solves and many cycles the alternating procedure
    converges to the dense solution Mhat^-1 r (a wrong sign or a stale residual between the colours diverges or
    stalls); (2) the first colour sees the original residual, so on colour-0 blocks one cycle equals the (densely
    pinned) additive K, and the second colour equals the additive K of the residual updated with the FULL operator;
    (3) support and parity; (4) GCR preconditioned by K_sap reproduces the dense LU solution of M x = b."""
    dims, U, Tcl, b, kappa = four
    blk, p = (2, 2, 2, 2), 0
    par = inputs.parity_mask(dims)
    T_, Z_, Y_, X_ = b.shape[:4]
    t, z, y, x = np.meshgrid(np.arange(T_), np.arange(Z_), np.arange(Y_), np.arange(X_), indexing="ij")
    colour = ((x // blk[0]) + (y // blk[1]) + (z // blk[2]) + (t // blk[3])) & 1
    r = b * (par == p)[..., None, None]
    # (1) dense Schur complement solve
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    sp = np.repeat(par.ravel(), 12)
    ip, iq = np.where(sp == p)[0], np.where(sp != p)[0]
    S = Md[np.ix_(ip, ip)] - Md[np.ix_(ip, iq)] @ np.linalg.solve(Md[np.ix_(iq, iq)], Md[np.ix_(iq, ip)])
    want = np.zeros(r.size, dtype=complex)
    want[ip] = np.linalg.solve(S, r.ravel()[ip])
    got = oracle.schwarz_sap(r, U, Tcl, BC, kappa, p, blk, n_mr=60, n_cycle=40).ravel()
    assert _rel(got, want) < 1e-9
    e1 = _rel(oracle.schwarz_sap(r, U, Tcl, BC, kappa, p, blk, n_mr=60, n_cycle=1).ravel(), want)
    e3 = _rel(oracle.schwarz_sap(r, U, Tcl, BC, kappa, p, blk, n_mr=60, n_cycle=3).ravel(), want)
    assert e3 < e1 < 1.0                                        # the procedure contracts the error
    # (2) one cycle, colour by colour, against the additive K and the full operator
    m0, m1 = (colour == 0)[..., None, None], (colour == 1)[..., None, None]
    ks = oracle.schwarz_sap(r, U, Tcl, BC, kappa, p, blk, n_mr=5, n_cycle=1)
    y0 = oracle.schwarz(r * m0, U, Tcl, BC, kappa, p, blk, n_mr=5)
    assert np.max(np.abs(y0 * m1)) == 0.0
    assert _rel((ks * m0), y0) < 1e-13
    r1 = r - oracle.matpc(y0, U, Tcl, BC, kappa, p)
    y1 = oracle.schwarz(r1 * m1, U, Tcl, BC, kappa, p, blk, n_mr=5)
    assert _rel((ks * m1), y1) < 1e-13
    assert _rel((ks * m1), oracle.schwarz(r * m1, U, Tcl, BC, kappa, p, blk, n_mr=5)) > 1e-3    # and not the additive one
    # (3) parity
    assert np.max(np.abs(ks[par != p])) == 0.0
    # (4) GCR-SAP solve
    bhat = oracle.prepare_source(b, U, Tcl, BC, kappa, p)
    xg, ig = oracle.gcr_sap_pc(bhat, U, Tcl, BC, kappa, p, 1e-12 * np.linalg.norm(b), blk, n_mr=4, n_cycle=1)
    xs = np.zeros(r.size, dtype=complex)
    xs[ip] = np.linalg.solve(S, bhat.ravel()[ip])
    assert ig["status"] == 0 and _rel(xg.ravel(), xs) < 1e-10
    xa, ia = oracle.gcr_pc(bhat, U, Tcl, BC, kappa, p, 1e-12 * np.linalg.norm(b), block=blk, n_mr=4)
    assert ig["iterations"] <= ia["iterations"]                   # multiplicative beats additive per outer iteration here


def test_schwarz_ras_pins():
    """Overlapping restricted additive Schwarz (reading R18) against what fixes it, on 6x2x2x8 with blocks 2x2x2x4
    (partitioned in x and t, antiperiodic t, domains that reach through the lattice's wrap): (1) no overlap = the
    densely pinned K; (2) block by block, a dense restatement: the domain built from coordinates here, M cut to the
    domain entry by entry, its Schur complement on parity p, MR with one alpha, restriction to the block's own box;
    (3) the blocks add up; (4) support and parity; (5) a domain that would reach around the lattice is refused."""
    dims, kappa, p = (6, 2, 2, 8), 0.12, 0
    blk, ovl = (2, 2, 2, 4), 1
    U = inputs.random_gauge(dims, 0.5, 3)
    Tcl = oracle.clover_term(U, 1.0)
    b = inputs.gaussian_spinor(dims, 4)
    par = inputs.parity_mask(dims)
    r = b * (par == p)[..., None, None]
    # (1)
    assert _rel(oracle.schwarz_ras(r, U, Tcl, BC, kappa, p, blk, 0, n_mr=4), oracle.schwarz(r, U, Tcl, BC, kappa, p, blk, n_mr=4)) < 1e-14
    # (2)
    Md = _dense(lambda v: oracle.M(v, U, Tcl, BC, kappa), b.shape)
    T_, Z_, Y_, X_ = b.shape[:4]
    t, z, y, x = np.meshgrid(np.arange(T_), np.arange(Z_), np.arange(Y_), np.arange(X_), indexing="ij")
    sp = np.repeat(par.ravel(), 12)
    total = np.zeros(r.size, dtype=complex)
    nbx, nbt = dims[0] // blk[0], dims[3] // blk[3]
    for bt in range(nbt):
        for bx in range(nbx):
            box = bx + nbx * bt                                   # y, z are not partitioned
            dx, dt = (x - bx * blk[0]) % dims[0], (t - bt * blk[3]) % dims[3]
            own = (dx < blk[0]) & (dt < blk[3])
            dom = ((dx < blk[0] + ovl) | (dx >= dims[0] - ovl)) & ((dt < blk[3] + ovl) | (dt >= dims[3] - ovl))
            assert dom.sum() == (blk[0] + 2) * 2 * 2 * (blk[3] + 2) and (own & ~dom).sum() == 0
            sd = np.repeat(dom.ravel(), 12)
            ip, iq = np.where(sd & (sp == p))[0], np.where(sd & (sp != p))[0]
            S = Md[np.ix_(ip, ip)] - Md[np.ix_(ip, iq)] @ np.linalg.solve(Md[np.ix_(iq, iq)], Md[np.ix_(iq, ip)])
            rho = r.ravel()[ip].copy()
            xb = np.zeros_like(rho)
            for _ in range(3):
                w = S @ rho
                a = np.vdot(w, rho) / np.vdot(w, w).real
                xb += a * rho
                rho -= a * w
            want = np.zeros(r.size, dtype=complex)
            want[ip] = xb
            want *= np.repeat(own.ravel(), 12)
            got = oracle.schwarz_ras(r, U, Tcl, BC, kappa, p, blk, ovl, n_mr=3, only_block=box).ravel()
            assert _rel(got, want) < 1e-12, box
            total += want
    # (3), (4)
    full = oracle.schwarz_ras(r, U, Tcl, BC, kappa, p, blk, ovl, n_mr=3)
    assert _rel(full.ravel(), total) < 1e-12
    assert np.max(np.abs(full[par != p])) == 0.0
    # the overlap changes the result (it is not silently ignored) and still approximates Mhat^-1
    assert _rel(full, oracle.schwarz(r, U, Tcl, BC, kappa, p, blk, n_mr=3)) > 1e-3
    res = r - oracle.matpc(oracle.schwarz_ras(r, U, Tcl, BC, kappa, p, blk, ovl, n_mr=10), U, Tcl, BC, kappa, p)
    assert np.linalg.norm(res) < 0.5 * np.linalg.norm(r)
    # (5)
    with pytest.raises(ValueError):
        oracle.schwarz_ras(r, U, Tcl, BC, kappa, p, blk, 2)       # x: 2 + 4 = 6 = L
