"""GPU solver parity (-m gpu): lqcd_invert / lqcd_schwarz through the C ABI against the oracle.

Iterates and iteration counts differ between precisions and implementations (several correct
answers); what is unique is compared: the solution x = M^-1 b (<= 1e-8 relative) and the true
residual ||b - M x||/||b|| recomputed by the ORACLE's operator (<= 1e-10).
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs
from test_gpu_parity import Case, _rel, BC

pytestmark = pytest.mark.gpu


def _solve(c, b, params):
    x = torch.zeros(b.shape, dtype=torch.complex128, device="cuda")
    info = c.ctx.invert(x, torch.from_numpy(b).cuda(), params)
    torch.cuda.synchronize()
    return x.cpu().numpy(), info


@pytest.fixture(scope="module")
def cfg1():
    return Case((4, 4, 4, 4), 0.5)


@pytest.fixture(scope="module")
def mid():
    return Case((8, 8, 8, 16), 0.2)


def test_cfg1_bicgstab_fp64(cfg1):
    """BASELINE.json config 1: 4^4, kappa = 0.12, c_sw = 1, BiCGstab to 1e-12."""
    c = cfg1
    lq = c.lqcd
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, 0.12, parity=0, tol=1e-12)
    assert io["status"] == 0
    for parity in (0, 1):
        p = c.ctx.make_params(0.12, 1.0, 1e-12, solver=lq.SOLVER_BICGSTAB, prec=(0, 0, 0), recon=(18, 18, 18), parity=parity)
        x, info = _solve(c, b, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-12
        res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, 0.12)) / np.linalg.norm(b)
        assert res <= 2e-12
        assert _rel(x, xo) <= 1e-10


@pytest.mark.parametrize("sloppy,recon", [(1, 12), (2, 12), (1, 8), (2, 18)])
def test_mixed_precision_bicgstab(mid, sloppy, recon):
    c = mid
    lq = c.lqcd
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 2)
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_BICGSTAB, prec=(0, sloppy, sloppy), recon=(18, recon, recon))
    x, info = _solve(c, b, p)
    assert info["status"] == 0 and info["true_residual"] <= 1e-10
    assert info["restarts"] >= 1
    res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
    assert res <= 1.05e-10
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    assert _rel(x, xo) <= 1e-8


def test_schwarz_matches_oracle(mid):
    c = mid
    kappa, blk = 0.124, (4, 4, 4, 8)
    r = inputs.gaussian_spinor(c.dims, 4)
    for parity in (0, 1):
        # Dirichlet operator alone, through K with one MR step: K r = alpha_b r per block
        want1 = oracle.schwarz(r, c.U, c.T, c.bc, kappa, parity, blk, n_mr=1)
        want5 = oracle.schwarz(r, c.U, c.T, c.bc, kappa, parity, blk, n_mr=5)
        for prec, t1, t5 in ((0, 1e-12, 1e-11), (1, 1e-5, 5e-5), (2, 5e-3, 2e-2)):
            got1 = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, parity, kappa, blk, 1, 1.0, prec, 12, 0), r, parity, parity, 0)
            got5 = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, parity, kappa, blk, 5, 1.0, prec, 12, 0), r, parity, parity, 0)
            assert _rel(got1, want1) <= t1, (parity, prec)
            assert _rel(got5, want5) <= t5, (parity, prec)
    # support on one block stays exactly inside it (bitwise zero elsewhere), even in half precision
    T_, Z_, Y_, X_ = r.shape[:4]
    t, z, y, x = np.meshgrid(np.arange(T_), np.arange(Z_), np.arange(Y_), np.arange(X_), indexing="ij")
    inside = (x // 4 == 1) & (y // 4 == 0) & (z // 4 == 1) & (t // 8 == 1)
    src = r * inside[..., None, None]
    got = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, 0, kappa, blk, 4, 1.0, 2, 12, 1), src, 0, 0, 1)
    assert np.max(np.abs(got[~inside])) == 0.0
    assert np.max(np.abs(got[inside])) > 0.0


@pytest.mark.parametrize("sloppy,precond", [(0, 0), (1, 2), (2, 2)])
def test_gcr_dd(mid, sloppy, precond):
    c = mid
    lq = c.lqcd
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 2)
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, prec=(0, sloppy, precond), recon=(18, 12, 12),
                          gcr_kmax=16, schwarz_block=(4, 4, 4, 8), mr_steps=10, delta=0.1)
    x, info = _solve(c, b, p)
    assert info["status"] == 0 and info["true_residual"] <= 1e-10
    res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
    assert res <= 1.05e-10
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    assert _rel(x, xo) <= 1e-8
    # unpreconditioned GCR needs more outer iterations than GCR-DD
    if sloppy == 0:
        p2 = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, prec=(0, 0, 0), recon=(18, 18, 18),
                               gcr_kmax=16, precondition=False)
        x2, info2 = _solve(c, b, p2)
        assert info2["true_residual"] <= 1e-10 and _rel(x2, xo) <= 1e-8
        assert info["iterations"] < info2["iterations"]
        # fp64 GCR-DD follows Algorithm 1 like the oracle: same number of outer iterations (+-1)
        xo2, io2 = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-10, solver=oracle.GCR_DD, kmax=16,
                                 delta=0.1, block=(4, 4, 4, 8), n_mr=10)
        assert abs(io2["iterations"] - info["iterations"]) <= 1


def test_invert_host_and_apply_host(cfg1):
    c = cfg1
    lq = c.lqcd
    b = inputs.gaussian_spinor(c.dims, 2)
    bh = torch.from_numpy(b).pin_memory()
    xh = torch.zeros_like(bh).pin_memory()
    p = c.ctx.make_params(0.12, 1.0, 1e-12, prec=(0, 1, 1), recon=(18, 12, 12))
    info = c.ctx.invert_host(xh, bh, p)
    assert info["true_residual"] <= 1e-12
    res = np.linalg.norm(b - oracle.M(xh.numpy(), c.U, c.T, c.bc, 0.12)) / np.linalg.norm(b)
    assert res <= 2e-12
    out = torch.zeros_like(bh).pin_memory()
    c.ctx.apply_host(out, bh, 0, 0, False, 0.12, 0, 18)
    assert _rel(out.numpy(), oracle.dslash(b, c.U, c.bc)) <= 1e-13
    c.ctx.apply_host(out, bh, 1, 1, True, 0.12, 0, 12)
    assert _rel(out.numpy(), oracle.matpc(b, c.U, c.T, c.bc, 0.12, 1, dagger=True)) <= 1e-13


def test_apply_host_slab_pipeline_equals_device_path():
    """lqcd_apply_host (t-slab pipeline, HOST buffers) against the device-resident calls on a ragged
    lattice with 8 slabs: bit-identical in every precision (same kernels on site sub-ranges), and
    within the operator tolerance of the oracle."""
    c = Case((6, 4, 10, 8), 0.3, bc=(-1, 1, 1, -1))
    kappa = 0.124
    psi = inputs.gaussian_spinor(c.dims, 7)
    hin = torch.from_numpy(psi).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    d = torch.from_numpy(psi).cuda()
    for prec, tol in ((0, 1e-13), (1, 1e-5), (2, 5e-3)):
        for dagger in (False, True):
            # op 0: D on both parities
            hout.fill_(7.0)
            c.ctx.apply_host(hout, hin, 0, 0, dagger, kappa, prec, 12)
            ref = torch.zeros_like(d)
            for p in (0, 1):
                fo = c.ctx.new_field(prec)
                c.ctx.dslash(fo, c.ctx.pack_spinor(d, 1 - p, prec), p, dagger, prec, 12)
                c.ctx.unpack_spinor(ref, fo, p, prec)
            assert torch.equal(hout, ref.cpu())
            assert _rel(hout.numpy(), oracle.dslash(psi, c.U, c.bc, dagger=dagger)) <= tol
            # op 1: Mhat on one parity, zero elsewhere
            for parity in (0, 1):
                hout.fill_(7.0)
                c.ctx.apply_host(hout, hin, 1, parity, dagger, kappa, prec, 12)
                ref = torch.zeros_like(d)
                fo = c.ctx.new_field(prec)
                c.ctx.matpc(fo, c.ctx.pack_spinor(d, parity, prec), parity, dagger, kappa, prec, 12)
                c.ctx.unpack_spinor(ref, fo, parity, prec)
                assert torch.equal(hout, ref.cpu())
                assert _rel(hout.numpy(), oracle.matpc(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)) <= tol


def test_cfg4_full_size_solves_true_residual_by_oracle():
    """BASELINE.json config 4 at full size (32^3x64, eps = 0.2, kappa = 0.124, c_sw = 1, Gaussian source):
    mixed-precision BiCGstab (inner fp32 and half) and GCR-DD to 1e-10; the true residual
    ||b - M x|| / ||b|| is recomputed with the ORACLE's full-lattice operator.  (The oracle's own
    solve at this size takes minutes; x = M^-1 b is unique, so the residual pins it.)"""
    from paper_1109_2935_b200 import lqcd
    dims, kappa = (32, 32, 32, 64), 0.124
    Ut = inputs.random_gauge_torch(dims, 0.2, 11, device="cuda")
    bt = inputs.gaussian_spinor_torch(dims, 12, device="cuda")
    ctx = lqcd.Context(dims, BC, 0)
    ctx.load_gauge(Ut)
    ctx.build_clover(1.0)
    U, b = Ut.cpu().numpy(), bt.cpu().numpy()
    del Ut
    T = oracle.clover_term(U, 1.0)
    bn = np.linalg.norm(b)
    runs = [(lqcd.SOLVER_BICGSTAB, (0, 1, 1), {}), (lqcd.SOLVER_BICGSTAB, (0, 2, 2), {}),
            (lqcd.SOLVER_GCR_DD, (0, 1, 2), dict(gcr_kmax=16, schwarz_block=(8, 8, 8, 16), mr_steps=10))]
    for solver, prec, kw in runs:
        p = ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=prec, recon=(18, 12, 12), **kw)
        x = torch.zeros_like(bt)
        info = ctx.invert(x, bt, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-10
        res = np.linalg.norm(b - oracle.M(x.cpu().numpy(), U, T, BC, kappa)) / bn
        assert res <= 1.05e-10, (solver, prec, res)
        assert abs(res - info["true_residual"]) <= 0.05 * res      # the library's fp64 residual is the oracle's
    ctx.close()


def test_cfg5_full_size_gcr_dd_and_bicgstab_true_residual_by_oracle():
    """BASELINE.json config 5 at full size (48^3x96 = 10.6 M sites, eps = 0.2, kappa = 0.124, c_sw = 1, Gaussian
    source, seeds 21 / 22): GCR(16)-DD with 256 Schwarz blocks of 12^3x24 and 10 MR steps in half precision
    (fp64 outer; sloppy fp32 and the paper's single-half-half flavour, sloppy half), against
    mixed-precision BiCGstab on the same system (Figs. 7-8), all to 1e-10.  The true residual
    ||b - M x|| / ||b|| is recomputed with the ORACLE's full-lattice operator (x = M^-1 b is unique, so the
    residual pins it; the oracle's own solve at this size would take an hour), and the solvers' solutions
    must agree with each other to 1e-8."""
    from paper_1109_2935_b200 import lqcd
    dims, kappa, blk = (48, 48, 48, 96), 0.124, (12, 12, 12, 24)
    Ut = inputs.random_gauge_torch(dims, 0.2, 21, device="cuda")
    bt = inputs.gaussian_spinor_torch(dims, 22, device="cuda")
    ctx = lqcd.Context(dims, BC, 0)
    ctx.load_gauge(Ut)
    ctx.build_clover(1.0)
    U, b = Ut.cpu().numpy(), bt.cpu().numpy()
    del Ut
    T = oracle.clover_term(U, 1.0)
    bn = np.linalg.norm(b)
    runs = [("gcr-dd fp64/fp32/half", lqcd.SOLVER_GCR_DD, (0, 1, 2), dict(gcr_kmax=16, schwarz_block=blk, mr_steps=10)),
            ("gcr-dd fp64/half/half", lqcd.SOLVER_GCR_DD, (0, 2, 2), dict(gcr_kmax=16, schwarz_block=blk, mr_steps=10)),
            ("bicgstab fp64/half", lqcd.SOLVER_BICGSTAB, (0, 2, 2), {}),
            ("bicgstab fp64/fp32", lqcd.SOLVER_BICGSTAB, (0, 1, 1), {})]
    xs = []
    for name, solver, prec, kw in runs:
        p = ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=prec, recon=(18, 12, 12), **kw)
        x = torch.zeros_like(bt)
        info = ctx.invert(x, bt, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-10, (name, info)
        xh = x.cpu().numpy()
        res = np.linalg.norm((b - oracle.M(xh, U, T, BC, kappa)).ravel()) / bn
        assert res <= 1.05e-10, (name, res)
        assert abs(res - info["true_residual"]) <= 0.05 * res, (name, res, info["true_residual"])
        if solver == lqcd.SOLVER_GCR_DD:
            assert info["matpc_precond"] == 10 * info["iterations"]          # 10 MR steps per outer iteration
        xs.append(x)
        del xh
    for x in xs[1:]:
        assert float(torch.linalg.vector_norm(x - xs[0]) / torch.linalg.vector_norm(xs[0])) <= 1e-8
    ctx.close()


@pytest.mark.parametrize("prec", [(0, 0, 0), (0, 1, 1), (0, 2, 2)])
def test_cgnr(mid, prec):
    """CGNR in fp64 and mixed precision: same unique solution as the oracle's solve, true
    residual by the oracle's operator; in fp64 the iteration count equals the oracle's CGNR (+-1: same
    recurrence, different summation order); CGNR needs more operator applications than BiCGstab."""
    c = mid
    lq = c.lqcd
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 2)
    for parity in (0, 1):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_CGNR, prec=prec, recon=(18, 12, 12), parity=parity)
        x, info = _solve(c, b, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-10
        res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
        assert res <= 1.05e-10
        xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=parity, tol=1e-10, solver=oracle.CGNR)
        assert _rel(x, xo) <= 1e-8
        if prec == (0, 0, 0):
            assert abs(info["iterations"] - io["iterations"]) <= 1
            assert info["matpc_sloppy"] == 2 * info["iterations"]      # Mhat^dag r0, then (Mhat p, Mhat^dag r) per step, none after the last
    pb = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_BICGSTAB, prec=prec, recon=(18, 12, 12))
    xb, ib = _solve(c, b, pb)
    assert ib["matpc_sloppy"] < info["matpc_sloppy"]


def test_symmetric_even_odd_form(mid):
    """LQCD_MATPC_SYMMETRIC: lqcd_matpc_sym against the oracle's Mhat_s (and its adjoint) in every precision;
    BiCGstab and CGNR through the symmetric system reach the same unique solution with the FULL-system
    criterion ||b - M x|| <= tol ||b|| (oracle's operator); GCR-DD refuses it."""
    c = mid
    lq = c.lqcd
    kappa = 0.124
    psi = inputs.gaussian_spinor(c.dims, 3)
    for prec, tol in ((0, 1e-13), (1, 1e-5), (2, 5e-3)):
        for parity in (0, 1):
            for dagger in (False, True):
                want = oracle.matpc_sym(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)
                got = c.gpu_parity_op(lambda o, i: c.ctx.matpc_sym(o, i, parity, dagger, kappa, prec, 12), psi, parity, parity, prec)
                assert _rel(got, want) <= tol, (prec, parity, dagger)
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    for solver in (lq.SOLVER_BICGSTAB, lq.SOLVER_CGNR):
        for prec in ((0, 0, 0), (0, 1, 1), (0, 2, 2)):
            p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=prec, recon=(18, 12, 12), matpc_type=lq.MATPC_SYMMETRIC)
            x, info = _solve(c, b, p)
            assert info["status"] == 0 and info["true_residual"] <= 1e-10
            res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
            assert res <= 1.05e-10, (solver, prec, res)
            assert _rel(x, xo) <= 1e-8
    xs, isym = oracle.invert_sym(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-10)
    assert _rel(xs, xo) <= 1e-8
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, schwarz_block=(4, 4, 4, 8), matpc_type=lq.MATPC_SYMMETRIC)
    with pytest.raises(lq.LqcdError) as e:
        _solve(c, b, p)
    assert e.value.code == lq.EINVAL


@pytest.mark.parametrize("prec", [(0, 0, 0), (0, 1, 1), (0, 2, 2)])
def test_cgne(mid, prec):
    """CGNE / Craig's method, fp64 and mixed precision, both even-odd forms: the oracle's
    solution and the full-system residual by the oracle's operator; in fp64 the iteration count of the
    oracle's CGNE (+-1)."""
    c = mid
    lq = c.lqcd
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-10, solver=oracle.CGNE)
    for mt in (lq.MATPC_ASYMMETRIC, lq.MATPC_SYMMETRIC):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_CGNE, prec=prec, recon=(18, 12, 12), matpc_type=mt)
        x, info = _solve(c, b, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-10
        res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
        assert res <= 1.05e-10
        assert _rel(x, xo) <= 1e-8
        if prec == (0, 0, 0) and mt == lq.MATPC_ASYMMETRIC:
            assert abs(info["iterations"] - io["iterations"]) <= 1


def test_beyond_critical_kappa_cgnr_converges_where_bicgstab_does_not():
    """kappa = 0.138 on these rough links is beyond kappa_c: M is indefinite.  BiCGstab (the oracle's plain fp64
    one as well) does not converge there; it must end with LQCD_ENOCONV or LQCD_EBREAKDOWN and an honest true
    residual, never with a false success.  CGNR and GCR-DD converge to the oracle's solution."""
    c = Case((8, 8, 8, 16), 0.2)
    lq = c.lqcd
    kappa = 0.138
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-10, solver=oracle.CGNR)
    assert io["status"] == 0
    for solver, kw in ((lq.SOLVER_CGNR, {}), (lq.SOLVER_CGNE, {}), (lq.SOLVER_GCR_DD, dict(schwarz_block=(4, 4, 4, 8), mr_steps=4))):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=(0, 1, 2), recon=(18, 12, 12), max_iter=5000, **kw)
        x, info = _solve(c, b, p)
        assert info["status"] == 0
        assert np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b) <= 1.05e-10
        assert _rel(x, xo) <= 1e-7
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_BICGSTAB, prec=(0, 2, 2), recon=(18, 12, 12), max_iter=400)
    x = torch.zeros(b.shape, dtype=torch.complex128, device="cuda")
    info = c.ctx.invert(x, torch.from_numpy(b).cuda(), p, allow_fail=True)
    if info["status"] == 0:
        assert info["true_residual"] <= 1e-10
    else:
        assert info["status"] in (lq.ENOCONV, lq.EBREAKDOWN)
        res = np.linalg.norm(b - oracle.M(x.cpu().numpy(), c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
        assert abs(res - info["true_residual"]) <= 1e-6 * res       # the reported residual is the real one
    c.ctx.close()


def test_schwarz_block_groups_and_residual_history(mid):
    """SURVEY NEXT-1 block-group schedule: K applied group by group (all MR steps on a group of blocks before the
    next group) is bit-identical to K applied to all blocks at once, for every group size, and still the oracle's K;
    GCR-DD with groups reaches the same solution.  The optional residual history has one entry per iteration, ends
    below the stopping threshold and starts near ||bhat|| / ||b||."""
    c = mid
    lq = c.lqcd
    kappa, blk = 0.124, (4, 4, 4, 8)
    r = inputs.gaussian_spinor(c.dims, 7)
    d = torch.from_numpy(r).cuda()
    fin = c.ctx.pack_spinor(d, 0, 2)
    outs = []
    for group in (0, 1, 3, 5, 1000):
        c.ctx.set_schwarz_group(group)
        out = c.ctx.new_field(2)
        c.ctx.schwarz(out, fin, 0, kappa, blk, 4, 1.0, 2, 12, 2)
        outs.append(out)
    c.ctx.set_schwarz_group(0)
    for o in outs[1:]:
        assert torch.equal(o, outs[0])
    got = torch.zeros_like(d)
    c.ctx.unpack_spinor(got, outs[2], 0, 2)
    want = oracle.schwarz(r, c.U, c.T, c.bc, kappa, 0, blk, n_mr=4)
    assert _rel(got.cpu().numpy(), want) <= 2e-2
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    for solver, kw in ((lq.SOLVER_GCR_DD, dict(schwarz_block=blk, mr_steps=4, schwarz_group=3)), (lq.SOLVER_BICGSTAB, {}),
                       (lq.SOLVER_CGNR, {})):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=(0, 1, 2), recon=(18, 12, 12), history_len=4000, **kw)
        x, info = _solve(c, b, p)
        assert info["status"] == 0 and _rel(x, xo) <= 1e-8
        h = info["residual_history"]
        assert len(h) == info["iterations"] and all(v == v and v >= 0 for v in h)
        assert 0.1 < h[0] < 3.0 and min(h) <= 1.2e-10
    with pytest.raises(lq.LqcdError):
        c.ctx.set_schwarz_group(-1)


def test_multiplicative_schwarz_sap(mid):
    """Multiplicative Schwarz (SAP; R16) against the oracle: K_sap in every
    precision (1 and 2 cycles), support on the solve parity, and GCR preconditioned by it (fp64 / mixed) against the
    oracle's solution and, in fp64, its outer-iteration count; the additive preconditioner still works on the
    colour-major block layout SAP leaves behind."""
    c = mid
    lq = c.lqcd
    kappa, blk = 0.124, (4, 4, 4, 8)
    r = inputs.gaussian_spinor(c.dims, 7)
    d = torch.from_numpy(r).cuda()
    for prec, tol in ((0, 1e-11), (1, 5e-5), (2, 2e-2)):
        for parity in (0, 1):
            for ncyc in (1, 2):
                want = oracle.schwarz_sap(r, c.U, c.T, c.bc, kappa, parity, blk, n_mr=4, n_cycle=ncyc)
                fin, out = c.ctx.pack_spinor(d, parity, prec), c.ctx.new_field(prec)
                c.ctx.schwarz_sap(out, fin, parity, kappa, blk, 4, 1.0, ncyc, prec, 12, prec, 12)
                got = torch.zeros_like(d)
                c.ctx.unpack_spinor(got, out, parity, prec)
                g = got.cpu().numpy()
                assert np.max(np.abs(g[c.par != parity])) == 0.0
                assert _rel(g, want) <= tol, (prec, parity, ncyc)
    # additive K on the colour-major layout
    want = oracle.schwarz(r, c.U, c.T, c.bc, kappa, 0, blk, n_mr=4)
    out = c.ctx.new_field(0)
    c.ctx.schwarz(out, c.ctx.pack_spinor(d, 0, 0), 0, kappa, blk, 4, 1.0, 0, 18, 0)
    got = torch.zeros_like(d)
    c.ctx.unpack_spinor(got, out, 0, 0)
    assert _rel(got.cpu().numpy(), want) <= 1e-11
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    bhat = oracle.prepare_source(b, c.U, c.T, c.bc, kappa, 0)
    xs, isap = oracle.gcr_sap_pc(bhat, c.U, c.T, c.bc, kappa, 0, 1e-10 * np.linalg.norm(b), blk, n_mr=4, n_cycle=1)
    for prec in ((0, 0, 0), (0, 1, 2), (0, 2, 2)):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, prec=prec, recon=(18, 12, 12), schwarz_block=blk,
                              mr_steps=4, schwarz_type=lq.SCHWARZ_MULTIPLICATIVE, sap_cycles=1)
        x, info = _solve(c, b, p)
        assert info["status"] == 0 and info["true_residual"] <= 1e-10 and _rel(x, xo) <= 1e-8
        if prec == (0, 0, 0):
            assert abs(info["iterations"] - isap["iterations"]) <= 1
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, schwarz_block=(8, 4, 4, 8), schwarz_type=lq.SCHWARZ_MULTIPLICATIVE)
    with pytest.raises(lq.LqcdError) as e:                        # one block in x: no two-colouring
        _solve(c, b, p)
    assert e.value.code == lq.EINVAL


def test_apply_host_complex64_equals_device_path():
    """lqcd_apply_host_c64: complex64 host arrays (half the PCIe bytes) for fp32 / half compute give bit for bit
    what the device path gives on the same single-precision values; fp64 compute is refused."""
    from paper_1109_2935_b200 import lqcd
    c = Case((8, 4, 6, 8), 0.3)
    kappa = 0.12
    psi = inputs.gaussian_spinor(c.dims, 5)
    h32 = torch.from_numpy(psi).to(torch.complex64).pin_memory()
    d = h32.to(torch.complex128).cuda()
    out32 = torch.empty_like(h32).pin_memory()
    for prec in (1, 2):
        for op, parity, dagger in ((0, 0, False), (0, 0, True), (1, 0, False), (1, 1, True)):
            c.ctx.apply_host(out32, h32, op, parity, dagger, kappa, prec, 12)
            ref = torch.zeros_like(d)
            if op == 0:
                for p in (0, 1):
                    fo = c.ctx.new_field(prec)
                    c.ctx.dslash(fo, c.ctx.pack_spinor(d, 1 - p, prec), p, dagger, prec, 12)
                    c.ctx.unpack_spinor(ref, fo, p, prec)
            else:
                fo = c.ctx.new_field(prec)
                c.ctx.matpc(fo, c.ctx.pack_spinor(d, parity, prec), parity, dagger, kappa, prec, 12)
                c.ctx.unpack_spinor(ref, fo, parity, prec)
            assert torch.equal(out32, ref.to(torch.complex64).cpu()), (prec, op, parity, dagger)
    with pytest.raises(lqcd.LqcdError) as e:
        c.ctx.apply_host(out32, h32, 0, 0, False, kappa, 0, 18)
    assert e.value.code == lqcd.EINVAL
    c.ctx.close()


@pytest.mark.parametrize("solver", ["bicgstab", "cgnr"])
def test_fused_reductions_are_bit_reproducible(mid, solver):
    """SURVEY 8(a) a8 "deterministic reductions": the sums fused into M-hat's second launch (per-CTA partials, added
    in a fixed order by dots_finalize_kernel) and the BLAS-1 sums give the same bits on every run — two identical
    solves return bitwise identical x, iteration counts and residual histories, in every inner precision."""
    c = mid
    lq = c.lqcd
    b = inputs.gaussian_spinor(c.dims, 5)
    for sloppy in (0, 1, 2):
        runs = []
        for _ in range(2):
            p = c.ctx.make_params(0.124, 1.0, 1e-10, solver=lq.SOLVER_BICGSTAB if solver == "bicgstab" else lq.SOLVER_CGNR,
                                  prec=(0, sloppy, sloppy), recon=(18, 12, 12), history_len=4000)
            x, info = _solve(c, b, p)
            assert info["status"] == 0
            runs.append((x, info["iterations"], list(info["residual_history"])))
        assert runs[0][1] == runs[1][1]
        assert runs[0][2] == runs[1][2]
        assert np.array_equal(runs[0][0], runs[1][0])


def test_overlapping_schwarz(mid):
    """Overlapping (restricted additive) Schwarz domains (R18): K with every block grown by
    one site on both sides of every direction against the oracle's block-by-block schwarz_ras, in every precision and
    on both parities (antiperiodic t: domains at the t edges contain the sign plane); overlap 0 afterwards is the
    non-overlapping K again; GCR-DD preconditioned by it reaches the oracle's solution; impossible overlaps are refused."""
    c = mid
    lq = c.lqcd
    kappa, blk = 0.124, (4, 4, 4, 8)
    r = inputs.gaussian_spinor(c.dims, 7)
    d = torch.from_numpy(r).cuda()
    try:
        c.ctx.set_schwarz_overlap(1)
        for prec, tol in ((0, 1e-11), (1, 5e-5), (2, 2e-2)):
            for parity in (0, 1):
                want = oracle.schwarz_ras(r, c.U, c.T, c.bc, kappa, parity, blk, 1, n_mr=4)
                out = c.ctx.new_field(prec)
                c.ctx.schwarz(out, c.ctx.pack_spinor(d, parity, prec), parity, kappa, blk, 4, 1.0, prec, 12, prec)
                got = torch.zeros_like(d)
                c.ctx.unpack_spinor(got, out, parity, prec)
                g = got.cpu().numpy()
                assert np.max(np.abs(g[c.par != parity])) == 0.0
                assert _rel(g, want) <= tol, (prec, parity, _rel(g, want))
        # the overlap is not silently ignored
        assert _rel(want, oracle.schwarz(r, c.U, c.T, c.bc, kappa, 1, blk, n_mr=4)) > 1e-3
        # two partitioned directions (z, t), x and y keep their wrap; block groups give the same bits
        blk2 = (8, 8, 4, 8)
        want = oracle.schwarz_ras(r, c.U, c.T, c.bc, kappa, 0, blk2, 1, n_mr=3)
        outs = []
        for group in (0, 3):
            c.ctx.set_schwarz_group(group)
            out = c.ctx.new_field(0)
            c.ctx.schwarz(out, c.ctx.pack_spinor(d, 0, 0), 0, kappa, blk2, 3, 1.0, 0, 18, 0)
            outs.append(out)
        c.ctx.set_schwarz_group(0)
        assert torch.equal(outs[0], outs[1])
        got = torch.zeros_like(d)
        c.ctx.unpack_spinor(got, outs[0], 0, 0)
        assert _rel(got.cpu().numpy(), want) <= 1e-11
        with pytest.raises(lq.LqcdError):                               # 4 + 2*2 = 8 = extent
            c.ctx.set_schwarz_overlap(2)
            c.ctx.schwarz(out, c.ctx.pack_spinor(d, 0, 2), 0, kappa, blk, 4, 1.0, 2, 12, 2)
        with pytest.raises(lq.LqcdError):                               # three partitioned directions x 1: odd
            c.ctx.set_schwarz_overlap(1)
            c.ctx.schwarz(out, c.ctx.pack_spinor(d, 0, 2), 0, kappa, (8, 4, 4, 8), 4, 1.0, 2, 12, 2)
    finally:
        c.ctx.set_schwarz_overlap(0)
    want = oracle.schwarz(r, c.U, c.T, c.bc, kappa, 0, blk, n_mr=4)
    out = c.ctx.new_field(0)
    c.ctx.schwarz(out, c.ctx.pack_spinor(d, 0, 0), 0, kappa, blk, 4, 1.0, 0, 18, 0)
    got = torch.zeros_like(d)
    c.ctx.unpack_spinor(got, out, 0, 0)
    assert _rel(got.cpu().numpy(), want) <= 1e-11
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-12)
    its = {}
    for ovl in (0, 1):
        for prec in ((0, 0, 0), (0, 2, 2)):
            p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, prec=prec, recon=(18, 12, 12), schwarz_block=blk,
                                  mr_steps=4, schwarz_overlap=ovl)
            x, info = _solve(c, b, p)
            assert info["status"] == 0 and info["true_residual"] <= 1e-10 and _rel(x, xo) <= 1e-8
            its[(ovl, prec)] = info["iterations"]
    assert its[(1, (0, 0, 0))] <= its[(0, (0, 0, 0))]                  # the overlap does not cost outer iterations
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, schwarz_block=blk, schwarz_type=lq.SCHWARZ_MULTIPLICATIVE, schwarz_overlap=1)
    with pytest.raises(lq.LqcdError):
        _solve(c, b, p)


def test_overlapping_schwarz_three_blocks_in_x():
    """An odd number of blocks in a direction (12 x 4 x 4 x 16, blocks 4 x 4 x 4 x 8: 3 x 1 x 1 x 2): every x domain
    overlaps both its neighbours, block 0 and block 2 through the lattice's wrap; y and z are not partitioned."""
    c = Case((12, 4, 4, 16), 0.3)
    kappa, blk = 0.124, (4, 4, 4, 8)
    r = inputs.gaussian_spinor(c.dims, 9)
    d = torch.from_numpy(r).cuda()
    try:
        c.ctx.set_schwarz_overlap(1)
        for prec, tol in ((0, 1e-11), (2, 2e-2)):
            for parity in (0, 1):
                want = oracle.schwarz_ras(r, c.U, c.T, c.bc, kappa, parity, blk, 1, n_mr=3)
                out = c.ctx.new_field(prec)
                c.ctx.schwarz(out, c.ctx.pack_spinor(d, parity, prec), parity, kappa, blk, 3, 1.0, prec, 12, prec)
                got = torch.zeros_like(d)
                c.ctx.unpack_spinor(got, out, parity, prec)
                assert _rel(got.cpu().numpy(), want) <= tol, (prec, parity)
    finally:
        c.ctx.set_schwarz_overlap(0)
