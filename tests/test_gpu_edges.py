"""Edge and degenerate cases of the hot path on the GPU (-m gpu), each against the oracle:
extent-2 directions (forward and backward neighbour coincide), c_sw = 0 and
kappa = 0, zero and one-site sources, exact initial guess, iteration cap, a single Schwarz block
(B = dims keeps the wrap, R7), the parity-1 Schur system, the size limit of lqcd_create."""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs
from test_gpu_parity import Case, _rel, TOL

pytestmark = pytest.mark.gpu


def _solve(c, b, params, x0=None, allow_fail=False):
    x = torch.zeros(b.shape, dtype=torch.complex128, device="cuda") if x0 is None else torch.from_numpy(x0).cuda()
    info = c.ctx.invert(x, torch.from_numpy(b).cuda(), params, allow_fail=allow_fail)
    torch.cuda.synchronize()
    return x.cpu().numpy(), info


@pytest.mark.parametrize("dims,bc", [((2, 2, 4, 6), (1, -1, 1, -1)), ((4, 6, 2, 2), (-1, 1, -1, 1)), ((2, 2, 2, 2), (1, 1, 1, -1))])
def test_extent_two_directions(dims, bc):
    """L_mu = 2: x+mu and x-mu are the same site and both terms are added, with the boundary sign on
    the one that wraps; X = 2 also makes the checkerboarded row one site long (Xh = 1)."""
    c = Case(dims, 0.4, bc=bc)
    kappa = 0.11
    psi = inputs.gaussian_spinor(dims, 5)
    for prec in (0, 1, 2):
        for recon in (18, 12, 8):
            tol = TOL[prec]        # fp64 recon-8 included (R10: measured <= 1.2e-14)
            for parity in (0, 1):
                for dagger in (False, True):
                    want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
                    got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, dagger, prec, recon), psi, 1 - parity, parity, prec)
                    assert _rel(got, want) <= tol, (prec, recon, parity, dagger)
                want = oracle.matpc(psi, c.U, c.T, c.bc, kappa, parity)
                got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, parity, False, kappa, prec, recon), psi, parity, parity, prec)
                assert _rel(got, want) <= tol, (prec, recon, parity)
    lq = c.lqcd
    b = inputs.gaussian_spinor(dims, 6)
    for solver, prec in ((lq.SOLVER_BICGSTAB, (0, 1, 1)), (lq.SOLVER_GCR_DD, (0, 0, 1))):
        p = c.ctx.make_params(kappa, 1.0, 1e-11, solver=solver, prec=prec, recon=(18, 12, 12), schwarz_block=(2, 2, 2, 2), mr_steps=4)
        x, info = _solve(c, b, p)
        assert np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b) <= 1.05e-11
    c.ctx.close()


def test_csw_zero_and_kappa_zero():
    """c_sw = 0: A = 1, so the clover apply is the identity and Mhat = 1 - kappa^2 D D (Wilson);
    kappa = 0: Mhat = 1 exactly."""
    c = Case((4, 4, 4, 6), 0.3, c_sw=0.0)
    psi = inputs.gaussian_spinor(c.dims, 8)
    assert np.max(np.abs(c.T)) == 0.0
    for prec in (0, 1):
        got = c.gpu_parity_op(lambda o, i: c.ctx.clover(o, i, 0, False, 0.124, prec), psi, 0, 0, prec)
        assert _rel(got, psi * c.mask(0)) <= (0.0 if prec == 0 else 1e-7)
        got = c.gpu_parity_op(lambda o, i: c.ctx.clover(o, i, 1, True, 0.124, prec), psi, 1, 1, prec)
        assert _rel(got, psi * c.mask(1)) <= (0.0 if prec == 0 else 1e-7)
        want = oracle.matpc(psi, c.U, c.T, c.bc, 0.124, 0)
        got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, 0, False, 0.124, prec, 12), psi, 0, 0, prec)
        assert _rel(got, want) <= TOL[prec]
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, 1, False, 0.0, 0, 18), psi, 1, 1, 0)
    assert np.array_equal(got, psi * c.mask(1))
    c.ctx.close()


@pytest.fixture(scope="module")
def small():
    return Case((4, 4, 4, 8), 0.3)


def test_zero_and_point_sources(small):
    c = small
    lq = c.lqcd
    kappa = 0.12
    zero = np.zeros((8, 4, 4, 4, 4, 3), dtype=np.complex128)
    for prec in (0, 1, 2):      # a zero field stays exactly zero through the half-precision quantiser (norm 0)
        got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, 0, False, kappa, prec, 12), zero, 0, 0, prec)
        assert np.max(np.abs(got)) == 0.0
    p = c.ctx.make_params(kappa, 1.0, 1e-10, prec=(0, 2, 2), recon=(18, 12, 12))
    x, info = _solve(c, zero, p)
    assert info["status"] == 0 and info["iterations"] == 0 and np.max(np.abs(x)) == 0.0
    # point source: one nonzero component on an odd site (outside the solved parity)
    b = zero.copy()
    b[3, 2, 1, 1, 2, 1] = 1.0 - 0.5j
    for solver in (lq.SOLVER_BICGSTAB, lq.SOLVER_GCR_DD):
        p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=(0, 1, 2), recon=(18, 12, 12), schwarz_block=(2, 2, 4, 4))
        x, info = _solve(c, b, p)
        assert np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b) <= 1.05e-10
    # Dslash of a point source touches exactly its 8 neighbours
    got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, 0, False, 0, 18), b, 1, 0, 0)
    assert np.count_nonzero(np.abs(got).sum(axis=(4, 5))) == 8


def test_initial_guess_and_iteration_cap(small):
    c = small
    lq = c.lqcd
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 9)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=0, tol=1e-13)
    # exact initial guess: accepted without iterating
    p = c.ctx.make_params(kappa, 1.0, 1e-10, prec=(0, 1, 1), recon=(18, 12, 12), use_initial_guess=True)
    x, info = _solve(c, b, p, x0=xo)
    assert info["iterations"] == 0 and info["true_residual"] <= 1e-10 and _rel(x, xo) <= 1e-12
    # a poor guess is improved, not discarded
    p = c.ctx.make_params(kappa, 1.0, 1e-10, prec=(0, 1, 1), recon=(18, 12, 12), use_initial_guess=True)
    x, info = _solve(c, b, p, x0=xo + 0.01 * inputs.gaussian_spinor(c.dims, 10))
    assert info["iterations"] > 0 and _rel(x, xo) <= 1e-8
    # iteration cap: LQCD_ENOCONV, and the result struct still reports the true residual reached
    for solver in (lq.SOLVER_BICGSTAB, lq.SOLVER_GCR_DD):
        p = c.ctx.make_params(kappa, 1.0, 1e-12, solver=solver, prec=(0, 1, 1), recon=(18, 12, 12), max_iter=2,
                              schwarz_block=(2, 2, 2, 2), mr_steps=2)
        x, info = _solve(c, b, p, allow_fail=True)
        assert info["status"] == lq.ENOCONV and info["iterations"] == 2
        res = np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b)
        assert 1e-12 < res < 1.0 and abs(res - info["true_residual"]) <= 1e-8 * res + 1e-13
        with pytest.raises(lq.LqcdError) as e:
            _solve(c, b, p)
        assert e.value.code == lq.ENOCONV


def test_single_schwarz_block_keeps_the_wrap(small):
    """B = dims: one block, nothing is cut (R7), so K = n_MR global MR steps on Mhat with its
    (anti)periodic wrap, and GCR-DD still converges to the oracle's solution."""
    c = small
    lq = c.lqcd
    kappa, blk = 0.124, c.dims
    r = inputs.gaussian_spinor(c.dims, 4)
    want = oracle.schwarz(r, c.U, c.T, c.bc, kappa, 0, blk, n_mr=3)
    got = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, 0, kappa, blk, 3, 1.0, 0, 18, 0), r, 0, 0, 0)
    assert _rel(got, want) <= 1e-12
    # three global MR steps written out with the oracle's operator
    rho, x = r * c.mask(0), 0
    for _ in range(3):
        w = oracle.matpc(rho, c.U, c.T, c.bc, kappa, 0)
        a = np.vdot(w.ravel(), rho.ravel()) / np.vdot(w.ravel(), w.ravel())
        x, rho = x + a * rho, rho - a * w
    assert _rel(got, x) <= 1e-12
    b = inputs.gaussian_spinor(c.dims, 2)
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, prec=(0, 1, 2), recon=(18, 12, 12), schwarz_block=blk, mr_steps=5)
    x, info = _solve(c, b, p)
    assert np.linalg.norm(b - oracle.M(x, c.U, c.T, c.bc, kappa)) / np.linalg.norm(b) <= 1.05e-10


@pytest.mark.parametrize("solver", [0, 1])
def test_parity_one_mixed_precision(small, solver):
    c = small
    kappa = 0.124
    b = inputs.gaussian_spinor(c.dims, 2)
    xo, io = oracle.invert(b, c.U, c.T, c.bc, kappa, parity=1, tol=1e-13)
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=solver, prec=(0, 2, 2), recon=(18, 8, 12), parity=1,
                          schwarz_block=(2, 2, 2, 4), mr_steps=6)
    x, info = _solve(c, b, p)
    assert info["status"] == 0 and info["true_residual"] <= 1e-10
    assert _rel(x, xo) <= 1e-8


def test_create_rejects_oversized_and_bad_arguments():
    from paper_1109_2935_b200 import lqcd
    for dims in ((1024, 1024, 64, 64), (0, 4, 4, 4), (4, 4, 4, -2)):       # Vh must fit a 32-bit index
        with pytest.raises(lqcd.LqcdError):
            lqcd.Context(dims, (1, 1, 1, -1), 0)
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((4, 4, 4, 4), (1, 1, 0, -1), 0)                          # boundary must be +-1
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((4, 4, 4, 4), (1, 1, 1, -1), 99)                         # no such device
    ctx = lqcd.Context((4, 4, 4, 8), (1, 1, 1, -1), 0)
    U = torch.from_numpy(inputs.random_gauge((4, 4, 4, 8), 0.3, 1)).cuda()
    ctx.load_gauge(U)
    ctx.build_clover(1.0)
    f, g = ctx.new_field(1), ctx.new_field(1)
    for blk in ((3, 4, 4, 8), (4, 4, 4, 6), (4, 4, 4, 0)):                    # odd / not dividing / zero block
        with pytest.raises(lqcd.LqcdError) as e:
            ctx.schwarz(f, g, 0, 0.12, blk, 2, 1.0, 1, 12, 1)
        assert e.value.code == lqcd.EINVAL
    p = ctx.make_params(0.12, 0.5, 1e-8)                                      # c_sw differs from the built one
    x = torch.zeros((8, 4, 4, 4, 4, 3), dtype=torch.complex128, device="cuda")
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.invert(x, x.clone(), p)
    assert e.value.code == lqcd.ESTATE
    ctx.close()


def test_context_lifecycle_releases_device_memory():
    """Create / use / destroy repeatedly (all precisions, both solvers, host pipeline, Schwarz blocks):
    lqcd_destroy returns every byte the context allocated; two contexts can be alive at once and do not
    share state."""
    from paper_1109_2935_b200 import lqcd
    dims = (8, 8, 8, 8)
    U = torch.from_numpy(inputs.random_gauge(dims, 0.3, 1)).cuda()
    b = torch.from_numpy(inputs.gaussian_spinor(dims, 2)).cuda()
    bh = b.cpu().pin_memory()
    oh = torch.empty_like(bh).pin_memory()

    def cycle():
        ctx = lqcd.Context(dims, (1, 1, 1, -1), 0)
        ctx.load_gauge(U)
        ctx.build_clover(1.0)
        x = torch.zeros_like(b)
        for solver, prec in ((lqcd.SOLVER_BICGSTAB, (0, 1, 1)), (lqcd.SOLVER_GCR_DD, (0, 1, 2)), (lqcd.SOLVER_CGNR, (0, 2, 2))):
            info = ctx.invert(x, b, ctx.make_params(0.12, 1.0, 1e-9, solver=solver, prec=prec, recon=(18, 12, 8), schwarz_block=(4, 4, 4, 4)))
            assert info["true_residual"] <= 1e-9
        ctx.apply_host(oh, bh, 1, 0, False, 0.12, 2, 12)
        f = ctx.new_fields(1, 5)
        ctx.matpc_mrhs(ctx.new_fields(1, 5), f.zero_(), 5, 0, False, 0.12, 1, 12)
        torch.cuda.synchronize()
        ctx.close()
        return x

    x0 = cycle()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(5):
        x1 = cycle()
        assert torch.equal(x0, x1)                        # deterministic from a fresh context
    torch.cuda.synchronize()
    assert abs(torch.cuda.mem_get_info()[0] - free0) <= (8 << 20)      # nothing accumulates (allocator granularity only)
    # two live contexts with different kappa / lattices do not interfere
    c1 = lqcd.Context(dims, (1, 1, 1, -1), 0)
    c2 = lqcd.Context((4, 4, 4, 8), (1, 1, 1, 1), 0)
    c1.load_gauge(U)
    c1.build_clover(1.0)
    U2 = torch.from_numpy(inputs.random_gauge((4, 4, 4, 8), 0.4, 5)).cuda()
    c2.load_gauge(U2)
    c2.build_clover(0.7)
    f1 = c1.pack_spinor(b, 0, 0)
    o1a, o1b = c1.new_field(0), c1.new_field(0)
    c1.matpc(o1a, f1, 0, False, 0.12, 0, 18)
    b2 = torch.from_numpy(inputs.gaussian_spinor((4, 4, 4, 8), 3)).cuda()
    c2.matpc(c2.new_field(0), c2.pack_spinor(b2, 0, 0), 0, False, 0.11, 0, 18)
    c1.matpc(o1b, f1, 0, False, 0.12, 0, 18)
    assert torch.equal(o1a, o1b)
    c1.close()
    c2.close()


def test_recon8_rejects_unit_gauge_and_compression_rejects_non_su3():
    """recon-8 cannot hold a link with first row (a1, 0, 0) (N = |a2|^2 + |a3|^2 = 0, e.g. the cold start
    U = 1; R10): the library must say so (LQCD_EINVAL) instead of returning NaN fields, in every
    precision, and recon-12 / 18 must keep working on the same context.  Links that are not SU(3) are
    refused by recon-12 and recon-8 (both reconstruct unitary links only) and accepted by recon-18."""
    from paper_1109_2935_b200 import lqcd
    dims = (4, 4, 4, 4)
    psi = torch.from_numpy(inputs.gaussian_spinor(dims, 2)).cuda()
    ctx = lqcd.Context(dims, (1, 1, 1, -1), 0)
    ctx.load_gauge(torch.from_numpy(inputs.unit_gauge(dims)).cuda())
    ctx.build_clover(1.0)
    for prec in (0, 1, 2):
        fin, fout = ctx.pack_spinor(psi, 1, prec), ctx.new_field(prec)
        with pytest.raises(lqcd.LqcdError) as e:
            ctx.dslash(fout, fin, 0, False, prec, 8)
        assert e.value.code == lqcd.EINVAL and "recon 8" in str(e.value)
        with pytest.raises(lqcd.LqcdError) as e:                   # still refused on the second call (nothing half-built is cached)
            ctx.matpc(fout, fin, 0, False, 0.12, prec, 8)
        assert e.value.code == lqcd.EINVAL
        for recon in (12, 18):
            ctx.dslash(fout, fin, 0, False, prec, recon)
            got = torch.zeros_like(psi)
            ctx.unpack_spinor(got, fout, 0, prec)
            assert bool(torch.isfinite(torch.view_as_real(got)).all())
    p = ctx.make_params(0.12, 1.0, 1e-8, prec=(0, 1, 1), recon=(18, 8, 8))
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.invert(torch.zeros_like(psi), psi, p)
    assert e.value.code == lqcd.EINVAL
    # one link of an otherwise valid field scaled by 1.001: not unitary
    U = inputs.random_gauge(dims, 0.4, 3)
    U[2, 1, 2, 3, 0] *= 1.001
    ctx.load_gauge(torch.from_numpy(U).cuda())
    ctx.build_clover(1.0)
    fin, fout = ctx.pack_spinor(psi, 1, 0), ctx.new_field(0)
    for recon in (12, 8):
        with pytest.raises(lqcd.LqcdError) as e:
            ctx.dslash(fout, fin, 0, False, 0, recon)
        assert e.value.code == lqcd.EINVAL and "SU(3)" in str(e.value)
    ctx.dslash(fout, fin, 0, False, 0, 18)                         # recon-18 stores what it is given
    got = torch.zeros_like(psi)
    ctx.unpack_spinor(got, fout, 0, 0)
    par = inputs.parity_mask(dims)
    want = oracle.dslash(psi.cpu().numpy() * (par == 1)[..., None, None], U, (1, 1, 1, -1)) * (par == 0)[..., None, None]
    assert _rel(got.cpu().numpy(), want) <= 1e-13
    ctx.close()


def test_recon8_fp64_near_unit_links():
    """Smooth gauge fields (eps = 0.02: N ~ 1e-4 on a typical link) in fp64 / recon-8 at the north_star tolerance:
    the reconstruction takes |c1|^2 = N - |b1|^2 (core.cuh), so its error does not grow as N -> 0."""
    c = Case((4, 6, 4, 8), 0.02)
    psi = inputs.gaussian_spinor(c.dims, 9)
    for parity in (0, 1):
        want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc) * c.mask(parity)
        got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, False, 0, 8), psi, 1 - parity, parity, 0)
        assert _rel(got, want) <= 1e-13
    want = oracle.matpc(psi, c.U, c.T, c.bc, 0.12, 0)
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, 0, False, 0.12, 0, 8), psi, 0, 0, 0)
    assert _rel(got, want) <= 1e-13
    c.ctx.close()


def test_staggered_links_survive_growing_mrhs_workspace():
    """One context serving both paths: loading staggered links, then multi-right-hand-side Mhat calls whose
    temporary has to grow (more sources, then a wider precision), must leave the staggered links loaded."""
    from paper_1109_2935_b200 import lqcd
    dims, bc = (4, 4, 4, 8), (1, 1, 1, -1)
    c = Case(dims, 0.3)
    ctx = c.ctx
    fat, lng = inputs.staggered_links(dims, 0.3, 4)
    ctx.load_staggered_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), 0.0)
    chi = inputs.gaussian_colour_vector(dims, 5)
    d = torch.from_numpy(chi).cuda()

    def stag():
        out = ctx.new_staggered_field(1)
        ctx.staggered_dslash(out, ctx.pack_staggered(d, 1, 1), 0, 1)
        got = torch.zeros_like(d)
        ctx.unpack_staggered(got, out, 0, 1)
        return got

    ref = stag()
    for prec, nrhs in ((1, 2), (1, 5), (0, 5), (0, 9)):
        fin = ctx.new_fields(prec, nrhs).zero_()
        ctx.matpc_mrhs(ctx.new_fields(prec, nrhs), fin, nrhs, 0, False, 0.12, prec, 12)
        assert torch.equal(stag(), ref)
    ctx.close()
