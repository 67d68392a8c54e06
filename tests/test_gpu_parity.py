"""GPU-vs-oracle parity (-m gpu): every call goes through the C ABI (include/lqcd.h) via the
ctypes binding and is compared element by element with oracle/ on the same seeded inputs.

Tolerances (relative L2 per operator application) are BASELINE.json's north_star:
fp64 1e-13, fp32 1e-5, half 5e-3; solves: true residual <= 1e-10, solution within 1e-8.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL = {0: 1e-13, 1: 1e-5, 2: 5e-3}


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


class Case:
    """One lattice + gauge field loaded into a GPU context, with the oracle's clover term."""

    def __init__(self, dims, eps, c_sw=1.0, bc=BC, gauge_seed=1):
        from paper_1109_2935_b200 import lqcd
        self.lqcd = lqcd
        self.dims, self.bc, self.c_sw = dims, bc, c_sw
        self.U = inputs.random_gauge(dims, eps, gauge_seed)
        self.ctx = lqcd.Context(dims, bc, 0)
        self.ctx.load_gauge(torch.from_numpy(self.U).cuda())
        self.ctx.build_clover(c_sw)
        self.T = oracle.clover_term(self.U, c_sw)
        self.par = inputs.parity_mask(dims)

    def mask(self, p):
        return (self.par == p)[..., None, None]

    def gpu_parity_op(self, fn, psi, p_in, p_out, prec):
        """pack parity p_in of psi, run fn(out, in), unpack to a zero-initialised canonical array."""
        ctx = self.ctx
        d = torch.from_numpy(np.ascontiguousarray(psi)).cuda()
        fin = ctx.pack_spinor(d, p_in, prec)
        fout = ctx.new_field(prec)
        fn(fout, fin)
        res = torch.zeros_like(d)
        ctx.unpack_spinor(res, fout, p_out, prec)
        torch.cuda.synchronize()
        return res.cpu().numpy()


@pytest.fixture(scope="module")
def cfg1():
    return Case((4, 4, 4, 4), 0.5)


@pytest.fixture(scope="module")
def ragged():
    # Vh = 6*4*10*8/2 = 960 = 7.5 CTAs of 128 threads: several tiles and a ragged tail
    return Case((6, 4, 10, 8), 0.3, bc=(-1, 1, 1, -1))


def test_pack_unpack_roundtrip(ragged):
    c = ragged
    psi = inputs.gaussian_spinor(c.dims, 2)
    for prec, tol in ((0, 0.0), (1, 1e-7), (2, 3e-5)):
        for p in (0, 1):
            got = c.gpu_parity_op(lambda o, i: o.copy_(i), psi, p, p, prec)
            want = psi * c.mask(p)
            if tol == 0.0:
                assert np.array_equal(got, want)
            else:
                assert _rel(got, want) <= tol
            assert np.max(np.abs(got[c.par != p])) == 0.0


@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("dagger", [False, True])
@pytest.mark.parametrize("parity", [0, 1])
def test_cfg1_dslash_fp64(cfg1, parity, dagger, recon):
    c = cfg1
    psi = inputs.gaussian_spinor(c.dims, 2)
    want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
    got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, dagger, 0, recon), psi, 1 - parity, parity, 0)
    assert _rel(got, want) <= 1e-13   # recon-8 included: measured 5e-16 here (R10)


@pytest.mark.parametrize("dagger", [False, True])
@pytest.mark.parametrize("parity", [0, 1])
def test_cfg1_matpc_and_clover_fp64(cfg1, parity, dagger):
    c = cfg1
    kappa = 0.12
    psi = inputs.gaussian_spinor(c.dims, 2)
    want = oracle.matpc(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, parity, dagger, kappa, 0, 18), psi, parity, parity, 0)
    assert _rel(got, want) <= 1e-13
    for inverse in (False, True):
        want = oracle.clover_apply(psi, c.T, kappa, inverse=inverse, parity=parity)
        got = c.gpu_parity_op(lambda o, i: c.ctx.clover(o, i, parity, inverse, kappa, 0), psi, parity, parity, 0)
        assert _rel(got, want) <= 1e-13


@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_ragged_all_precisions(ragged, prec, recon):
    c = ragged
    kappa = 0.124
    psi = inputs.gaussian_spinor(c.dims, 3)
    tol = TOL[prec]                  # fp64 recon-8 measured 1.7e-15 on this lattice (R10)
    for parity in (0, 1):
        for dagger in (False, True):
            want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
            got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, dagger, prec, recon), psi, 1 - parity, parity, prec)
            assert _rel(got, want) <= tol, ("dslash", parity, dagger)
            assert np.max(np.abs(got[c.par != parity])) == 0.0
            want = oracle.matpc(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)
            got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, parity, dagger, kappa, prec, recon), psi, parity, parity, prec)
            assert _rel(got, want) <= tol, ("matpc", parity, dagger)
        for inverse in (False, True):
            want = oracle.clover_apply(psi, c.T, kappa, inverse=inverse, parity=parity)
            got = c.gpu_parity_op(lambda o, i: c.ctx.clover(o, i, parity, inverse, kappa, prec), psi, parity, parity, prec)
            assert _rel(got, want) <= TOL[prec], ("clover", parity, inverse)


def test_free_field_plane_wave_on_gpu():
    """U = 1 (recon-18/12; recon-8 is singular at U = 1): closed form M(p)."""
    dims, bc, kappa = (8, 4, 4, 6), (1, 1, 1, -1), 0.12
    c = Case(dims, 0.0)
    assert np.allclose(c.U, inputs.unit_gauge(dims))
    X, Y, Z, T = dims
    n = np.array([1, 0, 3, 2])
    p = 2 * np.pi * (n + np.where(np.array(bc) < 0, 0.5, 0.0)) / np.array(dims)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    u = np.random.default_rng(5).standard_normal((4, 3)) + 0j
    psi = phase[..., None, None] * u
    g = [oracle.gamma(m) for m in range(4)]
    Dp = sum((np.eye(4) - g[m]) * np.exp(1j * p[m]) + (np.eye(4) + g[m]) * np.exp(-1j * p[m]) for m in range(4))
    want = phase[..., None, None] * (Dp @ u)
    for recon in (18, 12):
        for parity in (0, 1):
            got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, False, 0, recon), psi, 1 - parity, parity, 0)
            assert _rel(got, want * c.mask(parity)) <= 1e-13


def test_cfg2_fp32_recon12():
    """BASELINE.json config 2: 16^3x32, fp32 storage, recon-12, eps = 0.3."""
    c = Case((16, 16, 16, 32), 0.3)
    psi = inputs.gaussian_spinor(c.dims, 2)
    for parity in (0, 1):
        for dagger in (False, True):
            want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
            got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, dagger, 1, 12), psi, 1 - parity, parity, 1)
            assert _rel(got, want) <= 1e-5
        want = oracle.clover_apply(psi, c.T, 0.124, parity=parity)
        got = c.gpu_parity_op(lambda o, i: c.ctx.clover(o, i, parity, False, 0.124, 1), psi, parity, parity, 1)
        assert _rel(got, want) <= 1e-5
    # half precision on the same lattice
    want = oracle.matpc(psi, c.U, c.T, c.bc, 0.124, 0)
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, 0, False, 0.124, 2, 12), psi, 0, 0, 2)
    assert _rel(got, want) <= 5e-3


def test_blas_reductions(ragged):
    c = ragged
    x = inputs.gaussian_spinor(c.dims, 11)
    y = inputs.gaussian_spinor(c.dims, 12)
    for prec, tol in ((0, 1e-14), (1, 1e-6), (2, 2e-4)):
        fx = c.ctx.pack_spinor(torch.from_numpy(x).cuda(), 0, prec)
        fy = c.ctx.pack_spinor(torch.from_numpy(y).cuda(), 0, prec)
        xm, ym = x * c.mask(0), y * c.mask(0)
        d = c.ctx.cdot(fx, fy, prec)
        assert abs(d - np.vdot(xm.ravel(), ym.ravel())) <= tol * np.linalg.norm(xm) * np.linalg.norm(ym)
        n2 = c.ctx.axpy_norm(0.37, fx, fy, prec)
        want = ym + 0.37 * xm
        assert abs(n2 - np.linalg.norm(want) ** 2) <= 10 * tol * np.linalg.norm(want) ** 2
        res = torch.zeros(x.shape, dtype=torch.complex128, device="cuda")
        c.ctx.unpack_spinor(res, fy, 0, prec)
        assert _rel(res.cpu().numpy(), want) <= max(tol, 1e-15) * 10
        # bit-reproducible reductions
        assert c.ctx.cdot(fx, fy, prec) == c.ctx.cdot(fx, fy, prec)


def test_error_codes(cfg1):
    from paper_1109_2935_b200 import lqcd
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((3, 4, 4, 4), BC, 0)                       # odd extent
    ctx = lqcd.Context((4, 4, 4, 4), BC, 0)
    f = ctx.new_field(0)
    g = ctx.new_field(0)
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.dslash(f, g, 0, False, 0, 18)                       # before load_gauge
    assert e.value.code == lqcd.ESTATE
    with pytest.raises(lqcd.LqcdError) as e:
        cfg1.ctx.dslash(f, g, 0, False, 0, 10)                  # bad recon
    assert e.value.code == lqcd.EINVAL
    with pytest.raises(lqcd.LqcdError) as e:
        cfg1.ctx.dslash(f, f, 0, False, 0, 18)                  # aliasing
    assert e.value.code == lqcd.EINVAL
    ctx.close()


def test_cfg3_full_size_all_precisions():
    """BASELINE.json config 3 at full size, 32^3x64 (eps = 0.3, kappa = 0.124, c_sw = 1): the launch
    configuration bench.py times (8192 CTAs x 128 threads per parity).  Dslash in every precision x
    compression and Mhat in every precision, element by element against the oracle on the same
    arrays (the oracle applies D to the full lattice in well under a second)."""
    from paper_1109_2935_b200 import lqcd
    dims, kappa = (32, 32, 32, 64), 0.124
    Ut = inputs.random_gauge_torch(dims, 0.3, 1, device="cuda")
    pt = inputs.gaussian_spinor_torch(dims, 2, device="cuda")
    ctx = lqcd.Context(dims, BC, 0)
    ctx.load_gauge(Ut)
    ctx.build_clover(1.0)
    U, psi = Ut.cpu().numpy(), pt.cpu().numpy()
    del Ut
    want_d = oracle.dslash(psi, U, BC)                      # both parities at once
    want_ddag = oracle.dslash(psi, U, BC, dagger=True)
    T = oracle.clover_term(U, 1.0)
    want_m = oracle.matpc(psi, U, T, BC, kappa, 0)
    del T
    par = torch.from_numpy(inputs.parity_mask(dims)).cuda()
    wd, wdd, wm = (torch.from_numpy(w).cuda() for w in (want_d, want_ddag, want_m))
    even = (par == 0)[..., None, None]
    for prec in (0, 1, 2):
        fin = [ctx.pack_spinor(pt, p, prec) for p in (0, 1)]
        fo = [ctx.new_field(prec) for _ in (0, 1)]
        for recon in (18, 12, 8):
            tol = TOL[prec]          # fp64 recon-8: measured 1.2e-14 at this size (min N = 1.7e-6; R10)
            for dagger, want in ((False, wd), (True, wdd)):
                got = torch.zeros_like(pt)
                for p in (0, 1):
                    ctx.dslash(fo[p], fin[1 - p], p, dagger, prec, recon)
                    ctx.unpack_spinor(got, fo[p], p, prec)
                err = float(torch.linalg.vector_norm(got - want) / torch.linalg.vector_norm(want))
                assert err <= tol, ("dslash", prec, recon, dagger, err)
            got = torch.zeros_like(pt)
            ctx.matpc(fo[0], fin[0], 0, False, kappa, prec, recon)
            ctx.unpack_spinor(got, fo[0], 0, prec)
            assert float(torch.count_nonzero(got * ~even)) == 0
            err = float(torch.linalg.vector_norm(got - wm) / torch.linalg.vector_norm(wm))
            assert err <= tol, ("matpc", prec, recon, err)
    ctx.close()


def test_cfg5_full_size_operator_and_schwarz():
    """BASELINE.json config 5 at full size, 48^3x96 (10.6 M sites, eps = 0.2, kappa = 0.124, c_sw = 1):
    Dslash (fp32 and half, recon-12), Mhat (half) and the Schwarz preconditioner K with 256 blocks
    of 12^3x24 and 10 MR steps in half precision, and the multiplicative variant (SAP) on the same blocks, element by
    element against the oracle on the same arrays.  K's tolerance is the one of DESIGN.md R7 / SURVEY 8(c).8 (error compounds over steps)."""
    from paper_1109_2935_b200 import lqcd
    dims, kappa, blk = (48, 48, 48, 96), 0.124, (12, 12, 12, 24)
    Ut = inputs.random_gauge_torch(dims, 0.2, 21, device="cuda")
    pt = inputs.gaussian_spinor_torch(dims, 22, device="cuda")
    ctx = lqcd.Context(dims, BC, 0)
    ctx.load_gauge(Ut)
    ctx.build_clover(1.0)
    U, psi = Ut.cpu().numpy(), pt.cpu().numpy()
    del Ut
    par = torch.from_numpy(inputs.parity_mask(dims)).cuda()
    even = (par == 0)[..., None, None]
    want_d = torch.from_numpy(oracle.dslash(psi, U, BC)).cuda()
    for prec in (1, 2):
        fin = [ctx.pack_spinor(pt, p, prec) for p in (0, 1)]
        got = torch.zeros_like(pt)
        for p in (0, 1):
            fo = ctx.new_field(prec)
            ctx.dslash(fo, fin[1 - p], p, False, prec, 12)
            ctx.unpack_spinor(got, fo, p, prec)
        err = float(torch.linalg.vector_norm(got - want_d) / torch.linalg.vector_norm(want_d))
        assert err <= TOL[prec], ("dslash", prec, err)
    del want_d
    T = oracle.clover_term(U, 1.0)
    want_m = torch.from_numpy(oracle.matpc(psi, U, T, BC, kappa, 0)).cuda()
    fo = ctx.new_field(2)
    ctx.matpc(fo, fin[0], 0, False, kappa, 2, 12)
    got = torch.zeros_like(pt)
    ctx.unpack_spinor(got, fo, 0, 2)
    err = float(torch.linalg.vector_norm(got - want_m) / torch.linalg.vector_norm(want_m))
    assert err <= TOL[2], ("matpc", err)
    del want_m
    for n_mr, tol in ((1, 5e-3), (10, 2e-2)):
        want_k = torch.from_numpy(oracle.schwarz(psi, U, T, BC, kappa, 0, blk, n_mr=n_mr)).cuda()
        fk = ctx.new_field(1)
        ctx.schwarz(fk, ctx.pack_spinor(pt, 0, 1), 0, kappa, blk, n_mr, 1.0, 2, 12, 1)
        got = torch.zeros_like(pt)
        ctx.unpack_spinor(got, fk, 0, 1)
        assert float(torch.count_nonzero(got * ~even)) == 0
        err = float(torch.linalg.vector_norm(got - want_k) / torch.linalg.vector_norm(want_k))
        assert err <= tol, ("schwarz", n_mr, err)
    # multiplicative Schwarz (SAP, R16) on the same 256 blocks in the colour-major block order: one cycle,
    # 2 MR steps per half-step, half precision inside, fp32 outside
    want_k = torch.from_numpy(oracle.schwarz_sap(psi, U, T, BC, kappa, 0, blk, n_mr=2, n_cycle=1)).cuda()
    fk = ctx.new_field(1)
    ctx.schwarz_sap(fk, ctx.pack_spinor(pt, 0, 1), 0, kappa, blk, 2, 1.0, 1, 2, 12, 1, 12)
    got = torch.zeros_like(pt)
    ctx.unpack_spinor(got, fk, 0, 1)
    assert float(torch.count_nonzero(got * ~even)) == 0
    err = float(torch.linalg.vector_norm(got - want_k) / torch.linalg.vector_norm(want_k))
    assert err <= 1e-2, ("schwarz_sap", err)
    # overlapping domains (R18), 256 domains of 14^3x26: the GPU applies all of them, the oracle two of them
    # (block 0, whose domain reaches through the wrap in every direction and holds the antiperiodic plane, and an
    # interior one); compared on those blocks' own boxes, where nothing else contributes
    ctx.set_schwarz_overlap(1)
    fk = ctx.new_field(1)
    ctx.schwarz(fk, ctx.pack_spinor(pt, 0, 1), 0, kappa, blk, 2, 1.0, 2, 12, 1)
    ctx.set_schwarz_overlap(0)
    got = torch.zeros_like(pt)
    ctx.unpack_spinor(got, fk, 0, 1)
    g = got.cpu().numpy()
    for box in (0, 1 + 4 * (2 + 4 * (1 + 4 * 2))):
        want = oracle.schwarz_ras(psi, U, T, BC, kappa, 0, blk, 1, n_mr=2, only_block=box)
        own = np.abs(want).sum(axis=(-1, -2)) > 0
        assert own.sum() == 12 * 12 * 12 * 24 // 2
        err = np.linalg.norm((g - want)[own]) / np.linalg.norm(want[own])
        assert err <= 1e-2, ("schwarz_ras", box, err)
    ctx.close()


@pytest.mark.parametrize("dims", [(16, 16, 16, 32), (24, 8, 4, 6), (32, 8, 2, 4)])
def test_tile_form_is_bit_identical_to_thread_form(dims):
    """Half precision, plain hopping term: the CTA-tile kernel with bulk-async (TMA engine) staging
    (csrc/dslash_tile.cuh; T = 128 or 96 sites per CTA, y / z / t wraps inside a tile, antiperiodic t) computes
    bit for bit what the one-thread-per-site kernel with per-thread cp.async staging computes, 20 launches in a
    row (the refill of a stage races with its readers unless ordered by the proxy fence), and meets the
    oracle."""
    import os
    c = Case(dims, 0.3, bc=(1, -1, 1, -1))
    psi = inputs.gaussian_spinor(dims, 4)
    d = torch.from_numpy(psi).cuda()
    try:
        for recon in (12, 18):
            for parity in (0, 1):
                for dagger in (False, True):
                    fin = c.ctx.pack_spinor(d, 1 - parity, 2)
                    os.environ["LQCD_B200_NO_TILE"] = "1"
                    ref = c.ctx.new_field(2)
                    c.ctx.dslash(ref, fin, parity, dagger, 2, recon)
                    os.environ["LQCD_B200_NO_TILE"] = "0"
                    for _ in range(20 if (recon == 12 and parity == 0) else 2):
                        out = c.ctx.new_field(2)
                        c.ctx.dslash(out, fin, parity, dagger, 2, recon)
                        assert torch.equal(out, ref), (recon, parity, dagger)
                    got = torch.zeros_like(d)
                    c.ctx.unpack_spinor(got, out, parity, 2)
                    want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
                    assert _rel(got.cpu().numpy(), want) <= TOL[2]
    finally:
        os.environ.pop("LQCD_B200_NO_TILE", None)
        c.ctx.close()
