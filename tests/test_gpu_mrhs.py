"""Multi-right-hand-side Dslash / Mhat (-m gpu): every right-hand side of lqcd_dslash_mrhs and
lqcd_matpc_mrhs against the oracle applied to that source alone, and against the single-source
calls (same arithmetic per site: bit-identical), on a ragged lattice (Vh = 960 = 30 CTAs of 32
sites) and for right-hand-side counts that are not multiples of the 4 a CTA handles."""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs
from test_gpu_parity import Case, _rel, TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ragged():
    return Case((6, 4, 10, 8), 0.3, bc=(-1, 1, 1, -1))


@pytest.mark.parametrize("prec", [0, 1, 2])
@pytest.mark.parametrize("nrhs", [1, 3, 4, 6])
def test_mrhs_matches_oracle_and_single(ragged, prec, nrhs):
    c = ragged
    ctx, kappa = c.ctx, 0.124
    srcs = [inputs.gaussian_spinor(c.dims, 100 + r) * (1.0 + r) for r in range(nrhs)]    # different norms per source
    dev = [torch.from_numpy(s).cuda() for s in srcs]
    for recon in (18, 12, 8):
        tol = TOL[prec]        # fp64 recon-8 included (R10: measured <= 1.2e-14)
        for parity in (0, 1):
            for dagger in (False, True):
                fin = ctx.new_fields(prec, nrhs)
                fout = ctx.new_fields(prec, nrhs)
                for r in range(nrhs):
                    ctx.pack_spinor(dev[r], 1 - parity, prec, out=fin[r])
                ctx.dslash_mrhs(fout, fin, nrhs, parity, dagger, prec, recon)
                for r in range(nrhs):
                    got = torch.zeros_like(dev[r])
                    ctx.unpack_spinor(got, fout[r], parity, prec)
                    want = oracle.dslash(srcs[r] * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
                    assert _rel(got.cpu().numpy(), want) <= tol, ("dslash", recon, parity, dagger, r)
                    single = ctx.new_field(prec)
                    ctx.dslash(single, fin[r], parity, dagger, prec, recon)
                    assert torch.equal(single, fout[r]), ("dslash vs single", recon, parity, dagger, r)
            fin = ctx.new_fields(prec, nrhs)
            fout = ctx.new_fields(prec, nrhs)
            for r in range(nrhs):
                ctx.pack_spinor(dev[r], parity, prec, out=fin[r])
            ctx.matpc_mrhs(fout, fin, nrhs, parity, False, kappa, prec, recon)
            for r in range(nrhs):
                got = torch.zeros_like(dev[r])
                ctx.unpack_spinor(got, fout[r], parity, prec)
                want = oracle.matpc(srcs[r], c.U, c.T, c.bc, kappa, parity)
                assert _rel(got.cpu().numpy(), want) <= tol, ("matpc", recon, parity, r)
                single = ctx.new_field(prec)
                ctx.matpc(single, fin[r], parity, False, kappa, prec, recon)
                assert torch.equal(single, fout[r]), ("matpc vs single", recon, parity, r)


def test_mrhs_argument_errors(ragged):
    c = ragged
    lq = c.lqcd
    f = c.ctx.new_fields(1, 2)
    g = c.ctx.new_fields(1, 2)
    for bad in (0, -1, 65):
        with pytest.raises(lq.LqcdError) as e:
            c.ctx.dslash_mrhs(f, g, bad, 0, False, 1, 12)
        assert e.value.code == lq.EINVAL
    with pytest.raises(lq.LqcdError) as e:
        c.ctx.matpc_mrhs(f, f, 2, 0, False, 0.12, 1, 12)            # aliasing
    assert e.value.code == lq.EINVAL


@pytest.mark.parametrize("sloppy", [0, 1, 2])
def test_invert_mrhs(sloppy):
    """lqcd_invert_mrhs: 5 sources (one zero, one 100x larger, one a point source) solved in lockstep;
    every source meets its own full-system criterion by the ORACLE's operator and equals the
    single-source lqcd_invert solution."""
    c = Case((8, 8, 8, 16), 0.2)
    lq = c.lqcd
    kappa, nrhs = 0.124, 5
    srcs = [inputs.gaussian_spinor(c.dims, 200 + r) for r in range(nrhs)]
    srcs[1] = np.zeros_like(srcs[1])
    srcs[2] = 100.0 * srcs[2]
    srcs[3] = np.zeros_like(srcs[3])
    srcs[3][5, 2, 1, 1, 2, 1] = 1.0 - 0.5j
    b = torch.from_numpy(np.stack(srcs)).cuda()
    x = torch.zeros_like(b)
    p = c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_BICGSTAB, prec=(0, sloppy, sloppy), recon=(18, 12, 12))
    infos = c.ctx.invert_mrhs(x, b, p)
    xs = x.cpu().numpy()
    for r in range(nrhs):
        assert infos[r]["status"] == 0, r
        if r == 1:
            assert np.max(np.abs(xs[r])) == 0.0 and infos[r]["iterations"] == 0
            continue
        res = np.linalg.norm(srcs[r] - oracle.M(xs[r], c.U, c.T, c.bc, kappa)) / np.linalg.norm(srcs[r])
        assert res <= 1.05e-10, (r, res)
        assert abs(res - infos[r]["true_residual"]) <= 0.05 * res + 1e-14
        x1 = torch.zeros_like(b[r])
        c.ctx.invert(x1, b[r].contiguous(), p)
        assert _rel(xs[r], x1.cpu().numpy()) <= 1e-8, r
    # iteration cap: every unfinished source reports LQCD_ENOCONV with its true residual
    p2 = c.ctx.make_params(kappa, 1.0, 1e-12, solver=lq.SOLVER_BICGSTAB, prec=(0, sloppy, sloppy), recon=(18, 12, 12), max_iter=3)
    x.zero_()
    infos = c.ctx.invert_mrhs(x, b, p2, allow_fail=True)
    assert [i["status"] for i in infos] == [lq.ENOCONV, 0, lq.ENOCONV, lq.ENOCONV, lq.ENOCONV]
    xs = x.cpu().numpy()
    for r in (0, 2, 3, 4):
        res = np.linalg.norm(srcs[r] - oracle.M(xs[r], c.U, c.T, c.bc, kappa)) / np.linalg.norm(srcs[r])
        assert infos[r]["iterations"] == 3 and 1e-12 < res < 1.0 and abs(res - infos[r]["true_residual"]) <= 1e-6 * res
    # the single-source solver still works on scalar set 0 afterwards, GCR-DD is refused in batched mode
    x1 = torch.zeros_like(b[0])
    assert c.ctx.invert(x1, b[0].contiguous(), p)["true_residual"] <= 1e-10
    with pytest.raises(lq.LqcdError) as e:
        c.ctx.invert_mrhs(x, b, c.ctx.make_params(kappa, 1.0, 1e-10, solver=lq.SOLVER_GCR_DD, schwarz_block=(4, 4, 4, 8)))
    assert e.value.code == lq.EINVAL
    c.ctx.close()
