"""Improved staggered path on the GPU (-m gpu) against oracle/staggered_oracle.cpp on the same seeded
inputs: pack/unpack round trip, the hopping term on both parities, M^dag M + sigma, free-field closed
form, on a ragged lattice (Vh = 1440 sites = 11.25 CTAs) with mixed boundary conditions."""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs

pytestmark = pytest.mark.gpu
STOL = {0: 1e-13, 1: 1e-5}


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


class SCase:
    def __init__(self, dims, eps, bc, seed=1, unit=False, long_scale=0.0):
        from paper_1109_2935_b200 import lqcd
        self.lqcd, self.dims, self.bc = lqcd, dims, bc
        if unit:
            one = inputs.unit_gauge(dims)
            self.fat, self.lng = 1.125 * one, (-1.0 / 24.0) * one
        else:
            self.fat, self.lng = inputs.staggered_links(dims, eps, seed)
        self.ctx = lqcd.Context(dims, bc, 0)
        self.ctx.load_staggered_links(torch.from_numpy(self.fat).cuda(), torch.from_numpy(self.lng).cuda(), long_scale)
        self.par = inputs.parity_mask(dims)

    def mask(self, p):
        return (self.par == p)[..., None]

    def op(self, fn, chi, p_in, p_out, prec):
        d = torch.from_numpy(np.ascontiguousarray(chi)).cuda()
        fin = self.ctx.pack_staggered(d, p_in, prec)
        fout = self.ctx.new_staggered_field(prec)
        fn(fout, fin)
        res = torch.zeros_like(d)
        self.ctx.unpack_staggered(res, fout, p_out, prec)
        torch.cuda.synchronize()
        return res.cpu().numpy()


@pytest.fixture(scope="module")
def ragged():
    return SCase((6, 4, 10, 12), 0.4, (-1, 1, 1, -1))


def test_pack_unpack_roundtrip(ragged):
    c = ragged
    chi = inputs.gaussian_colour_vector(c.dims, 2)
    for prec in (0, 1):
        for p in (0, 1):
            got = c.op(lambda o, i: o.copy_(i), chi, p, p, prec)
            want = chi * c.mask(p)
            if prec == 0:
                assert np.array_equal(got, want)
            else:
                assert _rel(got, want) <= 1e-7 and np.max(np.abs(got[c.par != p])) == 0.0


@pytest.mark.parametrize("prec", [0, 1])
def test_dslash_and_mdagm(ragged, prec):
    c = ragged
    chi = inputs.gaussian_colour_vector(c.dims, 3)
    for p in (0, 1):
        want = oracle.stag_dslash(chi * c.mask(1 - p), c.fat, c.lng, c.bc) * c.mask(p)
        got = c.op(lambda o, i: c.ctx.staggered_dslash(o, i, p, prec), chi, 1 - p, p, prec)
        assert _rel(got, want) <= STOL[prec], ("dslash", p)
        assert np.max(np.abs(got[c.par != p])) == 0.0
        for mass, sigma in ((0.05, 0.0), (0.3, 0.7)):
            want = oracle.stag_MdagM(chi * c.mask(p), c.fat, c.lng, c.bc, mass, sigma) * c.mask(p)
            got = c.op(lambda o, i: c.ctx.staggered_mdagm(o, i, p, mass, sigma, prec), chi, p, p, prec)
            assert _rel(got, want) <= STOL[prec], ("mdagm", p, mass, sigma)


def test_free_field_closed_form_on_gpu():
    dims, bc, n = (8, 4, 6, 12), (1, -1, 1, -1), (3, 1, 2, 5)
    c = SCase(dims, 0.0, bc, unit=True)
    X, Y, Z, T = dims
    p = 2 * np.pi * (np.array(n) + np.where(np.array(bc) < 0, 0.5, 0.0)) / np.array(dims)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    chi = phase[..., None] * np.array([0.3 - 1.0j, 2.0, -0.5 + 0.25j])
    m, sigma = 0.07, 0.4
    lam = m * m + sigma + np.sum((1.125 * np.sin(p) - np.sin(3 * p) / 24.0) ** 2)
    for par in (0, 1):
        got = c.op(lambda o, i: c.ctx.staggered_mdagm(o, i, par, m, sigma, 0), chi, par, par, 0)
        assert _rel(got, lam * chi * c.mask(par)) <= 1e-13
    c.ctx.close()


def test_staggered_errors():
    from paper_1109_2935_b200 import lqcd
    ctx = lqcd.Context((4, 4, 4, 4), (1, 1, 1, -1), 0)
    f, g = ctx.new_staggered_field(1), ctx.new_staggered_field(1)
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.staggered_dslash(f, g, 0, 1)                        # links not loaded
    assert e.value.code == lqcd.ESTATE
    assert ctx.lib.lqcd_field_bytes(ctx.h, lqcd.FIELD_STAGGERED_PARITY, 2) == 0     # no half-precision staggered fields
    ctx.close()
    ctx = lqcd.Context((2, 4, 4, 4), (1, 1, 1, -1), 0)
    one = torch.from_numpy(inputs.unit_gauge((2, 4, 4, 4))).cuda()
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.load_staggered_links(one, one)                      # extent 2 < 4
    assert e.value.code == lqcd.EINVAL
    ctx.close()


@pytest.mark.parametrize("ms_prec", [1, 0])
@pytest.mark.parametrize("parity", [0, 1])
def test_multishift_solver(ragged, parity, ms_prec):
    """lqcd_staggered_multishift (single-precision multi-shift CG + mixed-precision refinement):
    every x_i equals the oracle's own CG solution of (M^dag M + sigma_i) x = b on that parity, and the true
    residual recomputed with the ORACLE's operator meets the tolerance."""
    c = ragged
    mass, sigmas, tol = 0.08, [0.0, 0.01, 0.1, 0.5, 2.0], 1e-10
    b = inputs.gaussian_colour_vector(c.dims, 5) * c.mask(parity)
    x = torch.zeros((len(sigmas),) + b.shape, dtype=torch.complex128, device="cuda")
    infos = c.ctx.staggered_multishift(x, torch.from_numpy(b).cuda(), parity, mass, sigmas, tol, multishift_prec=ms_prec)
    xs = x.cpu().numpy()
    assert infos[0]["matpc_precond"] > 0                    # the multi-shift phase ran
    for i, sg in enumerate(sigmas):
        assert infos[i]["status"] == 0 and infos[i]["true_residual"] <= tol
        assert np.max(np.abs(xs[i][c.par != parity])) == 0.0
        res = np.linalg.norm(b - oracle.stag_MdagM(xs[i], c.fat, c.lng, c.bc, mass, sg)) / np.linalg.norm(b)
        assert res <= 1.05 * tol, (i, res)
        xo, io = oracle.stag_cg(b, c.fat, c.lng, c.bc, mass, sg, tol=1e-13)
        assert io["status"] == 0 and _rel(xs[i], xo) <= 1e-8, i
    # larger shifts are better conditioned: their refinement needs no more iterations than the smallest shift's
    assert infos[-1]["iterations"] <= infos[0]["iterations"]
    if ms_prec == 0:      # the fp64 multi-shift phase reaches the tolerance by itself: the refinement only confirms
        assert sum(i["iterations"] for i in infos) <= 3 * len(sigmas)


def test_multishift_edges(ragged):
    c = ragged
    lq = c.lqcd
    b = torch.from_numpy(inputs.gaussian_colour_vector(c.dims, 6)).cuda()
    x = torch.zeros((2,) + tuple(b.shape), dtype=torch.complex128, device="cuda")
    for bad in ([0.5, 0.1], [-0.1, 0.2], [0.3, 0.3]):         # not ascending / negative / repeated
        with pytest.raises(lq.LqcdError) as e:
            c.ctx.staggered_multishift(x, b, 0, 0.1, bad, 1e-8)
        assert e.value.code == lq.EINVAL
    # zero source: x = 0 at once
    infos = c.ctx.staggered_multishift(x, torch.zeros_like(b), 0, 0.1, [0.0, 1.0], 1e-10)
    assert all(i["status"] == 0 and i["iterations"] == 0 for i in infos) and float(x.abs().max()) == 0.0
    # a single shift and a loose tolerance that the single-precision phase meets by itself
    x1 = torch.zeros((1,) + tuple(b.shape), dtype=torch.complex128, device="cuda")
    infos = c.ctx.staggered_multishift(x1, b, 1, 0.2, [0.0], 1e-4)
    assert infos[0]["status"] == 0 and infos[0]["true_residual"] <= 1e-4 and infos[0]["iterations"] == 0
    # iteration cap
    infos = c.ctx.staggered_multishift(x, b, 0, 0.01, [0.0, 0.5], 1e-12, max_iter=3, allow_fail=True)
    assert infos[0]["status"] == lq.ENOCONV and 0 < infos[0]["true_residual"] < 1.0


@pytest.mark.parametrize("prec", [0, 1])
def test_long_links_stored_as_12_reals(prec):
    """long_scale = c3 declares the long links c3 x SU(3): 12 reals per long link, third row reconstructed.
    Same operator as the 18-real storage, against the oracle; a field that is not c3 x SU(3) is refused."""
    dims, bc = (6, 4, 10, 12), (-1, 1, 1, -1)
    c = SCase(dims, 0.4, bc, long_scale=-1.0 / 24.0)
    chi = inputs.gaussian_colour_vector(dims, 3)
    for p in (0, 1):
        want = oracle.stag_dslash(chi * c.mask(1 - p), c.fat, c.lng, c.bc) * c.mask(p)
        got = c.op(lambda o, i: c.ctx.staggered_dslash(o, i, p, prec), chi, 1 - p, p, prec)
        assert _rel(got, want) <= STOL[prec]
        want = oracle.stag_MdagM(chi * c.mask(p), c.fat, c.lng, c.bc, 0.1, 0.3) * c.mask(p)
        got = c.op(lambda o, i: c.ctx.staggered_mdagm(o, i, p, 0.1, 0.3, prec), chi, p, p, prec)
        assert _rel(got, want) <= STOL[prec]
    lq = c.lqcd
    fat, lng = torch.from_numpy(c.fat).cuda(), torch.from_numpy(c.lng).cuda()
    for bad_lng, scale in ((lng, -1.0 / 20.0), (fat, 1.125), (lng * np.exp(0.3j), -1.0 / 24.0)):   # wrong scale / not unitary / det != 1
        with pytest.raises(lq.LqcdError) as e:
            c.ctx.load_staggered_links(fat, bad_lng.contiguous(), scale)
        assert e.value.code == lq.EINVAL
    with pytest.raises(lq.LqcdError) as e:
        c.ctx.staggered_dslash(c.ctx.new_staggered_field(1), c.ctx.new_staggered_field(1), 0, 1)      # a refused load leaves no links
    assert e.value.code == lq.ESTATE
    c.ctx.close()


def test_extent_four_three_hop_wraps_to_the_backward_neighbour():
    """L_mu = 4: x + 3 mu and x - mu are the same site (and x - 3 mu = x + mu), reached once through the long
    link with the wrap's boundary sign and once through the fat link; every hop of a 4^4 lattice wraps
    somewhere.  Operator and a full multi-shift solve against the oracle."""
    dims, bc = (4, 4, 4, 4), (-1, 1, -1, -1)
    c = SCase(dims, 0.5, bc, seed=9)
    chi = inputs.gaussian_colour_vector(dims, 3)
    for prec in (0, 1):
        for p in (0, 1):
            want = oracle.stag_dslash(chi * c.mask(1 - p), c.fat, c.lng, c.bc) * c.mask(p)
            got = c.op(lambda o, i: c.ctx.staggered_dslash(o, i, p, prec), chi, 1 - p, p, prec)
            assert _rel(got, want) <= STOL[prec]
    b = chi * c.mask(1)
    sig = [0.0, 0.3]
    x = torch.zeros((2,) + b.shape, dtype=torch.complex128, device="cuda")
    infos = c.ctx.staggered_multishift(x, torch.from_numpy(b).cuda(), 1, 0.1, sig, 1e-11)
    for i, sg in enumerate(sig):
        xo, _ = oracle.stag_cg(b, c.fat, c.lng, c.bc, 0.1, sg, tol=1e-13)
        assert infos[i]["status"] == 0 and _rel(x[i].cpu().numpy(), xo) <= 1e-9
    c.ctx.close()


def test_full_size_32x64_operator_and_solve():
    """32^3x64 (the size bench.py --op staggered times): Dslash fp32/fp64 with 18- and 12-real long links
    against the oracle on the full lattice, and a 3-shift solve whose true residuals are recomputed by
    the oracle's operator."""
    from paper_1109_2935_b200 import lqcd
    dims, bc = (32, 32, 32, 64), (1, 1, 1, -1)
    fat = (inputs.random_gauge_torch(dims, 0.3, 31, device="cuda") * 1.125).contiguous()
    lng = (inputs.random_gauge_torch(dims, 0.3, 33, device="cuda") * (-1.0 / 24.0)).contiguous()
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    chi = torch.view_as_complex(torch.randn((64, 32, 32, 32, 3, 2), generator=g, dtype=torch.float64, device="cuda")).contiguous()
    fn, ln, cn = fat.cpu().numpy(), lng.cpu().numpy(), chi.cpu().numpy()
    want = torch.from_numpy(oracle.stag_dslash(cn, fn, ln, bc)).cuda()
    ctx = lqcd.Context(dims, bc, 0)
    for long_scale in (0.0, -1.0 / 24.0):
        ctx.load_staggered_links(fat, lng, long_scale)
        for prec in (0, 1):
            got = torch.zeros_like(chi)
            for p in (0, 1):
                o = ctx.new_staggered_field(prec)
                ctx.staggered_dslash(o, ctx.pack_staggered(chi, 1 - p, prec), p, prec)
                ctx.unpack_staggered(got, o, p, prec)
            err = float(torch.linalg.vector_norm(got - want) / torch.linalg.vector_norm(want))
            assert err <= STOL[prec], (long_scale, prec, err)
    par = torch.from_numpy(inputs.parity_mask(dims) == 0).cuda()[..., None]
    b = (chi * par).contiguous()
    sig, mass, tol = [0.0, 0.02, 0.5], 0.05, 1e-10
    x = torch.zeros((3,) + tuple(chi.shape), dtype=torch.complex128, device="cuda")
    infos = ctx.staggered_multishift(x, b, 0, mass, sig, tol)
    bn = b.cpu().numpy()
    for i, sg in enumerate(sig):
        res = np.linalg.norm(bn - oracle.stag_MdagM(x[i].cpu().numpy(), fn, ln, bc, mass, sg)) / np.linalg.norm(bn)
        assert infos[i]["status"] == 0 and res <= 1.05 * tol, (i, res)
    ctx.close()


@pytest.mark.parametrize("ms_prec", [1, 0])
def test_multishift_wide_shift_range_and_small_mass(ms_prec):
    """Eight shifts over six decades (0 ... 100) at mass 0.005: the zeta recurrences of the converged (large)
    shifts underflow while the small ones still iterate; every solution meets 1e-11 by the oracle's operator."""
    dims, bc = (8, 8, 8, 16), (1, 1, 1, -1)
    c = SCase(dims, 0.4, bc, seed=3, long_scale=-1.0 / 24.0)
    b = inputs.gaussian_colour_vector(dims, 4) * c.mask(0)
    sig = [0.0, 1e-4, 1e-3, 1e-2, 0.1, 1.0, 10.0, 100.0]
    x = torch.zeros((len(sig),) + b.shape, dtype=torch.complex128, device="cuda")
    infos = c.ctx.staggered_multishift(x, torch.from_numpy(b).cuda(), 0, 0.005, sig, 1e-11, max_iter=20000, multishift_prec=ms_prec)
    for i, sg in enumerate(sig):
        res = np.linalg.norm(b - oracle.stag_MdagM(x[i].cpu().numpy(), c.fat, c.lng, c.bc, 0.005, sg)) / np.linalg.norm(b)
        assert infos[i]["status"] == 0 and res <= 1.05e-11, (i, res)
    c.ctx.close()
