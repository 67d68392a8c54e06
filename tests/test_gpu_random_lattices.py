"""Seeded random sweep over lattice shapes, boundary conditions, precisions and compressions (-m gpu):
Dslash, Mhat (both even-odd forms), the Schwarz operator through one MR step, the multi-right-hand-side
kernels and the staggered Dslash, each against the oracle.  Shapes include extents 2, odd X/2 and
lattices smaller than one CTA; the draw is fixed by the seed, so a failure is reproducible."""
import numpy as np
import pytest
import torch

import oracle
from paper_1109_2935_b200 import inputs
from test_gpu_parity import Case, _rel, TOL

pytestmark = pytest.mark.gpu

EXTENTS = [2, 4, 6, 8, 10, 12]


def _draw(seed):
    rng = np.random.default_rng(1000 + seed)
    dims = tuple(int(rng.choice(EXTENTS)) for _ in range(4))
    while np.prod(dims) > 12000:
        dims = tuple(int(rng.choice(EXTENTS)) for _ in range(4))
    bc = tuple(int(rng.choice([1, -1])) for _ in range(4))
    return rng, dims, bc


@pytest.mark.parametrize("seed", range(12))
def test_random_wilson_clover(seed):
    rng, dims, bc = _draw(seed)
    c = Case(dims, float(rng.uniform(0.1, 0.6)), c_sw=float(rng.uniform(0.0, 1.5)), bc=bc, gauge_seed=seed)
    kappa = float(rng.uniform(0.05, 0.11))                      # kappa * c_sw < 1/6: A positive definite
    psi = inputs.gaussian_spinor(dims, 50 + seed)
    prec, recon = int(rng.integers(0, 3)), int(rng.choice([18, 12, 8]))
    parity, dagger = int(rng.integers(0, 2)), bool(rng.integers(0, 2))
    tol = TOL[prec] if not (prec == 0 and recon == 8) else 1e-10
    want = oracle.dslash(psi * c.mask(1 - parity), c.U, c.bc, dagger=dagger) * c.mask(parity)
    got = c.gpu_parity_op(lambda o, i: c.ctx.dslash(o, i, parity, dagger, prec, recon), psi, 1 - parity, parity, prec)
    assert _rel(got, want) <= tol, ("dslash", dims, bc, prec, recon)
    want = oracle.matpc(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc(o, i, parity, dagger, kappa, prec, recon), psi, parity, parity, prec)
    assert _rel(got, want) <= tol, ("matpc", dims, bc, prec, recon)
    want = oracle.matpc_sym(psi, c.U, c.T, c.bc, kappa, parity, dagger=dagger)
    got = c.gpu_parity_op(lambda o, i: c.ctx.matpc_sym(o, i, parity, dagger, kappa, prec, recon), psi, parity, parity, prec)
    assert _rel(got, want) <= tol, ("matpc_sym", dims, bc, prec, recon)
    # Schwarz operator with a random admissible block (even extents dividing dims), one MR step
    blk = tuple(int(rng.choice([b for b in (2, 4, 6) if d % b == 0] + [d])) for d in dims)
    want = oracle.schwarz(psi, c.U, c.T, c.bc, kappa, parity, blk, n_mr=1)
    got = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, parity, kappa, blk, 1, 1.0, prec, recon if recon != 8 else 12, prec), psi, parity, parity, prec)
    assert _rel(got, want) <= 3 * tol, ("schwarz", dims, bc, blk, prec)
    # three right-hand sides at once
    nrhs = 3
    dev = [torch.from_numpy(inputs.gaussian_spinor(dims, 70 + seed + r)).cuda() for r in range(nrhs)]
    fin, fout = c.ctx.new_fields(prec, nrhs), c.ctx.new_fields(prec, nrhs)
    for r in range(nrhs):
        c.ctx.pack_spinor(dev[r], parity, prec, out=fin[r])
    c.ctx.matpc_mrhs(fout, fin, nrhs, parity, dagger, kappa, prec, recon)
    for r in range(nrhs):
        single = c.ctx.new_field(prec)
        c.ctx.matpc(single, fin[r], parity, dagger, kappa, prec, recon)
        assert torch.equal(single, fout[r]), ("mrhs", dims, r)
    c.ctx.close()


@pytest.mark.parametrize("seed", range(8))
def test_random_staggered(seed):
    from paper_1109_2935_b200 import lqcd
    rng, dims, bc = _draw(100 + seed)
    dims = tuple(max(4, d) for d in dims)
    fat, lng = inputs.staggered_links(dims, float(rng.uniform(0.1, 0.6)), seed)
    use12 = bool(rng.integers(0, 2))
    ctx = lqcd.Context(dims, bc, 0)
    ctx.load_staggered_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), (-1.0 / 24.0) if use12 else 0.0)
    chi = inputs.gaussian_colour_vector(dims, 60 + seed)
    par = inputs.parity_mask(dims)
    prec, p = int(rng.integers(0, 2)), int(rng.integers(0, 2))
    mass, sigma = float(rng.uniform(0.01, 0.5)), float(rng.uniform(0.0, 1.0))
    d = torch.from_numpy(chi).cuda()
    out = ctx.new_staggered_field(prec)
    ctx.staggered_mdagm(out, ctx.pack_staggered(d, p, prec), p, mass, sigma, prec)
    got = torch.zeros_like(d)
    ctx.unpack_staggered(got, out, p, prec)
    mask = (par == p)[..., None]
    want = oracle.stag_MdagM(chi * mask, fat, lng, bc, mass, sigma) * mask
    assert _rel(got.cpu().numpy(), want) <= (1e-13 if prec == 0 else 1e-5), (dims, bc, prec, use12)
    ctx.close()


@pytest.mark.parametrize("seed", [0, 1, 5, 6, 14, 16, 17, 22, 25, 27])
def test_random_overlapping_schwarz(seed):
    """Overlapping Schwarz domains (R18) on drawn shapes: directions of extent 8 or 12 are cut into blocks of 4
    (an even number of them), the others stay whole; one site of overlap; random boundary signs, so that antiperiodic
    planes fall inside grown domains in x, y, z as well as t; against the oracle's block-by-block schwarz_ras."""
    rng, dims, bc = _draw(seed)
    blk = [4 if d in (8, 12) else d for d in dims]
    parts = [m for m in range(4) if blk[m] != dims[m]]
    if len(parts) % 2:
        blk[parts[0]] = dims[parts[0]]
        parts = parts[1:]
    assert len(parts) >= 2, "seed list and draw disagree"
    c = Case(dims, float(rng.uniform(0.1, 0.6)), c_sw=float(rng.uniform(0.0, 1.5)), bc=bc, gauge_seed=seed)
    kappa = float(rng.uniform(0.05, 0.11))
    psi = inputs.gaussian_spinor(dims, 90 + seed)
    prec, parity, n_mr = int(rng.integers(0, 3)), int(rng.integers(0, 2)), int(rng.integers(1, 4))
    want = oracle.schwarz_ras(psi, c.U, c.T, c.bc, kappa, parity, tuple(blk), 1, n_mr=n_mr)
    try:
        c.ctx.set_schwarz_overlap(1)
        got = c.gpu_parity_op(lambda o, i: c.ctx.schwarz(o, i, parity, kappa, tuple(blk), n_mr, 1.0, prec, 12, prec), psi, parity, parity, prec)
    finally:
        c.ctx.set_schwarz_overlap(0)
    assert _rel(got, want) <= 3 * n_mr * TOL[prec], ("schwarz_ras", dims, bc, blk, prec, n_mr)
