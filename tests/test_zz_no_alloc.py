"""lqcd_cdot_static (-m gpu): the allocation-free reduction entry point against the existing path (lqcd_cdot).

Collected last on purpose (file name): the suite runs with `pytest -x`.  Both paths form the same per-site sums in
the field's arithmetic type and add them in fp64; only the order of the fp64 additions differs, so they agree to the
tolerance test_gpu_parity.py::test_blas_reductions uses for lqcd_cdot against numpy.
"""
import numpy as np
import pytest
import torch

from paper_1109_2935_b200 import inputs, lqcd

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL = ((0, 1e-14), (1, 1e-6), (2, 2e-4))      # test_blas_reductions


def _fields(ctx, dims, prec, seeds):
    return [ctx.pack_spinor(torch.from_numpy(inputs.gaussian_spinor(dims, s)).cuda(), 0, prec) for s in seeds]


def _norm(ctx, f, prec):
    return abs(ctx.cdot(f, f, prec)) ** 0.5


@pytest.mark.parametrize("dims", [(6, 4, 10, 8), (8, 8, 8, 16)])     # 960 sites: 4 CTAs, ragged tail; 4096: 16 CTAs
def test_cdot_static_matches_cdot_on_two_calls_in_a_row(dims):
    ctx = lqcd.Context(dims, BC, 0)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device="cuda")
    for prec, tol in TOL:
        fx, fy = _fields(ctx, dims, prec, (11, 12))
        scale = _norm(ctx, fx, prec) * _norm(ctx, fy, prec)
        # first call: <x,y>; second call straight after it, other operands: <y,x> (the scratch keeps the first call's partials)
        ctx.cdot_static(fx, fy, prec, out)
        first = out.cpu().numpy().copy()
        ctx.cdot_static(fy, fx, prec, out)
        second = out.cpu().numpy().copy()
        want_xy, want_yx = ctx.cdot(fx, fy, prec), ctx.cdot(fy, fx, prec)
        assert abs(complex(first[0], first[1]) - want_xy) <= tol * scale
        assert abs(complex(second[0], second[1]) - want_yx) <= tol * scale
        assert abs(first[2] - ctx.cdot(fy, fy, prec).real) <= tol * scale
        assert abs(second[2] - ctx.cdot(fx, fx, prec).real) <= tol * scale
        # fixed summation order: a repeat gives the same bits
        ctx.cdot_static(fy, fx, prec, out)
        assert np.array_equal(out.cpu().numpy(), second)


def test_cdot_static_small_field_after_large_field_and_no_allocation():
    """The partials of a larger earlier call stay in the array; a smaller call must not read them.  And the call does
    not change the device's free memory (no cudaMalloc behind it)."""
    big, small = (8, 8, 8, 16), (4, 4, 4, 4)
    cb, cs = lqcd.Context(big, BC, 0), lqcd.Context(small, BC, 0)
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    bx, by = _fields(cb, big, 1, (3, 4))
    sx, sy = _fields(cs, small, 1, (5, 6))
    want = cs.cdot(sx, sy, 1)
    scale = _norm(cs, sx, 1) * _norm(cs, sy, 1)
    cb.cdot_static(bx, by, 1, out)               # also the first call of a fresh process: looks the address up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    cb.cdot_static(bx, by, 1, out)
    cs.cdot_static(sx, sy, 1, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    got = out.cpu().numpy()
    assert abs(complex(got[0], got[1]) - want) <= 1e-6 * scale


def test_cdot_static_rejects_fields_beyond_the_static_maximum():
    ctx = lqcd.Context((128, 64, 64, 64), BC, 0)     # 16,777,216 sites per parity > 2^23; the context holds no fields
    out = torch.zeros(3, dtype=torch.float64, device="cuda")
    dummy = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(lqcd.LqcdError) as e:
        ctx.cdot_static(dummy, dummy, 0, out)
    assert "maximum" in str(e.value) and "8388608" in str(e.value)
    with pytest.raises(lqcd.LqcdError):
        lqcd.Context((4, 4, 4, 4), BC, 0).cdot_static(dummy, dummy, 3, out)      # bad precision
