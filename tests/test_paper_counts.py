"""Byte / flop bookkeeping against the counts the paper prints (tests/golden/paper_counts.txt): the byte
model bench.py reports rooflines with (CPU), and the packed field sizes of the library (GPU)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _golden():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_counts.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = int(line[1])
    return out


def test_bench_byte_model_uses_the_papers_counts():
    import bench
    g = _golden()
    size = {0: 8, 1: 4, 2: 2}
    for prec in (0, 1, 2):
        norm = 4 if prec == 2 else 0
        assert bench.SPINOR_B[prec] == g["spinor_reals_per_site"] * size[prec] + norm
        assert bench.CLOVER_B[prec] == g["clover_reals_per_site"] * size[prec] + norm
        for recon in (g["link_reals_full"], g["link_reals_recon12"], g["link_reals_recon8"]):
            # compulsory bytes: input + output spinor and one link per neighbour (each link is read once)
            assert bench.dslash_bytes(prec, recon) == 2 * bench.SPINOR_B[prec] + g["dslash_neighbours"] * recon * size[prec]
            assert bench.matpc_bytes(prec, recon) == 5 * bench.SPINOR_B[prec] + 2 * g["dslash_neighbours"] * recon * size[prec] + 2 * bench.CLOVER_B[prec]
    # flop conventions of BASELINE.json re-derived: 8 hops x (12 projection adds + 2 SU(3) matvecs of 66) + 7 x 24 accumulations
    assert bench.FLOP_DSLASH == g["dslash_neighbours"] * (12 + 2 * 66) + (g["dslash_neighbours"] - 1) * g["spinor_reals_per_site"]
    # clover: two Hermitian 6x6 blocks: 6 real-diagonal x complex (2 flop each component -> 12) + 30 complex MACs (8 flop) each
    assert 2 * (6 * 2 + 30 * 8) == 504
    assert bench.FLOP_MATPC == 2 * bench.FLOP_DSLASH + 2 * 504 + 48


@pytest.mark.gpu
def test_packed_field_sizes_follow_the_papers_counts():
    from paper_1109_2935_b200 import lqcd
    g = _golden()
    dims = (4, 6, 8, 4)
    vh = 4 * 6 * 8 * 4 // 2
    ctx = lqcd.Context(dims, (1, 1, 1, -1), 0)
    assert ctx.field_bytes(lqcd.PREC_DOUBLE) == vh * g["spinor_reals_per_site"] * 8
    assert ctx.field_bytes(lqcd.PREC_SINGLE) == vh * g["spinor_reals_per_site"] * 4
    assert ctx.field_bytes(lqcd.PREC_HALF) == vh * (g["spinor_reals_per_site"] * 2 + 4)          # + one fp32 norm per site (R9)
    assert ctx.lib.lqcd_field_bytes(ctx.h, lqcd.FIELD_STAGGERED_PARITY, lqcd.PREC_DOUBLE) == vh * g["staggered_reals_per_site"] * 8
    assert ctx.lib.lqcd_field_bytes(ctx.h, lqcd.FIELD_STAGGERED_PARITY, lqcd.PREC_SINGLE) == vh * g["staggered_reals_per_site"] * 4
    p = ctx.make_params(0.12, 1.0, 1e-8)
    assert p.mr_steps == g["gcr_mr_steps"] and p.gcr_kmax == 16
    ctx.close()
