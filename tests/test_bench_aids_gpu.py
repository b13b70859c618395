"""The measurement aids of bench.py on a GPU: the probes behind the roofline's denominator and behind the
operand-delivery bound of DESIGN.md section 6 return what the analysis rests on."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu


def test_fma_chain_rates_are_near_the_derived_peaks():
    import bench_aids
    ffma = bench_aids.pipe_probe(0, 8192)["gfma_per_s"]
    dfma = bench_aids.pipe_probe(2, 8192)["gfma_per_s"]
    # 148 SM x 128 (64) lanes x 1.965 GHz = 37.2e3 (18.6e3) G lane-ops/s at the maximum clock: the chains cannot exceed
    # that, reach most of it (whatever clock this box runs at), and the FP64 pipe has half the lanes
    assert 0.5 * 37224 <= ffma <= 1.02 * 37224, ffma
    assert 0.5 * 18612 <= dfma <= 1.02 * 18612, dfma
    assert 1.8 <= ffma / dfma <= 2.2, (ffma, dfma)


def test_operand_forms_cost_what_the_analysis_says():
    """Two register pairs (or an immediate) run at the pipe's rate; a third distinct 64-bit register operand costs a third
    cycle; the operand-reuse cache and the 32-bit scalar form lie in between (profiles/r2_allpairs_sass_analysis.md)."""
    import bench_aids
    r = {bench_aids.OPERAND_FORMS[k]: bench_aids.operand_probe(k, 4, 4096)["tlaneops_per_s"] for k in range(8)}
    print(r)
    two, three = r["ffma2_two_pairs"], r["ffma2_three_pairs"]
    assert abs(r["ffma2_two_pairs_imm"] / two - 1) <= 0.03
    assert 0.60 <= three / two <= 0.72                                               # ~2/3: three cycles instead of two
    assert three < r["ffma2_two_pairs_one_scalar"] < r["ffma2_three_pairs_one_reused"] < two
    assert 0.60 <= r["dfma_three_regs"] / r["dfma_two_regs"] <= 0.72
    assert r["dfma_three_regs"] < r["dfma_three_regs_one_reused"] < r["dfma_two_regs"]
    assert 1.8 <= two / r["dfma_two_regs"] <= 2.2
