"""Host-side logic that needs no GPU: the algorithmic-work model bench.py reports against
(SURVEY.md section 8 / 8d table), wave partitioning, the ragged length recipe."""
import importlib.util
import os

from paper_2606_01143_b200 import inputs, schedule

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(spec)
spec.loader.exec_module(bench)


def test_flop_model_matches_survey_table():
    f = bench.flops(inputs.config_7b())
    # A 0.188, B-fwd 0.662, B-bwd 1.654, C 0.470 TF; step 2.97, replay 7.58, ideal 2.55x
    assert abs(f["A"] / 1e12 - 0.188) < 1e-3 and abs(f["B_fwd"] / 1e12 - 0.6615) < 1e-3
    assert abs(f["B_bwd"] / 1e12 - 1.6537) < 1e-3 and abs(f["C"] / 1e12 - 0.4699) < 1e-3
    assert abs(f["step"] / 1e12 - 2.973) < 1e-3 and abs(f["replay"] / 1e12 - 7.578) < 1e-3
    assert abs(f["ideal_speedup"] - 2.549) < 1e-3
    # fwd : bwd = 4 : 10 on the same pair set, so the pair model is weight-free
    assert f["B_bwd"] * 4 == f["B_fwd"] * 10 and f["C"] * 4 == f["A"] * 10


def test_speedup_model_grows_with_prefix_ratio_and_group_size():
    """the amortisation model is monotone in both knobs."""
    sp = {(r, n): bench.flops(inputs.config_sweep(r, n))["ideal_speedup"]
          for r in (20, 50, 83, 95) for n in (2, 4, 8, 16)}
    for r in (20, 50, 83, 95):
        assert sp[(r, 2)] < sp[(r, 4)] < sp[(r, 8)] < sp[(r, 16)]
    for n in (2, 4, 8, 16):
        assert sp[(20, n)] < sp[(50, n)] < sp[(83, n)] < sp[(95, n)]
    assert abs(sp[(95, 16)] - 6.74) < 0.01 and abs(sp[(20, 2)] - 1.02) < 0.01


def test_wave_partition_and_ragged_recipe():
    assert schedule._waves(5, 2) == [[0, 1], [2, 3], [4]]
    assert schedule._waves(3, 0) == [[0], [1], [2]] and schedule._waves(0, 4) == []
    Ls = inputs.config_ragged().Ls
    assert len(Ls) == 16 and all(256 <= x <= 2048 for x in Ls) and Ls == inputs.config_ragged().Ls


def test_bwd_split_model_is_host_only_deterministic_and_even():
    """The backward item split comes from a list-scheduling simulation on the host (prefixflow.cu
    SplitModel): no GPU needed.  configs[1], one packed wave on 148 SMs: 8 x 7 = 56 pairs in 4 even
    chunks of 14 with all prefix items first, 5 chunks of 12 in the default interleaved launch order
    (profiles/r2_kernel_experiments.md)."""
    from paper_2606_01143_b200 import binding as pf
    d = pf.make_desc(28, 4, 128)
    cu8 = [1024 * i for i in range(9)]
    a, b = pf.pf_bwd_split_model(d, 5120, cu8)
    assert (a, b) == pf.pf_bwd_split_model(d, 5120, cu8)
    assert 8 <= a <= 14 and 1 <= b <= 7          # 4-7 chunks of the 56 pairs: about one round of CTAs per chunk
    # Phase C / replay: no prefix source, one sequence: only the heads-per-item choice matters
    a1, b1 = pf.pf_bwd_split_model(d, 0, [0, 5120])
    assert 1 <= b1 <= 7 and a1 >= 1
    # one call per suffix: fewer pairs per item than the packed wave (more parallelism is needed)
    a2, _ = pf.pf_bwd_split_model(d, 5120, [0, 1024])
    assert 1 <= a2 < a
    # a tiny launch on a big GPU is split as finely as it can be; a one-SM GPU gets whole key tiles
    assert pf.pf_bwd_split_model(pf.make_desc(2, 2, 64), 256, [0, 64], 148)[0] == 1
    assert pf.pf_bwd_split_model(d, 5120, cu8, 1) == (56, 7)
    with __import__("pytest").raises(pf.PrefixFlowError):
        pf.pf_bwd_split_model(d, 5120, [0, 10, 5])
