"""GPU parity: the CUDA path (through the C ABI) vs the fp64 oracle, teacher-forced
on identical seeded inputs (SURVEY.md section 8(c) comparison protocol).
Selection bit-exact; attention within 2e-3 (fp32) / 1.5e-2 (bf16) of max|out|."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

SMALL = ["cfg1", "f32_gqa", "cfg2_small", "cfg3_small", "cfg4_small", "cfg5_small", "paper_small"]


@pytest.mark.parametrize("name", SMALL)
def test_teacher_forced_parity(name):
    from _parity import run_teacher_forced
    rep = run_teacher_forced(wl.get_config(name))
    bad = [r for r in rep if not r[2]]
    assert not bad, f"{name}: {bad}\nfull report: {rep}"
    assert any(r[0] == "topk" for r in rep) and any(r[0] == "attn" for r in rep)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5", "paper_b1"])
def test_full_size_parity(name):
    """BASELINE.json's full sizes in bench.py's launch configuration (DecodePass under CUDA-graph replay):
    all selections bit-exact, append bitwise, sampled attention rows within tolerance."""
    from _parity import run_full_size
    rep = run_full_size(wl.get_config(name))
    bad = [r for r in rep if not r[2]]
    assert not bad, f"{name}: {bad}\nfull report: {rep}"


@pytest.mark.parametrize("name", ["cfg2", "cfg4", "cfg5", "paper_b1"])
def test_full_size_parity_from_logits(name):
    """The same pass with the selection fed RAW logits (stark_beam_topk_logits, reading R22; bench.py
    --from-logits): every level's (score, parent, code) bit-exact vs oracle.select_beams_from_logits, the
    tree that results still appended and attended correctly."""
    from _parity import run_full_size
    rep = run_full_size(wl.get_config(name), n_samples=3, from_logits=True)
    bad = [r for r in rep if not r[2]]
    assert not bad, f"{name}: {bad}\nfull report: {rep}"
