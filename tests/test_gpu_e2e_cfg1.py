"""Config 1 (BASELINE.json configs[0], fp32) FREE-RUNNING end to end: the GPU path and the oracle each run the
whole beam search on their own (nothing teacher-forced) and must produce identical beams (north star:
"End-to-end beam sets on the fp32 config must be identical").

Why identity is robust: the oracle records the selection margins of seed 0 (key gap between rank W and rank
W+1 per level, >= 9.8e-3) and its adjacent-rank gaps inside the beam (>= 1.07e-2); the fp32 attention + fp32
projection differ from the fp64 oracle by ~1e-6 relative, four orders of magnitude less."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("from_logits", [False, True], ids=["logprob_topk", "raw_logits_topk"])
def test_cfg1_free_running_identical_beams(from_logits):
    from _free_running import run_free_running
    cfg = wl.get_config("cfg1")
    gpu, oracle = run_free_running(cfg, seed=0, from_logits=from_logits)
    for u, tr in enumerate(oracle):
        gaps = [float(np.min(-np.diff(s.astype(np.float64)))) for s in tr.scores]
        print(f"user {u}: selection margins {tr.margins}; min adjacent gap inside the beam {gaps}")
        assert min(tr.margins) > 1e-4 and min(gaps) > 1e-4      # recorded, seed 0
        for t in range(cfg.d):
            assert np.array_equal(gpu["parent"][t][u], tr.parents[t]), f"level {t + 1}: parents differ"
            assert np.array_equal(gpu["code"][t][u], tr.codes[t]), f"level {t + 1}: codes differ"
            # scores: fp32 attention/projection vs fp64 -- close, not bitwise
            assert np.abs(gpu["score"][t][u].astype(np.float64) - tr.scores[t].astype(np.float64)).max() < 1e-4
            ref = tr.attn_out[t]
            err = np.abs(gpu["attn"][t][u] - ref).max() / np.abs(ref).max()
            assert err <= 2e-3, f"step {t}: attention rel err {err:.3e}"
        assert np.array_equal(gpu["paths"][u], tr.paths), "final SID paths differ"
        assert len({tuple(p) for p in gpu["paths"][u]}) == tr.paths.shape[0]      # a set of distinct paths
