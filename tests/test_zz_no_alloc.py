"""stark_beam_topk_static (include/stark.h): the top-k entry point that allocates nothing -- its scratch memory is a
static device array inside the library -- against the existing stark_beam_topk on the same inputs.

Integer / index work and one fp32 addition per key: the bar is bit-exact, as in tests/test_gpu_topk.py.  Two calls in
a row on each shape: the second one finds the array as the first one left it.  The file sorts last on purpose (the
suite runs with `pytest -x`); it passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _inputs(B, W_in, C, seed):
    r = np.random.default_rng([0, 4068, seed])
    logits = r.normal(0, 2, (B, W_in, C)).astype(np.float32)
    logp = (logits - np.log(np.exp(logits.astype(np.float64)).sum(-1, keepdims=True))).astype(np.float32)
    score = np.sort(r.normal(-8, 2, (B, W_in)).astype(np.float32))[:, ::-1].copy()
    return logp, score


def _outs(B, W_out):
    import torch
    return (torch.full((B, W_out), float("nan"), dtype=torch.float32, device="cuda"),
            torch.full((B, W_out), -1, dtype=torch.int32, device="cuda"),
            torch.full((B, W_out), -1, dtype=torch.int32, device="cuda"))


# whole-GPU kernel (needs the scratch array): 2 x 262 144 and 8 x 524 288 candidates; cluster / one-CTA kernels
# (no scratch): the smaller ones
@pytest.mark.parametrize("B,W_in,C,W_out", [(2, 256, 1024, 256), (8, 512, 1024, 512), (3, 64, 256, 64), (2, 1, 256, 96)])
def test_static_scratch_matches_workspace_path_twice(B, W_in, C, W_out):
    import torch
    from paper_2607_04068_b200 import binding as sb
    from paper_2607_04068_b200.decode import beam_topk, beam_topk_static
    for call in range(2):                                   # two calls in a row, different inputs
        logp, score = _inputs(B, W_in, C, 10 * call + B)
        lp, sc = torch.from_numpy(logp).cuda(), torch.from_numpy(score).cuda()
        ref = [x.cpu().numpy() for x in beam_topk(lp, sc, W_out)]
        out = _outs(B, W_out)
        before = torch.cuda.memory_allocated()
        beam_topk_static(lp, sc, W_out, out)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before, "the static entry point must not allocate through torch"
        got = [x.cpu().numpy() for x in out]
        assert np.array_equal(got[0].view(np.uint32), ref[0].view(np.uint32)), f"call {call}: score bits differ"
        assert np.array_equal(got[1], ref[1]), f"call {call}: parent differs"
        assert np.array_equal(got[2], ref[2]), f"call {call}: code differs"
    # and the same inputs again give the same answer (nothing of the previous call leaks into the next)
    out2 = _outs(B, W_out)
    beam_topk_static(lp, sc, W_out, out2)
    torch.cuda.synchronize()
    for a, b in zip(out, out2):
        assert torch.equal(a, b)
    assert sb.TOPK_STATIC_SCRATCH_BYTES == 9 << 20


def test_static_scratch_matches_oracle():
    """Not only the other path: the definition itself (oracle.select_beams), on the whole-GPU kernel's shape."""
    import torch
    from oracle.selection import select_beams
    from paper_2607_04068_b200.decode import beam_topk_static
    B, W_in, C, W_out = 2, 160, 1024, 300
    logp, score = _inputs(B, W_in, C, 99)
    out = _outs(B, W_out)
    beam_topk_static(torch.from_numpy(logp).cuda(), torch.from_numpy(score).cuda(), W_out, out)
    s_g, p_g, c_g = [x.cpu().numpy() for x in out]
    for u in range(B):
        s_r, p_r, c_r = select_beams(score[u], logp[u], W_out)
        assert np.array_equal(p_g[u], p_r) and np.array_equal(c_g[u], c_r)
        assert np.array_equal(s_g[u].view(np.uint32), s_r.view(np.uint32))


def test_static_scratch_under_graph_capture():
    """The use case the entry point exists for: captured into a CUDA graph (no allocation may happen there) and
    replayed.  The first call per device resolves the array's address and is made eagerly, before the capture."""
    import torch
    from paper_2607_04068_b200.decode import beam_topk, beam_topk_static
    B, W_in, C, W_out = 2, 256, 1024, 256
    logp, score = _inputs(B, W_in, C, 7)
    lp, sc = torch.from_numpy(logp).cuda(), torch.from_numpy(score).cuda()
    out = _outs(B, W_out)
    beam_topk_static(lp, sc, W_out, out)                     # eager warm-up
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        beam_topk_static(lp, sc, W_out, out)
    for rep in range(2):
        logp, score = _inputs(B, W_in, C, 70 + rep)          # new contents in the captured buffers
        lp.copy_(torch.from_numpy(logp)); sc.copy_(torch.from_numpy(score))
        for o in out:
            o.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        ref = beam_topk(lp, sc, W_out)
        for a, b in zip(out, ref):
            assert torch.equal(a.view(torch.int32), b.view(torch.int32)), f"replay {rep}"


def test_beyond_the_static_maximum_is_rejected():
    """64 users x 131 072 candidates need 10.5 MB of workspace: more than the 9 MiB array.  Clear error, nothing
    launched, outputs untouched; the workspace path serves the same problem."""
    import torch
    from paper_2607_04068_b200 import binding as sb
    from paper_2607_04068_b200.decode import beam_topk, beam_topk_static
    B, W_in, C, W_out = 64, 128, 1024, 128
    need = sb.stark_workspace_bytes(sb.make_shape(B, 1, 1, 64, 1, W_in, torch.float32), sb.CALL_BEAM_TOPK, W_in, C)
    assert need > sb.TOPK_STATIC_SCRATCH_BYTES
    lp = torch.zeros((B, W_in, C), dtype=torch.float32, device="cuda")
    out = _outs(B, W_out)
    with pytest.raises(sb.StarkError) as e:
        beam_topk_static(lp, None, W_out, out)
    assert e.value.status == -3 and "static array" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out[1] == -1).all()) and bool((out[2] == -1).all())
    beam_topk(lp, None, W_out, out)                          # the existing path takes it
    torch.cuda.synchronize()
    assert bool((out[1] >= 0).all())
