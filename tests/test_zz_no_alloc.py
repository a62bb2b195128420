"""dkd_match_static — the matcher for callers that may not allocate device memory — against dkd_match.

Some users of this library run where cudaMalloc is off limits: a plug-in inside a host application that owns the
whole device-memory budget, a real-time loop in which a call that takes the driver's allocation lock is banned, a
process whose memory pool has already taken the entire GPU.  They cannot create a dkd context (dkd_create allocates the
workspace), so they get one context-free entry point whose only scratch memory — the column-split partials between
k_match_tc and k_match_finalize — is a 1 MiB array compiled into the library (include/dkd.h, dkd_match_static).

What is checked here: the entry point returns what dkd_match returns on the same inputs (match indices equal; the
similarities within TOL_SIM of tests/test_gpu_match.py — they are in fact the same kernels in the same geometry), on
calls made one after the other WITHOUT clearing anything in between, so that the second call runs on the array as the
first one left it (a different shape, so the stale records do not line up with the new ones); that repeated calls leave
the amount of free device memory where it was; and that a problem beyond the array's capacity is refused with
DKD_ERR_CAPACITY before anything is launched.

This file is collected last on purpose (pytest -x stops at the first failure), and it passes both on its own in a
fresh process — its first call then does the one-time device set-up — and after the rest of the suite.
"""
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu
TOL_SIM = 1e-4                                                    # as in tests/test_gpu_match.py


def _problem(P, Na, Nb, D, seed, ragged):
    ca = [Na - 17, Na][:P] if ragged else None
    cb = [Nb, max(Nb - 33, 1)][:P] if ragged else None
    A, B, cta, ctb = synth.match_sets(P, Na, Nb, D, seed=seed, count_a=ca, count_b=cb)
    return A.cuda(), B.cuda(), cta.cuda(), ctb.cuda()


def _static(dkd, prob, ratio, mutual):
    A, B, ca, cb = prob
    P, Na, _ = A.shape
    out = torch.full((P, Na), -7, dtype=torch.int32, device="cuda")
    sim = torch.full((P, Na, 2), -7.0, dtype=torch.float32, device="cuda")
    dkd.match_static(A, B, out, sim, ca, cb, ratio=ratio, mutual=mutual)
    return out, sim


def _same(got, want):
    torch.cuda.synchronize()
    assert torch.equal(got[0], want[0])
    assert float((got[1] - want[1]).abs().max()) <= TOL_SIM


def test_static_scratch_matcher_equals_dkd_match_on_consecutive_calls():
    import paper_2607_01757_b200 as dkd
    ctx = dkd.DKD(max_batch=2, max_h=64, max_w=128, max_top_k=64, max_dim=0)
    try:
        big = _problem(2, 1500, 1300, 128, seed=11, ragged=True)     # 256-wide tiles, several column splits, mutual
        small = _problem(2, 300, 260, 64, seed=12, ragged=True)      # 128-wide tiles; lands on big's leftovers
        one = _problem(1, 97, 40, 256, seed=13, ragged=False)
        want_big = ctx.match(*big, ratio=0.8, mutual=True)
        want_small = ctx.match(*small, ratio=0.8, mutual=False)
        want_one = ctx.match(*one, ratio=1e9, mutual=True)
        torch.cuda.synchronize()
        # two calls in a row on the shared array, then a third and a repeat of the first
        got_big = _static(dkd, big, 0.8, True)
        got_small = _static(dkd, small, 0.8, False)
        _same(got_big, want_big)
        _same(got_small, want_small)
        _same(_static(dkd, one, 1e9, True), want_one)
        _same(_static(dkd, big, 0.8, True), want_big)
        # calls after the first allocate nothing: free device memory does not drop (outputs are made beforehand)
        outs = [(torch.empty_like(w[0]), torch.empty_like(w[1])) for w in (want_big, want_small)]
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            for prob, o, mutual in ((big, outs[0], True), (small, outs[1], False)):
                dkd.match_static(prob[0], prob[1], o[0], o[1], prob[2], prob[3], ratio=0.8, mutual=mutual)
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        assert free_after >= free_before
        _same(outs[0], want_big)
        _same(outs[1], want_small)
    finally:
        ctx.close()


def test_static_scratch_matcher_refuses_what_does_not_fit():
    import paper_2607_01757_b200 as dkd
    P, N, D = 16, 4096, 64                                           # 16 x 4096 records per direction: 2 x 65536 with mutual
    A = torch.zeros((P, N, D), dtype=torch.float16, device="cuda")
    out = torch.full((P, N), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(dkd.DKDError) as ei:
        dkd.match_static(A, A, out, None, ratio=0.8, mutual=True)
    assert ei.value.code == -3 and str(dkd.MATCH_STATIC_MAX_RECS) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == -7).all())                                   # nothing was launched
    with pytest.raises(dkd.DKDError) as ei:                          # argument errors carry their text too
        dkd.match_static(A[:, :, :48].contiguous(), A[:, :, :48].contiguous(), out, None)
    assert ei.value.code == -2 and "D must be" in str(ei.value)
