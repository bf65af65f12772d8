"""mlp_pipe_run_static: the CTA-pipelined pass for callers that must not allocate device memory.

Some users of this library cannot let it call cudaMalloc: an inference server whose own memory manager took all free HBM
at start-up (a later cudaMalloc fails, or eats into a budget the library does not know about), or a decode loop that
shares the GPU with other streams (cudaMalloc / cudaFree can stall the whole device, not only the calling stream).  For
them `mlp_pipe_run_static` keeps everything the kernel needs beyond X, W and Y -- hidden activations, split-K partials,
tickets, counters, unit tables -- in one fixed 32 MiB array inside the library instead of in a handle's cudaMalloc'ed
buffers (include/mlp_pipe.h).

What is checked here: its output against the existing path (`mlp_pipe_create` + `mlp_pipe_run`, default mode -- the same
plan), on calls IN A ROW, because every call shares that one array and finds the previous call's counters, tables and
activations in it; and that a problem beyond the array's size is refused with a message that says so.  The measure and
the bound are those of tests/test_gpu_parity.py (bit-equal in exact mode, err <= 2e-2 otherwise).

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It depends on nothing the other tests leave behind and leaves nothing behind for them.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07862_b200 import binding as B
from paper_2607_07862_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 2e-2   # tests/test_gpu_parity.py


def handle_path(cfg, X, Ws):
    """The existing path: a default CTA_PIPELINED handle (it owns cudaMalloc'ed scratch)."""
    p = B.MlpPipe(cfg.M, cfg.widths, cfg.act, None)
    try:
        Y = p.run(X, Ws)
        torch.cuda.synchronize()
        st = p.stats()
        assert st.status == 0 and st.ready_ok == 1
        return inputs.as_u16(Y.cpu())
    finally:
        p.close()


def device_inputs(cfg, reseed=0):
    if reseed:
        cfg = inputs.Config(cfg.name, cfg.M, cfg.widths, cfg.act, cfg.dist, cfg.seed + reseed, cfg.note)
    X, Ws = inputs.make_inputs(cfg)
    return cfg, X.cuda(), [w.cuda() for w in Ws]


def same(cfg, got, want):
    if cfg.dist == "exact":
        assert np.array_equal(got, want), "exact mode: the two paths must agree bit for bit"
    else:
        e = oracle.rel_err(got, want)
        assert e["nan"] == 0 and e["err"] <= TOL, e


@pytest.mark.parametrize("idx,dist", [(0, "exact"), (0, "uniform"), (1, "normal")])
def test_two_calls_in_a_row_match_the_handle_path(idx, dist):
    """Two calls back to back on one stream, no host synchronisation between them, different inputs: the second call
    starts from the first one's leftovers in the shared array and must still agree with the handle path."""
    cfg_a, Xa, Wa = device_inputs(inputs.get_config(idx, dist))
    cfg_b, Xb, Wb = device_inputs(inputs.get_config(idx, dist), reseed=100)
    Ya = torch.full((cfg_a.M, cfg_a.widths[-1]), float("nan"), dtype=torch.bfloat16, device="cuda")
    Yb = torch.full_like(Ya, float("nan"))
    B.run_static(Xa, Wa, cfg_a.act, Ya)
    B.run_static(Xb, Wb, cfg_b.act, Yb)
    torch.cuda.synchronize()
    same(cfg_a, inputs.as_u16(Ya.cpu()), handle_path(cfg_a, Xa, Wa))
    same(cfg_b, inputs.as_u16(Yb.cpu()), handle_path(cfg_b, Xb, Wb))
    assert not np.array_equal(inputs.as_u16(Ya.cpu()), inputs.as_u16(Yb.cpu())), "the two calls had different inputs"


def test_shape_changes_between_calls():
    """tiny -> decode -> 4-layer chain -> tiny, back to back: every call lays the array out anew over whatever the call
    before wrote there (the chain's 24 MiB cover what the small shapes use)."""
    seq = [inputs.get_config(0, "exact"), inputs.get_config(1), inputs.get_config(4), inputs.get_config(0, "exact")]
    runs = []
    for cfg in seq:
        cfg, X, Ws = device_inputs(cfg)
        Y = torch.full((cfg.M, cfg.widths[-1]), float("nan"), dtype=torch.bfloat16, device="cuda")
        B.run_static(X, Ws, cfg.act, Y)
        runs.append((cfg, X, Ws, Y))
    torch.cuda.synchronize()
    for cfg, X, Ws, Y in runs:
        same(cfg, inputs.as_u16(Y.cpu()), handle_path(cfg, X, Ws))


def test_too_large_is_refused_and_the_next_call_still_works():
    """M = 4096 on 8192 -> 8192 -> 8192 needs 64 MiB of hidden activations alone: refused before anything is enqueued,
    with the limit named in the message; the entry point stays usable."""
    M, w = 4096, [8192, 8192, 8192]
    X = torch.zeros((M, w[0]), dtype=torch.bfloat16, device="cuda")
    Ws = [torch.zeros((w[l + 1], w[l]), dtype=torch.bfloat16, device="cuda") for l in range(2)]
    with pytest.raises(B.MlpError) as ei:
        B.run_static(X, Ws, B.MLP_ACT_NONE)
    assert ei.value.status == B.MLP_ERR_UNSUPPORTED
    assert "MLP_STATIC_SCRATCH_BYTES" in str(ei.value) and str(B.MLP_STATIC_SCRATCH_BYTES) in str(ei.value)
    del X, Ws
    cfg, X, Ws = device_inputs(inputs.get_config(0, "exact"))
    Y = B.run_static(X, Ws, cfg.act)
    torch.cuda.synchronize()
    same(cfg, inputs.as_u16(Y.cpu()), handle_path(cfg, X, Ws))


def test_free_device_memory_does_not_move():
    """After one warm-up call (which may load the library's device code), calls for new shapes -- each replans and lays the
    array out again -- leave the device's free memory exactly where it was: nothing is allocated, nothing is freed."""
    small, X0, W0 = device_inputs(inputs.get_config(0, "uniform"))
    big, X1, W1 = device_inputs(inputs.get_config(1))
    Y0 = torch.empty((small.M, small.widths[-1]), dtype=torch.bfloat16, device="cuda")
    Y1 = torch.empty((big.M, big.widths[-1]), dtype=torch.bfloat16, device="cuda")
    B.run_static(X0, W0, small.act, Y0)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        B.run_static(X1, W1, big.act, Y1)
        B.run_static(X0, W0, small.act, Y0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
