"""Host logic of the ticket scheduler (step a1) checked WITHOUT a GPU: the unit tables
that mlp_pipe_plan_units returns are what the persistent kernel walks ticket by ticket, so their invariants are
the deadlock-freedom argument of DESIGN.md written as assertions."""
import pytest

from paper_2607_07862_b200 import binding as B
from paper_2607_07862_b200 import inputs

S, MB, P = B.MLP_SEQUENTIAL, B.MLP_MICROBATCH, B.MLP_CTA_PIPELINED

SHAPES = [(c.M, tuple(c.widths)) for c in inputs.CONFIGS] + [
    (1, (8, 8, 8)), (7, (72, 136, 8)), (300, (136, 264, 136)), (130, (264, 392, 200)), (16, (64, 128, 128, 128)),
    (1024, (8192, 8192, 8192)), (40, (136, 200)), (24, (64, 128, 72, 136, 64, 128, 64, 200, 64)),  # L = 1 and L = MLP_MAX_LAYERS
]
MODES = [
    dict(kind=P), dict(kind=S), dict(kind=MB, chunks=1), dict(kind=P, sm_split=0.5), dict(kind=P, split_k=4),
    dict(kind=P, split_k=3, flags=B.MLP_FLAG_DEBUG_REVERSE), dict(kind=P, tile_n=256, tile_m=64), dict(kind=P, tile_n=128),
    dict(kind=P, split_k_layer=[2, 9]), dict(kind=S, split_k=16), dict(kind=P, flags=B.MLP_FLAG_PAIR), dict(kind=S, flags=B.MLP_FLAG_PAIR, split_k=3),
    dict(kind=MB, chunks=1, flags=B.MLP_FLAG_MB_CORESIDENT), dict(kind=P, flags=B.MLP_FLAG_TWO_KERNEL, sm_split=0.625),
]


def _check_tables(M, widths, plan, tables, pair=False):
    L = len(widths) - 1
    rows = M
    assert plan.tile_m % 16 == 0 and 16 <= plan.tile_m <= 256 and plan.tile_n in (128, 256)
    assert plan.m_blks * plan.tile_m >= rows
    acc_cols = plan.tile_m if pair else (plan.tile_n // 128) * plan.tile_m   # pair mode: each CTA keeps its own 128 rows
    assert plan.acc_stages * acc_cols <= 512, "accumulator ring must fit the 512 TMEM columns"
    if pair:
        assert plan.tile_n == 256 and plan.tile_m % 32 == 0 and plan.grid % 2 == 0
    assert plan.smem_bytes <= 227 * 1024
    for l in range(L):
        K, N = widths[l], widths[l + 1]
        kb_total = -(-K // 64)
        tiles = plan.m_blks * -(-N // plan.tile_n)
        assert plan.tiles[l] == tiles
        sp = plan.split_k[l]
        table = tables[l]
        assert len(table) == plan.units[l]
        mma = [u for u in table if u[1] == 0]
        red = [u for u in table if u[1] == 1]
        # every (tile, K-slice) exactly once, and the slices of a tile tile [0, kb_total) without gap or overlap
        assert len(mma) == tiles * sp
        assert len({(t, ks) for t, _, ks, _, _ in mma}) == tiles * sp
        per_tile = {}
        for t, _, ks, a, b in mma:
            assert 0 <= t < tiles and 0 <= ks < sp and a < b
            per_tile.setdefault(t, []).append((a, b))
        for t, spans in per_tile.items():
            spans.sort()
            assert spans[0][0] == 0 and spans[-1][1] == kb_total
            assert all(spans[i][1] == spans[i + 1][0] for i in range(len(spans) - 1))
        mode = plan.reduce_mode[l]
        if sp == 1:
            assert mode == 0 and not red and plan.ready_inc[l] == 1
        elif mode == 1:
            assert not red and plan.ready_inc[l] == 1
        else:
            assert mode == 2
            # the reduce units of a tile partition its token columns, and every one of them holds a HIGHER ticket
            # than all K-slices of its tile (a unit only ever waits on lower tickets: no deadlock)
            pos_last_slice = {}
            for i, u in enumerate(table):
                if u[1] == 0:
                    pos_last_slice[u[0]] = i
            cols = {}
            for i, u in enumerate(table):
                if u[1] == 1:
                    assert i > pos_last_slice[u[0]]
                    assert u[3] % 16 == 0 and u[3] < u[4] <= plan.tile_m
                    cols.setdefault(u[0], []).append((u[3], u[4]))
            assert set(cols) == set(range(tiles))
            for t, spans in cols.items():
                spans.sort()
                assert spans[0][0] == 0 and spans[-1][1] == plan.tile_m and len(spans) == plan.ready_inc[l]
                assert all(spans[i][1] == spans[i + 1][0] for i in range(len(spans) - 1))


@pytest.mark.parametrize("M,widths", SHAPES)
@pytest.mark.parametrize("mode", MODES, ids=[str(i) for i in range(len(MODES))])
def test_unit_tables_are_a_valid_schedule(M, widths, mode):
    kw = dict(mode)
    m = B.make_mode(**kw)
    if kw.get("tile_m") and kw["tile_m"] * 2 > 512:
        pytest.skip("shape not supported")
    pair = bool(kw.get("flags", 0) & B.MLP_FLAG_PAIR)
    if kw.get("flags", 0) & B.MLP_FLAG_TWO_KERNEL and len(widths) != 3:
        pytest.skip("the two-kernel pipeline is defined for 2 layers")
    if pair and (-(-min(M, 256) // 16) * 16) % 32 != 0 and M <= 256:
        pytest.skip("pair mode needs a token tile that is a multiple of 32")
    plan, tables = B.plan(M, widths, m, num_sms=148)
    if pair and plan.tile_m % 32 != 0:
        pytest.skip("pair mode needs a token tile that is a multiple of 32")
    _check_tables(M, widths, plan, tables, pair=pair)
    assert plan.model_us > 0


def test_plan_depends_on_sm_count_and_is_deterministic():
    cfg = inputs.CONFIGS[1]
    a, ta = B.plan(cfg.M, cfg.widths, B.make_mode(P), num_sms=148)
    b, tb = B.plan(cfg.M, cfg.widths, B.make_mode(P), num_sms=148)
    assert ta == tb and list(a.split_k) == list(b.split_k)
    c, tc = B.plan(cfg.M, cfg.widths, B.make_mode(P), num_sms=64)
    assert c.grid == 64
    _check_tables(cfg.M, cfg.widths, c, tc)


def test_pipelined_plan_orders_consumer_slices_by_k():
    """K-slice-major order of a many-slice consumer layer: its first tickets cover the lowest K range, i.e. depend on
    the producer's EARLIEST tiles only (what lets the consumer start while the producer is still running)."""
    cfg = inputs.CONFIGS[1]
    plan, tables = B.plan(cfg.M, cfg.widths, B.make_mode(P))
    if plan.split_k[1] > 4:
        first = tables[1][: plan.tiles[1]]
        assert all(u[2] == 0 and u[3] == 0 for u in first)


def test_coresident_and_two_kernel_grids():
    """MLP_FLAG_MB_CORESIDENT sizes every micro-batch launch so that the launches of the L streams fit on the device together;
    MLP_FLAG_TWO_KERNEL partitions the SMs between the producer and the consumer kernel."""
    cfg = inputs.CONFIGS[2]
    full, _ = B.plan(cfg.M, cfg.widths, B.make_mode(MB, chunks=2), num_sms=148)
    co, tco = B.plan(cfg.M, cfg.widths, B.make_mode(MB, chunks=2, flags=B.MLP_FLAG_MB_CORESIDENT), num_sms=148)
    assert full.grid == 148 and co.grid == 74
    co4, _ = B.plan(128, inputs.CONFIGS[4].widths, B.make_mode(MB, chunks=8, flags=B.MLP_FLAG_MB_CORESIDENT), num_sms=148)
    assert co4.grid == 148 // 4            # four layers = four streams
    tk, ttk = B.plan(cfg.M, cfg.widths, B.make_mode(P, flags=B.MLP_FLAG_TWO_KERNEL, sm_split=0.75), num_sms=148)
    assert tk.grid == 148 and tk.producer_ctas == 148   # (per-kernel grids are 111 + 37; the plan reports the device-wide grid)
    _check_tables(cfg.M, cfg.widths, tk, ttk)
    import ctypes
    out = B.mlp_plan()
    w4 = (ctypes.c_int * 5)(*inputs.CONFIGS[4].widths)
    bad = B.make_mode(S, flags=B.MLP_FLAG_TWO_KERNEL)
    assert B.load().mlp_pipe_plan(128, 4, w4, ctypes.byref(bad), 148, ctypes.byref(out)) == B.MLP_ERR_UNSUPPORTED
    bad = B.make_mode(P, flags=B.MLP_FLAG_MB_CORESIDENT)
    assert B.load().mlp_pipe_plan(128, 4, w4, ctypes.byref(bad), 148, ctypes.byref(out)) == B.MLP_ERR_INVALID


def test_two_kernel_needs_a_cta_for_each_kernel():
    """A grid of one CTA cannot be split into a producer and a consumer kernel: plan and plan_units refuse it (create runs
    the same check) instead of planning a producer launch of 0 CTAs; a grid of 2 is the smallest that works (1 + 1).  A chain
    that is not 2 layers long is refused by the planner as it is by create."""
    import ctypes
    lib = B.load()
    cfg = inputs.CONFIGS[0]
    w = (ctypes.c_int * 3)(*cfg.widths)
    out, units, n = B.mlp_plan(), (B.mlp_unit * 8)(), ctypes.c_int()
    for sms, grid in ((148, 1), (1, 0)):
        m = B.make_mode(P, flags=B.MLP_FLAG_TWO_KERNEL, grid=grid)
        assert lib.mlp_pipe_plan(cfg.M, 2, w, ctypes.byref(m), sms, ctypes.byref(out)) == B.MLP_ERR_UNSUPPORTED
        assert lib.mlp_pipe_plan_units(cfg.M, 2, w, ctypes.byref(m), sms, 0, units, 8, ctypes.byref(n)) == B.MLP_ERR_UNSUPPORTED
    ok, tables = B.plan(cfg.M, cfg.widths, B.make_mode(P, flags=B.MLP_FLAG_TWO_KERNEL, grid=2), num_sms=148)
    assert ok.grid == 2
    _check_tables(cfg.M, cfg.widths, ok, tables)
    w4 = (ctypes.c_int * 5)(*inputs.CONFIGS[4].widths)
    m = B.make_mode(P, flags=B.MLP_FLAG_TWO_KERNEL)
    assert lib.mlp_pipe_plan(128, 4, w4, ctypes.byref(m), 148, ctypes.byref(out)) == B.MLP_ERR_UNSUPPORTED


def test_plan_rejects_bad_arguments():
    import ctypes
    lib = B.load()
    w = (ctypes.c_int * 3)(64, 128, 128)
    out = B.mlp_plan()
    assert lib.mlp_pipe_plan(16, 2, w, None, 148, None) == B.MLP_ERR_INVALID
    assert lib.mlp_pipe_plan(0, 2, w, None, 148, ctypes.byref(out)) == B.MLP_ERR_INVALID
    assert lib.mlp_pipe_plan(16, 2, w, None, 0, ctypes.byref(out)) == B.MLP_ERR_INVALID
    bad = (ctypes.c_int * 3)(64, 100, 128)
    assert lib.mlp_pipe_plan(16, 2, bad, None, 148, ctypes.byref(out)) == B.MLP_ERR_INVALID
    assert lib.mlp_pipe_plan(16, 2, w, None, 148, ctypes.byref(out)) == B.MLP_OK
    # limits of the unit table's 16-bit fields: rejected before the planner runs (include/mlp_pipe.h, "limits")
    huge = (ctypes.c_int * 3)(64, 1 << 20, 128)
    assert lib.mlp_pipe_plan(1 << 20, 2, huge, None, 148, ctypes.byref(out)) == B.MLP_ERR_UNSUPPORTED
    deep = (ctypes.c_int * 3)(64 * 65536, 128, 128)
    assert lib.mlp_pipe_plan(16, 2, deep, None, 148, ctypes.byref(out)) == B.MLP_ERR_UNSUPPORTED
