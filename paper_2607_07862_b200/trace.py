"""Per-CTA unit timeline of one run, from the kernel's own timestamps (`mlp_pipe_cta_records`; the paper's
in-kernel instrumentation).

    python -m paper_2607_07862_b200.trace --config 1 [--mode pipelined|sequential] [--no-autotune] [--workqueue] [--pair] [--every 12]

Prints, for every `--every`-th CTA, when it started, requested its first weights, started its first MMA and exited,
what it waited for (SM cycles -> us at the SM clock), and its first units with their four timestamps (weight loader
starts the unit / has requested its last weights / accumulator complete / epilogue done), all in us relative to
the first CTA's first instruction.  Needs a B200; synthetic inputs of the BASELINE.json config.
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main() -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--mode", default="pipelined", choices=["pipelined", "sequential"])
    ap.add_argument("--no-autotune", action="store_true")
    ap.add_argument("--workqueue", action="store_true")
    ap.add_argument("--pair", action="store_true", help="CTA pairs (MLP_FLAG_PAIR)")
    ap.add_argument("--every", type=int, default=12)
    ap.add_argument("--split-k", type=str, default="")
    ap.add_argument("--tile-n", type=int, default=0)
    ap.add_argument("--act", type=int, default=-1, help="override the activation: 0 none, 1 ReLU, 2 GeLU-tanh")
    ap.add_argument("--sm-mhz", type=float, default=0.0,
                    help="SM clock for cycles -> us; 0 = the median clock sampled (NVML) while the timed runs executed")
    args = ap.parse_args()

    import torch

    from paper_2607_07862_b200 import binding as B
    from paper_2607_07862_b200 import inputs, timing

    cfg = inputs.CONFIGS[args.config]
    if args.act >= 0:
        cfg = inputs.Config(cfg.name + f"_act{args.act}", cfg.M, cfg.widths, args.act, cfg.dist, cfg.seed)
    kind = B.MLP_CTA_PIPELINED if args.mode == "pipelined" else B.MLP_SEQUENTIAL
    flags = (0 if args.no_autotune else B.MLP_FLAG_AUTOTUNE) | (B.MLP_FLAG_WORKQUEUE if args.workqueue else 0) | (B.MLP_FLAG_PAIR if args.pair else 0)
    X, sets = timing.device_inputs(torch, cfg, timing.weight_sets_for(cfg))
    Y = torch.empty((cfg.M, cfg.widths[-1]), dtype=torch.bfloat16, device="cuda")
    split = [int(x) for x in args.split_k.split(",")] if args.split_k else []
    p = B.MlpPipe(cfg.M, cfg.widths, cfg.act, B.make_mode(kind, flags=flags, split_k_layer=split, tile_n=args.tile_n))
    sampler = timing.ClockSampler(timing.nvml_index_for(torch, torch.cuda.current_device()))
    lat, clocks = timing.time_steps(torch, p, X, sets, Y, 50, 10, sampler)
    st = p.stats()
    L = cfg.n_layers
    print(f"{cfg.name}: CUDA-event median {lat['median']:.1f} us; unit tile {st.tile_n}x{st.tile_m}, stages {st.stages}, "
          f"K-split {list(st.split_k)[:L]}, reduce mode {list(st.reduce_mode)[:L]}, tickets {list(st.units)[:L]}")
    # SM cycles per us: the clock the runs really had (an idle-to-busy GPU is not at its maximum clock), else the maximum
    cyc = args.sm_mhz or (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0
    print(f"SM clock for cycle counts: {cyc:.0f} MHz ({'given' if args.sm_mhz else 'sampled during the timed runs'})")
    for cls in range(1 if kind == B.MLP_CTA_PIPELINED else L):
        recs = p.cta_records(cls)
        t0 = min(r.ts[0] for r in recs)
        span = (max(r.ts[7] for r in recs) - t0) / 1e3
        ends = sorted((r.ts[7] - t0) / 1e3 for r in recs)
        print(f"launch class {cls}: first CTA start -> last CTA exit {span:.1f} us; CTA exits min / median / max "
              f"{ends[0]:.1f} / {ends[len(ends) // 2]:.1f} / {ends[-1]:.1f} us")
        print("  columns: start, setup done, first unit known, first weights requested, first MMA, first accumulator, "
              "first unit stored, exit")
        for i in range(0, len(recs), max(1, args.every)):
            r = recs[i]
            ts = " ".join(f"{(int(t) - t0) / 1e3:6.1f}" if t else "     -" for t in r.ts)
            w = [int(x) / cyc for x in r.wait]
            print(f"  cta {i:3d}: {ts} | waits: W ring {w[0]:5.1f}  MMA on operands {w[2]:5.1f}  epilogue on accumulator {w[4]:5.1f}  "
                  f"flags {int(r.flag_stall_cycles) / cyc:5.1f}  gather {w[1]:4.1f}  partial {w[6]:4.1f}  direct {w[7]:4.1f}  arrival {w[5]:4.1f} us")
            for u in range(B.MLP_UNIT_TRACE if hasattr(B, "MLP_UNIT_TRACE") else 12):
                if r.unit_ts[u][0] == 0 or int(r.unit_ts[u][0]) < t0:
                    break
                uid = r.unit_id[u]
                t = [(int(x) - t0) / 1e3 for x in r.unit_ts[u]]
                kind_s = f"reduce cols {16 * (uid & 0x7f):3d}.." if uid & 0x80 else f"K-slice {uid & 0x7f:2d}"
                print(f"      layer {uid >> 28} tile {(uid >> 8) & 0xfffff:4d} {kind_s}: {t[0]:6.1f} {t[1]:6.1f} {t[2]:6.1f} {t[3]:6.1f}")
    p.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
