"""Time the real-space partner on one GPU: rbe_short_range (both force kernels, polynomial and tabulated pair term) and
rbe_rbl_forces.

    python -m paper_2407_09315_b200.time_short_range [--config water_nacl_1m] [--rs 10] [--rc 5] [--p 30] [--calls 10]

Prints one JSON line with the mean milliseconds per call (CUDA events, after warm-up).  Also the command the ncu
captures of these kernels under profiles/ are taken around (it only calls the public binding)."""
from __future__ import annotations

import argparse
import json


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="water_nacl_1m")
    ap.add_argument("--rs", type=float, default=10.0)
    ap.add_argument("--rc", type=float, default=5.0)
    ap.add_argument("--p", type=int, default=30)
    ap.add_argument("--calls", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--with-energy", action="store_true")
    args = ap.parse_args()

    import torch

    from . import inputs, rbe

    cfg = inputs.CONFIGS[args.config]
    ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    x = torch.from_numpy(inputs.make_atoms(cfg)).cuda()
    f = torch.empty_like(x)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(fn):
        for i in range(args.warmup):
            fn(i)
        torch.cuda.synchronize()
        e0.record()
        for i in range(args.calls):
            fn(args.warmup + i)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.calls

    out = {"config": cfg.name, "N": cfg.N, "r_s": args.rs, "r_c": args.rc, "p": args.p, "with_energy": args.with_energy}
    out["short_range_ms"] = timed(lambda i: ctx.rbe_short_range(x, args.rs, f, with_energy=args.with_energy))
    ctx.rbe_set_pair_table(True)
    out["short_range_table_ms"] = timed(lambda i: ctx.rbe_short_range(x, args.rs, f, with_energy=args.with_energy))
    ctx.rbe_set_pair_table(False)
    ctx.rbe_set_pair_kernel(1)            # fine cells, tensor-core cutoff test, ordered pairs
    out["short_range_cells_ms"] = timed(lambda i: ctx.rbe_short_range(x, args.rs, f, with_energy=args.with_energy))
    ctx.rbe_set_pair_table(True)
    out["short_range_cells_table_ms"] = timed(lambda i: ctx.rbe_short_range(x, args.rs, f, with_energy=args.with_energy))
    ctx.rbe_set_pair_table(False)
    ctx.rbe_set_pair_kernel(0)
    out["rbl_ms"] = timed(lambda i: ctx.rbe_rbl_forces(x, args.rc, args.rs, args.p, cfg.seed, i, f))
    print(json.dumps(out))


if __name__ == "__main__":
    main()
