#!/usr/bin/env python
"""bench.py -- RBE k-space ns/atom/step and fraction of roofline (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl reference]

One *step* = one pass of the whole hot path over one batch of synthetic input: rbe_step with a
fresh, pre-generated k-set = ONE cooperative launch (step_kernel: structure-factor phase, grid
barrier, distributed fixed-order reduction, grid barrier, force phase; the k-set rides in the
kernel parameters).  The two-launch form (rbe_set_kvectors + rbe_structure_factor + rbe_forces)
is timed beside it, call by call.
Workload at N = 1: BASELINE.json configs[2] (water + NaCl, N = 999 999, P = 200), the one the
metric is quoted on.  With N > 1 GPUs (torchrun) the atoms are sharded, one rank per GPU, the
k-set is replicated and the P complex structure factors are summed across ranks (weak
scaling: every rank owns 999 999 atoms of an n-times larger box at the same density).

Prints ONE JSON line (rank 0).  See DESIGN.md section 7 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "rbe_kspace_ns_per_atom_step"
UNIT = "ns/atom/step"
# SFU (MUFU) issue peak: 16 lanes/SM/clk x SMs x max SM clock (checked by
# the pipe microbenchmark in profiles/).  SURVEY.md s8(d): 2 sincos evaluations per (atom, k)
# pair per kernel are the algorithmic work that bounds this path.
MUFU_LANES_PER_SM = 16
FP32_LANES_PER_SM = 128
SFU_PER_PAIR_PER_KERNEL = 2
FMA_PER_PAIR_STEP = 13
BYTES_PER_ATOM_STEP = 48
# what the kernels EXECUTE per (atom, k) pair: the SF phase pairs atoms of equal |q|
# (3 MUFU per two pairs), the F phase uses the amplitude-phase form (1 MUFU per pair)
MUFU_EXECUTED_PER_PAIR = {"sf": 1.5, "f": 1.0}


def source_sha():
    """Fingerprint of the kernel sources: ncu counters in profiles/kernel_counters.csv are tied to it."""
    import hashlib
    h = hashlib.sha256()
    for f in ("rbe_kernels.cuh", "rbe_api.cu"):
        h.update(open(os.path.join(ROOT, "paper_2407_09315_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:12]


def read_counters(kernel, config):
    """dram bytes / warp instructions per launch from ONE `ncu --set full` capture (profiles/kernel_counters.csv)."""
    import csv
    path = os.path.join(ROOT, "profiles", "kernel_counters.csv")
    if not os.path.exists(path):
        return None
    for r in csv.DictReader(open(path)):
        if r["kernel"] == kernel and r["config"] == config:
            out = {"dram_bytes": float(r["dram_bytes"]), "inst_executed": float(r["inst_executed"]),
                   "inst_executed_pipe_xu": float(r["inst_executed_pipe_xu"]) if r.get("inst_executed_pipe_xu") else None,
                   "source_sha": r["source_sha"], "capture": r["capture"]}
            out["stale"] = out["source_sha"] != source_sha()
            if out["stale"]:
                print(f"bench: profiles/kernel_counters.csv row {kernel}:{config} was captured at source {out['source_sha']}, "
                      f"the kernels are now {source_sha()}: counters are stale", file=sys.stderr)
            return out
    return None


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


def roofline_times(n_atoms, P, num_sms, peaks):
    clk = peaks["sm_max_mhz"] * 1e6
    sfu_rate = num_sms * MUFU_LANES_PER_SM * clk
    fma_rate = num_sms * FP32_LANES_PER_SM * clk
    t_hbm = BYTES_PER_ATOM_STEP * n_atoms / (peaks["hbm_gbs"] * 1e9)
    t_fma = FMA_PER_PAIR_STEP * n_atoms * P / fma_rate
    t_sfu = 2 * SFU_PER_PAIR_PER_KERNEL * n_atoms * P / sfu_rate
    return {"hbm": t_hbm, "fma": t_fma, "sfu": t_sfu}, sfu_rate


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx, self.proc, self.path = gpu_index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "10"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        os.unlink(self.path)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def time_oracle(cfg_name, n_sample, steps, warmup, threads=None, last_kset=None):
    """The oracle as it stands, timed on the host cores, on the first n_sample atoms of the
    workload (cost is linear in atoms) with the workload's full batch of P wavevectors.
    last_kset: the k-set index of the LAST timed oracle step (the others keep 0, 1, ...), so that its result can be
    compared with what the GPU computed for that same k-set; the last (rho, F) are returned in `keep`."""
    import oracle
    from paper_2407_09315_b200 import inputs
    cfg = workload_config(cfg_name, 1)
    atoms = inputs.make_atoms(cfg)[:n_sample].copy()
    all_threads = oracle.max_threads()
    if threads:
        oracle.set_threads(threads)
    S = oracle.S(cfg.L, cfg.alpha)
    ts, keep = [], None
    for it in range(warmup + steps):
        k_idx = last_kset if (last_kset is not None and it == warmup + steps - 1) else it
        m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, k_idx)
        t0 = time.perf_counter()
        rho = oracle.rho(atoms, cfg.L, m)
        F = oracle.force(atoms, cfg.L, m, S, rho)
        dt = time.perf_counter() - t0
        if it >= warmup:
            ts.append(dt)
        keep = (k_idx, rho, F)
    per_step = sum(ts) / len(ts)
    used = oracle.max_threads()
    oracle.set_threads(all_threads)
    return per_step, per_step / n_sample * 1e9, used, cfg, keep


def workload_config(name, world):
    from paper_2407_09315_b200 import inputs
    if name.startswith("ions_"):
        parts = name.split("_")
        n = int(float(parts[1]))
        P = int(parts[2][1:]) if len(parts) > 2 else 200
        return inputs.ions_config(n, P)
    return inputs.CONFIGS[name]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    cfg0 = workload_config(args.config, 1)
    # The whole workload if the host cores manage it within the budget (N = 999 999, P = 200: ~0.7 s per step on 16
    # threads), else a prefix of the atoms (the cost is linear in atoms): sized from a probe on 20 000 atoms.
    n_probe = min(20_000, cfg0.N)
    t_probe, _, _, _, _ = time_oracle(args.config, n_probe, 1, 1)
    budget_s = 150.0
    n_fit = int(budget_s / ((steps + warmup) * max(t_probe / n_probe, 1e-12)))
    n_sample = cfg0.N if args.ref_atoms <= 0 else min(args.ref_atoms, cfg0.N)
    n_sample = max(min(n_sample, n_fit), min(1000, cfg0.N))
    per_step, ns_atom, cores, cfg, _ = time_oracle(args.config, n_sample, steps, warmup)
    what = "all" if n_sample == cfg.N else "first"
    sample = f"{what} {n_sample} atoms of {cfg.name} (N={cfg.N}), all P={cfg.P} wavevectors, oracle.rho + oracle.force"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": ns_atom, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": per_step * 1e3, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same keys the GPU arm prints for the workload (one rank runs the oracle: N_total = N_per_gpu = the config's N)
        "config": {"workload": cfg.name, "N_per_gpu": cfg.N, "N_total": cfg.N, "P": cfg.P, "L": cfg.L, "alpha": cfg.alpha,
                   "sample_atoms": n_sample},
        "cpu_baseline": {"value": ns_atom, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ns_atom, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", default="water_nacl_1m")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-atoms", type=int, default=0, help="--impl reference: atoms per oracle step (0 = the whole workload, "
                    "cut down only if the host cores cannot finish it within ~150 s)")
    ap.add_argument("--no-md", action="store_true")
    ap.add_argument("--cpu-baseline-atoms", type=int, default=1_000_000)
    ap.add_argument("--cpu-baseline-steps", type=int, default=15)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--no-short-range", action="store_true")
    ap.add_argument("--rs", type=float, default=10.0, help="cutoff radius of the real-space partner leg [A]")
    ap.add_argument("--exchange", default="fused", choices=["fused", "nccl"],
                    help="N > 1: how the structure factors are summed across ranks")
    ap.add_argument("--with-energy", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(3, args.warmup)

    import torch
    import torch.distributed as dist
    from paper_2407_09315_b200 import inputs, rbe

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the RBE path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    base = workload_config(args.config, world)
    # weak scaling: every rank owns base.N atoms of a box `world` times larger, same density
    L = base.L * world ** (1.0 / 3.0)
    n_local, n_total, P, alpha = base.N, base.N * world, base.P, base.alpha
    cfg_r = inputs.Config(base.name, base.N, base.L, base.P, base.seed + 1000 * rank, base.kind,
                          base.n_water, base.n_ion_pairs, base.alpha)
    atoms = inputs.make_atoms(cfg_r)
    if world > 1:
        atoms[:, :3] *= np.float32(L / base.L)  # spread the shard over the larger box

    ctx = rbe.Rbe(n_local, L, alpha, P)
    info = ctx.rbe_get_launch_info()
    # N > 1: the P complex structure factors are exchanged INSIDE the kernels over NVLink peer
    # memory (rbe_set_exchange); NCCL all_gather + rbe_set_rho only if symmetric memory is unavailable
    fused = False
    if world > 1 and args.exchange == "fused":
        ok = torch.ones(1, device="cuda")
        try:
            from paper_2407_09315_b200 import exchange
            exchange.setup_fused_exchange(ctx)
        except Exception as e:  # noqa: BLE001 - any failure here means "no peer mapping": use NCCL
            ok.zero_()
            if rank == 0:
                print(f"bench: fused exchange unavailable ({type(e).__name__}: {e}); using NCCL all_gather", file=sys.stderr)
        dist.all_reduce(ok, op=dist.ReduceOp.MIN)
        fused = bool(ok.item() > 0)
        if not fused:
            ctx.rbe_set_exchange(0, 0, None, 0)
    # inputs larger than L2: rotate over enough {xyzq, force} buffer pairs to exceed 126 MB
    n_rot = max(2, int(np.ceil(160e6 / max(1, 32 * n_local))))
    n_rot = min(n_rot, 64)
    xs = [torch.from_numpy(atoms).cuda() for _ in range(n_rot)]
    fs = [torch.empty((n_local, 4), dtype=torch.float32, device="cuda") for _ in range(n_rot)]
    n_k = args.warmup + args.steps
    ksets = [np.ascontiguousarray(inputs.sample_kset(L, alpha, P, base.seed, t), dtype=np.int32) for t in range(n_k)]
    rho_local = torch.empty((P, 2), dtype=torch.float64, device="cuda")
    gathered = torch.empty((world, P, 2), dtype=torch.float64, device="cuda") if world > 1 else None

    one_launch = world == 1 and bool(info["step_fused"])

    def step_two(i, ev=None):
        x, f = xs[i % n_rot], fs[i % n_rot]
        ctx.rbe_set_kvectors(ksets[i % n_k])
        if ev: ev[0].record()
        ctx.rbe_structure_factor(x, rho_local if world > 1 and not fused else None)
        if world > 1 and not fused:
            dist.all_gather_into_tensor(gathered, rho_local)
            ctx.rbe_set_rho(gathered.sum(0))  # fixed (rank) order
        if ev: ev[1].record()
        ctx.rbe_forces(x, f, args.with_energy)
        if ev: ev[2].record()

    # rbe_step with the tensors marshalled once per buffer set (the per-step host cost matters for the small configs)
    bound = [ctx.rbe_step_bound(xs[r], fs[r], with_energy=args.with_energy) for r in range(n_rot)] if world == 1 else None

    def step(i, ev=None):
        if world > 1:
            return step_two(i, ev)
        bound[i % n_rot](ksets[i % n_k])          # one launch (or two: large systems)

    # N > 1: before anything is timed, one step through the fused exchange is checked against the NCCL sum
    # (a mis-synchronised peer exchange that still arrives in time would otherwise give a timing line and no error)
    exchange_used = "none" if world == 1 else ("fused" if fused else "nccl")
    if fused:
        ref = rbe.Rbe(n_local, L, alpha, P)
        ref.rbe_set_kvectors(ksets[0])
        ref.rbe_structure_factor(xs[0], rho_local)
        dist.all_gather_into_tensor(gathered, rho_local)
        ref.rbe_set_rho(gathered.sum(0))
        u_ref = ref.rbe_kspace_energy()
        step_two(0)
        u_fused = ctx.rbe_kspace_energy()
        ctx.rbe_exchange_check()
        bad = torch.tensor([0.0 if u_fused == u_ref else 1.0], device="cuda")     # rank-ordered sums: bitwise equal
        dist.all_reduce(bad, op=dist.ReduceOp.MAX)
        if bad.item() > 0:
            if rank == 0:
                print(f"bench: fused exchange disagrees with the NCCL sum ({u_fused!r} vs {u_ref!r}); using NCCL", file=sys.stderr)
            ctx.rbe_set_exchange(0, 0, None, 0)
            fused = False
            exchange_used = "nccl (fused exchange failed its cross-check)"
        del ref

    def sync():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        step(i)
    sync()

    # ---- timed region A: exactly K steps, device-timed, nothing else on the stream
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    sync()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # one more UNTIMED step goes out right before the first event: the GPU has been idle since the synchronise (and the
    # sampler's start-up sleep), and without it the host-side latency of issuing the first timed step lands inside the
    # region (~100 us: 5 us per step of a 20-step run, 0.5 us of a 200-step run); with it the K timed steps run back to back
    step(args.warmup - 1)
    e0.record()
    for i in range(args.steps):
        step(args.warmup + i)
    e1.record()
    sync()
    ms_total = e0.elapsed_time(e1)
    # the forces the LAST timed step left in its buffer, for parity_in_run (compared with the oracle in the cpu_baseline leg)
    i_last = args.warmup + args.steps - 1
    F_last = fs[i_last % n_rot].cpu().numpy() if world == 1 else None
    rho_last, rerun_equal = None, None
    if world == 1:
        # the same step once more, untimed, into fresh buffers and with the structure factors returned: it must
        # reproduce the timed step's forces bit for bit (a timed step that skipped work would not)
        f_chk = torch.full((n_local, 4), float("nan"), dtype=torch.float32, device="cuda")
        rho_chk = torch.full((P, 2), float("nan"), dtype=torch.float64, device="cuda")
        ctx.rbe_step(ksets[i_last % n_k], xs[i_last % n_rot], f_chk, with_energy=args.with_energy, rho=rho_chk)
        sync()
        rerun_equal = bool(np.array_equal(f_chk.cpu().numpy(), F_last))
        rho_last = rho_chk.cpu().numpy()
        del f_chk, rho_chk

    # ---- region A2: the same K steps with CUDA events around every step, for the median and the minimum;
    # the headline stays region A's mean, which carries no per-step event
    evs_a = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    for i in range(args.steps):
        evs_a[i][0].record()
        step(args.warmup + i)
        evs_a[i][1].record()
    sync()
    t_step = sorted(e[0].elapsed_time(e[1]) for e in evs_a)

    # ---- region A3: the same K steps with the charge pairing of the structure-factor phase switched off
    # (rbe_set_pairing(0)): what a system whose atoms all carry different |q| would see -- 2 special-function
    # evaluations per pair there instead of the 1.5 that water's equal charges allow
    ms_unpaired = None
    if world == 1:
        ctx.rbe_set_pairing(0)
        for i in range(3):
            step(i)
        sync()
        e0.record()
        for i in range(args.steps):
            step(args.warmup + i)
        e1.record()
        sync()
        ms_unpaired = e0.elapsed_time(e1) / args.steps
        ctx.rbe_set_pairing(3)

    # ---- region A4: the same K steps through rbe_step_static (scratch in the library's own static device array: for callers
    # that cannot allocate; one 8-byte memset + the same kernel per step)
    ms_static = None
    if world == 1 and one_launch and P <= 512:
        sctx = rbe.Rbe(n_local, L, alpha, P, allocate=False)
        for i in range(3):
            sctx.rbe_step_static(ksets[i % n_k], xs[i % n_rot], fs[i % n_rot], with_energy=args.with_energy)
        sync()
        e0.record()
        for i in range(args.steps):
            j = args.warmup + i
            sctx.rbe_step_static(ksets[j % n_k], xs[j % n_rot], fs[j % n_rot], with_energy=args.with_energy)
        e1.record()
        sync()
        ms_static = e0.elapsed_time(e1) / args.steps
        if F_last is not None and not np.array_equal(fs[i_last % n_rot].cpu().numpy(), F_last):
            raise SystemExit("bench: rbe_step_static did not reproduce rbe_step's forces bit for bit")
        del sctx

    # ---- timed region B: the same K steps in the two-launch form with CUDA events around each call, for the
    # per-kernel durations of sf_kernel and f_kernel
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    for i in range(3):
        step_two(i)
    sync()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record()
    for i in range(args.steps):
        step_two(args.warmup + i, evs[i])
    e3.record()
    sync()
    ms_two = e2.elapsed_time(e3) / args.steps
    clocks = sampler.stop() if rank == 0 else None
    # issue rates of the pipes that bound the path, measured now on this device (rbe_probe_pipe_rates)
    pipe = ctx.rbe_probe_pipe_rates() if rank == 0 else None
    if fused:
        ctx.rbe_exchange_check()   # raises if any kernel gave up waiting for a peer
    t_sf = [e[0].elapsed_time(e[1]) for e in evs]
    t_f = [e[1].elapsed_time(e[2]) for e in evs]
    ms_sf, ms_f = sum(t_sf) / len(t_sf), sum(t_f) / len(t_f)

    # ---- the same K steps as ONE graph launch each: device sampler + SF + F,
    # no per-step host-to-device traffic; one context + graph per buffer set, so the inputs still rotate
    ms_graph = None
    if world == 1 and not args.no_graph:
        gctx = []
        for r in range(n_rot):
            g = rbe.Rbe(n_local, L, alpha, P)
            g.rbe_graph_capture(xs[r], fs[r], args.with_energy, base.seed, 1_000_000 * r)
            gctx.append(g)
        for i in range(args.warmup):
            gctx[i % n_rot].rbe_graph_launch()
        sync()
        e0.record()
        for i in range(args.steps):
            gctx[i % n_rot].rbe_graph_launch()
        e1.record()
        sync()
        ms_graph = e0.elapsed_time(e1) / args.steps
        del gctx

    # ---- real-space partner: Eq. 2.10 truncated at r_s = 10 A on the same atoms
    sr = None
    if world == 1 and not args.no_short_range and L >= 3 * args.rs:
        k_sr = max(3, min(args.steps, 20))
        for i in range(3):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        sync()
        e0.record()
        for i in range(k_sr):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        e1.record()
        sync()
        ms_sr = e0.elapsed_time(e1) / k_sr
        # the same sum with the paper's tabulated pair term instead of the polynomial erfc (rbe_set_pair_table)
        ctx.rbe_set_pair_table(True)
        for i in range(2):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        sync()
        e0.record()
        for i in range(k_sr):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        e1.record()
        sync()
        ms_sr_tab = e0.elapsed_time(e1) / k_sr
        ctx.rbe_set_pair_table(False)
        # ... and with the second force kernel (rbe_set_pair_kernel(1): fine cells, tensor-core cutoff test, ordered pairs)
        ctx.rbe_set_pair_kernel(1)
        for i in range(2):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        sync()
        e0.record()
        for i in range(k_sr):
            ctx.rbe_short_range(xs[i % n_rot], args.rs, fs[i % n_rot])
        e1.record()
        sync()
        ms_sr_cells = e0.elapsed_time(e1) / k_sr
        ctx.rbe_set_pair_kernel(0)
        # the paper's own estimator of the same force: random batch list, r_c = r_s / 2, p = 30
        for i in range(2):
            ctx.rbe_rbl_forces(xs[i % n_rot], args.rs / 2, args.rs, 30, base.seed, i, fs[i % n_rot])
        sync()
        e0.record()
        for i in range(3):
            ctx.rbe_rbl_forces(xs[i % n_rot], args.rs / 2, args.rs, 30, base.seed, 2 + i, fs[i % n_rot])
        e1.record()
        sync()
        ms_rbl = e0.elapsed_time(e1) / 3
        nbr = 4.0 / 3.0 * np.pi * args.rs ** 3 * n_local / L ** 3          # expected atoms inside the cutoff sphere
        sr = {"ms_per_call": ms_sr, "value": ms_sr * 1e6 / n_local, "unit": UNIT.replace("/step", "/call"),
              "r_s": args.rs, "neighbours_per_atom_expected": nbr, "calls": k_sr, "gpu_launches_per_call": 7,
              "pair_rate_G_per_s": nbr * n_local / (ms_sr * 1e-3) / 1e9,
              "pair_table": {"ms_per_call": ms_sr_tab, "note": "rbe_set_pair_table(1): tabulated pair term with cubic interpolation "
                             "(P:196) instead of the degree-8 polynomial erfc; one more launch (the table is rebuilt per call)"},
              "pair_kernel_cells": {"ms_per_call": ms_sr_cells, "note": "rbe_set_pair_kernel(1): one CTA per cell of side r_s / 2, cutoff test as a TF32 "
                                    "mma on the tensor cores, every ordered pair evaluated by one lane, no atomics"},
              "rbl": {"ms_per_call": ms_rbl, "r_c": args.rs / 2, "p": 30,
                      "note": "rbe_rbl_forces (Eqs. 2.13-2.16): cells of side r_c, warp per atom, parity-exact batch; still slower "
                              "than the deterministic sum on B200 (instruction budget: profiles/r02_rbl_README.md)"},
              "note": "rbe_short_range: bin + scan + scatter + sort + group boxes + pair kernel (every unordered pair "
                      "once, fixed-point integer atomics across warps) + finalise; not part of `value`"}

    # ---- one whole MD step (velocity Verlet P:78, NVE P:86): rbe_md_capture's graph -- kick +
    # drift, device sampler, k-space step, rbe_short_range (accumulate), kick -- replayed on ~1e6 ions at the
    # workload's density
    md = None
    if world == 1 and not args.no_md:
        cells = max(2, int(round((n_local / 2.0) ** (1.0 / 3.0))))
        a_cell = (2.0 / inputs.DENSITY) ** (1.0 / 3.0)                     # bcc cell side for 0.1 ions per A^3
        x_m, v_m, q_m, mass_m, L_m = inputs.plasma(cells, a=a_cell, seed=11, jitter=0.05, v_rms=0.04)
        n_m = x_m.shape[0]
        if L_m >= 3 * args.rs:
            mctx = rbe.Rbe(n_m, L_m, alpha, P)
            pos_m = torch.from_numpy(x_m).cuda()
            vel_m = torch.from_numpy(v_m).cuda()
            inv_m = torch.from_numpy(1.0 / mass_m).cuda()
            xyzq_m = torch.from_numpy(np.concatenate([x_m.astype(np.float32), q_m[:, None]], axis=1)).cuda().contiguous()
            force_m = torch.zeros((n_m, 4), dtype=torch.float32, device="cuda")
            mctx.rbe_sample_kvectors(base.seed, 0)
            mctx.rbe_step(None, xyzq_m, force_m)
            mctx.rbe_short_range(xyzq_m, args.rs, force_m, accumulate=True)
            mctx.rbe_md_capture(pos_m, vel_m, inv_m, xyzq_m, force_m, args.rs, 0.2, sampled=True, seed=base.seed, first_step=1)
            k_md = max(3, min(args.steps, 20))
            for i in range(3):
                mctx.rbe_graph_launch()
            sync()
            e0.record()
            for i in range(k_md):
                mctx.rbe_graph_launch()
            e1.record()
            sync()
            ms_md = e0.elapsed_time(e1) / k_md
            finite = bool(torch.isfinite(pos_m).all().item() and torch.isfinite(force_m).all().item())
            k_launch = 2 if bool(mctx.rbe_get_launch_info()["step_fused"]) else 3      # sampler + step (or + sf + f)
            md = {"ms_per_step": ms_md, "value": ms_md * 1e6 / n_m, "unit": UNIT, "N": n_m, "L": L_m, "r_s": args.rs, "dt_tau": 0.2,
                  "steps": k_md, "graph_launches_per_step": 1, "kernels_per_step": 2 + k_launch + 7, "memsets_per_step": 2,
                  "finite": finite,
                  "note": "rbe_md_capture replayed by rbe_graph_launch: kick+drift, sample_kernel, k-space step, rbe_short_range "
                          "(7 kernels, 2 memsets, accumulate), kick; one-component plasma (bcc, +1 e, implied background) at 0.1 ions/A^3, "
                          "positions and velocities fp64 resident on the device; not part of `value`"}
            del mctx, pos_m, vel_m, inv_m, xyzq_m, force_m

    if world > 1:
        t = torch.tensor([ms_total, ms_sf, ms_f, ms_two], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total, ms_sf, ms_f, ms_two = [float(v) for v in t.cpu()]
    ms_step = ms_total / args.steps
    value = ms_step * 1e6 / n_total            # whole job: all atoms of all ranks per step time

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        # page-locked host buffers from the library (rbe_host_alloc = cudaHostAlloc): on these hosts
        # H2D from memory pinned after allocation (torch pin_memory) is 2-4x slower and erratic
        hx_np = rbe.rbe_host_alloc((n_local, 4), np.float32)
        hf_np = rbe.rbe_host_alloc((n_local, 4), np.float32)
        hx_np[:] = atoms
        hx, hf = torch.from_numpy(hx_np), torch.from_numpy(hf_np)
        k_e2e = max(3, min(args.steps, 20))
        ms_e2e4 = None
        if world == 1:
            def time_host(fn):
                for i in range(3):
                    fn(i)
                sync()
                e0.record()
                for i in range(k_e2e):
                    fn(i)
                e1.record()
                sync()
                return e0.elapsed_time(e1) / k_e2e
            # float4 {x,y,z,q} in / float4 {F,e} out: 32 B per atom over PCIe
            ms_e2e4 = time_host(lambda i: ctx.rbe_step_host(hx, ksets[i % n_k], hf, with_energy=args.with_energy))
            # the MD-loop form: charges resident on the device, positions in / force vectors out: 24 B per atom
            hx3_np = rbe.rbe_host_alloc((n_local, 3), np.float32)
            hf3_np = rbe.rbe_host_alloc((n_local, 3), np.float32)
            hx3_np[:] = atoms[:, :3]
            ctx.rbe_set_charges(torch.from_numpy(atoms[:, 3].copy()).cuda())
            ms_e2e = time_host(lambda i: ctx.rbe_step_host_xyz(hx3_np, ksets[i % n_k], hf3_np))
        else:
            dx = torch.empty((n_local, 4), dtype=torch.float32, device="cuda")
            df = torch.empty((n_local, 4), dtype=torch.float32, device="cuda")

            def e2e_step(i):
                dx.copy_(hx, non_blocking=True)
                ctx.rbe_set_kvectors(ksets[i % n_k])
                ctx.rbe_structure_factor(dx, None if fused else rho_local)
                if not fused:
                    dist.all_gather_into_tensor(gathered, rho_local)
                    ctx.rbe_set_rho(gathered.sum(0))
                ctx.rbe_forces(dx, df, args.with_energy)
                hf.copy_(df, non_blocking=True)
                torch.cuda.current_stream().synchronize()
            for i in range(3):
                e2e_step(i)
            sync()
            e0.record()
            for i in range(k_e2e):
                e2e_step(i)
            e1.record()
            sync()
            t = torch.tensor([e0.elapsed_time(e1) / k_e2e], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_e2e = float(t.cpu()[0])
        compact = world == 1
        e2e = {"value": ms_e2e * 1e6 / n_total, "unit": UNIT, "ms_per_step": ms_e2e, "steps": k_e2e,
               "h2d_bytes_per_step": (12 if compact else 16) * n_local + 16 * P,
               "d2h_bytes_per_step": (12 if compact else 16) * n_local,
               "path": "rbe_step_host_xyz: pinned host positions float3[N] in -> forces float3[N] out (charges resident on "
                       "the device), copies chunked (<= 4) and overlapped with the kernels" if compact else
                       "H2D + rbe_* calls + exchange + D2H per rank",
               "float4_ms_per_step": ms_e2e4}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = read_peaks()
    tr, sfu_rate_nominal = roofline_times(n_local, P, info["num_sms"], peaks)
    t_roof = max(tr.values())
    pairs = n_local * P
    clk = peaks["sm_max_mhz"] * 1e6
    sms = info["num_sms"]
    # peaks: MEASURED lanes per SM per clock (this run) x SMs x the max SM clock
    mufu_rate = pipe["mufu"] * sms * clk
    issue_rate = 4 * sms * clk                     # warp instructions per second: 4 schedulers per SM, 1 per clock

    def roof(kernel, ms, alg_per_pair, exe_per_pair):
        """alu roofline of one kernel: algorithmic special-function evaluations (2 per pair per
        phase) against the measured MUFU rate; beside it what the kernel executes, and its issue bound."""
        cnt = read_counters(kernel, args.config)
        t = ms * 1e-3
        r = {"bound": "alu", "kernel": kernel, "achieved": alg_per_pair * pairs / t / 1e9, "peak": mufu_rate / 1e9,
             "unit": "G sincos-evaluation/s, ALGORITHMIC count (2 per pair per phase) against the measured MUFU rate",
             "frac": alg_per_pair * pairs / t / mufu_rate,
             "frac_is": "algorithmic work / measured peak (SURVEY.md s8(d)'s count, as the measurement contract defines it): a speed-of-"
                        "light ratio that can pass 1 because the kernels EXECUTE fewer special-function instructions than the 4 per "
                        "pair it counts; the pipe utilisation is executed.frac_of_mufu_peak / frac_of_xu_peak / frac_of_issue_bound",
             "executed": {"mufu_per_pair": exe_per_pair, "frac_of_mufu_peak": exe_per_pair * pairs / t / mufu_rate},
             "traffic": None if cnt is None else cnt["dram_bytes"],
             "peak_source": f"measured in this run: {pipe['mufu']:.2f} MUFU lanes/SM/clk (rbe_probe_pipe_rates) x {sms} SMs x "
                            f"{peaks['sm_max_mhz']:.0f} MHz"}
        if cnt is not None:
            t_issue = cnt["inst_executed"] / issue_rate
            r["executed"].update(warp_instructions=cnt["inst_executed"], issue_bound_us=t_issue * 1e6, frac_of_issue_bound=t_issue / t,
                                 counters=cnt["capture"], counters_stale=cnt["stale"])
            if cnt["inst_executed_pipe_xu"] is not None:
                # COUNTED, not assumed: warp instructions the XU pipe executed in one launch (sm__inst_executed_pipe_xu.sum:
                # MUFU plus whatever conversions share the pipe), 32 lanes each
                xu = cnt["inst_executed_pipe_xu"] * 32.0
                r["executed"].update(xu_warp_instructions=cnt["inst_executed_pipe_xu"], xu_per_pair=xu / pairs,
                                     frac_of_xu_peak=xu / t / mufu_rate,
                                     mufu_per_pair_source="design count (DESIGN.md section 5); xu_per_pair is the ncu count")
        return r

    main_kernel = "step_kernel" if one_launch else "sf_kernel"
    main_ms = ms_step if one_launch else ms_sf
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": base.name, "N_per_gpu": n_local, "N_total": n_total, "P": P, "L": L, "alpha": alpha,
                   "l2": f"inputs rotate over {n_rot} buffer sets ({32 * n_local * n_rot / 1e6:.0f} MB > 126 MB L2)",
                   "parallelism": f"atoms sharded over {world} GPU(s), k-set replicated" + (
                       "" if world == 1 else ", rho exchanged inside the kernels over NVLink peer memory (rbe_set_exchange)"
                       if fused else ", rho exchanged with NCCL all_gather + rank-ordered sum"),
                   "exchange": exchange_used,
                   "step": "rbe_step: one cooperative launch (step_kernel)" if one_launch else
                           "rbe_set_kvectors + rbe_structure_factor + rbe_forces: two launches",
                   "launch": info, "with_energy": bool(args.with_energy)},
        "kernels_ms": {"step_call": ms_step, "step_call_median": t_step[len(t_step) // 2], "step_call_min": t_step[0],
                       "two_launch_step": ms_two, "structure_factor_call": ms_sf, "forces_call": ms_f,
                       "structure_factor_call_median": statistics.median(t_sf), "structure_factor_call_min": min(t_sf),
                       "forces_call_median": statistics.median(t_f), "forces_call_min": min(t_f),
                       "note": "step_call = region A (rbe_step; _median / _min: region A2, per-step events); the rest = region B, the two-launch form with CUDA events around "
                               "each C-ABI call: structure_factor_call = sf_kernel (incl. its in-kernel second pass), forces_call = f_kernel"},
        "peaks": {"lanes_per_sm_per_clk": {k: pipe[k] for k in ("ffma", "imad", "i2fp", "mufu")},
                  "sm_mhz_during_probe": pipe["sm_mhz"], "sm_max_mhz": peaks["sm_max_mhz"], "hbm_gbs": peaks["hbm_gbs"],
                  "hbm_source": peaks["src"] + " (MEASURED_PEAKS.json)" if peaks["src"] == "measured" else peaks["src"],
                  "how": "rbe_probe_pipe_rates: dependent-free chains, 32 warps per SM, in-kernel clock64, in this run"},
        "roofline": roof(main_kernel, main_ms, 2 * SFU_PER_PAIR_PER_KERNEL if one_launch else SFU_PER_PAIR_PER_KERNEL,
                         MUFU_EXECUTED_PER_PAIR["sf"] + (MUFU_EXECUTED_PER_PAIR["f"] if one_launch else 0.0)),
        "roofline_kernels": [roof("sf_kernel", ms_sf, SFU_PER_PAIR_PER_KERNEL, MUFU_EXECUTED_PER_PAIR["sf"]),
                             roof("f_kernel", ms_f, SFU_PER_PAIR_PER_KERNEL, MUFU_EXECUTED_PER_PAIR["f"])],
        "roofline_step": {
            "t_roof_us": t_roof * 1e6, "t_hbm_us": tr["hbm"] * 1e6, "t_fma_us": tr["fma"] * 1e6, "t_sfu_us": tr["sfu"] * 1e6,
            "frac": t_roof / (ms_step * 1e-3), "ns_per_atom_at_roofline": t_roof * 1e9 / n_local,
            "hbm_peak_gbs": peaks["hbm_gbs"], "peaks": peaks["src"],
            "note": "SURVEY.md s8(d): 4 sincos + 13 FMA per (atom,k) pair per step, 48 B per atom, at the NOMINAL 16 MUFU / 128 FP32 "
                    "lanes per SM per clock (the survey's figures; `roofline` uses the rates measured in this run)",
        },
        "graph_step": None if ms_graph is None else {
            "ms_per_step": ms_graph, "value": ms_graph * 1e6 / n_total, "unit": UNIT, "gpu_launches_per_step": 2 if one_launch else 3,
            "note": "rbe_graph_launch: device sampler (Philox) + the k-space step replayed as one CUDA graph, "
                    "no per-step H2D; not the headline (the k-set there comes from the host each step)"},
        "static_step": None if ms_static is None else {
            "ms_per_step": ms_static, "value": ms_static * 1e6 / n_total, "unit": UNIT, "gpu_launches_per_step": 1, "memsets_per_step": 1,
            "note": "rbe_step_static: the same kernel with its scratch in a 1.5 MiB static __device__ array of librbe.so (no workspace, "
                    "no allocation anywhere on the path; P <= 512); forces checked bit-identical to rbe_step's in this run"},
        "short_range": sr,
        "md_step": md,
        "clocks": clocks,
        "gpu_launches": (1 if one_launch else 2) * args.steps,
        "paper_context": "8.20 ms/step, 1e6 atoms, A100, RBL+RBE nonbonded total, P=100 (PAPER.md P:284); 2.89 ms k-space at 1e5 atoms, P=200 (P:266)",
    }
    if ms_unpaired is not None:
        out["roofline"]["unpaired"] = {
            "ms_per_step": ms_unpaired, "value": ms_unpaired * 1e6 / n_total,
            "frac": 2 * SFU_PER_PAIR_PER_KERNEL * pairs / (ms_unpaired * 1e-3) / mufu_rate,   # of the whole step (both phases)
            "executed_mufu_per_pair": 2.0 + MUFU_EXECUTED_PER_PAIR["f"],
            "note": "the timed steps again with rbe_set_pairing(0): no two atoms share a special-function evaluation in the structure-"
                    "factor phase -- the figure a system with all-distinct |q| would see; `frac` as roofline.frac (algorithmic count)"}
    if e2e:
        out["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        n_s = min(args.cpu_baseline_atoms, base.N)
        k_cpu = max(1, args.cpu_baseline_steps)
        per_step, ns_cpu, cores, _, keep = time_oracle(args.config, n_s, k_cpu, 1, last_kset=i_last % n_k)
        # parity inside this run: the oracle's last timed step used the k-set of the GPU's last timed step, so its
        # output doubles as the check that the timed region did the work (no extra oracle time is spent)
        if n_s == base.N and F_last is not None:
            _, rho_o, F_o = keep
            qsum = float(np.abs(atoms[:, 3].astype(np.float64)).sum())
            d_f = F_last[:, :3].astype(np.float64) - F_o
            parity = {"F_relL2": float(np.linalg.norm(d_f) / np.linalg.norm(F_o)),
                      "rho_err": float(np.abs(rho_last - rho_o).max() / qsum),
                      "tolerance": {"F_relL2": 2e-5, "rho_err": 1e-6}, "atoms": int(n_s), "kset_step": int(i_last % n_k),
                      "timed_step_reproduced_bitwise": rerun_equal,
                      "what": "forces left by the LAST timed step (all 3N components) and rho of the same step re-run, against "
                              "oracle.rho / oracle.force on the same atoms and k-set (the cpu_baseline leg's last step)"}
            parity["passed"] = bool(parity["F_relL2"] <= 2e-5 and parity["rho_err"] <= 1e-6 and rerun_equal)
            out["parity_in_run"] = parity
        else:
            out["parity_in_run"] = {"passed": None, "timed_step_reproduced_bitwise": rerun_equal,
                                    "what": "the cpu_baseline sample is smaller than the workload: no oracle comparison in this run"}
        # the same oracle on ONE thread, on a sample sized for ~5 s: a bare core count would mislead
        n_1 = max(1000, min(n_s, 25_000))
        per_step1, ns_cpu1, _, _, _ = time_oracle(args.config, n_1, 1, 1, threads=1)
        out["cpu_baseline"] = {"value": ns_cpu, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "one_thread": {"value": ns_cpu1, "unit": UNIT, "sample_atoms": n_1},
                               "speedup_all_threads_vs_one": ns_cpu1 / ns_cpu,
                               "sample": f"first {n_s} atoms of {base.name} (N={base.N}), all P={P} wavevectors, oracle.rho + "
                                         f"oracle.force, {k_cpu} steps after 1 warm-up ({per_step * k_cpu:.1f} s of CPU work)"}
    if "parity_in_run" not in out:
        out["parity_in_run"] = {"passed": None, "timed_step_reproduced_bitwise": rerun_equal, "what": "no cpu_baseline leg in this run"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    if out["parity_in_run"]["passed"] is False or rerun_equal is False:
        print("bench: the timed step's output FAILED its in-run check: " + json.dumps(out["parity_in_run"]), file=sys.stderr)
        raise SystemExit(1)


if __name__ == "__main__":
    main()
