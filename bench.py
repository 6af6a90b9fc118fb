#!/usr/bin/env python
"""bench.py -- accepted electron moves/s of the delayed rank-K Slater-inverse update
(arXiv 1708.00744) on B200, through the C-ABI library (include/qmcd.h).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--config c1] [--K 32] [--mode bern0.99]

One "step" = one pass of the whole hot path over one batch of synthetic input:
adopt the inverse (F0), run every proposal of the config through ratio (F1) ->
accept/reject (F2) -> flush when K moves are queued (F3), and the final partial
flush (F5).  The default workload is BASELINE.json configs[1] (c1: 16 walkers,
N = 512, 4 sweeps, Bernoulli(0.99)).  Prints ONE JSON line (rank 0).

N > 1 GPUs: walkers are independent, so every rank runs its own
batch (per-rank seeds) with no data-path collective -> "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "accepted electron moves/s (fp64, batched walkers)"
UNIT = "moves/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c1")
    ap.add_argument("--K", type=int, default=32)
    ap.add_argument("--mode", default="bern0.99")
    ap.add_argument("--cluster", type=int, default=0, help="CTAs per walker (0 = library default)")
    ap.add_argument("--flush-path", type=int, default=0, help="0 auto, 1 CUDA-core, 2 DMMA")
    ap.add_argument("--opt", action="append", default=[], help="library option key=value (qmcd_set_option)")
    ap.add_argument("--N", type=int, default=0, help="with --config custom: matrix order")
    ap.add_argument("--batch", type=int, default=1, help="with --config custom: walkers")
    ap.add_argument("--sweeps", type=int, default=1, help="with --config custom: sweeps over the electrons")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--phases", action="store_true",
                    help="also time the ratio and flush kernels in isolation (per-call API)")
    return ap.parse_args()


def get_config(args):
    """BASELINE.json config c0..c4, or a custom shape (the paper's own grid, PAPER.md:103-113:
    one walker, N = 256 ... 8192, 100 % acceptance = --mode bern1.0)."""
    from paper_1708_00744_b200 import inputs
    if args.config == "custom":
        if args.N < 1:
            raise SystemExit("--config custom needs --N")
        return dict(batch=args.batch, N=args.N, sweeps=args.sweeps, Ks=(args.K,), modes=(args.mode,), seed=1)
    return inputs.CONFIGS[args.config]


def mode_inputs(wl, mode):
    """-> (mask or None, uniforms or None)"""
    if mode.startswith("bern"):
        return wl.bernoulli_mask(float(mode[4:])), None
    if mode == "metropolis":
        return None, wl.uniforms
    raise SystemExit(f"unknown mode {mode}")


def config_dict(args, cfg, wl, extra=None):
    d = {"workload": f"{args.config}: batch {wl.batch} walkers/GPU, N={wl.N}, {cfg['sweeps']} sweeps "
                     f"({wl.n_moves} proposals/walker), {args.mode}, delay K={args.K}",
         "config": args.config, "batch_per_gpu": wl.batch, "N": wl.N, "K": args.K,
         "proposals_per_walker": wl.n_moves, "acceptance": args.mode,
         "l2": "inputs per step (proposals + inverse + pristine copy) exceed the 126 MB L2"
               if (wl.proposals.nbytes + 2 * wl.Ainv.nbytes) > 126e6 else
               "L2 flushed between steps by writing a 256 MB buffer"}
    if extra:
        d.update(extra)
    return d


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for nm, val in zip(names, c[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            # "under load": samples in the upper half of what was seen
            hi = [x for x in sm if x >= 0.5 * max(sm)]
            out["sm_mhz"] = float(np.median(hi))
            out["sm_max_mhz"] = float(max(mx))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


# ----------------------------------------------------------------------------- accounting
def algorithmic_work(acc, N, K, lockstep=False):
    """Algorithmic flops / bytes of one step from the accept sequence acc [n_moves][batch]
    (SURVEY.md 8(d) / DESIGN.md 'Kernels'): F1 per proposal at queue length m:
    2N(2m+1)+2m^2 flops, 8N(2m+2)+8m^2 bytes; F2 per accept 4m^2 flops; F3 per rank-m
    flush 4N^2 m + 2 m^2 N flops, 16N^2 + 24mN bytes (final partial flush included).
    lockstep: the window closes after every K-th PROPOSAL with the rank m
    accepted in it; a rejected slot is a zero column of U and counts no work."""
    n_moves, batch = acc.shape
    f1f = f1b = f2f = f3f = f3b = 0.0
    flushes = 0
    for w in range(batch):
        m = 0
        a = acc[:, w]
        for t in range(n_moves):
            f1f += 2.0 * N * (2 * m + 1) + 2.0 * m * m
            f1b += 8.0 * N * (2 * m + 2) + 8.0 * m * m
            if a[t]:
                f2f += 4.0 * m * m
                m += 1
            if (m > 0 and (t + 1) % K == 0) if lockstep else (m == K):
                f3f += 4.0 * N * N * m + 2.0 * m * m * N
                f3b += 16.0 * N * N + 24.0 * m * N
                flushes += 1
                m = 0
        if m > 0:
            f3f += 4.0 * N * N * m + 2.0 * m * m * N
            f3b += 16.0 * N * N + 24.0 * m * N
            flushes += 1
    return dict(ratio_flops=f1f, ratio_bytes=f1b, accept_flops=f2f, flush_flops=f3f,
                flush_bytes=f3b, flushes=flushes, flops=f1f + f2f + f3f, bytes=f1b + f3b)


# ----------------------------------------------------------------------------- reference arm
def oracle_step(oracle, wl, K, mask, uniforms):
    B = wl.Ainv.copy()
    t0 = time.perf_counter()
    R, acc, thr = oracle.run(2, B, K, wl.proposals, mask=mask, uniforms=uniforms, final_flush=True)
    return time.perf_counter() - t0, acc, thr


def run_reference(args):
    """--impl reference: the CPU oracle as it stands (delayed rank-K path), timed on the host
    cores on the same config.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_1708_00744_b200 import inputs
    cfg = get_config(args)
    wl = inputs.make_workload(cfg["batch"], cfg["N"], cfg["sweeps"] * cfg["N"], seed=cfg["seed"])
    mask, uniforms = mode_inputs(wl, args.mode)
    for _ in range(min(args.warmup, 1)):
        oracle_step(oracle, wl, args.K, mask, uniforms)
    ts, accepted, thr = [], 0, 0
    for _ in range(args.steps):
        dt, acc, thr = oracle_step(oracle, wl, args.K, mask, uniforms)
        ts.append(dt); accepted = int(acc.sum())
    total = float(sum(ts))
    value = accepted * args.steps / total
    sample = f"the full {args.config} step ({wl.batch} walkers x {wl.n_moves} proposals), oracle path 2 (delayed rank-K)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(args, cfg, wl),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ----------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1708_00744_b200 import binding, buildlib, inputs
    from paper_1708_00744_b200 import dist as qdist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference "
                         "for the CPU oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        buildlib.build()
    if world > 1:
        dist.barrier()
    binding.load()

    cfg = get_config(args)
    wl = inputs.make_workload(cfg["batch"], cfg["N"], cfg["sweeps"] * cfg["N"],
                              seed=qdist.rank_seed(cfg["seed"], rank, cfg["batch"]))     # per-rank walkers
    N, K, batch, n_moves = wl.N, args.K, wl.batch, wl.n_moves
    mask, uniforms = mode_inputs(wl, args.mode)

    q = binding.Qmcd(N, K, batch)
    if args.cluster:
        q.set_option("cluster", args.cluster)
    if args.flush_path:
        q.set_option("flush_path", args.flush_path)
    for kv in args.opt:
        k_, v_ = kv.split("=")
        q.set_option(k_, int(v_))
    B0 = torch.from_numpy(wl.Ainv).cuda()
    B = torch.empty_like(B0)
    P = torch.from_numpy(wl.proposals).cuda()
    Md = None if mask is None else torch.from_numpy(mask).cuda()
    Ud = None if uniforms is None else torch.from_numpy(uniforms).cuda()
    R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((n_moves, batch), dtype=torch.uint8, device="cuda")
    need_l2_flush = (wl.proposals.nbytes + 2 * wl.Ainv.nbytes) <= 126e6
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if need_l2_flush else None

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(e_sweep=None):
        """One whole pass on device-resident inputs.  Kernels of ours launched: sweep, flush."""
        if scratch is not None:
            scratch.fill_(1)
        B.copy_(B0)                      # F0: a fresh inverse for this pass
        q.set_inverse(B)
        if e_sweep:
            e_sweep[0].record()
        q.sweep(0, P, mask=Md, uniforms=Ud, R_out=R, acc_out=acc)
        if e_sweep:
            e_sweep[1].record()
        q.flush()
    LAUNCHES_PER_STEP = 2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = ev(), ev()
    sweep_ev = [(ev(), ev()) for _ in range(args.steps)]
    barrier()
    e0.record()
    for i in range(args.steps):
        step(sweep_ev[i])
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    sweep_ms = float(np.mean([a.elapsed_time(b) for a, b in sweep_ev]))
    st, info = q.status()
    if st != 0:
        raise SystemExit(f"device status {st} {info}")
    acc_h = acc.cpu().numpy()
    accepted = int(acc_h.sum())
    ms_total, accepted_all = qdist.combine(ms_total, accepted, device="cuda")    # max time, summed moves
    ms_per_step = ms_total / args.steps
    value = qdist.moves_per_second(ms_total, args.steps, accepted_all)

    # ---- end to end: host buffers through qmcd_sweep_host (H2D of Ainv + proposals + mask,
    #      D2H of R + acc inside the timed region)
    e2e = None
    if not args.no_e2e:
        Ph = torch.from_numpy(wl.proposals).pin_memory()
        Bh = torch.from_numpy(wl.Ainv).pin_memory()
        Mh = None if mask is None else torch.from_numpy(mask).pin_memory()
        Uh = None if uniforms is None else torch.from_numpy(uniforms).pin_memory()
        Rh = torch.zeros((n_moves, batch), dtype=torch.float64).pin_memory()
        Ah = torch.zeros((n_moves, batch), dtype=torch.uint8).pin_memory()
        staging = torch.empty((64 << 20) + 256, dtype=torch.uint8, device="cuda")

        def e2e_step():
            B.copy_(Bh, non_blocking=True)
            q.set_inverse(B)
            q.sweep_host(0, Ph, mask=Mh, uniforms=Uh, R_out=Rh, acc_out=Ah, staging=staging)
            q.flush()
        n_e2e = max(2, min(args.steps, 5))
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        barrier()
        dt = (time.perf_counter() - t0) / n_e2e
        tt = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        h2d = Ph.numel() * 8 + Bh.numel() * 8 + (Mh.numel() if Mh is not None else Uh.numel() * 8)
        d2h = Rh.numel() * 8 + Ah.numel()
        assert np.array_equal(Ah.numpy(), acc_h)
        e2e = {"value": accepted_all / float(tt[0]), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * float(tt[0]), "steps": n_e2e,
               "api": "qmcd_sweep_host (pinned host buffers, chunked double-buffered copies)"}
    clocks = sampler.stop() if sampler else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the persistent sweep kernel: F1+F2+F3 fused)
    work = algorithmic_work(acc_h, N, K, lockstep=bool(q.get_option("lockstep")))
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    dmma = binding.probe_fp64(1, 20000)
    dfma = binding.probe_fp64(0, 20000)
    fl_final = 4.0 * N * N  # the final partial flush runs in the separate flush launch: negligible
    ach = work["flops"] / (sweep_ms * 1e-3) / 1e12
    traffic = None
    try:    # dram__bytes_read.sum + dram__bytes_write.sum of this kernel from the committed ncu capture
        for line in open(os.path.join(ROOT, "profiles", "r1_traffic.csv")).read().splitlines()[1:]:
            f = line.split(",")
            if f[0] == f"{args.config}:K{K}:{args.mode}":
                traffic = int(f[1])
    except (OSError, ValueError, IndexError):
        pass
    roofline = {"kernel": "qmcd_kernel_sweep (look-ahead + accept + flush fused, persistent, one launch/step)",
                "bound": "tensor", "achieved": ach, "peak": dmma, "unit": "TFLOP/s",
                "frac": ach / dmma, "traffic": traffic,
                "peak_source": "measured live: register-resident DMMA.8x8x4 fp64 loop (qmcd_probe_fp64); "
                               f"DFMA loop {dfma:.1f} TFLOP/s; MEASURED_PEAKS.json has no fp64 figure",
                "kernel_ms": sweep_ms, "algorithmic_flops_per_launch": work["flops"],
                "algorithmic_bytes_per_launch": work["bytes"],
                "hbm_equiv_gbs": work["bytes"] / (sweep_ms * 1e-3) / 1e9,
                "hbm_peak_gbs": peaks.get("hbm_gbs"),
                "share_of_step": sweep_ms / ms_per_step}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config_dict(args, cfg, wl, {"cluster": q.get_option("cluster"),
                                                 "clusters_per_walker": q.get_option("clusters_per_walker"),
                                                 "lookahead": "blocked" if (q.get_option("blocked_ok") and
                                                                            q.get_option("lookahead") == 0) else "per-move",
                                                 "flush_path": q.get_option("flush_path"),
                                                 "lockstep": q.get_option("lockstep"),
                                                 "accepted_per_step": accepted_all,
                                                 "flushes_per_step": work["flushes"]}),
           "clocks": clocks, "e2e": e2e, "gpu_launches": LAUNCHES_PER_STEP * args.steps,
           "roofline": roofline}

    # time split inside the sweep kernel (SM cycles of each walker's leader CTA, summed over the
    # steps since the last set_inverse = the last step): look-ahead products, per-move chain,
    # queue append, flush
    cyc = q.counters().cpu().numpy()[:, 2:7].astype(np.float64)
    tot = np.maximum(cyc[:, 4], 1.0)
    out["time_split"] = {k: float(np.mean(cyc[:, i] / tot)) for i, k in
                         enumerate(["lookahead_products", "chain", "queue_append", "flush"])}
    out["time_split"]["sweep_cycles_mean"] = float(np.mean(tot))
    if args.phases:
        out["phases"] = time_phases(binding, wl, K)

    if not args.no_cpu_baseline and world == 1:
        import oracle
        dt, acc_o, thr = oracle_step(oracle, wl, K, mask, uniforms)
        assert np.array_equal(acc_o, acc_h), "accept sequence differs from the oracle"
        out["cpu_baseline"] = {"value": int(acc_o.sum()) / dt, "unit": UNIT, "cores": thr, "kind": "oracle",
                               "sample": f"one full {args.config} step, oracle path 2 (delayed rank-K, K={K}), "
                                         f"{dt:.2f} s wall"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def time_phases(binding, wl, K, reps=5):
    """Ratio (F1) and flush (F3) kernels timed in isolation through the per-call API, on this
    workload's shapes: ratio at queue length m = K-1 (the most traffic), flush at rank K-1."""
    import torch
    N, batch = wl.N, wl.batch
    q = binding.Qmcd(N, K, batch)
    q.set_option("lookahead", 1)      # the fill below must stop at m = K-1 (the blocked sweep flushes a nearly full queue early)
    B = torch.from_numpy(wl.Ainv).cuda()
    q.set_inverse(B)
    P = torch.from_numpy(wl.proposals[:max(K, 2) + 64]).cuda()
    R = torch.zeros(batch, dtype=torch.float64, device="cuda")
    ones = torch.ones((K, batch), dtype=torch.uint8, device="cuda")
    m = K - 1
    ev = lambda: torch.cuda.Event(enable_timing=True)
    ratio_ms, flush_ms = [], []
    for rep in range(reps + 1):
        if m > 0:
            q.sweep(0, P[:m], mask=ones[:m])
            assert int(q.pending().min()) == m, "phase timing needs the queue at m = K-1"
        e0, e1 = ev(), ev()
        n_r = 32
        e0.record()
        for i in range(n_r):
            q.ratio(m + i, P[m + i], R)
        e1.record()
        q.reject()
        f0, f1 = ev(), ev()
        f0.record()
        q.flush()
        f1.record()
        torch.cuda.synchronize()
        if rep > 0:
            ratio_ms.append(e0.elapsed_time(e1) / n_r)
            flush_ms.append(f0.elapsed_time(f1))
    # set-up step: qmcd_invert of the batch; every one of the N elimination
    # steps streams each matrix once (read + write): 16 N^3 bytes per walker
    inv_ms = []
    if getattr(wl, "A", None) is not None:
        Ad = torch.from_numpy(wl.A).cuda()
        Xd = torch.empty_like(Ad)
        for rep in range(3):
            i0, i1 = ev(), ev()
            i0.record()
            q.invert(Ad, Ainv=Xd)
            i1.record()
            torch.cuda.synchronize()
            if rep > 0:
                inv_ms.append(i0.elapsed_time(i1))
        del Ad, Xd
    q.close()
    mm = max(m, 0)
    rb = batch * (8.0 * N * (2 * mm + 2) + 8.0 * mm * mm)
    ff = batch * (4.0 * N * N * mm + 2.0 * mm * mm * N)
    fb = batch * (16.0 * N * N + 24.0 * mm * N)
    r_ms, f_ms = float(np.median(ratio_ms)), float(np.median(flush_ms))
    inv = None
    if inv_ms:
        i_ms = float(np.median(inv_ms)); ib = batch * 16.0 * N ** 3
        inv = {"ms_per_launch": i_ms, "bytes": ib, "gbs": ib / (i_ms * 1e-3) / 1e9,
               "flops": batch * 2.0 * N ** 3, "walkers_per_s": batch / (i_ms * 1e-3)}
    return {"invert": inv, "ratio": {"m": mm, "ms_per_launch": r_ms, "bytes": rb, "gbs": rb / (r_ms * 1e-3) / 1e9},
            "flush": {"m": mm, "ms_per_launch": f_ms, "flops": ff, "bytes": fb,
                      "tflops": (ff / (f_ms * 1e-3) / 1e12) if mm else 0.0,
                      "gbs": fb / (f_ms * 1e-3) / 1e9}}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
