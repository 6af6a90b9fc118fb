#!/usr/bin/env python
"""bench.py -- accepted electron moves/s of the delayed rank-K Slater-inverse update
(arXiv 1708.00744) on B200, through the C-ABI library (include/qmcd.h).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--config c3] [--K 64] [--mode bern0.99]

One "step" = one pass of the whole hot path over one batch of synthetic input:
adopt the inverse (F0), run every proposal of the config through ratio (F1) ->
accept/reject (F2) -> flush when K moves are queued (F3), and the final partial
flush (F5).  The default workload is BASELINE.json configs[3] (c3: 32 walkers,
N = 2048, 2 sweeps, Bernoulli(0.99)) at delay K = 64 -- "electron counts in the
thousands" at the delay that is fastest on this machine (DESIGN.md
section 10 says why c3 and not c4).  Prints ONE JSON line (rank 0).

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
DEFAULT_CONFIG, DEFAULT_K, DEFAULT_MODE = "c3", 64, "bern0.99"
NCU_TRAFFIC_BYTES_DEFAULT = 232.9e9       # profiles/r2_ncu_c3_sweep.md: dram__bytes_read.sum + dram__bytes_write.sum per sweep launch


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULT_CONFIG)
    ap.add_argument("--K", type=int, default=DEFAULT_K)
    ap.add_argument("--mode", default=DEFAULT_MODE)
    ap.add_argument("--cluster", type=int, default=0, help="CTAs per leader cluster (0 = library default)")
    ap.add_argument("--flush-path", type=int, default=0, help="0 auto, 1 CUDA-core, 2 DMMA")
    ap.add_argument("--opt", action="append", default=[], help="library option key=value (qmcd_set_option)")
    ap.add_argument("--N", type=int, default=0, help="with --config custom: matrix order")
    ap.add_argument("--batch", type=int, default=1, help="with --config custom: walkers")
    ap.add_argument("--sweeps", type=int, default=1, help="with --config custom: sweeps over the electrons")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-k1", action="store_true", help="skip this library's own K = 1 baseline")
    ap.add_argument("--no-phases", action="store_true",
                    help="skip the ratio and flush kernels timed in isolation (per-call API)")
    ap.add_argument("--no-dgemm", action="store_true", help="skip the library fp64 GEMM ceiling (checker only)")
    ap.add_argument("--quick", action="store_true", help="= --no-cpu-baseline --no-e2e --no-k1 --no-phases --no-dgemm")
    ap.add_argument("--nvtx", action="store_true", help="NVTX ranges around each part of the run")
    ap.add_argument("--Ks", default="", help="comma-separated delays: one JSON line per K on ONE generated workload "
                                             "(K sweeps / the paper's grid; overrides --K)")
    a = ap.parse_args()
    if a.quick:
        a.no_cpu_baseline = a.no_e2e = a.no_k1 = a.no_phases = a.no_dgemm = True
    return a


def get_config(args):
    """BASELINE.json config c0..c4, or a custom shape (the paper's own grid, PAPER.md:103-113:
    one walker, N = 256 ... 8192, 100 % acceptance = --mode bern1.0)."""
    from paper_1708_00744_b200 import inputs
    if args.config == "custom":
        if args.N < 1:
            raise SystemExit("--config custom needs --N")
        return dict(batch=args.batch, N=args.N, sweeps=args.sweeps, Ks=(args.K,), modes=(args.mode,), seed=1)
    return inputs.CONFIGS[args.config]


def mode_inputs(wl, mode, n=None):
    """-> (mask or None, uniforms or None), the first n proposals (all by default)"""
    n = wl.n_moves if n is None else n
    if mode.startswith("bern"):
        return wl.bernoulli_mask(float(mode[4:]))[:n], None
    if mode == "metropolis":
        return None, wl.uniforms[:n]
    raise SystemExit(f"unknown mode {mode}")


def config_dict(args, cfg, batch, N, n_moves, big_inputs, extra=None):
    d = {"workload": f"{args.config}: batch {batch} walkers/GPU, N={N}, {cfg['sweeps']} sweeps "
                     f"({n_moves} proposals/walker), {args.mode}, delay K={args.K}",
         "config": args.config, "batch_per_gpu": batch, "N": N, "K": args.K,
         "proposals_per_walker": n_moves, "acceptance": args.mode,
         "l2": "inputs per step (proposals + inverse + pristine copy) exceed the 126 MB L2"
               if big_inputs else "L2 flushed between steps by writing a 256 MB buffer"}
    if extra:
        d.update(extra)
    return d


def inputs_exceed_l2(batch, N, n_moves):
    return (n_moves * batch * N * 8 + 2 * batch * N * N * 8) > 126e6


def sample_moves(n_moves, K):
    """Bounded sample for the CPU oracle and the K = 1 baseline: the first 2K proposals of every
    walker (>= 128: at least two full windows at the default delay), never more than the run."""
    return min(n_moves, max(2 * K, 128))


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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                s_, m_ = float(c[1]), float(c[2])
            except ValueError:
                continue
            try:
                p_ = float(c[3])
            except ValueError:
                p_ = float("nan")
            sm.append(s_); mx.append(m_); pw.append(p_)
            for nm, val in zip(names, c[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            # "under load": samples in the upper half of the power draw seen (an idle GPU sits at max clock too)
            fin = [p for p in pw if p == p]
            if fin:
                thr = 0.5 * (min(fin) + max(fin))
                hi = [s for s, p in zip(sm, pw) if p == p and p >= thr] or sm
                out["power_w_max"] = float(max(fin))
            else:
                hi = sm
            out["sm_mhz"] = float(np.median(hi))
            out["sm_max_mhz"] = float(max(mx))
            out["samples"] = len(sm)
            out["samples_under_load"] = len(hi)
        out["reasons"] = sorted(reasons)
        return out


# ----------------------------------------------------------------------------- accounting
def algorithmic_work(acc, N, K, lockstep=False):
    """Algorithmic flops / bytes of one step from the accept sequence acc [n_moves][batch]
    (SURVEY.md 8(d) / DESIGN.md 'Kernels'): F1 per proposal at queue length m:
    2N(2m+1)+2m^2 flops, 8N(2m+2)+8m^2 bytes; F2 per accept 4m^2 flops; F3 per rank-m
    flush 4N^2 m + 2 m^2 N flops, 16N^2 + 24mN bytes (final partial flush included).
    lockstep: the window closes after every K-th PROPOSAL with the rank m
    accepted in it; a rejected slot is a zero column of U and counts no work.
    The windows are cut where the METHOD cuts them (m == K); the library may flush a few moves
    early (qmcd.h, qmcd_sweep), which leaves the 4N^2 flops per accepted move unchanged and the
    2 m N term within 2 %: the measured flush count and mean rank are reported beside this."""
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
def oracle_step(oracle, wl, K, mask, uniforms, n):
    """The oracle's delayed rank-K path (path 2) on the first n proposals of every walker."""
    B = wl.Ainv.copy()
    t0 = time.perf_counter()
    R, acc, thr = oracle.run(2, B, K, wl.proposals[:n], mask=mask, uniforms=uniforms, final_flush=True)
    return time.perf_counter() - t0, acc, thr


def sample_text(args, batch, n, n_full):
    return (f"the first {n} of {n_full} proposals of every one of the {batch} walkers of {args.config} "
            f"(>= 2 windows of K={args.K} and the final partial flush), oracle path 2 (delayed rank-K), "
            f"OpenMP over walkers")


def run_reference(args):
    """--impl reference: the CPU oracle as it stands (delayed rank-K path), timed on the host
    cores on a bounded sample of the same config.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_1708_00744_b200 import inputs
    cfg = get_config(args)
    n_full = cfg["sweeps"] * cfg["N"]
    n = sample_moves(n_full, args.K)
    wl = inputs.make_workload(cfg["batch"], cfg["N"], n, seed=cfg["seed"], want_A=False)
    mask, uniforms = mode_inputs(wl, args.mode, n)
    for _ in range(args.warmup):
        oracle_step(oracle, wl, args.K, mask, uniforms, n)
    ts, accepted, thr = [], 0, 0
    for _ in range(args.steps):
        dt, acc, thr = oracle_step(oracle, wl, args.K, mask, uniforms, n)
        ts.append(dt); accepted = int(acc.sum())
    total = float(sum(ts))
    value = accepted * args.steps / total
    sample = sample_text(args, wl.batch, n, n_full)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": config_dict(args, cfg, wl.batch, wl.N, n_full, inputs_exceed_l2(wl.batch, wl.N, n_full)),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ----------------------------------------------------------------------------- our arm
class Nvtx:
    def __init__(self, on):
        self.on = on

    def __call__(self, name):
        import contextlib
        if not self.on:
            return contextlib.nullcontext()
        import torch
        return torch.cuda.nvtx.range(name)


def apply_opts(q, args):
    if args.cluster:
        q.set_option("cluster", args.cluster)
    if args.flush_path:
        q.set_option("flush_path", args.flush_path)
    for kv in args.opt:
        k_, v_ = kv.split("=")
        q.set_option(k_, int(v_))


def load_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


def run_ours(args, wl_cache=None):
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
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        buildlib.build()
    if world > 1:
        dist.barrier()
    binding.load()
    nvtx = Nvtx(args.nvtx)

    cfg = get_config(args)
    if wl_cache is not None and "wl" in wl_cache:
        wl = wl_cache["wl"]
    else:
        wl = inputs.make_workload(cfg["batch"], cfg["N"], cfg["sweeps"] * cfg["N"],
                                  seed=qdist.rank_seed(cfg["seed"], rank, cfg["batch"]), want_A=False)     # per-rank walkers
        if wl_cache is not None:
            wl_cache["wl"] = wl
    N, K, batch, n_moves = wl.N, args.K, wl.batch, wl.n_moves
    mask, uniforms = mode_inputs(wl, args.mode)
    big = inputs_exceed_l2(batch, N, n_moves)

    q = binding.Qmcd(N, K, batch)
    apply_opts(q, args)
    B0 = torch.from_numpy(wl.Ainv).cuda()
    B = torch.empty_like(B0)
    P = torch.from_numpy(wl.proposals).cuda()
    Md = None if mask is None else torch.from_numpy(mask).cuda()
    Ud = None if uniforms is None else torch.from_numpy(uniforms).cuda()
    R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((n_moves, batch), dtype=torch.uint8, device="cuda")
    scratch = None if big else torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

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

    n_warm = max(args.warmup, 3)
    with nvtx("warmup"):
        for _ in range(n_warm):
            step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = ev(), ev()
    sweep_ev = [(ev(), ev()) for _ in range(args.steps)]
    barrier()
    with nvtx("timed steps (sweep: F1 ratio + F2 accept + F3 flush; then the final flush F5)"):
        e0.record()
        for i in range(args.steps):
            step(sweep_ev[i])
        e1.record()
    barrier()
    clocks = sampler.stop() if sampler else None
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
    workers = worker_summary(q, batch, K)
    cyc = q.counters().cpu().numpy()[:, 2:7].astype(np.float64)

    # ---- end to end: host buffers through qmcd_sweep_host (H2D of Ainv + proposals + mask,
    #      D2H of R + acc inside the timed region)
    e2e = None
    if not args.no_e2e:
        with nvtx("end to end (qmcd_sweep_host)"):
            Ph = torch.from_numpy(wl.proposals).pin_memory()
            Bh = torch.from_numpy(wl.Ainv).pin_memory()
            Mh = None if mask is None else torch.from_numpy(mask).pin_memory()
            Uh = None if uniforms is None else torch.from_numpy(uniforms).pin_memory()
            Rh = torch.zeros((n_moves, batch), dtype=torch.float64).pin_memory()
            Ah = torch.zeros((n_moves, batch), dtype=torch.uint8).pin_memory()
            # two buffers of up to 1024 moves each (qmcd_sweep_host cuts the sweep into launches of 128, 256, ... moves)
            staging = torch.empty(2 * min(n_moves, 1024) * (batch * N * 8 + 64 * batch) + 4096, dtype=torch.uint8, device="cuda")

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
            del Ph, Bh, Rh, Ah, staging

    if rank != 0:
        if world > 1 and wl_cache is None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the persistent sweep kernel: F1+F2+F3 fused)
    lockstep = bool(q.get_option("lockstep"))
    work = algorithmic_work(acc_h, N, K, lockstep=lockstep)
    peaks = load_peaks()
    dmma = binding.probe_fp64(1, 20000)
    dfma = binding.probe_fp64(0, 20000)
    ach = work["flops"] / (sweep_ms * 1e-3) / 1e12
    roofline = {"kernel": "qmcd_kernel_sweep (look-ahead + accept + flush jobs; persistent: leader clusters + pool, one launch/step)",
                "bound": "tensor", "achieved": ach, "peak": dmma, "unit": "TFLOP/s",
                "frac": ach / dmma, "traffic": None,
                "traffic_note": "no ncu capture of this configuration; the capture of the default workload is "
                                "profiles/r2_ncu_c3_sweep.md",
                "peak_source": "measured live: register-resident DMMA.8x8x4 fp64 loop (qmcd_probe_fp64) = 148 SMs x SM clock x "
                               f"128 flop/clk; DFMA loop {dfma:.1f} TFLOP/s; MEASURED_PEAKS.json has no fp64 figure",
                "kernel_ms": sweep_ms, "algorithmic_flops_per_launch": work["flops"],
                "algorithmic_bytes_per_launch": work["bytes"],
                "hbm_equiv_gbs": work["bytes"] / (sweep_ms * 1e-3) / 1e9,
                "hbm_peak_gbs": peaks.get("hbm_gbs"),
                "hbm_peak_source": "MEASURED_PEAKS.json (of measured)" if peaks else None,
                "share_of_step": sweep_ms / ms_per_step}

    if (args.config, K, args.mode) == (DEFAULT_CONFIG, DEFAULT_K, DEFAULT_MODE) and not args.cluster and not args.flush_path \
            and all(o.startswith("cooperative=") for o in args.opt):
        # dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of this kernel on this workload, from the ncu --set full
        # capture of this build (a constant of the build, not of this run: refreshed with every change of the kernel)
        roofline["traffic"] = NCU_TRAFFIC_BYTES_DEFAULT
        roofline["traffic_note"] = ("bytes per launch: dram__bytes_read.sum + dram__bytes_write.sum from "
                                    "profiles/r2_ncu_c3_sweep.md (ncu --set full of this kernel, this workload, this build); "
                                    "algorithmic flush bytes per launch: %.4g" % work["flush_bytes"])
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": n_warm, "ms_per_step": ms_per_step, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config_dict(args, cfg, batch, N, n_moves, big,
                                 {"cluster": q.get_option("cluster"), "pool_ctas": q.get_option("pool"),
                                  "tile_rows": q.get_option("tile_rows"),
                                  "lookahead": "blocked" if (q.get_option("blocked_ok") and
                                                             q.get_option("lookahead") == 0) else "per-move",
                                  "flush_path": q.get_option("flush_path"), "lockstep": int(lockstep),
                                  "accepted_per_step": accepted_all,
                                  "flushes_per_step_ideal": work["flushes"],
                                  "flushes_measured": workers["flushes_measured"],
                                  "mean_flush_rank": workers["mean_flush_rank"]}),
           "clocks": clocks, "e2e": e2e, "gpu_launches": LAUNCHES_PER_STEP * args.steps,
           "roofline": roofline}

    # time split inside the sweep kernel (SM cycles of each walker's leader CTA over the last step):
    # look-ahead products, per-move chain, queue append, flush (job posted -> all its tiles finished)
    tot = np.maximum(cyc[:, 4], 1.0)
    out["time_split"] = {k: float(np.mean(cyc[:, i] / tot)) for i, k in
                         enumerate(["lookahead_products", "chain", "queue_append", "flush"])}
    out["time_split"]["sweep_cycles_mean"] = float(np.mean(tot))
    out["workers"] = workers
    q.close()
    del q, B0, B, P, R, acc

    if not args.no_phases:
        with nvtx("phases (ratio and flush kernels alone)"):
            ph = time_phases(binding, wl, K, args)
            for k_, pk, un in (("ratio", peaks.get("hbm_gbs"), "gbs"), ("flush", dmma, "tflops")):
                if ph.get(k_) and pk:
                    ph[k_]["frac_of_peak"] = ph[k_][un] / pk
            out["phases"] = ph
    if not args.no_k1 and K != 1:
        with nvtx("own K = 1 baseline"):
            out["k1_baseline"] = k1_baseline(binding, wl, args, mask, uniforms, value / max(world, 1), peaks)
    if not args.no_dgemm:
        with nvtx("library fp64 GEMM ceiling"):
            roofline["dgemm_ceiling"] = dgemm_ceiling()

    if not args.no_cpu_baseline and world == 1:
        import oracle
        n = sample_moves(n_moves, K)
        m_s, u_s = mode_inputs(wl, args.mode, n)
        dt, acc_o, thr = oracle_step(oracle, wl, K, m_s, u_s, n)
        assert np.array_equal(acc_o, acc_h[:n]), "accept sequence differs from the oracle"
        out["cpu_baseline"] = {"value": int(acc_o.sum()) / dt, "unit": UNIT, "cores": thr, "kind": "oracle",
                               "sample": sample_text(args, batch, n, n_moves) + f", {dt:.2f} s wall"}
    print(json.dumps(out), flush=True)
    if world > 1 and wl_cache is None:
        dist.destroy_process_group()


def worker_summary(q, batch, K):
    """Where the CTAs of the sweep / flush grids spent the last step (qmcd_worker_stats): pool CTAs
    (flush workers serving every walker) and the leader clusters' CTAs."""
    st, fr = q.worker_stats()
    st = st.cpu().numpy().astype(np.float64); fr = fr.cpu().numpy().astype(np.float64)
    S, pool = q.get_option("cluster"), q.get_option("pool")
    nl = min(batch * S, 512)
    lead, pl = st[:nl], st[nl:min(nl + pool, 512)]
    cnt = q.counters().cpu().numpy().astype(np.float64)
    out = {"leader_ctas": int(batch * S), "pool_ctas": int(pool),
           "flushes_measured": int(cnt[:, 1].sum()),
           "mean_flush_rank": float(fr.sum() / max(cnt[:, 1].sum(), 1.0))}
    if len(lead):
        tot = np.maximum(lead[:, 3], 1.0)
        out["leader"] = {"tiles_per_cta": float(lead[:, 0].mean()), "frac_in_own_tiles": float((lead[:, 1] / tot).mean()),
                         "frac_waiting_for_tiles": float((lead[:, 2] / tot).mean())}
    if len(pl):
        tot = np.maximum(pl[:, 3], 1.0)
        out["pool"] = {"tiles_per_cta": float(pl[:, 0].mean()), "frac_in_tiles": float((pl[:, 1] / tot).mean()),
                       "frac_seeking": float((pl[:, 2] / tot).mean()),
                       "cycles_per_tile": float(pl[:, 1].sum() / max(pl[:, 0].sum(), 1.0))}
    return out


def k1_baseline(binding, wl, args, mask, uniforms, value_per_gpu, peaks):
    """This library's own K = 1 Sherman-Morrison path (F4; the paper quotes every speed-up against
    K = 1) on a bounded sample of the same workload: the first proposals of
    every walker.  HBM-bound: >= 16 N^2 bytes per accepted move."""
    import torch
    N, batch = wl.N, wl.batch
    n = sample_moves(wl.n_moves, args.K)
    q = binding.Qmcd(N, 1, batch)
    apply_opts(q, args)
    B = torch.from_numpy(wl.Ainv).cuda()
    P = torch.from_numpy(wl.proposals[:n]).cuda()
    Md = None if mask is None else torch.from_numpy(mask[:n]).cuda()
    Ud = None if uniforms is None else torch.from_numpy(uniforms[:n]).cuda()
    acc = torch.zeros((n, batch), dtype=torch.uint8, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    ms = []
    for rep in range(3):
        q.set_inverse(B)                 # (the inverse walks on from rep to rep; the cost does not depend on it)
        e0, e1 = ev(), ev()
        e0.record()
        q.sweep(0, P, mask=Md, uniforms=Ud, acc_out=acc)
        e1.record()
        torch.cuda.synchronize()
        if rep > 0:
            ms.append(e0.elapsed_time(e1))
    accepted = int(acc.sum().item())
    q.close()
    t = float(np.median(ms)) * 1e-3
    v = accepted / t
    gbs = accepted * 16.0 * N * N / t / 1e9
    return {"value": v, "unit": UNIT, "K": 1, "sample": f"the first {n} proposals of every walker, one launch, median of 2",
            "hbm_gbs": gbs, "frac_of_hbm_peak": (gbs / peaks["hbm_gbs"]) if peaks.get("hbm_gbs") else None,
            "speedup_of_headline_over_k1": value_per_gpu / v}


def dgemm_ceiling():
    """the library DGEMM (torch.matmul fp64, 8192^3) on this device, after the timed
    region, as a second opinion on what a tuned fp64 contraction reaches.  Checker only."""
    import torch
    n = 8192
    a = torch.randn((n, n), dtype=torch.float64, device="cuda")
    b = torch.randn((n, n), dtype=torch.float64, device="cuda")
    c = torch.empty_like(a)
    torch.matmul(a, b, out=c)
    torch.cuda.synchronize()
    best = 1e30
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); torch.matmul(a, b, out=c); e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return {"tflops": 2.0 * n ** 3 / (best * 1e-3) / 1e12, "what": "torch.matmul fp64 8192^3 (cuBLAS), best of 3"}


def time_phases(binding, wl, K, args, reps=5):
    """Ratio (F1) and flush (F3) kernels timed in isolation through the per-call API, on this
    workload's shapes: ratio at queue length m = K-1 (the most traffic), flush at rank K-1."""
    import torch
    N, batch = wl.N, wl.batch
    q = binding.Qmcd(N, K, batch)
    apply_opts(q, args)
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
    # set-up step (outside the hot path): batched on-device inversion, timed on the inverse itself (any well-conditioned matrix)
    inv_ms = []
    Xinv = torch.empty_like(B)
    for rep in range(2):
        i0, i1 = ev(), ev()
        i0.record()
        q.invert(B, Ainv=Xinv)
        i1.record()
        torch.cuda.synchronize()
        inv_ms.append(i0.elapsed_time(i1))
    del Xinv
    q.close()
    mm = max(m, 0)
    rb = batch * (8.0 * N * (2 * mm + 2) + 8.0 * mm * mm)
    ff = batch * (4.0 * N * N * mm + 2.0 * mm * mm * N)
    fb = batch * (16.0 * N * N + 24.0 * mm * N)
    r_ms, f_ms = float(np.median(ratio_ms)), float(np.median(flush_ms))
    return {"ratio": {"m": mm, "ms_per_launch": r_ms, "bytes": rb, "gbs": rb / (r_ms * 1e-3) / 1e9,
                      "note": "back-to-back launches: the queue rows are L2-resident; HBM-cold figure under profiles/"},
            "flush": {"m": mm, "ms_per_launch": f_ms, "flops": ff, "bytes": fb,
                      "tflops": (ff / (f_ms * 1e-3) / 1e12) if mm else 0.0,
                      "gbs": fb / (f_ms * 1e-3) / 1e9},
            "invert": {"ms": float(min(inv_ms)), "what": "qmcd_invert of the whole batch (blocked Gauss-Jordan, set-up step outside the timed path)"}}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.Ks:
        cache = {}
        for k in [int(x) for x in args.Ks.split(",")]:
            args.K = k
            run_ours(args, cache)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
