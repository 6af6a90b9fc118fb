"""K (and launch shape) autotuner (the paper: "K ... can be autotuned",
PAPER.md:89,109): time a bounded run of the device-resident sweep for each candidate delay K --
and, on request, each candidate number of CTAs per leader cluster (option "cluster": the
library's default is a rule fitted to the BASELINE shapes) -- on the caller's shape and
return the measured accepted moves/s.  It drives the same C-ABI calls as everything else
(qmcd_create / set_inverse / sweep / flush); there is no model and no CPU path.

    python -m paper_1708_00744_b200.autotune --batch 32 --N 2048 --Ks 16,32,64,128
    python -m paper_1708_00744_b200.autotune --batch 8 --N 4096 --Ks 64 --clusters 1,2,4
"""
from __future__ import annotations

import argparse
import json


def autotune_K(N: int, batch: int, Ks=(16, 32, 64, 128), acceptance: float = 0.99,
               n_moves: int | None = None, reps: int = 2, seed: int = 1, clusters=None) -> dict:
    """-> {"best_K": k, "moves_per_s": {k: rate}, "n_moves": n}.  Synthetic inputs with the
    recipe of BASELINE.json (inputs.make_workload); n_moves defaults to 4 windows of the largest
    K (at least 256), so every candidate sees several full flushes.
    clusters: candidate CTAs per leader cluster (powers of two); None = the library's default only.
    With clusters the result also holds "best_cluster" and "by_cluster" {k: {S: rate}}; a (K, S) pair the
    library refuses (shared memory, divisibility) is skipped."""
    import torch
    from . import binding, inputs
    Ks = [int(k) for k in Ks if 1 <= int(k) <= N]
    if not Ks:
        raise ValueError("no admissible K (need 1 <= K <= N)")
    if n_moves is None:
        n_moves = max(256, 4 * max(Ks))
    wl = inputs.make_workload(batch, N, n_moves, seed=seed, want_A=False)
    mask = wl.bernoulli_mask(acceptance)
    accepted = int(mask.sum())
    B0 = torch.from_numpy(wl.Ainv).cuda()
    P = torch.from_numpy(wl.proposals).cuda()
    M = torch.from_numpy(mask).cuda()
    B = torch.empty_like(B0)
    rates, by_cluster, best_S = {}, {}, {}
    for K in Ks:
        for S in (list(clusters) if clusters else [None]):
            q = binding.Qmcd(N, K, batch)
            if S is not None:
                try:
                    q.set_option("cluster", int(S))
                except binding.QmcdError:
                    q.close()
                    continue
            S_used = q.get_option("cluster")
            best = float("inf")
            for rep in range(reps + 1):                      # the first repetition warms up
                B.copy_(B0)
                q.set_inverse(B)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                q.sweep(0, P, mask=M)
                q.flush()
                e1.record()
                torch.cuda.synchronize()
                if rep > 0:
                    best = min(best, e0.elapsed_time(e1))
            st, _ = q.status()
            q.close()
            if st != 0:
                raise RuntimeError(f"device status {st} at K={K}")
            rate = accepted / (best * 1e-3)
            by_cluster.setdefault(K, {})[S_used] = rate
            if rate > rates.get(K, 0.0):
                rates[K], best_S[K] = rate, S_used
    best_K = max(rates, key=rates.get)
    out = {"best_K": best_K, "moves_per_s": rates, "n_moves": n_moves, "accepted": accepted}
    if clusters:
        out.update(best_cluster=best_S[best_K], by_cluster=by_cluster)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, required=True)
    ap.add_argument("--batch", type=int, required=True)
    ap.add_argument("--Ks", default="16,32,64,128")
    ap.add_argument("--acceptance", type=float, default=0.99)
    ap.add_argument("--clusters", default="", help="comma-separated CTAs per leader cluster to try (default: the library's choice)")
    a = ap.parse_args()
    cl = [int(c) for c in a.clusters.split(",")] if a.clusters else None
    print(json.dumps(autotune_K(a.N, a.batch, [int(k) for k in a.Ks.split(",")], a.acceptance, clusters=cl)))


if __name__ == "__main__":
    main()
