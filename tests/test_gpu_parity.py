"""GPU parity: the CUDA path (through the C-ABI / binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json's north_star: identical
accept sequence, every ratio to relative error <= 1e-10, max|A.Ainv - I| <= 1e-8 after every
flush (fp64)."""
import numpy as np
import pytest

import oracle
from paper_1708_00744_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL_RATIO = 1e-10
TOL_RESID = 1e-8


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _rel(a, b):
    return np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-300))


def gpu_sweep(qmcd, wl, K, mask=None, uniforms=None, final_flush=True, cluster=None, j_begin=0,
              flush_path=None, lookahead=None, lockstep=None, G=None, split=None, tile_rows=None, pool=None, tma=None, la_tma=None, stagger=None):
    import torch
    q = qmcd.Qmcd(wl.N, K, wl.batch)
    if lockstep is not None:
        q.set_option("lockstep", lockstep)
    if stagger is not None:
        q.set_option("stagger", stagger)
    if cluster is not None:
        q.set_option("cluster", cluster)
    if flush_path is not None:
        q.set_option("flush_path", flush_path)
    if lookahead is not None:
        q.set_option("lookahead", lookahead)
    if G is not None:
        q.set_option("clusters_per_walker", G)       # round-1 name: 1 = leader clusters only, > 1 = with the pool
    if pool is not None:
        q.set_option("pool", pool)
    if tma is not None:
        q.set_option("tma", tma)                     # 0: the cp.async flush kernels also for K <= 64
        q.set_option("la_tma", 2 if tma else 0)      # ... and the TMA-ring look-ahead on every shape that fits / never
    if la_tma is not None:
        q.set_option("la_tma", la_tma)
    if tile_rows is not None:
        q.set_option("tile_rows", tile_rows)
    blocked = bool(q.get_option("blocked_ok")) and q.get_option("lookahead") == 0
    B = _dev(wl.Ainv)
    q.set_inverse(B)
    P = _dev(wl.proposals)
    R = torch.zeros((wl.n_moves, wl.batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, wl.batch), dtype=torch.uint8, device="cuda")
    Md = None if mask is None else _dev(mask)
    Ud = None if uniforms is None else _dev(uniforms)
    cuts = [0] + list(split or []) + [wl.n_moves]
    for a, b in zip(cuts[:-1], cuts[1:]):          # one launch per piece
        q.sweep((j_begin + a) % wl.N, P[a:b], mask=None if Md is None else Md[a:b],
                uniforms=None if Ud is None else Ud[a:b], R_out=R[a:b], acc_out=acc[a:b])
    if final_flush:
        q.flush()
    st, info = q.status()
    cnt = q.counters().cpu().numpy()
    pend = q.pending().cpu().numpy()
    out = dict(R=R.cpu().numpy(), acc=acc.cpu().numpy(), B=B.cpu().numpy(), status=st, info=info,
               counters=cnt, pending=pend, S=q.get_option("cluster"), blocked=blocked, pool=q.get_option("pool"),
               tma=q.get_option("tma"), la_tma=q.get_option("la_tma"))
    q.close()
    return out


def gpu_calls(qmcd, wl, K, mask, flush_every=None, residual_cb=None, ratio_kernel=None):
    """The per-call API: ratio -> accept(mask) per move."""
    import torch
    q = qmcd.Qmcd(wl.N, K, wl.batch)
    if ratio_kernel is not None:
        q.set_option("ratio_kernel", ratio_kernel)
    B = _dev(wl.Ainv)
    q.set_inverse(B)
    P = _dev(wl.proposals)
    Md = _dev(mask)
    R = torch.zeros((wl.n_moves, wl.batch), dtype=torch.float64, device="cuda")
    for t in range(wl.n_moves):
        q.ratio(t % wl.N, P[t], R[t])
        q.accept(Md[t])
        if flush_every and (t + 1) % flush_every == 0:
            q.flush()
        if residual_cb is not None:
            residual_cb(t, q, B)
    q.flush()
    st, _ = q.status()
    out = dict(R=R.cpu().numpy(), B=B.cpu().numpy(), status=st, counters=q.counters().cpu().numpy())
    q.close()
    return out


def check_residuals(wl, acc, B):
    for w in range(wl.batch):
        A_cur = inputs.current_matrix(wl.A[w], wl.proposals[:, w, :], acc[:, w], wl.n_moves)
        res = np.max(np.abs(A_cur @ B[w] - np.eye(wl.N)))
        assert res <= TOL_RESID, (w, res)


# ------------------------------------------------------------------ config 0, every check
def test_c0_calls_vs_oracle_delayed_rank1_and_residual_after_every_flush(qmcd):
    """BASELINE.json configs[0]: N=64, K=4, 2 sweeps, Bernoulli(0.99); per-call API."""
    wl = inputs.make_config("c0")
    mask = wl.bernoulli_mask(0.99)
    K = 4
    B1 = wl.Ainv.copy(); R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, mask=mask)
    B2 = wl.Ainv.copy(); R2, acc2, _ = oracle.run(2, B2, K, wl.proposals, mask=mask)
    seen = {"flushes": 0, "last": 0}

    def cb(t, q, B):
        c = int(q.counters()[0, 1].item())
        if c != seen["last"]:           # a flush happened inside this accept
            seen["last"] = c; seen["flushes"] += 1
            assert int(q.pending()[0].item()) == 0
            A_cur = inputs.current_matrix(wl.A[0], wl.proposals[:, 0, :], mask[:, 0], t + 1)
            res = np.max(np.abs(A_cur @ B[0].cpu().numpy() - np.eye(wl.N)))
            assert res <= TOL_RESID, (t, res)

    g = gpu_calls(qmcd, wl, K, mask, residual_cb=cb)
    assert g["status"] == 0
    assert seen["flushes"] == int(mask.sum()) // K
    assert _rel(g["R"], R2) <= RTOL_RATIO and _rel(g["R"], R1) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - B2)) <= 1e-11 and np.max(np.abs(g["B"] - B1)) <= 1e-11
    check_residuals(wl, mask, g["B"])
    assert int(g["counters"][0, 0]) == int(mask.sum())
    # explicit LU at sampled moves (path 0)
    A = wl.A[0].copy()
    for t in range(wl.n_moves):
        if t % 9 == 0:
            Rb = oracle.ratio_bruteforce(A, t % wl.N, wl.proposals[t, 0])
            assert abs(g["R"][t, 0] - Rb) <= RTOL_RATIO * abs(Rb)
        if mask[t, 0]:
            A[:, t % wl.N] = wl.proposals[t, 0]


# ------------------------------------------------------------------ ragged sizes, several tiles
@pytest.mark.parametrize("N,K,batch,cluster", [
    (100, 7, 3, 1), (100, 7, 3, 2), (130, 16, 2, 4), (257, 33, 2, 8), (96, 96, 1, 1), (64, 1, 2, 1),
    (520, 40, 2, 16), (33, 5, 150, 1),
])
def test_sweep_matches_oracle_ragged(qmcd, N, K, batch, cluster):
    wl = inputs.make_workload(batch, N, n_moves=min(2 * N + 3, 300), seed=7)
    mask = wl.bernoulli_mask(0.8)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster)
    assert g["status"] == 0 and g["S"] == cluster
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    check_residuals(wl, mask, g["B"])
    assert np.array_equal(g["counters"][:, 0], mask.sum(axis=0))
    assert np.all(g["pending"] == 0)


@pytest.mark.parametrize("N,K,batch,cluster,p", [
    (128, 16, 2, 1, 0.8),      # one 128-row tile, ragged final rank
    (128, 5, 2, 2, 1.0),       # rank 5 -> padded to 8, 64-row tiles
    (256, 40, 2, 4, 0.8),      # 64 rows per CTA, rank 40
    (256, 64, 3, 2, 0.95),     # full 64-wide block, 128-row tiles
    (512, 96, 2, 4, 0.9),      # two m-blocks (64 + 32), R = 64 layout
    (256, 200, 1, 1, 0.9),     # four m-blocks, several M row blocks
    (320, 24, 2, 1, 0.7),      # N = 5 chunks, rows 320 = 2.5 tiles of 128
    (192, 1, 2, 1, 0.9),       # rank 1 through the tensor path
])
def test_dmma_flush_matches_oracle(qmcd, N, K, batch, cluster, p):
    """The FP64 tensor-core flush (flush_path = 2 forces it whenever N and N/S are multiples
    of 64) against the oracle's delayed path: every ratio, the accept sequence, the inverse."""
    wl = inputs.make_workload(batch, N, n_moves=N + K + 7, seed=17)
    mask = wl.bernoulli_mask(p)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, flush_path=2)
    assert g["status"] == 0 and g["S"] == cluster
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    check_residuals(wl, mask, g["B"])
    # and the CUDA-core path gives the same inverse to rounding
    s = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, flush_path=1)
    assert np.max(np.abs(g["B"] - s["B"])) <= 1e-11


@pytest.mark.parametrize("N,K,batch,cluster,G", [(512, 32, 3, 4, 2), (512, 16, 2, 2, 4), (256, 8, 4, 1, 4),
                                                 (1024, 64, 2, 4, 4), (384, 24, 2, 2, 3)])
def test_helper_clusters_share_the_flush(qmcd, N, K, batch, cluster, G):
    """With the pool (round-1 option name clusters_per_walker > 1): the leader cluster of a walker runs
    the look-ahead and posts its flush jobs; its own CTAs and the pool CTAs take the row tiles."""
    wl = inputs.make_workload(batch, N, n_moves=N + 2 * K + 5, seed=31)
    mask = wl.bernoulli_mask(0.9)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    import torch
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("cluster", cluster)
    q.set_option("clusters_per_walker", G)
    assert q.get_option("pool") > 0
    B = _dev(wl.Ainv); q.set_inverse(B)
    R = torch.zeros((wl.n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, batch), dtype=torch.uint8, device="cuda")
    half = wl.n_moves // 2
    P, Md = _dev(wl.proposals), _dev(mask)
    q.sweep(0, P[:half], mask=Md[:half], R_out=R[:half], acc_out=acc[:half])
    q.flush()                                    # explicit flush launch with helpers, mid-run
    q.sweep(half % N, P[half:], mask=Md[half:], R_out=R[half:], acc_out=acc[half:])
    q.flush()
    assert q.status()[0] == 0
    assert np.array_equal(acc.cpu().numpy(), acco)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10
    check_residuals(wl, mask, B.cpu().numpy())
    q.close()


def test_sweep_equals_call_by_call(qmcd):
    """qmcd_sweep must reproduce the ratio -> accept(mask) sequence (include/qmcd.h)."""
    wl = inputs.make_workload(4, 128, 200, seed=3)
    mask = wl.bernoulli_mask(0.7)
    a = gpu_sweep(qmcd, wl, 8, mask=mask, lookahead=1)      # per-move look-ahead ...
    b = gpu_calls(qmcd, wl, 8, mask, ratio_kernel=0)        # ... and qmcd_ratio through the same device function: same arithmetic
    assert not a["blocked"]
    assert np.array_equal(a["R"], b["R"])
    assert np.array_equal(a["B"], b["B"])
    b = gpu_calls(qmcd, wl, 8, mask)                        # the dedicated ratio kernel (default): another summation order
    assert _rel(b["R"], a["R"]) <= 1e-12 and np.max(np.abs(a["B"] - b["B"])) <= 1e-12
    c = gpu_sweep(qmcd, wl, 8, mask=mask)                   # blocked look-ahead: other summation order
    assert c["blocked"]
    assert _rel(c["R"], b["R"]) <= 1e-12
    assert np.max(np.abs(c["B"] - b["B"])) <= 1e-12


@pytest.mark.parametrize("N,K,batch,cluster,p,j_begin", [
    (128, 16, 2, 1, 0.8, 0),       # one CTA per walker
    (128, 5, 3, 2, 1.0, 3),        # K not a multiple of 8, every move accepted
    (256, 40, 2, 4, 0.5, 250),     # wrap-around of the electron index inside a block
    (512, 96, 2, 4, 0.9, 0),       # 26 output tiles per block
    (64, 64, 2, 1, 0.3, 0),        # K = N with many rejections: electrons repeat inside a window
    (48, 24, 2, 2, 0.4, 5),        # ragged chunk (24 columns per CTA), repeats
    (1024, 32, 2, 16, 0.99, 0),    # 16 CTAs per walker, one strip row per owner
    (512, 128, 2, 2, 0.9, 0),      # K = 128: M stays in GLOBAL memory, staged 16 rows at a time (qmcd_blk_xy_global)
    (256, 150, 2, 1, 0.5, 3),      # K = 150 (ragged panels, K not a multiple of 8), many rejections
    (1024, 128, 3, 4, 0.99, 1000), # clusters of 4: the leader CTA alone writes M, the others read it after the barrier
])
def test_blocked_lookahead_matches_oracle_and_per_move(qmcd, N, K, batch, cluster, p, j_begin):
    """qmcd_sweep's blocked look-ahead (qmcd_block.cuh) against the oracle's delayed path and
    against the per-move look-ahead of the same library."""
    wl = inputs.make_workload(batch, N, n_moves=3 * N, seed=23)
    # move t proposes electron (j_begin + t) % N: take the proposal the generator built around
    # that column (keeps the matrices as well conditioned as in the BASELINE configs)
    n_moves = 2 * N + 11
    t = np.arange(n_moves)
    pick = (t % N + j_begin) % N + N * (t // N)
    wl.proposals = np.ascontiguousarray(wl.proposals[pick]); wl.uniforms = np.ascontiguousarray(wl.uniforms[pick])
    wl.n_moves = n_moves
    mask = wl.bernoulli_mask(p)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, j_begin=j_begin, mask=mask)
    # la_tma = 0: the 16-proposal blocks of qmcd_block.cuh (LDG / cp.async strips) -- the path of K > 64 and of shapes the
    # super-block ring does not take; the default (super-blocks where they fit) is checked below and in the next test
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, j_begin=j_begin, la_tma=0)
    assert g["status"] == 0 and g["S"] == cluster and g["blocked"] and g["la_tma"] == 0
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    assert np.array_equal(g["counters"][:, 0], mask.sum(axis=0))
    assert np.all(g["pending"] == 0)
    pm = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, j_begin=j_begin, lookahead=1)
    assert not pm["blocked"]
    assert np.max(np.abs(g["R"] - pm["R"])) <= 1e-11
    assert np.max(np.abs(g["B"] - pm["B"])) <= 1e-11
    # the library's default for this shape: super-blocks through the TMA ring when K <= 64 and the slices are whole
    # 16-column chunks -- wrap-around cuts the super-block, a repeated electron cuts it or flushes first
    gt = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, j_begin=j_begin)
    fits = N >= 128 and N % 64 == 0 and ((K <= 64 and (N // cluster) % 16 == 0) or (64 < K <= 128 and K % 2 == 0 and (N // cluster) % 8 == 0))
    assert gt["la_tma"] == (1 if fits else 0)
    assert gt["blocked"] and gt["status"] == 0
    assert np.array_equal(gt["acc"], acco)
    assert _rel(gt["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(gt["B"] - Bo)) <= 1e-10


@pytest.mark.parametrize("N,K,batch,cluster,mode,j_begin,lockstep", [
    (256, 64, 2, 1, "bern0.99", 0, 0),     # one 64-proposal super-block per window, tiles of D only
    (256, 64, 2, 2, "bern0.5", 200, 0),    # rate-adaptive length (64 proposals at queue length 32), wrap-around, cluster-wide sum
    (512, 64, 2, 4, "bern0.3", 0, 0),      # over-long super-blocks: the queue fills inside one and the rest is looked at again
    (128, 64, 2, 1, "bern0.2", 0, 0),      # K near N with many rejections: queued electrons come round again (cut / flush first)
    (256, 48, 3, 2, "bern0.7", 5, 0),      # K = 48: shapes 64 -> 32 -> 16 as the queue fills
    (192, 20, 2, 1, "bern0.9", 0, 0),      # K not a multiple of 8, N = 3 x 64
    (256, 3, 2, 1, "bern1.0", 0, 0),       # K smaller than a block
    (256, 64, 2, 8, "metropolis", 0, 0),   # 8 CTAs per walker (32-column slices), Metropolis decisions on the ratios
    (1024, 64, 2, 2, "bern0.8", 1000, 0),  # long slices: queue append in several pieces per warp
    (512, 128, 2, 2, "bern0.9", 0, 0),     # K = 128: M in global memory, one k-group per stage, shapes 64 -> 32 -> 32
    (1024, 128, 2, 4, "bern0.5", 1000, 0), # ... at 50 % acceptance, clusters of 4 (the leader CTA alone writes M), wrap-around
    (256, 100, 2, 1, "bern0.7", 0, 0),     # K = 100: ragged queue boxes (rows past K zero-filled by TMA)
    (256, 64, 2, 1, "bern0.5", 0, 1),      # lock-step windows (oracle path 3)
    (256, 40, 2, 2, "bern0.1", 3, 1),      # lock-step with few acceptances
])
def test_superblock_lookahead_matches_oracle(qmcd, N, K, batch, cluster, mode, j_begin, lockstep):
    """qmcd_sweep's super-block look-ahead (qmcd_superblock.cuh: P | Q | D of up to 64 proposals from one pass over the
    operands, queue entries accepted inside the super-block read out of D) against the oracle's delayed path (path 2;
    lock-step: the literal path 3), every ratio, decision and the final inverse; launches cut at odd places."""
    wl = inputs.make_workload(batch, N, n_moves=3 * N, seed=31)
    n_moves = 2 * N + 37
    t = np.arange(n_moves)
    pick = (t % N + j_begin) % N + N * (t // N)
    wl.proposals = np.ascontiguousarray(wl.proposals[pick]); wl.uniforms = np.ascontiguousarray(wl.uniforms[pick])
    wl.n_moves = n_moves
    mask = wl.bernoulli_mask(float(mode[4:])) if mode.startswith("bern") else None
    u = wl.uniforms if mode == "metropolis" else None
    Bo = wl.Ainv.copy()
    if lockstep:
        Ao = wl.A.copy()
        Ro, acco, _, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, j_begin=j_begin, mask=mask, uniforms=u)
    else:
        Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, j_begin=j_begin, mask=mask, uniforms=u)
    for split in (None, [7, 100, N + 1]):
        g = gpu_sweep(qmcd, wl, K, mask=mask, uniforms=u, cluster=cluster, j_begin=j_begin, lockstep=lockstep or None, split=split)
        assert g["status"] == 0 and g["S"] == cluster and g["blocked"] and g["la_tma"] == 1
        if u is not None:
            near_tie = np.abs(u - np.minimum(1.0, Ro * Ro)) < 1e-9            # reading G20
            assert np.array_equal(g["acc"][~near_tie], acco[~near_tie])
        else:
            assert np.array_equal(g["acc"], acco)
        assert _rel(g["R"], Ro) <= RTOL_RATIO
        assert np.max(np.abs(g["B"] - Bo)) <= 1e-10 * max(1.0, np.abs(Bo).max())
        assert np.array_equal(g["counters"][:, 0], acco.sum(axis=0))
        assert np.all(g["pending"] == 0)


@pytest.mark.parametrize("N,K,batch,cluster,p", [(256, 64, 5, 1, 0.99), (512, 32, 8, 2, 0.6), (256, 8, 3, 1, 1.0), (256, 32, 8, 1, 0.05)])
def test_staggered_first_windows_are_neutral(qmcd, N, K, batch, cluster, p):
    """Option "stagger" (default for 2 ... 8 walkers with N >= 2048, forced here): the first window of walker b in a launch
    is cut short to K (b mod 8 + 1) / 8 moves so that the walkers' flushes do not coincide -- the same ratios, decisions and
    inverse as without, at most one more flush per walker and launch."""
    wl = inputs.make_workload(batch, N, n_moves=2 * N + 9, seed=41)
    mask = wl.bernoulli_mask(p)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    out = {}
    for st in (1, 0):
        g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, stagger=st, split=[N + 3])
        assert g["status"] == 0 and g["la_tma"] == 1
        assert np.array_equal(g["acc"], acco)
        assert _rel(g["R"], Ro) <= RTOL_RATIO
        assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
        out[st] = g["counters"][:, 1]
    assert np.all(out[1] >= out[0])              # (the shortened first window costs a flush unless the final partial one absorbs it)


@pytest.mark.timeout(120, method="thread")
@pytest.mark.parametrize("K,lockstep", [(1, 0), (1, 1), (8, 0)])
def test_launch_starting_with_a_rejection_and_room_for_one_move(qmcd, K, lockstep):
    """Regression, found by a randomized soak: the super-block length is the room left in the queue over the acceptance rate
    seen so far in the launch; with room for ONE move and the launch's first proposal rejected it came out as 0 proposals and
    the sweep never advanced.  K = 1, and K = 8 with 7 moves carried over from the launch before."""
    N, batch = 128, 2
    wl = inputs.make_workload(batch, N, n_moves=60, seed=5)
    mask = np.ones((60, batch), dtype=np.uint8)
    first = 0 if K == 1 else K - 1                       # the launch that starts at `first` begins with rejections
    mask[first:first + 3] = 0
    mask[20:25, 1] = 0
    Bo = wl.Ainv.copy()
    if lockstep:
        Ao = wl.A.copy()
        Ro, acco, _, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, mask=mask)
    else:
        Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=1, lockstep=lockstep or None, split=[first] if first else None)
    assert g["status"] == 0 and g["la_tma"] == 1
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10


@pytest.mark.parametrize("N,K,batch,cluster,p", [
    (128, 1, 3, 1, 0.9),       # K = 1: the classic Sherman-Morrison update (Eqs. 1-2)
    (192, 1, 2, 2, 1.0),       # N a multiple of 64 but not of 128
    (1024, 1, 2, 1, 0.5),      # 8 tiles per flush through the pool
    (2048, 2, 2, 1, 0.8),      # K = 2: ranks 1 and 2
    (4096, 2, 1, 2, 0.99),
    (256, 2, 40, 1, 0.7),      # 40 walkers, 64-row tiles
])
def test_rank1_and_rank2_flush_matches_oracle(qmcd, N, K, batch, cluster, p):
    """K <= 2 (in particular K = 1, the classic Sherman-Morrison baseline of Eqs. 1-2): rank-1 / rank-2 flush jobs through
    the tile kernels and the pool against the oracle's rank-1 path (path 1), launches cut in two."""
    import torch
    n_moves = min(N, 300) + 7
    wl = inputs.make_workload(batch, N, n_moves=n_moves, seed=77)
    mask = wl.bernoulli_mask(p)
    B1 = wl.Ainv.copy(); R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, mask=mask)      # K-independent
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("cluster", cluster)
    B = _dev(wl.Ainv)
    q.set_inverse(B)
    R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((n_moves, batch), dtype=torch.uint8, device="cuda")
    q.sweep(0, _dev(wl.proposals[:100]), mask=_dev(mask[:100]), R_out=R[:100], acc_out=acc[:100])
    q.sweep(100 % N, _dev(wl.proposals[100:]), mask=_dev(mask[100:]), R_out=R[100:], acc_out=acc[100:])
    q.flush()
    st, _ = q.status()
    cnt = q.counters().cpu().numpy()
    q.close()
    assert st == 0
    assert np.array_equal(acc.cpu().numpy(), acc1)
    assert _rel(R.cpu().numpy(), R1) <= RTOL_RATIO
    assert np.max(np.abs(B.cpu().numpy() - B1)) <= 1e-10 * max(1.0, np.abs(B1).max())
    assert np.array_equal(cnt[:, 0], acc1.sum(axis=0))


@pytest.mark.parametrize("K", [1, 16, 32])
def test_c1_full_size_vs_rank1_oracle(qmcd, K):
    """BASELINE.json configs[1] at full size, in bench.py's launch configuration (qmcd_sweep):
    ratios and accept sequence are K-independent, so one rank-1 oracle run is the
    reference for every K."""
    wl = inputs.make_config("c1")
    mask = wl.bernoulli_mask(0.99)
    ref = getattr(test_c1_full_size_vs_rank1_oracle, "_ref", None)
    if ref is None:
        B1 = wl.Ainv.copy(); R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, mask=mask)
        ref = (R1, acc1, B1)
        test_c1_full_size_vs_rank1_oracle._ref = ref
    R1, acc1, B1 = ref
    g = gpu_sweep(qmcd, wl, K, mask=mask)
    assert g["status"] == 0
    assert np.array_equal(g["acc"], acc1)
    assert _rel(g["R"], R1) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - B1)) <= 1e-9
    check_residuals(wl, mask, g["B"])


def test_metropolis_accept_sequence_identical(qmcd):
    """BASELINE.json configs[2] rule u < min(1, R^2), reduced size."""
    wl = inputs.make_workload(8, 256, 512, seed=11)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, 16, wl.proposals, uniforms=wl.uniforms)
    g = gpu_sweep(qmcd, wl, 16, uniforms=wl.uniforms)
    near_tie = np.abs(wl.uniforms - np.minimum(1.0, Ro * Ro)) < 1e-9      # reading G20
    assert np.array_equal(g["acc"][~near_tie], acco[~near_tie])
    assert near_tie.sum() == 0
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert 0.9 < acco.mean() < 1.0
    check_residuals(wl, acco, g["B"])


def test_metropolis_per_call(qmcd):
    import torch
    wl = inputs.make_workload(3, 96, 120, seed=5)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, 6, wl.proposals, uniforms=wl.uniforms)
    q = qmcd.Qmcd(wl.N, 6, wl.batch)
    B = _dev(wl.Ainv); q.set_inverse(B)
    P, U = _dev(wl.proposals), _dev(wl.uniforms)
    R = torch.zeros((wl.n_moves, wl.batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, wl.batch), dtype=torch.uint8, device="cuda")
    for t in range(wl.n_moves):
        q.ratio(t % wl.N, P[t], R[t])
        q.accept_metropolis(U[t], acc[t])
    q.flush()
    assert q.status()[0] == 0
    assert np.array_equal(acc.cpu().numpy(), acco)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10


def test_flush_neutrality_and_K_independence(qmcd):
    """delayed == one at a time; inserting qmcd_flush anywhere changes no ratio."""
    wl = inputs.make_workload(2, 128, 256, seed=13)
    mask = wl.bernoulli_mask(0.9)
    base = gpu_calls(qmcd, wl, 16, mask)
    for fe in (1, 5, 37):
        o = gpu_calls(qmcd, wl, 16, mask, flush_every=fe)
        assert _rel(o["R"], base["R"]) <= 1e-11
        assert np.max(np.abs(o["B"] - base["B"])) <= 1e-11
    for K in (1, 3, 128):
        o = gpu_sweep(qmcd, wl, K, mask=mask)
        assert _rel(o["R"], base["R"]) <= 1e-11
        assert np.max(np.abs(o["B"] - base["B"])) <= 1e-11


def test_repeated_electron_in_window_and_ratio_jv(qmcd):
    """Reading G7: the delta term keeps the ratio exact for an already-queued electron, and
    accepting it flushes first.  Uses per-walker electron indices (qmcd_ratio_jv)."""
    import torch
    N, K, batch = 48, 6, 3
    wl = inputs.make_workload(batch, N, 12, seed=21)
    js = np.array([[0, 5, 9], [1, 5, 3], [0, 7, 9], [2, 5, 9], [0, 5, 1], [4, 4, 4], [4, 4, 4]], dtype=np.int32)
    q = qmcd.Qmcd(N, K, batch)
    B = _dev(wl.Ainv); q.set_inverse(B)
    P = _dev(wl.proposals)
    R = torch.zeros(batch, dtype=torch.float64, device="cuda")
    D = [oracle.Delayed(wl.Ainv[w].copy(), K) for w in range(batch)]
    A = [wl.A[w].copy() for w in range(batch)]
    for t in range(js.shape[0]):
        q.ratio(_dev(js[t]), P[t], R)
        q.accept()
        Rg = R.cpu().numpy()
        for w in range(batch):
            Ro = D[w].ratio(int(js[t, w]), wl.proposals[t, w])
            Rb = oracle.ratio_bruteforce(A[w], int(js[t, w]), wl.proposals[t, w])
            assert abs(Rg[w] - Ro) <= RTOL_RATIO * abs(Ro)
            assert abs(Rg[w] - Rb) <= 1e-9 * abs(Rb)
            D[w].accept()
            A[w][:, js[t, w]] = wl.proposals[t, w]
    pend = q.pending().cpu().numpy()
    assert list(pend) == [D[w].pending for w in range(batch)]
    q.flush()
    assert q.status()[0] == 0
    Bg = B.cpu().numpy()
    for w in range(batch):
        assert np.max(np.abs(A[w] @ Bg[w] - np.eye(N))) <= TOL_RESID
    q.close()


def test_closed_form_current_column_gives_one_and_linear_combination(qmcd):
    """Pin P2 on the GPU: v = A_cur alpha  =>  R = alpha_j exactly, mid-window too."""
    import torch
    N, K = 80, 8
    wl = inputs.make_workload(1, N, 5, seed=4)
    q = qmcd.Qmcd(N, K, 1)
    B = _dev(wl.Ainv); q.set_inverse(B)
    R = torch.zeros(1, dtype=torch.float64, device="cuda")
    A = wl.A[0].copy()
    for t in range(5):                                   # queue 5 moves
        q.ratio(t, _dev(wl.proposals[t]), R); q.accept()
        A[:, t] = wl.proposals[t, 0]
    rng = np.random.default_rng(0)
    alpha = rng.standard_normal(N)
    for j in (2, 40):                                    # queued and not queued electron
        q.ratio(j, _dev((A @ alpha)[None, :]), R); q.reject()
        assert abs(R.item() - alpha[j]) <= 1e-11 * max(1, abs(alpha[j]))
        q.ratio(j, _dev(A[:, j][None, :].copy()), R); q.reject()
        assert abs(R.item() - 1.0) <= 1e-12
    q.close()


def test_state_machine_and_singular_status(qmcd):
    import torch
    N = 32
    wl = inputs.make_workload(1, N, 2, seed=2)
    q = qmcd.Qmcd(N, 4, 1)
    R = torch.zeros(1, dtype=torch.float64, device="cuda")
    v = _dev(wl.proposals[0])
    with pytest.raises(qmcd.QmcdError) as e:
        q.ratio(0, v, R)                                 # no inverse yet
    assert e.value.code == qmcd.ESTATE
    B = _dev(wl.Ainv); q.set_inverse(B)
    with pytest.raises(qmcd.QmcdError):
        q.accept()                                       # IDLE
    with pytest.raises(qmcd.QmcdError):
        q.ratio(N, v, R)                                 # j out of range
    q.ratio(0, v, R)
    with pytest.raises(qmcd.QmcdError):
        q.flush()                                        # PROPOSED
    q.ratio(1, v, R)                                     # replaces the staged proposal
    q.reject()
    q.flush()                                            # legal when idle, no-op
    assert q.status()[0] == 0
    # singular: new column = another column of A  ->  R ~ 0 exactly only if forced; use zeros
    q.ratio(3, torch.zeros((1, N), dtype=torch.float64, device="cuda"), R)
    q.accept()
    st, info = q.status()
    assert R.item() == 0.0 and st == qmcd.ESINGULAR and info[0] == 0
    assert int(q.pending()[0].item()) == 0               # the move was dropped
    q.close()


def test_sweep_host_matches_device_sweep(qmcd):
    """The end-to-end path (host buffers, chunked double-buffered copies) gives the same results."""
    import torch
    wl = inputs.make_workload(4, 128, 300, seed=9)
    mask = wl.bernoulli_mask(0.9)
    ref = gpu_sweep(qmcd, wl, 8, mask=mask)
    q = qmcd.Qmcd(wl.N, 8, wl.batch)
    B = _dev(wl.Ainv); q.set_inverse(B)
    Ph = torch.from_numpy(wl.proposals).pin_memory()
    Mh = torch.from_numpy(mask).pin_memory()
    Rh = torch.zeros((wl.n_moves, wl.batch), dtype=torch.float64).pin_memory()
    Ah = torch.zeros((wl.n_moves, wl.batch), dtype=torch.uint8).pin_memory()
    need = qmcd.load().qmcd_sweep_host_min_staging(wl.N, wl.batch)
    staging = torch.empty(need * 7 + 256, dtype=torch.uint8, device="cuda")   # forces many chunks
    q.sweep_host(0, Ph, mask=Mh, R_out=Rh, acc_out=Ah, staging=staging)
    q.flush()          # (between flushes the stale inverse depends on where the launches were cut)
    # chunk boundaries cut the look-ahead blocks elsewhere: same numbers to rounding
    assert _rel(Rh.numpy(), ref["R"]) <= 1e-12
    assert np.array_equal(Ah.numpy(), ref["acc"])
    assert np.max(np.abs(B.cpu().numpy() - ref["B"])) <= 1e-12
    q.close()


# ------------------------------------------------------------------ full-size configs, bench launch configuration
def test_blocked_sweep_singular_move_is_dropped_and_reported(qmcd):
    """Reading G13 inside qmcd_sweep (blocked look-ahead): a proposal with R == 0 that the mask
    accepts sets the sticky status, is NOT queued, and the rest of the run is unaffected."""
    import torch
    wl = inputs.make_workload(2, 128, 200, seed=41)
    mask = wl.bernoulli_mask(0.9)
    t_bad, w_bad = 37, 1
    wl.proposals[t_bad, w_bad, :] = 0.0               # zero column: det(A_new) = 0 exactly
    mask[t_bad, w_bad] = 1
    ref_mask = mask.copy(); ref_mask[t_bad, w_bad] = 0  # what must effectively happen
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, 16, wl.proposals, mask=ref_mask)
    g = gpu_sweep(qmcd, wl, 16, mask=mask)
    assert g["blocked"] and g["status"] == qmcd.ESINGULAR and g["info"][0] == w_bad
    assert g["R"][t_bad, w_bad] == 0.0 and g["acc"][t_bad, w_bad] == 0
    assert np.array_equal(g["acc"], ref_mask)
    ok = np.ones_like(mask, dtype=bool); ok[t_bad, w_bad] = False
    assert _rel(g["R"][ok], Ro[ok]) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10


def test_helper_clusters_with_metropolis_and_single_moves(qmcd):
    """Helper clusters under the Metropolis rule, driven by sweeps of 1, 2, 3, ... proposals
    (blocks and windows cut at every launch boundary; M, J, m live in global memory in between)."""
    import torch
    N, K, batch = 256, 8, 3
    wl = inputs.make_workload(batch, N, 120, seed=43)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, uniforms=wl.uniforms)
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("cluster", 2); q.set_option("clusters_per_walker", 2)
    B = _dev(wl.Ainv); q.set_inverse(B)
    P, U = _dev(wl.proposals), _dev(wl.uniforms)
    R = torch.zeros((wl.n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, batch), dtype=torch.uint8, device="cuda")
    t, step = 0, 1
    while t < wl.n_moves:
        n = min(step, wl.n_moves - t)
        q.sweep(t % N, P[t:t + n], uniforms=U[t:t + n], R_out=R[t:t + n], acc_out=acc[t:t + n])
        t += n; step += 1
    q.flush()
    assert q.status()[0] == 0
    assert np.array_equal(acc.cpu().numpy(), acco)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10
    q.close()


def test_autotune_K_picks_a_tensor_bound_delay(qmcd):
    """the autotuner times the real sweep per candidate K.  On a c2-shaped problem
    the classic K = 1 path must lose by a wide margin and the winner must be a delay >= 16."""
    from paper_1708_00744_b200 import autotune
    r = autotune.autotune_K(1024, 16, Ks=(1, 16, 32, 64), n_moves=256, reps=1)
    assert set(r["moves_per_s"]) == {1, 16, 32, 64}
    assert r["best_K"] in (16, 32, 64)
    assert r["moves_per_s"][r["best_K"]] > 5 * r["moves_per_s"][1]
    # the launch shape too: CTAs per leader cluster (the default is a rule fitted to the BASELINE shapes)
    r = autotune.autotune_K(1024, 16, Ks=(64,), n_moves=256, reps=1, clusters=(1, 2, 4, 3))
    assert set(r["by_cluster"][64]) == {1, 2, 4}                     # 3 is refused by the library and skipped
    assert r["best_cluster"] in (1, 2, 4) and r["moves_per_s"][64] == max(r["by_cluster"][64].values())


def test_randomized_shapes_seeds_modes_and_launch_splits(qmcd):
    """A short randomized soak (fixed generator): shapes with and without the pool of flush workers, random
    seeds, acceptance 0.2 ... 0.99 or the Metropolis rule, the run cut into 1 ... 4 sweep launches at
    random places, staggered first windows on or off -- every run against the oracle's delayed path.  (Longer
    versions of this loop outside the suite: 3500 runs over N = 72 ... 1024, K = 1 ... 200,
    found the zero-length super-block of `test_launch_starting_with_a_rejection_and_room_for_one_move` and are
    green since, worst deviation 1.7e-14.)"""
    import torch
    rng = np.random.default_rng(123)
    shapes = [(256, 16, 8, 2, 2), (512, 32, 6, 4, 2), (128, 8, 10, 1, 2), (384, 24, 4, 2, 3),
              (1024, 64, 3, 4, 4), (320, 40, 5, 1, 1), (192, 192, 2, 1, 1),
              (320, 1, 4, 2, 2), (640, 96, 2, 2, 2), (256, 64, 5, 8, 2), (200, 20, 3, 1, 2), (512, 128, 2, 4, 2)]
    for run in range(24):
        N, K, batch, S, G = shapes[run % len(shapes)]
        seed = int(rng.integers(1, 1 << 30)); p = float(rng.choice([0.99, 0.9, 0.5, 0.2, 0.05]))
        n_moves = int(rng.integers(N // 2, 2 * N))
        wl = inputs.make_workload(batch, N, n_moves, seed=seed)
        metro = bool(rng.integers(0, 2))
        mask = None if metro else wl.bernoulli_mask(p)
        uni = wl.uniforms if metro else None
        Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask, uniforms=uni)
        q = qmcd.Qmcd(N, K, batch)
        q.set_option("cluster", S)
        if G > 1:
            q.set_option("clusters_per_walker", G)
        q.set_option("stagger", int(rng.integers(0, 2)))
        B = _dev(wl.Ainv); q.set_inverse(B)
        P = _dev(wl.proposals)
        R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
        acc = torch.zeros((n_moves, batch), dtype=torch.uint8, device="cuda")
        cuts = sorted(set([0, n_moves] + [int(c) for c in rng.integers(1, n_moves, size=int(rng.integers(0, 4)))]))
        for a, b in zip(cuts[:-1], cuts[1:]):
            q.sweep(a % N, P[a:b], mask=None if mask is None else _dev(mask[a:b]),
                    uniforms=None if uni is None else _dev(uni[a:b]), R_out=R[a:b], acc_out=acc[a:b])
        q.flush()
        assert q.status()[0] == 0
        q.close()
        ctx = (N, K, batch, S, G, seed, p, metro)
        assert np.array_equal(acc.cpu().numpy(), acco), ctx
        assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO, ctx
        assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10, ctx


@pytest.mark.parametrize("N,K,batch,cluster,path,pool,p", [
    (256, 16, 5, 1, "tma", -1, 0.9),        # S = 1 leaders, everything else is pool; TMA-fed tiles, NB = 2
    (256, 16, 5, 1, "cp64", -1, 0.9),       # the cp.async kernels on 64-row tiles
    (256, 16, 5, 1, "cp128", -1, 0.9),      # ... on 128-row tiles: two tiles per job
    (512, 64, 3, 2, "tma", -1, 0.99),       # full-rank local jobs, NB = 8
    (512, 64, 3, 2, "cp128", -1, 0.99),
    (512, 64, 3, 2, "cp64", 3, 0.99),       # a pool of one cluster (3 CTAs asked, rounded down to whole clusters)
    (512, 96, 2, 4, "cp64", -1, 0.9),       # K > 64: the Y = M W job, then the row job with Y
    (256, 200, 2, 1, "cp64", -1, 0.9),      # four m-blocks, several M row blocks, two-phase jobs
    (320, 24, 40, 1, "tma", -1, 0.5),       # 40 walkers drifting apart at 50 % acceptance; 320 rows = 2.5 tiles (TMA clips)
    (320, 24, 40, 1, "cp64", -1, 0.5),
    (192, 1, 3, 1, "tma", -1, 0.9),         # rank-1 jobs (K = 1 Sherman-Morrison) through the pool, NB = 1
    (192, 5, 3, 1, "tma", -1, 1.0),         # K not a multiple of 8: queue rows past K are zero-filled by TMA
    (1024, 64, 2, 8, "tma", -1, 0.99),      # clusters of 8: 15 fit, 13 of them pool
    (1024, 40, 2, 2, "tma", -1, 0.3),       # NB = 8 with ranks 33 ... 40 and low-rank final flushes
    (512, 32, 4, 2, "tma128", -1, 0.9),     # TMA-fed tiles of 128 rows forced on a small N (default there: 64 rows)
    (2048, 64, 2, 1, "tma64", -1, 0.99),    # ... and 64-row TMA tiles forced on a large N
    (512, 96, 2, 4, "tma", -1, 0.9),        # 64 < K <= 128: Y = M W job (cp.async), then 64-row TMA tiles multiplying by Y
    (1024, 128, 3, 1, "tma", -1, 0.99),     # K = 128, full rank, blocked look-ahead with M in global memory
    (256, 100, 2, 2, "tma", -1, 0.5),       # K = 100 (not a multiple of 8), ranks 93 ... 100
    (128, 32, 140, 1, "tma", -1, 0.8),      # 140 leaders + 8 pool CTAs, one tile per job
    (128, 32, 140, 1, "cp64", -1, 0.8),
])
def test_pool_flush_jobs_match_oracle(qmcd, N, K, batch, cluster, path, pool, p):
    """Flush jobs taken tile by tile by the leader's own CTAs and by the pool (qmcd_kernel.cuh), through the
    TMA-fed tile kernel (qmcd_flush_tma.cuh) or the cp.async kernels: every ratio, the accept sequence and
    the inverse against the oracle's delayed path, with launches cut in the middle of a window; and the
    same run without the pool."""
    wl = inputs.make_workload(batch, N, n_moves=min(2 * N, 700) + K + 3, seed=61)
    mask = wl.bernoulli_mask(p)
    Bo = wl.Ainv.copy(); Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    kw = dict(tma=1) if path == "tma" else dict(tma=1, tile_rows=int(path[3:])) if path.startswith("tma") else dict(tma=0, tile_rows=int(path[2:]))
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, pool=pool,
                  split=[wl.n_moves // 3, wl.n_moves // 3 + 5], **kw)
    assert g["status"] == 0 and g["S"] == cluster
    assert g["tma"] == (1 if path.startswith("tma") else 0)
    assert g["pool"] > 0 and g["pool"] % cluster == 0
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    check_residuals(wl, mask, g["B"])
    g0 = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, pool=0, **kw)
    assert g0["pool"] == 0 and np.array_equal(g0["acc"], acco)
    assert np.max(np.abs(g0["B"] - Bo)) <= 1e-10 and _rel(g0["R"], Ro) <= RTOL_RATIO


def test_tma_flush_per_call_api_partial_ranks_and_stale_M(qmcd):
    """The TMA-fed flush behind the per-call API: a long window (rank 48) followed by short ones (ranks 3, 9)
    flushed explicitly -- M's 64 x 64 tile in global memory still holds the long window's entries outside the
    short windows' m x m blocks and must be zero-padded before the flush multiplies by the whole tile."""
    import torch
    N, K, batch = 256, 48, 3
    wl = inputs.make_workload(batch, N, n_moves=48 + 3 + 9, seed=77)
    q = qmcd.Qmcd(N, K, batch)
    assert q.get_option("tma") == 0                    # no inverse adopted yet: no tensor map of B
    B = _dev(wl.Ainv); q.set_inverse(B)
    assert q.get_option("tma") == 1
    P = _dev(wl.proposals)
    R = torch.zeros(batch, dtype=torch.float64, device="cuda")
    Bo = wl.Ainv.copy()
    D = [oracle.Delayed(Bo[w], K) for w in range(batch)]
    t = 0
    for win in (48, 3, 9):
        for _ in range(win):
            q.ratio(t % N, P[t], R)
            Rg = R.cpu().numpy()
            for w in range(batch):
                assert abs(D[w].ratio(t % N, wl.proposals[t, w]) / Rg[w] - 1) <= RTOL_RATIO
                D[w].accept()
            q.accept()
            t += 1
        q.flush()
        for w in range(batch):
            D[w].flush()
        assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10, win
    assert q.status()[0] == 0
    q.close()


def test_cluster_option_rejects_non_powers_of_two(qmcd):
    """the blocked look-ahead deals its 16 strip rows over the CTAs of a cluster, which
    needs a power of two; 3, 5, 6, 7 used to be accepted and raced."""
    q = qmcd.Qmcd(768, 16, 2)
    for bad in (3, 5, 6, 7, 12, 0, 17):
        with pytest.raises(qmcd.QmcdError):
            q.set_option("cluster", bad)
    for ok in (1, 2, 4, 8):
        q.set_option("cluster", ok)
        assert q.get_option("cluster") == ok
    q.close()


# ------------------------------------------------------------------ the dedicated ratio kernel (per-call API)
@pytest.mark.parametrize("N,K,batch,n_moves", [
    (33, 5, 7, 40),          # odd N: 8-byte loads, one slice
    (100, 7, 3, 60),         # even, ragged slice
    (257, 33, 2, 80),        # odd N, several slices, K not a multiple of 8
    (1024, 64, 4, 150),      # several slices x row groups, two full windows
    (2048, 200, 1, 230),     # one walker: 8 row groups; M (200 x 200) read from global memory by the last CTA
])
def test_ratio_kernel_per_call_vs_oracle(qmcd, N, K, batch, n_moves):
    """qmcd_ratio through the dedicated kernel (qmcd_ratio.cuh): every ratio of a call-by-call run against the
    oracle's delayed path at every queue length 0 ... K-1, with accepts and rejects in between; and the
    same calls through the cluster kernel's look-ahead (option ratio_kernel = 0) agree to rounding."""
    import torch
    wl = inputs.make_workload(batch, N, n_moves, seed=29)
    mask = wl.bernoulli_mask(0.85)
    Bo = wl.Ainv.copy()
    D = [oracle.Delayed(Bo[w], K) for w in range(batch)]
    runs = {}
    for opt in (1, 0):
        q = qmcd.Qmcd(N, K, batch)
        q.set_option("ratio_kernel", opt)
        B = _dev(wl.Ainv); q.set_inverse(B)
        P, Md = _dev(wl.proposals), _dev(mask)
        R = torch.zeros(batch, dtype=torch.float64, device="cuda")
        Rs = np.zeros((n_moves, batch))
        for t in range(n_moves):
            q.ratio(t % N, P[t], R)
            q.accept(Md[t])
            Rs[t] = R.cpu().numpy()
        q.flush()
        assert q.status()[0] == 0
        runs[opt] = (Rs, B.cpu().numpy())
        q.close()
    for t in range(n_moves):
        for w in range(batch):
            Ro = D[w].ratio(t % N, wl.proposals[t, w])
            assert abs(runs[1][0][t, w] / Ro - 1) <= RTOL_RATIO, (t, w)
            if mask[t, w]:
                D[w].accept()
            else:
                D[w].reject()
    for w in range(batch):
        D[w].flush()
    assert np.max(np.abs(runs[1][1] - Bo)) <= 1e-10
    assert np.max(np.abs(runs[1][0] / runs[0][0] - 1)) <= 1e-11
    assert np.max(np.abs(runs[1][1] - runs[0][1])) <= 1e-11


# ------------------------------------------------------------------ slot replacement (reading G7)
@pytest.mark.parametrize("N,K,batch,cluster,p,j_begin", [
    (64, 64, 2, 1, 0.3, 0),        # K = N at 30 % acceptance: every window revisits queued electrons
    (48, 24, 3, 2, 0.4, 5),        # clusters of 2, ragged slices
    (128, 100, 2, 1, 0.5, 0),      # M in shared memory, K > 64 flush path
    (256, 200, 1, 4, 0.6, 250),    # M in GLOBAL memory (K too large for shared memory), wrap-around
])
def test_slot_replacement_sweep_matches_oracle_path4(qmcd, N, K, batch, cluster, p, j_begin):
    """Option "slot_replace": an electron accepted again before the queue is applied replaces the column of
    its queue slot (column-replacement Sherman-Morrison on M) instead of flushing first.  Against the
    oracle's literal path 4 (rebuilds S, LU-solves): ratios, decisions, inverse, and the same, smaller
    number of flushes; flush-first (the default) must give the same inverse with more flushes."""
    # proposals are generated for electron t mod N: start the stream at j_begin so that move t perturbs the
    # column of the electron it moves (otherwise the walk duplicates columns and becomes singular)
    full = inputs.make_workload(batch, N, n_moves=4 * N + 7 + j_begin, seed=23)
    wl = inputs.Workload(batch=batch, N=N, n_moves=4 * N + 7, seed=23, A=full.A, Ainv=full.Ainv,
                         proposals=np.ascontiguousarray(full.proposals[j_begin:]),
                         uniforms=np.ascontiguousarray(full.uniforms[j_begin:]))
    mask = wl.bernoulli_mask(p)
    jseq = ((j_begin + np.arange(wl.n_moves)) % N).astype(np.int32)
    Bo = wl.Ainv.copy()
    Ro, acco, flo, _ = oracle.run_jseq(Bo, K, wl.proposals, jseq, True, mask=mask)
    import torch
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("cluster", cluster); q.set_option("slot_replace", 1)
    assert q.get_option("slot_replace") == 1 and q.get_option("blocked_ok") == 0
    B = _dev(wl.Ainv); q.set_inverse(B)
    R = torch.zeros((wl.n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, batch), dtype=torch.uint8, device="cuda")
    q.sweep(j_begin, _dev(wl.proposals), mask=_dev(mask), R_out=R, acc_out=acc)
    q.flush()
    assert q.status()[0] == 0
    cnt = q.counters().cpu().numpy()
    q.close()
    assert np.array_equal(acc.cpu().numpy(), acco)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    # the walk replaces every column several times at small N: entries of the inverse reach ~1e2 here, so the
    # element-wise bar is relative to the largest entry (the ratios above and the residual below are the
    # north_star's bars)
    btol = 1e-10 * max(1.0, float(np.max(np.abs(Bo))))
    Bg = B.cpu().numpy()
    assert np.max(np.abs(Bg - Bo)) <= btol
    for w in range(batch):
        A_cur = wl.A[w].copy()
        for t in range(wl.n_moves):
            if mask[t, w]:
                A_cur[:, jseq[t]] = wl.proposals[t, w]
        assert np.max(np.abs(A_cur @ Bg[w] - np.eye(N))) <= 1e-8
    assert np.array_equal(cnt[:, 0], mask.sum(axis=0))
    assert np.array_equal(cnt[:, 1], flo)                       # Eq. 4 applied exactly as often as in the oracle
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, j_begin=j_begin, lookahead=1)     # flush-first
    assert np.max(np.abs(g["B"] - Bo)) <= btol
    assert (g["counters"][:, 1] >= cnt[:, 1]).all() and g["counters"][:, 1].sum() > cnt[:, 1].sum()


def test_slot_replacement_per_call_sequence(qmcd):
    """The (1, 4, 1, 4, 4, 2) sequence of the oracle pin P12 through qmcd_ratio / qmcd_accept."""
    import torch
    N, K, batch = 64, 6, 2
    wl = inputs.make_workload(batch, N, n_moves=12, seed=13)
    js = (1, 4, 1, 4, 4, 2, 2, 9, 1, 4, 30, 1)
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("slot_replace", 1)
    B = _dev(wl.Ainv); q.set_inverse(B)
    Bo = wl.Ainv.copy()
    D = [oracle.Delayed(Bo[w], K, replace=True) for w in range(batch)]
    R = torch.zeros(batch, dtype=torch.float64, device="cuda")
    A = wl.A.copy()
    for t, j in enumerate(js):
        v = A[:, :, j] + 0.3 * (wl.proposals[t] - wl.A[:, :, t % N]) * 8.0 / np.sqrt(N) + 0.05     # a new column for electron j
        q.ratio(j, _dev(v), R)
        Rg = R.cpu().numpy()
        for w in range(batch):
            An = A[w].copy(); An[:, j] = v[w]
            truth = np.linalg.det(An) / np.linalg.det(A[w])
            assert abs(D[w].ratio(j, v[w]) / truth - 1) <= 1e-10
            assert abs(Rg[w] / truth - 1) <= 1e-10, (t, j, w)
            D[w].accept()
            A[w] = An
        q.accept()
        pend = q.pending().cpu().numpy()
        assert all(int(pend[w]) == D[w].pending for w in range(batch)), (t, pend)
    q.flush()
    for w in range(batch):
        D[w].flush()
    assert q.status()[0] == 0
    assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10
    for w in range(batch):
        assert np.max(np.abs(A[w] @ B.cpu().numpy()[w] - np.eye(N))) <= 1e-8
    q.close()


# ------------------------------------------------------------------ lock-step variant
def _windows_with_accepts(acc, K):
    n = (acc.shape[0] // K) * K
    return acc[:n].reshape(-1, K, acc.shape[1]).any(axis=1).sum(axis=0)


@pytest.mark.parametrize("N,K,batch,cluster,G,p,lookahead,split", [
    (128, 16, 3, 1, None, 0.5, 0, None),        # blocked look-ahead, one block per window
    (128, 16, 3, 2, None, 0.5, 1, None),        # per-move look-ahead
    (256, 40, 2, 4, None, 0.5, 0, [37, 301]),   # windows of 16 + 16 + 8 proposals, launches cut mid-window
    (512, 32, 3, 4, 2, 0.99, 0, None),          # the pool shares the flushes
    (512, 64, 2, 4, None, 0.3, 0, [5]),         # DMMA flush of low, varying rank
    (96, 7, 2, 1, None, 0.1, 0, None),          # windows with no accepted move at all
    (64, 1, 2, 1, None, 0.5, 0, None),          # K = 1
    (256, 24, 3, 2, 2, 0.5, 0, [100]),          # TMA-ring look-ahead (la_tma forced on below) + pool, windows of 16 + 8
])
def test_lockstep_sweep_matches_oracle_path3(qmcd, N, K, batch, cluster, G, p, lookahead, split):
    """Option "lockstep" against the oracle's literal path 3 (a rejected move
    queues the unchanged column): same ratios, decisions and inverse; every walker flushes in
    the same move, once per K proposals."""
    n_moves = 2 * N + 13
    wl = inputs.make_workload(batch, N, n_moves=n_moves, seed=41)
    mask = wl.bernoulli_mask(p)
    Ao, Bo = wl.A.copy(), wl.Ainv.copy()
    Ro, acco, flo, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, mask=mask, final_flush=False)
    la = 2 if (N, K) == (256, 24) else None       # that case: the TMA-ring look-ahead, forced on
    g = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, G=G, lookahead=lookahead, lockstep=1,
                  split=split, final_flush=False, la_tma=la)
    assert g["status"] == 0 and (la is None or g["la_tma"] == 1)
    if lookahead == 1:
        assert not g["blocked"]
    assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    assert np.all(flo == n_moves // K)
    assert np.array_equal(g["counters"][:, 1], _windows_with_accepts(mask, K))   # empty windows cost nothing
    assert np.all(g["counters"][:, 7] == n_moves % K)
    assert np.array_equal(g["pending"], mask[(n_moves // K) * K:].sum(axis=0))
    # the other reading (only accepted moves take slots) reaches the same inverse
    g2 = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, lookahead=lookahead)
    g1 = gpu_sweep(qmcd, wl, K, mask=mask, cluster=cluster, G=G, lookahead=lookahead, lockstep=1, split=split)
    assert np.max(np.abs(g1["B"] - g2["B"])) <= 1e-10
    check_residuals(wl, acco, g1["B"])


def test_lockstep_metropolis_and_per_call_api(qmcd):
    """Lock-step through ratio / accept / accept_metropolis / reject, and a Metropolis sweep."""
    import torch
    N, K, batch, n_moves = 64, 6, 3, 100
    wl = inputs.make_workload(batch, N, n_moves=n_moves, seed=42)
    u = wl.uniforms
    Ao, Bo = wl.A.copy(), wl.Ainv.copy()
    Ro, acco, flo, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, uniforms=u, final_flush=False)
    g = gpu_sweep(qmcd, wl, K, uniforms=u, lockstep=1, final_flush=False)
    assert g["status"] == 0 and np.array_equal(g["acc"], acco) and _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-10
    # per-call: every third proposal is dropped with qmcd_reject, the others decided by Metropolis
    u2 = u.copy(); u2[::3] = 2.0                     # u >= 1 > min(1, R^2): rejected
    Ao, Bo = wl.A.copy(), wl.Ainv.copy()
    Ro, acco, flo, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, uniforms=u2, final_flush=False)
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("lockstep", 1)
    B = _dev(wl.Ainv); q.set_inverse(B)
    P = _dev(wl.proposals); Ud = _dev(u2)
    R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((n_moves, batch), dtype=torch.uint8, device="cuda")
    for t in range(n_moves):
        q.ratio(t % N, P[t], R[t])
        if t % 3 == 0:
            q.reject()
        else:
            q.accept_metropolis(Ud[t], acc[t])
        if (t + 1) % K == 0:
            assert np.all(q.pending().cpu().numpy() == 0), t      # the window closed in this move
    st, _ = q.status()
    cnt = q.counters().cpu().numpy()
    assert st == 0
    assert np.array_equal(acc.cpu().numpy(), acco)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    assert np.max(np.abs(B.cpu().numpy() - Bo)) <= 1e-10
    assert np.all(cnt[:, 7] == n_moves % K)
    q.flush()
    assert np.all(q.counters().cpu().numpy()[:, 7] == 0)
    q.close()


# ------------------------------------------------------------------ on-device inversion
@pytest.mark.parametrize("N,batch,seed", [(1, 2, 3), (7, 3, 4), (64, 1, 1), (130, 5, 6), (512, 16, 7), (1024, 3, 8)])
def test_invert_matches_oracle_lu_inverse(qmcd, N, batch, seed):
    """qmcd_invert (Gauss-Jordan, partial pivoting) against the oracle's LU inverse and the
    north_star residual; a leading zero forces a row exchange in walker 0."""
    import torch
    wl = inputs.make_workload(batch, N, n_moves=1, seed=seed)
    A = wl.A.copy()
    if N > 1:
        A[0, 0, 0] = 0.0
    q = qmcd.Qmcd(N, 1, batch)
    Ad = _dev(A)
    X, info = q.invert(Ad)
    torch.cuda.synchronize()
    assert np.all(info.cpu().numpy() == 0)
    assert torch.equal(Ad, _dev(A))                       # the input is left alone
    Xh = X.cpu().numpy()
    for w in range(min(batch, 4)):
        Xo = oracle.inverse(A[w])
        assert np.max(np.abs(Xh[w] - Xo)) <= 1e-10 * max(1.0, np.abs(Xo).max())
        assert np.max(np.abs(A[w] @ Xh[w] - np.eye(N))) <= TOL_RESID
    # in place, then adopted: the ratios of a sweep agree with the oracle started from ITS inverse
    q.invert(Ad, Ainv=Ad)
    torch.cuda.synchronize()
    assert np.array_equal(Ad.cpu().numpy(), Xh)
    q.close()


@pytest.mark.parametrize("N,batch", [(7, 3), (33, 2), (130, 5), (512, 16), (1000, 3)])
def test_invert_blocked_equals_unblocked_kernel(qmcd, N, batch):
    """The blocked Gauss-Jordan kernel (panels of 16 pivot columns, the default) against the unblocked one (option
    invert_blocked = 0): the same pivots and the same arithmetic in the same order, so the results agree to the last
    bits; both against the oracle's LU inverse.  Walker 0 starts with a zero (row exchange), the last one holds a NaN."""
    import torch
    wl = inputs.make_workload(batch, N, n_moves=1, seed=91)
    A = wl.A.copy()
    A[0, 0, 0] = 0.0
    A[batch - 1, N // 2, N // 3] = np.nan
    out = {}
    for blk in (1, 0):
        q = qmcd.Qmcd(N, 1, batch)
        q.set_option("invert_blocked", blk)
        assert q.get_option("invert_blocked") == blk
        X, info = q.invert(_dev(A))
        torch.cuda.synchronize()
        out[blk] = (X.cpu().numpy(), info.cpu().numpy())
        q.close()
    # the NaN walker is reported by both (the blocked kernel at the first column whose candidates hold the NaN, the unblocked
    # one when the NaN reaches a pivot), the others are fine
    for blk in (1, 0):
        assert out[blk][1][batch - 1] != 0 and np.all(out[blk][1][:batch - 1] == 0)
    for w in range(batch - 1):
        Xo = oracle.inverse(A[w])
        for blk in (1, 0):
            assert np.max(np.abs(out[blk][0][w] - Xo)) <= 1e-10 * max(1.0, np.abs(Xo).max())
        assert np.max(np.abs(out[1][0][w] - out[0][0][w])) <= 1e-13 * max(1.0, np.abs(Xo).max())


def test_invert_permutation_singular_and_pipeline(qmcd):
    import torch
    N, batch, K = 96, 3, 8
    rng = np.random.default_rng(5)
    A = np.zeros((batch, N, N))
    perm = rng.permutation(N)
    A[0, np.arange(N), perm] = 2.0                         # scaled permutation: every step pivots
    A[1] = np.eye(N); A[1, 5, 5] = 0.0                     # exactly singular
    wl = inputs.make_workload(1, N, n_moves=2 * N, seed=9)
    A[2] = wl.A[0]
    q = qmcd.Qmcd(N, K, batch)
    X, info = q.invert(_dev(A))
    torch.cuda.synchronize()
    info = info.cpu().numpy(); Xh = X.cpu().numpy()
    assert info[0] == 0 and info[2] == 0 and info[1] == 6  # first zero pivot at step k = 5
    assert np.array_equal(Xh[0], A[0].T / 4.0)             # closed form, exact in fp64
    # walker 2: invert -> set_inverse -> sweep, against the oracle run from its own LU inverse
    q.close()
    q = qmcd.Qmcd(N, K, 1)
    Bd, _ = q.invert(_dev(wl.A))
    q.set_inverse(Bd)
    mask = wl.bernoulli_mask(0.7)
    R = torch.zeros((wl.n_moves, 1), dtype=torch.float64, device="cuda")
    q.sweep(0, _dev(wl.proposals), mask=_dev(mask), R_out=R)
    q.flush()
    Bo = oracle.inverse(wl.A[0])[None].copy()
    Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    assert _rel(R.cpu().numpy(), Ro) <= RTOL_RATIO
    assert np.max(np.abs(Bd.cpu().numpy() - Bo)) <= 1e-10
    q.close()


def test_invert_c4_full_size_residual_and_lapack(qmcd):
    """qmcd_invert at BASELINE configs[4]'s size (8 walkers, N = 4096, 512 threads x 2 CTAs/SM,
    37 CTAs per walker): the north_star residual max|A.Ainv - I| <= 1e-8 for every walker (fp64
    product on the device, a library call used as a checker only) and agreement with the LAPACK
    inverse the input generator made."""
    import torch
    wl = inputs.make_workload(8, 4096, n_moves=1, seed=44)
    q = qmcd.Qmcd(4096, 1, 8)
    Ad = _dev(wl.A)
    X, info = q.invert(Ad)
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    eye = torch.eye(4096, dtype=torch.float64, device="cuda")
    for w in range(8):
        assert float((Ad[w] @ X[w] - eye).abs().max()) <= TOL_RESID
        assert float((X[w] @ Ad[w] - eye).abs().max()) <= TOL_RESID
    assert float((X - _dev(wl.Ainv)).abs().max()) <= 1e-9
    q.close()


@pytest.mark.parametrize("mode", ["bern0.5", "metropolis"])
def test_c1_full_size_lockstep_default_launch_vs_oracle_path3(qmcd, mode):
    """Lock-step at BASELINE configs[1]'s full size in the library's default launch configuration
    (pool, look-ahead in super-blocks, kernel entry qmcd_kernel_sweep_ls) against the oracle's
    literal path 3, every walker, every ratio."""
    wl = inputs.make_config("c1")
    K = 32
    mask = wl.bernoulli_mask(0.5) if mode == "bern0.5" else None
    u = wl.uniforms if mode == "metropolis" else None
    Ao, Bo = wl.A.copy(), wl.Ainv.copy()
    Ro, acco, flo, _ = oracle.run_lockstep(Ao, Bo, K, wl.proposals, mask=mask, uniforms=u)
    g = gpu_sweep(qmcd, wl, K, mask=mask, uniforms=u, lockstep=1)
    assert g["status"] == 0 and g["blocked"]
    if u is not None:
        near_tie = np.abs(u - np.minimum(1.0, Ro * Ro)) < 1e-9            # reading G20
        assert np.array_equal(g["acc"][~near_tie], acco[~near_tie])
    else:
        assert np.array_equal(g["acc"], acco)
    assert _rel(g["R"], Ro) <= RTOL_RATIO
    assert np.max(np.abs(g["B"] - Bo)) <= 1e-9
    assert np.all(flo == wl.n_moves // K) and np.all(g["counters"][:, 1] <= wl.n_moves // K)
    check_residuals(wl, acco, g["B"])
