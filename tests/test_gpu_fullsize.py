"""Full-size parity matrix: every (config, acceptance mode) of BASELINE.json c2, c3, c4
runs the ORACLE once, over the WHOLE run, on sampled walkers (path 2 at one K: ratios and decisions do not
depend on K), and EVERY K of that config's list is compared with it element by element in the
launch configuration bench.py times (library defaults): identical accept sequence, every ratio to
relative error <= 1e-10, the final inverse to 1e-10, max|A.Ainv - I| <= 1e-8 (north_star).
No comparison here is GPU against GPU.  c4 additionally checks the residual after every launch of K
proposals (BASELINE.json configs[4]: "max|A.Ainv - I| checked after every flush")."""
import numpy as np
import pytest

import oracle
from paper_1708_00744_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL_RATIO = 1e-10
SAMPLED = {"c2": (0, 31, 63), "c3": (0, 13, 31), "c4": (0, 3, 7)}
ORACLE_K = 64

_wl_cache = {}
_or_cache = {}


def _workload(cfg):
    if cfg not in _wl_cache:
        _wl_cache.clear(); _or_cache.clear()          # one full-size workload in host memory at a time
        _wl_cache[cfg] = inputs.make_config(cfg)
    return _wl_cache[cfg]


def _mode_inputs(wl, mode):
    if mode == "metropolis":
        return None, wl.uniforms
    return wl.bernoulli_mask(float(mode[4:])), None


def _oracle(cfg, mode):
    """Oracle path 2 (delayed rank-K, K = 64) over the whole run on the sampled walkers only."""
    key = (cfg, mode)
    if key not in _or_cache:
        wl = _workload(cfg)
        ws = list(SAMPLED[cfg])
        mask, uni = _mode_inputs(wl, mode)
        B = np.ascontiguousarray(wl.Ainv[ws])
        P = np.ascontiguousarray(wl.proposals[:, ws, :])
        R, acc, _ = oracle.run(2, B, ORACLE_K, P, mask=None if mask is None else np.ascontiguousarray(mask[:, ws]),
                               uniforms=None if uni is None else np.ascontiguousarray(uni[:, ws]))
        _or_cache[key] = (R, acc, B)
    return _or_cache[key]


def _residual_device(torch, A0, props, acc_w, upto, B_dev_w, pending=0):
    """max|A_applied . B - I| on the device (torch.matmul is the checker here, not the product path);
    A_applied = the initial matrix with the accepted columns of moves [0, upto) except the last `pending`
    accepted ones (still queued, not yet in B)."""
    N = A0.shape[0]
    idx = np.nonzero(acc_w[:upto])[0]
    if pending:
        idx = idx[:-pending]
    A = A0.copy()
    for t in idx:                                   # later moves of the same electron overwrite earlier ones
        A[:, t % N] = props[t]
    Ad = torch.from_numpy(A).cuda()
    E = Ad @ B_dev_w
    E.diagonal().sub_(1.0)
    return float(E.abs().max())


def _run_gpu(qmcd, wl, K, mask, uni):
    import torch
    q = qmcd.Qmcd(wl.N, K, wl.batch)
    B = torch.from_numpy(wl.Ainv).cuda()
    q.set_inverse(B)
    P = torch.from_numpy(wl.proposals).cuda()
    R = torch.zeros((wl.n_moves, wl.batch), dtype=torch.float64, device="cuda")
    acc = torch.zeros((wl.n_moves, wl.batch), dtype=torch.uint8, device="cuda")
    q.sweep(0, P, mask=None if mask is None else torch.from_numpy(mask).cuda(),
            uniforms=None if uni is None else torch.from_numpy(uni).cuda(), R_out=R, acc_out=acc)
    q.flush()
    st = q.status()[0]
    launch = dict(S=q.get_option("cluster"), pool=q.get_option("pool"), tma=q.get_option("tma"),
                  blocked=q.get_option("blocked_ok") and q.get_option("lookahead") == 0)
    q.close()
    del P
    return R.cpu().numpy(), acc.cpu().numpy(), B, st, launch


def _check_against_oracle(qmcd, cfg, mode, K):
    import torch
    wl = _workload(cfg)
    ws = list(SAMPLED[cfg])
    mask, uni = _mode_inputs(wl, mode)
    Ro, acco, Bo = _oracle(cfg, mode)
    Rg, accg, Bdev, st, launch = _run_gpu(qmcd, wl, K, mask, uni)
    ctx = (cfg, mode, K, launch)
    assert st == 0, ctx
    # accept sequence: identical to the oracle's on the sampled walkers; on every walker it is the mask
    # (Bernoulli) or the Metropolis rule applied to the walker's own ratios, away from ties (reading G20)
    assert np.array_equal(accg[:, ws], acco), ctx
    if mask is not None:
        assert np.array_equal(accg, mask), ctx
    else:
        pa = np.minimum(1.0, Rg * Rg)
        tie = np.abs(uni - pa) < 1e-9
        assert np.array_equal(accg[~tie], (uni < pa)[~tie].astype(np.uint8)), ctx
    rel = np.max(np.abs(Rg[:, ws] - Ro) / np.abs(Ro))
    assert rel <= RTOL_RATIO, (ctx, rel)
    assert np.all(np.isfinite(Rg)), ctx
    for i, w in enumerate(ws):
        Bw = Bdev[w]
        err = float((Bw - torch.from_numpy(Bo[i]).cuda()).abs().max())
        assert err <= 1e-10, (ctx, w, err)
        res = _residual_device(torch, wl.A[w], wl.proposals[:, w, :], accg[:, w], wl.n_moves, Bw)
        assert res <= 1e-8, (ctx, w, res)
    del Bdev
    torch.cuda.empty_cache()


C2 = [(m, K) for m in ("bern0.99", "bern0.5", "metropolis") for K in (1, 16, 32, 64)]
C3 = [("bern0.99", K) for K in (1, 32, 64, 128)]
C4 = [(m, K) for m in ("bern0.99", "bern0.5") for K in (1, 16, 32, 64, 128, 256)]


@pytest.mark.parametrize("mode,K", C2)
def test_c2_full_size_every_K_and_mode_vs_oracle(qmcd, mode, K):
    _check_against_oracle(qmcd, "c2", mode, K)


@pytest.mark.parametrize("mode,K", C3)
def test_c3_full_size_every_K_vs_oracle(qmcd, mode, K):
    _check_against_oracle(qmcd, "c3", mode, K)


@pytest.mark.parametrize("mode,K", C4)
def test_c4_full_size_every_K_and_mode_vs_oracle(qmcd, mode, K):
    _check_against_oracle(qmcd, "c4", mode, K)


@pytest.mark.parametrize("K,every", [(64, 1), (256, 4)])
def test_c4_residual_after_every_flush(qmcd, K, every):
    """BASELINE.json configs[4]: the sweep is cut into launches of K proposals (one flush each at 99 %
    acceptance) and max|A_applied . Ainv - I| <= 1e-8 is checked after each (K = 256: after every 4th) for
    two walkers, A_applied = the accepted moves minus those still queued (qmcd_pending).  PAPER.md:107."""
    import torch
    wl = _workload("c4")
    mask = wl.bernoulli_mask(0.99)
    q = qmcd.Qmcd(wl.N, K, wl.batch)
    B = torch.from_numpy(wl.Ainv).cuda()
    q.set_inverse(B)
    P = torch.from_numpy(wl.proposals).cuda()
    Md = torch.from_numpy(mask).cuda()
    worst, checks, flushes_seen = 0.0, 0, 0
    for i, t0 in enumerate(range(0, wl.n_moves, K)):
        t1 = min(t0 + K, wl.n_moves)
        q.sweep(t0 % wl.N, P[t0:t1], mask=Md[t0:t1])
        if (i + 1) % every:
            continue
        pend = q.pending().cpu().numpy()
        flushes_seen = int(q.counters().cpu().numpy()[:, 1].min())
        for w in (1, 6):
            r = _residual_device(torch, wl.A[w], wl.proposals[:, w, :], mask[:, w], t1, B[w], pending=int(pend[w]))
            worst = max(worst, r); checks += 1
            assert r <= 1e-8, (K, t1, w, r)
    q.flush()
    assert q.status()[0] == 0
    for w in (1, 6):
        assert _residual_device(torch, wl.A[w], wl.proposals[:, w, :], mask[:, w], wl.n_moves, B[w]) <= 1e-8
    assert checks >= 2 * (wl.n_moves // (K * every))
    assert flushes_seen >= (wl.n_moves // K) - 2          # about one flush per launch of K proposals at 99 % acceptance
    q.close()


@pytest.mark.parametrize("N,K,batch,S,n_moves", [
    (8192, 64, 1, 8, 160),       # the paper grid's largest shape: clusters of 8 (1 leader + pool clusters)
    (2048, 64, 1, 16, 200),      # 16 CTAs per leader cluster
    (2048, 256, 1, 16, 300),     # K = 256 on a 16-CTA cluster
    (4096, 128, 2, 4, 300),
])
def test_paper_grid_launch_shapes_vs_oracle(qmcd, N, K, batch, S, n_moves):
    """One parity test per launch shape the paper's own grid runs on:
    one or two walkers spread over large clusters, 100 % acceptance, reduced sweeps."""
    import torch
    wl = inputs.make_workload(batch, N, n_moves, seed=5)
    mask = np.ones((n_moves, batch), dtype=np.uint8)
    Bo = wl.Ainv.copy()
    Ro, acco, _ = oracle.run(2, Bo, K, wl.proposals, mask=mask)
    q = qmcd.Qmcd(N, K, batch)
    q.set_option("cluster", S)
    B = torch.from_numpy(wl.Ainv).cuda()
    q.set_inverse(B)
    R = torch.zeros((n_moves, batch), dtype=torch.float64, device="cuda")
    q.sweep(0, torch.from_numpy(wl.proposals).cuda(), mask=torch.from_numpy(mask).cuda(), R_out=R)
    q.flush()
    assert q.status()[0] == 0 and q.get_option("cluster") == S
    assert np.max(np.abs(R.cpu().numpy() - Ro) / np.abs(Ro)) <= RTOL_RATIO
    assert float((B - torch.from_numpy(Bo).cuda()).abs().max()) <= 1e-10
    q.close()
