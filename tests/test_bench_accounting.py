"""Host-side checks of bench.py's accounting (no GPU): the algorithmic flops / bytes per step are
the per-unit figures of DESIGN.md section 7 applied to the accept sequence."""
import importlib.util
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(spec)
spec.loader.exec_module(bench)


def test_algorithmic_work_all_accepted_full_windows():
    N, K, n_moves, batch = 64, 4, 16, 2
    acc = np.ones((n_moves, batch), dtype=np.uint8)
    w = bench.algorithmic_work(acc, N, K)
    # every window: queue lengths 0..K-1 at the proposals, one rank-K flush
    windows = n_moves // K * batch
    ratio_flops = windows * sum(2.0 * N * (2 * m + 1) + 2.0 * m * m for m in range(K))
    ratio_bytes = windows * sum(8.0 * N * (2 * m + 2) + 8.0 * m * m for m in range(K))
    flush_flops = windows * (4.0 * N * N * K + 2.0 * K * K * N)
    flush_bytes = windows * (16.0 * N * N + 24.0 * K * N)
    assert w["flushes"] == windows
    assert w["ratio_flops"] == ratio_flops and w["ratio_bytes"] == ratio_bytes
    assert w["flush_flops"] == flush_flops and w["flush_bytes"] == flush_bytes
    assert w["accept_flops"] == windows * sum(4.0 * m * m for m in range(K))
    assert w["flops"] == ratio_flops + flush_flops + w["accept_flops"]


def test_algorithmic_work_rejections_and_final_partial_flush():
    N, K = 32, 4
    acc = np.array([[1], [0], [1], [1], [0], [1], [1]], dtype=np.uint8)    # 5 accepts: one full window + 1
    w = bench.algorithmic_work(acc, N, K)
    assert w["flushes"] == 2                                   # rank 4, then the final rank-1 flush
    assert w["flush_flops"] == (4.0 * N * N * 4 + 2.0 * 16 * N) + (4.0 * N * N * 1 + 2.0 * 1 * N)
    # queue lengths seen by the 7 proposals: 0,1,1,2,3,3,0
    ms = [0, 1, 1, 2, 3, 3, 0]
    assert w["ratio_bytes"] == sum(8.0 * N * (2 * m + 2) + 8.0 * m * m for m in ms)


def test_k1_is_sherman_morrison_traffic():
    N = 128
    acc = np.ones((10, 1), dtype=np.uint8)
    w = bench.algorithmic_work(acc, N, 1)
    assert w["flushes"] == 10 and w["flush_bytes"] == 10 * (16.0 * N * N + 24.0 * N)


def test_mode_inputs_and_config_names():
    from paper_1708_00744_b200 import inputs
    wl = inputs.make_workload(2, 16, 8, seed=1)
    m, u = bench.mode_inputs(wl, "bern0.5")
    assert u is None and m.shape == (8, 2) and set(np.unique(m)) <= {0, 1}
    m, u = bench.mode_inputs(wl, "metropolis")
    assert m is None and np.array_equal(u, wl.uniforms)
    m, u = bench.mode_inputs(wl, "bern0.99", 5)            # the bounded sample of the oracle / K = 1 legs
    assert m.shape == (5, 2) and np.array_equal(m, wl.bernoulli_mask(0.99)[:5])
    assert bench.sample_moves(4096, 64) == 128 and bench.sample_moves(4096, 256) == 512 and bench.sample_moves(100, 64) == 100
    assert bench.DEFAULT_CONFIG in ("c3", "c4")          # the headline is a large configuration
    assert set(inputs.CONFIGS) == {"c0", "c1", "c2", "c3", "c4"}


def test_lockstep_accounting_flushes_every_K_proposals():
    """one flush per window of K proposals, rank = accepts in it; none if empty."""
    N, K = 16, 4
    acc = np.array([[1, 0, 0, 0,  0, 0, 0, 0,  1, 1, 1, 1,  1, 0]], dtype=np.uint8).T
    w = bench.algorithmic_work(acc, N, K, lockstep=True)
    assert w["flushes"] == 3                      # ranks 1, (empty), 4, and the final partial 1
    assert w["flush_flops"] == sum(4.0 * N * N * m + 2.0 * m * m * N for m in (1, 4, 1))
    w2 = bench.algorithmic_work(acc, N, K, lockstep=False)
    assert w2["flushes"] == 2                     # ranks 4 and 2
