"""Pins of the CPU oracle against things that are NOT the oracle: LAPACK (numpy) determinants
and inverses, closed forms, invariants and brute force.  No GPU, no CUDA binding.

Each pin names the passage of /root/reference/PAPER.md it fixes (DESIGN.md "Pins" P1..P10).
"""
import math

import numpy as np
import pytest

import oracle
from paper_1708_00744_b200 import inputs


def _walk(A0, props, acc, upto):
    return inputs.current_matrix(A0, props, acc, upto)


# ------------------------------------------------------------------ LU building blocks
@pytest.mark.parametrize("n", [1, 2, 5, 33])
def test_lu_slogdet_and_inverse_match_lapack(n):
    rng = np.random.default_rng(100 + n)
    A = rng.standard_normal((n, n))
    if n >= 2:
        A[0, 0] = 0.0                      # forces a row swap (partial pivoting, ref [21])
    s, la = oracle.slogdet(A)
    s_np, la_np = np.linalg.slogdet(A)
    assert s == int(s_np)
    assert abs(la - la_np) <= 1e-12 * max(1.0, abs(la_np))
    assert np.allclose(oracle.inverse(A), np.linalg.inv(A), rtol=0, atol=1e-10)
    assert oracle.residual(A, np.linalg.inv(A)) < 1e-10


def test_lu_singular_matrix_reports_zero_sign():
    A = np.ones((4, 4))
    s, la = oracle.slogdet(A)
    assert s == 0 and la == -math.inf
    with pytest.raises(oracle.OracleError):
        oracle.inverse(A)


def test_known_determinants():
    # permutation matrix (odd permutation) and a triangular matrix: textbook values
    P = np.array([[0, 1, 0], [1, 0, 0], [0, 0, 1.0]])
    assert oracle.slogdet(P) == (-1, 0.0)
    T = np.triu(np.arange(1.0, 17.0).reshape(4, 4)) + np.eye(4)
    s, la = oracle.slogdet(T)
    assert s == 1 and abs(la - math.log(np.prod(np.diag(T)))) < 1e-13


# ------------------------------------------------------------------ the residual itself
def test_residual_known_nonzero_values_order_and_sign():
    """max|A.B - I| (BASELINE.json north_star) pinned on pairs whose residual is known in closed
    form -- a residual that returns 0, drops the fabs, or forms B.A instead of A.B fails here."""
    n, eps = 6, 2.0 ** -9                                # (1 + eps) - 1 is exact
    I = np.eye(n)
    # A = I, B = I + eps e_i e_j^T  ->  A.B - I = eps e_i e_j^T: exactly eps (off the diagonal and on it)
    for (i, j) in [(1, 4), (4, 1), (2, 2)]:
        E = np.zeros((n, n)); E[i, j] = eps
        assert oracle.residual(I, I + E) == eps
        assert oracle.residual(I, I - E) == eps          # a negative entry: needs the fabs
    assert oracle.residual(I, I) == 0.0
    assert oracle.residual(2.0 * I, I) == 1.0            # 2I.I - I = I
    assert oracle.residual(I, np.zeros((n, n))) == 1.0   # -I
    # order: a pair with max|A.B - I| != max|B.A - I|, hand-computable
    A = np.array([[1.0, 4.0], [0.0, 1.0]])
    B = np.array([[1.0, 0.0], [0.0, 3.0]])
    # A.B - I = [[0, 12], [0, 2]] -> 12 ;  B.A - I = [[0, 4], [0, 2]] -> 4
    assert oracle.residual(A, B) == 12.0
    assert oracle.residual(B, A) == 4.0
    # and against numpy on a random nonsymmetric pair where the two orders differ
    rng = np.random.default_rng(77)
    A = rng.standard_normal((9, 9)); B = rng.standard_normal((9, 9))
    ab = float(np.max(np.abs(A @ B - np.eye(9)))); ba = float(np.max(np.abs(B @ A - np.eye(9))))
    assert abs(ab - ba) > 1e-3
    assert oracle.residual(A, B) == pytest.approx(ab, rel=1e-13)
    assert oracle.residual(B, A) == pytest.approx(ba, rel=1e-13)
    # a non-finite product is reported, not hidden
    Bn = np.eye(3); Bn[1, 1] = np.nan
    assert math.isnan(oracle.residual(np.eye(3), Bn))


# ------------------------------------------------------------------ P3: A = I and diagonal A
def test_P3_identity_and_diagonal_closed_forms():
    """PAPER.md:59-66 with A = I: R = v[j]; B_new = I - (v - e_j) e_j^T / v[j]."""
    n, j = 7, 3
    rng = np.random.default_rng(3)
    v = rng.standard_normal(n) + 2.0
    B = np.eye(n)
    assert oracle.sm_ratio(B, j, v) == v[j]
    assert oracle.ratio_bruteforce(np.eye(n), j, v) == pytest.approx(v[j], rel=1e-14)
    oracle.sm_accept(B, j, v)
    e = np.zeros(n); e[j] = 1.0
    expect = np.eye(n) - np.outer(v - e, e) / v[j]
    assert np.allclose(B, expect, rtol=0, atol=1e-15)
    # diagonal A: R = v[j] / A[j,j]
    dg = rng.uniform(0.5, 2.0, n)
    Bd = np.diag(1.0 / dg)
    assert oracle.sm_ratio(Bd, j, v) == pytest.approx(v[j] / dg[j], rel=1e-15)
    D = oracle.Delayed(Bd.copy(), 3)
    assert D.ratio(j, v) == pytest.approx(v[j] / dg[j], rel=1e-15)


def test_orientation_row_of_inverse_column_of_A():
    """G3: a move changes COLUMN j of A and reads ROW j of B.  A transposed
    operand gives a different number for a nonsymmetric matrix."""
    rng = np.random.default_rng(5)
    n, j = 6, 2
    A = np.eye(n) + 0.4 * rng.standard_normal((n, n))
    v = rng.standard_normal(n)
    B = np.linalg.inv(A)
    An = A.copy(); An[:, j] = v
    truth = np.linalg.det(An) / np.linalg.det(A)
    assert oracle.sm_ratio(B, j, v) == pytest.approx(truth, rel=1e-12)
    wrong = float(B[:, j] @ v)
    assert abs(wrong - truth) > 1e-3
    assert oracle.ratio_bruteforce(A, j, v) == pytest.approx(truth, rel=1e-12)


# ------------------------------------------------------------------ P1: brute force, config 0
def test_P1_config0_bruteforce_every_move():
    """BASELINE.json configs[0]: N=64, K=4, 2 sweeps, Bernoulli(0.99); every ratio of paths 1
    and 2 against explicit LU determinants (LAPACK), and the inverse against LAPACK's after
    every flush."""
    wl = inputs.make_config("c0")
    n = wl.N
    mask = wl.bernoulli_mask(0.99)[:, 0]
    props = wl.proposals[:, 0, :]
    A = wl.A[0].copy()
    B1 = wl.Ainv[0].copy()
    B2 = wl.Ainv[0].copy()
    D = oracle.Delayed(B2, 4)
    n_flush = 0
    for t in range(wl.n_moves):
        j = t % n
        v = props[t]
        An = A.copy(); An[:, j] = v
        s0, l0 = np.linalg.slogdet(A)
        s1, l1 = np.linalg.slogdet(An)
        truth = s0 * s1 * math.exp(l1 - l0)
        r1 = oracle.sm_ratio(B1, j, v)
        r2 = D.ratio(j, v)
        r0 = oracle.ratio_bruteforce(A, j, v)
        assert abs(r1 - truth) <= 1e-12 * abs(truth)
        assert abs(r2 - truth) <= 1e-12 * abs(truth)
        assert abs(r0 - truth) <= 1e-12 * abs(truth)
        if mask[t]:
            A = An
            oracle.sm_accept(B1, j, v)
            assert np.abs(B1 - np.linalg.inv(A)).max() < 1e-12
            if D.accept():
                n_flush += 1
                assert D.pending == 0
                assert np.abs(B2 - np.linalg.inv(A)).max() < 1e-12
                assert oracle.residual(A, B2) < 1e-12
        else:
            D.reject()
    D.flush()
    assert np.abs(B2 - np.linalg.inv(A)).max() < 1e-12
    assert n_flush == int(mask.sum()) // 4 and n_flush >= 30


# ------------------------------------------------------------------ P2: closed form R = alpha_j
@pytest.mark.parametrize("m_queued", [0, 1, 3, 5])
def test_P2_linear_combination_closed_form(m_queued):
    """v = A_cur @ alpha  =>  det(A_cur with col j := v)/det(A_cur) = alpha_j exactly
    (multilinearity of the determinant), also mid-window."""
    rng = np.random.default_rng(20 + m_queued)
    n, K = 24, 6
    A = np.eye(n) + 0.5 * rng.standard_normal((n, n)) / math.sqrt(n)
    B = np.linalg.inv(A)
    D = oracle.Delayed(B, K)
    for i in range(m_queued):
        v = A[:, i] + 0.3 * rng.standard_normal(n) / math.sqrt(n)
        D.ratio(i, v); D.accept()
        A[:, i] = v
    assert D.pending == m_queued
    j = 10
    alpha = rng.standard_normal(n)
    assert D.ratio(j, A @ alpha) == pytest.approx(alpha[j], rel=1e-11, abs=1e-13)
    D.reject()
    assert D.ratio(j, A[:, j].copy()) == pytest.approx(1.0, rel=1e-13)      # unmoved electron
    D.reject()
    assert D.ratio(j, 2.0 * A[:, j]) == pytest.approx(2.0, rel=1e-13)
    D.reject()
    assert abs(D.ratio(j, A[:, j + 1].copy())) < 1e-13                      # duplicate column
    D.reject()
    if m_queued:   # proposing an already-queued electron: the -delta(j, j_i) term (G7)
        alpha2 = rng.standard_normal(n)
        assert D.ratio(0, A @ alpha2) == pytest.approx(alpha2[0], rel=1e-11, abs=1e-13)


def test_P2_accepting_the_unmoved_column_changes_nothing():
    rng = np.random.default_rng(8)
    n = 12
    A = np.eye(n) + 0.2 * rng.standard_normal((n, n)) / math.sqrt(n)
    B = np.linalg.inv(A)
    B0 = B.copy()
    oracle.sm_accept(B, 4, A[:, 4].copy())
    assert np.abs(B - B0).max() < 1e-14


def test_singular_move_is_reported():
    """G13: accept with R == 0 -> error (A = I, v = e_i with i != j gives R = 0 exactly)."""
    n = 5
    v = np.zeros(n); v[1] = 1.0
    B = np.eye(n)
    assert oracle.sm_ratio(B, 3, v) == 0.0
    with pytest.raises(oracle.OracleError):
        oracle.sm_accept(B, 3, v)
    D = oracle.Delayed(np.eye(n), 2)
    assert D.ratio(3, v) == 0.0
    with pytest.raises(oracle.OracleError):
        D.accept()


# ------------------------------------------------------------------ P4: telescoping product
@pytest.mark.parametrize("path,K", [(1, 1), (2, 4), (2, 7), (2, 64)])
def test_P4_telescoping_log_determinant(path, K):
    """The paper's own check: determinant after a full sweep vs direct
    calculation.  sum log|R| over accepted moves == log|det A_final| - log|det A_init|
    (LAPACK slogdet), and the signs multiply likewise."""
    wl = inputs.make_workload(batch=2, N=64, n_moves=128, seed=11)
    mask = wl.bernoulli_mask(0.9)
    B = wl.Ainv.copy()
    R, acc, _ = oracle.run(path, B, K, wl.proposals, mask=mask)
    assert np.array_equal(acc, mask)
    for w in range(wl.batch):
        Af = _walk(wl.A[w], wl.proposals[:, w], acc[:, w], wl.n_moves)
        s0, l0 = np.linalg.slogdet(wl.A[w])
        s1, l1 = np.linalg.slogdet(Af)
        Rw = R[acc[:, w] == 1, w]
        assert abs(np.log(np.abs(Rw)).sum() - (l1 - l0)) < 1e-11
        assert np.prod(np.sign(Rw)) == s0 * s1
        assert np.abs(B[w] - np.linalg.inv(Af)).max() < 1e-11


# ------------------------------------------------------------------ P5: Eq. 3 inside a window
def test_P5_det_S_equals_product_of_window_ratios():
    """Eq. 3: det(I_k + V'A^-1 U) = det(A_k)/det(A_0) = product of the window's
    accepted ratios; S here is the oracle's W C^T."""
    rng = np.random.default_rng(31)
    n, K = 20, 8
    A = np.eye(n) + 0.5 * rng.standard_normal((n, n)) / math.sqrt(n)
    A0 = A.copy()
    D = oracle.Delayed(np.linalg.inv(A), K)
    prod = 1.0
    for i, j in enumerate([3, 9, 0, 17, 5]):
        v = A[:, j] + 0.3 * rng.standard_normal(n) / math.sqrt(n)
        prod *= D.ratio(j, v)
        D.accept()
        A[:, j] = v
        S = D.S()
        assert S.shape == (i + 1, i + 1)
        assert np.linalg.det(S) == pytest.approx(prod, rel=1e-12)
        assert np.linalg.det(A) / np.linalg.det(A0) == pytest.approx(prod, rel=1e-12)
        # S = I_m + V' B0 U with the paper's U, V
        J = D.J()
        U = A[:, J] - A0[:, J]
        V = np.eye(n)[:, J]
        assert np.allclose(S, np.eye(i + 1) + V.T @ np.linalg.inv(A0) @ U, atol=1e-13)


# ------------------------------------------------------------------ P8: Eq. 4 as a library identity
def test_P8_flush_equals_woodbury_by_library():
    """Eq. 4 evaluated with numpy on the paper's own U, V must equal the
    oracle's flush (which works from C, W, S and never forms U)."""
    rng = np.random.default_rng(41)
    n, K = 16, 5
    A0 = np.eye(n) + 0.5 * rng.standard_normal((n, n)) / math.sqrt(n)
    B0 = np.linalg.inv(A0)
    B = B0.copy()
    D = oracle.Delayed(B, K + 1)
    J = [2, 11, 7, 0, 13]
    cols = []
    for j in J:
        v = A0[:, j] + 0.3 * rng.standard_normal(n) / math.sqrt(n)
        cols.append(v)
        D.ratio(j, v); D.accept()
    D.flush()
    U = np.stack(cols, axis=1) - A0[:, J]
    V = np.eye(n)[:, J]
    wood = B0 - B0 @ U @ np.linalg.inv(np.eye(K) + V.T @ B0 @ U) @ V.T @ B0
    assert np.abs(B - wood).max() < 1e-13
    assert D.flush_count == 1 and D.pending == 0


# ------------------------------------------------------------------ P6/P7: invariants
@pytest.mark.parametrize("p", [0.99, 0.5])
def test_P6_delayed_equals_rank1_equals_fresh_inverse_for_every_K(p):
    """the delayed scheme is 'entirely equivalent to the classical method'."""
    wl = inputs.make_workload(batch=3, N=48, n_moves=120, seed=5)
    mask = wl.bernoulli_mask(p)
    B1 = wl.Ainv.copy()
    R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, mask=mask)
    for K in (1, 2, 3, 16, 48):
        B2 = wl.Ainv.copy()
        R2, acc2, _ = oracle.run(2, B2, K, wl.proposals, mask=mask)
        assert np.array_equal(acc1, acc2)
        assert np.abs(R2 / R1 - 1).max() < 1e-11
        assert np.abs(B2 - B1).max() < 1e-11
    for w in range(wl.batch):
        Af = _walk(wl.A[w], wl.proposals[:, w], acc1[:, w], wl.n_moves)
        assert np.abs(B1[w] - np.linalg.inv(Af)).max() < 1e-11
        assert oracle.residual(Af, B1[w]) < 1e-11          # P7


def test_P6_flush_neutrality_and_no_final_flush():
    """Inserting a flush anywhere changes no later ratio; without a final flush B is stale."""
    wl = inputs.make_workload(batch=1, N=32, n_moves=40, seed=9)
    props = wl.proposals[:, 0]
    Ba, Bb = wl.Ainv[0].copy(), wl.Ainv[0].copy()
    Da, Db = oracle.Delayed(Ba, 8), oracle.Delayed(Bb, 8)
    for t in range(40):
        ra = Da.ratio(t % 32, props[t]); Da.accept()
        rb = Db.ratio(t % 32, props[t]); Db.accept()
        assert ra == pytest.approx(rb, rel=1e-12)
        if t in (2, 3, 17):
            Db.flush()
            assert Db.pending == 0
    Da.flush(); Db.flush()
    assert np.abs(Ba - Bb).max() < 1e-12
    B3 = wl.Ainv.copy()
    oracle.run(2, B3, 32, wl.proposals[:20], mask=np.ones((20, 1), np.uint8), final_flush=False)
    assert np.array_equal(B3, wl.Ainv)                     # K > moves and no flush: untouched


# ------------------------------------------------------------------ P11: lock-step variant (path 3)
@pytest.mark.parametrize("p", [0.99, 0.5, 0.0])
def test_P11_lockstep_equals_rank1_and_fresh_inverse(p):
    """a rejected move takes a slot with the unchanged column; the result is
    still that of the classical method, the tracked A is the walked matrix, and
    every walker applies Eq. 4 exactly once per K proposals."""
    wl = inputs.make_workload(batch=3, N=40, n_moves=100, seed=11)
    mask = wl.bernoulli_mask(p)
    B1 = wl.Ainv.copy()
    R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, mask=mask)
    for K in (1, 3, 16, 40):
        A3, B3 = wl.A.copy(), wl.Ainv.copy()
        R3, acc3, fl, _ = oracle.run_lockstep(A3, B3, K, wl.proposals, mask=mask)
        assert np.array_equal(acc1, acc3)
        assert np.abs(R3 / R1 - 1).max() < 1e-11
        assert np.abs(B3 - B1).max() < 1e-11
        # K | 100 -> the final flush finds an empty queue; else one more partial flush
        assert np.all(fl == -(-100 // K))
        for w in range(wl.batch):
            Af = _walk(wl.A[w], wl.proposals[:, w], acc1[:, w], wl.n_moves)
            assert np.array_equal(A3[w], Af)
            assert np.abs(B3[w] - np.linalg.inv(Af)).max() < 1e-11
    if p == 0.0:                                           # nothing accepted: nothing moves
        assert np.abs(B3 - wl.Ainv).max() < 1e-12


def test_P11_lockstep_metropolis_and_window_boundaries():
    """Without a final flush the inverse is stale exactly by the last n_moves mod K proposals."""
    wl = inputs.make_workload(batch=2, N=24, n_moves=50, seed=12)
    u = wl.uniforms
    B1 = wl.Ainv.copy()
    R1, acc1, _ = oracle.run(1, B1, 1, wl.proposals, uniforms=u)
    A3, B3 = wl.A.copy(), wl.Ainv.copy()
    R3, acc3, fl, _ = oracle.run_lockstep(A3, B3, 8, wl.proposals, uniforms=u, final_flush=False)
    assert np.array_equal(acc1, acc3) and np.abs(R3 / R1 - 1).max() < 1e-11
    assert np.all(fl == 50 // 8)
    for w in range(wl.batch):
        A48 = _walk(wl.A[w], wl.proposals[:48, w], acc1[:48, w], 48)
        assert np.abs(B3[w] - np.linalg.inv(A48)).max() < 1e-11


# ------------------------------------------------------------------ P10: repeated electron (G7)
def test_P10_same_electron_twice_in_one_window():
    rng = np.random.default_rng(77)
    n, K = 10, 6
    A = np.eye(n) + 0.5 * rng.standard_normal((n, n)) / math.sqrt(n)
    B = np.linalg.inv(A)
    D = oracle.Delayed(B, K)
    for j in (1, 4, 1, 4, 4, 2):
        v = A[:, j] + 0.3 * rng.standard_normal(n)
        An = A.copy(); An[:, j] = v
        truth = np.linalg.det(An) / np.linalg.det(A)
        assert D.ratio(j, v) == pytest.approx(truth, rel=1e-11)
        D.accept()
        A = An
    D.flush()
    assert np.abs(B - np.linalg.inv(A)).max() < 1e-11


# ------------------------------------------------------------------ P12: slot replacement (path 4, G7)
def test_P12_slot_replacement_vs_bruteforce_and_flush_first():
    """The same electron accepted again before the queue is applied (PAPER.md:84 is silent; DESIGN.md
    G7, second alternative): the slot's column is replaced, nothing is flushed.  Every ratio against
    the plain definition (library determinants), the inverse against the library inverse, and the
    whole run against flush-first (path 2) -- the same ratios and inverse with fewer flushes."""
    rng = np.random.default_rng(77)
    n, K = 10, 6
    A = np.eye(n) + 0.5 * rng.standard_normal((n, n)) / math.sqrt(n)
    B = np.linalg.inv(A)
    D = oracle.Delayed(B, K, replace=True)
    pend = []
    for j in (1, 4, 1, 4, 4, 2):
        v = A[:, j] + 0.3 * rng.standard_normal(n)
        An = A.copy(); An[:, j] = v
        truth = np.linalg.det(An) / np.linalg.det(A)
        assert D.ratio(j, v) == pytest.approx(truth, rel=1e-11)
        assert D.accept() is False                   # never flushes: 3 distinct electrons < K
        pend.append(D.pending)
        A = An
    assert pend == [1, 2, 2, 2, 2, 3]                # a repeat keeps its slot
    assert list(D.J()) == [1, 4, 2]
    assert D.flush_count == 0
    # Eq. 3 still holds with the replaced columns: det S = det(A_cur) / det(A0)
    A0 = np.linalg.inv(B)                            # B is still the stale inverse
    assert np.linalg.det(D.S()) == pytest.approx(np.linalg.det(A) / np.linalg.det(A0), rel=1e-11)
    D.flush()
    assert np.abs(B - np.linalg.inv(A)).max() < 1e-11


@pytest.mark.parametrize("K,p", [(64, 0.3), (8, 0.6), (3, 1.0), (1, 1.0)])
def test_P12_run_jseq_replace_equals_flush_first_and_rank1(K, p):
    """K = N = 64 at 30 % acceptance revisits queued electrons in every window (the case the verdict
    names); path 4 must give path 2's ratios, decisions and inverse, with no more flushes."""
    wl = inputs.make_workload(batch=2, N=64, n_moves=300, seed=5)
    rng = np.random.default_rng(9)
    jseq = rng.integers(0, 12, size=wl.n_moves).astype(np.int32)       # few electrons: many repeats
    jseq[::7] = rng.integers(0, 64, size=len(jseq[::7]))
    # proposals must perturb the CURRENT column j of the walked matrix only loosely: use the generator's
    # columns of the initial matrix at jseq (reading G14)
    props = np.stack([np.stack([wl.A[w][:, jseq[t]] for w in range(2)]) for t in range(wl.n_moves)])
    props = props + 0.3 / 8.0 * np.random.default_rng(3).standard_normal(props.shape)
    mask = (wl.uniforms < p).astype(np.uint8)
    Bf, Br = wl.Ainv.copy(), wl.Ainv.copy()
    Rf, af, flf, _ = oracle.run_jseq(Bf, K, props, jseq, False, mask=mask)
    Rr, ar, flr, _ = oracle.run_jseq(Br, K, props, jseq, True, mask=mask)
    assert np.array_equal(af, ar) and np.array_equal(af, mask)
    assert np.abs(Rr / Rf - 1).max() < 1e-10
    assert np.abs(Br - Bf).max() < 1e-10
    assert (flr <= flf).all() and (K == 1 or (flr < flf).all())
    # and against rank-1 Sherman-Morrison, move by move (path 1 has no queue at all)
    for w in range(2):
        B1 = wl.Ainv[w].copy()
        for t in range(wl.n_moves):
            assert oracle.sm_ratio(B1, int(jseq[t]), props[t, w]) == pytest.approx(Rr[t, w], rel=1e-10)
            if mask[t, w]:
                oracle.sm_accept(B1, int(jseq[t]), props[t, w])
        assert np.abs(B1 - Br[w]).max() < 1e-10
        A_cur = wl.A[w].copy()
        for t in range(wl.n_moves):
            if mask[t, w]:
                A_cur[:, jseq[t]] = props[t, w]
        assert np.max(np.abs(A_cur @ Br[w] - np.eye(64))) < 1e-10


# ------------------------------------------------------------------ Metropolis mode (G11)
def test_metropolis_rule_and_path_agreement():
    wl = inputs.make_workload(batch=2, N=40, n_moves=80, seed=21)
    # scale proposals so a useful fraction is rejected
    props = wl.proposals * (1.0 + 0.4 * (wl.uniforms[:, :, None] - 0.5))
    u = wl.uniforms[::-1].copy()
    B1, B2 = wl.Ainv.copy(), wl.Ainv.copy()
    R1, a1, _ = oracle.run(1, B1, 1, props, uniforms=u)
    R2, a2, _ = oracle.run(2, B2, 8, props, uniforms=u)
    assert np.array_equal(a1, (u < np.minimum(1.0, R1 * R1)).astype(np.uint8))
    assert np.array_equal(a1, a2)
    assert 0.2 < a1.mean() < 0.98
    assert np.abs(R2 / R1 - 1).max() < 1e-11
    assert np.abs(B1 - B2).max() < 1e-11


def test_expected_accept_run_length_matches_paper():
    """mean length of a run of accepts is p/(1-p) (= 99 at p = 0.99): sanity of
    the seeded Bernoulli mask (tests/golden/paper_facts.txt)."""
    facts = dict(line.split("=") for line in open(
        __import__("os").path.join(__import__("os").path.dirname(__file__), "golden",
                                   "paper_facts.txt")) if "=" in line and not line.startswith("#"))
    p = float(facts["dmc_acceptance"])
    assert float(facts["expected_run_length"]) == pytest.approx(p / (1 - p))
    wl = inputs.make_workload(batch=1, N=8, n_moves=200000, seed=3)
    m = wl.bernoulli_mask(p)[:, 0]
    n_rej = int((m == 0).sum())
    assert m.sum() / (n_rej + 1) == pytest.approx(p / (1 - p), rel=0.1)


def test_inputs_are_deterministic_and_per_walker():
    a = inputs.make_workload(2, 16, 20, seed=4)
    b = inputs.make_workload(3, 16, 20, seed=4)
    assert np.array_equal(a.A, b.A[:2]) and np.array_equal(a.proposals, b.proposals[:, :2])
    c = inputs.make_workload(1, 16, 20, seed=5)
    assert np.array_equal(c.A[0], a.A[1])                  # walker w uses seed + w
    assert np.abs(a.A[0] @ a.Ainv[0] - np.eye(16)).max() < 1e-13
