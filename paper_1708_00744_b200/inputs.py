"""Seeded synthetic inputs shaped like the paper's / BASELINE.json's workloads.

This module serves BOTH the oracle-side tests and the CUDA path, and therefore
holds none of the method's arithmetic: it only draws random numbers and calls
the library LU inverse once for the initial ``Ainv`` ("Ainv from LU",
BASELINE.json configs[0]).  It imports neither ``oracle`` nor the CUDA binding.

Recipe (BASELINE.json configs; the paper's own test
application used synthetic matrices too):

  per walker w:  seed s_w = seed + w;  SeedSequence(s_w).spawn(3) -> PCG64
                 generators g_A, g_P, g_U
  A      = I + 0.5 * G / sqrt(N),   G = g_A.standard_normal((N, N))
  Ainv   = numpy.linalg.inv(A)                       (library LU)
  move t (sweep s = t // N, electron j = t % N), drawn in t order:
      v_t = A[:, j] + 0.3 * g / sqrt(N),  g = g_P.standard_normal(N)
            (A = the INITIAL matrix: reading G14)
      u_t = g_U.random()
  Bernoulli(p) mode accepts iff u_t < p; Metropolis mode accepts iff
  u_t < min(1, R^2) (decided by whoever computes R).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# BASELINE.json `configs`, in order.  K lists and acceptance modes as given there.
CONFIGS = {
    "c0": dict(batch=1, N=64, sweeps=2, Ks=(4,), modes=("bern0.99",), seed=1),
    "c1": dict(batch=16, N=512, sweeps=4, Ks=(1, 16, 32), modes=("bern0.99",), seed=1),
    "c2": dict(batch=64, N=1024, sweeps=4, Ks=(1, 16, 32, 64),
               modes=("bern0.99", "bern0.5", "metropolis"), seed=1),
    "c3": dict(batch=32, N=2048, sweeps=2, Ks=(1, 32, 64, 128), modes=("bern0.99",), seed=1),
    "c4": dict(batch=8, N=4096, sweeps=1, Ks=(1, 16, 32, 64, 128, 256),
               modes=("bern0.99", "bern0.5"), seed=1),
}


@dataclass
class Workload:
    batch: int
    N: int
    n_moves: int
    seed: int
    A: np.ndarray            # [batch][N][N]  initial Slater matrices
    Ainv: np.ndarray         # [batch][N][N]  library LU inverse of A
    proposals: np.ndarray    # [n_moves][batch][N]  new columns v_t
    uniforms: np.ndarray     # [n_moves][batch]     u_t in [0, 1)
    meta: dict = field(default_factory=dict)

    def electron(self, t: int, j_begin: int = 0) -> int:
        return (j_begin + t) % self.N

    def bernoulli_mask(self, p: float) -> np.ndarray:
        """[n_moves][batch] uint8, 1 iff u_t < p."""
        return (self.uniforms < p).astype(np.uint8)


def make_workload(batch: int, N: int, n_moves: int, seed: int = 1,
                  want_A: bool = True, dtype=np.float64) -> Workload:
    """Generate the tensors of one run.  Deterministic in (batch, N, n_moves, seed);
    walker w's data depend only on (N, n_moves, seed + w)."""
    A = np.empty((batch, N, N), dtype=dtype)
    Ainv = np.empty((batch, N, N), dtype=dtype)
    proposals = np.empty((n_moves, batch, N), dtype=dtype)
    uniforms = np.empty((n_moves, batch), dtype=dtype)
    rs = 1.0 / np.sqrt(N)
    for w in range(batch):
        g_A, g_P, g_U = (np.random.Generator(np.random.PCG64(s))
                         for s in np.random.SeedSequence(seed + w).spawn(3))
        Aw = np.eye(N) + (0.5 * rs) * g_A.standard_normal((N, N))
        A[w] = Aw
        Ainv[w] = np.linalg.inv(Aw)
        AT = np.ascontiguousarray(Aw.T)              # AT[j] = column j of A
        done = 0
        while done < n_moves:                        # (s, j) order == t order
            cnt = min(n_moves - done, max(1, (1 << 22) // N))
            g = g_P.standard_normal((cnt, N))
            js = (np.arange(done, done + cnt)) % N
            proposals[done:done + cnt, w, :] = AT[js] + (0.3 * rs) * g
            done += cnt
        uniforms[:, w] = g_U.random(n_moves)
    return Workload(batch=batch, N=N, n_moves=n_moves, seed=seed,
                    A=A if want_A else None, Ainv=Ainv, proposals=proposals,
                    uniforms=uniforms, meta=dict(recipe="I+0.5G/sqrtN; v=A[:,j]+0.3g/sqrtN"))


def make_config(name: str, sweeps: int | None = None, batch: int | None = None) -> Workload:
    """Workload of BASELINE.json config c0..c4 (optionally with fewer sweeps / walkers,
    for bounded samples -- the caller must say so wherever the result is reported)."""
    cfg = CONFIGS[name]
    s = cfg["sweeps"] if sweeps is None else sweeps
    b = cfg["batch"] if batch is None else batch
    wl = make_workload(b, cfg["N"], s * cfg["N"], seed=cfg["seed"])
    wl.meta.update(config=name, sweeps=s)
    return wl


def current_matrix(A0: np.ndarray, proposals_w: np.ndarray, acc_w: np.ndarray,
                   upto: int, j_begin: int = 0) -> np.ndarray:
    """A_cur of ONE walker after moves [0, upto): the initial matrix with column j_t
    overwritten by v_t at every accepted move (bookkeeping only -- used for residual
    checks, holds no arithmetic of the method)."""
    N = A0.shape[0]
    A = A0.copy()
    for t in range(upto):
        if acc_w[t]:
            A[:, (j_begin + t) % N] = proposals_w[t]
    return A
