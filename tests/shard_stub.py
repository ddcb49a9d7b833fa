"""A numpy stand-in for `binding.ShardPlan` (same methods), used by the CPU test of the sharded-mode HOST PROTOCOL
(tests/test_shard_protocol_gloo.py: world_size 2 over gloo).  TEST INFRASTRUCTURE: it shares no code with the CUDA
path; it restates the paper's scheme with one process per block, written densely:

  shard r owns rows lo..hi-1 of  T psi' = T^dagger psi  (Eq. 4); its last row J_r = hi-1 is its joint line
  (PAPER.md:90-94), the rows before it are its interior I.  With A = T[I, I]:
      psi'_I = y - psi'_{J_{r-1}} u - psi'_{J_r} v,   y = A^-1 d_I,  u = A^-1 (b e_first),  v = A^-1 (c e_last)     (SS)
  and row J_r becomes one row of the reduced system on the joint lines (RS):
      (-b u_last) X_{r-1} + (a_J - b v_last - c u'_first) X_r + (-c v'_first) X_{r+1} = d_J - b y_last - c y'_first
  (primed: the next shard).  What a process sends: FOUR matrix values once ("collecting four values per
  process") and, the matrix being pre-factored, TWO right-hand-side values per step; it gets the support values
  X_{r-1}, X_r back -- here from the reduced system solved redundantly by every process.
The explicit half-step d = T^dagger psi (Eq. 3) needs psi on the rows next to the shard: the row above is the previous
shard's joint line (its old value is the previous step's support value, or the exchanged edge value before step 1);
the row below the joint belongs to the next shard, which therefore sends conj(c) psi_first inside its second value.
"""
import numpy as np


class NumpyShard:
    def __init__(self, N_local, dx, dt, V_local, shard, nshards):
        self.n, self.r, self.S = N_local, shard, nshards
        s = dt / (4 * dx * dx)
        self.b = self.c = -1j * s                                   # off-diagonals of T (reading R3)
        self.a = 1 + 1j * (2 * s + 0.5 * dt * np.asarray(V_local, float))
        ni = N_local - 1                                            # interior rows
        A = np.diag(self.a[:ni]) + np.diag(np.full(ni - 1, self.b), -1) + np.diag(np.full(ni - 1, self.c), 1)
        self.Ainv = np.linalg.inv(A)
        e0, e1 = np.zeros(ni, complex), np.zeros(ni, complex)
        e0[0], e1[-1] = self.b if shard > 0 else 0.0, self.c
        self.u, self.v = self.Ainv @ e0, self.Ainv @ e1
        self.above_old = 0.0                                        # old psi on the row above this shard
        self.pending = None                                         # (y, d_J without its psi_{J+1} term)

    def counts(self):
        return 4, 2

    # ---- matrix side -------------------------------------------------------------------------------------------
    def factorize_local(self, send):
        rec = send.numpy()
        rec[0] = -self.b * self.u[-1]                               # sub of my joint row
        rec[1] = self.a[-1] - self.b * self.v[-1]                   # my part of its diagonal
        rec[2] = -self.c * self.u[0] if self.r > 0 else 0.0         # what I add to the diagonal of the joint above
        rec[3] = -self.c * self.v[0] if self.r > 0 else 0.0         # its coupling to my joint

    def factorize_finish(self, gathered):
        g = gathered.numpy().reshape(self.S, 4)
        M = np.zeros((self.S, self.S), complex)
        for r in range(self.S):
            M[r, r] = g[r, 1] + (g[r + 1, 2] if r + 1 < self.S else 0.0)
            if r > 0:
                M[r, r - 1] = g[r, 0]
            if r + 1 < self.S:
                M[r, r + 1] = g[r + 1, 3]
        self.Minv = np.linalg.inv(M)

    # ---- one run -----------------------------------------------------------------------------------------------
    def edge(self, psi, edge):
        edge.numpy()[0] = psi.numpy()[-1]

    def _reduce(self, psi, send):
        x = psi.numpy()
        lo = np.concatenate([[self.above_old], x[:-1]])
        hi = np.concatenate([x[1:], [0.0]])                         # the joint row's psi_{J+1} term comes from the next shard
        d = np.conj(self.b) * lo + np.conj(self.a) * x + np.conj(self.c) * hi
        y = self.Ainv @ d[:-1]
        rec = send.numpy()
        rec[0] = d[-1] - self.b * y[-1]                                                # JD
        rec[1] = (np.conj(self.c) * x[0] - self.c * y[0]) if self.r > 0 else 0.0       # JU (to the joint above)
        self.pending = y

    def _substitute(self, psi, gathered):
        g = gathered.numpy().reshape(self.S, 2)
        rhs = np.array([g[r, 0] + (g[r + 1, 1] if r + 1 < self.S else 0.0) for r in range(self.S)])
        X = self.Minv @ rhs                                          # RS, replicated
        xa = X[self.r - 1] if self.r > 0 else 0.0
        x = psi.numpy()
        x[:-1] = self.pending - xa * self.u - X[self.r] * self.v     # SS
        x[-1] = X[self.r]
        self.above_old = xa

    def prologue(self, psi, edges, send):
        self.above_old = edges.numpy()[self.r - 1] if self.r > 0 else 0.0
        self._reduce(psi, send)

    def advance(self, psi, gathered, send):
        self._substitute(psi, gathered)
        self._reduce(psi, send)

    def epilogue(self, psi, gathered):
        self._substitute(psi, gathered)
