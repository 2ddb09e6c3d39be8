"""Exact enumeration on tiny tori, written from the model's definition alone (test helper).

Independent of oracle/ and of the CUDA path: it enumerates every zero-tilt octahedron surface of an L x L torus
(heights with all nearest-neighbour differences +-1, modulo a global shift) row by row, and builds exact
single-site / tile / MCS transition matrices in *height* language for the schedule of DESIGN.md.
"""
from __future__ import annotations

import itertools
from fractions import Fraction

import numpy as np


def row_patterns(L):
    """All +-1 sequences of length L with zero sum, as relative heights r[x] (r[0] = 0)."""
    pats = []
    for ups in itertools.combinations(range(1, L + 1), L // 2):
        s = np.full(L + 1, -1, dtype=np.int64)
        s[list(ups)] = 1
        s[0] = 0
        r = np.cumsum(s)           # r[x] = sum_{l=1..x} s_l ; r[L] = 0
        pats.append(r[:L])
    return np.array(pats)          # [P, L]


def enumerate_states(L):
    """-> (B, Pidx, pats): B[n, y] = base height of row y (B[n,0] = 0), Pidx[n, y] = pattern index of row y."""
    pats = row_patterns(L)
    P = len(pats)
    # compat[d][p] = array of p' such that row (b+d, p') may sit above row (b, p)
    compat = {d: [np.array([pp for pp in range(P)
                            if np.all(np.abs(d + pats[pp] - pats[p]) == 1)], dtype=np.int64)
                  for p in range(P)] for d in (-1, 1)}
    B = np.zeros((P, 1), dtype=np.int8)
    PI = np.arange(P, dtype=np.int8).reshape(P, 1)
    for y in range(1, L):
        newB, newP = [], []
        for d in (-1, 1):
            for p in range(P):
                sel = np.nonzero(PI[:, -1] == p)[0]
                nxt = compat[d][p]
                if len(sel) == 0 or len(nxt) == 0:
                    continue
                rep = np.repeat(sel, len(nxt))
                til = np.tile(nxt, len(sel))
                newB.append(np.concatenate([B[rep], (B[rep, -1] + d).reshape(-1, 1).astype(np.int8)], axis=1))
                newP.append(np.concatenate([PI[rep], til.reshape(-1, 1).astype(np.int8)], axis=1))
        B = np.concatenate(newB)
        PI = np.concatenate(newP)
    # closure: row 0 = (0, p0) must be compatible above row L-1 = (b, p)
    ok = np.zeros(len(B), dtype=bool)
    for d in (-1, 1):
        for p in range(P):
            sel = np.nonzero((PI[:, -1] == p) & (B[:, -1] == -d))[0]
            if len(sel) == 0:
                continue
            good = np.zeros(P, dtype=bool)
            good[compat[d][p]] = True
            ok[sel] = good[PI[sel, 0]]
    return B[ok], PI[ok], pats


def sums_per_state(B, PI, pats):
    """-> (S1, S2) int64 arrays: sum of h and of h^2 per state (h(0,0) = 0 gauge)."""
    L = pats.shape[1]
    s1 = pats.sum(axis=1)
    s2 = (pats * pats).sum(axis=1)
    b = B.astype(np.int64)
    S1 = (L * b + s1[PI]).sum(axis=1)
    S2 = (L * b * b + 2 * b * s1[PI] + s2[PI]).sum(axis=1)
    return S1, S2


def heights_of(B, PI, pats):
    """-> H[n, y, x]"""
    return B.astype(np.int64)[:, :, None] + pats[PI]


def w2_fraction(S1, S2, N):
    """exact W^2 = (N*S2 - S1^2)/N^2 as a Fraction (scalars)"""
    return Fraction(int(N) * int(S2) - int(S1) ** 2, int(N) ** 2)


def key_of(h):
    """gauge-invariant key of a height field [y, x]: heights relative to h(0,0)"""
    h = np.asarray(h, dtype=np.int64)
    return (h - h[0, 0]).astype(np.int8).tobytes()


class ExactChain:
    """Exact Markov chain of the DESIGN.md schedule on an L x L torus with tile edge T (g = 1), dense matrices."""

    def __init__(self, L, T, p, q):
        assert T % 4 != 0, "exact chain helper assumes offset granularity 1"
        self.L, self.T, self.p, self.q = L, T, p, q
        B, PI, pats = enumerate_states(L)
        self.H = heights_of(B, PI, pats)                 # gauge h(0,0) = 0
        self.n = len(self.H)
        self.index = {key_of(h): i for i, h in enumerate(self.H)}
        S1, S2 = sums_per_state(B, PI, pats)
        N = L * L
        self.w2 = (N * S2 - S1 * S1) / float(N * N)
        self._site = {}

    def site_kernel(self, x, y):
        """K[s, s'] for one attempt at site (x, y) -- the rule in height language."""
        if (x, y) in self._site:
            return self._site[(x, y)]
        L, n = self.L, self.n
        K = np.zeros((n, n))
        for i, h in enumerate(self.H):
            c = h[y, x]
            nb = (h[y, (x - 1) % L], h[y, (x + 1) % L], h[(y - 1) % L, x], h[(y + 1) % L, x])
            if all(v == c + 1 for v in nb):
                h2 = h.copy(); h2[y, x] += 2
                j = self.index[key_of(h2)]
                K[i, j] += self.p; K[i, i] += 1 - self.p
            elif all(v == c - 1 for v in nb):
                h2 = h.copy(); h2[y, x] -= 2
                j = self.index[key_of(h2)]
                K[i, j] += self.q; K[i, i] += 1 - self.q
            else:
                K[i, i] = 1.0
        self._site[(x, y)] = K
        return K

    def tile_kernel(self, X0, Y0):
        """T*T sequential attempts, each at a uniformly random site of the tile with origin (X0, Y0)."""
        L, T = self.L, self.T
        one = sum(self.site_kernel((X0 + lx) % L, (Y0 + ly) % L) for lx in range(T) for ly in range(T)) / (T * T)
        return np.linalg.matrix_power(one, T * T)

    def mcs_kernel(self):
        """Average over offsets (uniform on [0,T)^2) and over the 24 colour orders of the 4 colour passes."""
        L, T = self.L, self.T
        NT = L // T
        M = np.zeros((self.n, self.n))
        for ox in range(T):
            for oy in range(T):
                passes = []
                for colour in range(4):
                    Pm = np.eye(self.n)
                    for ty in range(colour >> 1, NT, 2):
                        for tx in range(colour & 1, NT, 2):
                            Pm = Pm @ self.tile_kernel(ox + tx * T, oy + ty * T)
                    passes.append(Pm)
                for perm in itertools.permutations(range(4)):
                    A = np.eye(self.n)
                    for c in perm:
                        A = A @ passes[c]
                    M += A
        return M / (T * T * 24)

    def rs_mcs_kernel(self):
        """True random-sequential: L*L attempts at uniformly random sites."""
        L = self.L
        one = sum(self.site_kernel(x, y) for x in range(L) for y in range(L)) / (L * L)
        return np.linalg.matrix_power(one, L * L)

    @staticmethod
    def stationary(M):
        """stationary row vector by repeated squaring (rows renormalised to stay stochastic in floating point)"""
        n = len(M)
        A = M.copy()
        for _ in range(40):
            A = A @ A
            A /= A.sum(axis=1, keepdims=True)
        v = np.full(n, 1.0 / n) @ A
        return v / v.sum()

    def min_density(self):
        L = self.L
        d = np.zeros(self.n)
        for i, h in enumerate(self.H):
            cnt = 0
            for y in range(L):
                for x in range(L):
                    c = h[y, x]
                    if (h[y, (x - 1) % L] == c + 1 and h[y, (x + 1) % L] == c + 1 and
                            h[(y - 1) % L, x] == c + 1 and h[(y + 1) % L, x] == c + 1):
                        cnt += 1
            d[i] = cnt / (L * L)
        return d
