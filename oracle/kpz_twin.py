"""Pure-Python twin of the oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

An independent restatement, for tiny lattices only, of the same schedule in a *different representation*:
it keeps the height field h(x,y) itself (not the slopes) and applies the octahedron rule in height language
(a site whose four neighbours are all one unit higher is a local minimum and rises by 2 with
probability p; one whose four neighbours are all one unit lower is a local maximum and drops by 2 with
probability q).  Slopes are derived from the heights only when asked for.  tests/test_oracle_twin.py requires
this and oracle/kpz_oracle.cpp to agree bit for bit; together with the paper-fixed pins this is what stands in
for the schedule details the paper does not define ("parity unpinned" items).

Shares no code with the C++ oracle or with the CUDA path.
"""
from __future__ import annotations

M0, M1 = 0xD2511F53, 0xCD9E8D57
W0, W1 = 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    """Philox4x32-10 (Salmon et al., SC'11): 10 rounds, key bumped by (W0, W1) before rounds 2..10."""
    c = [int(v) & MASK for v in ctr]
    k = [int(v) & MASK for v in key]
    for rnd in range(10):
        if rnd:
            k = [(k[0] + W0) & MASK, (k[1] + W1) & MASK]
        p0 = M0 * c[0]
        p1 = M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & MASK, (p0 >> 32) ^ c[3] ^ k[1], p0 & MASK]
    return c


def mulhi32(a, n):
    return (a * n) >> 32


def threshold(prob):
    if prob >= 1.0:
        return 1 << 32
    if prob <= 0.0:
        return 0
    return int(prob * 4294967296.0)


class Twin:
    def __init__(self, L, p, q, T, seed, replica=0, schedule="colours", sub_sweeps=1, poisson=False):
        assert T >= 1 and L % (2 * T) == 0 and schedule in ("colours", "dead_border")
        assert sub_sweeps >= 1 and (T * T) % sub_sweeps == 0
        self.schedule, self.K, self.poisson = schedule, sub_sweeps, poisson
        self.attempts = 0
        self.L, self.T, self.p, self.q, self.seed, self.replica = L, T, p, q, seed, replica
        if poisson:
            self._poisson_table()
        self.g = 4 if T % 4 == 0 else 1
        self.key = (seed & MASK, (seed >> 32) & MASK)
        self.thr_p, self.thr_q = threshold(p), threshold(q)
        self.h = None
        self.mcs = 0
        self.deposits = self.removals = 0
        self.trace = None     # optional list of (x, y, dir) per attempt

    def init_flat(self):
        L = self.L
        self.h = [[(x + y) & 1 for x in range(L)] for y in range(L)]   # h[y][x]
        self.mcs = 0
        self.deposits = self.removals = 0

    def _attempt(self, x, y, accept):
        L, h = self.L, self.h
        c = h[y][x]
        nb = (h[y][(x - 1) % L], h[y][(x + 1) % L], h[(y - 1) % L][x], h[(y + 1) % L][x])
        d = 0
        if all(v == c + 1 for v in nb):
            if accept < self.thr_p:
                d = 1
        elif all(v == c - 1 for v in nb):
            if accept < self.thr_q:
                d = -1
        if d:
            h[y][x] = c + 2 * d
            if d > 0:
                self.deposits += 1
            else:
                self.removals += 1
        if self.trace is not None:
            self.trace.append((x, y, d))

    def _poisson_table(self):
        """DESIGN.md S7, in Python integers: weights 2^52 at the mode lambda = T^2/K, multiplied / divided down the two
        sides with floor divisions, over |k - lambda| <= ceil(12 sqrt(lambda)) + 16; thresholds floor(2^32 C_k / S)."""
        import math
        lam = self.T * self.T // self.K
        W = math.isqrt(144 * lam - 1) + 1 + 16 if lam > 0 else 16       # ceil(12 sqrt(lambda)) + 16
        kmin, kmax = max(0, lam - W), lam + W
        q = {lam: 1 << 52}
        for k in range(lam + 1, kmax + 1):
            q[k] = q[k - 1] * lam // k
        for k in range(lam - 1, kmin - 1, -1):
            q[k] = q[k + 1] * (k + 1) // lam
        S = sum(q.values())
        self.kmin, self.thr, C = kmin, [], 0
        for k in range(kmin, kmax + 1):
            C += q[k]
            self.thr.append((C << 32) // S)

    def _poisson_count(self, m, sub, tile_id):
        u = philox4x32_10((0x7FFFFFFF - sub, tile_id, m, self.replica), self.key)[0]
        return self.kmin + sum(1 for t in self.thr[:-1] if t <= u)

    def global_draw(self, m, sub=0):
        G = philox4x32_10((sub, MASK, m, self.replica), self.key)
        n = self.T // self.g
        ox = self.g * mulhi32(G[0], n)
        oy = self.g * mulhi32(G[1], n)
        pidx = mulhi32(G[2], 24)
        pool = [0, 1, 2, 3]
        perm = [pool.pop(pidx // 6), pool.pop((pidx % 6) // 2), pool.pop(pidx % 2)]
        perm.append(pool[0])
        return ox, oy, perm

    def run(self, n_mcs):
        L, T = self.L, self.T
        NT = L // T
        for _ in range(n_mcs):
            m = self.mcs
            # S6: K sub-sweeps; sub-sweep j has its own draw (offset, colour order) and runs steps
            # [j T^2/K, (j+1) T^2/K) of every tile's stream of this MCS
            for j in range(self.K):
                ox, oy, perm = self.global_draw(m, j)
                # S4: the four colours in the drawn order; S5 (dead borders): every tile in one pass
                passes = [[(tx, ty) for ty in range(c >> 1, NT, 2) for tx in range(c & 1, NT, 2)] for c in perm] \
                    if self.schedule == "colours" else [[(tx, ty) for ty in range(NT) for tx in range(NT)]]
                for tiles in passes:
                    for (tx, ty) in tiles:
                        tile_id = ty * NT + tx
                        s0, s1 = j * T * T // self.K, (j + 1) * T * T // self.K
                        if self.poisson:       # S7: own stream region per sub-sweep, Poissonised length
                            s0 = j << 16
                            s1 = s0 + self._poisson_count(m, j, tile_id)
                        self.attempts += s1 - s0
                        for s in range(s0, s1):
                            # DESIGN.md S3: a site word is a base-T*T fraction with two digits; step s uses digit
                            # s % 2 of word (s // 2) % 4 of call s // 8; accept word = word s % 4 of call s // 4 + 2^31
                            if s % 8 == 0 or s == s0:
                                sites = philox4x32_10((s // 8, tile_id, m, self.replica), self.key)
                            if s % 4 == 0 or s == s0:
                                accepts = philox4x32_10((s // 4 + 0x80000000, tile_id, m, self.replica), self.key)
                            word = sites[(s // 2) % 4]
                            if s % 2 == 1:
                                word = (word * T * T) & MASK
                            idx = mulhi32(word, T * T)
                            if self.schedule == "dead_border" and (idx % T == T - 1 or idx // T == T - 1):
                                continue      # a site on the +x / +y edge of its tile: the attempt does nothing
                            x = (ox + tx * T + idx % T) % L
                            y = (oy + ty * T + idx // T) % L
                            self._attempt(x, y, accepts[s % 4])
            self.mcs += 1

    def slopes(self):
        L, h = self.L, self.h
        sx = [[h[y][x] - h[y][(x - 1) % L] for x in range(L)] for y in range(L)]
        sy = [[h[y][x] - h[(y - 1) % L][x] for x in range(L)] for y in range(L)]
        return sx, sy

    def sums(self):
        s1 = sum(sum(r) for r in self.h)
        s2 = sum(sum(v * v for v in r) for r in self.h)
        return s1, s2
