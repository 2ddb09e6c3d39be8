"""C++ oracle vs the independent height-language Python twin, bit for bit, plus distribution tests of the
schedule's own definitions (colour order, offsets, site choice) which the paper does not pin."""
import numpy as np
import pytest

from oracle import Oracle
from oracle import kpz_twin


@pytest.mark.parametrize("L,T,p,q,seed,rep,n", [
    (8, 4, 1.0, 0.0, 1, 0, 5),
    (16, 4, 0.75, 0.25, 7, 0, 4),
    (16, 8, 0.5, 0.5, 0xDEADBEEFCAFE, 3, 3),
    (32, 16, 1.0, 0.0, 42, 0, 3),
    (32, 8, 0.3, 0.6, 2**63 + 5, 1023, 3),
    (12, 3, 0.75, 0.25, 3, 2, 4),
    (4, 2, 1.0, 0.0, 9, 0, 6),
    (6, 1, 0.9, 0.1, 5, 0, 6),
    (18, 3, 1.0, 0.0, 5, 0, 3),
])
def test_oracle_equals_twin(L, T, p, q, seed, rep, n):
    o = Oracle(L, p, q, T, seed, replica=rep)
    t = kpz_twin.Twin(L, p, q, T, seed, replica=rep)
    o.init_flat(); t.init_flat()
    for step in range(n):
        assert o.global_draw(step) == t.global_draw(step)
        o.run(1); t.run(1)
        sx, sy = o.slopes()
        tsx, tsy = t.slopes()
        assert np.array_equal(sx, np.array(tsx, dtype=np.int8))
        assert np.array_equal(sy, np.array(tsy, dtype=np.int8))
        s1, s2, _ = o.measure()
        assert (s1, s2) == t.sums()                 # absolute heights: h00 bookkeeping vs true height field
        c = o.counters()
        assert (c["deposits"], c["removals"]) == (t.deposits, t.removals)


def test_global_draw_distribution():
    """24 colour orders and (T/4)^2 offsets are (statistically) uniform; all 24 orders are valid permutations."""
    o = Oracle(64, 1.0, 0.0, 32, seed=12345)
    n = 48000
    perms, offs = {}, {}
    for m in range(n):
        ox, oy, perm = o.global_draw(m)
        assert sorted(perm) == [0, 1, 2, 3] and ox % 4 == 0 and oy % 4 == 0 and ox < 32 and oy < 32
        perms[tuple(perm)] = perms.get(tuple(perm), 0) + 1
        offs[(ox, oy)] = offs.get((ox, oy), 0) + 1
    assert len(perms) == 24 and len(offs) == 64
    chi_p = sum((c - n / 24) ** 2 / (n / 24) for c in perms.values())
    chi_o = sum((c - n / 64) ** 2 / (n / 64) for c in offs.values())
    assert chi_p < 60.0      # dof 23, P(chi2 > 60) ~ 4e-5
    assert chi_o < 120.0     # dof 63, P(chi2 > 120) ~ 2e-5


def test_site_choice_uniform_within_tile():
    L, T = 32, 16
    tw = kpz_twin.Twin(L, 0.0, 0.0, T, seed=77)
    tw.init_flat(); tw.trace = []
    tw.run(40)
    cnt = np.zeros((L, L))
    for (x, y, d) in tw.trace:
        cnt[y, x] += 1
    exp = 40.0
    chi = ((cnt - exp) ** 2 / exp).sum()
    dof = L * L - (L // T) ** 2          # each tile's total is fixed (T^2 per MCS)
    assert abs(chi - dof) < 6 * np.sqrt(2 * dof)
