"""Host-side check of the parity-free tile encoding used by the T >= 32 update kernel.

The kernel keeps u = h1 ^ E(x, y) in shared memory, with h1 = bit 1 of the height and
E(x, y) = ((x + (y & 1)) >> 1 & 1) ^ (y >> 1 & 1), and tests eq. 2 as
  local minimum <=> u(x+1,y) == u, u(x-1,y) != u, u(x,y+1) == u, u(x,y-1) != u      (maximum: all four reversed).
Here the claim is checked against the definition on heights for every neighbour configuration and every phase of
(x, y) mod 4, and the two constants of `enc_word` are re-derived from E.  (GPU parity with the oracle covers the
kernel itself; this pins the algebra the kernel relies on, with no GPU.)
"""
import itertools

import numpy as np


def E(x, y):
    return (((x + (y & 1)) >> 1) & 1) ^ ((y >> 1) & 1)


def test_minimum_and_maximum_tests_are_parity_free():
    for x, y in itertools.product(range(-4, 8), repeat=2):
        for h in range(-6, 7):
            if (h & 1) != ((x + y) & 1):        # low bit of the height is the checkerboard (x+y)&1
                continue
            for dl, dr, dd, du in itertools.product((-1, 1), repeat=4):
                hs = {"o": h, "l": h + dl, "r": h + dr, "d": h + dd, "u": h + du}
                pos = {"o": (x, y), "l": (x - 1, y), "r": (x + 1, y), "d": (x, y - 1), "u": (x, y + 1)}
                u = {k: ((hs[k] >> 1) & 1) ^ E(*pos[k]) for k in hs}
                is_min = (dl, dr, dd, du) == (1, 1, 1, 1)
                is_max = (dl, dr, dd, du) == (-1, -1, -1, -1)
                t_min = u["r"] == u["o"] and u["l"] != u["o"] and u["u"] == u["o"] and u["d"] != u["o"]
                t_max = u["r"] != u["o"] and u["l"] == u["o"] and u["u"] != u["o"] and u["d"] == u["o"]
                assert t_min == is_min and t_max == is_max, (x, y, h, dl, dr, dd, du)


def test_enc_word_constants():
    # bit j of an own word is column 32k + j; E has period 4 in x, so every word of a row carries the same pattern
    for y, want in ((0, 0xCCCCCCCC), (1, 0x66666666), (2, 0x33333333), (3, 0x99999999), (-1, 0x99999999)):
        word = sum(E(j, y) << j for j in range(32))
        assert word == want
        assert sum(E(64 + j, y) << j for j in range(32)) == want
    # halo columns x = T (== 0 mod 4) and x = -1
    for y in range(-1, 8):
        assert E(64, y) == (y >> 1) & 1
        assert E(-1, y) == ((y & 1) ^ 1) ^ ((y >> 1) & 1)


def test_lop3_truth_tables():
    # LOP3 immediates of the kernel: inputs a = 0xF0, b = 0xCC, c = 0xAA
    a, b, c = 0xF0, 0xCC, 0xAA
    assert ((a ^ (~b & 0xFF)) | (a ^ c)) == 0xDB       # not a minimum along x: (o ^ ~l) | (o ^ r)
    assert ((a ^ b) | (a ^ (~c & 0xFF))) == 0xBD       # not a minimum along y: (o ^ u) | (o ^ ~d)
