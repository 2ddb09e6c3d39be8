"""Seeded synthetic input generators shared by the oracle tests and the CUDA parity tests.

Holds none of the method's arithmetic (no update rule, no schedule, no RNG of the method, no width formula):
it only builds valid octahedron surfaces h(x,y) (all nearest-neighbour differences +-1, periodic) from closed
forms and turns a height field into the two slope arrays by their definition (backward differences,
DESIGN.md reading R3).  All arrays are indexed [y, x].
"""
from __future__ import annotations

import numpy as np


def heights_to_slopes(h):
    """sx(x,y) = h(x,y) - h(x-1,y), sy(x,y) = h(x,y) - h(x,y-1), periodic; int8 arrays [y, x]."""
    h = np.asarray(h, dtype=np.int64)
    sx = (h - np.roll(h, 1, axis=1)).astype(np.int8)
    sy = (h - np.roll(h, 1, axis=0)).astype(np.int8)
    assert np.all(np.abs(sx) == 1) and np.all(np.abs(sy) == 1), "not an octahedron surface"
    return sx, sy


def flat_heights(L):
    """The zig-zag start of P:88: h = (x + y) mod 2."""
    y, x = np.mgrid[0:L, 0:L]
    return ((x + y) & 1).astype(np.int64)


def raised_flat_heights(L, seed, frac=0.5):
    """Flat zig-zag with a seeded random subset of its (mutually non-adjacent) even-parity sites raised by 2.
    Every result is a valid surface; the subset is uniform with density `frac`."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:L, 0:L]
    h = ((x + y) & 1).astype(np.int64)
    mask = (rng.random((L, L)) < frac) & (((x + y) & 1) == 0)
    return h + 2 * mask


def triangle_heights(L, A):
    """h = tri_A(x) + tri_A(y), tri_A the triangle wave of period 2A taking 0,1,..,A,..,1 (2A must divide L)."""
    assert L % (2 * A) == 0
    t = np.arange(L) % (2 * A)
    tri = np.where(t <= A, t, 2 * A - t).astype(np.int64)
    return tri[None, :] + tri[:, None]


def staircase_heights(L, seed):
    """A valid surface with long-wavelength structure: sum of seeded zero-sum +-1 walks in x and in y
    (h = u(x) + v(y)); exercises large |h| for the int64 reductions."""
    rng = np.random.default_rng(seed)
    def walk():
        s = np.array([1] * (L // 2) + [-1] * (L // 2), dtype=np.int64)
        rng.shuffle(s)
        return np.concatenate([[0], np.cumsum(s)[:-1]])
    return walk()[None, :] + walk()[:, None]
