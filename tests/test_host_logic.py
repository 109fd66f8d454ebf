"""Host logic of the library that needs no GPU: the ownership and slot colouring of the angular edges (edges.cpp) that the tile kernel's
angular exchange is built on (Eq.25: every unique edge flux is formed once and enters both of its angles with opposite signs)."""
import numpy as np
import pytest

from paper_2302_04283_b200 import binding as B
from paper_2302_04283_b200 import build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return B.lib()


@pytest.mark.parametrize("angles", [("geodesic", 1), ("geodesic", 2), ("geodesic", 3), ("geodesic", 4), ("geodesic", 5), ("geodesic", 7),
                                    ("latlon", 5, 16), ("latlon", 8, 16), ("latlon", 4, 8), ("latlon", 1, 4), ("latlon", 3, 1), ("latlon", 7, 9)])
def test_edge_ownership_is_a_balanced_orientation_with_a_proper_slot_colouring(lib, angles):
    t = B.rad_edge_ownership(angles)
    N, E, lo, hi, own, par, pull = t["N"], t["E"], t["edge_lo"], t["edge_hi"], t["own_edge"], t["own_partner"], t["pull_pos"]
    # every unique edge is owned exactly once, by one of its two angles, and the partner entry is its other end
    owned = own[own >= 0]
    assert sorted(owned.tolist()) == list(range(E))
    deg = np.zeros(N, int)
    for e in range(E):
        deg[lo[e]] += 1; deg[hi[e]] += 1
    for n in range(N):
        for k in range(3):
            e = own[n, k]
            if e < 0:
                assert par[n, k] == -1
                continue
            assert n in (lo[e], hi[e]) and par[n, k] == (hi[e] if lo[e] == n else lo[e])
    # balanced: an angle owns between floor(deg/2) and ceil(deg/2) of its edges (so it owns <= 3 and receives <= 3)
    nown = (own >= 0).sum(1)
    assert (nown >= deg // 2).all() and (nown <= (deg + 1) // 2).all() and nown.max() <= 3
    # the slots colour the edges properly on the receiving side too: entry k of pull_pos comes from slot k of its owner, every edge
    # that joins two different angles is received exactly once, and by the right angle
    seen = set()
    for n in range(N):
        for k in range(3):
            q = pull[n, k]
            if q < 0:
                continue
            assert q // N == k
            v = q % N
            e = own[v, k]
            assert e >= 0 and par[v, k] == n and v != n
            assert e not in seen
            seen.add(e)
    assert seen == {e for e in range(E) if lo[e] != hi[e]}


def test_edge_ownership_is_deterministic(lib):
    a, b = B.rad_edge_ownership(("geodesic", 4)), B.rad_edge_ownership(("geodesic", 4))
    assert all(np.array_equal(a[k], b[k]) for k in ("own_edge", "own_partner", "pull_pos"))
