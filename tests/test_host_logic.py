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


def explicit_tables(A):
    """rad_angles kind 2 tables (rad.h) of an oracle angle grid: per (angle, slot) edge data, the normal pointing from the angle to its neighbour"""
    N = A.N
    tab = dict(nhat=A.nhat.copy(), domega=A.domega.copy(), nnbr=A.nnbr.copy(), nbr=A.nbr.copy(),
               edge_len=np.zeros((N, 6)), edge_mid=np.zeros((N, 6, 3)), edge_nrm=np.zeros((N, 6, 3)))
    for q in range(N):
        for s in range(6):
            e = A.nbr_edge[q, s]
            if e >= 0:
                tab["edge_len"][q, s] = A.edge_len[e]; tab["edge_mid"][q, s] = A.edge_mid[e]
                tab["edge_nrm"][q, s] = A.edge_nrm[e] if A.edge_lo[e] == q else -A.edge_nrm[e]
    return tab


@pytest.mark.parametrize("angles", [("geodesic", 2), ("latlon", 4, 8)])
def test_edge_ownership_of_explicit_tables(lib, oracle, angles):
    """an ("explicit", tables) grid goes through the same marshalling as rad_create's and gives the named grid's ownership;
    edge midpoints that are not finite unit vectors and non-finite edge normals are refused instead of poisoning the stored coefficients"""
    A = oracle.Angles(*angles)
    tab = explicit_tables(A)
    a, b = B.rad_edge_ownership(angles), B.rad_edge_ownership(("explicit", tab))
    assert a["N"] == b["N"] and a["E"] == b["E"]
    if angles[0] == "geodesic":  # the explicit builder numbers the unique edges in the geodesic grid's own order (first occurrence)
        assert all(np.array_equal(a[k], b[k]) for k in ("edge_lo", "edge_hi", "own_edge", "own_partner", "pull_pos"))
    else:                        # latitude-longitude: another numbering of the same edges; every one of them owned once
        assert sorted(zip(a["edge_lo"].tolist(), a["edge_hi"].tolist())) == sorted(zip(b["edge_lo"].tolist(), b["edge_hi"].tolist()))
        assert sorted(b["own_edge"][b["own_edge"] >= 0].tolist()) == list(range(b["E"]))
    e0 = int(np.argmax(A.nbr_edge[0] >= 0))  # a slot of angle 0 that holds an edge whose lower angle is 0
    for key, val in (("edge_mid", np.nan), ("edge_nrm", np.inf), ("edge_mid", 3.0), ("edge_nrm", np.nan)):
        bad = dict(tab, **{key: tab[key].copy()})
        bad[key][0, e0, 1] = val
        with pytest.raises(B.RadError) as e:
            B.rad_edge_ownership(("explicit", bad))
        assert e.value.status == 1 and "edge_mid must be finite unit vectors" in str(e.value)
    with pytest.raises(ValueError):
        B.rad_edge_ownership(("icosahedral", 2))
