// edges.cpp -- host-side ownership of the unique angular edges (used by the fused stage kernel).
//
// Every unique edge e = (lo, hi) of the angular grid carries one upwind flux (Eq.25) that enters
// the flux divergence of both of its angles with opposite signs.  The stage kernel computes it once, in the
// thread of the edge's OWNER angle, and hands it to the PARTNER angle through shared memory.  For a fixed
// trip count per thread the ownership is balanced: an orientation of the edge graph in which every angle owns
// at most ceil(deg/2) <= 3 of its <= 6 edges (and therefore receives at most 3).  Such an orientation always
// exists (pair up odd-degree vertices and follow Euler circuits); it is found here by reversing paths from
// overloaded to underloaded vertices, in a fixed deterministic order.  The owned edges of an angle then get SLOTS 0..2 by an
// edge colouring (below) under which the received edges of every angle have different slots as well.
#include <algorithm>
#include <queue>

#include "rad_internal.h"

namespace rad {

bool build_edge_ownership(const AngleTables &a, EdgeOwnership &o, std::string &err) {
    const int N = a.N, E = a.E;
    std::vector<int> owner(E), deg(N, 0), out(N, 0);
    for (int e = 0; e < E; e++) { owner[e] = a.edge_lo[e]; deg[a.edge_lo[e]]++; deg[a.edge_hi[e]]++; out[a.edge_lo[e]]++; }
    for (int n = 0; n < N; n++)
        if (deg[n] > 2 * kMaxOwn) { err = "angle with more than 6 edges"; return false; }
    // incident edge lists
    std::vector<std::vector<int>> inc(N);
    for (int e = 0; e < E; e++) { inc[a.edge_lo[e]].push_back(e); if (a.edge_hi[e] != a.edge_lo[e]) inc[a.edge_hi[e]].push_back(e); }
    // balance: floor(deg/2) <= out <= ceil(deg/2), hence out <= 3 and in = deg - out <= 3
    auto hi = [&](int v) { return (deg[v] + 1) / 2; };
    auto lo = [&](int v) { return deg[v] / 2; };
    auto other = [&](int e, int u) { return (a.edge_lo[e] == u) ? a.edge_hi[e] : a.edge_lo[e]; };
    // shed == true : v owns too many; walk owned edges to a vertex that can take one more; reverse the path
    // shed == false: v owns too few; walk edges owned by the far end to a vertex that can give one; reverse
    auto rebalance = [&](int v, bool shed) -> bool {
        std::vector<int> via(N, -1), seen(N, 0);
        std::queue<int> q;
        q.push(v); seen[v] = 1;
        int target = -1;
        while (!q.empty() && target < 0) {
            const int u = q.front(); q.pop();
            for (int e : inc[u]) {
                const int p = other(e, u);
                if ((shed ? owner[e] != u : owner[e] != p) || p == u || seen[p]) continue;
                seen[p] = 1; via[p] = e;
                if (shed ? out[p] < hi(p) : out[p] > lo(p)) { target = p; break; }
                q.push(p);
            }
        }
        if (target < 0) return false;
        int p = target;
        while (p != v) {  // every edge on the path changes owner
            const int e = via[p];
            const int u = other(e, p);
            owner[e] = shed ? p : u;
            p = u;
        }
        if (shed) { out[v]--; out[target]++; } else { out[v]++; out[target]--; }
        return true;
    };
    for (int v = 0; v < N; v++) {
        while (out[v] > hi(v)) if (!rebalance(v, true)) { err = "edge ownership could not be balanced"; return false; }
        while (out[v] < lo(v)) if (!rebalance(v, false)) { err = "edge ownership could not be balanced"; return false; }
    }
    for (int v = 0; v < N; v++)
        if (out[v] > hi(v) || out[v] < lo(v)) {  // a later reversal never unbalances a settled vertex, but check
            err = "edge ownership is not balanced"; return false;
        }
    // Slots.  The slot of an edge at its owner is a COLOUR in {0, 1, 2} chosen so that the edges an angle owns have different colours
    // (one slot each) and the edges it receives have different colours too: then the k-th flux an angle pulls always sits in slot k
    // of its owner, and a kernel needs only the owner's angle index per pulled edge.  Such a colouring is a proper edge colouring of
    // the bipartite graph (owner side, partner side) of maximum degree 3, which exists by Koenig's theorem; it is found by the
    // alternating-path argument of its proof, in a fixed deterministic order (increasing edge id).
    std::vector<int> colour(E, -1);
    std::vector<int> atX((size_t)N * kMaxOwn, -1), atY((size_t)N * kMaxOwn, -1);  // edge of colour c at owner side x / partner side y
    auto partner = [&](int e) { const int v = owner[e]; return (a.edge_lo[e] == v) ? a.edge_hi[e] : a.edge_lo[e]; };
    for (int e = 0; e < E; e++) {
        const int x = owner[e], y = partner(e);
        int ca = -1, cb = -1;
        for (int c = kMaxOwn - 1; c >= 0; c--) { if (atX[(size_t)x * kMaxOwn + c] < 0) ca = c; if (atY[(size_t)y * kMaxOwn + c] < 0) cb = c; }
        if (ca < 0 || cb < 0) { err = "edge colouring: a vertex has more than 3 edges on one side"; return false; }
        if (atY[(size_t)y * kMaxOwn + ca] >= 0) {
            // colour ca is taken at y: swap ca <-> cb along the maximal path that leaves y on colour ca (it cannot reach x, where ca is free)
            std::vector<int> path;
            int side = 1, v = y, want = ca;  // side 1: at a partner-side vertex, follow `want`
            while (true) {
                const int f = side ? atY[(size_t)v * kMaxOwn + want] : atX[(size_t)v * kMaxOwn + want];
                if (f < 0) break;
                path.push_back(f);
                v = side ? owner[f] : partner(f);
                side ^= 1;
                want = (want == ca) ? cb : ca;
            }
            for (int f : path) { atX[(size_t)owner[f] * kMaxOwn + colour[f]] = -1; atY[(size_t)partner(f) * kMaxOwn + colour[f]] = -1; }
            for (int f : path) {
                colour[f] = (colour[f] == ca) ? cb : ca;
                atX[(size_t)owner[f] * kMaxOwn + colour[f]] = f; atY[(size_t)partner(f) * kMaxOwn + colour[f]] = f;
            }
        }
        colour[e] = ca;
        atX[(size_t)x * kMaxOwn + ca] = e; atY[(size_t)y * kMaxOwn + ca] = e;
    }
    o.own_edge.assign((size_t)N * kMaxOwn, -1);
    o.own_partner.assign((size_t)N * kMaxOwn, -1);
    o.pull_pos.assign((size_t)N * kMaxOwn, -1);
    for (int e = 0; e < E; e++) {
        const int v = owner[e], p = partner(e), c = colour[e];
        if (o.own_edge[(size_t)v * kMaxOwn + c] >= 0) { err = "edge colouring: owner slot used twice"; return false; }
        o.own_edge[(size_t)v * kMaxOwn + c] = e;
        o.own_partner[(size_t)v * kMaxOwn + c] = p;
        if (p == v) continue;  // degenerate self edge (npsi = 1): carries no net flux
        if (o.pull_pos[(size_t)p * kMaxOwn + c] >= 0) { err = "edge colouring: partner slot used twice"; return false; }
        o.pull_pos[(size_t)p * kMaxOwn + c] = c * N + v;  // the k-th pull of an angle comes from slot k of its owner
    }
    return true;
}

}  // namespace rad
