// edges.cpp -- host-side ownership of the unique angular edges (used by the fused stage kernel).
//
// Every unique edge e = (lo, hi) of the angular grid carries one upwind flux (Eq.25) that enters
// the flux divergence of both of its angles with opposite signs.  The stage kernel computes it once, in the
// thread of the edge's OWNER angle, and hands it to the PARTNER angle through shared memory.  For a fixed
// trip count per thread the ownership is balanced: an orientation of the edge graph in which every angle owns
// at most ceil(deg/2) <= 3 of its <= 6 edges (and therefore receives at most 3).  Such an orientation always
// exists (pair up odd-degree vertices and follow Euler circuits); it is found here by reversing paths from
// overloaded to underloaded vertices, in a fixed deterministic order.
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
    o.own_edge.assign((size_t)N * kMaxOwn, -1);
    o.own_partner.assign((size_t)N * kMaxOwn, -1);
    o.pull_pos.assign((size_t)N * kMaxOwn, -1);
    std::vector<int> nown(N, 0), npull(N, 0), slot_of_edge(E, -1);
    for (int e = 0; e < E; e++) {  // increasing edge id => slots in increasing edge id per owner
        const int v = owner[e];
        if (nown[v] >= kMaxOwn) { err = "owner overflow"; return false; }
        const int p = (a.edge_lo[e] == v) ? a.edge_hi[e] : a.edge_lo[e];
        slot_of_edge[e] = nown[v];
        o.own_edge[(size_t)v * kMaxOwn + nown[v]] = e;
        o.own_partner[(size_t)v * kMaxOwn + nown[v]] = p;
        nown[v]++;
    }
    for (int e = 0; e < E; e++) {
        const int v = owner[e];
        const int p = (a.edge_lo[e] == v) ? a.edge_hi[e] : a.edge_lo[e];
        if (p == v) continue;  // degenerate self edge (npsi = 1): carries no net flux
        if (npull[p] >= kMaxOwn) { err = "partner overflow"; return false; }
        o.pull_pos[(size_t)p * kMaxOwn + npull[p]] = slot_of_edge[e] * N + v;
        npull[p]++;
    }
    return true;
}

}  // namespace rad
