// xs_graph.cpp -- a-1 of DESIGN.md: seeded instance generator of the library (host, once).
//
// N spins, N triplets, every spin in exactly 3 triplets, 3 distinct spins in a
// triplet (random regular hypergraph of degree 3).  PAPER.md L279-L291: greedy partition into
// sets of mutually non-adjacent spins, permutation array + set sizes, N x 6 adjacency.
// Readings: configuration model on 3N stubs shuffled by sorting Philox keys,
// whole-attempt rejection; gauge bits from Philox; ascending scan order for the greedy sets.
// Written independently of oracle/ -- the two must agree byte for byte
// (tests/test_abi_cpu.py::test_generator_matches_oracle_generator).
#include <algorithm>
#include <numeric>

#include "xs_internal.h"

namespace xs {

void philox4x32_10_host(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t x0 = ctr[0], x1 = ctr[1], x2 = ctr[2], x3 = ctr[3];
    uint32_t ka = key[0], kb = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t pa = 0xD2511F53ull * x0;   // M0 * c0
        const uint64_t pb = 0xCD9E8D57ull * x2;   // M1 * c2
        const uint32_t y0 = static_cast<uint32_t>(pb >> 32) ^ x1 ^ ka;
        const uint32_t y2 = static_cast<uint32_t>(pa >> 32) ^ x3 ^ kb;
        x1 = static_cast<uint32_t>(pb);
        x3 = static_cast<uint32_t>(pa);
        x0 = y0;
        x2 = y2;
        ka += 0x9E3779B9u;
        kb += 0xBB67AE85u;
    }
    out[0] = x0; out[1] = x1; out[2] = x2; out[3] = x3;
}

namespace {

inline void rng(uint32_t a, uint32_t b, uint32_t c, uint32_t tag, uint64_t seed, uint32_t o[4])
{
    const uint32_t ctr[4] = {a, b, c, tag};
    const uint32_t key[2] = {static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32)};
    philox4x32_10_host(ctr, key, o);
}

// Fills nbr / cls from tri; false if some spin is not in exactly three triplets or an index
// is out of range or repeated inside a triplet.
bool derive_adjacency(HostGraph& g, std::string& err)
{
    const uint32_t n = g.n;
    g.nbr.assign(6ull * n, 0);
    g.cls.assign(3ull * n, 0);
    std::vector<uint8_t> deg(n, 0);
    for (uint32_t t = 0; t < n; ++t) {
        const uint32_t* m = &g.tri[3ull * t];
        if (m[0] >= n || m[1] >= n || m[2] >= n) { err = "triplet index out of range"; return false; }
        if (m[0] == m[1] || m[1] == m[2] || m[0] == m[2]) { err = "repeated spin inside a triplet"; return false; }
        static const int other[3][2] = {{1, 2}, {0, 2}, {0, 1}};
        for (int s = 0; s < 3; ++s) {
            const uint32_t v = m[s];
            if (deg[v] == 3) { err = "a spin enters more than 3 triplets"; return false; }
            const uint32_t r = deg[v]++;
            g.cls[3ull * v + r] = t;
            g.nbr[6ull * v + 2 * r] = m[other[s][0]];
            g.nbr[6ull * v + 2 * r + 1] = m[other[s][1]];
        }
    }
    for (uint32_t v = 0; v < n; ++v)
        if (deg[v] != 3) { err = "a spin enters fewer than 3 triplets"; return false; }
    return true;
}

// Greedy independent sets (L279): per round, ascending scan; a spin joins the round's set if
// it is still free, no earlier member of the set is adjacent to it, and the cap allows.
void greedy_sets(HostGraph& g, uint32_t cap)
{
    const uint32_t n = g.n;
    g.order.clear();
    g.order.reserve(n);
    g.set_start.assign(1, 0);
    std::vector<uint32_t> taken_round(n, 0);    // 0 = free, else round in which it was placed
    std::vector<uint32_t> blocked_round(n, 0);  // last round in which a neighbour was placed
    uint32_t round = 0;
    while (g.order.size() < n) {
        ++round;
        uint32_t members = 0;
        for (uint32_t v = 0; v < n; ++v) {
            if (taken_round[v] != 0 || blocked_round[v] == round) continue;
            if (cap != 0 && members == cap) break;
            taken_round[v] = round;
            g.order.push_back(v);
            ++members;
            for (int q = 0; q < 6; ++q) blocked_round[g.nbr[6ull * v + q]] = round;
        }
        g.set_start.push_back(static_cast<uint32_t>(g.order.size()));
    }
}

// Balanced sets (L281: set sizes chosen "to keep the processing of components as balanced as
// possible"; DESIGN.md R-balance): an equitable colouring with n_col colours found by a tabu
// search over colour swaps into max(4, ceil(N / S)) sets, S = the set cap or a power of two near
// N / 4: few barriers per sweep and evenly filled rounds instead of the greedy partition's 6-7
// ragged ones (4 colours are the fewest a graph made of triangles of degree 6 admits in practice).  All integer, deterministic;
// random choices come from Philox(ctr = (step, 0, 0, TAG_PARTITION), key = graph seed).
// Returns false (g.order untouched) if no proper colouring was found within the step budget.
bool balanced_sets(HostGraph& g, uint64_t seed, uint32_t n_col, uint32_t step_budget)
{
    const uint32_t n = g.n;
    if (n_col < 2 || n_col > n) return false;
    std::vector<uint32_t> colour(n);
    std::vector<int32_t> same(static_cast<size_t>(n) * n_col, 0);   // same[v][c]: neighbours of v coloured c
    std::vector<uint32_t> forbidden_until(static_cast<size_t>(n) * n_col, 0);
    auto S = [&](uint32_t v, uint32_t c) -> int32_t& { return same[static_cast<size_t>(v) * n_col + c]; };
    auto F = [&](uint32_t v, uint32_t c) -> uint32_t& { return forbidden_until[static_cast<size_t>(v) * n_col + c]; };
    for (uint32_t v = 0; v < n; ++v) colour[v] = v % n_col;
    for (uint32_t v = 0; v < n; ++v)
        for (int e = 0; e < 6; ++e) ++S(v, colour[g.nbr[6ull * v + e]]);
    int64_t clashes = 0;      // sum over spins of same-coloured neighbour entries (2 x edges)
    for (uint32_t v = 0; v < n; ++v) clashes += S(v, colour[v]);
    int64_t record = clashes;
    std::vector<uint32_t> clashing;
    clashing.reserve(n);
    for (uint32_t step = 1; step <= step_budget && clashes > 0; ++step) {
        clashing.clear();
        for (uint32_t v = 0; v < n; ++v)
            if (S(v, colour[v]) > 0) clashing.push_back(v);
        uint32_t r[4];
        rng(step, 0, 0, TAG_PARTITION, seed, r);
        const uint32_t v = clashing[r[0] % clashing.size()];
        const uint32_t cv = colour[v];
        const uint32_t* nv = &g.nbr[6ull * v];
        int64_t best_gain = 0;
        uint32_t partner = n;           // n = none yet
        for (uint32_t u = 0; u < n; ++u) {
            const uint32_t cu = colour[u];
            if (cu == cv) continue;
            const int32_t links = static_cast<int32_t>(std::count(nv, nv + 6, u));
            const int64_t gain = static_cast<int64_t>(S(v, cu)) - S(v, cv) + S(u, cv) - S(u, cu) - 2 * links;
            const bool blocked = F(v, cu) >= step || F(u, cv) >= step;
            if (blocked && clashes + 2 * gain >= record) continue;     // aspiration: a new record
            if (partner == n || gain < best_gain) { partner = u; best_gain = gain; }
        }
        if (partner == n) continue;
        const uint32_t u = partner, cu = colour[u];
        for (int e = 0; e < 6; ++e) { const uint32_t w = nv[e]; --S(w, cv); ++S(w, cu); }
        for (int e = 0; e < 6; ++e) { const uint32_t w = g.nbr[6ull * u + e]; --S(w, cu); ++S(w, cv); }
        colour[v] = cu;
        colour[u] = cv;
        clashes += 2 * best_gain;
        F(v, cv) = step + 5 + r[1] % 10;
        F(u, cu) = step + 5 + r[2] % 10;
        record = std::min(record, clashes);
    }
    if (clashes != 0) return false;
    g.order.clear();
    g.order.reserve(n);
    g.set_start.assign(1, 0);
    for (uint32_t c = 0; c < n_col; ++c) {
        for (uint32_t v = 0; v < n; ++v)
            if (colour[v] == c) g.order.push_back(v);
        g.set_start.push_back(static_cast<uint32_t>(g.order.size()));
    }
    return true;
}

// The update order of a generated instance: balanced on request, else (or on failure) greedy.
void make_sets(HostGraph& g, uint64_t seed, uint32_t set_cap, bool balanced)
{
    if (balanced && g.n <= 8192u) {     // the search costs O(N) per step: small instances only
        // default set size: the largest of 16, 32, 64, 128, 256 that still leaves at least 4 sets
        // (N = 256 -> 4 x 64, N = 192 -> 6 x 32, N = 512 -> 4 x 128): sets that fill a CTA of
        // 4 x size threads exactly
        uint32_t size = set_cap;
        if (size == 0) {
            size = 16;
            while (size < 256 && 2 * size <= g.n / 4) size *= 2;
        }
        const uint32_t n_col = std::max(4u, (g.n + size - 1) / size);
        if (balanced_sets(g, seed, n_col, 1000u + 200u * g.n)) return;
    }
    greedy_sets(g, set_cap);
}

}  // namespace

bool build_graph_from_seed(uint32_t n, uint64_t graph_seed, bool gauge, uint32_t set_cap,
                           bool balanced, HostGraph& g, std::string& err)
{
    g.n = n;
    const uint32_t n_stub = 3u * n;
    std::vector<uint64_t> key(n_stub);
    std::vector<uint32_t> perm(n_stub);
    g.tri.assign(3ull * n, 0);
    g.attempt = -1;
    for (uint32_t attempt = 0; attempt < 100000u; ++attempt) {
        for (uint32_t j = 0; j < n_stub; ++j) {
            uint32_t o[4];
            rng(j, attempt, 0, TAG_GRAPH, graph_seed, o);
            key[j] = (static_cast<uint64_t>(o[0]) << 32) | o[1];
        }
        std::iota(perm.begin(), perm.end(), 0u);
        std::sort(perm.begin(), perm.end(), [&](uint32_t a, uint32_t b) {
            return key[a] != key[b] ? key[a] < key[b] : a < b;
        });
        bool simple = true;
        for (uint32_t t = 0; t < n && simple; ++t) {
            const uint32_t a = perm[3 * t] / 3, b = perm[3 * t + 1] / 3, c = perm[3 * t + 2] / 3;
            simple = (a != b) && (b != c) && (a != c);
        }
        if (!simple) continue;
        for (uint32_t s = 0; s < n_stub; ++s) g.tri[s] = perm[s] / 3;
        g.attempt = static_cast<int>(attempt);
        break;
    }
    if (g.attempt < 0) { err = "configuration model: no simple hypergraph found"; return false; }

    g.jbit.assign(n, 0);
    if (gauge) {
        std::vector<uint8_t> tau(n);
        for (uint32_t i = 0; i < n; ++i) {
            uint32_t o[4];
            rng(i, 0, 0, TAG_GAUGE, graph_seed, o);
            tau[i] = static_cast<uint8_t>(o[0] & 1u);
        }
        for (uint32_t t = 0; t < n; ++t)
            g.jbit[t] = tau[g.tri[3ull * t]] ^ tau[g.tri[3ull * t + 1]] ^ tau[g.tri[3ull * t + 2]];
    }
    if (!derive_adjacency(g, err)) return false;
    make_sets(g, graph_seed, set_cap, balanced);
    return true;
}

bool build_graph_from_arrays(uint32_t n, const uint32_t* tri, const uint8_t* jbit,
                             const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
                             HostGraph& g, std::string& err)
{
    g.n = n;
    g.attempt = -1;
    g.tri.assign(tri, tri + 3ull * n);
    g.jbit.resize(n);
    for (uint32_t t = 0; t < n; ++t) g.jbit[t] = jbit[t] ? 1 : 0;
    if (!derive_adjacency(g, err)) return false;
    // order must be a permutation; every set an anti-clique (L277).
    std::vector<int64_t> set_of(n, -1);
    g.order.assign(order, order + n);
    g.set_start.assign(1, 0);
    uint64_t pos = 0;
    for (uint32_t s = 0; s < n_sets; ++s) {
        if (set_size[s] == 0) { err = "empty independent set"; return false; }
        for (uint32_t q = 0; q < set_size[s]; ++q, ++pos) {
            if (pos >= n) { err = "set sizes exceed N"; return false; }
            const uint32_t v = order[pos];
            if (v >= n || set_of[v] >= 0) { err = "order is not a permutation"; return false; }
            set_of[v] = s;
        }
        g.set_start.push_back(static_cast<uint32_t>(pos));
    }
    if (pos != n) { err = "set sizes do not sum to N"; return false; }
    for (uint32_t v = 0; v < n; ++v)
        for (int q = 0; q < 6; ++q)
            if (set_of[g.nbr[6ull * v + q]] == set_of[v]) {
                err = "a set contains two adjacent spins";
                return false;
            }
    return true;
}

}  // namespace xs
