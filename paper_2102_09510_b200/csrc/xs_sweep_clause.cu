// xs_sweep_clause.cu -- host side of the clause-word sweep kernel (xs_sweep_clause.cuh): the
// round structure of an update order on a CTA of n_slots slots, the conflict-free placement of
// the clause rows in shared memory, eligibility, table upload and the dispatch to the
// instantiation units xs_sweep_clause_r<R>.cu.
#include <algorithm>
#include <cstdlib>

#include "xs_sweep_clause.cuh"

namespace xs {

void count_launch(uint64_t n);   // xs_diag.cu

extern template cudaError_t launch_clause_unit<4>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit<5>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit<6>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit<7>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit<8>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<9>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<10>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<11>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<12>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<13>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<14>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<15>(const ClauseArgs&, const ClauseLaunch&);
extern template cudaError_t launch_clause_unit_long<16>(const ClauseArgs&, const ClauseLaunch&);

namespace {

constexpr uint32_t CL_RMIN = 4, CL_RMAX = 16;     // rounds per sweep the kernel is instantiated for
constexpr uint32_t CL_RCAP = 8;                   // ... under the 128-register cap of the dense launch classes
constexpr uint32_t CL_SMEM_MAX = 227u * 1024u;

inline uint32_t clause_off_misc(uint32_t N, uint32_t n_slots) { return (N + n_slots / 2u) * 128u; }
inline uint32_t clause_smem(uint32_t N, uint32_t n_slots)
{
    return clause_off_misc(N, n_slots) + (6u * CL_T + 4u) * 4u + 128u;
}

struct Rng {
    uint64_t s;
    uint32_t next() { s ^= s << 13; s ^= s >> 7; s ^= s << 17; return (uint32_t)(s >> 32); }
};

}  // namespace

// Rounds a CTA of n_slots slots needs for one sweep of g's update order: a set of sz spins takes
// ceil(sz / n_slots) rounds.
uint32_t clause_rounds(const HostGraph& g, uint32_t n_slots)
{
    uint32_t r = 0;
    for (size_t s = 0; s + 1 < g.set_start.size(); ++s)
        r += (g.set_start[s + 1] - g.set_start[s] + n_slots - 1) / n_slots;
    return r;
}

// Placement for one instance on a CTA of n_slots slots (n_slots even).
//   half[t] in {0, 1} for every clause: the row of clause t is the lower / upper half of line t;
//   per set, the spins are paired: a spin whose clauses have halves (h1, h2, h3) with k ones pairs
//   with a spin of 3 - k ones; the first lists its clauses by ascending half, the second by
//   descending half, so that slots (2m, 2m+1), which share a shared-memory phase, touch opposite
//   halves in each of their three accesses.  A spin without a partner gets an idle neighbour slot,
//   which works on the opposite halves of scratch line N + m.  A set that needs nr = ceil(sz /
//   n_slots) rounds must fit its pairs into nr * n_slots / 2 slot pairs:
//       2 (max(a0, a3) + max(a1, a2)) <= nr * n_slots,  a_k = spins of the set with k upper halves,
//   which a randomised local search over half[] establishes (all integer, deterministic).
// Outputs: crec[e], e = round * n_slots + slot, for n_rounds rounds (entries of rounds >= the
// instance's own count are idle); cplace[t]; bar_mask bit r = round r ends a set; mode = the
// kernel MODE this instance allows (1 / 2: no idle slot, sets of one / two rounds; else 0).
// Returns false if the order does not fit (more than n_rounds rounds, more than 2 N entries) or
// no placement was found.
bool clause_placement(const HostGraph& g, uint32_t n_slots, uint32_t n_rounds, CRec* crec,
                      uint32_t* cplace, uint32_t* bar_mask, uint32_t* mode)
{
    const uint32_t N = g.n;
    const uint32_t n_sets = (uint32_t)g.set_start.size() - 1;
    if (n_slots < 2 || (n_slots & 1u) || n_rounds > CL_RMAX || (uint64_t)n_rounds * n_slots > 2ull * N)
        return false;
    if (clause_rounds(g, n_slots) > n_rounds) return false;
    std::vector<uint32_t> set_of(N), nr(n_sets), cap(n_sets);
    for (uint32_t s = 0; s < n_sets; ++s) {
        const uint32_t sz = g.set_start[s + 1] - g.set_start[s];
        nr[s] = (sz + n_slots - 1) / n_slots;
        cap[s] = nr[s] * n_slots;
        for (uint32_t p = g.set_start[s]; p < g.set_start[s + 1]; ++p) set_of[g.order[p]] = s;
    }
    std::vector<uint8_t> half(N), k(N, 0);
    std::vector<int> cnt((size_t)n_sets * 4, 0);
    Rng rng{0x9E3779B97F4A7C15ull ^ ((uint64_t)N << 32) ^ g.tri[0] ^ ((uint64_t)g.tri[1] << 16) ^
            ((uint64_t)n_slots << 48)};
    for (uint32_t t = 0; t < N; ++t) half[t] = (uint8_t)(rng.next() & 1u);
    for (uint32_t v = 0; v < N; ++v) {
        for (int c = 0; c < 3; ++c) k[v] += half[g.cls[3ull * v + c]];
        ++cnt[set_of[v] * 4 + k[v]];
    }
    auto set_cost = [&](uint32_t s) {
        const int* a = &cnt[s * 4];
        const int need = 2 * (std::max(a[0], a[3]) + std::max(a[1], a[2]));
        return std::max(0, need - (int)cap[s]);
    };
    auto total_cost = [&]() { int c = 0; for (uint32_t s = 0; s < n_sets; ++s) c += set_cost(s); return c; };
    auto toggle = [&](uint32_t t) {
        // every occurrence of clause t in a spin's clause list moves that spin's count by one
        const int d = half[t] ? -1 : 1;
        half[t] ^= 1u;
        for (int c = 0; c < 3; ++c) {
            const uint32_t v = g.tri[3ull * t + c];
            --cnt[set_of[v] * 4 + k[v]];
            k[v] = (uint8_t)(k[v] + d);
            ++cnt[set_of[v] * 4 + k[v]];
        }
    };
    int cost = total_cost();
    for (uint64_t it = 0; cost > 0 && it < 2000ull * N + 100000ull; ++it) {
        const uint32_t t = rng.next() % N;
        toggle(t);
        const int nc = total_cost();
        if (nc <= cost || (rng.next() & 15u) == 0u) cost = nc;
        else toggle(t);
    }
    if (cost != 0) return false;

    for (uint32_t t = 0; t < N; ++t) cplace[t] = (t << 7) | ((uint32_t)half[t] << 6);
    const uint32_t pairs_per_round = n_slots / 2;
    uint32_t round0 = 0, bm = 0;
    bool all_one = true, all_two = true, any_idle = false;
    // first slot of a pair: clauses by ascending half; second slot: descending
    auto rows = [&](uint32_t v, bool descending, uint32_t (&off)[3]) {
        uint32_t cl[3] = {g.cls[3ull * v], g.cls[3ull * v + 1], g.cls[3ull * v + 2]};
        std::stable_sort(cl, cl + 3, [&](uint32_t a, uint32_t b) {
            return descending ? half[a] > half[b] : half[a] < half[b];
        });
        for (int c = 0; c < 3; ++c) off[c] = cplace[cl[c]];
    };
    for (uint32_t s = 0; s < n_sets; ++s) {
        std::vector<uint32_t> by_k[4];
        for (uint32_t p = g.set_start[s]; p < g.set_start[s + 1]; ++p) by_k[k[g.order[p]]].push_back(g.order[p]);
        // slot pairs of the set: (first, second) with CL_IDLE where a spin has no partner
        std::vector<std::pair<uint32_t, uint32_t>> pairs;
        for (int lo = 0; lo < 2; ++lo) {
            const std::vector<uint32_t>&a = by_k[lo], &b = by_k[3 - lo];
            const size_t m = std::min(a.size(), b.size());
            for (size_t q = 0; q < m; ++q) pairs.push_back({a[q], b[q]});
            for (size_t q = m; q < a.size(); ++q) pairs.push_back({a[q], CL_IDLE});
            for (size_t q = m; q < b.size(); ++q) pairs.push_back({CL_IDLE, b[q]});
        }
        if (pairs.size() > (size_t)nr[s] * pairs_per_round) return false;
        size_t next = 0;
        for (uint32_t q = 0; q < nr[s]; ++q) {
            // the set's rounds get equal shares of its pairs
            const size_t left = pairs.size() - next, rounds_left = nr[s] - q;
            const size_t take = std::min<size_t>((left + rounds_left - 1) / rounds_left, pairs_per_round);
            for (uint32_t m = 0; m < pairs_per_round; ++m) {
                CRec* e = crec + (size_t)(round0 + q) * n_slots + 2 * m;
                const uint32_t scratch = (N + m) << 7;
                uint32_t va = CL_IDLE, vb = CL_IDLE;
                if (m < take) { va = pairs[next + m].first; vb = pairs[next + m].second; }
                uint32_t oa[3] = {scratch, scratch, scratch};
                uint32_t ob[3] = {scratch | 64u, scratch | 64u, scratch | 64u};
                if (va != CL_IDLE) rows(va, false, oa);
                if (vb != CL_IDLE) rows(vb, true, ob);
                // an idle slot mirrors its neighbour on the scratch line
                if (va == CL_IDLE && vb != CL_IDLE)
                    for (int c = 0; c < 3; ++c) oa[c] = scratch | ((ob[c] & 64u) ^ 64u);
                if (vb == CL_IDLE && va != CL_IDLE)
                    for (int c = 0; c < 3; ++c) ob[c] = scratch | ((oa[c] & 64u) ^ 64u);
                e[0] = CRec{oa[0], oa[1], oa[2], va};
                e[1] = CRec{ob[0], ob[1], ob[2], vb};
                if (va == CL_IDLE || vb == CL_IDLE) any_idle = true;
                // check: the two slots of a shared-memory phase touch opposite halves
                if (!(((oa[0] ^ ob[0]) & (oa[1] ^ ob[1]) & (oa[2] ^ ob[2])) & 64u)) return false;
            }
            next += take;
        }
        if (next != pairs.size()) return false;
        round0 += nr[s];
        bm |= 1u << (round0 - 1);
        if (nr[s] != 1) all_one = false;
        if (nr[s] != 2) all_two = false;
    }
    // rounds this instance does not have: idle on the scratch lines
    for (uint32_t r = round0; r < n_rounds; ++r)
        for (uint32_t m = 0; m < pairs_per_round; ++m) {
            const uint32_t scratch = (N + m) << 7;
            crec[(size_t)r * n_slots + 2 * m] = CRec{scratch, scratch, scratch, CL_IDLE};
            crec[(size_t)r * n_slots + 2 * m + 1] = CRec{scratch | 64u, scratch | 64u, scratch | 64u, CL_IDLE};
            any_idle = true;
        }
    // bits 16-18 of an entry's spin field: this round is the LAST touch of its clause 0 / 1 / 2 in a
    // sweep (the kernels for tables with w0 > 0 OR the clause words there: all clear <=> E = -N)
    {
        std::vector<uint32_t> round_of(N, 0), last_round(N, 0);
        for (uint32_t e = 0; e < round0 * n_slots; ++e)
            if (crec[e].spin != CL_IDLE) round_of[crec[e].spin] = e / n_slots;
        for (uint32_t t = 0; t < N; ++t)
            last_round[t] = std::max({round_of[g.tri[3ull * t]], round_of[g.tri[3ull * t + 1]],
                                      round_of[g.tri[3ull * t + 2]]});
        for (uint32_t e = 0; e < round0 * n_slots; ++e) {
            CRec& c = crec[e];
            if (c.spin == CL_IDLE) continue;
            const uint32_t r = e / n_slots;
            const uint32_t off[3] = {c.off0, c.off1, c.off2};
            for (int k = 0; k < 3; ++k)
                if (last_round[off[k] >> 7] == r) c.spin |= 1u << (16 + k);
        }
    }
    if (bar_mask) *bar_mask = bm;
    if (mode) *mode = any_idle ? 0u : all_one ? 1u : all_two ? 2u : 0u;
    return true;
}

// Called after choose_geometry: moves an on-chip batch with the quasi-greedy table to the clause
// kernel (variant 2) when its update orders fit, and uploads the placement tables on first use.
int clause_prepare(xs_batch& b, void* stream)
{
    TileGeom& g = b.geom;
    const xs_geometry& rq = b.req;
    if (rq.variant != XS_GEOM_AUTO && rq.variant != 2u) return 0;   // another kernel was asked for
    if (g.regime != 0 || (b.p.flags & XS_FLAG_STREAMING)) return 0;
    // flip tables: the quasi-greedy form (0, w1, 1, 1) and, on full lists (MODE 1), the family
    // (w0, w1, 1, 1) with 0 < w0 <= w1 (L69: Metropolis w0 = w1^3); anything else: generic kernel
    const bool family = b.ft.general && b.ft.always == 0xCu && b.ft.lo[0] > 0u && b.ft.lo[0] <= b.ft.lo[1];
    if (b.ft.general && !family) return 0;
    const bool special = family || b.ft.per_clone;     // forms that exist for the full 4-8 round lists only
    if (rq.tile_words && rq.tile_words != CL_T) return 0;
    const uint32_t N = b.p.n_spins, I = b.p.n_instances, W = b.p.n_words;
    if (W % CL_T || N < 64u || N >= (1u << 14)) return 0;
    // CTA size: the one that needs the fewest rounds per sweep (ties: the smaller CTA)
    uint32_t threads = 0, rounds = ~0u;
    for (uint32_t thr : {128u, 256u, 512u}) {
        if (rq.threads && rq.threads != thr) continue;
        const uint32_t ns = thr / CL_LPS;
        if (clause_smem(N, ns) > CL_SMEM_MAX) continue;
        uint32_t r = 0;
        for (const HostGraph& hg : b.graphs) r = std::max(r, clause_rounds(hg, ns));
        r = std::max(r, CL_RMIN);
        if (r > CL_RMAX || (uint64_t)r * ns > 2ull * N) continue;
        if (r > CL_RCAP && thr > 256u) continue;           // long lists: CTAs of at most 256 threads
        if (r < rounds) { rounds = r; threads = thr; }
    }
    if (!threads) return 0;
    const uint32_t n_slots = threads / CL_LPS;
    // Measured: with ragged sets that leave more than 30 % of the slots idle
    // (greedy orders at N = 512: 7 rounds on 128 slots) the generic kernel on 16-column tiles, where
    // the rule found one per SM, is faster (20.7 k against 19.1 k updates/ns)
    if (rq.variant == XS_GEOM_AUTO && g.variant == 0 && g.T == 16 &&
        (uint64_t)N * 10u < (uint64_t)rounds * n_slots * 7u)
        return 0;
    if (b.clause_state == 2 && b.clause_slots == n_slots) return 0;   // placement failed earlier
    if (b.clause_state != 1 || b.clause_slots != n_slots || b.clause_rounds != rounds) {
        const size_t ent = crec_entries(b.p);
        std::vector<CRec> crec((size_t)I * ent, CRec{0u, 0u, 0u, CL_IDLE});
        std::vector<uint32_t> cplace((size_t)I * N), cbar(I);
        uint32_t mode = 3;
        b.clause_slots = n_slots;
        for (uint32_t i = 0; i < I; ++i) {
            uint32_t m = 0;
            if (!clause_placement(b.graphs[i], n_slots, rounds, crec.data() + (size_t)i * ent,
                                  cplace.data() + (size_t)i * N, &cbar[i], &m)) {
                b.clause_state = 2;
                return 0;
            }
            mode = (mode == 3 || mode == m) ? m : 0u;
        }
        cudaStream_t st = (cudaStream_t)stream;
        cudaError_t e = cudaMemcpyAsync(b.d.crec, crec.data(), crec.size() * sizeof(CRec),
                                        cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(b.d.cplace, cplace.data(), cplace.size() * 4, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(b.d.cbar, cbar.data(), cbar.size() * 4, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // staging vectors die at return
        if (e != cudaSuccess) return (int)e;
        b.clause_state = 1;
        b.warp_passes = 0;         // the latency kernel's tables (same buffer) are gone
        b.clause_rounds = rounds;
        b.clause_mode = mode == 3 ? 0u : mode;
    }
    if (special && (b.clause_mode != 1u || rounds > CL_RCAP)) return 0;     // w0 > 0 / per-clone noise: full lists
    if (b.clause_thr != (uint64_t)b.p.w1_threshold) {
        // compare constants of the noise (xs_sweep_clause.cuh): 2^32 - thr, and the forced carry for thr = 0
        const uint32_t h[2] = {0u - b.p.w1_threshold, b.p.w1_threshold == 0u ? 1u : 0u};
        cudaStream_t st = (cudaStream_t)stream;
        cudaError_t e = cudaMemcpyAsync(b.d.cthr, h, sizeof h, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return (int)e;
        b.clause_thr = b.p.w1_threshold;
    }
    g.variant = 2;
    // detection pass + tile store every 256 sweeps (measured +3 % over 64; a replay, which happens
    // when a clone first reaches E = -N, re-runs at most one batch).  xs_geometry.batch_sweeps overrides.
    g.batch = rq.batch_sweeps ? rq.batch_sweeps : 256u;
    g.T = CL_T;
    g.CW = 2;
    g.threads = threads;
    g.ctas = I * (W / CL_T);
    g.smem = clause_smem(N, n_slots);
    g.rb = 0;
    return 0;
}

int launch_sweep_clause(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    const TileGeom& g = b.geom;
    ClauseArgs A;
    A.d = b.d;
    A.N = b.p.n_spins; A.W = b.p.n_words; A.n_sweeps = n_sweeps;
    A.flags = b.p.flags; A.batch = g.batch;
    A.n_slots = g.threads / CL_LPS;
    A.ent = crec_entries(b.p);
    A.off_misc = clause_off_misc(b.p.n_spins, A.n_slots);
    A.thr = b.ft.general ? b.ft.lo[1] : b.p.w1_threshold;
    A.thr0 = b.ft.general ? b.ft.lo[0] : 0u;
    A.one = 1u;
    A.zero = 0u;
    ClauseLaunch L;
    L.threads = g.threads; L.smem = g.smem; L.mode = b.clause_mode;
    L.w0 = b.ft.general != 0u;
    L.pcn = b.ft.per_clone != 0u;
    A.clone_m = b.ft.clone_m;
    L.dense = g.ctas > b.num_sms;
    L.st = (cudaStream_t)stream;
    const uint32_t tiles = b.p.n_words / CL_T;
    for (uint32_t i0 = 0; i0 < b.p.n_instances; i0 += CL_MAXI) {
        const uint32_t ni = std::min(CL_MAXI, b.p.n_instances - i0);
        A.inst0 = i0;
        for (uint32_t i = 0; i < CL_MAXI; ++i) A.seed[i] = i < ni ? b.run_seeds[i0 + i] : 0ull;
        L.ctas = ni * tiles;
        cudaError_t e;
        switch (b.clause_rounds) {
            case 4: e = launch_clause_unit<4>(A, L); break;
            case 5: e = launch_clause_unit<5>(A, L); break;
            case 6: e = launch_clause_unit<6>(A, L); break;
            case 7: e = launch_clause_unit<7>(A, L); break;
            case 8: e = launch_clause_unit<8>(A, L); break;
            case 9: e = launch_clause_unit_long<9>(A, L); break;
            case 10: e = launch_clause_unit_long<10>(A, L); break;
            case 11: e = launch_clause_unit_long<11>(A, L); break;
            case 12: e = launch_clause_unit_long<12>(A, L); break;
            case 13: e = launch_clause_unit_long<13>(A, L); break;
            case 14: e = launch_clause_unit_long<14>(A, L); break;
            case 15: e = launch_clause_unit_long<15>(A, L); break;
            default: e = launch_clause_unit_long<16>(A, L); break;
        }
        if (e != cudaSuccess) return (int)e;
        count_launch(1);
    }
    return 0;
}

}  // namespace xs
