/*
 * xs_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the quasi-greedy (QG) clone sweep of
 * arXiv 2102.09510.  One spin per byte (+1 / -1), scalar loops, no bit tricks,
 * no blocking, no code shared with the CUDA library under paper_2102_09510_b200/csrc.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may load it.
 *
 * What it follows (PAPER.md line numbers; readings R1..Rn are listed in DESIGN.md):
 *   - Hamiltonian H = -sum_{(i,j,k) in E} J_ijk s_i s_j s_k, N spins, N triplets, every
 *     spin in exactly 3 triplets, 3 distinct spins per triplet        (L41 Eq.(1))
 *   - QG rule: flip with prob. w_k, k = # unsatisfied interactions of the spin,
 *     w0 = 0, w1 = 0.055, w2 = w3 = 1                                 (L65-L67, L101)
 *   - clones = independent copies from random initial states          (L73-L85)
 *   - one random number per word of clones                            (L87)
 *   - sweep = sets of mutually non-adjacent spins one after another, which equals a
 *     sequential sweep in the order of the permutation array          (L277-L289)
 *   - exact sweep of first ground-state hit per clone; TTS = min over clones (L293, L111)
 *   - PRNG: Philox4x32-10 (BASELINE.json north_star; the paper's Parisi-Rapuano generator
 *     is only cited, L287)
 *
 * Pins (tests/test_oracle_*.py): Philox known-answer vectors; generator invariants;
 * planted state E = -N; brute force N <= 20 (min E = -N, #minima = 2^nullity, L59 fn.1);
 * Delta E = 6 - 4k against full recomputation; gauge covariance; set-parallel ==
 * sequential; absorbing ground state; stationary <E>/N ~ -(1-w1)/(1+w1).
 * "parity unpinned": absolute TTS seconds of Table 1 (V100 wall clock, instances missing).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define XSO_TAG_GRAPH 1u
#define XSO_TAG_GAUGE 2u
#define XSO_TAG_INIT  3u
#define XSO_TAG_SWEEP 4u

/* ---- Philox4x32-10 (Salmon et al. 2011, the Random123 definition) -------------------
 * per round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * then k0 += 0x9E3779B9, k1 += 0xBB67AE85 ; M0 = 0xD2511F53, M1 = 0xCD9E8D57.          */
void xso_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_seeded(uint32_t a, uint32_t b, uint32_t c, uint32_t tag, uint64_t seed,
                          uint32_t out[4])
{
    uint32_t ctr[4] = { a, b, c, tag };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    xso_philox4x32_10(ctr, key, out);
}

/* ---- instance: random 3-regular 3-uniform hypergraph (L43; DESIGN.md R-graph) --------
 * Configuration model.  Stub j = 0..3N-1 belongs to node j/3.  Attempt a = 0,1,...:
 * sort the stubs by the 64-bit key (o0<<32)|o1 of Philox(ctr=(j,a,0,GRAPH), key=seed),
 * ties by j; consecutive triples of the sorted stubs are the triplets.  The first attempt
 * whose triplets all have three distinct nodes is accepted.                              */
typedef struct { uint64_t key; uint32_t stub; } stub_key;

static int cmp_stub_key(const void* pa, const void* pb)
{
    const stub_key* a = (const stub_key*)pa;
    const stub_key* b = (const stub_key*)pb;
    if (a->key < b->key) return -1;
    if (a->key > b->key) return 1;
    if (a->stub < b->stub) return -1;
    if (a->stub > b->stub) return 1;
    return 0;
}

/* tri: [N][3].  Returns the accepted attempt index (>= 0), or -1 on allocation failure
 * or if max_attempts attempts were all rejected. */
int xso_gen_triplets(uint32_t N, uint64_t graph_seed, uint32_t max_attempts, uint32_t* tri)
{
    uint32_t n_stub = 3u * N;
    stub_key* sk = (stub_key*)malloc(sizeof(stub_key) * (size_t)n_stub);
    if (!sk) return -1;
    for (uint32_t a = 0; a < max_attempts; ++a) {
        for (uint32_t j = 0; j < n_stub; ++j) {
            uint32_t o[4];
            philox_seeded(j, a, 0u, XSO_TAG_GRAPH, graph_seed, o);
            sk[j].key = ((uint64_t)o[0] << 32) | (uint64_t)o[1];
            sk[j].stub = j;
        }
        qsort(sk, n_stub, sizeof(stub_key), cmp_stub_key);
        int ok = 1;
        for (uint32_t t = 0; t < N; ++t) {
            uint32_t i = sk[3 * t + 0].stub / 3u;
            uint32_t j = sk[3 * t + 1].stub / 3u;
            uint32_t k = sk[3 * t + 2].stub / 3u;
            tri[3 * t + 0] = i; tri[3 * t + 1] = j; tri[3 * t + 2] = k;
            if (i == j || j == k || i == k) ok = 0;
        }
        if (ok) { free(sk); return (int)a; }
    }
    free(sk);
    return -1;
}

/* ---- planted gauge (BASELINE.json configs; L43 explains why the paper needs none) ----
 * taubit_i = o0 & 1 of Philox(ctr=(i,0,0,GAUGE), key=graph seed); tau_i = 1 - 2 taubit_i;
 * J_t = tau_i tau_j tau_k, stored as jbit_t = taubit_i ^ taubit_j ^ taubit_k (1 <=> J=-1). */
void xso_gen_gauge(uint32_t N, uint64_t graph_seed, uint8_t* taubit)
{
    for (uint32_t i = 0; i < N; ++i) {
        uint32_t o[4];
        philox_seeded(i, 0u, 0u, XSO_TAG_GAUGE, graph_seed, o);
        taubit[i] = (uint8_t)(o[0] & 1u);
    }
}

void xso_couplings_from_gauge(uint32_t N, const uint32_t* tri, const uint8_t* taubit,
                              uint8_t* jbit)
{
    for (uint32_t t = 0; t < N; ++t) {
        int J = 1;
        for (int m = 0; m < 3; ++m) J *= (taubit[tri[3 * t + m]] ? -1 : 1);
        jbit[t] = (uint8_t)(J < 0 ? 1 : 0);
    }
}

/* ---- adjacency: the "N x 6 matrix" of L287 ------------------------------------------
 * For spin i, its three clauses in ascending clause id r = 0,1,2; nbr[i][2r], nbr[i][2r+1]
 * are the other two members in their stored order; cls[i][r] is the clause id.
 * Returns 0, or -1 if some spin is not in exactly three clauses. */
int xso_adjacency(uint32_t N, const uint32_t* tri, uint32_t* nbr, uint32_t* cls)
{
    uint32_t* deg = (uint32_t*)calloc(N, sizeof(uint32_t));
    if (!deg) return -1;
    int rc = 0;
    for (uint32_t t = 0; t < N && rc == 0; ++t) {
        for (int m = 0; m < 3; ++m) {
            uint32_t i = tri[3 * t + m];
            if (i >= N || deg[i] >= 3u) { rc = -1; break; }
            uint32_t r = deg[i]++;
            cls[3 * i + r] = t;
            int q = 0;
            for (int m2 = 0; m2 < 3; ++m2) {
                if (m2 == m) continue;
                nbr[6 * i + 2 * r + q] = tri[3 * t + m2];
                ++q;
            }
        }
    }
    for (uint32_t i = 0; i < N && rc == 0; ++i) if (deg[i] != 3u) rc = -1;
    free(deg);
    return rc;
}

/* ---- update order: greedy independent sets (L279, L289; DESIGN.md R-order) -----------
 * Repeat until every node is assigned: S = [], blocked = {}; scan v = 0..N-1 ascending;
 * if v is unassigned, not blocked and (cap == 0 or |S| < cap): append v to S, mark it
 * assigned, block its 6 neighbours.  Append S to order, |S| to set_size.
 * Returns the number of sets, or -1 on failure. */
int xso_update_order(uint32_t N, const uint32_t* nbr, uint32_t cap, uint32_t* order,
                     uint32_t* set_size)
{
    uint8_t* assigned = (uint8_t*)calloc(N, 1);
    uint8_t* blocked = (uint8_t*)malloc(N);
    if (!assigned || !blocked) { free(assigned); free(blocked); return -1; }
    uint32_t n_done = 0, n_sets = 0;
    while (n_done < N) {
        memset(blocked, 0, N);
        uint32_t sz = 0;
        for (uint32_t v = 0; v < N; ++v) {
            if (assigned[v] || blocked[v]) continue;
            if (cap != 0u && sz >= cap) continue;
            order[n_done + sz] = v;
            ++sz;
            assigned[v] = 1;
            for (int q = 0; q < 6; ++q) blocked[nbr[6 * v + q]] = 1;
        }
        set_size[n_sets++] = sz;
        n_done += sz;
    }
    free(assigned); free(blocked);
    return (int)n_sets;
}

/* ---- update order, balanced variant (L281: sets sized "to keep the processing of components
 * as balanced as possible"; DESIGN.md R-balance) ---------------------------------------------
 * q sets of equal size (within one), found by a tabu search over colour swaps.  Every step is
 * integer and deterministic:
 *   col[i] = i mod q;  cnt[v][c] = number of the 6 entries nbr[v][.] with colour c;
 *   conf = sum_v cnt[v][col[v]];  best = conf;  tabu[v][c] = 0.
 *   for it = 1 .. max_it, while conf > 0:
 *     L = spins with cnt[v][col[v]] > 0, ascending;  rnd = Philox(ctr=(it,0,0,5), key=seed);
 *     v = L[rnd[0] mod |L|], a = col[v];
 *     among all u (ascending) with b = col[u] != a, m = multiplicity of u in nbr[v][.]:
 *         d = cnt[v][b] - cnt[v][a] + cnt[u][a] - cnt[u][b] - 2m      (change of conf / 2)
 *         u is skipped if (tabu[v][b] >= it or tabu[u][a] >= it) and not conf + 2d < best;
 *         keep the first u with the smallest d;
 *     none: next it.  Else swap the colours of v and u, update cnt of their neighbours,
 *     conf += 2d, tabu[v][a] = it + 5 + rnd[1] mod 10, tabu[u][b] = it + 5 + rnd[2] mod 10,
 *     best = min(best, conf).
 * conf == 0: set c = the spins of colour c in ascending order, sets in colour order; returns q.
 * Otherwise (or if q < 2 or q > N) returns 0 and the caller uses the greedy order. */
#define XSO_TAG_PARTITION 5u
int xso_balanced_order(uint32_t N, const uint32_t* nbr, uint64_t seed, uint32_t q,
                       uint32_t max_it, uint32_t* order, uint32_t* set_size)
{
    if (q < 2u || q > N) return 0;
    uint32_t* col = (uint32_t*)malloc(sizeof(uint32_t) * N);
    int32_t* cnt = (int32_t*)calloc((size_t)N * q, sizeof(int32_t));
    uint32_t* tabu = (uint32_t*)calloc((size_t)N * q, sizeof(uint32_t));
    uint32_t* L = (uint32_t*)malloc(sizeof(uint32_t) * N);
    if (!col || !cnt || !tabu || !L) { free(col); free(cnt); free(tabu); free(L); return -1; }
    const uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    for (uint32_t i = 0; i < N; ++i) col[i] = i % q;
    for (uint32_t v = 0; v < N; ++v)
        for (int k = 0; k < 6; ++k) cnt[(size_t)v * q + col[nbr[6 * v + k]]] += 1;
    int64_t conf = 0;
    for (uint32_t v = 0; v < N; ++v) conf += cnt[(size_t)v * q + col[v]];
    int64_t best = conf;
    for (uint32_t it = 1; it <= max_it && conf > 0; ++it) {
        uint32_t nL = 0;
        for (uint32_t v = 0; v < N; ++v)
            if (cnt[(size_t)v * q + col[v]] > 0) L[nL++] = v;
        const uint32_t ctr[4] = { it, 0u, 0u, XSO_TAG_PARTITION };
        uint32_t rnd[4];
        xso_philox4x32_10(ctr, key, rnd);
        const uint32_t v = L[rnd[0] % nL], a = col[v];
        int found = 0;
        uint32_t bu = 0;
        int32_t bd = 0;
        for (uint32_t u = 0; u < N; ++u) {
            const uint32_t b = col[u];
            if (b == a) continue;
            int32_t m = 0;
            for (int k = 0; k < 6; ++k) m += (nbr[6 * v + k] == u);
            const int32_t d = cnt[(size_t)v * q + b] - cnt[(size_t)v * q + a] +
                              cnt[(size_t)u * q + a] - cnt[(size_t)u * q + b] - 2 * m;
            const int is_tabu = tabu[(size_t)v * q + b] >= it || tabu[(size_t)u * q + a] >= it;
            if (is_tabu && !(conf + 2 * (int64_t)d < best)) continue;
            if (!found || d < bd) { found = 1; bu = u; bd = d; }
        }
        if (!found) continue;
        const uint32_t u = bu, b = col[u];
        for (int k = 0; k < 6; ++k) {
            const uint32_t w = nbr[6 * v + k];
            cnt[(size_t)w * q + a] -= 1; cnt[(size_t)w * q + b] += 1;
        }
        for (int k = 0; k < 6; ++k) {
            const uint32_t w = nbr[6 * u + k];
            cnt[(size_t)w * q + b] -= 1; cnt[(size_t)w * q + a] += 1;
        }
        col[v] = b; col[u] = a;
        conf += 2 * (int64_t)bd;
        tabu[(size_t)v * q + a] = it + 5u + rnd[1] % 10u;
        tabu[(size_t)u * q + b] = it + 5u + rnd[2] % 10u;
        if (conf < best) best = conf;
    }
    int rc = 0;
    if (conf == 0) {
        uint32_t p = 0;
        for (uint32_t c = 0; c < q; ++c) {
            uint32_t sz = 0;
            for (uint32_t v = 0; v < N; ++v)
                if (col[v] == c) { order[p++] = v; ++sz; }
            set_size[c] = sz;
        }
        rc = (int)q;
    }
    free(col); free(cnt); free(tabu); free(L);
    return rc;
}

/* 1 if every set is an anti-clique (no member is a neighbour of another member) and
 * order is a permutation of 0..N-1; else 0.  (L277: "nodes that are not directly
 * connected can be processed in parallel") */
int xso_check_order(uint32_t N, const uint32_t* nbr, const uint32_t* order,
                    const uint32_t* set_size, uint32_t n_sets)
{
    int32_t* set_of = (int32_t*)malloc(sizeof(int32_t) * N);
    if (!set_of) return 0;
    for (uint32_t v = 0; v < N; ++v) set_of[v] = -1;
    uint32_t p = 0;
    int ok = 1;
    for (uint32_t s = 0; s < n_sets && ok; ++s)
        for (uint32_t q = 0; q < set_size[s]; ++q, ++p) {
            if (p >= N || order[p] >= N || set_of[order[p]] != -1) { ok = 0; break; }
            set_of[order[p]] = (int32_t)s;
        }
    if (p != N) ok = 0;
    for (uint32_t v = 0; v < N && ok; ++v)
        for (int q = 0; q < 6; ++q)
            if (set_of[nbr[6 * v + q]] == set_of[v]) ok = 0;
    free(set_of);
    return ok;
}

/* ---- clones: random initial states (L77; DESIGN.md R-init) ---------------------------
 * word(i,w) = o0 | (o1 << 32) of Philox(ctr=(i,w,0,INIT), key=run seed); clone c = 64w+b
 * has s_i = -1 iff bit b of word(i,w) is set.  s: [64W][N] bytes, clone-major. */
void xso_init_spins(uint32_t N, uint32_t W, uint64_t run_seed, int8_t* s)
{
    for (uint32_t i = 0; i < N; ++i)
        for (uint32_t w = 0; w < W; ++w) {
            uint32_t o[4];
            philox_seeded(i, w, 0u, XSO_TAG_INIT, run_seed, o);
            uint64_t word = (uint64_t)o[0] | ((uint64_t)o[1] << 32);
            for (uint32_t b = 0; b < 64u; ++b) {
                size_t c = (size_t)64u * w + b;
                s[c * N + i] = ((word >> b) & 1u) ? (int8_t)-1 : (int8_t)1;
            }
        }
}

/* ---- energy (L41 Eq.(1) with couplings): E = -sum_t J_t s_i s_j s_k, full sum -------- */
int32_t xso_energy(uint32_t N, const uint32_t* tri, const uint8_t* jbit, const int8_t* s1)
{
    int32_t E = 0;
    for (uint32_t t = 0; t < N; ++t) {
        int J = jbit[t] ? -1 : 1;
        E -= J * s1[tri[3 * t + 0]] * s1[tri[3 * t + 1]] * s1[tri[3 * t + 2]];
    }
    return E;
}

/* k = number of unsatisfied interactions of spin i in one clone (L65: "flipping a spin
 * entering k unsatisfied interactions"); interaction r is unsatisfied iff
 * J_r s_i s_a s_b = -1. */
static int unsat_count(uint32_t i, const uint32_t* nbr, const uint32_t* cls,
                       const uint8_t* jbit, const int8_t* s1)
{
    int k = 0;
    for (int r = 0; r < 3; ++r) {
        int J = jbit[cls[3 * i + r]] ? -1 : 1;
        int prod = J * s1[i] * s1[nbr[6 * i + 2 * r]] * s1[nbr[6 * i + 2 * r + 1]];
        if (prod == -1) ++k;
    }
    return k;
}

/* ---- one QG sweep, number t (1-based), over words [w_begin, w_end) -------------------
 * (L65-L67, L87, L101, L277-L289; DESIGN.md R-noise, R-thr)
 * for p = 0..N-1: i = order[p]; for each word w:
 *     u = Philox(ctr=(i, w>>2, t, SWEEP), key=run seed)[w & 3];  R = (u < w1_threshold)
 *     for each clone c of word w: flip s_i iff k >= 2, or k == 1 and R.
 * mode 0: sequential in `order`.  mode 1: every set is updated from a snapshot taken at
 * the start of the set (the paper's parallel-inside-a-set semantics, L277); both must
 * agree bit for bit because sets are anti-cliques.
 * n_flips (optional) counts accepted flips; dE_mismatch (optional) counts flips whose
 * incremental Delta E = 6 - 4k differs from E_after - E_before by full recomputation
 * (only evaluated when check_dE != 0; very slow). */
/* General flip table (L67: "w_k the probability of flipping a spin entering k unsatisfied
 * interactions"; L69: w0 = w1^3 with w2 = w3 = 1 satisfies detailed balance = Metropolis): thr4[k] in [0, 2^32], the spin
 * flips iff u < thr4[k], with the SAME number u for every k (one number per word, L87).
 * The quasi-greedy rule of L67/L101 is thr4 = (0, floor(0.055 2^32), 2^32, 2^32). */
void xso_sweep_w(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
                 const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
                 const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
                 uint64_t run_seed, uint32_t t, const uint64_t* thr4, int mode,
                 int check_dE, int8_t* s, uint64_t* n_flips, uint64_t* dE_mismatch)
{
    int8_t* snap = NULL;
    if (mode == 1) snap = (int8_t*)malloc(N);
    for (uint32_t w = w_begin; w < w_end; ++w) {
        for (uint32_t b = 0; b < 64u; ++b) {
            int8_t* s1 = s + ((size_t)64u * w + b) * N;
            uint32_t p = 0;
            for (uint32_t st = 0; st < n_sets; ++st) {
                if (mode == 1) memcpy(snap, s1, N);
                for (uint32_t q = 0; q < set_size[st]; ++q, ++p) {
                    uint32_t i = order[p];
                    uint32_t o[4];
                    philox_seeded(i, w >> 2, t, XSO_TAG_SWEEP, run_seed, o);
                    uint64_t u = (uint64_t)o[w & 3u];
                    int k = unsat_count(i, nbr, cls, jbit, mode == 1 ? snap : s1);
                    int flip = (u < thr4[k]) ? 1 : 0;
                    if (!flip) continue;
                    if (check_dE) {
                        int32_t e0 = xso_energy(N, tri, jbit, s1);
                        s1[i] = (int8_t)-s1[i];
                        int32_t e1 = xso_energy(N, tri, jbit, s1);
                        if (e1 - e0 != 6 - 4 * k && dE_mismatch) ++*dE_mismatch;
                    } else {
                        s1[i] = (int8_t)-s1[i];
                    }
                    if (n_flips) ++*n_flips;
                }
            }
        }
    }
    free(snap);
}

/* The quasi-greedy table w = (0, w1, 1, 1) of L67 / L101. */
static void qg_table(uint32_t w1_threshold, uint64_t thr4[4])
{
    thr4[0] = 0;
    thr4[1] = (uint64_t)w1_threshold;
    thr4[2] = (uint64_t)1 << 32;
    thr4[3] = (uint64_t)1 << 32;
}

void xso_sweep(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
               const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
               const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
               uint64_t run_seed, uint32_t t, uint32_t w1_threshold, int mode,
               int check_dE, int8_t* s, uint64_t* n_flips, uint64_t* dE_mismatch)
{
    uint64_t thr4[4];
    qg_table(w1_threshold, thr4);
    xso_sweep_w(N, w_begin, w_end, tri, jbit, nbr, cls, order, set_size, n_sets, run_seed, t, thr4,
                mode, check_dE, s, n_flips, dE_mismatch);
}

/* ---- run: sweeps t_begin+1 .. t_begin+n_sweeps over words [w_begin,w_end) ------------
 * After each sweep, E_c by FULL recomputation; first_hit[c] = t at the first sweep after
 * which E_c = -N (L293 "the exact iteration ... is saved", L111).  first_hit must be
 * initialised by the caller (0xFFFFFFFF = none; xso_mark_initial handles t = 0).
 * No freezing of solved clones: E = -N is a fixed point because w0 = 0 (L65(iii), L69). */
void xso_mark_initial(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
                      const uint8_t* jbit, const int8_t* s, uint32_t* first_hit)
{
    for (size_t c = (size_t)64u * w_begin; c < (size_t)64u * w_end; ++c) {
        first_hit[c] = 0xFFFFFFFFu;
        if (xso_energy(N, tri, jbit, s + c * N) == -(int32_t)N) first_hit[c] = 0u;
    }
}

void xso_run_w(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
               const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
               const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
               uint64_t run_seed, uint32_t t_begin, uint32_t n_sweeps, const uint64_t* thr4,
               int8_t* s, uint32_t* first_hit)
{
    for (uint32_t t = t_begin + 1u; t <= t_begin + n_sweeps; ++t) {
        xso_sweep_w(N, w_begin, w_end, tri, jbit, nbr, cls, order, set_size, n_sets, run_seed,
                    t, thr4, 0, 0, s, NULL, NULL);
        for (size_t c = (size_t)64u * w_begin; c < (size_t)64u * w_end; ++c)
            if (first_hit[c] == 0xFFFFFFFFu &&
                xso_energy(N, tri, jbit, s + c * N) == -(int32_t)N)
                first_hit[c] = t;
    }
}

/* ---- per-clone noise variant (DESIGN.md R-clone) ------------------
 * L87: the paper draws ONE random number per word ("the same random number for the 32 clones in
 * the same word"), which couples the k = 1 decisions of word mates.  This variant gives every
 * clone its own number: for spin i, word w, sweep t and clone bit b,
 *     U = sum_{k=0..6} bit_b(r_k) 2^k,   r_{2j} = o0 | o1 << 32,  r_{2j+1} = o2 | o3 << 32
 *     with (o0..o3) = Philox(ctr = (i, 4w + j, t, 6), key = run seed), j = 0..3  (r_7 unused),
 * and a spin with k = 1 flips iff U < m, i.e. w1 = m / 128 (m = 7: 0.0547, inside the paper's
 * 0.054(1), L91).  k >= 2 always flips, k = 0 never (L67).  Same order, same sets as xso_sweep. */
#define XSO_TAG_CLONE 6u
void xso_sweep_clone(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint8_t* jbit,
                     const uint32_t* nbr, const uint32_t* cls, const uint32_t* order,
                     uint64_t run_seed, uint32_t t, uint32_t m, int8_t* s)
{
    for (uint32_t w = w_begin; w < w_end; ++w) {
        for (uint32_t p = 0; p < N; ++p) {           /* clones are independent: spin outer, clone inner */
            const uint32_t i = order[p];
            uint64_t r[8];
            for (uint32_t j = 0; j < 4u; ++j) {
                uint32_t o[4];
                philox_seeded(i, 4u * w + j, t, XSO_TAG_CLONE, run_seed, o);
                r[2 * j] = (uint64_t)o[0] | ((uint64_t)o[1] << 32);
                r[2 * j + 1] = (uint64_t)o[2] | ((uint64_t)o[3] << 32);
            }
            for (uint32_t b = 0; b < 64u; ++b) {
                int8_t* s1 = s + ((size_t)64u * w + b) * N;
                uint32_t U = 0;
                for (uint32_t k = 0; k < 7u; ++k) U |= (uint32_t)((r[k] >> b) & 1u) << k;
                const int k_unsat = unsat_count(i, nbr, cls, jbit, s1);
                const int flip = (k_unsat >= 2) || (k_unsat == 1 && U < m);
                if (flip) s1[i] = (int8_t)-s1[i];
            }
        }
    }
}

void xso_run_clone(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
                   const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
                   const uint32_t* order, uint64_t run_seed, uint32_t t_begin, uint32_t n_sweeps,
                   uint32_t m, int8_t* s, uint32_t* first_hit)
{
    for (uint32_t t = t_begin + 1u; t <= t_begin + n_sweeps; ++t) {
        xso_sweep_clone(N, w_begin, w_end, jbit, nbr, cls, order, run_seed, t, m, s);
        for (size_t c = (size_t)64u * w_begin; c < (size_t)64u * w_end; ++c)
            if (first_hit[c] == 0xFFFFFFFFu &&
                xso_energy(N, tri, jbit, s + c * N) == -(int32_t)N)
                first_hit[c] = t;
    }
}

void xso_run(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
             const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
             const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
             uint64_t run_seed, uint32_t t_begin, uint32_t n_sweeps, uint32_t w1_threshold,
             int8_t* s, uint32_t* first_hit)
{
    uint64_t thr4[4];
    qg_table(w1_threshold, thr4);
    xso_run_w(N, w_begin, w_end, tri, jbit, nbr, cls, order, set_size, n_sets, run_seed, t_begin,
              n_sweeps, thr4, s, first_hit);
}

/* Same as xso_run but words are distributed over OpenMP threads (words evolve
 * independently, L87).  Used only for the timed CPU baseline. */
void xso_run_omp(uint32_t N, uint32_t w_begin, uint32_t w_end, const uint32_t* tri,
                 const uint8_t* jbit, const uint32_t* nbr, const uint32_t* cls,
                 const uint32_t* order, const uint32_t* set_size, uint32_t n_sets,
                 uint64_t run_seed, uint32_t t_begin, uint32_t n_sweeps,
                 uint32_t w1_threshold, int8_t* s, uint32_t* first_hit)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t w = (int64_t)w_begin; w < (int64_t)w_end; ++w)
        xso_run(N, (uint32_t)w, (uint32_t)w + 1u, tri, jbit, nbr, cls, order, set_size,
                n_sets, run_seed, t_begin, n_sweeps, w1_threshold, s, first_hit);
}

/* ---- conversion between the oracle's bytes and the boundary's bit-packed words --------
 * x[i][w] bit b <-> clone 64w+b, bit 1 <=> s = -1 (DESIGN.md layout). */
void xso_pack(uint32_t N, uint32_t W, const int8_t* s, uint64_t* x)
{
    for (uint32_t i = 0; i < N; ++i)
        for (uint32_t w = 0; w < W; ++w) {
            uint64_t word = 0;
            for (uint32_t b = 0; b < 64u; ++b)
                if (s[((size_t)64u * w + b) * N + i] < 0) word |= (uint64_t)1 << b;
            x[(size_t)i * W + w] = word;
        }
}

void xso_unpack(uint32_t N, uint32_t W, const uint64_t* x, int8_t* s)
{
    for (uint32_t i = 0; i < N; ++i)
        for (uint32_t w = 0; w < W; ++w)
            for (uint32_t b = 0; b < 64u; ++b)
                s[((size_t)64u * w + b) * N + i] =
                    ((x[(size_t)i * W + w] >> b) & 1u) ? (int8_t)-1 : (int8_t)1;
}

#ifdef _OPENMP
#include <omp.h>
#endif
int xso_omp_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
