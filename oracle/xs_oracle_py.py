"""Second opinion for the C oracle: the same algorithm in ~100 lines of pure Python ints.

TEST INFRASTRUCTURE.  Written separately from xs_oracle.c (no shared code, Python big ints
instead of C unsigned arithmetic, lists instead of arrays) so that a slip in one of them
(a wrong index, a wrong counter slot, a sign) shows up as a disagreement in
tests/test_oracle_pins.py.  Small sizes only.  Citations: PAPER.md lines as in xs_oracle.c.
"""
M32 = 0xFFFFFFFF
GRAPH, GAUGE, INIT, SWEEP = 1, 2, 3, 4


def philox4x32_10(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = (p1 >> 32) ^ c1 ^ k0, p1 & M32, (p0 >> 32) ^ c3 ^ k1, p0 & M32
        k0 = (k0 + 0x9E3779B9) & M32
        k1 = (k1 + 0xBB67AE85) & M32
    return [c0, c1, c2, c3]


def _rng(a, b, c, tag, seed):
    return philox4x32_10([a, b, c, tag], [seed & M32, seed >> 32])


def gen_triplets(N, seed):
    """L43: N triplets, 3 distinct indices each, each index in exactly 3 triplets."""
    a = 0
    while True:
        keys = []
        for j in range(3 * N):
            o = _rng(j, a, 0, GRAPH, seed)
            keys.append(((o[0] << 32) | o[1], j))
        keys.sort()
        tri = [tuple(keys[3 * t + m][1] // 3 for m in range(3)) for t in range(N)]
        if all(len(set(t)) == 3 for t in tri):
            return tri, a
        a += 1


def gen_taubit(N, seed):
    return [_rng(i, 0, 0, GAUGE, seed)[0] & 1 for i in range(N)]


def clauses_of(N, tri):
    """L287: per spin its 3 clauses (ascending id) as (clause id, partner a, partner b)."""
    adj = [[] for _ in range(N)]
    for t, trip in enumerate(tri):
        for m, i in enumerate(trip):
            others = [trip[q] for q in range(3) if q != m]
            adj[i].append((t, others[0], others[1]))
    return adj


def update_order(N, adj, cap=0):
    """L279: greedy scan, sets of mutually non-adjacent nodes."""
    assigned, order, sizes = set(), [], []
    while len(assigned) < N:
        S, blocked = [], set()
        for v in range(N):
            if v in assigned or v in blocked or (cap and len(S) >= cap):
                continue
            S.append(v)
            assigned.add(v)
            for (_, a, b) in adj[v]:
                blocked.add(a)
                blocked.add(b)
        order += S
        sizes.append(len(S))
    return order, sizes


def init_spins(N, W, run_seed):
    """s[c][i] = +-1, clone c = 64w + b <- bit b of o0 | o1<<32 (L77)."""
    s = [[1] * N for _ in range(64 * W)]
    for i in range(N):
        for w in range(W):
            o = _rng(i, w, 0, INIT, run_seed)
            word = o[0] | (o[1] << 32)
            for b in range(64):
                if (word >> b) & 1:
                    s[64 * w + b][i] = -1
    return s


def energy(tri, J, s1):
    """Eq. (1), with couplings J_t = +-1."""
    return -sum(J[t] * s1[i] * s1[j] * s1[k] for t, (i, j, k) in enumerate(tri))


def sweep_table(N, W, adj, J, order, run_seed, t, thr4, s):
    """L67, L69: flip with probability w_k = thr4[k] / 2^32, the same number for every k."""
    for i in order:
        for w in range(W):
            u = _rng(i, w >> 2, t, SWEEP, run_seed)[w & 3]
            for b in range(64):
                s1 = s[64 * w + b]
                k = sum(1 for (c, a, bb) in adj[i] if J[c] * s1[i] * s1[a] * s1[bb] == -1)
                if u < thr4[k]:
                    s1[i] = -s1[i]


def sweep(N, W, adj, J, order, run_seed, t, thr, s):
    """L65-L67, L87, L101: w0 = 0, w1 = thr / 2^32, w2 = w3 = 1, one number per word."""
    for i in order:
        for w in range(W):
            R = _rng(i, w >> 2, t, SWEEP, run_seed)[w & 3] < thr
            for b in range(64):
                s1 = s[64 * w + b]
                k = sum(1 for (c, a, bb) in adj[i] if J[c] * s1[i] * s1[a] * s1[bb] == -1)
                if k >= 2 or (k == 1 and R):
                    s1[i] = -s1[i]


def sweep_clone(N, W, adj, J, order, run_seed, t, m, s):
    """SURVEY.md 8(f) NEXT-2 (DESIGN.md R-clone): every clone draws its own 7-bit number U from
    Philox(ctr=(i, 4w+j, t, 6)), j = 0..3; a k = 1 spin flips iff U < m (w1 = m / 128)."""
    for i in order:
        for w in range(W):
            r = []
            for j in range(4):
                o = _rng(i, 4 * w + j, t, 6, run_seed)
                r += [o[0] | (o[1] << 32), o[2] | (o[3] << 32)]
            for b in range(64):
                U = sum(((r[k] >> b) & 1) << k for k in range(7))
                s1 = s[64 * w + b]
                k = sum(1 for (c, a, bb) in adj[i] if J[c] * s1[i] * s1[a] * s1[bb] == -1)
                if k >= 2 or (k == 1 and U < m):
                    s1[i] = -s1[i]
