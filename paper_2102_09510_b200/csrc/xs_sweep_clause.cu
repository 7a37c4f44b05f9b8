// xs_sweep_clause.cu -- the clause-word sweep kernel: same tile ownership, static task list, noise
// and first-hit logic as k_sweep_static (xs_sweep_static.cuh), but shared memory holds the
// CLAUSE words instead of the spin words:
//
//     c_t = x_i ^ x_j ^ x_k ^ Jmask_t      (bit = 1 <=> interaction t unsatisfied)
//
// A spin's update then needs only its three clause words: k = number of set bits among
// (c_1, c_2, c_3) (L67), M = maj, P = parity, flip = M | (P & R) (k >= 2 always, k = 1 with the
// word's noise mask R, k = 0 never: L65, L101), and flipping the spin toggles its three clauses:
// c_r ^= flip, x ^= flip.  The spin words themselves live only in the registers of the thread
// that owns the spin (and in global memory at batch boundaries).  Per task (128 clones of one
// spin): 3 LDS.128 + 3 STS.128 against the 6 + 2 accesses of the spin-word kernel, and the same 7
// logic operations per 32 clones.  Spins of one independent set share no clause (L277),
// so the read-modify-write of the clause rows is race free inside a round.
//
// Bank conflicts: a T = 8 clause row is 64 B = half of a 128-byte line, and the 8 lanes of one
// shared-memory phase serve two slots.  The host places every clause in the lower or upper half
// of its own line (half[t]) and pairs the spins of every set so that the two slots of a phase
// touch opposite halves in each of their three accesses (clause_placement below): single copy,
// conflict free, no second store.
//
// Eligibility (clause_prepare): quasi-greedy table, T = 8, 2 words per lane, exactly 4 or 6 sets that
// fill all slots of the CTA (balanced sets, DESIGN.md R-balance).  Everything else runs on
// k_sweep_static / k_sweep_tile.  The update order inside a set is free (L277), so results are
// bit-identical to the oracle's.
#include <algorithm>
#include <cstdlib>
#include <type_traits>

#include <cuda_runtime.h>

#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

void count_launch(uint64_t n);   // xs_diag.cu

namespace {

constexpr int CL_RMAX = 6;     // rounds (= sets) per sweep: 4 or 6
constexpr int CL_H = 4;        // uint32 halves per lane (2 uint64 words)
constexpr uint32_t CL_T = 8;   // tile width in uint64 columns
constexpr uint32_t CL_LPS = 4; // lanes per slot

struct ClauseArgs {
    DevPtrs d;
    uint32_t N, W, n_sweeps, thr, flags, batch;
    uint32_t off_misc;
};

__device__ __forceinline__ void lds4(uint32_t addr, uint32_t (&o)[4])
{
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void sts4(uint32_t addr, const uint32_t (&o)[4])
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "r"(addr), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
}
__device__ __forceinline__ uint32_t prmt_b(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
constexpr int LUT_OR_AND = 0xF8;   // a | (b & c)

template <int CL_R, int MAXTHREADS, int MINB>
__global__ void __launch_bounds__(MAXTHREADS, MINB) k_sweep_clause(ClauseArgs A)
{
    constexpr uint32_t NL = 2;         // lanes sharing a Philox call = sweeps per noise period
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t N = A.N, W = A.W;
    const uint32_t tiles = W / CL_T;
    const uint32_t inst = blockIdx.x / tiles;
    const uint32_t w0 = (blockIdx.x % tiles) * CL_T;
    const xs_tts_rec rec0 = A.d.rec[inst];
    if (rec0.solved && !(A.flags & XS_FLAG_NO_SKIP)) return;   // stop rule (L129, L293)

    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    uint32_t* det32 = reinterpret_cast<uint32_t*>(smem + A.off_misc);
    uint32_t* known32 = det32 + 2 * CL_T;
    uint32_t* flag = known32 + 2 * CL_T;

    const uint32_t slot = threadIdx.x / CL_LPS, n_slots = blockDim.x / CL_LPS;
    const uint32_t j = threadIdx.x % CL_LPS;
    const uint32_t lane_off = base + j * 16u;

    const uint64_t seed = A.d.run_seed[inst];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w0;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w0) * 64;

    // ---- static task list: round r = set r, this thread's spin = entry r * n_slots + slot -----
    uint32_t ca[CL_R][3];     // shared addresses of the spin's three clause rows
    uint32_t spin[CL_R];
    uint32_t x[CL_R][CL_H];   // the spin's words: registers only
    uint32_t rm[CL_R], rmn[CL_R];
    {
        const uint4* cr = reinterpret_cast<const uint4*>(A.d.crec + (size_t)inst * N);
#pragma unroll
        for (int r = 0; r < CL_R; ++r) {
            const uint4 v = cr[r * n_slots + slot];
            ca[r][0] = lane_off + v.x;
            ca[r][1] = lane_off + v.y;
            ca[r][2] = lane_off + v.z;
            spin[r] = v.w;
            rm[r] = 0;
            rmn[r] = 0;
        }
    }

    // a-3: clause rows from the spin words in global memory; own words into registers
    auto load_state = [&]() {
        const ClauseRec* cl = A.d.clause + (size_t)inst * N;
        const uint32_t* place = A.d.cplace + (size_t)inst * N;
        for (uint32_t e = threadIdx.x; e < N * CL_T; e += blockDim.x) {
            const uint32_t t = e / CL_T, lw = e - t * CL_T;
            const ClauseRec c = cl[t];
            const uint64_t v = xg[(size_t)c.i * W + lw] ^ xg[(size_t)c.j * W + lw] ^
                               xg[(size_t)c.k * W + lw] ^ (c.jbit ? ~0ull : 0ull);
            *reinterpret_cast<uint64_t*>(smem + place[t] + 8u * lw) = v;
        }
#pragma unroll
        for (int r = 0; r < CL_R; ++r) {
            const uint4 v = *reinterpret_cast<const uint4*>(xg + (size_t)spin[r] * W + 2u * j);
            x[r][0] = v.x; x[r][1] = v.y; x[r][2] = v.z; x[r][3] = v.w;
        }
    };
    // a-10: every spin is owned by exactly one slot
    auto store_state = [&]() {
#pragma unroll
        for (int r = 0; r < CL_R; ++r)
            *reinterpret_cast<uint4*>(xg + (size_t)spin[r] * W + 2u * j) =
                make_uint4(x[r][0], x[r][1], x[r][2], x[r][3]);
    };
    load_state();
    for (uint32_t e = threadIdx.x; e < 64 * CL_T; e += blockDim.x) {
        const bool kn = fhg[e] != XS_NO_HIT;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, kn);
        if ((threadIdx.x & 31) == 0) known32[e >> 5] = m;
    }
    __syncthreads();

    // ---- noise (a-6), as in k_sweep_static with CW = 2: the two lanes that share a Philox word
    // group each compute one sweep of a two-sweep period and exchange the threshold bytes ------
    const uint32_t grp = (w0 + 2u * j) >> 2;
    const uint32_t jl = j % NL;
    const uint32_t sub = (2u * j) & 3u;
    const int lane_base = (int)(threadIdx.x & 31u) - (int)jl;
    const uint32_t thr = A.thr;
    auto noise_call = [&](int r, uint32_t q) -> uint32_t {
        uint32_t o[4];
        philox4x32_10(spin[r], grp, NL * q + jl, TAG_SWEEP, k0, k1, o);
        const uint32_t v = (o[0] < thr ? 0xFFu : 0u) | (o[1] < thr ? 0xFF00u : 0u) |
                           (o[2] < thr ? 0xFF0000u : 0u) | (o[3] < thr ? 0xFF000000u : 0u);
        const uint32_t s0 = __shfl_sync(0xFFFFFFFFu, v, lane_base);
        const uint32_t s1 = __shfl_sync(0xFFFFFFFFu, v, lane_base + 1);
        return prmt_b(s0, s1, sub ? 0x7632u : 0x5410u);
    };
    auto produce_all = [&](uint32_t q) {
#pragma unroll
        for (int r = 0; r < CL_R; ++r) rm[r] = noise_call(r, q);
    };

    // ---- one sweep (a-4..a-8); h = index of the sweep inside the noise period; the Philox calls
    // of period qn for the rounds r = h (mod NL) sit in the latency shadow of the loads ---------
    auto sweep = [&](auto hc, uint32_t qn) {
        constexpr uint32_t h = decltype(hc)::value;
        constexpr uint32_t sel0 = 0x8888u + 0x1111u * (2u * h);
#pragma unroll
        for (int r = 0; r < CL_R; ++r) {
            uint32_t c0[CL_H], c1[CL_H], c2[CL_H];
            lds4(ca[r][0], c0); lds4(ca[r][1], c1); lds4(ca[r][2], c2);
            uint32_t R[2];
            R[0] = prmt_b(rm[r], 0u, sel0);
            R[1] = prmt_b(rm[r], 0u, sel0 + 0x1111u);
            if ((uint32_t)r % NL == h) rmn[r] = noise_call(r, qn);   // compile-time test
#pragma unroll
            for (int c = 0; c < CL_H; ++c) {
                const uint32_t M = lop3<LUT_MAJ>(c0[c], c1[c], c2[c]);    // k >= 2
                const uint32_t P = lop3<LUT_XOR3>(c0[c], c1[c], c2[c]);   // k odd
                const uint32_t f = lop3<LUT_OR_AND>(M, P, R[c >> 1]);     // flip mask (a-7)
                c0[c] ^= f; c1[c] ^= f; c2[c] ^= f;
                x[r][c] ^= f;
            }
            sts4(ca[r][0], c0); sts4(ca[r][1], c1); sts4(ca[r][2], c2);
            __syncthreads();                                          // a-8
        }
    };

    // ---- solved mask of the tile -> det32 (bit set = some interaction unsatisfied) ----------
    auto detect = [&]() {
        for (uint32_t e = threadIdx.x; e < 2 * CL_T; e += blockDim.x) det32[e] = 0;
        if (threadIdx.x == 0) *flag = 0;
        __syncthreads();
        uint32_t acc[CL_H] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int r = 0; r < CL_R; ++r) {
            uint32_t c0[CL_H], c1[CL_H], c2[CL_H];
            lds4(ca[r][0], c0); lds4(ca[r][1], c1); lds4(ca[r][2], c2);
#pragma unroll
            for (int c = 0; c < CL_H; ++c) acc[c] |= c0[c] | c1[c] | c2[c];
        }
#pragma unroll
        for (int c = 0; c < CL_H; ++c)
            if (acc[c]) atomicOr(&det32[CL_H * j + c], acc[c]);
        __syncthreads();
    };

    // sweeps t0+1 .. t0+n; exact: record first hits after every sweep (L293)
    auto run_range = [&](uint32_t t0, uint32_t n, bool exact) {
        const uint32_t t_first = t0 + 1, t_last = t0 + n;
        const uint32_t q_last = t_last / NL;
        bool have_next = false;
        for (uint32_t q = t_first / NL; q <= q_last; ++q) {
            if (have_next) {
#pragma unroll
                for (int r = 0; r < CL_R; ++r) rm[r] = rmn[r];
            } else {
                produce_all(q);
            }
            const bool fuse = (NL * q >= t_first) && (NL * q + NL - 1 <= t_last) && (q < q_last);
            auto step = [&](auto hc) {
                const uint32_t t = NL * q + decltype(hc)::value;
                if (t < t_first || t > t_last) return;
                sweep(hc, q + 1);
                if (exact) {
                    detect();
                    for (uint32_t e = threadIdx.x; e < 2 * CL_T; e += blockDim.x) {
                        uint32_t newly = ~det32[e] & ~known32[e];
                        known32[e] |= newly;
                        while (newly) {
                            const int bit = __ffs(newly) - 1;
                            newly &= newly - 1;
                            fhg[32 * e + bit] = t;
                        }
                    }
                    __syncthreads();
                }
            };
            step(std::integral_constant<uint32_t, 0>{});
            step(std::integral_constant<uint32_t, 1>{});
            have_next = fuse;
        }
    };

    uint32_t t = (uint32_t)rec0.sweeps_done;
    uint32_t remaining = A.n_sweeps;
    while (remaining) {
        const uint32_t nb = min(A.batch, remaining);
        run_range(t, nb, false);
        detect();
        for (uint32_t e = threadIdx.x; e < 2 * CL_T; e += blockDim.x)
            if (~det32[e] & ~known32[e]) *flag = 1;
        __syncthreads();
        const bool replay = *flag != 0;
        __syncthreads();
        if (replay) {
            load_state();          // global copy = state at the start of this batch
            __syncthreads();
            run_range(t, nb, true);
        }
        store_state();             // a-10 (also the replay checkpoint of the next batch)
        t += nb;
        remaining -= nb;
    }
}

inline uint32_t clause_off_misc(uint32_t N) { return N * 128u; }
inline uint32_t clause_smem(uint32_t N) { return clause_off_misc(N) + (4u * CL_T + 4u) * 4u + 128u; }

template <int R, int MT, int MINB>
cudaError_t launch_k(const ClauseArgs& A, uint32_t ctas, uint32_t threads, uint32_t smem, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(k_sweep_clause<R, MT, MINB>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_sweep_clause<R, MT, MINB><<<ctas, threads, smem, st>>>(A);
    return cudaGetLastError();
}
template <int R>
cudaError_t launch_r(const ClauseArgs& A, const TileGeom& g, uint32_t num_sms, cudaStream_t st)
{
    const bool dense = g.ctas > num_sms;   // more tiles than SMs: cap the registers, 16 warps per SM
    if (g.threads == 128) return launch_k<R, 128, 4>(A, g.ctas, g.threads, g.smem, st);
    if (g.threads == 256) return dense ? launch_k<R, 256, 2>(A, g.ctas, g.threads, g.smem, st)
                                       : launch_k<R, 256, 1>(A, g.ctas, g.threads, g.smem, st);
    if (g.threads == 1024) return launch_k<R, 1024, 1>(A, g.ctas, g.threads, g.smem, st);
    return launch_k<R, 512, 1>(A, g.ctas, g.threads, g.smem, st);
}

struct Rng {
    uint64_t s;
    uint32_t next() { s ^= s << 13; s ^= s >> 7; s ^= s << 17; return (uint32_t)(s >> 32); }
};

}  // namespace

// Placement for one instance: half[t] in {0, 1} for every clause and, per set, a pairing of the
// spins such that the spins on slots (2m, 2m+1) see opposite halves in each of their three
// accesses.  A spin whose clauses have halves (h1, h2, h3), k ones, pairs with a spin of 3 - k
// ones: the first lists its clauses by ascending half, the second by descending half.  Needed per
// set: #(k = 0) = #(k = 3) and #(k = 1) = #(k = 2); found by a randomised local search over
// half[] (2 constraints per set, N free bits).  All integer, deterministic.
// crec[e] = (row offset of clause 1, 2, 3, spin) for entry e = set * n_slots + slot;
// cplace[t] = row offset of clause t.  Returns false if the instance is not eligible.
bool clause_placement(const HostGraph& g, uint32_t n_slots, CRec* crec, uint32_t* cplace)
{
    const uint32_t N = g.n;
    const int CL_R = (int)g.set_start.size() - 1;
    if ((CL_R != 4 && CL_R != 6) || (n_slots & 1u) || N != (uint32_t)CL_R * n_slots) return false;
    for (int s = 0; s < CL_R; ++s)
        if (g.set_start[s + 1] - g.set_start[s] != n_slots) return false;
    std::vector<uint8_t> set_of(N), half(N), k(N, 0);
    for (uint32_t pos = 0; pos < N; ++pos) set_of[g.order[pos]] = (uint8_t)(pos / n_slots);
    int cnt[CL_RMAX][4] = {};
    Rng rng{0x9E3779B97F4A7C15ull ^ ((uint64_t)N << 32) ^ g.tri[0] ^ ((uint64_t)g.tri[1] << 16)};
    for (uint32_t t = 0; t < N; ++t) half[t] = (uint8_t)(rng.next() & 1u);
    for (uint32_t v = 0; v < N; ++v) {
        for (int c = 0; c < 3; ++c) k[v] += half[g.cls[3ull * v + c]];
        ++cnt[set_of[v]][k[v]];
    }
    auto set_cost = [&](int s) { return std::abs(cnt[s][0] - cnt[s][3]) + std::abs(cnt[s][1] - cnt[s][2]); };
    auto total_cost = [&]() { int c = 0; for (int s = 0; s < CL_R; ++s) c += set_cost(s); return c; };
    auto toggle = [&](uint32_t t) {
        // every occurrence of clause t in a spin's clause list moves that spin's count by one
        const int d = half[t] ? -1 : 1;
        half[t] ^= 1u;
        for (int c = 0; c < 3; ++c) {
            const uint32_t v = g.tri[3ull * t + c];
            --cnt[set_of[v]][k[v]];
            k[v] = (uint8_t)(k[v] + d);
            ++cnt[set_of[v]][k[v]];
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
    for (int s = 0; s < CL_R; ++s) {
        std::vector<uint32_t> by_k[4];
        for (uint32_t q = 0; q < n_slots; ++q) {
            const uint32_t v = g.order[g.set_start[s] + q];
            by_k[k[v]].push_back(v);
        }
        uint32_t e = (uint32_t)s * n_slots;
        auto emit = [&](uint32_t v, bool descending) {
            uint32_t cl[3] = {g.cls[3ull * v], g.cls[3ull * v + 1], g.cls[3ull * v + 2]};
            std::stable_sort(cl, cl + 3, [&](uint32_t a, uint32_t b) {
                return descending ? half[a] > half[b] : half[a] < half[b];
            });
            crec[e++] = CRec{cplace[cl[0]], cplace[cl[1]], cplace[cl[2]], v};
        };
        for (int lo = 0; lo < 2; ++lo)
            for (size_t m = 0; m < by_k[lo].size(); ++m) {
                emit(by_k[lo][m], false);
                emit(by_k[3 - lo][m], true);
            }
        // check: the two slots of every shared-memory phase touch opposite halves
        for (uint32_t m = (uint32_t)s * n_slots; m < e; m += 2) {
            const CRec a = crec[m], b = crec[m + 1];
            if (!(((a.off0 ^ b.off0) & (a.off1 ^ b.off1) & (a.off2 ^ b.off2)) & 64u)) return false;
        }
    }
    return true;
}

// Called after choose_geometry: switches an eligible static-kernel geometry to the clause kernel
// (variant 2) and uploads the placement tables on first use.
int clause_prepare(xs_batch& b, void* stream)
{
    TileGeom& g = b.geom;
    if (b.req.variant != XS_GEOM_AUTO && b.req.variant != 2u) return 0;   // another kernel was asked for
    if (g.regime != 0 || g.variant != 1 || g.CW != 2 || b.ft.general || b.ft.per_clone) return 0;
    if (b.clause_state == 2) return 0;                        // placement failed earlier
    const uint32_t N = b.p.n_spins, I = b.p.n_instances;
    uint32_t threads = g.threads;
    if (g.T == 4 && b.p.n_words % CL_T == 0 && b.max_set_size == 256) {
        // sets of 256 spins (N = 1024): the static kernel runs them on T = 4 tiles with 512 threads;
        // here one 1024-thread CTA (32 warps, 64 registers) keeps a T = 8 tile
        threads = 1024;
    } else if (g.T != CL_T) {
        return 0;
    }
    const uint32_t n_slots = threads / CL_LPS;
    if (threads != 128 && threads != 256 && threads != 512 && threads != 1024) return 0;
    if (clause_smem(N) > 227u * 1024u) return 0;
    if (b.clause_state == 0 || b.clause_slots != n_slots) {
        std::vector<CRec> crec((size_t)I * N);
        std::vector<uint32_t> cplace((size_t)I * N);
        for (uint32_t i = 0; i < I; ++i)
            if (!clause_placement(b.graphs[i], n_slots, crec.data() + (size_t)i * N,
                                  cplace.data() + (size_t)i * N)) {
                b.clause_state = 2;
                return 0;
            }
        cudaStream_t st = (cudaStream_t)stream;
        cudaError_t e = cudaMemcpyAsync(b.d.crec, crec.data(), crec.size() * sizeof(CRec),
                                        cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(b.d.cplace, cplace.data(), cplace.size() * 4, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // staging vectors die at return
        if (e != cudaSuccess) return (int)e;
        b.clause_state = 1;
        b.clause_slots = n_slots;
        b.clause_rounds = (uint32_t)b.graphs[0].set_start.size() - 1;   // equal for all instances (N = rounds x slots)
    }
    g.variant = 2;
    // detection pass + tile store every 256 sweeps (measured +3 % over 64; a replay, which happens
    // when a clone first reaches E = -N, re-runs at most one batch).  xs_geometry.batch_sweeps overrides.
    if (!b.req.batch_sweeps) g.batch = 256;
    g.T = CL_T;
    g.threads = threads;
    g.ctas = I * (b.p.n_words / CL_T);
    g.smem = clause_smem(N);
    return 0;
}

int launch_sweep_clause(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    const TileGeom& g = b.geom;
    ClauseArgs A;
    A.d = b.d;
    A.N = b.p.n_spins; A.W = b.p.n_words; A.n_sweeps = n_sweeps;
    A.thr = b.p.w1_threshold; A.flags = b.p.flags; A.batch = g.batch;
    A.off_misc = clause_off_misc(b.p.n_spins);
    cudaStream_t st = (cudaStream_t)stream;
    const cudaError_t e = b.clause_rounds == 6 ? launch_r<6>(A, g, b.num_sms, st) : launch_r<4>(A, g, b.num_sms, st);
    if (e != cudaSuccess) return (int)e;
    count_launch(1);
    return 0;
}

}  // namespace xs
