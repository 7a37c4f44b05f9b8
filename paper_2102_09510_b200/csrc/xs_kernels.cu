// xs_kernels.cu -- the CUDA path of the quasi-greedy clone sweep (sm_100a).
//
// Kernels:
//   k_init          a-2   random initial clone words from Philox(INIT)
//   k_sweep_tile    a-3..a-10  on-chip regime: a CTA owns (instance, T word columns), keeps the
//                   tile in shared memory for all sweeps of the call               (L293-L295)
//   k_stream_set    a-4..a-9   streaming regime: one launch per independent set, state in HBM/L2;
//                   <CW, true>: per-clone noise variant
//   (k_sweep_static, the register-resident work-list kernel of configs 2-4, lives in
//    xs_sweep_static.cuh)
//   k_unsat_or / k_mark / k_stream_commit   a-9/a-11  ground-state detection, first-hit table
//   k_energy_*      a-11  per-clone energies                                       (L41 Eq.(1))
//   k_finalize      a-11/a-12  per-instance min first-hit, solved flag, sweep counter (L111)
//
// The update itself (a-4..a-7), per 32 clones, all Boolean (L87 "multi-spin coding"):
//   w_r = x_a ^ x_b ^ Jmask_r            r = 0,1,2      clause fields without the spin itself
//   M = maj(w_0,w_1,w_2), P = w_0^w_1^w_2               bit-sliced adder of the three
//   unsatisfied-clause count of the spin: k = 2 (M^x) + (P^x) by self-duality of maj / parity
//   QG rule w = (0, w1, 1, 1) (L65-L67, L101): flip = (M^x) | ((P^x) & R)
//     R = 0  -> x_new = M ;  R = ~0 -> x_new = maj(M, P, ~x)
//   R = all-ones iff the word's 32-bit Philox output is below w1_threshold (L87: one random
//   number per word of clones).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

// ------------------------------------------------------------------------------------------
// a-2: initial state.  word(i,w) = o0 | o1 << 32 of Philox(ctr = (i, w, 0, INIT), key = run seed)
// ------------------------------------------------------------------------------------------
__global__ void k_init(DevPtrs d, uint32_t N, uint32_t W, uint32_t I)
{
    const uint64_t total = (uint64_t)I * N * W;
    for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t w = (uint32_t)(e % W);
        const uint32_t i = (uint32_t)((e / W) % N);
        const uint32_t inst = (uint32_t)(e / ((uint64_t)W * N));
        const uint64_t seed = d.run_seed[inst];
        uint32_t o[4];
        philox4x32_10(i, w, 0u, TAG_INIT, (uint32_t)seed, (uint32_t)(seed >> 32), o);
        d.x[e] = (uint64_t)o[0] | ((uint64_t)o[1] << 32);
    }
}

// ------------------------------------------------------------------------------------------
// a-9 / a-11: ground-state detection from global memory.
// det[inst][w] |= OR over clauses of (x_i ^ x_j ^ x_k ^ Jmask): bit c set <=> clone c has an
// unsatisfied clause <=> E_c > -N (L41: each of the N terms is >= -1).
// grid = (clause chunks, I); a thread owns words w = tid, tid + blockDim, ...
// ------------------------------------------------------------------------------------------
__global__ void k_unsat_or(DevPtrs d, uint32_t N, uint32_t W, uint32_t chunk, uint64_t* det)
{
    const uint32_t inst = blockIdx.y;
    const uint32_t c0 = blockIdx.x * chunk;
    const uint32_t c1 = min(c0 + chunk, N);
    const ClauseRec* cl = d.clause + (size_t)inst * N;
    const uint64_t* x = d.x + (size_t)inst * N * W;
    for (uint32_t w = blockIdx.z * blockDim.x + threadIdx.x; w < W; w += gridDim.z * blockDim.x) {
        uint64_t acc = 0;
        for (uint32_t c = c0; c < c1; ++c) {
            const ClauseRec r = cl[c];
            const uint64_t jm = r.jbit ? ~0ull : 0ull;
            acc |= x[(size_t)r.i * W + w] ^ x[(size_t)r.j * W + w] ^ x[(size_t)r.k * W + w] ^ jm;
        }
        if (acc) atomicOr(reinterpret_cast<unsigned long long*>(det + (size_t)inst * W + w), acc);
    }
}

// first_hit[clone] = sweeps_done[inst] for clones whose det bit is clear.  reset != 0: rewrite
// the whole table (XS_NO_HIT elsewhere); reset == 0: only fill entries that are XS_NO_HIT.
__global__ void k_mark(DevPtrs d, uint32_t W, uint32_t I, const uint64_t* det, int reset,
                       uint32_t t_add)
{
    const uint64_t total = (uint64_t)I * W * 64;
    for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t inst = (uint32_t)(e / ((uint64_t)W * 64));
        const uint64_t word = det[e >> 6];
        const bool solved = ((word >> (e & 63)) & 1ull) == 0;
        const uint32_t t_now = (uint32_t)d.rec[inst].sweeps_done + t_add;
        if (reset)
            d.first_hit[e] = solved ? t_now : XS_NO_HIT;
        else if (solved && d.first_hit[e] == XS_NO_HIT)
            d.first_hit[e] = t_now;
    }
}

// ------------------------------------------------------------------------------------------
// a-11: energies.  E_c = -N + 2 U_c, U_c = number of unsatisfied clauses of clone c.
// Bit-sliced vertical counters per thread (multi-spin coding of the count, L87), then expanded.
// grid = (W, I, clause chunks)
// ------------------------------------------------------------------------------------------
constexpr uint32_t EN_THREADS = 256;
constexpr uint32_t EN_MAX_CPT = 252;     // clauses per thread: 8 count planes hold <= 255; multiple of 4

__global__ void k_energy_fill(int32_t* out, uint64_t total, int32_t value)
{
    for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (uint64_t)gridDim.x * blockDim.x)
        out[e] = value;
}

// LANES <-> CONSECUTIVE WORDS of a spin row (LW = 2^lw_shift <= 32 of them), so that every gather
// x[i][w0 .. w0+LW) is one contiguous, fully used 8 LW-byte segment; the 256 / LW lane groups of a
// CTA take different clauses of the CTA's chunk.  Per thread the unsatisfied-clause count of its
// word's 64 clones is kept bit-sliced in 8 planes; four clause words enter per step through a
// carry-save adder tree (full adder = one XOR3 + one MAJ per 32 clones).
// grid = (word blocks x clause chunks, I)
__global__ void __launch_bounds__(EN_THREADS) k_energy_acc(DevPtrs d, uint32_t N, uint32_t W,
                                                          uint32_t lw_shift, uint32_t wblocks,
                                                          uint32_t cpt, int32_t* out)
{
    __shared__ int cnt[32 * 64];
    const uint32_t inst = blockIdx.y;
    const uint32_t wblock = blockIdx.x % wblocks, chunk = blockIdx.x / wblocks;
    const uint32_t LW = 1u << lw_shift, groups = EN_THREADS >> lw_shift;
    const uint32_t wl = threadIdx.x & (LW - 1u), cg = threadIdx.x >> lw_shift;
    const uint32_t w = wblock * LW + wl;
    const bool valid = w < W;
    for (uint32_t e = threadIdx.x; e < LW * 64u; e += EN_THREADS) cnt[e] = 0;
    __syncthreads();
    const ClauseRec* cl = d.clause + (size_t)inst * N;
    const uint64_t* x = d.x + (size_t)inst * N * W + (valid ? w : 0u);
    const uint32_t c_first = chunk * groups * cpt + cg;      // this thread: c_first, + groups, ...
    auto unsat = [&](uint32_t c) -> uint64_t {
        if (c >= N || !valid) return 0ull;
        const ClauseRec r = cl[c];
        return x[(size_t)r.i * W] ^ x[(size_t)r.j * W] ^ x[(size_t)r.k * W] ^ (r.jbit ? ~0ull : 0ull);
    };
    uint64_t pl[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (uint32_t q = 0; q < cpt; q += 4) {
        const uint32_t c = c_first + q * groups;
        const uint64_t u0 = unsat(c), u1 = unsat(c + groups), u2 = unsat(c + 2 * groups),
                       u3 = unsat(c + 3 * groups);
        const uint64_t s1 = u0 ^ u1 ^ u2, c1 = (u0 & u1) | (u2 & (u0 ^ u1));          // weight 1, 2
        const uint64_t s2 = s1 ^ u3 ^ pl[0], c2 = (s1 & u3) | (pl[0] & (s1 ^ u3));    // weight 1, 2
        pl[0] = s2;
        const uint64_t s3 = c1 ^ c2 ^ pl[1];
        uint64_t carry = (c1 & c2) | (pl[1] & (c1 ^ c2));                             // weight 4
        pl[1] = s3;
#pragma unroll
        for (int p = 2; p < 8; ++p) {
            const uint64_t t = pl[p] ^ carry;
            carry &= pl[p];
            pl[p] = t;
        }
    }
    if (valid) {
        for (int b = 0; b < 64; ++b) {
            int v = 0;
#pragma unroll
            for (int p = 0; p < 8; ++p) v |= (int)((pl[p] >> b) & 1ull) << p;
            if (v) atomicAdd(&cnt[wl * 64u + b], v);
        }
    }
    __syncthreads();
    int32_t* o = out + ((size_t)inst * W + (size_t)wblock * LW) * 64;
    const uint32_t n_valid = min(LW, W - wblock * LW) * 64u;
    for (uint32_t e = threadIdx.x; e < n_valid; e += EN_THREADS)
        if (cnt[e]) atomicAdd(o + e, 2 * cnt[e]);
}

// ------------------------------------------------------------------------------------------
// a-11 / a-12: per-instance record.  TTS = min_c first_hit (L111); smallest clone on ties.
// One CTA per instance.
// ------------------------------------------------------------------------------------------
constexpr uint32_t FIN_THREADS = 1024;

__global__ void __launch_bounds__(FIN_THREADS) k_finalize(DevPtrs d, uint32_t W, uint32_t n_sweeps,
                                                          uint32_t flags)
{
    __shared__ unsigned long long best[FIN_THREADS / 32];
    const uint32_t inst = blockIdx.x;
    const uint32_t C = 64 * W;                       // multiple of 64: 16-byte loads of four entries
    const uint4* fh = reinterpret_cast<const uint4*>(d.first_hit + (size_t)inst * C);
    unsigned long long m = ~0ull;
    for (uint32_t q = threadIdx.x; q < C / 4; q += FIN_THREADS) {
        const uint4 v = fh[q];
        const uint32_t t[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const unsigned long long key = ((unsigned long long)t[k] << 32) | (4u * q + k);
            m = key < m ? key : m;
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long v = __shfl_xor_sync(0xFFFFFFFFu, m, o);
        m = v < m ? v : m;
    }
    if ((threadIdx.x & 31) == 0) best[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (uint32_t q = 1; q < FIN_THREADS / 32; ++q) m = best[q] < m ? best[q] : m;
        xs_tts_rec r = d.rec[inst];
        const bool skipped = r.solved && !(flags & XS_FLAG_NO_SKIP);
        if (!skipped) r.sweeps_done += n_sweeps;
        const uint32_t t = (uint32_t)(m >> 32);
        r.solved = (t != XS_NO_HIT) ? 1u : 0u;
        r.tts_sweeps = t;
        r.clone = (t != XS_NO_HIT) ? (uint32_t)m : XS_NO_HIT;
        r._pad = 0;
        d.rec[inst] = r;
    }
}

// ------------------------------------------------------------------------------------------
// a-3 .. a-10: on-chip regime.
//
// A CTA owns tile (inst, word columns [w0, w0 + T)) for the whole call: the N x T uint64 tile
// lives in shared memory as rows x[i][0..T) (copy in, ~100 sweeps, copy
// out).  Unlike the paper's lanes <-> spins mapping (L277), LANES <-> CLONE WORDS of one spin
// row: the LPS = T / CW lanes that share a spin read the same partner rows, so every gather is
// a contiguous row read and the partner indices are shared by the lane group.  Different lane
// groups ("slots") take different spins of the current independent set; __syncthreads() after
// each set (L277).
//
// Noise: the Philox outputs of a whole chunk of sweeps are turned into one byte per
// (sweep, position, word) (0xFF <=> u32 < w1_threshold) by all threads in a produce phase, so
// that each Philox call (4 words) is computed once and off the update's critical path.
//
// Ground-state detection (a-9) without touching the hot loop: every `batch` sweeps the CTA
// runs a detection pass (k != 0 accumulate over all spins).  If a clone not yet in the
// first-hit table is solved, the batch is replayed from the copy of the tile in global memory
// (written at every batch boundary) with a detection pass after every sweep, which yields the
// exact first-hit sweep (L293); counter-based noise makes the replay bit-identical.
// ------------------------------------------------------------------------------------------
struct TileArgs {
    DevPtrs d;
    FlipTable ft;
    uint32_t N, W, T, n_sweeps, thr, flags, batch, rb;
    uint32_t off_rec, off_rbuf, off_sets, off_misc;   // byte offsets in dynamic shared memory
};

template <int CW>
struct TileCtx {
    unsigned char* state;     // [N][T] uint64
    const uint4* rec;         // [N][2]: {o0,o1,o2,o3}, {o4,o5,own offset, coupling bytes}
    unsigned char* rbuf;      // [rb][N][T] bytes
    const uint32_t* sets;     // [n_sets + 1]
    uint32_t* det32;          // [2T]
    uint32_t* known32;        // [2T]
    uint32_t* flag;
    uint32_t N, T, n_sets, slot, n_slots, joff /* byte offset of this lane's words in a row */,
        jw /* first local word of this lane */, row_shift /* log2(bytes of a row) */;
};

template <int CW>
__device__ __forceinline__ void tile_gather(const TileCtx<CW>& c, uint32_t p, uint32_t (&a)[3][2 * CW],
                                            uint32_t (&b)[3][2 * CW], uint32_t (&x)[2 * CW],
                                            uint32_t (&jm)[3], uint32_t& self_off)
{
    const uint4 r0 = c.rec[2 * p], r1 = c.rec[2 * p + 1];
    vload<CW>(c.state + r0.x + c.joff, a[0]);
    vload<CW>(c.state + r0.y + c.joff, b[0]);
    vload<CW>(c.state + r0.z + c.joff, a[1]);
    vload<CW>(c.state + r0.w + c.joff, b[1]);
    vload<CW>(c.state + r1.x + c.joff, a[2]);
    vload<CW>(c.state + r1.y + c.joff, b[2]);
    vload<CW>(c.state + r1.z + c.joff, x);
    self_off = r1.z;
    // coupling masks from the bytes 0x00 / 0xFF of r1.w (sign extension = one PRMT each)
    jm[0] = (uint32_t)(int32_t)(int8_t)(r1.w & 0xFFu);
    jm[1] = (uint32_t)(int32_t)(int8_t)((r1.w >> 8) & 0xFFu);
    jm[2] = (uint32_t)(int32_t)(int8_t)((r1.w >> 16) & 0xFFu);
}

// one sweep over all sets, sweep slot `rs` of the random-byte ring
template <int CW, bool GEN>
__device__ __forceinline__ void tile_sweep(const TileCtx<CW>& c, uint32_t rs)
{
    const unsigned char* rb = c.rbuf + (size_t)rs * c.N * c.T + c.jw;
    for (uint32_t s = 0; s < c.n_sets; ++s) {
        const uint32_t p1 = c.sets[s + 1];
        for (uint32_t p = c.sets[s] + c.slot; p < p1; p += c.n_slots) {
            uint32_t a[3][2 * CW], b[3][2 * CW], x[2 * CW], jm[3], self_off;
            tile_gather<CW>(c, p, a, b, x, jm, self_off);
            uint32_t nb[CW];          // noise byte of each word
            if (CW == 2) {
                const uint32_t two = *reinterpret_cast<const unsigned short*>(rb + (size_t)p * c.T);
                nb[0] = two & 0xFFu;
                nb[CW - 1] = two >> 8;
            } else {
                nb[0] = rb[(size_t)p * c.T];
            }
            uint32_t xn[2 * CW];
            if (GEN) {
                // general table: bit k of the byte <=> number below the threshold of w_k
#pragma unroll
                for (int h = 0; h < 2 * CW; ++h) {
                    const uint32_t v = nb[h >> 1];
                    xn[h] = table_update(a[0][h], b[0][h], jm[0], a[1][h], b[1][h], jm[1], a[2][h],
                                         b[2][h], jm[2], x[h], 0u - (v & 1u), 0u - ((v >> 1) & 1u),
                                         0u - ((v >> 2) & 1u), 0u - ((v >> 3) & 1u));
                }
            } else {
#pragma unroll
                for (int h = 0; h < 2 * CW; ++h)
                    xn[h] = qg_update(a[0][h], b[0][h], jm[0], a[1][h], b[1][h], jm[1], a[2][h], b[2][h],
                                      jm[2], x[h], (uint32_t)(int32_t)(int8_t)nb[h >> 1]);
            }
            vstore<CW>(c.state + self_off + c.joff, xn);
        }
        __syncthreads();
    }
}

// det32[] |= words with bit set where some spin of the clone has k != 0 (clone not in a ground
// state).  Caller zeroes det32 and puts barriers around.
template <int CW>
__device__ __forceinline__ void tile_detect_acc(const TileCtx<CW>& c)
{
    uint32_t acc[2 * CW];
#pragma unroll
    for (int h = 0; h < 2 * CW; ++h) acc[h] = 0;
    for (uint32_t p = c.slot; p < c.N; p += c.n_slots) {
        uint32_t a[3][2 * CW], b[3][2 * CW], x[2 * CW], jm[3], self_off;
        tile_gather<CW>(c, p, a, b, x, jm, self_off);
#pragma unroll
        for (int h = 0; h < 2 * CW; ++h)
            acc[h] |= qg_nonzero_k(a[0][h], b[0][h], jm[0], a[1][h], b[1][h], jm[1], a[2][h], b[2][h],
                                   jm[2], x[h]);
    }
#pragma unroll
    for (int h = 0; h < 2 * CW; ++h)
        if (acc[h]) atomicOr(&c.det32[2 * c.jw + h], acc[h]);
}

// Noise bytes for sweeps t_first .. t_first + ns - 1 (a-6).  One Philox call per (sweep,
// position, group of 4 words); round keys precomputed; G is a power of two (no divisions).
template <int CW>
__device__ __forceinline__ void tile_produce(const TileCtx<CW>& c, uint32_t t_first, uint32_t ns,
                                             uint32_t w0, const uint32_t (&ks)[10][2],
                                             const FlipTable& ft)
{
    const uint32_t thr = ft.lo[1];
    // noise byte of one word: quasi-greedy 0xFF / 0x00 (k = 1 threshold); general table: bit k
    auto nbyte = [&](uint32_t u) -> uint32_t {
        if (!ft.general) return u < thr ? 0xFFu : 0u;
        uint32_t v = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k)
            v |= ((((ft.always >> k) & 1u) != 0u) || (u < ft.lo[k])) ? (1u << k) : 0u;
        return v;
    };
    const uint32_t G = c.T >= 4 ? c.T / 4 : 1;
    const uint32_t gsh = (uint32_t)__ffs((int)G) - 1u;
    const uint32_t per_sweep = c.N << gsh;
    const uint32_t grp0 = w0 >> 2;
    for (uint32_t s = 0; s < ns; ++s) {
        unsigned char* row = c.rbuf + (size_t)s * c.N * c.T;
        const uint32_t t = t_first + s;
        for (uint32_t q = threadIdx.x; q < per_sweep; q += blockDim.x) {
            const uint32_t p = q >> gsh, g = q & (G - 1u);
            const uint32_t spin = c.rec[2 * p + 1].z >> c.row_shift;
            uint32_t o[4];
            philox4x32_10_ks(spin, grp0 + g, t, TAG_SWEEP, ks, o);
            unsigned char* dst = row + (size_t)p * c.T;
            if (c.T >= 4) {
                const uint32_t v = nbyte(o[0]) | (nbyte(o[1]) << 8) | (nbyte(o[2]) << 16) |
                                   (nbyte(o[3]) << 24);
                *reinterpret_cast<uint32_t*>(dst + 4 * g) = v;
            } else {
                for (uint32_t lw = 0; lw < c.T; ++lw)
                    dst[lw] = (unsigned char)nbyte(o[(w0 + lw) & 3u]);
            }
        }
    }
}

template <int CW>
__global__ void __launch_bounds__(1024, 1) k_sweep_tile(TileArgs A)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t N = A.N, W = A.W, T = A.T;
    const uint32_t tiles = W / T;
    const uint32_t inst = blockIdx.x / tiles;
    const uint32_t w0 = (blockIdx.x % tiles) * T;
    const xs_tts_rec rec0 = A.d.rec[inst];
    if (rec0.solved && !(A.flags & XS_FLAG_NO_SKIP)) return;   // stop rule (L129, L293)

    TileCtx<CW> c;
    c.state = smem;
    uint4* rec_w = reinterpret_cast<uint4*>(smem + A.off_rec);
    c.rec = rec_w;
    c.rbuf = smem + A.off_rbuf;
    uint32_t* sets_w = reinterpret_cast<uint32_t*>(smem + A.off_sets);
    c.sets = sets_w;
    c.det32 = reinterpret_cast<uint32_t*>(smem + A.off_misc);
    c.known32 = c.det32 + 2 * T;
    c.flag = c.known32 + 2 * T;
    c.N = N; c.T = T;
    c.row_shift = 2u + (uint32_t)__ffs((int)T);      // T is a power of two: log2(8 T)
    c.n_sets = A.d.n_sets[inst];
    const uint32_t LPS = T / CW;
    c.slot = threadIdx.x / LPS;
    c.n_slots = blockDim.x / LPS;
    c.jw = (threadIdx.x % LPS) * CW;
    c.joff = c.jw * 8;

    const uint64_t seed = A.d.run_seed[inst];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint32_t ks[10][2];
    philox_key_schedule(k0, k1, ks);
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w0;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w0) * 64;
    const uint32_t row_bytes = T * 8;

    // ---- a-3: tile load -------------------------------------------------------------------
    const AdjRec* adj = A.d.adj + (size_t)inst * N;
    for (uint32_t p = threadIdx.x; p < N; p += blockDim.x) {
        const AdjRec r = adj[p];
        rec_w[2 * p] = make_uint4(r.nbr[0] * row_bytes, r.nbr[1] * row_bytes, r.nbr[2] * row_bytes,
                                  r.nbr[3] * row_bytes);
        rec_w[2 * p + 1] = make_uint4(r.nbr[4] * row_bytes, r.nbr[5] * row_bytes, r.self * row_bytes,
                                      ((r.jbits & 1u) ? 0xFFu : 0u) | ((r.jbits & 2u) ? 0xFF00u : 0u) |
                                          ((r.jbits & 4u) ? 0xFF0000u : 0u));
    }
    for (uint32_t s = threadIdx.x; s <= c.n_sets; s += blockDim.x)
        sets_w[s] = A.d.set_start[(size_t)inst * (N + 1) + s];
    auto load_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            reinterpret_cast<uint64_t*>(smem)[e] = xg[(size_t)i * W + lw];
        }
    };
    auto store_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            xg[(size_t)i * W + lw] = reinterpret_cast<const uint64_t*>(smem)[e];
        }
    };
    load_state();
    // known32: bit set <=> the clone already has a first-hit entry
    for (uint32_t e = threadIdx.x; e < ((64 * T + 31) / 32) * 32; e += blockDim.x) {
        const bool k = fhg[e] != XS_NO_HIT;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, k);
        if ((threadIdx.x & 31) == 0) c.known32[e >> 5] = m;
    }
    __syncthreads();

    // solved mask of the current tile -> det32 (bit set = NOT solved); ends with a barrier
    auto detect = [&]() {
        for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x) c.det32[e] = 0;
        if (threadIdx.x == 0) *c.flag = 0;
        __syncthreads();
        tile_detect_acc<CW>(c);
        __syncthreads();
    };
    // sweeps t0+1 .. t0+n; exact: record first hits after every sweep
    auto run_range = [&](uint32_t t0, uint32_t n, bool exact) {
        for (uint32_t s0 = 0; s0 < n; s0 += A.rb) {
            const uint32_t ns = min(A.rb, n - s0);
            tile_produce<CW>(c, t0 + s0 + 1, ns, w0, ks, A.ft);
            __syncthreads();
            for (uint32_t s = 0; s < ns; ++s) {
                if (A.ft.general) tile_sweep<CW, true>(c, s); else tile_sweep<CW, false>(c, s);
                if (exact) {
                    detect();
                    const uint32_t t = t0 + s0 + s + 1;
                    for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x) {
                        uint32_t newly = ~c.det32[e] & ~c.known32[e];
                        c.known32[e] |= newly;
                        while (newly) {
                            const int bit = __ffs(newly) - 1;
                            newly &= newly - 1;
                            fhg[32 * e + bit] = t;
                        }
                    }
                    __syncthreads();
                }
            }
        }
    };

    uint32_t t = (uint32_t)rec0.sweeps_done;
    uint32_t remaining = A.n_sweeps;
    while (remaining) {
        const uint32_t nb = min(A.batch, remaining);
        if (A.ft.lo[0] != 0u || (A.ft.always & 1u)) {
            // w0 > 0: a ground state can be left again (L69), so the batch-end check could miss
            // a visit -> check after every sweep
            run_range(t, nb, true);
        } else {
            run_range(t, nb, false);
            detect();
            for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x)
                if (~c.det32[e] & ~c.known32[e]) *c.flag = 1;
            __syncthreads();
            const bool replay = *c.flag != 0;
            __syncthreads();
            if (replay) {
                load_state();          // global copy = state at the start of this batch
                __syncthreads();
                run_range(t, nb, true);
            }
        }
        store_state();             // a-10 (also the replay checkpoint of the next batch)
        t += nb;
        remaining -= nb;
    }
}

// ------------------------------------------------------------------------------------------
// a-4 .. a-9: streaming regime (tile does not fit on chip, e.g. N = 2^20).
// One launch per independent set; a lane owns CW words of one spin row and gathers the six
// partner rows from global memory (HBM / L2).  Spins of a set are mutually non-adjacent
// (L277), so the in-place update is race free inside a launch; launch order gives the set
// order.  k != 0 words are OR-reduced per sweep into det[inst][w] (registers -> shared ->
// one global atomic per CTA and word), and k_stream_commit turns clear bits into first hits.
// ------------------------------------------------------------------------------------------
constexpr uint32_t ST_THREADS = 256;

// Programmatic dependent launch: the streaming regime is a chain of short dependent launches
// (one per independent set).  Launched with programmatic stream serialization, a kernel may
// start while its predecessor drains; it must wait here before touching anything the
// predecessor wrote, and lets its own successor start launching right away.
__device__ __forceinline__ void pdl_wait_and_release()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// PC: per-clone noise instead of one number per word.
template <int CW, bool PC>
__global__ void __launch_bounds__(ST_THREADS) k_stream_set(DevPtrs d, uint32_t N, uint32_t W,
                                                          uint32_t set_idx, uint32_t s_rel,
                                                          FlipTable ft, uint32_t flags, uint64_t* det)
{
    __shared__ uint32_t sdet[1024];
    pdl_wait_and_release();
    const uint32_t thr = ft.lo[1];
    const uint32_t inst = blockIdx.y;
    const xs_tts_rec rec = d.rec[inst];
    if (rec.solved && !(flags & XS_FLAG_NO_SKIP)) return;
    if (set_idx >= d.n_sets[inst]) return;
    const uint32_t* ss = d.set_start + (size_t)inst * (N + 1);
    const uint32_t p0 = ss[set_idx], p1 = ss[set_idx + 1];
    const uint32_t nchunk = W / CW;
    const uint64_t total = (uint64_t)(p1 - p0) * nchunk;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const bool fixed = (stride % nchunk == 0) && (2 * W <= 1024);
    const uint32_t t = (uint32_t)rec.sweeps_done + s_rel;
    const uint64_t seed = d.run_seed[inst];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint64_t* x = d.x + (size_t)inst * N * W;
    uint32_t* det32 = reinterpret_cast<uint32_t*>(det + (size_t)inst * W);
    const AdjRec* adj = d.adj + (size_t)inst * N;

    if (fixed) {
        for (uint32_t e = threadIdx.x; e < 2 * W; e += blockDim.x) sdet[e] = 0;
        __syncthreads();
    }
    uint32_t acc[2 * CW];
#pragma unroll
    for (int h = 0; h < 2 * CW; ++h) acc[h] = 0;
    uint32_t my_w = 0;
    for (uint64_t task = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; task < total; task += stride) {
        const uint32_t q = (uint32_t)(task / nchunk);
        const uint32_t ch = (uint32_t)(task - (uint64_t)q * nchunk);
        const uint32_t w = ch * CW;
        my_w = w;
        const uint4* rp = reinterpret_cast<const uint4*>(adj + p0 + q);
        const uint4 r0 = __ldg(rp), r1 = __ldg(rp + 1);
        uint32_t a[3][2 * CW], b[3][2 * CW], xo[2 * CW];
        vload<CW>(x + (size_t)r0.x * W + w, a[0]);
        vload<CW>(x + (size_t)r0.y * W + w, b[0]);
        vload<CW>(x + (size_t)r0.z * W + w, a[1]);
        vload<CW>(x + (size_t)r0.w * W + w, b[1]);
        vload<CW>(x + (size_t)r1.x * W + w, a[2]);
        vload<CW>(x + (size_t)r1.y * W + w, b[2]);
        uint64_t* own = x + (size_t)r1.z * W + w;
        vload<CW>(own, xo);
        const uint32_t jm0 = (r1.w & 1u) ? ~0u : 0u, jm1 = (r1.w & 2u) ? ~0u : 0u,
                       jm2 = (r1.w & 4u) ? ~0u : 0u;
        uint32_t o[4];
        if (!PC) philox4x32_10(r1.z, w >> 2, t, TAG_SWEEP, k0, k1, o);
        uint32_t xn[2 * CW];
        uint32_t Rc[2 * CW];       // PC: k = 1 flip masks of the lane's half words
        if (PC) {
#pragma unroll
            for (int c = 0; c < CW; ++c) {
                uint32_t rl[8], rh[8];   // low / high halves of r_0 .. r_7 of word w + c
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    uint32_t q4[4];
                    philox4x32_10(r1.z, 4u * (w + c) + jj, t, TAG_CLONE, k0, k1, q4);
                    rl[2 * jj] = q4[0]; rh[2 * jj] = q4[1];
                    rl[2 * jj + 1] = q4[2]; rh[2 * jj + 1] = q4[3];
                }
                const uint32_t lo7[7] = {rl[0], rl[1], rl[2], rl[3], rl[4], rl[5], rl[6]};
                const uint32_t hi7[7] = {rh[0], rh[1], rh[2], rh[3], rh[4], rh[5], rh[6]};
                Rc[2 * c] = clone_noise_mask(lo7, ft.clone_m);
                Rc[2 * c + 1] = clone_noise_mask(hi7, ft.clone_m);
            }
        }
#pragma unroll
        for (int h = 0; h < 2 * CW; ++h) {
            const uint32_t u = PC ? 0u : (((w + (h >> 1)) & 3u) == 0u) ? o[0] : (((w + (h >> 1)) & 3u) == 1u) ? o[1]
                               : (((w + (h >> 1)) & 3u) == 2u) ? o[2] : o[3];
            const uint32_t nz = qg_nonzero_k(a[0][h], b[0][h], jm0, a[1][h], b[1][h], jm1, a[2][h],
                                             b[2][h], jm2, xo[h]);
            if (PC) {
                xn[h] = qg_update(a[0][h], b[0][h], jm0, a[1][h], b[1][h], jm1, a[2][h], b[2][h], jm2,
                                  xo[h], Rc[h]);
            } else if (ft.general) {
                uint32_t Rk[4];
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    Rk[k] = ((((ft.always >> k) & 1u) != 0u) || (u < ft.lo[k])) ? ~0u : 0u;
                xn[h] = table_update(a[0][h], b[0][h], jm0, a[1][h], b[1][h], jm1, a[2][h], b[2][h],
                                     jm2, xo[h], Rk[0], Rk[1], Rk[2], Rk[3]);
            } else {
                xn[h] = qg_update(a[0][h], b[0][h], jm0, a[1][h], b[1][h], jm1, a[2][h], b[2][h], jm2,
                                  xo[h], u < thr ? ~0u : 0u);
            }
            if (fixed) acc[h] |= nz;
            else if (nz) atomicOr(&det32[2 * w + h], nz);
        }
        vstore<CW>(own, xn);
    }
    if (fixed) {
#pragma unroll
        for (int h = 0; h < 2 * CW; ++h)
            if (acc[h]) atomicOr(&sdet[2 * my_w + h], acc[h]);
        __syncthreads();
        for (uint32_t e = threadIdx.x; e < 2 * W; e += blockDim.x)
            if (sdet[e]) atomicOr(&det32[e], sdet[e]);
    }
}

// After the last set of relative sweep s_rel: a clear bit in det_cur means every spin of the
// clone saw k = 0 during the sweep, i.e. the clone was in a ground state when the sweep
// started -> first hit = t - 1.  Also clears det_next for the following sweep.
__global__ void k_stream_commit(DevPtrs d, uint32_t W, uint32_t I, const uint64_t* det_cur,
                                uint64_t* det_next, uint32_t s_rel, uint32_t flags)
{
    pdl_wait_and_release();
    const uint64_t total = (uint64_t)I * W * 64;
    for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t inst = (uint32_t)(e / ((uint64_t)W * 64));
        const xs_tts_rec rec = d.rec[inst];
        if (!(rec.solved && !(flags & XS_FLAG_NO_SKIP))) {
            const bool solved = ((det_cur[e >> 6] >> (e & 63)) & 1ull) == 0;
            if (solved && d.first_hit[e] == XS_NO_HIT)
                d.first_hit[e] = (uint32_t)rec.sweeps_done + s_rel - 1u;
        }
        if (e < (uint64_t)I * W) det_next[e] = 0;
    }
}

// first-hit marking at the end of a streaming call for instances that were swept
__global__ void k_mark_swept(DevPtrs d, uint32_t W, uint32_t I, const uint64_t* det,
                             uint32_t n_sweeps, uint32_t flags)
{
    const uint64_t total = (uint64_t)I * W * 64;
    for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t inst = (uint32_t)(e / ((uint64_t)W * 64));
        const xs_tts_rec rec = d.rec[inst];
        if (rec.solved && !(flags & XS_FLAG_NO_SKIP)) continue;
        const bool solved = ((det[e >> 6] >> (e & 63)) & 1ull) == 0;
        if (solved && d.first_hit[e] == XS_NO_HIT)
            d.first_hit[e] = (uint32_t)rec.sweeps_done + n_sweeps;
    }
}

// ------------------------------------------------------------------------------------------
// host side: geometry and launchers
// ------------------------------------------------------------------------------------------
namespace {
constexpr uint32_t SMEM_MAX = 227u * 1024u;   // per-CTA opt-in limit on sm_100a

inline uint32_t round_up(uint32_t v, uint32_t m) { return (v + m - 1) / m * m; }

struct TileSmem { uint32_t off_rec, off_rbuf, off_sets, off_misc, total; };
TileSmem tile_smem(uint32_t N, uint32_t T, uint32_t rb, uint32_t n_sets_max)
{
    TileSmem s;
    uint64_t o = ((uint64_t)N * T * 8 + 15) / 16 * 16;   // records are read as 16-byte vectors
    s.off_rec = (uint32_t)o;           o += (uint64_t)N * 32;
    s.off_rbuf = (uint32_t)o;          o += round_up(rb * N * T, 16);
    s.off_sets = (uint32_t)o;          o += round_up((n_sets_max + 1) * 4, 16);
    s.off_misc = (uint32_t)o;          o += round_up((4 * T + 4) * 4, 16);
    s.total = o > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)o;
    return s;
}
}  // namespace

bool choose_geometry(const xs_batch& b, TileGeom& g, std::string& err)
{
    const xs_params& p = b.p;
    g = TileGeom{};
    const xs_geometry& rq = b.req;                  // explicit requests (xs_set_geometry), 0 = rule
    const uint32_t NUM_SMS = std::max(1u, b.num_sms);
    g.batch = rq.batch_sweeps ? rq.batch_sweeps : 64u;
    const uint32_t force_T = rq.tile_words;
    uint32_t bestT = 0;
    // Measured on B200: with at least one 16-column tile per SM
    // the generic kernel with T = 16 (128-byte rows: conflict-free, several CTAs per SM overlap
    // their load / compute / barrier phases) is the fastest choice; with fewer tiles than SMs
    // (config 2) the static-task kernel with T = 8 wins because one CTA per SM must hide its
    // own latencies.  xs_geometry.variant: AUTO / 2 = this rule, 0 = generic only, 1 = static if feasible.
    const uint32_t want_variant = (rq.variant == XS_GEOM_AUTO || rq.variant > 1u) ? 2u : rq.variant;
    const bool many_tiles = (p.n_words % 16 == 0) &&
                            (uint64_t)p.n_instances * (p.n_words / 16) >= NUM_SMS &&
                            tile_smem(p.n_spins, 16, 1, b.n_sets_max).total <= SMEM_MAX;
    uint32_t auto_T = 0;
    if (want_variant == 2 && many_tiles && !force_T) auto_T = 16;
    // Measured: when the update order has few, evenly filled sets
    // (XS_FLAG_BALANCED: 4 sets of N/4), the static-task kernel on T = 8 tiles with one task per
    // thread and round (threads = 4 x set size, registers capped so that 16 warps share an SM)
    // beats the generic kernel also when there are many tiles: 4 barriers per sweep, 8 instead of
    // 11 shared-memory accesses per task.
    // Larger N (sets of more than 128 spins): T = 4 tiles (two lanes per spin, four row copies).
    if (want_variant == 2 && !force_T && !(p.flags & XS_FLAG_STREAMING) && !b.ft.general &&
        p.n_words % 8 == 0 && (uint64_t)p.n_instances * (p.n_words / 8) >= NUM_SMS) {
        const uint32_t max_rounds = (p.flags & XS_FLAG_BALANCED) ? 6u : 4u;
        for (uint32_t lim : {4u, max_rounds}) {
            for (uint32_t T : {8u, 4u}) {
                for (uint32_t thr : {128u, 256u, 512u}) {
                    if (!static_feasible(b, T, 2, thr) || static_rounds(b, T, 2, thr) > lim) continue;
                    g.regime = 0;
                    g.variant = 1;
                    g.T = T;
                    g.CW = 2;
                    g.threads = thr;
                    g.ctas = p.n_instances * (p.n_words / T);
                    g.smem = static_smem_bytes(p.n_spins, T);
                    g.rb = 0;
                    return true;
                }
            }
        }
    }
    // 1) static-task kernel (xs_sweep_static.cu): work list in registers, T in {8,16,32,64}
    // many small tiles (e.g. 20,000 runs of W = 4): the generic kernel's high occupancy wins
    const bool few_tiles = (uint64_t)p.n_instances * ((p.n_words + 7) / 8) < 2ull * NUM_SMS;
    if (!(p.flags & XS_FLAG_STREAMING) && !b.ft.general &&     // static kernel: quasi-greedy table only
        (want_variant == 1 || (want_variant == 2 && !auto_T && few_tiles))) {
        const uint32_t force_thr = rq.threads;
        const uint32_t force_cw = rq.words_per_lane;
        uint32_t sT = 0, sThr = 0, sCW = 0;
        uint64_t s_cost = ~0ull;
        for (uint32_t T = 64; T >= 4; T >>= 1) {
            if (force_T && T != force_T) continue;
            for (uint32_t cw = 2; cw >= 1; --cw) {
                if (force_cw && cw != force_cw) continue;
                for (uint32_t thr = 128; thr <= 512; thr *= 2) {
                    if (force_thr && thr != force_thr) continue;
                    if (!static_feasible(b, T, cw, thr)) continue;
                    const uint32_t smem = static_smem_bytes(p.n_spins, T);
                    const uint64_t ctas = (uint64_t)p.n_instances * (p.n_words / T);
                    if (smem > SMEM_MAX) continue;
                    // work of the busiest SM ~ (CTAs it gets) x T columns; then fewer rounds
                    // (= fewer barriers per sweep); 512-thread CTAs are register-capped at 128
                    const uint64_t per_sm = (ctas + NUM_SMS - 1) / NUM_SMS;
                    const uint64_t cost = per_sm * T * 16 + static_rounds(b, T, cw, thr) +
                                          (thr == 512 ? 2 : 0) + (cw == 1 ? 1 : 0);
                    if (cost < s_cost) { s_cost = cost; sT = T; sThr = thr; sCW = cw; }
                }
            }
        }
        if (sT) {
            g.regime = 0;
            g.variant = 1;
            g.T = sT;
            g.CW = sCW;
            g.threads = sThr;
            g.ctas = p.n_instances * (p.n_words / sT);
            g.smem = static_smem_bytes(p.n_spins, sT);
            g.rb = 0;
            return true;
        }
    }
    // 2) generic tile kernel
    if (!(p.flags & XS_FLAG_STREAMING) && (uint64_t)p.n_spins * 8 < SMEM_MAX) {
        // Widest tile (up to a 128-byte row) that still gives every SM two CTAs, else one CTA,
        // else the narrowest tile (most CTAs).  Wider tiles share records and Philox calls
        // between more clone words; narrow rows cost bank conflicts.
        auto ok = [&](uint32_t T) {
            if (p.n_words % T) return false;
            if (force_T && T != force_T) return false;
            if (auto_T && T != auto_T) return false;
            return tile_smem(p.n_spins, T, 1, b.n_sets_max).total <= SMEM_MAX;
        };
        auto n_ctas = [&](uint32_t T) { return (uint64_t)p.n_instances * (p.n_words / T); };
        for (uint64_t want : {2ull * NUM_SMS, 1ull * NUM_SMS}) {
            for (uint32_t T = 16; T >= 1 && !bestT; T >>= 1)
                if (ok(T) && n_ctas(T) >= want) bestT = T;
            if (bestT) break;
        }
        for (uint32_t T = 1; T <= 64 && !bestT; T <<= 1)
            if (ok(T)) bestT = T;
    }
    if (bestT == 0) {
        g.regime = 1;
        g.T = p.n_words;
        g.CW = (p.n_words % 2 == 0) ? 2 : 1;
        g.threads = ST_THREADS;
        const uint64_t tasks = (uint64_t)b.max_set_size * (p.n_words / g.CW);
        g.ctas = (uint32_t)std::min<uint64_t>((tasks + ST_THREADS - 1) / ST_THREADS, NUM_SMS * 8);
        g.ctas = std::max(g.ctas, 1u);
        g.smem = 0;
        g.batch = 1;
        g.rb = 0;
        (void)err;
        return true;
    }
    g.regime = 0;
    g.T = bestT;
    g.CW = bestT >= 2 ? 2 : 1;
    const uint32_t LPS = g.T / g.CW;
    const uint32_t want = round_up(std::max(b.max_set_size, 1u) * LPS, 32);
    g.threads = std::min(1024u, std::max(128u, want));
    if (rq.threads) g.threads = std::min(1024u, std::max(32u, rq.threads / 32 * 32));
    g.ctas = p.n_instances * (p.n_words / g.T);
    uint32_t rb = std::max(1u, std::min(g.batch, rq.noise_sweeps ? rq.noise_sweeps : 8u));
    while (rb > 1 && tile_smem(p.n_spins, g.T, rb, b.n_sets_max).total > SMEM_MAX) --rb;
    // Two CTAs per SM overlap each other's load / compute / barrier phases (measured +19 % on
    // config 3, profiles/r01_ncu_summary.md): shrink the noise ring and the CTA until two fit
    // (228 KB shared memory and 64 K registers per SM; this kernel uses 56 registers).
    if (!rq.noise_sweeps && g.ctas >= 2 * NUM_SMS) {
        const uint32_t sm_smem = 228u * 1024u, reserved = 1024u;
        uint32_t r2 = rb;
        while (r2 > 1 && 2 * (tile_smem(p.n_spins, g.T, r2, b.n_sets_max).total + reserved) > sm_smem) r2 /= 2;
        if (2 * (tile_smem(p.n_spins, g.T, r2, b.n_sets_max).total + reserved) <= sm_smem) {
            rb = r2;
            if (!rq.threads) g.threads = std::min(g.threads, 512u);
        }
    }
    g.rb = rb;
    g.smem = tile_smem(p.n_spins, g.T, rb, b.n_sets_max).total;
    return true;
}

#define XS_CU(call)                                         \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return (int)e_;              \
    } while (0)

void count_launch(uint64_t n);   // xs_diag.cu

static inline uint32_t grid_for(uint64_t total, uint32_t threads)
{
    return (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>((total + threads - 1) / threads, 148u * 16u));
}

int launch_init(const xs_batch& b, void* stream)
{
    const xs_params& p = b.p;
    const uint64_t total = (uint64_t)p.n_instances * p.n_spins * p.n_words;
    k_init<<<grid_for(total, 256), 256, 0, (cudaStream_t)stream>>>(b.d, p.n_spins, p.n_words, p.n_instances);
    count_launch(1);
    return (int)cudaGetLastError();
}

// det slot 0 <- unsat OR of the current global state
static int launch_unsat_or(const xs_batch& b, cudaStream_t st)
{
    const xs_params& p = b.p;
    XS_CU(cudaMemsetAsync(b.d.det, 0, (size_t)p.n_instances * p.n_words * 8, st));
    const uint32_t thr = std::min(256u, round_up(p.n_words, 32));
    const uint32_t wblocks = std::min(64u, (p.n_words + thr - 1) / thr);
    // clauses per CTA: 64, fewer when that leaves SMs without a CTA (small single instances)
    const uint64_t ctas64 = (uint64_t)((p.n_spins + 63) / 64) * p.n_instances * wblocks;
    uint32_t chunk = 64;
    while (chunk > 4 && ctas64 * (64 / chunk) < 2ull * b.num_sms) chunk /= 2;
    dim3 grid((p.n_spins + chunk - 1) / chunk, p.n_instances, wblocks);
    k_unsat_or<<<grid, thr, 0, st>>>(b.d, p.n_spins, p.n_words, chunk, b.d.det);
    count_launch(1);
    return (int)cudaGetLastError();
}

int launch_mark(const xs_batch& b, bool reset_first_hit, void* stream)
{
    const xs_params& p = b.p;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = launch_unsat_or(b, st);
    if (rc) return rc;
    const uint64_t total = (uint64_t)p.n_instances * p.n_words * 64;
    k_mark<<<grid_for(total, 256), 256, 0, st>>>(b.d, p.n_words, p.n_instances, b.d.det,
                                                 reset_first_hit ? 1 : 0, 0u);
    count_launch(1);
    return (int)cudaGetLastError();
}

int launch_finalize(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    k_finalize<<<b.p.n_instances, FIN_THREADS, 0, (cudaStream_t)stream>>>(b.d, b.p.n_words, n_sweeps, b.p.flags);
    count_launch(1);
    return (int)cudaGetLastError();
}

int launch_energy(const xs_batch& b, int32_t* dev_out, void* stream)
{
    const xs_params& p = b.p;
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t total = (uint64_t)p.n_instances * p.n_words * 64;
    k_energy_fill<<<grid_for(total, 256), 256, 0, st>>>(dev_out, total, -(int32_t)p.n_spins);
    count_launch(1);
    // lanes <-> words: LW = smallest power of two >= W, at most 32
    uint32_t lw_shift = 0;
    while (lw_shift < 5 && (1u << lw_shift) < p.n_words) ++lw_shift;
    const uint32_t LW = 1u << lw_shift, groups = EN_THREADS >> lw_shift;
    const uint32_t wblocks = (p.n_words + LW - 1) / LW;
    // clauses per thread: as many as the count planes hold, fewer when that leaves SMs without a CTA
    const uint64_t want_chunks = std::max<uint64_t>(1, (4ull * b.num_sms) / ((uint64_t)wblocks * p.n_instances));
    uint64_t cpt = ((uint64_t)p.n_spins + groups * want_chunks - 1) / (groups * want_chunks);
    cpt = std::min<uint64_t>(EN_MAX_CPT, std::max<uint64_t>(4, (cpt + 3) / 4 * 4));
    const uint32_t chunks = (uint32_t)(((uint64_t)p.n_spins + groups * cpt - 1) / (groups * cpt));
    dim3 grid(wblocks * chunks, p.n_instances);
    k_energy_acc<<<grid, EN_THREADS, 0, st>>>(b.d, p.n_spins, p.n_words, lw_shift, wblocks, (uint32_t)cpt, dev_out);
    count_launch(1);
    return (int)cudaGetLastError();
}

int launch_sweeps(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    const xs_params& p = b.p;
    const TileGeom& g = b.geom;
    cudaStream_t st = (cudaStream_t)stream;
    if (n_sweeps == 0) return 0;
    if (g.regime == 0 && g.variant == 3) return launch_sweep_warp(b, n_sweeps, stream);
    if (g.regime == 0 && g.variant == 2) return launch_sweep_clause(b, n_sweeps, stream);
    if (g.regime == 0 && g.variant == 1) return launch_sweep_static(b, n_sweeps, stream);
    if (g.regime == 0) {
        const TileSmem s = tile_smem(p.n_spins, g.T, g.rb, b.n_sets_max);
        TileArgs A;
        A.d = b.d;
        A.N = p.n_spins; A.W = p.n_words; A.T = g.T; A.n_sweeps = n_sweeps;
        A.thr = p.w1_threshold; A.flags = p.flags; A.batch = g.batch; A.rb = g.rb;
        A.ft = b.ft;
        A.off_rec = s.off_rec; A.off_rbuf = s.off_rbuf; A.off_sets = s.off_sets; A.off_misc = s.off_misc;
        if (g.CW == 2) {
            XS_CU(cudaFuncSetAttribute(k_sweep_tile<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.total));
            k_sweep_tile<2><<<g.ctas, g.threads, s.total, st>>>(A);
            count_launch(1);
        } else {
            XS_CU(cudaFuncSetAttribute(k_sweep_tile<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.total));
            k_sweep_tile<1><<<g.ctas, g.threads, s.total, st>>>(A);
            count_launch(1);
        }
        return (int)cudaGetLastError();
    }
    // streaming regime
    const size_t det_words = (size_t)p.n_instances * p.n_words;
    uint64_t* det[2] = {b.d.det, b.d.det + det_words};
    XS_CU(cudaMemsetAsync(b.d.det, 0, 2 * det_words * 8, st));
    dim3 grid(g.ctas, p.n_instances);
    const uint64_t clones = det_words * 64;
    cudaLaunchAttribute pdl_attr[1];
    pdl_attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    pdl_attr[0].val.programmaticStreamSerializationAllowed = 1;
    for (uint32_t s = 1; s <= n_sweeps; ++s) {
        uint64_t* cur = det[s & 1];
        for (uint32_t set = 0; set < b.n_sets_max; ++set) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = grid;
            cfg.blockDim = dim3(ST_THREADS);
            cfg.stream = st;
            cfg.attrs = pdl_attr;
            cfg.numAttrs = 1;
            auto kern = b.ft.per_clone ? (g.CW == 2 ? k_stream_set<2, true> : k_stream_set<1, true>)
                                       : (g.CW == 2 ? k_stream_set<2, false> : k_stream_set<1, false>);
            XS_CU(cudaLaunchKernelEx(&cfg, kern, b.d, p.n_spins, p.n_words, set, s, b.ft, p.flags, cur));
            count_launch(1);
        }
        if (b.ft.lo[0] != 0u || (b.ft.always & 1u)) {
            // w0 > 0: ground states are not absorbing (L69): look at the state after every sweep
            int rc = launch_unsat_or(b, st);
            if (rc) return rc;
            k_mark_swept<<<grid_for(clones, 256), 256, 0, st>>>(b.d, p.n_words, p.n_instances, b.d.det,
                                                               s, p.flags);
            count_launch(1);
            XS_CU(cudaMemsetAsync(b.d.det, 0, 2 * det_words * 8, st));
        } else {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(grid_for(clones, 256));
            cfg.blockDim = dim3(256);
            cfg.stream = st;
            cfg.attrs = pdl_attr;
            cfg.numAttrs = 1;
            XS_CU(cudaLaunchKernelEx(&cfg, k_stream_commit, b.d, p.n_words, p.n_instances,
                                     (const uint64_t*)cur, det[(s + 1) & 1], s, p.flags));
            count_launch(1);
        }
        XS_CU(cudaGetLastError());
    }
    int rc = launch_unsat_or(b, st);
    if (rc) return rc;
    k_mark_swept<<<grid_for(clones, 256), 256, 0, st>>>(b.d, p.n_words, p.n_instances, b.d.det,
                                                       n_sweeps, p.flags);
    count_launch(1);
    return (int)cudaGetLastError();
}

}  // namespace xs
