// xs_sweep_clause.cuh -- the clause-word sweep kernel (template).  Included by the instantiation
// units xs_sweep_clause_r<R>.cu (one per number of rounds, so that they compile in parallel) and by
// the host side xs_sweep_clause.cu.
//
// Shared memory holds the CLAUSE words instead of the spin words:
//
//     c_t = x_i ^ x_j ^ x_k ^ Jmask_t      (bit = 1 <=> interaction t unsatisfied)
//
// A spin's update needs only its three clause words: k = number of set bits among (c_1, c_2, c_3)
// (L67), M = maj (k >= 2), P = parity (k odd), flip = M | (P & R) (k >= 2 always, k = 1 with the
// word's noise mask R, k = 0 never: L65, L101), and flipping the spin toggles its three clauses:
// c_r ^= flip, x ^= flip: 7 three-input logic operations per 32 clones.  The spin words live only
// in the registers of the thread that owns the spin (and in global memory at batch boundaries).
// Per task (128 clones of one spin): 3 LDS.128 + 3 STS.128.  Spins of one independent set share no
// clause (L277), so the read-modify-write of the clause rows is race free between barriers.
//
// Work list: a CTA of 4 n_slots threads owns (instance, 8 word columns); "round" r of a sweep puts
// one spin on every slot (4 lanes x 16 bytes = the 64-byte clause row).  A set of at most n_slots
// spins is one round, a larger set several rounds with no barrier between them; slots without a
// spin in a round work on a scratch row (MODE 0) -- the list (3 row addresses, spin index, the
// spin's words) stays in registers for the whole call.
//
// Bank conflicts: a clause row is half of a 128-byte line and the 8 lanes of one shared-memory
// phase serve two slots.  The host places every clause in the lower or upper half of its own line
// and pairs the spins of every round so that the two slots of a phase touch opposite halves in
// each of their three accesses (clause_placement): single copy, conflict free.
//
// Noise (a-6): one Philox4x32-10 call yields the numbers of 4 consecutive words of a spin for one
// sweep.  The two lanes that share a word group each compute the call of one sweep of a two-sweep
// period and exchange the threshold bytes by shuffles (one register per round; even and odd
// rounds renew it in alternate sweeps, so every round carries half a call).  The 10 round keys are CTA-uniform: the
// run seed comes from the kernel parameters (constant bank), so the key schedule lives in uniform
// registers and costs no vector ALU work.  The comparison u < thr runs on the FMA pipe: the carry
// of u + (2^32 - thr) is the high word of a 64-bit multiply-add, and the four carries are packed
// into threshold bytes by integer multiply-adds; the ALU pipe, which bounds this kernel together
// with shared memory, only sees the 20 three-input XORs of a call.  (cthr[0] = 2^32 - thr mod 2^32,
// cthr[1] = 1 iff thr = 0, where "u >= thr" always holds: the carry is forced.)
//
// Ground-state detection / exact first hit: detection pass (OR of all clause words) every `batch`
// sweeps; if a clone not yet in the table is solved, the batch is replayed from the global copy
// with a pass after every sweep (L293; counter-based noise makes the replay bit-identical).
#pragma once
#include <type_traits>

#include <cuda_runtime.h>

#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

constexpr int CL_H = 4;             // uint32 halves per lane (2 uint64 words)
constexpr uint32_t CL_T = 8;        // tile width in uint64 columns
constexpr uint32_t CL_LPS = 4;      // lanes per slot
constexpr uint32_t CL_MAXI = 256;   // instances per launch (their run seeds travel in the parameters)
constexpr uint32_t CL_IDLE = 0xFFFFFFFFu;   // CRec.spin of a slot without a spin in that round

struct ClauseArgs {
    DevPtrs d;
    uint32_t N, W, n_sweeps, flags, batch;
    uint32_t n_slots;        // slots per CTA = threads / 4
    uint32_t ent;            // task-table entries per instance (crec_entries)
    uint32_t inst0;          // first instance of this launch
    uint32_t off_misc;       // byte offset of det32 / known32 / flag in dynamic shared memory
    uint32_t thr;            // noise threshold: a k = 1 spin flips iff u < thr
    uint32_t thr0;           // W0 kernels: a k = 0 spin flips iff u < thr0 (thr0 <= thr)
    uint32_t clone_m;        // PCN kernels: a k = 1 spin flips iff its clone's 7-bit number U < clone_m
    uint32_t one;            // the multiplier 1, as data, so that the compare stays a multiply-add
    uint32_t zero;           // the multiplier 0, as data: ties the last store of a round to its Philox call
    uint64_t seed[CL_MAXI];  // run seeds of instances inst0 .. (constant bank -> uniform registers)
};

__device__ __forceinline__ void cl_lds4(uint32_t addr, uint32_t (&o)[4])
{
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void cl_sts4(uint32_t addr, const uint32_t (&o)[4])
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "r"(addr), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
}
__device__ __forceinline__ uint32_t cl_prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
__device__ __forceinline__ uint64_t cl_mad_wide(uint32_t a, uint32_t b, uint64_t c)
{
    uint64_t d;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(d) : "r"(a), "r"(b), "l"(c));
    return d;
}
__device__ __forceinline__ uint32_t cl_mad_lo(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
constexpr int LUT_OR_ANDN = 0xF4;   // a | (b & ~c)

// R: rounds per sweep (unrolled; the task list of R rounds lives in registers).
// MODE 0: general -- slots may be idle in a round (scratch rows; warps without any spin skip the
//         round) and the barriers follow the per-instance mask cbar (bit r: barrier after round r);
// MODE 1: every slot has a spin in every round, barrier after every round (R sets of n_slots);
// MODE 2: every slot busy, barrier after every second round (R / 2 sets of 2 n_slots spins).
// W0: flip table (w0, w1, 1, 1) with 0 < w0 <= w1 (the Metropolis table w0 = w1^3;
//     SURVEY.md 8(f) NEXT-1), MODE 1 only.  A k = 0 spin flips iff the word's number u < thr0, so a second
//     threshold bit per word is kept (flip = M | (P & u<thr) | u<thr0), and a ground state can be
//     left again: the first hit is looked for after EVERY sweep, without extra loads, by OR-ing
//     every clause word at its LAST touch of the sweep (a static 3-bit mask per task, from the host).
// PCN: per-clone noise (XS_FLAG_CLONE_NOISE; DESIGN.md R-clone), MODE 1 only: every
//     clone draws its own 7-bit number U from four Philox calls per (spin, word, sweep); a k = 1 spin
//     flips iff U < clone_m.  Each lane computes the masks of its two words in the round itself (16 times
//     the Philox work of the shared-number rule: this form is ALU bound).
template <int R, int MAXTHREADS, int MINB, int MODE, bool W0 = false, bool PCN = false>
__global__ void __launch_bounds__(MAXTHREADS, MINB) k_sweep_clause(const __grid_constant__ ClauseArgs A)
{
    // One CTA per SM with few warps (fewer tiles than SMs, e.g. BASELINE.json configs[1]): the
    // kernel is bound by the dependent chain of a round, not by a pipe.  Measured (DESIGN.md
    // section 7): the multiply-add compare and the store-address tie of the noise cost 3 % there
    // and gain 10 % on the dense shapes, so the two launch classes take different forms.
    constexpr bool SPARSE = (MINB == 1 && MAXTHREADS <= 256);
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t N = A.N, W = A.W;
    const uint32_t tiles = W / CL_T;
    const uint32_t il = blockIdx.x / tiles;                 // instance inside this launch
    const uint32_t inst = A.inst0 + il;
    const uint32_t w0 = (blockIdx.x % tiles) * CL_T;
    const xs_tts_rec rec0 = A.d.rec[inst];
    if (rec0.solved && !(A.flags & XS_FLAG_NO_SKIP)) return;   // stop rule (L129, L293)

    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    uint32_t* det32 = reinterpret_cast<uint32_t*>(smem + A.off_misc);
    uint32_t* known32 = det32 + 4 * CL_T;         // det32: two buffers of 2 T words (W0: by sweep parity)
    uint32_t* flag = known32 + 2 * CL_T;

    const uint32_t n_slots = A.n_slots;
    const uint32_t slot = threadIdx.x / CL_LPS;
    const uint32_t j = threadIdx.x % CL_LPS;
    const uint32_t lane_off = base + j * 16u;

    // CTA-uniform key from the constant bank: the 10 round keys of Philox stay in uniform registers
    const uint64_t seed = A.seed[il];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w0;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w0) * 64;

    // ---- static task list: this thread's spin of round r = entry r * n_slots + slot -----------
    uint32_t ca[R][3];        // shared addresses of the spin's three clause rows
    uint32_t x[R][CL_H];      // the spin's words: registers only
    // threshold bytes of the current two-sweep noise period.  Only bit 7 of each byte is looked at
    // (sign-replicating PRMT); with 7 or 8 rounds the spin index rides in bits 0-6 of bytes 0 and 1
    // (N < 2^14): one register per round less, which keeps the 8-round list of N = 1024 free of
    // spills under the 128-register cap.  (Measured: the unpacking costs 6 % with 4 rounds, where
    // there is room, and gains 3 % with 8.)
    constexpr bool PACK = (R >= 7);
    uint32_t rm[R] = {};
    uint32_t spin[PACK ? 1 : R] = {};
    auto spin_of = [&](int r) -> uint32_t {
        return PACK ? ((rm[r] & 0x7Fu) | ((rm[r] >> 1) & 0x3F80u)) : spin[PACK ? 0 : r];
    };
    uint32_t rm0[W0 ? R : 1];         // W0: the same bytes for the k = 0 threshold
    uint32_t last = 0;                // W0: bit 3 r + k <=> round r is the last touch of its clause k in a sweep
    uint32_t act = 0, wact = 0, bar = 0;
    {
        const uint4* cr = reinterpret_cast<const uint4*>(A.d.crec + (size_t)inst * A.ent);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const uint4 v = cr[r * n_slots + slot];
            ca[r][0] = lane_off + v.x;
            ca[r][1] = lane_off + v.y;
            ca[r][2] = lane_off + v.z;
            if (PACK) {
                rm[r] = (v.w & 0x7Fu) | ((v.w & 0x3F80u) << 1);
            } else {
                rm[r] = 0;
                spin[PACK ? 0 : r] = v.w & 0xFFFFu;      // bits 16-18: last-touch mask
            }
            if (W0) {
                rm0[r] = 0;
                last |= ((v.w >> 16) & 7u) << (3 * r);
            }
            if (MODE == 0) {
                const bool a = v.w != CL_IDLE;
                if (a) act |= 1u << r;
                if (__ballot_sync(0xFFFFFFFFu, a)) wact |= 1u << r;
            }
        }
        if (MODE == 0) bar = __shfl_sync(0xFFFFFFFFu, A.d.cbar[inst], 0);
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
        for (int r = 0; r < R; ++r) {
            if (MODE != 0 || ((act >> r) & 1u)) {
                const uint4 v = *reinterpret_cast<const uint4*>(xg + (size_t)spin_of(r) * W + 2u * j);
                x[r][0] = v.x; x[r][1] = v.y; x[r][2] = v.z; x[r][3] = v.w;
            } else {
                x[r][0] = x[r][1] = x[r][2] = x[r][3] = 0u;
            }
        }
    };
    // a-10: every spin is owned by exactly one slot
    auto store_state = [&]() {
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (MODE != 0 || ((act >> r) & 1u))
                *reinterpret_cast<uint4*>(xg + (size_t)spin_of(r) * W + 2u * j) =
                    make_uint4(x[r][0], x[r][1], x[r][2], x[r][3]);
    };
    load_state();
    for (uint32_t e = threadIdx.x; e < 4 * CL_T; e += blockDim.x) det32[e] = 0;
    for (uint32_t e = threadIdx.x; e < 64 * CL_T; e += blockDim.x) {
        const bool kn = fhg[e] != XS_NO_HIT;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, kn);
        if ((threadIdx.x & 31) == 0) known32[e >> 5] = m;
    }
    __syncthreads();

    // ---- noise (a-6) --------------------------------------------------------------------------
    const uint32_t grp = (w0 + 2u * j) >> 2;              // Philox word group of this lane
    const uint32_t jl = j & 1u;                           // which sweep of the period this lane computes
    const uint32_t sub_sel = ((2u * j) & 3u) ? 0x7632u : 0x5410u;
    const int lane_base = (int)(threadIdx.x & 31u) - (int)jl;
    // the 64-bit addend (thr_zero : neg_thr) comes from global memory so that it sits in ordinary
    // registers: with a uniform-register addend the compiler splits the multiply-add into a
    // multiply and a two-instruction 64-bit add on the ALU pipe
    const uint2 ta = *reinterpret_cast<const uint2*>(A.d.cthr);
    const uint64_t addend = ((uint64_t)ta.y << 32) | ta.x;
    const uint32_t one = A.one;
    // Noise periods: round r works in periods of two sweeps with phase phi = r & 1: period k of round
    // r covers sweeps 2k - phi and 2k - phi + 1, so that half of the rounds renew their threshold
    // bytes in even sweeps and the other half in odd sweeps (every round of every sweep carries
    // the same work: 7 logic operations per 32 clones + half a Philox call).
    // bytes of the result: byte 2h + c = 0xFF iff word c of this lane does NOT flip k = 1 spins in
    // sweep h of the period (u >= thr)
    auto noise_call = [&](int r, uint32_t k, uint32_t& own) -> uint32_t {
        uint32_t o[4];
        philox4x32_10(spin_of(r), grp, 2u * k - (uint32_t)(r & 1) + jl, TAG_SWEEP, k0, k1, o);
        uint32_t v = 0;
        if (W0) {
            const uint32_t thr = A.thr, thr0 = A.thr0;
            v = (o[0] >= thr ? 0xFFu : 0u) | (o[1] >= thr ? 0xFF00u : 0u) |
                (o[2] >= thr ? 0xFF0000u : 0u) | (o[3] >= thr ? 0xFF000000u : 0u);
            const uint32_t v0 = (o[0] >= thr0 ? 0xFFu : 0u) | (o[1] >= thr0 ? 0xFF00u : 0u) |
                                (o[2] >= thr0 ? 0xFF0000u : 0u) | (o[3] >= thr0 ? 0xFF000000u : 0u);
            const uint32_t z0 = __shfl_sync(0xFFFFFFFFu, v0, lane_base);
            const uint32_t z1 = __shfl_sync(0xFFFFFFFFu, v0, lane_base + 1);
            rm0[W0 ? r : 0] = cl_prmt(z0, z1, sub_sel);
        } else if (SPARSE) {
            // plain compares: the shortest dependent chain (set-predicate, select, OR)
            const uint32_t thr = A.thr;
            v = (o[0] >= thr ? 0xFFu : 0u) | (o[1] >= thr ? 0xFF00u : 0u) |
                (o[2] >= thr ? 0xFF0000u : 0u) | (o[3] >= thr ? 0xFF000000u : 0u);
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint32_t ge = (uint32_t)(cl_mad_wide(o[i], one, addend) >> 32);   // 1 iff o[i] >= thr
                v = cl_mad_lo(ge, 0xFFu << (8 * i), v);
            }
        }
        own = v;
        const uint32_t s0 = __shfl_sync(0xFFFFFFFFu, v, lane_base);
        const uint32_t s1 = __shfl_sync(0xFFFFFFFFu, v, lane_base + 1);
        const uint32_t nb = cl_prmt(s0, s1, sub_sel);
        // PACK: new threshold bits (bit 7 of every byte), the spin index bits stay
        return PACK ? lop3<0xE4>(nb, rm[r], 0x80808080u) : nb;             // c ? a : b
    };
    // threshold bytes of the periods that contain sweep t
    auto produce_all = [&](uint32_t t) {
        if (!PCN) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                uint32_t own;
                rm[r] = noise_call(r, (t + (uint32_t)(r & 1)) >> 1, own);
            }
        }
    };

    // ---- sweep t (a-4..a-8); h = t & 1.  A round in the second sweep of its period replaces its
    // threshold bytes by those of the next period right after their last use; the Philox chain sits
    // in the latency shadow of the round's loads. ------------------------------------------------
    auto sweep = [&](auto hc, uint32_t t) {
        constexpr uint32_t h = decltype(hc)::value;
        uint32_t lacc[CL_H] = {0u, 0u, 0u, 0u};      // W0: OR of the clause words at their last touch
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (MODE != 0 || ((wact >> r) & 1u)) {
                const uint32_t hp = h ^ (uint32_t)(r & 1);          // sweep index inside the round's period
                const uint32_t sel0 = 0x8888u + 0x1111u * (2u * hp);
                uint32_t c0[CL_H], c1[CL_H], c2[CL_H];
                cl_lds4(ca[r][0], c0); cl_lds4(ca[r][1], c1); cl_lds4(ca[r][2], c2);
                uint32_t nf[2];
                nf[0] = cl_prmt(rm[r], 0u, sel0);
                nf[1] = cl_prmt(rm[r], 0u, sel0 + 0x1111u);
                uint32_t n0[2] = {0u, 0u};
                if (W0) {
                    n0[0] = cl_prmt(rm0[W0 ? r : 0], 0u, sel0);
                    n0[1] = cl_prmt(rm0[W0 ? r : 0], 0u, sel0 + 0x1111u);
                }
                // The address of the round's last store is made to depend (times zero) on the call's
                // result: the instruction scheduler then treats the Philox chain as the critical path
                // of the round and issues it first, interleaved with the update, in the shadow of
                // the loads, instead of leaving the loads' latency exposed and the chain for later.
                uint32_t a2 = ca[r][2];
                uint32_t rc[CL_H] = {0u, 0u, 0u, 0u};     // PCN: k = 1 flip masks of the lane's four half words
                if (PCN) {
#pragma unroll
                    for (int cw = 0; cw < 2; ++cw) {
                        uint32_t rl[8], rh[8];            // low / high halves of r_0 .. r_7 of word w0 + 2 j + cw
#pragma unroll
                        for (int jj = 0; jj < 4; ++jj) {
                            uint32_t q4[4];
                            philox4x32_10(spin_of(r), 4u * (w0 + 2u * j + (uint32_t)cw) + (uint32_t)jj, t, TAG_CLONE,
                                          k0, k1, q4);
                            rl[2 * jj] = q4[0]; rh[2 * jj] = q4[1];
                            rl[2 * jj + 1] = q4[2]; rh[2 * jj + 1] = q4[3];
                        }
                        const uint32_t lo7[7] = {rl[0], rl[1], rl[2], rl[3], rl[4], rl[5], rl[6]};
                        const uint32_t hi7[7] = {rh[0], rh[1], rh[2], rh[3], rh[4], rh[5], rh[6]};
                        rc[2 * cw] = clone_noise_mask(lo7, A.clone_m);
                        rc[2 * cw + 1] = clone_noise_mask(hi7, A.clone_m);
                    }
                }
                if (!PCN && hp == 1) {
                    uint32_t own;
                    rm[r] = noise_call(r, ((t + (uint32_t)(r & 1)) >> 1) + 1u, own);
                    if (!SPARSE) a2 = cl_mad_lo(own, A.zero, a2);
                }
#pragma unroll
                for (int c = 0; c < CL_H; ++c) {
                    const uint32_t M = lop3<LUT_MAJ>(c0[c], c1[c], c2[c]);     // k >= 2
                    const uint32_t P = lop3<LUT_XOR3>(c0[c], c1[c], c2[c]);    // k odd
                    uint32_t f = PCN ? lop3<0xF8>(M, P, rc[c])                 // M | (P & R_clone)
                                     : lop3<LUT_OR_ANDN>(M, P, nf[c >> 1]);    // flip mask (a-7)
                    if (W0) f = lop3<0xF3>(f, n0[c >> 1], 0u);                 // | (u < thr0): the k = 0 move
                    c0[c] ^= f; c1[c] ^= f; c2[c] ^= f;
                    x[r][c] ^= f;
                }
                if (W0) {
                    const uint32_t l0 = 0u - ((last >> (3 * r)) & 1u), l1 = 0u - ((last >> (3 * r + 1)) & 1u),
                                   l2 = 0u - ((last >> (3 * r + 2)) & 1u);
#pragma unroll
                    for (int c = 0; c < CL_H; ++c) {
                        lacc[c] = lop3<0xEA>(c0[c], l0, lacc[c]);              // (a & b) | c
                        lacc[c] = lop3<0xEA>(c1[c], l1, lacc[c]);
                        lacc[c] = lop3<0xEA>(c2[c], l2, lacc[c]);
                    }
                }
                cl_sts4(ca[r][0], c0); cl_sts4(ca[r][1], c1); cl_sts4(a2, c2);
            }
            if (W0 && r == R - 1) {
                // every clause word has had its last touch: clones with a set bit are not in a ground state
                uint32_t* det = det32 + (t & 1u) * 2u * CL_T;
#pragma unroll
                for (int c = 0; c < CL_H; ++c) {
                    lacc[c] |= __shfl_xor_sync(0xFFFFFFFFu, lacc[c], 4);
                    lacc[c] |= __shfl_xor_sync(0xFFFFFFFFu, lacc[c], 8);
                    lacc[c] |= __shfl_xor_sync(0xFFFFFFFFu, lacc[c], 16);
                    if ((threadIdx.x & 31u) < CL_LPS && lacc[c]) atomicOr(&det[CL_H * j + c], lacc[c]);
                }
            }
            if (MODE == 1 || (MODE == 2 && (r & 1)) || (MODE == 0 && ((bar >> r) & 1u)))
                __syncthreads();                                              // a-8
        }
    };

    // W0: after the last barrier of sweep t, record the clones whose clause words are all clear and
    // clear the buffer for sweep t + 2
    auto w0_commit = [&](uint32_t t) {
        uint32_t* det = det32 + (t & 1u) * 2u * CL_T;
        for (uint32_t e = threadIdx.x; e < 2 * CL_T; e += blockDim.x) {
            uint32_t newly = ~det[e] & ~known32[e];
            det[e] = 0;
            known32[e] |= newly;
            while (newly) {
                const int bit = __ffs(newly) - 1;
                newly &= newly - 1;
                fhg[32 * e + bit] = t;
            }
        }
    };

    // ---- solved mask of the tile -> det32 (bit set = some interaction unsatisfied) ----------
    auto detect = [&]() {
        for (uint32_t e = threadIdx.x; e < 2 * CL_T; e += blockDim.x) det32[e] = 0;
        if (threadIdx.x == 0) *flag = 0;
        __syncthreads();
        uint32_t acc[CL_H] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (MODE != 0 || ((act >> r) & 1u)) {
                uint32_t c0[CL_H], c1[CL_H], c2[CL_H];
                cl_lds4(ca[r][0], c0); cl_lds4(ca[r][1], c1); cl_lds4(ca[r][2], c2);
#pragma unroll
                for (int c = 0; c < CL_H; ++c) acc[c] |= c0[c] | c1[c] | c2[c];
            }
        }
#pragma unroll
        for (int c = 0; c < CL_H; ++c)
            if (acc[c]) atomicOr(&det32[CL_H * j + c], acc[c]);
        __syncthreads();
    };

    // sweeps t0+1 .. t0+n; exact: record first hits after every sweep (L293)
    auto run_range = [&](uint32_t t0, uint32_t n, bool exact) {
        auto post = [&](uint32_t t) {
            if (W0) { w0_commit(t); return; }
            if (!exact) return;
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
        };
        uint32_t t = t0 + 1;
        const uint32_t t_last = t0 + n;
        produce_all(t);
        if (t & 1u) {
            sweep(std::integral_constant<uint32_t, 1>{}, t);
            post(t);
            ++t;
        }
        for (; t < t_last; t += 2) {
            sweep(std::integral_constant<uint32_t, 0>{}, t);
            post(t);
            sweep(std::integral_constant<uint32_t, 1>{}, t + 1);
            post(t + 1);
        }
        if (t == t_last) {
            sweep(std::integral_constant<uint32_t, 0>{}, t);
            post(t);
        }
    };

    uint32_t t = (uint32_t)rec0.sweeps_done;
    uint32_t remaining = A.n_sweeps;
    while (remaining) {
        const uint32_t nb = min(A.batch, remaining);
        run_range(t, nb, false);
        if (W0) {                  // first hits are already exact; no detection pass, no replay
            store_state();
            t += nb;
            remaining -= nb;
            continue;
        }
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

// ---- launch of one R family; each family is instantiated in its own translation unit ---------
struct ClauseLaunch {
    uint32_t threads, ctas, smem, mode;
    bool w0;             // flip table with w0 > 0 (MODE 1 only)
    bool pcn;            // per-clone noise (MODE 1 only)
    bool dense;          // more CTAs than SMs: prefer the register-capped variants
    cudaStream_t st;
};

template <int R, int MT, int MINB, int MODE, bool W0 = false, bool PCN = false>
cudaError_t launch_clause_k(const ClauseArgs& A, const ClauseLaunch& L)
{
    cudaError_t e = cudaFuncSetAttribute(k_sweep_clause<R, MT, MINB, MODE, W0, PCN>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);
    if (e != cudaSuccess) return e;
    k_sweep_clause<R, MT, MINB, MODE, W0, PCN><<<L.ctas, L.threads, L.smem, L.st>>>(A);
    return cudaGetLastError();
}

template <int R, int MT, int MINB>
cudaError_t launch_clause_m(const ClauseArgs& A, const ClauseLaunch& L)
{
    if (L.mode == 1 && L.pcn) return launch_clause_k<R, MT, MINB, 1, false, true>(A, L);
    if (L.mode == 1 && L.w0) return launch_clause_k<R, MT, MINB, 1, true>(A, L);
    if (L.mode == 1) return launch_clause_k<R, MT, MINB, 1>(A, L);
    if (L.mode == 2 && R % 2 == 0) return launch_clause_k<R, MT, MINB, (R % 2 == 0 ? 2 : 0)>(A, L);
    return launch_clause_k<R, MT, MINB, 0>(A, L);
}

template <int R>
cudaError_t launch_clause_unit(const ClauseArgs& A, const ClauseLaunch& L)
{
    if (L.threads == 128) return launch_clause_m<R, 128, 4>(A, L);
    if (L.threads == 256) return L.dense ? launch_clause_m<R, 256, 2>(A, L) : launch_clause_m<R, 256, 1>(A, L);
    return launch_clause_m<R, 512, 1>(A, L);
}

// 9 .. 16 rounds per sweep (orders with many small sets, e.g. the paper's cap-32 sets, L279): the
// general form only, without a register cap (one CTA of at most 256 threads per launch bound).
template <int R>
cudaError_t launch_clause_unit_long(const ClauseArgs& A, const ClauseLaunch& L)
{
    if (L.threads == 128) return launch_clause_k<R, 128, 1, 0>(A, L);
    return launch_clause_k<R, 256, 1, 0>(A, L);
}

}  // namespace xs
