// xs_sweep_static.cuh -- the static-task sweep kernel (template).  Included by the instantiation
// units xs_sweep_static_i*.cu (one per (CW, NC), so that they compile in parallel) and by the host
// side xs_sweep_static.cu (declarations only).
//
// Same tile ownership as k_sweep_tile (a CTA keeps (instance, T word columns) in shared
// memory for the whole call; lanes <-> clone words of one spin row, sets
// separated by __syncthreads, L277), but the work list of every thread is fixed for the whole
// call and lives in REGISTERS: in "round" r of a sweep, thread (slot, j) updates words
// CW*j .. CW*j+CW-1 of the spin at position set_start[s(r)] + q(r) * n_slots + slot.  Because
// the update order is instance data (L289), the 6 partner addresses, the 3 coupling masks and
// the thread's own spin words of each round stay in registers; the hot loop has no index
// loads, no address arithmetic and never re-reads its own row.
//
// Noise (a-6): each Philox4x32-10 call yields the numbers of 4 consecutive words of a spin.
// The NL = 4 / CW lanes that share a word group each compute the call of one sweep of a period
// of NL sweeps and exchange the threshold bytes by warp shuffles, so every call is evaluated
// exactly once and nothing goes through shared memory.
//
// Bank conflicts: for T = 8 a spin row is 64 B, so the two spins served by one 128-byte phase
// of a shared load collide when their rows have the same parity.  The kernel keeps NC = 16 / T
// copies of every row in one 128 B line (T = 8: banks 0-15 and 16-31; T = 4: four quarters);
// slot s reads copy s % NC, and a write updates all copies in NC conflict-free stores (in
// store c, slot s writes copy (s + c) % NC).  T >= 16 rows are whole 128 B lines and need no
// copy.  Lanes without a task in a round work on a scratch line, so the hot loop has no
// per-lane branch; warps without any task skip the round.
//
// Ground-state detection / exact first hit: as in k_sweep_tile (detection pass every `batch`
// sweeps, replay of the batch from the global copy with a pass after every sweep, L293).
#pragma once
#include <type_traits>

#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

struct StaticArgs {
    DevPtrs d;
    uint32_t N, W, T, n_sweeps, thr, flags, batch;
    uint32_t line_shift;   // log2(bytes of one spin line in shared memory)
    uint32_t off_misc;     // byte offset of det32 / known32 / flag in dynamic shared memory
};

// CW uint64 words = 2*CW uint32 per lane, by 32-bit shared address
template <int CW> __device__ __forceinline__ void lds(uint32_t addr, uint32_t (&o)[2 * CW]);
template <> __device__ __forceinline__ void lds<2>(uint32_t addr, uint32_t (&o)[4])
{
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]) : "r"(addr) : "memory");
}
template <> __device__ __forceinline__ void lds<1>(uint32_t addr, uint32_t (&o)[2])
{
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(o[0]), "=r"(o[1]) : "r"(addr) : "memory");
}
template <int CW> __device__ __forceinline__ void sts(uint32_t addr, const uint32_t (&o)[2 * CW]);
template <> __device__ __forceinline__ void sts<2>(uint32_t addr, const uint32_t (&o)[4])
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "r"(addr), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
}
template <> __device__ __forceinline__ void sts<1>(uint32_t addr, const uint32_t (&o)[2])
{
    asm volatile("st.shared.v2.u32 [%0], {%1,%2};" :: "r"(addr), "r"(o[0]), "r"(o[1]) : "memory");
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// Per-round register state of a thread.
template <int MAXT, int CW>
struct Tasks {
    uint32_t a[MAXT][6];       // shared addresses of the partner words (incl. lane and copy offset)
    uint32_t self[MAXT];       // shared address of the own words (copy read by this thread)
    uint32_t jm[MAXT][3];      // coupling masks
    uint32_t rmn[MAXT];        // noise bytes of the next period (produced inside the sweeps)
    uint32_t rm[MAXT];         // noise bytes of the current period: byte CW*h + c = 0xFF iff word c
                               // flips k=1 spins in sweep h of the period
    uint32_t x[MAXT][2 * CW];  // the thread's own spin words (mirror of shared memory)
    uint32_t act;              // bit r: this thread has a task in round r
    uint32_t wact;             // bit r: some lane of this warp has a task in round r
    uint32_t bar;              // bit r: round r is the last of its set (CTA-uniform)
    uint32_t n_rounds;         // CTA-uniform
};

// MAXT: unrolled rounds per sweep; MAXTHREADS / MINB: launch bounds (MINB > 1 caps the registers so
// that several CTAs share an SM when there are more tiles than SMs).
// FULL: every instance has exactly MAXT sets of one round each and every warp has a task in every
// round (balanced sets on a matching CTA size): the round loop carries no tests at all.
template <int MAXT, int CW, int NC, int MAXTHREADS, int MINB, bool FULL>
__global__ void __launch_bounds__(MAXTHREADS, MINB) k_sweep_static(StaticArgs A)
{
    constexpr int H = 2 * CW;          // uint32 halves per lane
    constexpr uint32_t NL = 4 / CW;    // lanes sharing a Philox call = sweeps per noise period
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t N = A.N, W = A.W, T = A.T;
    const uint32_t tiles = W / T;
    const uint32_t inst = blockIdx.x / tiles;
    const uint32_t w0 = (blockIdx.x % tiles) * T;
    const xs_tts_rec rec0 = A.d.rec[inst];
    if (rec0.solved && !(A.flags & XS_FLAG_NO_SKIP)) return;   // stop rule (L129, L293)

    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t shift = A.line_shift;
    uint32_t* det32 = reinterpret_cast<uint32_t*>(smem + A.off_misc);
    uint32_t* known32 = det32 + 2 * T;
    uint32_t* flag = known32 + 2 * T;

    const uint32_t LPS = T / CW;
    const uint32_t slot = threadIdx.x / LPS, n_slots = blockDim.x / LPS;
    const uint32_t j = threadIdx.x % LPS;
    // NC copies of every row in its 128-byte line; slot s reads copy s % NC (conflict-free phases)
    constexpr uint32_t ROWB = 128u / NC;                  // bytes of one copy (= 8 T when NC > 1)
    const uint32_t sm = slot % NC;
    const uint32_t cpy = NC > 1 ? sm * ROWB : 0u;
    const uint32_t lane_off = base + cpy + j * (8u * CW);

    const uint64_t seed = A.d.run_seed[inst];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w0;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w0) * 64;

    // ---- static task list (a-1 tables -> registers) ---------------------------------------
    Tasks<MAXT, CW> tk;
    tk.act = 0; tk.wact = 0; tk.bar = 0; tk.n_rounds = 0;
    {
        const AdjRec* adj = A.d.adj + (size_t)inst * N;
        const uint32_t* ss = A.d.set_start + (size_t)inst * (N + 1);
        const uint32_t n_sets = A.d.n_sets[inst];
        uint32_t s = 0, q = 0;
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            const bool valid = s < n_sets;
            const uint32_t p0 = valid ? ss[s] : 0u, p1 = valid ? ss[s + 1] : 0u;
            const uint32_t pos = p0 + q * n_slots + slot;
            const bool active = valid && pos < p1;
            const bool last = valid && (p0 + (q + 1) * n_slots >= p1);
            // lanes without a task work on the scratch line N: no per-lane branch in the hot loop
            uint4 r0 = make_uint4(N, N, N, N), r1 = make_uint4(N, N, N, 0);
            if (__ballot_sync(0xFFFFFFFFu, active)) tk.wact |= 1u << r;
            if (active) {
                const uint4* rp = reinterpret_cast<const uint4*>(adj + pos);
                r0 = rp[0];
                r1 = rp[1];
                tk.act |= 1u << r;
            }
            tk.a[r][0] = lane_off + (r0.x << shift);
            tk.a[r][1] = lane_off + (r0.y << shift);
            tk.a[r][2] = lane_off + (r0.z << shift);
            tk.a[r][3] = lane_off + (r0.w << shift);
            tk.a[r][4] = lane_off + (r1.x << shift);
            tk.a[r][5] = lane_off + (r1.y << shift);
            tk.self[r] = lane_off + (r1.z << shift);
            tk.jm[r][0] = (r1.w & 1u) ? ~0u : 0u;
            tk.jm[r][1] = (r1.w & 2u) ? ~0u : 0u;
            tk.jm[r][2] = (r1.w & 4u) ? ~0u : 0u;
            tk.rm[r] = 0;
            tk.rmn[r] = 0;
            if (valid) tk.n_rounds = r + 1;
            if (last) { tk.bar |= 1u << r; ++s; q = 0; } else { ++q; }
        }
    }

    tk.n_rounds = __shfl_sync(0xFFFFFFFFu, tk.n_rounds, 0);   // tell the compiler: warp-uniform
    tk.bar = __shfl_sync(0xFFFFFFFFu, tk.bar, 0);

    auto load_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            const uint64_t v = xg[(size_t)i * W + lw];
            unsigned char* line = smem + ((size_t)i << shift);
            reinterpret_cast<uint64_t*>(line)[lw] = v;
#pragma unroll
            for (int c = 1; c < NC; ++c) reinterpret_cast<uint64_t*>(line + c * ROWB)[lw] = v;
        }
    };
    auto store_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            xg[(size_t)i * W + lw] = reinterpret_cast<const uint64_t*>(smem + ((size_t)i << shift))[lw];
        }
    };
    auto reload_x = [&]() {
#pragma unroll
        for (int r = 0; r < MAXT; ++r) lds<CW>(tk.self[r], tk.x[r]);
    };
    load_state();
    for (uint32_t e = threadIdx.x; e < 64 * T; e += blockDim.x) {
        const bool kn = fhg[e] != XS_NO_HIT;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, kn);
        if ((threadIdx.x & 31) == 0) known32[e >> 5] = m;
    }
    __syncthreads();
    reload_x();

    // ---- noise (a-6): threshold bytes of this lane's words for the NL sweeps of a period ---
    const uint32_t grp = (w0 + CW * j) >> 2;              // Philox word group of this lane
    const uint32_t jl = j % NL;                           // which sweep of the period this lane computes
    const uint32_t sub = (CW * j) & 3u;                   // first byte of this lane's words in a call
    const int lane_base = (int)(threadIdx.x & 31u) - (int)jl;
    const uint32_t thr = A.thr;
    auto noise_call = [&](int r, uint32_t q) -> uint32_t {
        const uint32_t spin = (tk.self[r] - lane_off) >> shift;
        uint32_t o[4];
        philox4x32_10(spin, grp, NL * q + jl, TAG_SWEEP, k0, k1, o);
        const uint32_t v = (o[0] < thr ? 0xFFu : 0u) | (o[1] < thr ? 0xFF00u : 0u) |
                           (o[2] < thr ? 0xFF0000u : 0u) | (o[3] < thr ? 0xFF000000u : 0u);
        const uint32_t s0 = __shfl_sync(0xFFFFFFFFu, v, lane_base);
        const uint32_t s1 = __shfl_sync(0xFFFFFFFFu, v, lane_base + 1);
        if (CW == 2) return prmt(s0, s1, sub ? 0x7632u : 0x5410u);
        const uint32_t s2 = __shfl_sync(0xFFFFFFFFu, v, lane_base + 2);
        const uint32_t s3 = __shfl_sync(0xFFFFFFFFu, v, lane_base + 3);
        const uint32_t pick = sub | ((4u + sub) << 4);
        return prmt(prmt(s0, s1, pick), prmt(s2, s3, pick), 0x5410u);
    };
    // all rounds of period q at once (branch-free: the calls interleave)
    auto produce_all = [&](uint32_t q) {
#pragma unroll
        for (int r = 0; r < MAXT; ++r) tk.rm[r] = noise_call(r, q);
    };

    // ---- one sweep (a-4..a-8); h = index of the sweep inside the noise period.  With `fuse`
    // the Philox calls of period qn for the rounds r = h (mod NL) are issued right after the
    // round's shared loads, i.e. in their latency shadow. --------------------------------------
    auto sweep = [&](auto hc, uint32_t qn) {
        constexpr uint32_t h = decltype(hc)::value;
        constexpr uint32_t sel0 = 0x8888u + 0x1111u * (CW * h);
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            if (FULL || r < (int)tk.n_rounds) {
                if (FULL || ((tk.wact >> r) & 1u)) {
                    uint32_t a0[H], b0[H], a1[H], b1[H], a2[H], b2[H], xn[H];
                    lds<CW>(tk.a[r][0], a0); lds<CW>(tk.a[r][1], b0);
                    lds<CW>(tk.a[r][2], a1); lds<CW>(tk.a[r][3], b1);
                    lds<CW>(tk.a[r][4], a2); lds<CW>(tk.a[r][5], b2);
                    uint32_t R[CW];
#pragma unroll
                    for (int c = 0; c < CW; ++c) R[c] = prmt(tk.rm[r], 0u, sel0 + 0x1111u * c);
                    if ((uint32_t)r % NL == h) tk.rmn[r] = noise_call(r, qn);   // compile-time test
#pragma unroll
                    for (int c = 0; c < H; ++c)
                        xn[c] = qg_update(a0[c], b0[c], tk.jm[r][0], a1[c], b1[c], tk.jm[r][1], a2[c],
                                          b2[c], tk.jm[r][2], tk.x[r][c], R[c >> 1]);
                    sts<CW>(tk.self[r], xn);
                    // the other copies: in store c, slot s writes copy (s + c) % NC
#pragma unroll
                    for (int c = 1; c < NC; ++c)
                        sts<CW>(tk.self[r] + (((sm + c) % NC) - sm) * ROWB, xn);
#pragma unroll
                    for (int c = 0; c < H; ++c) tk.x[r][c] = xn[c];
                }
                if (FULL || ((tk.bar >> r) & 1u)) __syncthreads();
            }
        }
    };

    // ---- solved mask of the current tile -> det32 (bit set = NOT solved) -------------------
    auto detect = [&]() {
        for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x) det32[e] = 0;
        if (threadIdx.x == 0) *flag = 0;
        __syncthreads();
        uint32_t acc[H];
#pragma unroll
        for (int c = 0; c < H; ++c) acc[c] = 0;
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            if (r < (int)tk.n_rounds && ((tk.act >> r) & 1u)) {
                uint32_t a0[H], b0[H], a1[H], b1[H], a2[H], b2[H];
                lds<CW>(tk.a[r][0], a0); lds<CW>(tk.a[r][1], b0);
                lds<CW>(tk.a[r][2], a1); lds<CW>(tk.a[r][3], b1);
                lds<CW>(tk.a[r][4], a2); lds<CW>(tk.a[r][5], b2);
#pragma unroll
                for (int c = 0; c < H; ++c)
                    acc[c] |= qg_nonzero_k(a0[c], b0[c], tk.jm[r][0], a1[c], b1[c], tk.jm[r][1], a2[c],
                                           b2[c], tk.jm[r][2], tk.x[r][c]);
            }
        }
#pragma unroll
        for (int c = 0; c < H; ++c)
            if (acc[c]) atomicOr(&det32[H * j + c], acc[c]);
        __syncthreads();
    };

    // sweeps t0+1 .. t0+n; exact: record first hits after every sweep
    auto run_range = [&](uint32_t t0, uint32_t n, bool exact) {
        const uint32_t t_first = t0 + 1, t_last = t0 + n;
        const uint32_t q_last = t_last / NL;
        bool have_next = false;
        for (uint32_t q = t_first / NL; q <= q_last; ++q) {
            if (have_next) {
#pragma unroll
                for (int r = 0; r < MAXT; ++r) tk.rm[r] = tk.rmn[r];
            } else {
                produce_all(q);
            }
            // the next period's noise can be produced inside this period's sweeps iff all NL
            // sweeps of this period run and there is a next period
            const bool fuse = (NL * q >= t_first) && (NL * q + NL - 1 <= t_last) && (q < q_last);
            auto step = [&](auto hc) {
                const uint32_t t = NL * q + decltype(hc)::value;
                if (t < t_first || t > t_last) return;
                sweep(hc, q + 1);
                if (exact) {
                    detect();
                    for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x) {
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
            if (NL > 1) step(std::integral_constant<uint32_t, 1 % NL>{});
            if (NL > 2) {
                step(std::integral_constant<uint32_t, 2 % NL>{});
                step(std::integral_constant<uint32_t, 3 % NL>{});
            }
            have_next = fuse;
        }
    };

    uint32_t t = (uint32_t)rec0.sweeps_done;
    uint32_t remaining = A.n_sweeps;
    while (remaining) {
        const uint32_t nb = min(A.batch, remaining);
        run_range(t, nb, false);
        detect();
        for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x)
            if (~det32[e] & ~known32[e]) *flag = 1;
        __syncthreads();
        const bool replay = *flag != 0;
        __syncthreads();
        if (replay) {
            load_state();          // global copy = state at the start of this batch
            __syncthreads();
            reload_x();
            run_range(t, nb, true);
        }
        store_state();             // a-10 (also the replay checkpoint of the next batch)
        t += nb;
        remaining -= nb;
    }
}


// ---- launch of one (CW, NC) family; each family is instantiated in its own translation unit ----
struct StaticLaunch {
    uint32_t rounds;     // rounds per sweep (<= 8)
    uint32_t threads, ctas, smem;
    bool dense;          // more CTAs than SMs: prefer the register-capped variants
    bool full;           // see FULL
    cudaStream_t st;
};

template <int MAXT, int CW, int NC, int MT, int MINB, bool FULL>
cudaError_t launch_static_k(const StaticArgs& A, const StaticLaunch& L)
{
    cudaError_t e = cudaFuncSetAttribute(k_sweep_static<MAXT, CW, NC, MT, MINB, FULL>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);
    if (e != cudaSuccess) return e;
    k_sweep_static<MAXT, CW, NC, MT, MINB, FULL><<<L.ctas, L.threads, L.smem, L.st>>>(A);
    return cudaGetLastError();
}

template <int CW, int NC, int MT, int MINB>
cudaError_t launch_static_t(const StaticArgs& A, const StaticLaunch& L)
{
    // fewer unrolled rounds = fewer registers
    if (L.rounds == 4 && L.full) return launch_static_k<4, CW, NC, MT, MINB, true>(A, L);
    if (L.rounds <= 4) return launch_static_k<4, CW, NC, MT, MINB, false>(A, L);
    if (L.rounds <= 6) return launch_static_k<6, CW, NC, MT, MINB, false>(A, L);
    return launch_static_k<8, CW, NC, MT, MINB, false>(A, L);
}

template <int CW, int NC>
cudaError_t launch_static_unit(const StaticArgs& A, const StaticLaunch& L)
{
    if (L.threads <= 128) return launch_static_t<CW, NC, 128, 4>(A, L);
    if (L.threads <= 256) return L.dense ? launch_static_t<CW, NC, 256, 2>(A, L)
                                         : launch_static_t<CW, NC, 256, 1>(A, L);
    if (L.threads <= 384) return launch_static_t<CW, NC, 384, 1>(A, L);
    return launch_static_t<CW, NC, 512, 1>(A, L);
}

}  // namespace xs
