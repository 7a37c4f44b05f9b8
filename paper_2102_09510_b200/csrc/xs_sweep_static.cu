// xs_sweep_static.cu -- a-3..a-10, on-chip regime, "static task" variant of the sweep kernel.
//
// Same tile ownership as k_sweep_tile (a CTA keeps (instance, T word columns) in shared
// memory for the whole call; lanes <-> clone words of one spin row, sets
// separated by __syncthreads, L277), but the work list of every thread is fixed for the whole
// call and lives in REGISTERS: in "round" r of a sweep, thread (slot, j) updates words
// 2j, 2j+1 of the spin at position set_start[s(r)] + q(r) * n_slots + slot.  Because the
// update order is instance data (L289), the 7 shared-memory addresses and the 3 coupling masks
// of each round are loaded once; the hot loop has no index loads and no address arithmetic.
//
// Noise (a-6): each Philox4x32-10 call yields the numbers of 4 consecutive words of a spin.
// The two lanes (j, j^1) that share a word group compute the calls of the even and the odd
// sweep of a sweep pair and exchange the 4 threshold bytes by one warp shuffle, so every call
// is evaluated exactly once and nothing goes through shared memory.
//
// Bank conflicts: for T = 8 a spin row is 64 B, so the two spins served by one quarter-warp
// phase of an LDS.128 collide when their rows have the same parity.  DUP keeps two copies of
// every row in one 128 B line (banks 0-15 and 16-31); even slots read copy 0, odd slots copy
// 1, and a write updates both copies in two conflict-free stores.  T >= 16 rows are whole
// 128 B lines and need no copy.
//
// Ground-state detection / exact first hit: as in k_sweep_tile (detection pass every `batch`
// sweeps, replay of the batch from the global copy with a pass after every sweep, L293).
#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

void count_launch(uint64_t n);

struct StaticArgs {
    DevPtrs d;
    uint32_t N, W, T, n_sweeps, thr, flags, batch;
    uint32_t line_shift;   // log2(bytes of one spin line in shared memory)
    uint32_t off_misc;     // byte offset of det32 / known32 / flag in dynamic shared memory
};

__device__ __forceinline__ void lds128(uint32_t addr, uint32_t (&o)[4])
{
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint32_t (&o)[4])
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "r"(addr), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// Per-round register state of a thread.
template <int MAXT>
struct Tasks {
    uint32_t a[MAXT][6];   // shared addresses of the partner words (incl. lane and copy offset)
    uint32_t self[MAXT];   // shared address of the own words (copy read by this thread)
    uint32_t jm[MAXT][3];  // coupling masks
    uint32_t rm[MAXT];     // noise: byte 2h+c = 0xFF iff word c flips k=1 spins in sweep h of the pair
    uint32_t act;          // bit r: this thread has a task in round r
    uint32_t bar;          // bit r: round r is the last of its set (CTA-uniform)
    uint32_t n_rounds;     // CTA-uniform
};

template <int MAXT, bool DUP, int MAXTHREADS>
__global__ void __launch_bounds__(MAXTHREADS, 1) k_sweep_static(StaticArgs A)
{
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

    const uint32_t LPS = T / 2;
    const uint32_t slot = threadIdx.x / LPS, n_slots = blockDim.x / LPS;
    const uint32_t j = threadIdx.x % LPS;
    const uint32_t cpy = DUP ? (slot & 1u) * 64u : 0u;
    const uint32_t lane_off = base + cpy + j * 16u;

    const uint64_t seed = A.d.run_seed[inst];
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w0;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w0) * 64;

    // ---- static task list (a-1 tables -> registers) ---------------------------------------
    Tasks<MAXT> tk;
    tk.act = 0; tk.bar = 0; tk.n_rounds = 0;
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
            uint4 r0 = make_uint4(0, 0, 0, 0), r1 = make_uint4(0, 0, 0, 0);
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
            if (valid) tk.n_rounds = r + 1;
            if (last) { tk.bar |= 1u << r; ++s; q = 0; } else { ++q; }
        }
    }

    auto load_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            const uint64_t v = xg[(size_t)i * W + lw];
            unsigned char* line = smem + ((size_t)i << shift);
            reinterpret_cast<uint64_t*>(line)[lw] = v;
            if (DUP) reinterpret_cast<uint64_t*>(line + 64)[lw] = v;
        }
    };
    auto store_state = [&]() {
        for (uint32_t e = threadIdx.x; e < N * T; e += blockDim.x) {
            const uint32_t i = e / T, lw = e - i * T;
            xg[(size_t)i * W + lw] = reinterpret_cast<const uint64_t*>(smem + ((size_t)i << shift))[lw];
        }
    };
    load_state();
    for (uint32_t e = threadIdx.x; e < 64 * T; e += blockDim.x) {
        const bool kn = fhg[e] != XS_NO_HIT;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, kn);
        if ((threadIdx.x & 31) == 0) known32[e >> 5] = m;
    }
    __syncthreads();

    // ---- noise of sweep pair q: sweeps 2q (h = 0) and 2q + 1 (h = 1) ----------------------
    const uint32_t grp = (w0 >> 2) + (j >> 1);
    const uint32_t selj = (j & 1u) ? 0x3276u : 0x5410u;
    auto produce = [&](uint32_t q) {
        const uint32_t t_mine = 2u * q + (j & 1u);
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            if (r < (int)tk.n_rounds) {
                uint32_t v = 0;
                if ((tk.act >> r) & 1u) {
                    const uint32_t spin = (tk.self[r] - lane_off) >> shift;
                    uint32_t o[4];
                    philox4x32_10(spin, grp, t_mine, TAG_SWEEP, k0, k1, o);
                    v = (o[0] < A.thr ? 0xFFu : 0u) | (o[1] < A.thr ? 0xFF00u : 0u) |
                        (o[2] < A.thr ? 0xFF0000u : 0u) | (o[3] < A.thr ? 0xFF000000u : 0u);
                }
                const uint32_t other = __shfl_xor_sync(0xFFFFFFFFu, v, 1);
                tk.rm[r] = prmt(v, other, selj);
            }
        }
    };

    // ---- one sweep (a-4..a-8); h selects the sweep of the pair -----------------------------
    auto sweep = [&](uint32_t h) {
        const uint32_t sel0 = 0x8888u + 0x2222u * h, sel1 = sel0 + 0x1111u;
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            if (r < (int)tk.n_rounds) {
                if ((tk.act >> r) & 1u) {
                    uint32_t a0[4], b0[4], a1[4], b1[4], a2[4], b2[4], x[4], xn[4];
                    lds128(tk.a[r][0], a0); lds128(tk.a[r][1], b0);
                    lds128(tk.a[r][2], a1); lds128(tk.a[r][3], b1);
                    lds128(tk.a[r][4], a2); lds128(tk.a[r][5], b2);
                    lds128(tk.self[r], x);
                    const uint32_t R0 = prmt(tk.rm[r], 0u, sel0), R1 = prmt(tk.rm[r], 0u, sel1);
#pragma unroll
                    for (int c = 0; c < 4; ++c)
                        xn[c] = qg_update(a0[c], b0[c], tk.jm[r][0], a1[c], b1[c], tk.jm[r][1], a2[c],
                                          b2[c], tk.jm[r][2], x[c], c < 2 ? R0 : R1);
                    sts128(tk.self[r], xn);
                    if (DUP) sts128(tk.self[r] ^ 64u, xn);
                }
                if ((tk.bar >> r) & 1u) __syncthreads();
            }
        }
    };

    // ---- solved mask of the current tile -> det32 (bit set = NOT solved) -------------------
    auto detect = [&]() {
        for (uint32_t e = threadIdx.x; e < 2 * T; e += blockDim.x) det32[e] = 0;
        if (threadIdx.x == 0) *flag = 0;
        __syncthreads();
        uint32_t acc[4] = {0, 0, 0, 0};
#pragma unroll
        for (int r = 0; r < MAXT; ++r) {
            if (r < (int)tk.n_rounds && ((tk.act >> r) & 1u)) {
                uint32_t a0[4], b0[4], a1[4], b1[4], a2[4], b2[4], x[4];
                lds128(tk.a[r][0], a0); lds128(tk.a[r][1], b0);
                lds128(tk.a[r][2], a1); lds128(tk.a[r][3], b1);
                lds128(tk.a[r][4], a2); lds128(tk.a[r][5], b2);
                lds128(tk.self[r], x);
#pragma unroll
                for (int c = 0; c < 4; ++c)
                    acc[c] |= qg_nonzero_k(a0[c], b0[c], tk.jm[r][0], a1[c], b1[c], tk.jm[r][1], a2[c],
                                           b2[c], tk.jm[r][2], x[c]);
            }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (acc[c]) atomicOr(&det32[4 * j + c], acc[c]);
        __syncthreads();
    };

    // sweeps t0+1 .. t0+n; exact: record first hits after every sweep
    auto run_range = [&](uint32_t t0, uint32_t n, bool exact) {
        const uint32_t t_first = t0 + 1, t_last = t0 + n;
        for (uint32_t q = t_first >> 1; q <= (t_last >> 1); ++q) {
            produce(q);
            for (uint32_t h = 0; h < 2; ++h) {
                const uint32_t t = 2u * q + h;
                if (t < t_first || t > t_last) continue;
                sweep(h);
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
            }
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
            run_range(t, nb, true);
        }
        store_state();             // a-10 (also the replay checkpoint of the next batch)
        t += nb;
        remaining -= nb;
    }
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
constexpr int STATIC_MAXT = 8;
constexpr uint32_t STATIC_SMEM_MAX = 227u * 1024u;

static uint32_t static_line_shift(uint32_t T)
{
    uint32_t bytes = (T == 8) ? 128u : T * 8u, sh = 0;
    while ((1u << sh) < bytes) ++sh;
    return sh;
}

uint32_t static_smem_bytes(uint32_t N, uint32_t T)
{
    const uint64_t state = (uint64_t)N << static_line_shift(T);
    const uint64_t total = state + (4ull * T + 4) * 4 + 128;
    return total > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)total;
}

// rounds a CTA of `threads` threads needs per sweep for tile width T (max over instances)
uint32_t static_rounds(const xs_batch& b, uint32_t T, uint32_t threads)
{
    const uint32_t n_slots = threads / (T / 2);
    if (n_slots == 0) return 0xFFFFFFFFu;
    uint32_t worst = 0;
    for (const HostGraph& g : b.graphs) {
        uint32_t r = 0;
        for (size_t s = 0; s + 1 < g.set_start.size(); ++s)
            r += (g.set_start[s + 1] - g.set_start[s] + n_slots - 1) / n_slots;
        worst = std::max(worst, r);
    }
    return worst;
}

bool static_feasible(const xs_batch& b, uint32_t T, uint32_t threads)
{
    if (T < 8 || T > 64 || (T & (T - 1)) || b.p.n_words % T) return false;
    if (threads % 32 || threads < 32 || threads > 512 || threads % (T / 2)) return false;
    if (static_smem_bytes(b.p.n_spins, T) > STATIC_SMEM_MAX) return false;
    return static_rounds(b, T, threads) <= (uint32_t)STATIC_MAXT;
}

int launch_sweep_static(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    const xs_params& p = b.p;
    const TileGeom& g = b.geom;
    StaticArgs A;
    A.d = b.d;
    A.N = p.n_spins; A.W = p.n_words; A.T = g.T; A.n_sweeps = n_sweeps;
    A.thr = p.w1_threshold; A.flags = p.flags; A.batch = g.batch;
    A.line_shift = static_line_shift(g.T);
    A.off_misc = (uint32_t)(((uint64_t)p.n_spins << A.line_shift) + 127) / 128 * 128;
    const uint32_t smem = g.smem;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
#define XS_LAUNCH(DUPV, MT)                                                                            \
    do {                                                                                               \
        e = cudaFuncSetAttribute(k_sweep_static<STATIC_MAXT, DUPV, MT>,                                \
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);              \
        if (e == cudaSuccess) k_sweep_static<STATIC_MAXT, DUPV, MT><<<g.ctas, g.threads, smem, st>>>(A); \
    } while (0)
    if (g.T == 8) {
        if (g.threads <= 256) XS_LAUNCH(true, 256); else XS_LAUNCH(true, 512);
    } else {
        if (g.threads <= 256) XS_LAUNCH(false, 256); else XS_LAUNCH(false, 512);
    }
#undef XS_LAUNCH
    if (e != cudaSuccess) return (int)e;
    count_launch(1);
    return (int)cudaGetLastError();
}

}  // namespace xs
