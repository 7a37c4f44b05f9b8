// xs_sweep_warp.cu -- the latency kernel: few clone words and few instances (BASELINE.json
// configs[0]: N = 64, one uint64 word of 64 clones, run until E = -N).  There is one warp of work
// per word column, so what counts is the length of the dependent chain of one sweep, not
// throughput ("config 1: latency; report sweeps/us").
//
// A CTA owns (instance, all W <= 4 word columns).  Warp w < W is the CONSUMER of column w: its 32
// lanes are 16 slots x the two uint32 halves of the column's word; a "pass" puts one spin of the
// current independent set on every slot (lanes <-> spins of the set, a warp
// synchronisation after each set -- with one word per spin the paper's own mapping is the right
// one).  Shared memory holds the column's CLAUSE words c_t = x_i ^ x_j ^ x_k ^ J_t (as in
// xs_sweep_clause.cuh): a pass is 3 loads, M = maj, P = parity, flip = M | (P & R), 3 stores,
// __syncwarp; the pass list (3 addresses, the spin's own half word) lives in registers.
// The remaining warps are PRODUCERS: the noise R(spin, word, sweep) does not depend on the state
// (counter-based Philox, a-6), so they compute it a chunk of 32 sweeps ahead into a two-buffer
// ring in shared memory (full / empty named barriers); the consumer's chain never waits for a
// Philox call.  Exact first hits (L293): detection (OR of all clause words, warp reduction) at
// the end of every chunk; if a clone not yet in the table is solved, the chunk is replayed from
// the global copy with a detection after every sweep, using the same noise buffer.
#include <algorithm>

#include <cuda_runtime.h>

#include "xs_device.cuh"
#include "xs_internal.h"

namespace xs {

void count_launch(uint64_t n);   // xs_diag.cu

namespace {

constexpr uint32_t WP_SLOTS = 16;     // spins per pass (x 2 halves = 32 lanes)
constexpr uint32_t WP_PROD = 3;       // producer warps
constexpr uint32_t WP_KB = 32;        // sweeps per noise chunk = detection batch
constexpr uint32_t WP_IDLE = 0xFFFFFFFFu;
constexpr uint32_t WP_SMEM_MAX = 227u * 1024u;
constexpr int LUT_OR_AND = 0xF8;   // a | (b & c)

struct WarpArgs {
    DevPtrs d;
    uint32_t N, W, n_sweeps, thr, flags;
    uint32_t n_pass;          // passes per sweep
    uint32_t ent;             // task-table entries per instance (crec_entries)
    uint32_t off_ring;        // byte offset of the noise ring in dynamic shared memory
};

__device__ __forceinline__ uint32_t wp_lds(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void wp_sts(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void bar_sync(uint32_t id, uint32_t count)
{
    asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(uint32_t id, uint32_t count)
{
    asm volatile("bar.arrive %0, %1;" :: "r"(id), "r"(count) : "memory");
}

// shared memory: [W][N + 16] uint64 clause words (+ one scratch word per slot), then the ring
// [2][WP_KB][n_pass * 16][W] uint32 noise masks
// NP: passes per sweep (exact: the pass loop carries no tests).
template <int NP>
__global__ void __launch_bounds__(32 * (4 + WP_PROD), 1) k_sweep_warp(WarpArgs A)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const uint32_t N = A.N, W = A.W;
    const uint32_t inst = blockIdx.x;
    const xs_tts_rec rec0 = A.d.rec[inst];
    if (rec0.solved && !(A.flags & XS_FLAG_NO_SKIP)) return;   // stop rule (L129, L293)

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t n_ent = A.n_pass * WP_SLOTS;
    const uint32_t n_part = blockDim.x;                          // threads at every named barrier
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t ring = base + A.off_ring;
    const uint32_t buf_bytes = WP_KB * n_ent * W * 4u;
    const CRec* cr = A.d.crec + (size_t)inst * A.ent;
    const uint32_t t0 = (uint32_t)rec0.sweeps_done;
    const uint32_t n_chunks = (A.n_sweeps + WP_KB - 1) / WP_KB;
    // named barriers: 1 + buf = "buffer full", 3 + buf = "buffer empty"

    if (warp >= W) {
        // ---- producers: R(spin, word, sweep) for chunk c into buffer c & 1 --------------------
        const uint64_t seed = A.d.run_seed[inst];
        const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
        const uint32_t ptid = threadIdx.x - 32u * W, n_prod = blockDim.x - 32u * W;
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t buf = c & 1u;
            if (c >= 2) bar_sync(3 + buf, n_part);
            const uint32_t ns = min(WP_KB, A.n_sweeps - c * WP_KB);
            for (uint32_t q = ptid; q < ns * n_ent; q += n_prod) {
                const uint32_t kb = q / n_ent, e = q - kb * n_ent;
                const uint32_t spin = cr[e].spin;
                if (spin == WP_IDLE) continue;
                uint32_t o[4];
                philox4x32_10(spin, 0u, t0 + c * WP_KB + kb + 1u, TAG_SWEEP, k0, k1, o);
                const uint32_t dst = ring + buf * buf_bytes + (kb * n_ent + e) * W * 4u;
#pragma unroll
                for (uint32_t w = 0; w < 4; ++w)
                    if (w < W) wp_sts(dst + 4u * w, o[w] < A.thr ? ~0u : 0u);
            }
            __syncwarp();
            bar_arrive(1 + buf, n_part);
        }
        return;
    }

    // ---- consumer of word column `warp` ----------------------------------------------------------
    const uint32_t w = warp;
    const uint32_t slot = lane >> 1, half = lane & 1u;
    const uint32_t col = base + w * (N + WP_SLOTS) * 8u;      // this column's clause words
    uint64_t* xg = A.d.x + (size_t)inst * N * W + w;
    uint32_t* fhg = A.d.first_hit + ((size_t)inst * W + w) * 64;

    uint32_t ca[NP][3], spin[NP], x[NP];
#pragma unroll
    for (int r = 0; r < NP; ++r) {
        const CRec v = cr[r * WP_SLOTS + slot];
        ca[r][0] = col + v.off0 + 4u * half;
        ca[r][1] = col + v.off1 + 4u * half;
        ca[r][2] = col + v.off2 + 4u * half;
        spin[r] = v.spin;
        x[r] = 0;
    }
    auto load_state = [&]() {
        const ClauseRec* cl = A.d.clause + (size_t)inst * N;
        for (uint32_t t = lane; t < N; t += 32) {
            const ClauseRec c = cl[t];
            const uint64_t v = xg[(size_t)c.i * W] ^ xg[(size_t)c.j * W] ^ xg[(size_t)c.k * W] ^
                               (c.jbit ? ~0ull : 0ull);
            wp_sts(col + 8u * t, (uint32_t)v);
            wp_sts(col + 8u * t + 4u, (uint32_t)(v >> 32));
        }
#pragma unroll
        for (int r = 0; r < NP; ++r)
            if (spin[r] != WP_IDLE)
                x[r] = reinterpret_cast<const uint32_t*>(xg + (size_t)spin[r] * W)[half];
        __syncwarp();
    };
    auto store_state = [&]() {
#pragma unroll
        for (int r = 0; r < NP; ++r)
            if (spin[r] != WP_IDLE)
                reinterpret_cast<uint32_t*>(xg + (size_t)spin[r] * W)[half] = x[r];
    };
    // clones with an unsatisfied interaction: OR of all clause words, same value in every lane
    auto detect = [&]() -> uint64_t {
        uint32_t lo = 0, hi = 0;
        for (uint32_t t = lane; t < N; t += 32) {
            lo |= wp_lds(col + 8u * t);
            hi |= wp_lds(col + 8u * t + 4u);
        }
        lo = __reduce_or_sync(0xFFFFFFFFu, lo);
        hi = __reduce_or_sync(0xFFFFFFFFu, hi);
        return ((uint64_t)hi << 32) | lo;
    };
    uint64_t known = 0;      // clones that already have a first-hit entry
    for (uint32_t b = lane; b < 64; b += 32)
        known |= (uint64_t)__ballot_sync(0xFFFFFFFFu, fhg[b] != XS_NO_HIT) << (b & 32u);
    known = ((uint64_t)__shfl_sync(0xFFFFFFFFu, (uint32_t)(known >> 32), 0) << 32) |
            __shfl_sync(0xFFFFFFFFu, (uint32_t)known, 0);
    load_state();

    // one sweep with the noise of slot `kb` of buffer `nbase`
    auto sweep = [&](uint32_t nrow) {
#pragma unroll
        for (int r = 0; r < NP; ++r) {
            {
                const uint32_t c0 = wp_lds(ca[r][0]), c1 = wp_lds(ca[r][1]), c2 = wp_lds(ca[r][2]);
                const uint32_t R = wp_lds(nrow + ((uint32_t)r * WP_SLOTS + slot) * W * 4u);
                const uint32_t M = lop3<LUT_MAJ>(c0, c1, c2);       // k >= 2
                const uint32_t P = lop3<LUT_XOR3>(c0, c1, c2);      // k odd
                const uint32_t f = lop3<LUT_OR_AND>(M, P, R);       // flip mask (a-7)
                wp_sts(ca[r][0], c0 ^ f);
                wp_sts(ca[r][1], c1 ^ f);
                wp_sts(ca[r][2], c2 ^ f);
                x[r] ^= f;
                __syncwarp();                                        // a-8
            }
        }
    };

    for (uint32_t c = 0; c < n_chunks; ++c) {
        const uint32_t buf = c & 1u;
        const uint32_t ns = min(WP_KB, A.n_sweeps - c * WP_KB);
        const uint32_t nb = ring + buf * buf_bytes + w * 4u;
        const uint32_t tc = t0 + c * WP_KB;
        bar_sync(1 + buf, n_part);
        for (uint32_t kb = 0; kb < ns; ++kb) sweep(nb + kb * n_ent * W * 4u);
        if (~detect() & ~known) {
            // a clone reached E = -N in this chunk: replay it from the global copy (= state at the
            // start of the chunk), looking after every sweep (L293)
            load_state();
            for (uint32_t kb = 0; kb < ns; ++kb) {
                sweep(nb + kb * n_ent * W * 4u);
                const uint64_t newly = ~detect() & ~known;
                known |= newly;
                for (uint32_t b = lane; b < 64; b += 32)
                    if ((newly >> b) & 1ull) fhg[b] = tc + kb + 1u;
            }
        }
        store_state();             // a-10 (also the replay checkpoint of the next chunk)
        if (c + 2 < n_chunks) bar_arrive(3 + buf, n_part);
    }
}

// passes of one sweep on 16 slots: a set of sz spins takes ceil(sz / 16) passes
uint32_t warp_passes(const HostGraph& g)
{
    uint32_t r = 0;
    for (size_t s = 0; s + 1 < g.set_start.size(); ++s)
        r += (g.set_start[s + 1] - g.set_start[s] + WP_SLOTS - 1) / WP_SLOTS;
    return r;
}
inline uint32_t warp_col_bytes(uint32_t N) { return (N + WP_SLOTS) * 8u; }
inline uint32_t warp_smem(uint32_t N, uint32_t W, uint32_t n_pass)
{
    return W * warp_col_bytes(N) + 2u * WP_KB * n_pass * WP_SLOTS * W * 4u;
}

}  // namespace

// Called after choose_geometry / clause_prepare: a batch of few instances with W <= 4 words and the
// quasi-greedy table runs on the latency kernel (variant 3).  Tables: entry pass * 16 + slot ->
// byte offsets of the spin's three clause words inside a column, spin index (idle: own scratch word).
int warp_prepare(xs_batch& b, void* stream)
{
    TileGeom& g = b.geom;
    const xs_geometry& rq = b.req;
    const uint32_t N = b.p.n_spins, I = b.p.n_instances, W = b.p.n_words;
    if (rq.variant != XS_GEOM_AUTO && rq.variant != 3u) return 0;
    if (g.regime != 0 || b.ft.general || b.ft.per_clone || (b.p.flags & XS_FLAG_STREAMING)) return 0;
    if (W > 4u || (rq.tile_words && rq.tile_words != W)) return 0;
    // latency regime only: with more instances than SMs the throughput kernels win
    if (rq.variant == XS_GEOM_AUTO && I > b.num_sms) return 0;
    uint32_t n_pass = 0;
    for (const HostGraph& hg : b.graphs) n_pass = std::max(n_pass, warp_passes(hg));
    if (n_pass == 0 || n_pass > 16u || n_pass * WP_SLOTS > crec_entries(b.p)) return 0;
    if (warp_smem(N, W, n_pass) > WP_SMEM_MAX) return 0;
    if (b.warp_passes != n_pass) {
        const size_t ent = crec_entries(b.p);
        std::vector<CRec> crec((size_t)I * ent, CRec{0u, 0u, 0u, WP_IDLE});
        for (uint32_t i = 0; i < I; ++i) {
            const HostGraph& hg = b.graphs[i];
            CRec* out = crec.data() + (size_t)i * ent;
            for (uint32_t e = 0; e < n_pass * WP_SLOTS; ++e) {
                const uint32_t scratch = (N + e % WP_SLOTS) * 8u;
                out[e] = CRec{scratch, scratch, scratch, WP_IDLE};
            }
            uint32_t pass = 0;
            for (size_t s = 0; s + 1 < hg.set_start.size(); ++s) {
                const uint32_t p0 = hg.set_start[s], sz = hg.set_start[s + 1] - p0;
                for (uint32_t q = 0; q < sz; ++q) {
                    const uint32_t v = hg.order[p0 + q];
                    out[(pass + q / WP_SLOTS) * WP_SLOTS + q % WP_SLOTS] =
                        CRec{hg.cls[3ull * v] * 8u, hg.cls[3ull * v + 1] * 8u, hg.cls[3ull * v + 2] * 8u, v};
                }
                pass += (sz + WP_SLOTS - 1) / WP_SLOTS;
            }
        }
        cudaStream_t st = (cudaStream_t)stream;
        cudaError_t e = cudaMemcpyAsync(b.d.crec, crec.data(), crec.size() * sizeof(CRec),
                                        cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // staging vector dies at return
        if (e != cudaSuccess) return (int)e;
        b.warp_passes = n_pass;
        b.clause_state = 0;        // the clause-word kernel's tables (same buffer) are gone
    }
    g.variant = 3;
    g.T = W;
    g.CW = 1;
    g.threads = 32u * (W + WP_PROD);
    g.ctas = I;
    g.smem = warp_smem(N, W, n_pass);
    g.batch = WP_KB;
    g.rb = WP_KB;
    return 0;
}

int launch_sweep_warp(const xs_batch& b, uint32_t n_sweeps, void* stream)
{
    const TileGeom& g = b.geom;
    WarpArgs A;
    A.d = b.d;
    A.N = b.p.n_spins; A.W = b.p.n_words; A.n_sweeps = n_sweeps;
    A.thr = b.p.w1_threshold; A.flags = b.p.flags;
    A.n_pass = b.warp_passes;
    A.ent = crec_entries(b.p);
    A.off_ring = A.W * warp_col_bytes(A.N);
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaErrorInvalidValue;
#define XS_WP_CASE(NP_)                                                                                        \
    case NP_:                                                                                                  \
        e = cudaFuncSetAttribute(k_sweep_warp<NP_>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem); \
        if (e != cudaSuccess) return (int)e;                                                                   \
        k_sweep_warp<NP_><<<g.ctas, g.threads, g.smem, st>>>(A);                                               \
        break;
    switch (A.n_pass) {
        XS_WP_CASE(1) XS_WP_CASE(2) XS_WP_CASE(3) XS_WP_CASE(4) XS_WP_CASE(5) XS_WP_CASE(6) XS_WP_CASE(7) XS_WP_CASE(8)
        XS_WP_CASE(9) XS_WP_CASE(10) XS_WP_CASE(11) XS_WP_CASE(12) XS_WP_CASE(13) XS_WP_CASE(14) XS_WP_CASE(15)
        XS_WP_CASE(16)
        default: return (int)cudaErrorInvalidValue;
    }
#undef XS_WP_CASE
    e = cudaGetLastError();
    if (e != cudaSuccess) return (int)e;
    count_launch(1);
    return 0;
}

}  // namespace xs
