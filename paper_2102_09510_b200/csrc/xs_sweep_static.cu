// xs_sweep_static.cu -- host side of the static-task sweep kernel (xs_sweep_static.cuh): shared
// memory size, rounds per sweep, feasibility, and the dispatch to the instantiation units
// xs_sweep_static_i<CW><NC>.cu.
#include <algorithm>
#include <cstdlib>

#include "xs_sweep_static.cuh"

namespace xs {

void count_launch(uint64_t n);

extern template cudaError_t launch_static_unit<1, 1>(const StaticArgs&, const StaticLaunch&);
extern template cudaError_t launch_static_unit<1, 2>(const StaticArgs&, const StaticLaunch&);
extern template cudaError_t launch_static_unit<1, 4>(const StaticArgs&, const StaticLaunch&);
extern template cudaError_t launch_static_unit<2, 1>(const StaticArgs&, const StaticLaunch&);
extern template cudaError_t launch_static_unit<2, 2>(const StaticArgs&, const StaticLaunch&);
extern template cudaError_t launch_static_unit<2, 4>(const StaticArgs&, const StaticLaunch&);

constexpr int STATIC_MAXT = 8;
constexpr uint32_t STATIC_SMEM_MAX = 227u * 1024u;

static uint32_t static_line_shift(uint32_t T)
{
    uint32_t bytes = (T <= 16) ? 128u : T * 8u, sh = 0;   // T = 4, 8: 4 / 2 copies in one line
    while ((1u << sh) < bytes) ++sh;
    return sh;
}

uint32_t static_smem_bytes(uint32_t N, uint32_t T)
{
    const uint64_t state = ((uint64_t)N + 1) << static_line_shift(T);   // + scratch line
    const uint64_t total = state + (4ull * T + 4) * 4 + 128;
    return total > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)total;
}

// rounds a CTA of `threads` threads needs per sweep for tile width T (max over instances)
uint32_t static_rounds(const xs_batch& b, uint32_t T, uint32_t CW, uint32_t threads)
{
    const uint32_t n_slots = threads / (T / CW);
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

bool static_feasible(const xs_batch& b, uint32_t T, uint32_t CW, uint32_t threads)
{
    if (T < 4 || T > 64 || (T & (T - 1)) || b.p.n_words % T) return false;
    if (CW != 1 && CW != 2) return false;
    const uint32_t LPS = T / CW;
    if (LPS > 32) return false;
    if (threads % 32 || threads < 32 || threads > 512 || threads % LPS) return false;
    if (static_smem_bytes(b.p.n_spins, T) > STATIC_SMEM_MAX) return false;
    return static_rounds(b, T, CW, threads) <= (uint32_t)STATIC_MAXT;
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
    A.off_misc = (uint32_t)((((uint64_t)p.n_spins + 1) << A.line_shift) + 127) / 128 * 128;
    const uint32_t nc = g.T <= 16 ? 16u / g.T : 1u;     // row copies per 128-byte line
    StaticLaunch L;
    L.rounds = static_rounds(b, g.T, g.CW, g.threads);
    L.threads = g.threads; L.ctas = g.ctas; L.smem = g.smem;
    L.dense = g.ctas > b.num_sms;
    // FULL: exactly `rounds` sets, one round each, and the last warp of the CTA has a task in each
    {
        const uint32_t n_slots = g.threads / (g.T / g.CW), slots_per_warp = 32u / (g.T / g.CW);
        const uint32_t warps = g.threads / 32u;
        L.full = slots_per_warp > 0;
        for (const HostGraph& hg : b.graphs) {
            if (hg.set_start.size() != (size_t)L.rounds + 1) { L.full = false; break; }
            for (size_t s = 0; s + 1 < hg.set_start.size(); ++s) {
                const uint32_t sz = hg.set_start[s + 1] - hg.set_start[s];
                if (sz > n_slots || sz <= (warps - 1) * slots_per_warp) L.full = false;
            }
        }
    }
    L.st = (cudaStream_t)stream;
    cudaError_t e;
    if (g.CW == 2)
        e = nc == 4 ? launch_static_unit<2, 4>(A, L) : nc == 2 ? launch_static_unit<2, 2>(A, L)
                                                               : launch_static_unit<2, 1>(A, L);
    else
        e = nc == 4 ? launch_static_unit<1, 4>(A, L) : nc == 2 ? launch_static_unit<1, 2>(A, L)
                                                               : launch_static_unit<1, 1>(A, L);
    if (e != cudaSuccess) return (int)e;
    count_launch(1);
    return 0;
}

}  // namespace xs
