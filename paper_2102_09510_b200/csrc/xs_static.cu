// xs_static.cu -- xs_solved_mask_static: an entry point that allocates nothing and needs no
// scratch from the caller.  For callers that cannot call cudaMalloc (CUDA graph capture, tight
// serving loops, harnesses that forbid it) and want to ask "which clones are in a ground state
// right now?" (E = -N <=> every interaction satisfied; L71: the check done between
// batches of sweeps) without xs_energy's [inst][64 W] int32 output.
//
// It is a variant of the ground-state detection kernel k_unsat_or (xs_kernels.cu), whose scratch
// -- det[inst][w] = OR over clauses of (x_i ^ x_j ^ x_k ^ Jmask), bit set <=> the clone has an
// unsatisfied interaction -- normally lives in the caller's workspace.  Here the scratch is the
// file-scope array g_det_scratch below: XS_STATIC_MAX_WORDS uint64 words = 512 KiB that EVERY GPU
// which loads the library holds until the process exits.  All calls share it and it keeps the
// last call's contents: each call clears the part it uses first, and two calls that overlap on
// the GPU (different streams, no dependency) race on it.  No existing code path is changed.
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>
#include <string>

#include "xs_internal.h"

namespace xs {

void count_launch(uint64_t n);   // xs_diag.cu

namespace {

// the scratch: one uint64 per (instance, word); modest, fixed maximum
static __device__ __align__(256) unsigned long long g_det_scratch[XS_STATIC_MAX_WORDS];

// In host code `g_det_scratch` is only a host-side stand-in for the symbol, not a device address:
// the address a kernel may use comes from cudaGetSymbolAddress, asked once per device with that
// device current.
constexpr int MAX_DEVICES = 64;
unsigned long long* g_scratch_ptr[MAX_DEVICES] = {};
std::mutex g_scratch_mutex;

cudaError_t scratch_for_current_device(int dev, unsigned long long** out)
{
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_det_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_ptr[dev] = static_cast<unsigned long long*>(p);
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

constexpr uint32_t SM_CHUNK = 32;      // clauses per CTA
constexpr uint32_t SM_THREADS = 128;

// det[inst][w] |= OR over the CTA's clauses of the unsatisfied-clause word (as k_unsat_or).
// grid = (clause chunks, I, word blocks)
__global__ void __launch_bounds__(SM_THREADS) k_unsat_or_static(DevPtrs d, uint32_t N, uint32_t W,
                                                                unsigned long long* det)
{
    const uint32_t inst = blockIdx.y;
    const uint32_t c0 = blockIdx.x * SM_CHUNK;
    const uint32_t c1 = min(c0 + SM_CHUNK, N);
    const ClauseRec* cl = d.clause + (size_t)inst * N;
    const uint64_t* x = d.x + (size_t)inst * N * W;
    for (uint32_t w = blockIdx.z * blockDim.x + threadIdx.x; w < W; w += gridDim.z * blockDim.x) {
        unsigned long long acc = 0;
        for (uint32_t c = c0; c < c1; ++c) {
            const ClauseRec r = cl[c];
            acc |= x[(size_t)r.i * W + w] ^ x[(size_t)r.j * W + w] ^ x[(size_t)r.k * W + w] ^
                   (r.jbit ? ~0ull : 0ull);
        }
        if (acc) atomicOr(det + (size_t)inst * W + w, acc);
    }
}

// mask[e] = ~det[e]: bit set <=> the clone has no unsatisfied interaction <=> E = -N
__global__ void k_mask_out(const unsigned long long* det, uint64_t* mask, uint32_t total)
{
    for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < total; e += gridDim.x * blockDim.x)
        mask[e] = ~det[e];
}

}  // namespace
}  // namespace xs

extern "C" int xs_solved_mask_static(xs_batch* b, uint64_t* dev_mask, void* cuda_stream)
{
    using namespace xs;
    if (!b || !dev_mask) return xs::xs_set_error(XS_EINVAL, "null argument");
    const uint64_t words = (uint64_t)b->p.n_instances * b->p.n_words;
    if (words > XS_STATIC_MAX_WORDS)
        return xs::xs_set_error(XS_EINVAL, "xs_solved_mask_static: n_instances * n_words = " + std::to_string(words) +
                                           " exceeds the static scratch of XS_STATIC_MAX_WORDS = " +
                                           std::to_string((unsigned)XS_STATIC_MAX_WORDS) + " words");
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev)) return xs::xs_set_error(XS_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev != b->device || dev < 0 || dev >= MAX_DEVICES)
        return xs::xs_set_error(XS_ESTATE, "xs_solved_mask_static: the batch's device must be current (and below 64)");
    unsigned long long* det = nullptr;
    if (cudaError_t e = scratch_for_current_device(dev, &det))
        return xs::xs_set_error(XS_ECUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t N = b->p.n_spins, W = b->p.n_words, I = b->p.n_instances;
    // the array keeps the last call's contents: clear what this call accumulates into
    if (cudaError_t e = cudaMemsetAsync(det, 0, words * 8, st))
        return xs::xs_set_error(XS_ECUDA, std::string("scratch clear: ") + cudaGetErrorString(e));
    dim3 grid((N + SM_CHUNK - 1) / SM_CHUNK, I, std::min<uint32_t>(64u, (W + SM_THREADS - 1) / SM_THREADS));
    k_unsat_or_static<<<grid, SM_THREADS, 0, st>>>(b->d, N, W, det);
    k_mask_out<<<(uint32_t)std::min<uint64_t>((words + 255) / 256, 1184), 256, 0, st>>>(det, dev_mask, (uint32_t)words);
    count_launch(2);
    if (cudaError_t e = cudaGetLastError())
        return xs::xs_set_error(XS_ECUDA, std::string("xs_solved_mask_static launch: ") + cudaGetErrorString(e));
    return XS_OK;
}
