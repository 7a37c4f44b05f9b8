// xs_diag.cu -- measurement helpers behind the C ABI (no arithmetic of the method).
//   xs_alu_peak        : measured LOP3 issue rate of the whole GPU (the integer-pipe roofline
//                        denominator of DESIGN.md "Roofline"; SURVEY.md 8(d) asks for it to be
//                        measured, MEASURED_PEAKS.json has no integer figure)
//   xs_kernel_launches : number of kernels this library has launched in this process
#include <cuda_runtime.h>

#include <atomic>

#include "xs_internal.h"

namespace xs {
std::atomic<uint64_t> g_launches{0};
void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

// 16 independent LOP3 chains per thread, ITER x 16 x UNROLL instructions, nothing else in the
// loop but the counter.  LUT 0x96 (xor3) on register operands.
constexpr int PEAK_CHAINS = 16;
constexpr int PEAK_UNROLL = 8;

__global__ void __launch_bounds__(1024) k_alu_peak(uint32_t iters, uint32_t seed, uint32_t* sink)
{
    uint32_t a[PEAK_CHAINS];
    const uint32_t b = seed * 2654435761u + threadIdx.x, c = seed ^ (blockIdx.x * 40503u);
#pragma unroll
    for (int q = 0; q < PEAK_CHAINS; ++q) a[q] = threadIdx.x * 0x9E3779B9u + q;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
            for (int q = 0; q < PEAK_CHAINS; ++q)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[q]) : "r"(b), "r"(c));
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int q = 0; q < PEAK_CHAINS; ++q) r ^= a[q];
    if (r == 0x12345678u) *sink = r;   // practically never; keeps the chains alive
}
}  // namespace xs

extern "C" {

uint64_t xs_kernel_launches(void) { return xs::g_launches.load(std::memory_order_relaxed); }

int xs_alu_peak(double* lane_ops_per_ns, double* kernel_ms, void* cuda_stream)
{
    if (!lane_ops_per_ns) return XS_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return XS_ECUDA;
    uint32_t* sink = nullptr;
    if (cudaMalloc(&sink, 4) != cudaSuccess) return XS_ECUDA;   // diagnostic only, not the product path
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const uint32_t iters = 4096;
    const int grid = sms * 2, threads = 1024;
    double best_ms = 1e30;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        xs::k_alu_peak<<<grid, threads, 0, st>>>(iters, 17u + rep, sink);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return XS_ECUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    xs::count_launch(4);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    const double ops = (double)grid * threads * iters * xs::PEAK_CHAINS * xs::PEAK_UNROLL;
    *lane_ops_per_ns = ops / (best_ms * 1e6);
    if (kernel_ms) *kernel_ms = best_ms;
    return XS_OK;
}

}  // extern "C"
