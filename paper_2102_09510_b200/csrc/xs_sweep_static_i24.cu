// Instantiation unit of the static-task sweep kernel: CW = 2 uint64 words per lane, NC = 4 row
// copies per 128-byte line (one unit per family so that the families compile in parallel).
#include "xs_sweep_static.cuh"

namespace xs {
template cudaError_t launch_static_unit<2, 4>(const StaticArgs&, const StaticLaunch&);
}  // namespace xs
