// Instantiation unit of the clause-word sweep kernel (xs_sweep_clause.cuh): 16 rounds per sweep.
#include "xs_sweep_clause.cuh"

namespace xs {
template cudaError_t launch_clause_unit_long<16>(const ClauseArgs&, const ClauseLaunch&);
}
