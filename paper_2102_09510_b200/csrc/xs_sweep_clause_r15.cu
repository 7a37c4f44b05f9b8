// Instantiation unit of the clause-word sweep kernel (xs_sweep_clause.cuh): 15 rounds per sweep.
#include "xs_sweep_clause.cuh"

namespace xs {
template cudaError_t launch_clause_unit_long<15>(const ClauseArgs&, const ClauseLaunch&);
}
