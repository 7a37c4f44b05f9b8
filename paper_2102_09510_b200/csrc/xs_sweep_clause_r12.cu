// Instantiation unit of the clause-word sweep kernel (xs_sweep_clause.cuh): 12 rounds per sweep.
#include "xs_sweep_clause.cuh"

namespace xs {
template cudaError_t launch_clause_unit_long<12>(const ClauseArgs&, const ClauseLaunch&);
}
