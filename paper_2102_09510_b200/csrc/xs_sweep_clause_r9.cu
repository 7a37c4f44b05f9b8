// Instantiation unit of the clause-word sweep kernel (xs_sweep_clause.cuh): 9 rounds per sweep.
#include "xs_sweep_clause.cuh"

namespace xs {
template cudaError_t launch_clause_unit_long<9>(const ClauseArgs&, const ClauseLaunch&);
}
