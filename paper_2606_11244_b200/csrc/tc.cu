// tc.cu -- placeholder until the tcgen05 kernel lands (next commit).
#include "common.cuh"
#include "kernels.h"
namespace spear {
bool tc_available() { return false; }
int run_tc(const TcProblem&, cudaStream_t) { return set_error(SPEAR_EUNSUPPORTED, "tcgen05 path not built"); }
}  // namespace spear
