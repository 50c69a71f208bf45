// rgrmhd_rhs_tiled.cu -- placeholder until the tiled kernel lands (the simple kernel is used).
#include "rgrmhd_rhs.cuh"
namespace rg {
bool rhs_tiled_supported(const GridView&) { return false; }
cudaError_t launch_rhs_tiled(const GridView&, double, int, int, cudaStream_t) { return cudaErrorNotSupported; }
}
