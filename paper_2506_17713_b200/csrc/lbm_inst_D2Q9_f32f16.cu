// Instantiation unit: lattice D2Q9, compute float, storage __half.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D2Q9, float, __half>(const LaunchArgs&); }
