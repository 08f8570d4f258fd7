// Instantiation unit: lattice D3Q19, compute float, storage __half.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D3Q19, float, __half>(const LaunchArgs&); }
