// Instantiation unit: lattice D3Q19, compute float, storage float.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D3Q19, float, float>(const LaunchArgs&); }
