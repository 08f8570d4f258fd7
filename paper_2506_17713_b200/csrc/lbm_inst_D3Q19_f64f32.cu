// Instantiation unit: lattice D3Q19, compute double, storage float.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D3Q19, double, float>(const LaunchArgs&); }
