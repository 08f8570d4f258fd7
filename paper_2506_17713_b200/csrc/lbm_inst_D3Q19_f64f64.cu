// Instantiation unit: lattice D3Q19, compute double, storage double.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D3Q19, double, double>(const LaunchArgs&); }
