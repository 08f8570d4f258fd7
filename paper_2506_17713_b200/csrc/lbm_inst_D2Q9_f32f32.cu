// Instantiation unit: lattice D2Q9, compute float, storage float.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D2Q9, float, float>(const LaunchArgs&); }
