// Instantiation unit: lattice D2Q9, compute double, storage float.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D2Q9, double, float>(const LaunchArgs&); }
