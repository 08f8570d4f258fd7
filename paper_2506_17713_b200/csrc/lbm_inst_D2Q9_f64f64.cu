// Instantiation unit: lattice D2Q9, compute double, storage double.
#define LBM_INSTANTIATE
#include "lbm_launch.cuh"
namespace lbmk { template cudaError_t launch<D2Q9, double, double>(const LaunchArgs&); }
