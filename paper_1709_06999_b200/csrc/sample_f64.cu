// sample_f64.cu — the per-point kernels in double precision.
#include "sample_launch.cuh"
namespace galb { GAL_INSTANTIATE_SAMPLE(double) }
