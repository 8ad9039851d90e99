// sample_f32.cu — the per-point kernels on single-precision arrays.
#include "sample_launch.cuh"
namespace galb { GAL_INSTANTIATE_SAMPLE(float) }
