// fft_f64.cu — the FFT passes in double precision.
#include "fft_launch.cuh"
namespace galb { GAL_INSTANTIATE_FFT(double) }
