// fft_f32.cu — the FFT passes in single precision.
#include "fft_launch.cuh"
namespace galb { GAL_INSTANTIATE_FFT(float) }
