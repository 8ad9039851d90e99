// redo_f32.cu — the conditional second pass of a speculative call (redo.cuh), single precision.
#include <cstring>
#include "redo.cuh"
namespace galb { GAL_INSTANTIATE_REDO(float) }
