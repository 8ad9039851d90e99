// redo_f64.cu — the conditional second pass of a speculative call (redo.cuh), double precision.
#include <cstring>
#include "redo.cuh"
namespace galb { GAL_INSTANTIATE_REDO(double) }
