// models_chaotic.cu -- kernel template instances of Chaotic, both precisions (see dispatch.cuh).
#include "dispatch.cuh"

namespace pycool {
PYCOOL_INSTANTIATE_MODEL(Chaotic)
}  // namespace pycool
