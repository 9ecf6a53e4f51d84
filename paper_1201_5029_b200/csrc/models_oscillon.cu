// models_oscillon.cu -- kernel template instances of Oscillon, both precisions (see dispatch.cuh).
#include "dispatch.cuh"

namespace pycool {
PYCOOL_INSTANTIATE_MODEL(Oscillon)
}  // namespace pycool
