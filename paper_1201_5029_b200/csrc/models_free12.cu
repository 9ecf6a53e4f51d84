// models_free12.cu -- kernel template instances of Free<1>, Free<2>, both precisions (see dispatch.cuh).
#include "dispatch.cuh"

namespace pycool {
PYCOOL_INSTANTIATE_MODEL(Free<1>)
PYCOOL_INSTANTIATE_MODEL(Free<2>)
}  // namespace pycool
