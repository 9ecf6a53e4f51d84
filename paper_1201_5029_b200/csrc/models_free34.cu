// models_free34.cu -- kernel template instances of Free<3>, Free<4>, both precisions (see dispatch.cuh).
#include "dispatch.cuh"

namespace pycool {
PYCOOL_INSTANTIATE_MODEL(Free<3>)
PYCOOL_INSTANTIATE_MODEL(Free<4>)
}  // namespace pycool
