// models_qball.cu -- kernel template instances of QBall, both precisions (see dispatch.cuh).
#include "dispatch.cuh"

namespace pycool {
PYCOOL_INSTANTIATE_MODEL(QBall)
}  // namespace pycool
