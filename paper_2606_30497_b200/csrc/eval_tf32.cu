// eval_tf32.cu -- tensor-core (tcgen05, TF32) variant of the eval pass (SURVEY.md 8(a) row a-T).
// Placeholder translation unit: the variant is reported as unsupported until the kernel lands.
#include "common.cuh"
#include "internal.h"

namespace mlp {

bool eval_tf32_supported(int hidden) {
    (void)hidden;
    return false;
}

cudaError_t launch_eval_tf32(const float*, const float*, int64_t, const float*, const float*, int,
                             double*, int, double*, cudaStream_t, int64_t*) {
    return cudaErrorNotSupported;
}

}  // namespace mlp
