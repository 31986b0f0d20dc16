// mlp_tc.cu -- tcgen05 / TMEM tensor-core MLP (GMNN_MLP_3XTF32, GMNN_MLP_TF32).  Placeholder
// until the kernel lands: selecting these precisions fails loudly, it never falls back.
#include "gmnn_internal.h"

namespace gmnn {

int launch_mlp_forward_tc(gmnn_system *, cudaStream_t) {
    set_error("tensor-core MLP (mlp_precision 1, 2) is not built yet");
    return GMNN_UNSUPPORTED;
}
int launch_mlp_backward_tc(gmnn_system *, const float *, cudaStream_t) {
    set_error("tensor-core MLP (mlp_precision 1, 2) is not built yet");
    return GMNN_UNSUPPORTED;
}

}  // namespace gmnn
