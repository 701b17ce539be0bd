// tuned.cu -- dispatch table of the per-class tuned kernels (filled in by the reg_*.cu / coop_*.cu units).
#include "launch.h"

namespace eri {

bool tuned_jk_info(int, int, int, int, int, int, TunedInfo*) { return false; }
cudaError_t launch_tuned_jk(const Work&, int, cudaStream_t) { return cudaErrorNotSupported; }
bool tuned_grad_info(int, int, int, int, int, int, TunedInfo*) { return false; }
cudaError_t launch_tuned_grad(const Work&, int, cudaStream_t) { return cudaErrorNotSupported; }

}  // namespace eri
