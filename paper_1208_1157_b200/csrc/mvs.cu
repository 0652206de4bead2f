// mvs.cu — placeholder until the MVS kernel lands (next commit): ens_integrate(ENS_MVS) returns ENS_EUNSUPPORTED.
#include "ens_internal.cuh"
namespace ensd {
KernelInfo mvs_kernel_for(int) { KernelInfo k; k.fn = nullptr; k.shape.L = k.shape.B = 0; k.threads = 0; return k; }
cudaError_t launch_mvs(const View&, const StepArgs&, int, cudaStream_t, int64_t*) { return cudaErrorNotSupported; }
}
