// mf_fused.cu — fused path (MF_PATH_FUSED): one kernel per RK stage.  Placeholder until the staged path is parity-green.
#include "mf_kernels.h"

namespace mf {

bool fused_supported(const Grid&) { return false; }

int launch_fused_stage(const Grid&, const Eos&, int, int, int, CState5, Stage, CState5, CState5, State5, Source, const StepState*, int, cudaStream_t)
{
    return 0;
}

} // namespace mf
