// helios_rt_k_sampling.cu -- instantiations of rt_step_kernel: one Gauss point per bin (opacity sampling, config 6)
// (NONISO, TOA, PPT, ROWS, WARPS, MAXT, MINB) / (NONISO, TOA, ROWS, WARPS, MAXT, MINB), in order of preference; see helios_rt_kernels.cuh.
// Planck values read from the workspace (BDIRECT); 1 point per thread.
#include "helios_rt_kernels.cuh"

namespace hrt_k {
const Variant kVariantsSampling[] = {
    HRT_KB(false, false, 0, 0, 640, 1),
    HRT_KB(false, true, 0, 0, 640, 1),
    HRT_KB(true, false, 0, 0, 512, 1),
    HRT_KB(true, true, 0, 0, 512, 1),
};
const int kNumSampling = (int)(sizeof(kVariantsSampling) / sizeof(kVariantsSampling[0]));
}  // namespace hrt_k
