// helios_rt_k_iso.cu -- instantiations of rt_step_kernel: isothermal layers, full outputs (BASELINE config 2, the headline)
// (NONISO, TOA, PPT, ROWS, WARPS, MAXT, MINB), in order of preference; see helios_rt_kernels.cuh.
// 2 points per thread, runtime block size (2 warps); ROWS 1 (k-table rows through the TMA ring) is a comparison build.
#include "helios_rt_kernels.cuh"

namespace hrt_k {
const Variant kVariantsIsoFull[] = {
    HRT_K(false, false, 2, 0, 0, 512, 1),
    HRT_K(false, false, 2, 1, 0, 512, 1),
    HRT_K(false, false, 1, 0, 0, 768, 1),
};
const int kNumIsoFull = (int)(sizeof(kVariantsIsoFull) / sizeof(kVariantsIsoFull[0]));
}  // namespace hrt_k
