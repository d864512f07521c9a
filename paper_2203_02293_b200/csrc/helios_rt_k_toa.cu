// helios_rt_k_toa.cu -- instantiations of rt_step_kernel: isothermal layers, TOA spectrum only (BASELINE config 5)
// (NONISO, TOA, PPT, ROWS, WARPS, MAXT, MINB), in order of preference; see helios_rt_kernels.cuh.
// 4 points per thread, 1 warp per block; 2 and 1 points per thread when n_gauss is not a multiple of 4 / 2.
#include "helios_rt_kernels.cuh"

namespace hrt_k {
const Variant kVariantsIsoToa[] = {
    HRT_K(false, true, 4, 0, 1, 384, 1),
    HRT_K(false, true, 4, 0, 0, 384, 1),
    HRT_K(false, true, 2, 0, 0, 512, 1),
    HRT_K(false, true, 1, 0, 0, 640, 1),
};
const int kNumIsoToa = (int)(sizeof(kVariantsIsoToa) / sizeof(kVariantsIsoToa[0]));
}  // namespace hrt_k
