// helios_rt_k_noniso.cu -- instantiations of rt_step_kernel: non-isothermal layers (BASELINE configs 3, 4)
// (NONISO, TOA, PPT, ROWS, WARPS, MAXT, MINB), in order of preference; see helios_rt_kernels.cuh.
// full outputs: 2 points per thread at 168 registers, 2 warps per block (config 3: 1.453 ms against 1.478 at 1 point per thread, 128 registers, 4 warps); TOA: 1 point per thread; ROWS 1 is a comparison build.
#include "helios_rt_kernels.cuh"

namespace hrt_k {
const Variant kVariantsNoniso[] = {
    HRT_K(true, false, 2, 0, 0, 384, 1),
    HRT_K(true, false, 1, 0, 4, 512, 1),
    HRT_K(true, false, 1, 0, 0, 512, 1),
    HRT_K(true, false, 1, 1, 0, 512, 1),
    HRT_K(true, true, 1, 0, 0, 512, 1),
};
const int kNumNoniso = (int)(sizeof(kVariantsNoniso) / sizeof(kVariantsNoniso[0]));
}  // namespace hrt_k
