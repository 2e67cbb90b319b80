// Instantiations of the fp32 kernel with g from erfcf/expf (PHOTONS_G_DIRECT).
#include "p2p_fp32_kernel.cuh"

namespace photons {

int launch_p32_direct(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    return launch_p32_shape<GM_DIRECT, 0>(c, a, count, st);
}

}  // namespace photons
