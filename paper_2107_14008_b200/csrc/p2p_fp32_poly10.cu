// Instantiations of the fp32 kernel with the degree-10 polynomial g (PHOTONS_G_POLY).
#include "p2p_fp32_kernel.cuh"

namespace photons {

template <>
int launch_p32_poly_deg<10>(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    return launch_p32_shape<GM_POLY, 10>(c, a, count, st);
}

}  // namespace photons
