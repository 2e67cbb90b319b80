// Instantiations of the fp32 kernel with Eq. 1 evaluated directly by the hand-fused routine (PHOTONS_G_FUSED).
#include "p2p_fp32_kernel.cuh"

namespace photons {

int launch_p32_fused(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    switch (c->fused_deg) {
        case 9: return launch_p32_shape<GM_FUSED, 9>(c, a, count, st);
        case 10: return launch_p32_shape<GM_FUSED, 10>(c, a, count, st);
        case 11: return launch_p32_shape<GM_FUSED, 11>(c, a, count, st);
        default: return fail(c, PHOTONS_EINVAL, "fused g: degree %d has no compiled kernel (9..11)", c->fused_deg);
    }
}

}  // namespace photons
