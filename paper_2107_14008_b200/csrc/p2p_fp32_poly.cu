// g from the FMA-pipe polynomial (PHOTONS_G_POLY): dispatch on the degree; one translation unit per degree
// (p2p_fp32_poly10.cu ... p2p_fp32_poly14.cu) so that they compile in parallel.
#include "p2p_fp32_kernel.cuh"

namespace photons {

int launch_p32_poly(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    switch (c->poly_deg) {
        case 10: return launch_p32_poly_deg<10>(c, a, count, st);
        case 11: return launch_p32_poly_deg<11>(c, a, count, st);
        case 12: return launch_p32_poly_deg<12>(c, a, count, st);
        case 13: return launch_p32_poly_deg<13>(c, a, count, st);
        case 14: return launch_p32_poly_deg<14>(c, a, count, st);
        default: return fail(c, PHOTONS_EINVAL, "poly_degree %d has no compiled kernel (10..14)", c->poly_deg);
    }
}

}  // namespace photons
