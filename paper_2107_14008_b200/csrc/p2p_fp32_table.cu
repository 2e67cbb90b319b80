// Instantiations of the fp32 kernel with g from the paper's shared-memory table, Eq. 2 (PHOTONS_G_TABLE).
#include "p2p_fp32_kernel.cuh"

namespace photons {

int launch_p32_table(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    switch (c->table.level) {
        case 0: return launch_p32_shape<GM_TABLE, 0>(c, a, count, st);
        case 1: return launch_p32_shape<GM_TABLE, 1>(c, a, count, st);
        case 2: return launch_p32_shape<GM_TABLE, 2>(c, a, count, st);
        case 3: return launch_p32_shape<GM_TABLE, 3>(c, a, count, st);
        default: return fail(c, PHOTONS_EINVAL, "table_level %d: the fp32 kernels keep T[0..3]; use FP64 for T[4]", c->table.level);
    }
}

}  // namespace photons
