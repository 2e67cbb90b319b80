// Host side of the fp32 / mixed P2P kernels: argument block, shared-memory sizing, g-mode dispatch.
#include <cmath>

#include "p2p_fp32_kernel.cuh"

namespace photons {

size_t p32_smem_bytes(Ctx* c, int T)
{
    const int W = c->p.warps_per_leaf;
    const bool mixed = c->p.precision == PHOTONS_MIXED;
    size_t b = (size_t)W * N_STAGES * c->p.chunk_max * 16 + (size_t)W * T * 32 * 3 * 8;
    b += mixed ? (size_t)((W * N_STAGES * 8 + 15) & ~15) + (size_t)W * N_STAGES * MAX_RUN_LEAVES * 16 : (size_t)W * N_STAGES * 8;
    if (c->p.g_mode == PHOTONS_G_TABLE) b += (size_t)(c->table.n + 1) * 8;
    return b;
}

void fill_p32_args(Ctx* c, P32Args& a, long long first, void* out, bool out_f32)
{
    a.p32 = c->d_p32; a.p64 = c->d_p64; a.ctr = c->d_leaf_ctr; a.slot_src = c->d_slot_src;
    a.chunk_ptr = c->d_chunk_ptr; a.chunks = c->d_chunks; a.order = c->d_order; a.first = first;
    a.maxleaf = c->p.maxleaf; a.log2m = 0;
    while ((1 << a.log2m) < a.maxleaf) ++a.log2m;
    a.chunk_max = c->p.chunk_max; a.mixed = c->p.precision == PHOTONS_MIXED;
    // kernel units: lengths / pscale, G m / gmscale (common.cuh); everything the pair core touches is O(1)
    const double ips = 1.0 / c->pscale;
    const double Ls = c->p.boxsize * ips, rs = c->r_s * ips, rcut = c->r_cut * ips;
    a.inv_pscale = ips;
    a.oscale = c->gmscale * ips * ips;
    a.inv_oscale = 1.0 / a.oscale;
    a.Lh = (float)Ls; a.Ll = (float)(Ls - (double)a.Lh); a.invL = (float)(1.0 / Ls);
    a.rcut2 = (float)(rcut * rcut);
    const double eps = c->p.softening * ips;
    a.r2add = std::fmax(R2_FLOOR, (float)(eps * eps));
    a.eps2_d = c->p.softening * c->p.softening;
    a.Ld = c->p.boxsize; a.inv2rs_d = 1.0 / (2.0 * c->r_s); a.rcut2_d = c->r_cut * c->r_cut;
    // exact path trigger: |fp32 partial of a run| > max|G m| / r_close^2 (one pair at r_close), in kernel units
    a.pth2 = 0.f;
    if (c->p.close_pair_radius > 0) {
        const double rc = c->p.close_pair_radius * ips;
        const double pth = (c->gm_max / c->gmscale) / (rc * rc);
        a.pth2 = (float)std::fmin(pth * pth, 1e37);
    }
    a.gmu = 1.0;
    if (c->ugm) {      // the runs' fp32 partial sums lack the common factor G m: it is applied when they are flushed
        a.gmu = c->gm_uniform / c->gmscale;
        a.pth2 = (float)std::fmin((double)a.pth2 / (a.gmu * a.gmu), 1e37);
    }
    a.inv2rs = (float)(1.0 / (2.0 * rs));
    const double smax = 0.25 * c->p.rcut_over_rs * c->p.rcut_over_rs;
    a.tk = (float)(2.0 / (smax * 4.0 * rs * rs));
    for (int i = 0; i <= POLY_MAX_DEG; ++i) a.pc[i] = c->p.g_mode == PHOTONS_G_FUSED ? c->fused_c[i] : c->poly_c[i];
    a.ek = (float)(-1.4426950408889634 / (4.0 * rs * rs));          // exp(-x^2) = 2^(-x^2 log2 e), x^2 = r^2 / 4 r_s^2
    a.tmap = (float)(2.0 / (0.5 * c->p.rcut_over_rs) / (2.0 * rs));   // t = 2 x / x_cut - 1 with x = r / 2 r_s folded in
    a.tn = c->table.n;
    a.h = a.tn ? (float)(3.0 / a.tn) : 0.f;
    a.uk = a.tn ? (float)(a.tn / 3.0 / (2.0 * rs)) : 0.f;
    a.rmax = (float)(3.0 * 2.0 * rs);       // x = 3 = the last node
    a.table = c->table.d_TE;
    a.out = out; a.out_f32 = out_f32 ? 1 : 0;
}

int launch_p2p_fp32(Ctx* c, long long first, long long count, void* out, bool out_f32, cudaStream_t st)
{
    P32Args a{};
    fill_p32_args(c, a, first, out, out_f32);
    switch (c->p.g_mode) {
        case PHOTONS_G_POLY: return launch_p32_poly(c, a, count, st);
        case PHOTONS_G_TABLE: return launch_p32_table(c, a, count, st);
        case PHOTONS_G_FUSED: return launch_p32_fused(c, a, count, st);
        default: return launch_p32_direct(c, a, count, st);
    }
}

}  // namespace photons
