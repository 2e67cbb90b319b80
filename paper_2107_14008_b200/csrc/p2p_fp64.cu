// fp64 P2P kernel (Alg. 1 + Alg. 2, the paper's DP run L196): one CTA per target leaf, the CTA's
// warps split the leaf's source list, lanes own targets, source runs arrive in shared memory by TMA bulk
// copies through a per-warp mbarrier ring (pipeline.cuh).  SURVEY.md §8(a) steps a4-a9.
//
// The pair core is bound by the FP64 pipe (64 lanes per SM: a warp-wide DFMA/DADD/DMUL/DSETP holds a scheduler's
// DP unit for two cycles), so the design rule is: as few DP-pipe instructions per pair as the tolerance allows.
//   - branch-free: self / coincident pairs are neutralised by a tiny start value of the r^2 chain (w * 0 = 0 with a
//     finite w), the cut is one DSETP + a select on the weight;
//   - 1/r from MUFU.RSQ64H (XU pipe, ~20 bits) and ONE third-order correction step (5 DP ops, error ~ e^3 = 2^-60)
//     instead of the library's rsqrt (two Newton steps plus special-case code, ~12 DP ops);
//   - U independent source chains per lane so that the dependent DFMA chains of one pair overlap with the others';
//   - the interpolation table lives in shared memory, in one of two layouts:
//       paper layout  {T_i, E_i}, Eq. 2's polynomials in x_i rebuilt per pair (L129-L151: 14 flops in the paper's count);
//       coefficient layout  c_k = T^(k)(x_i) h^k / k!, k = 0..level, per node: the same Taylor series about the same
//         node with the node polynomials folded in when the table is built (Horner only: `level` DFMAs).  The paper
//         tabulates two numbers per node "considering the suitable capacity of shared memory" (L143, 96 KB on V100);
//         with 227 KB per SM on B200 the 5-column table of 512 nodes (20 KB) is the cheaper trade.
//   - index by the magic-number add in fp64 (the low word of u + 1.5 * 2^52 is the nearest integer): no F2I/I2F;
//     u itself is never formed: fma(r, uk, MAGIC) and eps = fma(r, 1/2r_s, -x_i);
//   - the cut compare on the integer pipe (bit patterns of positive doubles are ordered).
#include "common.cuh"
#include "pipeline.cuh"

namespace photons {

constexpr double R2_FLOOR64 = 0x1p-600;   // start of every r^2 chain: 1/r^3 = 2^900 stays finite, w * 0 = 0 (A7)
constexpr double MAGIC64 = 6755399441055744.0;   // 1.5 * 2^52
// ring depth of the fp64 kernels: a stage is 4 KB per warp, and with 2 stages a fourth CTA fits per SM (measured:
// table 512/T[4] 262.8 -> 252.8 ms on config 4)
constexpr int N_STAGES64 = 2;
constexpr int TAB_STRIDE = 5;             // doubles per node in the coefficient layout (odd: fewer bank conflicts)

enum { G64_DIRECT = 0, G64_TABLE = 1, G64_COEF = 2, G64_QUAD = 3 };

struct P64Args {
    const double4* p64;       // n_slots x {x, y, z, G m}
    const int* slot_src;      // slot -> caller index (-1 = padding)
    const long long* chunk_ptr;
    const uint2* chunks;
    const int* order;         // CTA b works on leaf order[first + b]
    long long first;
    int maxleaf, chunk_max;
    double L, rcut2, inv2rs, r2add;
    const double* table;      // TABLE: {T_i, E_i} pairs; COEF: TAB_STRIDE doubles per node; i = 0..tn
    int tn, tab_doubles;      // number of doubles to stage in shared memory
    double uk, h;             // u = r * uk in node units; h = 3 / tn
    void* out;                // caller order, n x 3
    int out_f32;
};

// Eq. 1 by the special functions, x = r / 2 r_s
__device__ __forceinline__ double g_direct64(double x)
{
    return erfc(x) + 1.1283791670955125739 * x * exp(-x * x);
}

// 1/sqrt(x) for normal positive x: MUFU.RSQ64H seed on the high word, then y (1 + e/2 + 3 e^2/8), e = 1 - x y^2
__device__ __forceinline__ double rsqrt64(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double hx = x * y;
    const double e = fma(-hx, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(y, e * p, y);
}

// g(x) for NCH chains at once; r = r2 * idr is passed in
template <int GMODE, int LEVEL, int NCH>
__device__ __forceinline__ void g_eval(const P64Args& a, const double* __restrict__ tab, const double (&r)[NCH],
                                       const bool (&incut)[NCH], double (&g)[NCH])
{
    if constexpr (GMODE == G64_DIRECT) {
        // the library's erfc + exp cost ~90 DP instructions: skip them for sources no lane of the warp has inside the cut
#pragma unroll
        for (int c = 0; c < NCH; ++c) g[c] = __any_sync(0xffffffffu, incut[c]) ? g_direct64(r[c] * a.inv2rs) : 0.0;
    } else {
    double fi[NCH];
    int idx[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
        const double um = fma(r[c], a.uk, MAGIC64);    // u = r uk in node units; + 1.5 * 2^52 rounds to the nearest node (A14)
        fi[c] = um - MAGIC64;
        idx[c] = min(__double2loint(um), a.tn);        // beyond the table only for pairs the cut discards anyway
    }
    if (GMODE == G64_COEF) {
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const double eu = fma(r[c], a.uk, -fi[c]);     // |eu| <= 1/2, one rounding
            const double* t = tab + idx[c] * TAB_STRIDE;
            double p = t[LEVEL];
#pragma unroll
            for (int k = LEVEL - 1; k >= 0; --k) p = fma(p, eu, t[k]);
            g[c] = p;
        }
    } else if (GMODE == G64_QUAD) {
        // Eq. 2 with the brackets of T[3] and T[4] read from the table beside {T_i, E_i}: 9 DP instructions instead of 14
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const double2 te = reinterpret_cast<const double2*>(tab)[2 * idx[c]];
            const double2 hi = reinterpret_cast<const double2*>(tab)[2 * idx[c] + 1];
            const double xi = fi[c] * a.h;
            const double e = fma(r[c], a.inv2rs, -xi);
            const double xi2 = xi * xi;
            double poly = 0.0;
            if (LEVEL >= 4) poly = hi.y;
            if (LEVEL >= 3) poly = fma(poly, e, hi.x);
            if (LEVEL >= 2) poly = fma(poly, e, fma(-xi, xi2, xi));
            if (LEVEL >= 1) poly = fma(poly, e, xi2);
            g[c] = LEVEL >= 1 ? fma(te.y * e, poly, te.x) : te.x;
        }
    } else {
        // Eq. 2 to level LEVEL about the nearest node, the node polynomials rebuilt from x_i
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const double2 te = reinterpret_cast<const double2*>(tab)[idx[c]];
            const double xi = fi[c] * a.h;                 // the node
            const double e = fma(r[c], a.inv2rs, -xi);     // eps = x - x_i, one rounding
            const double xi2 = xi * xi;
            double poly = 0.0;   // sum_{k>=1} coefficient_k(x_i) e^(k-1), Horner from the highest kept level
            if (LEVEL >= 4) poly = -xi * fma(fma(xi2, 1.0 / 3.0, -1.5), xi2, 1.0);
            if (LEVEL >= 3) poly = fma(poly, e, fma(fma(xi2, 2.0 / 3.0, -5.0 / 3.0), xi2, 1.0 / 3.0));
            if (LEVEL >= 2) poly = fma(poly, e, fma(-xi, xi2, xi));
            if (LEVEL >= 1) poly = fma(poly, e, xi2);
            g[c] = LEVEL >= 1 ? fma(te.y * e, poly, te.x) : te.x;
        }
    }
    }
}

// LG lanes own the leaf's targets (T per lane); with LG = 16 the two half-warps take alternate sources
template <int T, int LG, int GMODE, int LEVEL>
__global__ void __launch_bounds__(256) p2p_fp64_kernel(P64Args a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const int M = a.maxleaf;
    const int stage_bytes = a.chunk_max * 32;
    unsigned char* ring = smem_raw + (size_t)warp * N_STAGES64 * stage_bytes;
    unsigned char* tail = smem_raw + (size_t)W * N_STAGES64 * stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(tail) + warp * N_STAGES64;
    uint2* meta = reinterpret_cast<uint2*>(tail + W * N_STAGES64 * 8) + warp * N_STAGES64;
    double* red = reinterpret_cast<double*>(tail + W * N_STAGES64 * 16);   // W x T x 32 x 3 doubles
    double* tab = red + (size_t)W * T * 32 * 3;

    constexpr int HS = 32 / LG;
    const int half = HS > 1 ? lane / LG : 0;

    if (GMODE != G64_DIRECT) {   // the interpolation table lives in shared memory (Fig. 1)
        for (int i = threadIdx.x; i < a.tab_doubles; i += blockDim.x) tab[i] = a.table[i];
        __syncthreads();
    }

    const long long leaf = a.order[a.first + blockIdx.x];
    const long long slot0 = leaf * M;

    double tx[T], ty[T], tz[T], ax[T], ay[T], az[T];
    int tslot[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        tslot[t] = (int)slot0 + (lane % LG) + LG * t;
        const double4 p = a.p64[tslot[t]];
        tx[t] = p.x; ty[t] = p.y; tz[t] = p.z;
        ax[t] = ay[t] = az[t] = 0.0;
    }

    const long long c0 = a.chunk_ptr[leaf], c1 = a.chunk_ptr[leaf + 1];
    const long long n_all = c1 - c0;
    const int n_my = n_all > warp ? (int)((n_all - warp + W - 1) / W) : 0;

    if (lane == 0) {
        for (int s = 0; s < N_STAGES64; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncwarp();
    auto issue = [&](int k) {
        const uint2 e = a.chunks[c0 + warp + (long long)k * W];
        const int st = k % N_STAGES64;
        meta[st] = e;
        const uint32_t bytes = (e.y & 0xffffu) * 32u;
        mbar_expect_tx(&bars[st], bytes);
        bulk_g2s(ring + (size_t)st * stage_bytes, a.p64 + e.x, bytes, &bars[st]);
    };
    if (lane == 0)
        for (int k = 0; k < N_STAGES64 && k < n_my; ++k) issue(k);

    for (int k = 0; k < n_my; ++k) {
        const int st = k % N_STAGES64;
        mbar_wait(&bars[st], (uint32_t)(k / N_STAGES64) & 1u);
        const uint2 e = meta[st];
        const int ns = (int)(e.y & 0xffffu);
        const double4* src = reinterpret_cast<const double4*>(ring + (size_t)st * stage_bytes);
        const bool per_pair = (e.y & ENTRY_PER_PAIR) != 0;
        // image shift of this entry, moved onto the targets: d = (r_j + s L) - r_i = r_j - (r_i - s L)
        double sx = 0, sy = 0, sz = 0;
        if (!per_pair) {
            sx = a.L * (double)((int)((e.y >> 16) & 3u) - 1);
            sy = a.L * (double)((int)((e.y >> 18) & 3u) - 1);
            sz = a.L * (double)((int)((e.y >> 20) & 3u) - 1);
        }
        double px[T], py[T], pz[T], qx[T], qy[T], qz[T];
#pragma unroll
        for (int t = 0; t < T; ++t) {
            px[t] = py[t] = pz[t] = 0.0;
            qx[t] = tx[t] - sx; qy[t] = ty[t] - sy; qz[t] = tz[t] - sz;
        }
        // U sources x T targets = NCH independent chains per iteration (ns is a multiple of maxleaf >= 16)
        constexpr int U = T == 1 ? 4 : T == 2 ? 2 : 1;
        constexpr int NCH = U * T;
        auto step = [&](const int j, const bool image) {
            double dx[NCH], dy[NCH], dz[NCH], r2[NCH], r[NCH], idr[NCH], gm[NCH], g[NCH];
            bool incut[NCH];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const double4 s = src[j + u * HS];
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const int c = u * T + t;
                    dx[c] = s.x - qx[t]; dy[c] = s.y - qy[t]; dz[c] = s.z - qz[t];
                    if (image) {      // degenerate geometry (tiny N): minimum image per pair
                        dx[c] -= a.L * rint(dx[c] / a.L);
                        dy[c] -= a.L * rint(dy[c] / a.L);
                        dz[c] -= a.L * rint(dz[c] / a.L);
                    }
                    gm[c] = s.w;
                }
            }
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                r2[c] = fma(dx[c], dx[c], fma(dy[c], dy[c], fma(dz[c], dz[c], a.r2add)));
                idr[c] = rsqrt64(r2[c]);
                r[c] = r2[c] * idr[c];
                // the cut (A8): positive doubles order like their bit patterns, so the compare runs on the integer
                // pipe instead of taking a slot of the FP64 pipe
                incut[c] = __double_as_longlong(r2[c]) < __double_as_longlong(a.rcut2);
            }
            g_eval<GMODE, LEVEL, NCH>(a, tab, r, incut, g);
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                const double v = (gm[c] * idr[c]) * (idr[c] * idr[c]) * g[c];
                const double w = incut[c] ? v : 0.0;             // also drops what g did beyond its range
                const int t = c % T;
                px[t] = fma(w, dx[c], px[t]); py[t] = fma(w, dy[c], py[t]); pz[t] = fma(w, dz[c], pz[t]);
            }
        };
        if (per_pair) {
            for (int j = half; j < ns; j += HS * U) step(j, true);
        } else {
            for (int j = half; j < ns; j += HS * U) step(j, false);
        }
#pragma unroll
        for (int t = 0; t < T; ++t) { ax[t] += px[t]; ay[t] += py[t]; az[t] += pz[t]; }
        __syncwarp();
        if (lane == 0 && k + N_STAGES64 < n_my) issue(k + N_STAGES64);
    }

#pragma unroll
    for (int o = 16; o >= LG; o >>= 1) {     // add the half-warps' partial sums (fixed order)
#pragma unroll
        for (int t = 0; t < T; ++t) {
            ax[t] += __shfl_xor_sync(0xffffffffu, ax[t], o);
            ay[t] += __shfl_xor_sync(0xffffffffu, ay[t], o);
            az[t] += __shfl_xor_sync(0xffffffffu, az[t], o);
        }
    }
    // sum the warps' partial accelerations (fixed order: deterministic), then scatter to caller order
    if (W > 1) {
#pragma unroll
        for (int t = 0; t < T; ++t) {
            double* rr = red + ((size_t)(warp * T + t) * 32 + lane) * 3;
            rr[0] = ax[t]; rr[1] = ay[t]; rr[2] = az[t];
        }
        __syncthreads();
        if (warp != 0) return;
#pragma unroll
        for (int t = 0; t < T; ++t) {
            for (int w = 1; w < W; ++w) {
                const double* rr = red + ((size_t)(w * T + t) * 32 + lane) * 3;
                ax[t] += rr[0]; ay[t] += rr[1]; az[t] += rr[2];
            }
        }
    }
#pragma unroll
    for (int t = 0; t < T; ++t) {
        if (lane >= LG) continue;
        const int dst = a.slot_src[tslot[t]];
        if (dst < 0) continue;
        if (a.out_f32) {
            float* o = reinterpret_cast<float*>(a.out) + 3 * (size_t)dst;
            o[0] = (float)ax[t]; o[1] = (float)ay[t]; o[2] = (float)az[t];
        } else {
            double* o = reinterpret_cast<double*>(a.out) + 3 * (size_t)dst;
            o[0] = ax[t]; o[1] = ay[t]; o[2] = az[t];
        }
    }
}

template <int T, int LG, int GMODE, int LEVEL>
static int launch_t(Ctx* c, const P64Args& a, long long count, int W, size_t smem, cudaStream_t st)
{
    auto kern = p2p_fp64_kernel<T, LG, GMODE, LEVEL>;
    if (smem > 227 * 1024) return fail(c, PHOTONS_EINVAL, "fp64 kernel: %zu bytes of shared memory (ring + table) exceed 227 KB; use a smaller table or chunk_max", smem);
    PH_CUDA(c, opt_in_smem(c, reinterpret_cast<const void*>(kern), smem));
    kern<<<(unsigned)count, 32 * W, smem, st>>>(a);
    ++c->launches;
    PH_CUDA(c, cudaGetLastError());
    return PHOTONS_OK;
}

template <int T, int LG, int GMODE>
static int launch_l(Ctx* c, const P64Args& a, long long count, int W, size_t smem, cudaStream_t st)
{
    switch (c->p.table_level) {
        case 0: return launch_t<T, LG, GMODE, 0>(c, a, count, W, smem, st);
        case 1: return launch_t<T, LG, GMODE, 1>(c, a, count, W, smem, st);
        case 2: return launch_t<T, LG, GMODE, 2>(c, a, count, W, smem, st);
        case 3: return launch_t<T, LG, GMODE, 3>(c, a, count, W, smem, st);
        default: return launch_t<T, LG, GMODE, 4>(c, a, count, W, smem, st);
    }
}

template <int T, int LG>
static int launch_g(Ctx* c, const P64Args& a, long long count, int W, size_t smem, cudaStream_t st)
{
    if (c->p.g_mode == PHOTONS_G_DIRECT) return launch_t<T, LG, G64_DIRECT, 0>(c, a, count, W, smem, st);
    if (c->p.table_layout == PHOTONS_TABLE_COEF) return launch_l<T, LG, G64_COEF>(c, a, count, W, smem, st);
    if (c->p.table_layout == PHOTONS_TABLE_QUAD) return launch_l<T, LG, G64_QUAD>(c, a, count, W, smem, st);
    return launch_l<T, LG, G64_TABLE>(c, a, count, W, smem, st);
}

int launch_p2p_fp64(Ctx* c, long long first, long long count, void* out, bool out_f32, cudaStream_t st)
{
    P64Args a{};
    a.p64 = c->d_p64; a.slot_src = c->d_slot_src; a.chunk_ptr = c->d_chunk_ptr; a.chunks = c->d_chunks;
    a.order = c->d_order; a.first = first; a.maxleaf = c->p.maxleaf; a.chunk_max = c->p.chunk_max;
    a.L = c->p.boxsize; a.rcut2 = c->r_cut * c->r_cut; a.inv2rs = 1.0 / (2.0 * c->r_s);
    // start value of the r^2 chain: eps^2 (A23), else a floor far below any separation, scaled with r_cut^2 so that
    // it means the same in any units
    a.r2add = c->p.softening > 0 ? c->p.softening * c->p.softening : R2_FLOOR64 * a.rcut2;
    const bool coef = c->p.table_layout == PHOTONS_TABLE_COEF, quad = c->p.table_layout == PHOTONS_TABLE_QUAD;
    a.table = nullptr; a.tn = 0; a.tab_doubles = 0;
    if (c->p.g_mode == PHOTONS_G_TABLE) {
        a.tn = c->table.n;
        a.table = coef ? c->table.d_C64 : quad ? c->table.d_Q64 : reinterpret_cast<const double*>(c->table.d_TE64);
        a.tab_doubles = (a.tn + 1) * (coef ? TAB_STRIDE : quad ? 4 : 2);
        a.h = 3.0 / a.tn;
        a.uk = a.tn / 3.0 * a.inv2rs;
    }
    a.out = out; a.out_f32 = out_f32 ? 1 : 0;
    const int W = c->p.warps_per_leaf;
    const int M = c->p.maxleaf;
    const int T = (M + 31) / 32;
    const size_t smem = (size_t)W * N_STAGES64 * c->p.chunk_max * 32 + (size_t)W * N_STAGES64 * 16 + (size_t)W * T * 32 * 3 * 8 +
                        (size_t)a.tab_doubles * 8;
    switch (M) {
        case 16: return launch_g<1, 16>(c, a, count, W, smem, st);
        case 32: return launch_g<1, 32>(c, a, count, W, smem, st);
        case 64: return launch_g<2, 32>(c, a, count, W, smem, st);
        default: return launch_g<4, 32>(c, a, count, W, smem, st);
    }
}

}  // namespace photons
