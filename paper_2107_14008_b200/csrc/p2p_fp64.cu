// fp64 P2P kernel (Alg. 1 + Alg. 2, the paper's DP run L196): one CTA per target leaf, the CTA's
// warps split the leaf's source list, lanes own targets, source runs arrive in shared memory by TMA bulk
// copies through a per-warp mbarrier ring (pipeline.cuh).  SURVEY.md §8(a) steps a4-a9.
#include "common.cuh"
#include "pipeline.cuh"

namespace photons {

struct P64Args {
    const double4* p64;       // n_slots x {x, y, z, G m}
    const int* slot_src;      // slot -> caller index (-1 = padding)
    const long long* chunk_ptr;
    const uint2* chunks;
    const int* order;         // CTA b works on leaf order[first + b]
    long long first;
    int maxleaf, chunk_max;
    double L, rcut2, inv2rs;
    const double2* table;     // TABLE mode: {T_i, E_i}, i = 0..tn
    int tn;
    void* out;                // caller order, n x 3
    int out_f32;
};

// Eq. 1 by the special functions, x = r / 2 r_s
__device__ __forceinline__ double g_direct64(double x)
{
    return erfc(x) + 1.1283791670955125739 * x * exp(-x * x);
}

// Eq. 2 to level LEVEL about the nearest node (A14)
template <int LEVEL>
__device__ __forceinline__ double g_table64(double x, const double2* __restrict__ table, int tn)
{
    const double h = 3.0 / tn;
    int i = (int)rint(x * (tn / 3.0));
    i = min(i, tn);
    const double xi = i * h;
    const double e = x - xi;
    const double2 te = __ldg(&table[i]);
    const double Ti = te.x, Ei = te.y;
    const double xi2 = xi * xi;
    double poly = 0.0;   // sum_{k>=1} coefficient_k(x_i) e^(k-1), Horner from the highest kept level
    if (LEVEL >= 4) poly = -xi * (xi2 * xi2 * (1.0 / 3.0) - 1.5 * xi2 + 1.0);
    if (LEVEL >= 3) poly = poly * e + ((2.0 / 3.0) * xi2 * xi2 - (5.0 / 3.0) * xi2 + (1.0 / 3.0));
    if (LEVEL >= 2) poly = poly * e - xi * (xi2 - 1.0);
    if (LEVEL >= 1) poly = poly * e + xi2;
    return LEVEL >= 1 ? Ti + Ei * e * poly : Ti;
}

template <int T, int GMODE, int LEVEL>
__global__ void __launch_bounds__(256) p2p_fp64_kernel(P64Args a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    const int M = a.maxleaf;
    const int stage_bytes = a.chunk_max * 32;
    unsigned char* ring = smem_raw + (size_t)warp * N_STAGES * stage_bytes;
    unsigned char* tail = smem_raw + (size_t)W * N_STAGES * stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(tail) + warp * N_STAGES;
    uint2* meta = reinterpret_cast<uint2*>(tail + W * N_STAGES * 8) + warp * N_STAGES;
    double* red = reinterpret_cast<double*>(tail + W * N_STAGES * 16);   // W x T x 32 x 3 doubles

    const long long leaf = a.order[a.first + blockIdx.x];
    const long long slot0 = leaf * M;

    double tx[T], ty[T], tz[T], ax[T], ay[T], az[T];
    bool live[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        const int l = lane + 32 * t;
        live[t] = l < M;
        const double4 p = a.p64[slot0 + (live[t] ? l : 0)];
        tx[t] = p.x; ty[t] = p.y; tz[t] = p.z;
        ax[t] = ay[t] = az[t] = 0.0;
    }

    const long long c0 = a.chunk_ptr[leaf], c1 = a.chunk_ptr[leaf + 1];
    const long long n_all = c1 - c0;
    const int n_my = n_all > warp ? (int)((n_all - warp + W - 1) / W) : 0;

    if (lane == 0) {
        for (int s = 0; s < N_STAGES; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncwarp();
    auto issue = [&](int k) {
        const uint2 e = a.chunks[c0 + warp + (long long)k * W];
        const int st = k % N_STAGES;
        meta[st] = e;
        const uint32_t bytes = (e.y & 0xffffu) * 32u;
        mbar_expect_tx(&bars[st], bytes);
        bulk_g2s(ring + (size_t)st * stage_bytes, a.p64 + e.x, bytes, &bars[st]);
    };
    if (lane == 0)
        for (int k = 0; k < N_STAGES && k < n_my; ++k) issue(k);

    for (int k = 0; k < n_my; ++k) {
        const int st = k % N_STAGES;
        mbar_wait(&bars[st], (uint32_t)(k / N_STAGES) & 1u);
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
        for (int j = 0; j < ns; ++j) {
            const double4 s = src[j];
#pragma unroll
            for (int t = 0; t < T; ++t) {
                double dx = s.x - qx[t], dy = s.y - qy[t], dz = s.z - qz[t];
                if (per_pair) {
                    dx -= a.L * rint(dx / a.L);
                    dy -= a.L * rint(dy / a.L);
                    dz -= a.L * rint(dz / a.L);
                }
                const double r2 = dx * dx + dy * dy + dz * dz;
                if (r2 < a.rcut2 && r2 > 0.0) {
                    const double idr = rsqrt(r2);
                    const double r = r2 * idr;
                    const double x = r * a.inv2rs;
                    const double g = GMODE == PHOTONS_G_DIRECT ? g_direct64(x) : g_table64<LEVEL>(x, a.table, a.tn);
                    const double w = s.w * g * (idr * idr * idr);
                    px[t] += w * dx; py[t] += w * dy; pz[t] += w * dz;
                }
            }
        }
#pragma unroll
        for (int t = 0; t < T; ++t) { ax[t] += px[t]; ay[t] += py[t]; az[t] += pz[t]; }
        __syncwarp();
        if (lane == 0 && k + N_STAGES < n_my) issue(k + N_STAGES);
    }

    // sum the warps' partial accelerations (fixed order: deterministic), then scatter to caller order
    if (W > 1) {
#pragma unroll
        for (int t = 0; t < T; ++t) {
            double* r = red + ((size_t)(warp * T + t) * 32 + lane) * 3;
            r[0] = ax[t]; r[1] = ay[t]; r[2] = az[t];
        }
        __syncthreads();
        if (warp != 0) return;
#pragma unroll
        for (int t = 0; t < T; ++t) {
            for (int w = 1; w < W; ++w) {
                const double* r = red + ((size_t)(w * T + t) * 32 + lane) * 3;
                ax[t] += r[0]; ay[t] += r[1]; az[t] += r[2];
            }
        }
    }
#pragma unroll
    for (int t = 0; t < T; ++t) {
        if (!live[t]) continue;
        const int dst = a.slot_src[slot0 + lane + 32 * t];
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

template <int T, int GMODE, int LEVEL>
static int launch_t(Ctx* c, const P64Args& a, long long count, int W, size_t smem, cudaStream_t st)
{
    auto kern = p2p_fp64_kernel<T, GMODE, LEVEL>;
    PH_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)count, 32 * W, smem, st>>>(a);
    ++c->launches;
    PH_CUDA(c, cudaGetLastError());
    return PHOTONS_OK;
}

template <int T>
static int launch_g(Ctx* c, const P64Args& a, long long count, int W, size_t smem, cudaStream_t st)
{
    if (c->p.g_mode == PHOTONS_G_DIRECT) return launch_t<T, PHOTONS_G_DIRECT, 0>(c, a, count, W, smem, st);
    switch (c->p.table_level) {
        case 0: return launch_t<T, PHOTONS_G_TABLE, 0>(c, a, count, W, smem, st);
        case 1: return launch_t<T, PHOTONS_G_TABLE, 1>(c, a, count, W, smem, st);
        case 2: return launch_t<T, PHOTONS_G_TABLE, 2>(c, a, count, W, smem, st);
        case 3: return launch_t<T, PHOTONS_G_TABLE, 3>(c, a, count, W, smem, st);
        default: return launch_t<T, PHOTONS_G_TABLE, 4>(c, a, count, W, smem, st);
    }
}

int launch_p2p_fp64(Ctx* c, long long first, long long count, void* out, bool out_f32, cudaStream_t st)
{
    P64Args a{};
    a.p64 = c->d_p64; a.slot_src = c->d_slot_src; a.chunk_ptr = c->d_chunk_ptr; a.chunks = c->d_chunks;
    a.order = c->d_order; a.first = first; a.maxleaf = c->p.maxleaf; a.chunk_max = c->p.chunk_max;
    a.L = c->p.boxsize; a.rcut2 = c->r_cut * c->r_cut; a.inv2rs = 1.0 / (2.0 * c->r_s);
    a.table = c->table.d_TE64; a.tn = c->table.n; a.out = out; a.out_f32 = out_f32 ? 1 : 0;
    const int W = c->p.warps_per_leaf;
    const int T = (c->p.maxleaf + 31) / 32;
    const size_t smem = (size_t)W * N_STAGES * c->p.chunk_max * 32 + (size_t)W * N_STAGES * 16 + (size_t)W * T * 32 * 3 * 8;
    switch (T) {
        case 1: return launch_g<1>(c, a, count, W, smem, st);
        case 2: return launch_g<2>(c, a, count, W, smem, st);
        default: return launch_g<4>(c, a, count, W, smem, st);
    }
}

}  // namespace photons
