// Truncated multipole-to-local operator (§2; A24-A26), fp64.
//
//   L_n(z_B) += sum over the listed source cells A of  sum_{|m| <= p - |n|} M_m(z_A) D_{n+m}(z_B - z_A),
//   D_n = grad^n psi,  psi(r) = erfc(r / 2 r_s) / r.
//
// Mapping: one warp per target cell; its lanes take the cell's source list 32 entries at a time.  A lane evaluates
// erfc and exp once per pair, obtains the radial derivatives f_(k) = (1/r d/dr)^k psi by the upward recurrence
//     B_0 = erfc(a r)/r,   B_k = [(2k-1) B_{k-1} + (2 a^2)^k exp(-a^2 r^2) / (a sqrt(pi))] / r^2,   f_(k) = (-1)^k B_k,
// a = 1/2r_s (equivalent to the paper's closed form L51, which is what the oracle evaluates), builds the derivative
// tensor and contracts it with the source multipoles in registers (generated straight-line code, m2l_generated.cuh),
// and the warp adds its lanes' partial L_n by shuffles in a fixed order.  Bound by the FP64 pipe.
#include "common.cuh"
#include "m2l_generated.cuh"

namespace photons {

struct M2LArgs {
    long long n_cells;
    const double* centres;      // n_cells x 3
    const double* multipoles;   // n_cells x NC
    const long long* pair_ptr;  // n_cells + 1
    const int* pair_src;
    const signed char* pair_shift;   // 3 per pair, or nullptr
    double* locals;             // n_cells x NC
    double alpha, boxsize;      // alpha = 1 / 2 r_s
};

template <int P>
__global__ void __launch_bounds__(128) m2l_kernel(M2LArgs a)
{
    constexpr int NC = M2LPair<P>::NC;
    const int lane = threadIdx.x & 31;
    const long long cell = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    if (cell >= a.n_cells) return;
    const double bx = a.centres[3 * cell], by = a.centres[3 * cell + 1], bz = a.centres[3 * cell + 2];
    double L[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) L[c] = 0.0;
    const double a2 = 2.0 * a.alpha * a.alpha;
    const double k0 = 1.0 / (a.alpha * 1.7724538509055160273);     // 1 / (alpha sqrt(pi))
    for (long long q = a.pair_ptr[cell] + lane; q < a.pair_ptr[cell + 1]; q += 32) {
        const int src = a.pair_src[q];
        double Rx = bx - a.centres[3 * (size_t)src], Ry = by - a.centres[3 * (size_t)src + 1], Rz = bz - a.centres[3 * (size_t)src + 2];
        if (a.pair_shift) {       // the source centre is moved by s box lengths (A26)
            Rx -= a.boxsize * (double)a.pair_shift[3 * q];
            Ry -= a.boxsize * (double)a.pair_shift[3 * q + 1];
            Rz -= a.boxsize * (double)a.pair_shift[3 * q + 2];
        }
        const double r2 = Rx * Rx + Ry * Ry + Rz * Rz;
        const double r = sqrt(r2);
        const double ir2 = 1.0 / r2;
        const double ar = a.alpha * r;
        double f[P + 1];
        double Bk = erfc(ar) / r;
        double gk = exp(-ar * ar) * k0;         // (2 a^2)^k exp(-a^2 r^2) / (a sqrt(pi)), k = 0
        f[0] = Bk;
#pragma unroll
        for (int k = 1; k <= P; ++k) {
            gk *= a2;
            Bk = ((2 * k - 1) * Bk + gk) * ir2;
            f[k] = (k & 1) ? -Bk : Bk;
        }
        M2LPair<P>::apply(Rx, Ry, Rz, f, a.multipoles + (size_t)src * NC, L);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) L[c] += __shfl_xor_sync(0xffffffffu, L[c], o);
    }
    if (lane == 0) {
#pragma unroll
        for (int c = 0; c < NC; ++c) a.locals[(size_t)cell * NC + c] = L[c];
    }
}

template <int P>
static cudaError_t launch_m2l(const M2LArgs& a, cudaStream_t st)
{
    const long long threads = a.n_cells * 32;
    m2l_kernel<P><<<(unsigned)((threads + 127) / 128), 128, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace photons

using namespace photons;

extern "C" int photons_m2l(int device, int p, double r_s, double boxsize, long long n_cells, const double* centres,
                           const double* multipoles, const long long* pair_ptr, const int* pair_src, const signed char* pair_shift,
                           double* locals, int mem_kind, void* cuda_stream, double* kernel_ms)
{
    if (p < 0 || p > 4 || !(r_s > 0) || n_cells < 1 || n_cells > (1LL << 26) || !centres || !multipoles || !pair_ptr || !locals) return PHOTONS_EINVAL;
    if (mem_kind != PHOTONS_MEM_HOST && mem_kind != PHOTONS_MEM_DEVICE) return PHOTONS_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return PHOTONS_ENODEVICE; }
    if (device < 0 || device >= ndev || cudaSetDevice(device) != cudaSuccess) return PHOTONS_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const int nc = (p + 1) * (p + 2) * (p + 3) / 6;
    M2LArgs a{};
    a.n_cells = n_cells; a.alpha = 1.0 / (2.0 * r_s); a.boxsize = boxsize;
    void* bufs[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    long long n_pairs = 0;
    int rc = PHOTONS_OK;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    auto cleanup = [&]() {
        for (void* b : bufs) if (b) cudaFree(b);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    };
#define M2L_CHECK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { cudaGetLastError(); cleanup(); \
        return e_ == cudaErrorMemoryAllocation ? PHOTONS_ENOMEM : PHOTONS_ECUDA; } } while (0)
    if (mem_kind == PHOTONS_MEM_HOST) {
        n_pairs = pair_ptr[n_cells];
        if (n_pairs < 0 || (n_pairs > 0 && !pair_src)) return PHOTONS_EINVAL;
        const size_t sz[6] = {sizeof(double) * 3 * n_cells, sizeof(double) * nc * n_cells, sizeof(long long) * (n_cells + 1),
                              sizeof(int) * (size_t)std::max<long long>(n_pairs, 1), pair_shift ? (size_t)3 * std::max<long long>(n_pairs, 1) : 0,
                              sizeof(double) * nc * n_cells};
        const void* src[5] = {centres, multipoles, pair_ptr, pair_src, pair_shift};
        for (int i = 0; i < 6; ++i) {
            if (!sz[i]) continue;
            M2L_CHECK(cudaMalloc(&bufs[i], sz[i]));
            if (i < 5 && src[i] && (i != 3 || n_pairs > 0) && (i != 4 || n_pairs > 0)) M2L_CHECK(cudaMemcpyAsync(bufs[i], src[i], sz[i], cudaMemcpyHostToDevice, st));
        }
        a.centres = (const double*)bufs[0]; a.multipoles = (const double*)bufs[1]; a.pair_ptr = (const long long*)bufs[2];
        a.pair_src = (const int*)bufs[3]; a.pair_shift = (const signed char*)bufs[4]; a.locals = (double*)bufs[5];
    } else {
        a.centres = centres; a.multipoles = multipoles; a.pair_ptr = pair_ptr; a.pair_src = pair_src; a.pair_shift = pair_shift; a.locals = locals;
    }
    M2L_CHECK(cudaEventCreate(&e0));
    M2L_CHECK(cudaEventCreate(&e1));
    M2L_CHECK(cudaEventRecord(e0, st));
    cudaError_t e = cudaSuccess;
    switch (p) {
        case 0: e = launch_m2l<0>(a, st); break;
        case 1: e = launch_m2l<1>(a, st); break;
        case 2: e = launch_m2l<2>(a, st); break;
        case 3: e = launch_m2l<3>(a, st); break;
        default: e = launch_m2l<4>(a, st); break;
    }
    M2L_CHECK(e);
    M2L_CHECK(cudaEventRecord(e1, st));
    if (mem_kind == PHOTONS_MEM_HOST) M2L_CHECK(cudaMemcpyAsync(locals, a.locals, sizeof(double) * nc * n_cells, cudaMemcpyDeviceToHost, st));
    M2L_CHECK(cudaStreamSynchronize(st));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (kernel_ms) *kernel_ms = ms;
#undef M2L_CHECK
    cleanup();
    return rc;
}
