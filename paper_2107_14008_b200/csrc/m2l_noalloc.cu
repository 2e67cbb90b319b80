// photons_m2l_noalloc: the truncated M2L operator (§2; A24-A26) for callers that cannot
// allocate - code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// A variant of m2l.cu's kernel that splits every target cell's source list into S segments (one warp each), so that a
// few hundred cells with long lists - the small-box / isolated case in which the paper says M2L matters, L224 - still
// fill the 148 SMs; the segments' partial L_n go through scratch memory and a second kernel adds them in a fixed order.
// That scratch is the file-scope array below: 8 MiB that every GPU which loads the library holds until the process
// exits.  Nothing is allocated, freed, created or synchronised by the entry point: it enqueues two kernels.
//
// The array's name is a host-side stand-in in host code, not a device address: the device address is looked up once per
// device with cudaGetSymbolAddress (that device current) and it is that pointer the kernels are given.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "common.cuh"
#include "m2l_generated.cuh"

namespace photons {

constexpr size_t NOALLOC_SCRATCH_DOUBLES = PHOTONS_M2L_NOALLOC_SCRATCH_BYTES / sizeof(double);
// partial L_n: [cell][segment][coefficient].  Shared by every call on the device and never cleared: each call writes
// every slot it later reads (empty segments write zeros), so nothing has to start at zero - and calls that overlap on
// the GPU (two streams, two host threads) race on it.
static __device__ __align__(256) double m2l_noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];

struct M2LSplitArgs {
    long long n_cells;
    int n_seg;
    const double* centres;
    const double* multipoles;
    const long long* pair_ptr;
    const int* pair_src;
    const signed char* pair_shift;
    double* partial;            // n_cells x n_seg x NC (the scratch array's device address)
    double* locals;             // n_cells x NC
    double alpha, boxsize;
};

// one warp per (target cell, segment of its source list); the pair arithmetic is m2l.cu's
template <int P>
__global__ void __launch_bounds__(128) m2l_split_kernel(M2LSplitArgs a)
{
    constexpr int NC = M2LPair<P>::NC;
    const int lane = threadIdx.x & 31;
    const long long w = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    if (w >= a.n_cells * a.n_seg) return;
    const long long cell = w / a.n_seg;
    const int seg = (int)(w - cell * a.n_seg);
    const long long q0 = a.pair_ptr[cell], q1 = a.pair_ptr[cell + 1];
    const long long per = (q1 - q0 + a.n_seg - 1) / a.n_seg;
    const long long s0 = q0 + seg * per, s1 = s0 + per < q1 ? s0 + per : q1;
    const double bx = a.centres[3 * cell], by = a.centres[3 * cell + 1], bz = a.centres[3 * cell + 2];
    double L[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) L[c] = 0.0;
    const double a2 = 2.0 * a.alpha * a.alpha;
    const double k0 = 1.0 / (a.alpha * 1.7724538509055160273);     // 1 / (alpha sqrt(pi))
    for (long long q = s0 + lane; q < s1; q += 32) {
        const int src = a.pair_src[q];
        double Rx = bx - a.centres[3 * (size_t)src], Ry = by - a.centres[3 * (size_t)src + 1], Rz = bz - a.centres[3 * (size_t)src + 2];
        if (a.pair_shift) {
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
        double gk = exp(-ar * ar) * k0;
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
        double* dst = a.partial + (size_t)w * NC;       // written even when the segment is empty: the array keeps the last call's contents
#pragma unroll
        for (int c = 0; c < NC; ++c) dst[c] = L[c];
    }
}

// one thread per (cell, coefficient): the segments' partial sums in ascending segment order (reproducible)
__global__ void m2l_split_reduce_kernel(long long n_out, int nc, int n_seg, const double* __restrict__ partial, double* __restrict__ locals)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_out) return;
    const long long cell = i / nc;
    const int c = (int)(i - cell * nc);
    const double* p = partial + (size_t)cell * n_seg * nc + c;
    double s = 0.0;
    for (int k = 0; k < n_seg; ++k) s += p[(size_t)k * nc];
    locals[i] = s;
}

constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex g_noalloc_mutex;
static double* g_noalloc_ptr[NOALLOC_MAX_DEVICES];    // device address of the scratch array, per device; null = not looked up yet
static int g_noalloc_sms[NOALLOC_MAX_DEVICES];

static int noalloc_fail(char* err_buf, int err_len, int code, const char* fmt, ...)
{
    if (err_buf && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err_buf, (size_t)err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace photons

using namespace photons;

extern "C" int photons_m2l_noalloc(int device, int p, double r_s, double boxsize, long long n_cells, const double* centres,
                                   const double* multipoles, const long long* pair_ptr, const int* pair_src,
                                   const signed char* pair_shift, double* locals, void* cuda_stream, char* err_buf, int err_len)
{
    if (p < 0 || p > 4 || !(r_s > 0) || n_cells < 1 || !centres || !multipoles || !pair_ptr || !pair_src || !locals)
        return noalloc_fail(err_buf, err_len, PHOTONS_EINVAL, "m2l_noalloc: p must be 0..4, r_s > 0, n_cells >= 1 and the device pointers non-null");
    const int nc = (p + 1) * (p + 2) * (p + 3) / 6;
    // the limit first: it needs no device
    if ((unsigned long long)n_cells * (unsigned long long)nc > NOALLOC_SCRATCH_DOUBLES)
        return noalloc_fail(err_buf, err_len, PHOTONS_EINVAL,
                            "m2l_noalloc: n_cells x NC(p) = %lld x %d partial sums need %llu bytes, the static scratch holds %llu "
                            "(PHOTONS_M2L_NOALLOC_SCRATCH_BYTES): at most %llu cells at order %d; use photons_m2l",
                            n_cells, nc, (unsigned long long)n_cells * nc * 8ULL, (unsigned long long)PHOTONS_M2L_NOALLOC_SCRATCH_BYTES,
                            (unsigned long long)(NOALLOC_SCRATCH_DOUBLES / nc), p);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return noalloc_fail(err_buf, err_len, PHOTONS_ENODEVICE, "m2l_noalloc: no CUDA device");
    }
    if (device < 0 || device >= ndev || device >= NOALLOC_MAX_DEVICES || cudaSetDevice(device) != cudaSuccess)
        return noalloc_fail(err_buf, err_len, PHOTONS_EINVAL, "m2l_noalloc: bad device %d", device);
    double* scratch = nullptr;
    int sms = 0;
    {
        // set-up, once per device, with that device current: the device address of the file-scope array
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_ptr[device]) {
            double* ptr = nullptr;
            cudaError_t e = cudaGetSymbolAddress((void**)&ptr, m2l_noalloc_scratch);
            if (e != cudaSuccess || !ptr) {
                cudaGetLastError();
                return noalloc_fail(err_buf, err_len, PHOTONS_ECUDA, "m2l_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            }
            int n = 0;
            e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device);
            if (e != cudaSuccess || n < 1) {
                cudaGetLastError();
                return noalloc_fail(err_buf, err_len, PHOTONS_ECUDA, "m2l_noalloc: cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
            }
            g_noalloc_sms[device] = n;
            g_noalloc_ptr[device] = ptr;
        }
        scratch = g_noalloc_ptr[device];
        sms = g_noalloc_sms[device];
    }
    // segments per cell: enough warps for ~16 per SM, at most 32, and no more than the scratch array holds
    long long n_seg = ((long long)sms * 16 + n_cells - 1) / n_cells;
    const long long fit = (long long)(NOALLOC_SCRATCH_DOUBLES / ((unsigned long long)n_cells * nc));
    if (n_seg > 32) n_seg = 32;
    if (n_seg > fit) n_seg = fit;
    if (n_seg < 1) n_seg = 1;
    M2LSplitArgs a{};
    a.n_cells = n_cells; a.n_seg = (int)n_seg; a.centres = centres; a.multipoles = multipoles; a.pair_ptr = pair_ptr;
    a.pair_src = pair_src; a.pair_shift = pair_shift; a.partial = scratch; a.locals = locals;
    a.alpha = 1.0 / (2.0 * r_s); a.boxsize = boxsize;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    const long long threads = n_cells * n_seg * 32;
    const unsigned blocks = (unsigned)((threads + 127) / 128);
    switch (p) {
        case 0: m2l_split_kernel<0><<<blocks, 128, 0, st>>>(a); break;
        case 1: m2l_split_kernel<1><<<blocks, 128, 0, st>>>(a); break;
        case 2: m2l_split_kernel<2><<<blocks, 128, 0, st>>>(a); break;
        case 3: m2l_split_kernel<3><<<blocks, 128, 0, st>>>(a); break;
        default: m2l_split_kernel<4><<<blocks, 128, 0, st>>>(a); break;
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        const long long n_out = n_cells * nc;
        m2l_split_reduce_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, st>>>(n_out, nc, (int)n_seg, scratch, locals);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return noalloc_fail(err_buf, err_len, PHOTONS_ECUDA, "m2l_noalloc: launch: %s", cudaGetErrorString(e));
    return PHOTONS_OK;
}
