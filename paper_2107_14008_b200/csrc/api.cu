// C ABI of the photons library (include/photons.h): context, parameter validation, particle intake,
// the short_range_acc driver (stream batches, output staging) and the test hooks.
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <new>

#include "common.cuh"

namespace photons {

int fail(Ctx* c, int code, const char* fmt, ...)
{
    char buf[1024];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    return code;
}

cudaError_t opt_in_smem(Ctx* c, const void* kernel, size_t bytes)
{
    for (const void* k : c->smem_opted)
        if (k == kernel) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) c->smem_opted.push_back(kernel);
    return e;
}

void* workspace(Ctx* c, int slot, size_t bytes)
{
    DevBuf& b = c->ws[slot];
    if (bytes == 0) bytes = 16;
    if (b.cap >= bytes) return b.p;
    if (b.p) { cudaFree(b.p); b.p = nullptr; b.cap = 0; }
    const cudaError_t e = cudaMalloc(&b.p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        b.p = nullptr;
        fail(c, PHOTONS_ENOMEM, "device allocation of %zu bytes failed (workspace slot %d): %s", bytes, slot, cudaGetErrorString(e));
        return nullptr;
    }
    b.cap = bytes;
    return b.p;
}

void workspace_free(Ctx* c)
{
    for (DevBuf& b : c->ws) {
        if (b.p) cudaFree(b.p);
        b.p = nullptr;
        b.cap = 0;
    }
}

static double now_ms()
{
    using namespace std::chrono;
    return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

// wrap into [0, L), flag non-finite values, find max |m| (the fp32 kernels' mass unit); src is fp64 or fp32.
// flags: [0] = non-finite input seen, [1] = bits of max |m| (non-negative doubles order like their bit patterns),
// [2] = bits of min |m| (starts at all ones), [3] = signs seen (1 = negative, 2 = positive): all masses are equal iff
// [1] == [2] and only one sign was seen
template <typename Tin>
__global__ void intake_kernel(long long n, const Tin* __restrict__ pos, const Tin* __restrict__ mass, double L, int periodic,
                              double default_mass, double* __restrict__ opos, double* __restrict__ omass,
                              unsigned long long* __restrict__ flags)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = i < n;
    if (!live) i = n - 1;
    bool ok = true;
    for (int a = 0; a < 3; ++a) {
        double x = (double)pos[3 * i + a];
        if (!isfinite(x)) { ok = false; x = 0.0; }
        if (periodic) {
            x -= L * floor(x / L);
            if (x >= L) x -= L;      // x/L rounding can leave x == L
            if (x < 0.0) x = 0.0;
        }
        if (live) opos[3 * i + a] = x;
    }
    double m = mass ? (double)mass[i] : default_mass;
    if (!isfinite(m)) { ok = false; m = 0.0; }
    if (live) omass[i] = m;
    if (!ok) atomicExch(&flags[0], 1ULL);
    unsigned long long mb = (unsigned long long)__double_as_longlong(fabs(m));
    for (int o = 16; o > 0; o >>= 1) mb = max(mb, __shfl_xor_sync(0xffffffffu, mb, o));
    // (a plain read first: once the flags hold the extremes - after the first few warps when all masses are equal -
    // no warp issues an atomic any more; 16.7 M particles: 1.13 -> 0.45 ms)
    const volatile unsigned long long* vf = flags;
    if ((threadIdx.x & 31) == 0 && mb > vf[1]) atomicMax(&flags[1], mb);
    unsigned long long mn = (unsigned long long)__double_as_longlong(fabs(m));
    unsigned sg = m < 0.0 ? 1u : m > 0.0 ? 2u : 0u;
    for (int o = 16; o > 0; o >>= 1) { mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o)); sg |= __shfl_xor_sync(0xffffffffu, sg, o); }
    if ((threadIdx.x & 31) == 0) {
        if (mn < vf[2]) atomicMin(&flags[2], mn);
        if ((vf[3] & sg) != sg) atomicOr(&flags[3], (unsigned long long)sg);
    }
}

// build_ms from the events recorded around photons_build_leaves' device work
static void resolve_build_ms(Ctx* c)
{
    if (!c->build_ms_pending) return;
    float ms = 0;
    if (cudaEventSynchronize(c->evb1) == cudaSuccess && cudaEventElapsedTime(&ms, c->evb0, c->evb1) == cudaSuccess) c->stats.build_ms = ms;
    else cudaGetLastError();
    c->build_ms_pending = false;
}

static void free_particles(Ctx* c)
{
    c->d_pos = nullptr;     // the buffers stay in the workspace
    c->d_mass = nullptr;
    c->n = 0;
}

}  // namespace photons

using namespace photons;

extern "C" {

void photons_default_params(photons_params* p)
{
    if (!p) return;
    memset(p, 0, sizeof *p);
    p->boxsize = 1.0;
    p->n_pm = 32;
    p->rs_over_cell = 1.2;
    p->rcut_over_rs = 6.0;
    p->G = 1.0;
    p->maxleaf = 32;
    p->precision = PHOTONS_FP32;
    p->g_mode = PHOTONS_G_POLY;
    p->table_nodes = 512;
    p->table_level = 2;
    p->n_streams = 1;
    p->device = 0;
    p->close_pair_radius = 0.0;
    p->chunk_max = 0;
    p->warps_per_leaf = 0;
    p->targets_per_lane = 0;
    p->poly_degree = 0;
    p->periodic = 1;
    p->softening = 0.0;
    p->table_layout = PHOTONS_TABLE_PAPER;
    p->leaf_order = 0;
    p->orb_method = 0;
    p->mass_path = 0;
}

static int create_fail(char* err_buf, int err_len, int code, const char* msg)
{
    if (err_buf && err_len > 0) snprintf(err_buf, err_len, "%s", msg);
    return code;
}

int photons_create(const photons_params* pp, photons_ctx** out, char* err_buf, int err_len)
{
    if (!pp || !out) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "null argument");
    photons_params p = *pp;
    if (!(p.boxsize > 0) || !std::isfinite(p.boxsize)) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "boxsize must be > 0");
    if (p.n_pm < 1) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "n_pm must be >= 1");
    if (!(p.rs_over_cell > 0) || !(p.rcut_over_rs > 0)) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "rs_over_cell and rcut_over_rs must be > 0");
    if (!std::isfinite(p.G)) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "G must be finite");
    if (p.maxleaf != 16 && p.maxleaf != 32 && p.maxleaf != 64 && p.maxleaf != 128)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "maxleaf must be 16, 32, 64 or 128");
    if (p.precision < PHOTONS_FP64 || p.precision > PHOTONS_MIXED) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "bad precision");
    if (p.g_mode < PHOTONS_G_DIRECT || p.g_mode > PHOTONS_G_FUSED) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "bad g_mode");
    if ((p.g_mode == PHOTONS_G_POLY || p.g_mode == PHOTONS_G_FUSED) && p.precision == PHOTONS_FP64)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "g_mode POLY / FUSED are fp32 approximations; use DIRECT or TABLE with FP64");
    if (p.g_mode != PHOTONS_G_DIRECT && p.rcut_over_rs > 6.0)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "TABLE, POLY and FUSED cover x = r/2r_s in [0,3]: rcut_over_rs must be <= 6");
    if (p.g_mode == PHOTONS_G_TABLE) {
        if (p.table_nodes < 64 || p.table_nodes > 4096) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "table_nodes must be 64..4096");
        if (p.table_level < 0 || p.table_level > 4) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "table_level must be 0..4");
        if (p.table_level > 3 && p.precision != PHOTONS_FP64)
            return create_fail(err_buf, err_len, PHOTONS_EINVAL, "table_level 4 needs PHOTONS_FP64 (the fp32 kernels keep T[0..3])");
        if (p.table_layout != PHOTONS_TABLE_PAPER && p.table_layout != PHOTONS_TABLE_COEF && p.table_layout != PHOTONS_TABLE_QUAD)
            return create_fail(err_buf, err_len, PHOTONS_EINVAL, "bad table_layout");
        if (p.table_layout != PHOTONS_TABLE_PAPER && p.precision != PHOTONS_FP64)
            return create_fail(err_buf, err_len, PHOTONS_EINVAL, "table_layout COEF / QUAD are options of the PHOTONS_FP64 path");
    }
    if (p.orb_method != 0 && p.orb_method != 1) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "orb_method must be 0 or 1");
    if (p.mass_path != 0 && p.mass_path != 1) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "mass_path must be 0 or 1");
    if (p.leaf_order != 0 && p.leaf_order != 1) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "leaf_order must be 0 or 1");
    if (p.n_streams < 1 || p.n_streams > 64) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "n_streams must be 1..64");
    if (p.close_pair_radius < 0 || !std::isfinite(p.close_pair_radius)) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "close_pair_radius must be >= 0");
    if (p.chunk_max == 0) p.chunk_max = p.maxleaf > 128 ? p.maxleaf : 128;
    if (p.chunk_max % p.maxleaf || p.chunk_max < p.maxleaf || p.chunk_max > 256)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "chunk_max must be a multiple of maxleaf, <= 256");
    if (p.warps_per_leaf == 0) p.warps_per_leaf = 4;
    if (p.warps_per_leaf != 1 && p.warps_per_leaf != 2 && p.warps_per_leaf != 4 && p.warps_per_leaf != 8)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "warps_per_leaf must be 1, 2, 4 or 8");
    if (p.targets_per_lane == 0) p.targets_per_lane = p.maxleaf <= 32 ? 1 : p.maxleaf / 32;
    {
        const int t = p.targets_per_lane, m = p.maxleaf;
        const bool ok = (m == 16 && (t == 1 || t == 2)) || (m == 32 && (t == 1 || t == 2)) || (m == 64 && t == 2) || (m == 128 && t == 4);
        if (!ok) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "targets_per_lane not available for this maxleaf");
    }
    if (p.g_mode == PHOTONS_G_FUSED) {
        if (p.poly_degree == 0) p.poly_degree = 10;
        if (p.poly_degree < 9 || p.poly_degree > 11) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "poly_degree must be 9..11 with g_mode FUSED");
    } else {
        if (p.poly_degree == 0) p.poly_degree = 12;
        if (p.poly_degree < 10 || p.poly_degree > 14) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "poly_degree must be 10..14");
    }

    const double r_s = p.rs_over_cell * p.boxsize / p.n_pm;
    const double r_cut = p.rcut_over_rs * r_s;
    if (p.periodic != 0 && p.periodic != 1) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "periodic must be 0 or 1");
    if (p.periodic && !(r_cut < 0.5 * p.boxsize)) return create_fail(err_buf, err_len, PHOTONS_EBOX, "r_cut >= boxsize/2: minimum image is not unique");
    if (p.close_pair_radius >= r_cut) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "close_pair_radius must be < r_cut");
    if (!(p.softening >= 0) || !std::isfinite(p.softening) || p.softening >= r_cut)
        return create_fail(err_buf, err_len, PHOTONS_EINVAL, "softening must be >= 0 and < r_cut");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return create_fail(err_buf, err_len, PHOTONS_ENODEVICE, "no CUDA device (this library has no CPU fallback)");
    }
    if (p.device < 0 || p.device >= ndev) return create_fail(err_buf, err_len, PHOTONS_EINVAL, "device ordinal out of range");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p.device) != cudaSuccess || cudaSetDevice(p.device) != cudaSuccess) {
        cudaGetLastError();
        return create_fail(err_buf, err_len, PHOTONS_ECUDA, "cannot select the CUDA device");
    }
    if (prop.major < 10) return create_fail(err_buf, err_len, PHOTONS_ENODEVICE, "kernels are built for sm_100a only (Blackwell B200)");

    Ctx* c = new (std::nothrow) Ctx;
    if (!c) return create_fail(err_buf, err_len, PHOTONS_ENOMEM, "host allocation failed");
    c->p = p;
    c->r_s = r_s;
    c->r_cut = r_cut;
    // length unit of the fp32 kernels: the power of two just below r_cut (an exact rescaling of fp32 data)
    c->pscale = std::ldexp(1.0, (int)std::floor(std::log2(r_cut)));
    c->sm_count = prop.multiProcessorCount;
    bool ok = true;
    c->streams.resize(p.n_streams);
    c->stream_done.resize(p.n_streams);
    for (int i = 0; i < p.n_streams; ++i) {
        c->streams[i] = nullptr; c->stream_done[i] = nullptr;
        ok = ok && cudaStreamCreateWithFlags(&c->streams[i], cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&c->stream_done[i], cudaEventDisableTiming) == cudaSuccess;
    }
    c->own_stream0 = c->streams[0];
    ok = ok && cudaEventCreate(&c->ev0) == cudaSuccess && cudaEventCreate(&c->ev1) == cudaSuccess;
    ok = ok && cudaEventCreate(&c->evb0) == cudaSuccess && cudaEventCreate(&c->evb1) == cudaSuccess;
    int rc = PHOTONS_OK;
    if (!ok) rc = fail(c, PHOTONS_ECUDA, "stream/event creation failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc == PHOTONS_OK && p.g_mode == PHOTONS_G_TABLE) rc = make_table(c);
    if (rc == PHOTONS_OK && p.g_mode == PHOTONS_G_POLY) rc = make_poly(c);
    if (rc == PHOTONS_OK && p.g_mode == PHOTONS_G_FUSED) rc = make_fused(c);
    if (rc != PHOTONS_OK) {
        create_fail(err_buf, err_len, rc, c->err.c_str());
        photons_destroy(reinterpret_cast<photons_ctx*>(c));
        return rc;
    }
    *out = reinterpret_cast<photons_ctx*>(c);
    return PHOTONS_OK;
}

int photons_set_stream(photons_ctx* ctx, void* cuda_stream)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    c->streams[0] = cuda_stream ? reinterpret_cast<cudaStream_t>(cuda_stream) : c->own_stream0;
    return PHOTONS_OK;
}

int photons_set_particles(photons_ctx* ctx, long long n, const void* pos, const void* mass, int dtype, int mem_kind,
                          void* cuda_stream)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    if (n < 1 || !pos) return fail(c, PHOTONS_EINVAL, "set_particles: n must be >= 1 and pos non-null");
    if (dtype != PHOTONS_DTYPE_F64 && dtype != PHOTONS_DTYPE_F32) return fail(c, PHOTONS_EINVAL, "set_particles: bad dtype");
    if (mem_kind != PHOTONS_MEM_HOST && mem_kind != PHOTONS_MEM_DEVICE) return fail(c, PHOTONS_EINVAL, "set_particles: bad mem_kind");
    if (2 * n + 256 >= (1LL << 31)) return fail(c, PHOTONS_EINVAL, "set_particles: too many particles for 32-bit slot indices");
    PH_CUDA(c, cudaSetDevice(c->p.device));
    free_leaves(c);
    free_particles(c);
    cudaStream_t st = cuda_stream ? reinterpret_cast<cudaStream_t>(cuda_stream) : c->streams[0];
    const size_t esz = dtype == PHOTONS_DTYPE_F64 ? 8 : 4;
    c->d_pos = static_cast<double*>(workspace(c, WS_POS, sizeof(double) * 3 * n));
    c->d_mass = static_cast<double*>(workspace(c, WS_MASS, sizeof(double) * n));
    unsigned long long* d_flags = static_cast<unsigned long long*>(workspace(c, WS_FLAG, 4 * sizeof(unsigned long long)));
    if (!c->d_pos || !c->d_mass || !d_flags) { free_particles(c); return PHOTONS_ENOMEM; }
    const void *src_pos = pos, *src_mass = mass;
    if (mem_kind == PHOTONS_MEM_HOST) {
        void* d_in_pos = workspace(c, WS_IN_POS, esz * 3 * n);
        if (!d_in_pos) { free_particles(c); return PHOTONS_ENOMEM; }
        PH_CUDA(c, cudaMemcpyAsync(d_in_pos, pos, esz * 3 * n, cudaMemcpyHostToDevice, st));
        src_pos = d_in_pos;
        if (mass) {
            void* d_in_mass = workspace(c, WS_IN_MASS, esz * n);
            if (!d_in_mass) { free_particles(c); return PHOTONS_ENOMEM; }
            PH_CUDA(c, cudaMemcpyAsync(d_in_mass, mass, esz * n, cudaMemcpyHostToDevice, st));
            src_mass = d_in_mass;
        }
    }
    PH_CUDA(c, cudaMemsetAsync(d_flags, 0, 4 * sizeof(unsigned long long), st));
    PH_CUDA(c, cudaMemsetAsync(d_flags + 2, 0xff, sizeof(unsigned long long), st));
    const int tb = 256;
    const unsigned nb = (unsigned)((n + tb - 1) / tb);
    if (dtype == PHOTONS_DTYPE_F64)
        intake_kernel<double><<<nb, tb, 0, st>>>(n, (const double*)src_pos, (const double*)src_mass, c->p.boxsize, c->p.periodic, 1.0 / (double)n, c->d_pos, c->d_mass, d_flags);
    else
        intake_kernel<float><<<nb, tb, 0, st>>>(n, (const float*)src_pos, (const float*)src_mass, c->p.boxsize, c->p.periodic, 1.0 / (double)n, c->d_pos, c->d_mass, d_flags);
    ++c->launches;
    unsigned long long h_flags[4] = {0, 0, 0, 0};
    cudaError_t e = cudaMemcpyAsync(h_flags, d_flags, sizeof h_flags, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { free_particles(c); return fail(c, PHOTONS_ECUDA, "set_particles: %s", cudaGetErrorString(e)); }
    if (h_flags[0]) { free_particles(c); return fail(c, PHOTONS_ENONFINITE, "set_particles: NaN or Inf in positions or masses"); }
    // mass unit of the fp32 kernels: the power of two >= max |G m| (exact rescaling; G m / unit in (1/2, 1])
    double m_max;
    memcpy(&m_max, &h_flags[1], sizeof m_max);
    const double gm_max = std::fabs(c->p.G) * m_max;
    c->gm_max = gm_max;
    c->gmscale = gm_max > 0 && std::isfinite(gm_max) ? std::ldexp(1.0, (int)std::ceil(std::log2(gm_max))) : 1.0;
    // all masses equal (the paper's runs: one particle species; Alg. 2 L177 carries a single GM): the fp32 kernels then
    // apply G m once per staged run instead of once per pair
    c->gm_uniform = 0.0;
    if (m_max > 0 && h_flags[1] == h_flags[2] && (h_flags[3] == 1 || h_flags[3] == 2))
        c->gm_uniform = c->p.G * (h_flags[3] == 1 ? -m_max : m_max);
    c->n = n;
    return PHOTONS_OK;
}

int photons_build_leaves(photons_ctx* ctx)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    if (c->n < 1) return fail(c, PHOTONS_ESTATE, "build_leaves: call set_particles first");
    PH_CUDA(c, cudaSetDevice(c->p.device));
    free_leaves(c);
    PH_CUDA(c, cudaEventRecord(c->evb0, c->streams[0]));
    int rc = build_leaves_impl(c);
    if (rc != PHOTONS_OK) { free_leaves(c); return rc; }
    PH_CUDA(c, cudaEventRecord(c->evb1, c->streams[0]));
    c->build_ms_pending = true;      // the tail of the build is still in flight: no host synchronisation here
    c->leaves_built = true;
    return PHOTONS_OK;
}

int photons_short_range_acc(photons_ctx* ctx, void* acc, int dtype, int mem_kind, photons_stats* stats)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    if (!c->leaves_built) return fail(c, PHOTONS_ESTATE, "short_range_acc: call build_leaves first");
    if (!acc) return fail(c, PHOTONS_EINVAL, "short_range_acc: acc is null");
    if (dtype != PHOTONS_DTYPE_F64 && dtype != PHOTONS_DTYPE_F32) return fail(c, PHOTONS_EINVAL, "short_range_acc: bad dtype");
    if (mem_kind != PHOTONS_MEM_HOST && mem_kind != PHOTONS_MEM_DEVICE) return fail(c, PHOTONS_EINVAL, "short_range_acc: bad mem_kind");
    PH_CUDA(c, cudaSetDevice(c->p.device));
    const double t0 = now_ms();
    const bool f32 = dtype == PHOTONS_DTYPE_F32;
    const size_t bytes = (f32 ? 4 : 8) * 3 * (size_t)c->n;
    void* d_out = acc;
    bool staged = false;
    if (mem_kind == PHOTONS_MEM_HOST) {
        // A pinned (page-locked, mapped) host buffer is written by the kernel itself: every CTA stores its leaf's
        // accelerations straight into caller order, so the device->host transfer rides along with the kernel instead
        // of following it (201 MB after a 94 ms kernel on config 4).  Pageable memory goes through a staging buffer.
        cudaPointerAttributes at{};
        if (c->p.n_streams >= 1 && cudaPointerGetAttributes(&at, acc) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) {
            d_out = at.devicePointer;
        } else {
            cudaGetLastError();
            d_out = workspace(c, WS_OUT, bytes);
            if (!d_out) return PHOTONS_ENOMEM;
            staged = true;
        }
    }

    // target-leaf batches round-robin over the streams (north_star: "stream concurrency between leaf
    // batches"; "concurrency management"): the order array (photons_params.leaf_order) is cut into
    // 4 n_streams contiguous blocks, block b goes to stream b mod n_streams.
    const int ns = (int)c->streams.size();
    const long long nl = c->n_leaves;
    const long long n_batches = ns == 1 ? 1 : (long long)ns * 4;
    const long long per = (nl + n_batches - 1) / n_batches;
    cudaStream_t s0 = c->streams[0];
    int rc = PHOTONS_OK;
    cudaError_t e = cudaEventRecord(c->ev0, s0);
    for (int s = 1; s < ns && e == cudaSuccess; ++s) e = cudaStreamWaitEvent(c->streams[s], c->ev0, 0);
    for (long long b = 0; b < n_batches && rc == PHOTONS_OK && e == cudaSuccess; ++b) {
        const long long first = b * per;
        const long long count = first + per <= nl ? per : nl - first;
        if (count <= 0) break;
        cudaStream_t st = c->streams[b % ns];
        rc = c->p.precision == PHOTONS_FP64 ? launch_p2p_fp64(c, first, count, d_out, f32, st)
                                            : launch_p2p_fp32(c, first, count, d_out, f32, st);
    }
    for (int s = 1; s < ns && e == cudaSuccess; ++s) {
        e = cudaEventRecord(c->stream_done[s], c->streams[s]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s0, c->stream_done[s], 0);
    }
    if (e == cudaSuccess) e = cudaEventRecord(c->ev1, s0);
    if (e == cudaSuccess && staged) e = cudaMemcpyAsync(acc, d_out, bytes, cudaMemcpyDeviceToHost, s0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s0);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (rc != PHOTONS_OK || e != cudaSuccess) {
        // a failed launch or event call may have left forked streams unjoined: nothing of this call may still be
        // writing the caller's buffer or the workspace when it returns
        for (cudaStream_t s : c->streams) cudaStreamSynchronize(s);
        cudaGetLastError();
    }
    if (rc != PHOTONS_OK) return rc;
    if (e != cudaSuccess) return fail(c, PHOTONS_ECUDA, "short_range_acc: %s", cudaGetErrorString(e));
    float ms = 0;
    cudaEventElapsedTime(&ms, c->ev0, c->ev1);
    c->stats.kernel_ms = ms;
    resolve_build_ms(c);
    c->stats.total_ms = now_ms() - t0;
    c->stats.kernel_launches = c->launches;
    if (stats) *stats = c->stats;
    return PHOTONS_OK;
}

int photons_get_leaf_order(photons_ctx* ctx, long long* perm, long long* leaf_start)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    if (!c->leaves_built) return fail(c, PHOTONS_ESTATE, "get_leaf_order: call build_leaves first");
    if (perm) {
        std::vector<uint32_t> h(c->n);
        PH_CUDA(c, cudaMemcpy(h.data(), c->d_perm, sizeof(uint32_t) * c->n, cudaMemcpyDeviceToHost));
        for (long long i = 0; i < c->n; ++i) perm[i] = h[i];
    }
    if (leaf_start)
        for (long long k = 0; k <= c->n_leaves; ++k) leaf_start[k] = k == c->n_leaves ? c->n : seg_start(c->n, c->depth, k);
    return PHOTONS_OK;
}

int photons_get_interaction_list(photons_ctx* ctx, long long* chunk_ptr, int* first_leaf, int* n_leaf, int* shift_code)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return PHOTONS_EINVAL;
    if (!c->leaves_built) return fail(c, PHOTONS_ESTATE, "get_interaction_list: call build_leaves first");
    if (chunk_ptr) PH_CUDA(c, cudaMemcpy(chunk_ptr, c->d_chunk_ptr, sizeof(long long) * (c->n_leaves + 1), cudaMemcpyDeviceToHost));
    if (first_leaf || n_leaf || shift_code) {
        std::vector<uint2> h(c->stats.n_chunks);
        PH_CUDA(c, cudaMemcpy(h.data(), c->d_chunks, sizeof(uint2) * h.size(), cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < h.size(); ++i) {
            if (first_leaf) first_leaf[i] = (int)(h[i].x / (unsigned)c->p.maxleaf);
            if (n_leaf) n_leaf[i] = (int)((h[i].y & 0xffffu) / (unsigned)c->p.maxleaf);
            if (shift_code) shift_code[i] = entry_shift_code(h[i].y);
        }
    }
    return PHOTONS_OK;
}

int photons_get_stats(photons_ctx* ctx, photons_stats* stats)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c || !stats) return PHOTONS_EINVAL;
    resolve_build_ms(c);
    c->stats.kernel_launches = c->launches;
    *stats = c->stats;
    return PHOTONS_OK;
}

const char* photons_last_error(const photons_ctx* ctx)
{
    const Ctx* c = reinterpret_cast<const Ctx*>(ctx);
    return c ? c->err.c_str() : "null context";
}

void photons_destroy(photons_ctx* ctx)
{
    Ctx* c = reinterpret_cast<Ctx*>(ctx);
    if (!c) return;
    cudaSetDevice(c->p.device);
    free_leaves(c);
    free_particles(c);
    workspace_free(c);
    cudaFree(c->table.d_TE);
    cudaFree(c->table.d_TE64);
    cudaFree(c->table.d_C64);
    cudaFree(c->table.d_Q64);
    if (!c->streams.empty()) c->streams[0] = c->own_stream0;
    for (auto s : c->streams) if (s) cudaStreamDestroy(s);
    for (auto e : c->stream_done) if (e) cudaEventDestroy(e);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->evb0) cudaEventDestroy(c->evb0);
    if (c->evb1) cudaEventDestroy(c->evb1);
    delete c;
}

}  // extern "C"
