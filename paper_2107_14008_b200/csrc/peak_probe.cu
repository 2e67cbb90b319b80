// Throughput micro-benchmarks behind photons_peak_probe (include/photons.h): what the B200 issues per second
// for the instruction classes of the pair core.  They give the measured roofline denominators of DESIGN.md §7
// next to the nominal SM-count x lanes x clock figure (PAPER.md L190 quotes its peak the same way).
#include "common.cuh"

namespace photons {

constexpr int PROBE_ITERS = 4096;
constexpr int CH = 16;   // independent dependency chains per thread

template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(float* out, float a_in, float b_in, int iters)
{
    __shared__ float4 sh[64];
    if (threadIdx.x < 64) sh[threadIdx.x] = make_float4(a_in, b_in, a_in, b_in);
    __syncthreads();
    float a = a_in, b = b_in;
    float x[CH];
    float2 y[CH / 2];
    double d[CH / 2];
#pragma unroll
    for (int i = 0; i < CH; ++i) x[i] = 1.0f + 0.001f * (threadIdx.x + i);
#pragma unroll
    for (int i = 0; i < CH / 2; ++i) { y[i] = make_float2(x[2 * i], x[2 * i + 1]); d[i] = x[i]; }
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    float4 acc4 = make_float4(0, 0, 0, 0);
    for (int it = 0; it < iters; ++it) {
        if (KIND == 0) {            // FFMA, three register operands
#pragma unroll
            for (int i = 0; i < CH; ++i) x[i] = fmaf(x[i], a, b);
        } else if (KIND == 1) {     // FFMA2
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) y[i] = __ffma2_rn(y[i], a2, b2);
        } else if (KIND == 2) {     // DFMA
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) d[i] = fma(d[i], (double)a, (double)b);
        } else if (KIND == 3) {     // MUFU.RSQ
#pragma unroll
            for (int i = 0; i < CH; ++i) x[i] = rsqrtf(x[i]);
        } else if (KIND == 5) {     // LDS.128, one address per warp (broadcast)
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const float4 v = sh[(it + i) & 63];
                acc4.x += v.x; acc4.y += v.y; acc4.z += v.z; acc4.w += v.w;
            }
        } else if (KIND == 8) {     // FADD2
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) y[i] = __fadd2_rn(y[i], a2);
        } else if (KIND == 9) {     // FMUL2
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) y[i] = __fmul2_rn(y[i], a2);
        } else if (KIND == 4) {     // MUFU.EX2
#pragma unroll
            for (int i = 0; i < CH; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
        } else if (KIND == 6) {     // DADD
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) d[i] = d[i] + (double)a;
        } else if (KIND == 7) {     // MUFU.RSQ64H (the seed of the fp64 kernel's reciprocal square root)
#pragma unroll
            for (int i = 0; i < CH / 2; ++i) asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(d[i]));
        } else if (KIND >= 11 && KIND <= 15) {
            // the pair core's instruction mix per step (two pairs per lane): 24 FFMA2-class in two dependent
            // chains (Horner), plus 11: 2 MUFU.RSQ (single instruction, ftz)   12: + 2 x (FSETP + FSEL)
            // 13: + 2 broadcast LDS.128 feeding the chains   15: all of them   14: the chains alone
            float2 c0 = b2, c1 = b2;
            if (KIND == 13 || KIND == 15) {
                const float4 v = sh[it & 63], w = sh[(it + 7) & 63];
                c0 = make_float2(v.x, v.y);
                c1 = make_float2(w.z, w.w);
            }
#pragma unroll
            for (int r = 0; r < 12; ++r) {
                y[0] = __ffma2_rn(y[0], a2, c0);
                y[1] = __ffma2_rn(y[1], a2, c1);
            }
            if (KIND != 14) {
                asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[0]));
                asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[1]));
            }
            if (KIND == 12 || KIND == 15) {
                x[2] = x[2] < a ? x[3] : 0.f;
                x[4] = x[4] < b ? x[5] : 0.f;
            }
        }
    }
    float s = acc4.x + acc4.y + acc4.z + acc4.w;
#pragma unroll
    for (int i = 0; i < CH; ++i) s += x[i];
#pragma unroll
    for (int i = 0; i < CH / 2; ++i) s += y[i].x + y[i].y + (float)d[i];
    if (s == 123.456f) out[0] = s;   // keeps the chains alive
}

static int g_blocks_per_sm = 8;   // 8 x 256 threads = 16 warps per scheduler; kinds >= 100 use fewer

template <int KIND>
static cudaError_t run_probe(int sms, float* d_out, float* ms)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 8;   // g_blocks_per_sm of them resident per SM (dynamic shared memory limits it)
    const size_t dyn = g_blocks_per_sm >= 8 ? 0 : (size_t)(200 * 1024 / g_blocks_per_sm - 2048);
    cudaFuncSetAttribute(probe_kernel<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    probe_kernel<KIND><<<grid, 256, dyn>>>(d_out, 0.999f, 0.001f, 64);   // warm-up
    cudaEventRecord(e0);
    probe_kernel<KIND><<<grid, 256, dyn>>>(d_out, 0.999f, 0.001f, PROBE_ITERS);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}

}  // namespace photons

using namespace photons;

extern "C" int photons_peak_probe(int device, int kind, double* out)
{
    // kind + 100 * b: the same probe with only b (1..7) resident blocks of 8 warps per SM (occupancy sweep)
    g_blocks_per_sm = 8;
    if (kind >= 100) { g_blocks_per_sm = kind / 100; kind %= 100; }
    const bool known = (kind >= 0 && kind <= 9) || (kind >= 11 && kind <= 15);
    if (!out || !known || g_blocks_per_sm < 1 || g_blocks_per_sm > 8) return PHOTONS_EINVAL;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) {
        cudaGetLastError();
        return PHOTONS_ENODEVICE;
    }
    float* d_out = nullptr;
    if (cudaMalloc(&d_out, 16) != cudaSuccess) return PHOTONS_ENOMEM;
    float ms = 0;
    cudaError_t e = cudaSuccess;
    double lane_ops_per_thread_iter = 0;   // FMA = 1 op per lane; f32x2 = 2
    switch (kind) {
        case 0: e = run_probe<0>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 1: e = run_probe<1>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 2: e = run_probe<2>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH / 2; break;
        case 3: e = run_probe<3>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 4: e = run_probe<4>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 5: e = run_probe<5>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;     // LDS.128 per lane
        case 6: e = run_probe<6>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH / 2; break;
        case 7: e = run_probe<7>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH / 2; break;
        case 8: e = run_probe<8>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 9: e = run_probe<9>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = CH; break;
        case 11: e = run_probe<11>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = 48; break;
        case 12: e = run_probe<12>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = 48; break;
        case 13: e = run_probe<13>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = 48; break;
        case 14: e = run_probe<14>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = 48; break;
        default: e = run_probe<15>(prop.multiProcessorCount, d_out, &ms); lane_ops_per_thread_iter = 48; break;
    }
    cudaFree(d_out);
    if (e != cudaSuccess) return PHOTONS_ECUDA;
    const double threads = (double)prop.multiProcessorCount * 8 * 256;
    *out = threads * PROBE_ITERS * lane_ops_per_thread_iter / (ms * 1e-3);
    return PHOTONS_OK;
}
