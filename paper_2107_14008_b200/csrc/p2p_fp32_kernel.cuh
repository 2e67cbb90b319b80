// fp32 / mixed-precision P2P kernel (Alg. 1 + Alg. 2, the paper's SP run L206), written for sm_100a.
//
// Mapping:
//   CTA            one target leaf (Alg. 1 L96); its W warps split the leaf's source list
//   lane           T targets in registers; the warp is split into 32 T / maxleaf lane groups that take
//                  alternate source pairs (maxleaf 16: the two half-warps take the same 16
//                  targets and alternate source pairs)
//   source staging runs of contiguous source leaves, one TMA bulk copy each into a per-warp mbarrier ring
//   pair core      two sources per lane per step in packed fp32 (add/mul/fma.rn.f32x2 -> FADD2/FMUL2/FFMA2),
//                  one MUFU.RSQ per pair; sources are read as two broadcast LDS.128 per step
//   accumulation   fp32 per staged run, flushed into fp64 per-lane sums (two-level, A12)
//   exact path     optional (close_pair_radius > 0): a staged run whose fp32 partial acceleration on a target exceeds
//                  what one pair at close_pair_radius would give is re-evaluated in fp64 from the exact coordinates
//                  for that target by the whole warp (nothing per pair in the fast path: three compares per run)
//   units          lengths in units of Ctx::pscale (a power of two near r_cut), G m in units of Ctx::gmscale (a power
//                  of two >= max |G m|): exact rescalings that keep every fp32 intermediate in range whatever the
//                  caller's units are; the fp64 sums are scaled back when they are stored
#pragma once
#include "common.cuh"
#include "pipeline.cuh"

#ifndef PHOTONS_UNROLL_T1
#define PHOTONS_UNROLL_T1 8   // source pairs per loop iteration with one target per lane (measured on config 4:
                              // 2: 103.2 ms, 4: 96.3 ms, 8: 94.4 ms)
#endif
#ifndef PHOTONS_UNROLL_T2
#define PHOTONS_UNROLL_T2 4   // ... with two targets per lane (MAXLEAF 64 on config 4: 2: 122.0 ms, 4 with two CTAs of 256 per SM: 119.6 ms)
#endif
#ifndef PHOTONS_PRED_ACC
#define PHOTONS_PRED_ACC 1    // two targets per lane, full-warp groups: the cut as a predicate on scalar accumulation FFMAs
                              // instead of a select on the weight (config 4, MAXLEAF 64: 117.3 against 119.6 ms; with one target
                              // per lane it changes nothing at MAXLEAF 32 and costs 3 % at MAXLEAF 16, so it stays off there)
#endif
#ifndef PHOTONS_MINBLOCKS_T1
#define PHOTONS_MINBLOCKS_T1 2   // __launch_bounds__(256, .) of the kernels with one target per lane and full-warp groups (MAXLEAF 32):
                                 // 2 leaves the compiler the 96 registers it asks for (5 CTAs of 128 threads per SM); 3 caps it at 80
                                 // (6 CTAs) at the price of re-computed addresses and a local-memory phase bit per list entry.
                                 // Config 4, 2 against 3: POLY 89.8 / 90.6 ms, FUSED 96.6 / 97.9, MIXED 95.1 / 97.4, TABLE 512 99.9 / 99.8,
                                 // TABLE 4096 104.1 / 112.9.  Half-warp groups (MAXLEAF 16) keep 3: 84.1 / 82.8 ms, MIXED 102.9 / 98.3
#endif
#ifndef PHOTONS_MINBLOCKS_T2
#define PHOTONS_MINBLOCKS_T2 2   // __launch_bounds__(256, .) of the kernels with two targets per lane
#endif

namespace photons {

constexpr int MAX_RUN_LEAVES = 16;        // chunk_max / maxleaf at most (256 / 16)
// Added to every r^2 (kernel length units, r_cut in [1, 2)): self / coincident pairs then give w * 0 = 0 with a finite
// w (A7): 1/r^3 = 1e36 and G m <= 1 in kernel units, so w cannot overflow.  With Plummer softening (A23) eps^2 takes
// its place.
constexpr float R2_FLOOR = 1e-24f;
constexpr float MAGIC = 12582912.0f;     // 1.5 * 2^23: float -> nearest-integer trick for the table index

struct P32Args {
    const float* p32;          // n_slots/2 x {x0 x1 y0 y1 z0 z1 Gm0 Gm1}
    const double4* p64;        // n_slots x {x, y, z, G m}: exact coordinates for the exact path
    const double* ctr;         // n_leaves x 3: origin of each leaf's offsets (MIXED), else unused
    const int* slot_src;
    const long long* chunk_ptr;
    const uint2* chunks;
    const int* order;
    long long first;
    int maxleaf, log2m, chunk_max, mixed;
    float Lh, Ll, invL;        // box length in kernel units as an unevaluated sum of two floats (exact image shifts)
    float rcut2;               // kernel units; compared with r^2 + r2add
    float pth2;                // exact path: square of the run-partial acceleration that triggers it (kernel units); 0 = off
    float r2add;               // max(R2_FLOOR, eps^2): start value of every r^2 chain
    double gmu;                // UGM kernels (all G m equal): the common G m in kernel units, applied once per run
    double Ld, inv2rs_d, rcut2_d, eps2_d;   // caller units, for the exact path
    double inv_pscale;         // 1 / Ctx::pscale
    double oscale, inv_oscale; // kernel-unit sums -> caller units: gmscale / pscale^2
    float inv2rs;              // 1 / 2 r_s (kernel units)
    float tk;                  // POLY: t = r2 * tk - 1
    float ek, tmap;            // FUSED: exp(-x^2) = ex2(r2 * ek); t = r * tmap - 1 maps r in [0, r_cut] to [-1, 1]
    float pc[POLY_MAX_DEG + 1];
    float uk, h, rmax;         // TABLE: u = r * uk in node units, h = 3/n, rmax = radius of the last node
    int tn;
    const float2* table;
    void* out;
    int out_f32;
};

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
// one MUFU.RSQ, no denormal fix-up code: r^2 carries r2add >= R2_FLOOR, so it is never subnormal
__device__ __forceinline__ float rsq(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// one MUFU.EX2
__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }
// 8-byte shared-memory load from a 32-bit shared address
__device__ __forceinline__ float2 lds_f2(uint32_t addr)
{
    float2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

// ---------------------------------------------------------------------------------------------------------
// g-dependent part of the pair core: returns w = G m_j g(r) / r^3 for two pairs at once.
//   r2 : r^2 (+floor, clamped to r_close^2 when close pairs are on)
//   gm : G m_j
// The value is only meaningful inside r_cut: the caller replaces it by 0 beyond the cut with a select
// (FSEL, ALU pipe), which also discards the Inf/NaN the polynomial can produce far outside its range.
// Keeping the cut out of the arithmetic saves two FMA-pipe multiplies per pair.
// ---------------------------------------------------------------------------------------------------------

template <int DEG>
__device__ __forceinline__ float2 weight_poly(const P32Args& a, float2 r2, float2 gm)
{
    const float2 idr = f2(rsq(r2.x), rsq(r2.y));
    const float2 t = __ffma2_rn(r2, dup(a.tk), dup(-1.0f));          // s mapped to [-1, 1]
    float2 q = dup(a.pc[0]);
#pragma unroll
    for (int k = 1; k <= DEG; ++k) q = __ffma2_rn(q, t, dup(a.pc[k]));
    const float2 idr2 = __fmul2_rn(idr, idr);
    const float2 u = __ffma2_rn(idr2, idr, f2(-q.x, -q.y));          // 1/r^3 - Q(s)/(2 r_s)^3
    return __fmul2_rn(u, gm);
}

template <int DEG>
__device__ __forceinline__ float2 weight_fused(const P32Args& a, float2 r2, float2 gm)
{
    const float2 idr = f2(rsq(r2.x), rsq(r2.y));
    const float2 t = __ffma2_rn(__fmul2_rn(r2, idr), dup(a.tmap), dup(-1.0f));
    const float2 y = __fmul2_rn(r2, dup(a.ek));
    const float2 e = f2(ex2(y.x), ex2(y.y));
    float2 q = dup(a.pc[0]);
#pragma unroll
    for (int k = 1; k <= DEG; ++k) q = __ffma2_rn(q, t, dup(a.pc[k]));
    const float2 idr2 = __fmul2_rn(idr, idr);
    return __fmul2_rn(__fmul2_rn(q, e), __fmul2_rn(idr2, __fmul2_rn(idr, gm)));
}

template <int LEVEL, bool UGM>
__device__ __forceinline__ float2 weight_table(const P32Args& a, const float2* __restrict__ tab, float2 r2, float2 gm)
{
    const float2 idr = f2(rsq(r2.x), rsq(r2.y));
    // r clamped to the last node's radius (FMNMX, ALU pipe) so that the index stays in range; the nearest node (A14) by
    // the magic-number add folded into one FMA: u = r uk in node units, bits(u + 1.5 * 2^23) = bits(MAGIC) + node
    float2 r = __fmul2_rn(r2, idr);
    r = f2(fminf(r.x, a.rmax), fminf(r.y, a.rmax));
    const float2 um = __ffma2_rn(r, dup(a.uk), dup(MAGIC));
    const float2 fi = __fadd2_rn(um, dup(-MAGIC));
    const float2 xi = __fmul2_rn(fi, dup(a.h));
    const float2 eps = __ffma2_rn(r, dup(a.inv2rs), f2(-xi.x, -xi.y));        // x - x_i, one rounding
    // table address straight from the float's bit pattern: (bits << 3) + (base - (bits(MAGIC) << 3)), one LEA per lookup
    const uint32_t tab_bias = smem_u32(tab) - (0x4B400000u << 3);
    const float2 te0 = lds_f2(((uint32_t)__float_as_int(um.x) << 3) + tab_bias);
    const float2 te1 = lds_f2(((uint32_t)__float_as_int(um.y) << 3) + tab_bias);
    const float2 Ti = f2(te0.x, te1.x), Ei = f2(te0.y, te1.y);
    float2 T = Ti;
    if (LEVEL >= 1) {
        // Eq. 2: T = T_i + E_i eps (x_i^2 - x_i (x_i^2 - 1) eps + (2/3 x_i^4 - 5/3 x_i^2 + 1/3) eps^2 - ...)
        const float2 xi2 = __fmul2_rn(xi, xi);
        float2 poly = xi2;
        if (LEVEL >= 2) {
            const float2 c2 = __ffma2_rn(f2(-xi.x, -xi.y), xi2, xi);                 // -x_i (x_i^2 - 1)
            float2 inner = c2;
            if (LEVEL >= 3) {
                const float2 c3 = __ffma2_rn(__ffma2_rn(xi2, dup(2.0f / 3.0f), dup(-5.0f / 3.0f)), xi2, dup(1.0f / 3.0f));
                inner = __ffma2_rn(c3, eps, c2);
            }
            poly = __ffma2_rn(inner, eps, xi2);
        }
        T = __ffma2_rn(__fmul2_rn(Ei, eps), poly, Ti);
    }
    const float2 idr2 = __fmul2_rn(idr, idr);
    const float2 idr3 = __fmul2_rn(idr2, idr);
    return UGM ? __fmul2_rn(idr3, T) : __fmul2_rn(__fmul2_rn(idr3, T), gm);
}

// Eq. 1 by the CUDA library special functions (what the paper's §3.3 L121 calls expensive)
__device__ __forceinline__ float weight_direct1(const P32Args& a, float r2, float gm)
{
    const float idr = rsq(r2);
    const float x = r2 * idr * a.inv2rs;
    const float g = erfcf(x) + 1.1283791671f * x * expf(-x * x);
    return gm * g * (idr * idr * idr);
}

enum { GM_POLY = 0, GM_TABLE = 1, GM_DIRECT = 2, GM_FUSED = 3 };

template <int GKIND, int GPAR, bool UGM = false>
__device__ __forceinline__ float2 weight2(const P32Args& a, const float2* tab, float2 r2, float2 gm)
{
    float2 w;
    if (GKIND == GM_POLY) w = weight_poly<GPAR>(a, r2, gm);
    else if (GKIND == GM_TABLE) w = weight_table<GPAR, UGM>(a, tab, r2, gm);
    else if (GKIND == GM_FUSED) w = weight_fused<GPAR>(a, r2, gm);
    else w = f2(weight_direct1(a, r2.x, gm.x), weight_direct1(a, r2.y, gm.y));
    // the cut (A8) and, with it, everything the approximations do outside their range
    return f2(r2.x < a.rcut2 ? w.x : 0.f, r2.y < a.rcut2 ? w.y : 0.f);
}

// The same for NCH independent chains (targets x unrolled source pairs) at once.  The polynomial is a chain
// of dependent FFMA2s, one every ~4 clocks per warp; writing the Horner steps of all chains side by side
// keeps NCH of them in flight, which is what lets a few warps per scheduler saturate the FMA pipe.
// kc: the loop constants (polynomial coefficients, tk, r_cut^2) as one local object
struct LoopConst {
    float pc[POLY_MAX_DEG + 1];
    float tk, rcut2, r2add, ek, tmap, inv2rs;
};

// SEL = false: the cut is left to the caller (acc_cut below), w is the raw value
template <int GKIND, int GPAR, int NCH, bool SEL, bool UGM>
__device__ __forceinline__ void weights(const P32Args& a, const LoopConst& kc, const float2* tab, const float2 (&r2)[NCH],
                                        const float2 (&gm)[NCH], float2 (&w)[NCH])
{
    if (GKIND == GM_POLY) {
        float2 idr[NCH], t[NCH], q[NCH];
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            idr[c] = f2(rsq(r2[c].x), rsq(r2[c].y));
            t[c] = __ffma2_rn(r2[c], dup(kc.tk), dup(-1.0f));
            q[c] = __ffma2_rn(dup(kc.pc[0]), t[c], dup(kc.pc[1]));
        }
#pragma unroll
        for (int k = 2; k <= GPAR; ++k) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) q[c] = __ffma2_rn(q[c], t[c], dup(kc.pc[k]));
        }
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const float2 idr2 = __fmul2_rn(idr[c], idr[c]);
            const float2 u = __ffma2_rn(idr2, idr[c], f2(-q[c].x, -q[c].y));
            const float2 v = UGM ? u : __fmul2_rn(u, gm[c]);
            w[c] = SEL ? f2(r2[c].x < kc.rcut2 ? v.x : 0.f, r2[c].y < kc.rcut2 ? v.y : 0.f) : v;
        }
    } else if (GKIND == GM_FUSED) {
        // Eq. 1 evaluated directly, hand-fused: g = exp(-x^2) H(x) with H = erfcx(x) + 2x/sqrt(pi), smooth on [0, 3]:
        // one MUFU.EX2 for the Gaussian (its argument straight from r^2) and a degree-GPAR polynomial for H on the
        // FMA pipe, against the stock erfcf + expf of GM_DIRECT (5 MUFU + 1 FRND + ~55 FP32 instructions per pair)
        float2 idr[NCH], t[NCH], q[NCH], e[NCH];
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            idr[c] = f2(rsq(r2[c].x), rsq(r2[c].y));
            t[c] = __ffma2_rn(__fmul2_rn(r2[c], idr[c]), dup(kc.tmap), dup(-1.0f));
            const float2 y = __fmul2_rn(r2[c], dup(kc.ek));
            e[c] = f2(ex2(y.x), ex2(y.y));
            q[c] = __ffma2_rn(dup(kc.pc[0]), t[c], dup(kc.pc[1]));
        }
#pragma unroll
        for (int k = 2; k <= GPAR; ++k) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) q[c] = __ffma2_rn(q[c], t[c], dup(kc.pc[k]));
        }
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
            const float2 idr2 = __fmul2_rn(idr[c], idr[c]);
            const float2 v = __fmul2_rn(__fmul2_rn(q[c], e[c]), __fmul2_rn(idr2, UGM ? idr[c] : __fmul2_rn(idr[c], gm[c])));
            w[c] = SEL ? f2(r2[c].x < kc.rcut2 ? v.x : 0.f, r2[c].y < kc.rcut2 ? v.y : 0.f) : v;
        }
    } else {
#pragma unroll
        for (int c = 0; c < NCH; ++c) w[c] = weight2<GKIND, GPAR, UGM>(a, tab, r2[c], gm[c]);    // (selects inside)
    }
}

// The cut (A8) as a predicate on the accumulation: acc += w d iff r2 < rcut2 - one FSETP and three predicated scalar
// FFMAs per pair, against FSETP + FSEL and 1.5 FFMA2: the same FMA-pipe time and one issue slot less.  A w that is
// Inf/NaN far outside the approximation's range is never touched.
__device__ __forceinline__ void acc_cut(float& ax, float& ay, float& az, float w, float dx, float dy, float dz, float r2, float rcut2)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f32 p, %7, %8;\n\t@p fma.rn.f32 %0, %3, %4, %0;\n\t@p fma.rn.f32 %1, %3, %5, %1;\n\t"
        "@p fma.rn.f32 %2, %3, %6, %2;\n\t}"
        : "+f"(ax), "+f"(ay), "+f"(az) : "f"(w), "f"(dx), "f"(dy), "f"(dz), "f"(r2), "f"(rcut2));
}

// Exact path (A12): one target against one staged run of sources, in fp64 from the exact coordinates with
// the library's erfc / exp — the oracle's arithmetic.  The whole warp works on it: the run's share of the target's owner
// lane — source PAIRS first, first + step, ... (sources 2p and 2p + 1), exactly what the fast path dealt that lane — is
// numbered m = 0, 1, ... and lane l takes m = l, l + 32, ...; the 32 partial sums are added in a fixed butterfly order,
// so every lane returns the same, reproducible sum.  Returns the acceleration in caller units.
// (scalars by value: a reference to the kernel's parameter block would make the compiler copy it to local memory)
static __device__ __noinline__ double3 exact_run(const double4* __restrict__ p64, double Ld, double eps2_d, double rcut2_d,
                                                 double inv2rs_d, int tslot, uint2 e, int first, int step)
{
    const int lane = threadIdx.x & 31;
    const int ns = (int)(e.y & 0xffffu);
    const bool per_pair = (e.y & ENTRY_PER_PAIR) != 0;
    const double sx = Ld * ((int)((e.y >> 16) & 3u) - 1), sy = Ld * ((int)((e.y >> 18) & 3u) - 1), sz = Ld * ((int)((e.y >> 20) & 3u) - 1);
    const double4 pi = p64[tslot];
    double ax = 0, ay = 0, az = 0;
    for (int m = lane;; m += 32) {
        const int j = 2 * (first + step * (m >> 1)) + (m & 1);
        if (j >= ns) break;
        const double4 pj = p64[e.x + j];
        double dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        if (per_pair) {
            dx -= Ld * rint(dx / Ld); dy -= Ld * rint(dy / Ld); dz -= Ld * rint(dz / Ld);
        } else {
            dx += sx; dy += sy; dz += sz;
        }
        const double r2 = dx * dx + dy * dy + dz * dz;
        const double r2e = r2 + eps2_d;
        if (r2 > 0.0 && r2e < rcut2_d) {
            const double r = sqrt(r2e);
            const double x = r * inv2rs_d;
            const double w = pj.w * (erfc(x) + 1.1283791670955125739 * x * exp(-x * x)) / (r2e * r);
            ax += w * dx; ay += w * dy; az += w * dz;
        }
    }
    __syncwarp();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ax += __shfl_xor_sync(0xffffffffu, ax, o);
        ay += __shfl_xor_sync(0xffffffffu, ay, o);
        az += __shfl_xor_sync(0xffffffffu, az, o);
    }
    return make_double3(ax, ay, az);
}

// ---------------------------------------------------------------------------------------------------------

template <int T, int HS, bool MIXED, int GKIND, int GPAR, bool UGM = false>
__global__ void __launch_bounds__(256, T == 1 ? (HS == 1 ? PHOTONS_MINBLOCKS_T1 : 3) : T == 2 ? PHOTONS_MINBLOCKS_T2 : 1) p2p_fp32_kernel(P32Args a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, W = blockDim.x >> 5;
    // the leaf size is fixed by the mapping (T targets per lane, HS lane groups): a build-time constant for the MIXED
    // kernels' walk over the source leaves of a run (trip counts and shifts known to the compiler)
    constexpr int MC = T * 32 / HS;
    constexpr int LOG2_MC = MC == 16 ? 4 : MC == 32 ? 5 : MC == 64 ? 6 : 7;
    const int M = MIXED ? MC : a.maxleaf;
    const int stage_bytes = a.chunk_max * 16;
    unsigned char* ring = smem_raw + (size_t)warp * N_STAGES * stage_bytes;
    unsigned char* tail = smem_raw + (size_t)W * N_STAGES * stage_bytes;
    uint64_t* bars = reinterpret_cast<uint64_t*>(tail) + warp * N_STAGES;
    // MIXED: per stage, the origin of every source leaf of the staged run minus the target leaf's origin
    // (the region exists in the MIXED kernels only; the others keep the barriers' plain size)
    const int bars_bytes = MIXED ? ((W * N_STAGES * 8 + 15) & ~15) : W * N_STAGES * 8;
    float4* cshift = reinterpret_cast<float4*>(tail + bars_bytes) + warp * N_STAGES * MAX_RUN_LEAVES;
    unsigned char* tail2 = tail + bars_bytes + (MIXED ? (size_t)W * N_STAGES * MAX_RUN_LEAVES * 16 : 0);
    double* red = reinterpret_cast<double*>(tail2);                             // W x T x 32 x 3 doubles
    float2* tab = reinterpret_cast<float2*>(tail2 + (size_t)W * T * 32 * 3 * 8);

    const long long leaf = a.order[a.first + blockIdx.x];
    const long long slot0 = leaf * M;
    // HS groups of LG = 32/HS lanes: a lane owns T targets (lane-in-group + LG t), the groups take alternate
    // source pairs.  MAXLEAF = T * LG.  More targets per lane = fewer shared-memory reads per pair.
    constexpr int LG = 32 / HS;
    const int half = HS > 1 ? lane / LG : 0;
    const int pstep = HS;

    if (GKIND == GM_TABLE) {   // the interpolation table lives in shared memory (Fig. 1)
        for (int i = threadIdx.x; i <= a.tn; i += blockDim.x) tab[i] = a.table[i];
        __syncthreads();
    }

    LoopConst kc;
    if (GKIND == GM_POLY || GKIND == GM_FUSED) {
#pragma unroll
        for (int k = 0; k <= GPAR; ++k) kc.pc[k] = a.pc[k];
    }
    kc.ek = a.ek; kc.tmap = a.tmap; kc.inv2rs = a.inv2rs;
    kc.tk = a.tk;
    kc.rcut2 = a.rcut2;
    kc.r2add = a.r2add;

    // targets -> registers (Alg. 1 L99)
    float tx[T], ty[T], tz[T];
    double ax[T], ay[T], az[T];
    int tslot[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        const int l = (lane % LG) + LG * t;
        tslot[t] = (int)slot0 + l;
        const float* b = a.p32 + (size_t)(tslot[t] >> 1) * 8 + (tslot[t] & 1);
        tx[t] = b[0]; ty[t] = b[2]; tz[t] = b[4];
        ax[t] = ay[t] = az[t] = 0.0;
    }
    double cix = 0, ciy = 0, ciz = 0;
    if (MIXED) { cix = a.ctr[3 * leaf]; ciy = a.ctr[3 * leaf + 1]; ciz = a.ctr[3 * leaf + 2]; }

    const long long c0 = a.chunk_ptr[leaf], c1 = a.chunk_ptr[leaf + 1];
    const long long n_all = c1 - c0;
    const int n_my = n_all > warp ? (int)((n_all - warp + W - 1) / W) : 0;

    if (lane == 0) {
        for (int s = 0; s < N_STAGES; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncwarp();
    // Interaction-list entries of this warp, 32 at a time in registers (one per lane, coalesced when W == 1)
    // and one batch ahead, so that neither the producer nor the consumer ever waits on a global load.
    const uint2* my_chunks = a.chunks + c0 + warp;
    auto load_batch = [&](int b) {
        const int idx = b * 32 + lane;
        return idx < n_my ? __ldg(&my_chunks[(long long)idx * W]) : make_uint2(0u, 0u);
    };
    uint2 dcur = load_batch(0), dnext = load_batch(1);
    auto entry = [&](int k, int cur_batch) {
        const uint2 v = (k >> 5) == cur_batch ? dcur : dnext;       // warp-uniform choice
        return make_uint2(__shfl_sync(0xffffffffu, v.x, k & 31), __shfl_sync(0xffffffffu, v.y, k & 31));
    };
    // stage st of the ring: shared-memory addresses kept in registers, stage index and phase bit stepped by hand
    const uint32_t ring_u32 = smem_u32(ring), bars_u32 = smem_u32(bars);
    auto issue = [&](int k, int cur_batch, int st) {
        const uint2 mine = (k >> 5) == cur_batch ? dcur : dnext;       // warp-uniform choice; lane (k & 31) holds entry k
        if (MIXED) {
            // origin differences in fp64, rounded once (A15); computed when the copy is issued, N_STAGES runs
            // ahead of their use, so the global loads of the origins are off the critical path
            const uint2 e = make_uint2(__shfl_sync(0xffffffffu, mine.x, k & 31), __shfl_sync(0xffffffffu, mine.y, k & 31));
            const int nleaf = (int)((e.y & 0xffffu) >> LOG2_MC);
            if (lane < nleaf) {
                const long long jl = (long long)(e.x >> LOG2_MC) + lane;
                const int sxi = (int)((e.y >> 16) & 3u) - 1, syi = (int)((e.y >> 18) & 3u) - 1, szi = (int)((e.y >> 20) & 3u) - 1;
                cshift[st * MAX_RUN_LEAVES + lane] = make_float4((float)(((a.ctr[3 * jl] + a.Ld * sxi) - cix) * a.inv_pscale),
                                                                 (float)(((a.ctr[3 * jl + 1] + a.Ld * syi) - ciy) * a.inv_pscale),
                                                                 (float)(((a.ctr[3 * jl + 2] + a.Ld * szi) - ciz) * a.inv_pscale), 0.f);
            }
            __syncwarp();   // the stores above are read by other lanes (first N_STAGES entries: before any loop barrier)
        }
        if (lane == (k & 31)) {      // the lane that holds the entry issues its copy: no shuffle on the producer side
            const uint32_t bytes = (mine.y & 0xffffu) * 16u;
            mbar_expect_tx_u32(bars_u32 + 8u * st, bytes);
            bulk_g2s_u32(ring_u32 + (uint32_t)(st * stage_bytes), a.p32 + (size_t)mine.x * 4, bytes, bars_u32 + 8u * st);
        }
    };
    for (int k = 0; k < N_STAGES && k < n_my; ++k) issue(k, 0, k);

    // stage and phase bit of entry k: with a power-of-two ring depth they are bit fields of k (no loop-carried state)
    constexpr bool POW2_STAGES = (N_STAGES & (N_STAGES - 1)) == 0;
    constexpr int LOG2_STAGES = N_STAGES == 2 ? 1 : N_STAGES == 4 ? 2 : N_STAGES == 8 ? 3 : 0;
    int st = 0;
    uint32_t phase = 0;
    for (int k = 0; k < n_my; ++k) {
        if (POW2_STAGES) { st = k & (N_STAGES - 1); phase = (uint32_t)(k >> LOG2_STAGES) & 1u; }
        const int batch = k >> 5;
        if ((k & 31) == 0 && k > 0) { dcur = dnext; dnext = load_batch(batch + 1); }
        const uint2 e = entry(k, batch);
        mbar_wait_u32(bars_u32 + 8u * st, phase);
        const int ns = (int)(e.y & 0xffffu);
        const float4* src = reinterpret_cast<const float4*>(ring + (size_t)st * stage_bytes);
        const bool per_pair = (e.y & ENTRY_PER_PAIR) != 0;
        const int sxi = (int)((e.y >> 16) & 3u) - 1, syi = (int)((e.y >> 18) & 3u) - 1, szi = (int)((e.y >> 20) & 3u) - 1;
        // MIXED: every source leaf of the run has its own origin; ABS: one block = the whole run
        const int blk = MIXED ? M : ns;

        float px[T], py[T], pz[T];       // fp32 partial sums of this run (level 1 of the accumulation)
#pragma unroll
        for (int t = 0; t < T; ++t) px[t] = py[t] = pz[t] = 0.f;

        // the same, packed (the two sources of a pair accumulate side by side).  MIXED: one set for all the blocks
        // (source leaves) of the run; ABS: one block per run, declared where it is used (shorter live ranges)
        float2 pax_run[T], pay_run[T], paz_run[T];
#pragma unroll
        for (int t = 0; t < T; ++t) pax_run[t] = pay_run[t] = paz_run[t] = dup(0.f);

        for (int b0 = 0; b0 < ns; b0 += blk) {
            // targets as seen from this block: d = (r_j + sadd) - q
            float qx[T], qy[T], qz[T];
            float sax = 0.f, say = 0.f, saz = 0.f;
            float4 dc = make_float4(0.f, 0.f, 0.f, 0.f);
            if (MIXED) {
                dc = cshift[st * MAX_RUN_LEAVES + (b0 >> LOG2_MC)];
#pragma unroll
                for (int t = 0; t < T; ++t) { qx[t] = tx[t] - dc.x; qy[t] = ty[t] - dc.y; qz[t] = tz[t] - dc.z; }
            } else {
                // L = Lh + Ll (two floats).  s = +1: move the target by -L: t - Lh is exact (it sits in the upper half
                // of the box), then - Ll; s = -1: move the sources by -Lh per pair (exact for the same reason) and
                // the target by +Ll.  With a box length that fp32 holds exactly Ll = 0.
                if (((e.y >> 16) & 0x3fu) == 0x15u) {        // no image shift on any axis (most entries): warp-uniform
#pragma unroll
                    for (int t = 0; t < T; ++t) { qx[t] = tx[t]; qy[t] = ty[t]; qz[t] = tz[t]; }
                } else {
                    sax = sxi < 0 ? -a.Lh : 0.f; say = syi < 0 ? -a.Lh : 0.f; saz = szi < 0 ? -a.Lh : 0.f;
#pragma unroll
                    for (int t = 0; t < T; ++t) {
                        qx[t] = sxi > 0 ? (tx[t] - a.Lh) - a.Ll : sxi < 0 ? tx[t] + a.Ll : tx[t];
                        qy[t] = syi > 0 ? (ty[t] - a.Lh) - a.Ll : syi < 0 ? ty[t] + a.Ll : ty[t];
                        qz[t] = szi > 0 ? (tz[t] - a.Lh) - a.Ll : szi < 0 ? tz[t] + a.Ll : tz[t];
                    }
                }
            }
            const bool seam = (sax != 0.f) | (say != 0.f) | (saz != 0.f);
            const float4* s4 = src + b0;             // two float4 per source pair
            const int np = blk / 2;

            if (per_pair) {
                // degenerate geometry (tiny N, leaves spanning half the box): minimum image per pair.  The image shift is
                // applied to an operand it is exact for, never to the rounded difference: ABS: x_j - x_i > L/2 puts x_j
                // in the upper half of the box, so x_j - Lh is exact (and x_i - Lh when the sign is the other way);
                // MIXED: to the origin difference.  A close pair across a box face then keeps its separation to one ulp
                // of the separation, not of the box length.
                auto image = [&](float xj, float xt, float dcx) {
                    if (MIXED) {
                        const float off = xj - xt;
                        const float i = rintf((off + dcx) * a.invL);
                        return off + fmaf(-a.Ll, i, fmaf(-a.Lh, i, dcx));
                    }
                    const float i = rintf((xj - xt) * a.invL);
                    const float xs = i > 0.f ? xj - a.Lh : xj, ts = i < 0.f ? xt - a.Lh : xt;
                    return fmaf(-a.Ll, i, xs - ts);
                };
                for (int p = half; p < np; p += pstep) {
                    const float4 A = s4[2 * p], B = s4[2 * p + 1];
#pragma unroll
                    for (int t = 0; t < T; ++t) {
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            const float dx = image(hh ? A.y : A.x, tx[t], dc.x), dy = image(hh ? A.w : A.z, ty[t], dc.y),
                                        dz = image(hh ? B.y : B.x, tz[t], dc.z);
                            float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, a.r2add)));
                            // equal-mass kernels: a padding slot sits at PAD_FAR instead of carrying zero mass, and MIXED
                            // wraps the offset by whole box lengths here - keep it beyond the cut
                            if (UGM && MIXED && (hh ? A.y : A.x) >= 0.5f * PAD_FAR) r2 = 3.0e30f;
                            const float2 w = weight2<GKIND, GPAR>(a, tab, dup(r2), dup(UGM ? 1.f : hh ? B.w : B.z));
                            px[t] = fmaf(w.x, dx, px[t]); py[t] = fmaf(w.x, dy, py[t]); pz[t] = fmaf(w.x, dz, pz[t]);
                        }
                    }
                }
            } else {
                float2 nqx[T], nqy[T], nqz[T], pax_blk[T], pay_blk[T], paz_blk[T];
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    nqx[t] = dup(-qx[t]); nqy[t] = dup(-qy[t]); nqz[t] = dup(-qz[t]);
                    pax_blk[t] = pay_blk[t] = paz_blk[t] = dup(0.f);
                }
                float2 (&pax)[T] = MIXED ? pax_run : pax_blk;
                float2 (&pay)[T] = MIXED ? pay_run : pay_blk;
                float2 (&paz)[T] = MIXED ? paz_run : paz_blk;
                const float2 sx2 = dup(sax), sy2 = dup(say), sz2 = dup(saz);
                // U source pairs x T targets = NCH independent chains per iteration
                // (with lane groups the leaf's np = maxleaf/2 source pairs are shared out, so fewer fit in one iteration)
                constexpr int U = T == 1 ? (HS == 1 ? PHOTONS_UNROLL_T1 : (PHOTONS_UNROLL_T1 / 2 > 4 ? 4 : PHOTONS_UNROLL_T1 / 2)) : T == 2 ? (HS == 4 ? 2 : PHOTONS_UNROLL_T2) : 1;
                static_assert(U * HS <= 16 * T / HS, "a leaf's source pairs must fill whole iterations");
                constexpr int NCH = U * T;
                auto step = [&](const int p, const bool with_seam) {
                    float2 dx[NCH], dy[NCH], dz[NCH], r2[NCH], gm[NCH], w[NCH];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const float4 A = s4[2 * (p + u * pstep)];
                        float4 B;
                        if (UGM) {   // all G m equal: only {z0, z1} of the second half is read (one LDS.64)
                            const float2 Bz = *reinterpret_cast<const float2*>(&s4[2 * (p + u * pstep) + 1]);
                            B = make_float4(Bz.x, Bz.y, 0.f, 0.f);
                        } else {
                            B = s4[2 * (p + u * pstep) + 1];
                        }
                        float2 xj = f2(A.x, A.y), yj = f2(A.z, A.w), zj = f2(B.x, B.y);
                        if (with_seam) { xj = __fadd2_rn(xj, sx2); yj = __fadd2_rn(yj, sy2); zj = __fadd2_rn(zj, sz2); }
#pragma unroll
                        for (int t = 0; t < T; ++t) {
                            const int c = u * T + t;
                            dx[c] = __fadd2_rn(xj, nqx[t]); dy[c] = __fadd2_rn(yj, nqy[t]); dz[c] = __fadd2_rn(zj, nqz[t]);
                            gm[c] = f2(B.z, B.w);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < NCH; ++c) {
                        r2[c] = __ffma2_rn(dx[c], dx[c], __ffma2_rn(dy[c], dy[c], __ffma2_rn(dz[c], dz[c], dup(kc.r2add))));
                    }
                    constexpr bool PRED = PHOTONS_PRED_ACC && T == 2 && HS == 1 && (GKIND == GM_POLY || GKIND == GM_FUSED);
                    weights<GKIND, GPAR, NCH, !PRED, UGM>(a, kc, tab, r2, gm, w);
#pragma unroll
                    for (int u = 0; u < U; ++u) {
#pragma unroll
                        for (int t = 0; t < T; ++t) {
                            const int c = u * T + t;
                            if (PRED) {
                                acc_cut(pax[t].x, pay[t].x, paz[t].x, w[c].x, dx[c].x, dy[c].x, dz[c].x, r2[c].x, kc.rcut2);
                                acc_cut(pax[t].y, pay[t].y, paz[t].y, w[c].y, dx[c].y, dy[c].y, dz[c].y, r2[c].y, kc.rcut2);
                            } else {
                                pax[t] = __ffma2_rn(w[c], dx[c], pax[t]);
                                pay[t] = __ffma2_rn(w[c], dy[c], pay[t]);
                                paz[t] = __ffma2_rn(w[c], dz[c], paz[t]);
                            }
                        }
                    }
                };
                // np is a multiple of U * pstep for every leaf size (np = 8 with two half-warps, else >= 16)
                if (seam) {
                    for (int p = half; p < np; p += pstep * U) step(p, true);
                } else {
                    for (int p = half; p < np; p += pstep * U) step(p, false);
                }
                if (!MIXED) {
#pragma unroll
                    for (int t = 0; t < T; ++t) { px[t] = pax[t].x + pax[t].y; py[t] = pay[t].x + pay[t].y; pz[t] = paz[t].x + paz[t].y; }
                }
            }
        }
        if (MIXED) {     // (px is non-zero only after the per-pair path, which does not use the packed sums)
#pragma unroll
            for (int t = 0; t < T; ++t) {
                px[t] += pax_run[t].x + pax_run[t].y; py[t] += pay_run[t].x + pay_run[t].y; pz[t] += paz_run[t].x + paz_run[t].y;
            }
        }
        // Exact path: a run whose partial sum is larger than one pair at close_pair_radius would give holds a pair
        // close enough for fp32 rounding (3 ulp of the rsqrt in 1/r^3) to show against the tolerance: redo the run
        // in fp64 for this target and drop the fp32 partial.
        if (a.pth2 > 0.f) {
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const bool trig = fmaf(px[t], px[t], fmaf(py[t], py[t], pz[t] * pz[t])) > a.pth2;
                unsigned todo = __ballot_sync(0xffffffffu, trig);
                while (todo) {                       // warp-uniform: the warp redoes the run for one owner lane at a time
                    const int owner = __ffs(todo) - 1;
                    todo &= todo - 1;
                    const int ts = __shfl_sync(0xffffffffu, tslot[t], owner);
                    const int fo = HS > 1 ? owner / LG : 0;
                    const double3 x = exact_run(a.p64, a.Ld, a.eps2_d, a.rcut2_d, a.inv2rs_d, ts, e, fo, pstep);
                    if (lane == owner) {
                        ax[t] += x.x * a.inv_oscale; ay[t] += x.y * a.inv_oscale; az[t] += x.z * a.inv_oscale;
                        px[t] = py[t] = pz[t] = 0.f;
                    }
                }
            }
        }
        // level 2 of the accumulation: flush the run's fp32 partial sums into the fp64 sums
#pragma unroll
        for (int t = 0; t < T; ++t) {
            if (UGM) { ax[t] = fma((double)px[t], a.gmu, ax[t]); ay[t] = fma((double)py[t], a.gmu, ay[t]); az[t] = fma((double)pz[t], a.gmu, az[t]); }
            else { ax[t] += (double)px[t]; ay[t] += (double)py[t]; az[t] += (double)pz[t]; }
        }
        __syncwarp();
        if (k + N_STAGES < n_my) issue(k + N_STAGES, batch, st);
        if (!POW2_STAGES) { if (++st == N_STAGES) { st = 0; phase ^= 1u; } }
    }

#pragma unroll
    for (int o = 16; o >= LG; o >>= 1) {     // add the groups' partial sums (fixed order)
#pragma unroll
        for (int t = 0; t < T; ++t) {
            ax[t] += __shfl_xor_sync(0xffffffffu, ax[t], o);
            ay[t] += __shfl_xor_sync(0xffffffffu, ay[t], o);
            az[t] += __shfl_xor_sync(0xffffffffu, az[t], o);
        }
    }
    // sum the warps' partial accelerations in a fixed order (deterministic), then scatter to caller order
    if (W > 1) {
#pragma unroll
        for (int t = 0; t < T; ++t) {
            double* r = red + ((size_t)(warp * T + t) * 32 + lane) * 3;
            r[0] = ax[t]; r[1] = ay[t]; r[2] = az[t];
        }
        __syncthreads();
        if (warp != 0) return;
#pragma unroll
        for (int t = 0; t < T; ++t)
            for (int w = 1; w < W; ++w) {
                const double* r = red + ((size_t)(w * T + t) * 32 + lane) * 3;
                ax[t] += r[0]; ay[t] += r[1]; az[t] += r[2];
            }
    }
#pragma unroll
    for (int t = 0; t < T; ++t) {
        if (lane >= LG) continue;
        const int dst = a.slot_src[tslot[t]];
        if (dst < 0) continue;
        // back to the caller's units (a power of two: exact)
        const double ox = ax[t] * a.oscale, oy = ay[t] * a.oscale, oz = az[t] * a.oscale;
        if (a.out_f32) {
            float* o = reinterpret_cast<float*>(a.out) + 3 * (size_t)dst;
            o[0] = (float)ox; o[1] = (float)oy; o[2] = (float)oz;
        } else {
            double* o = reinterpret_cast<double*>(a.out) + 3 * (size_t)dst;
            o[0] = ox; o[1] = oy; o[2] = oz;
        }
    }
}

// host side ------------------------------------------------------------------------------------------------
void fill_p32_args(Ctx* c, P32Args& a, long long first, void* out, bool out_f32);
size_t p32_smem_bytes(Ctx* c, int T);

template <int GKIND, int GPAR>
static int launch_p32_shape(Ctx* c, const P32Args& a, long long count, cudaStream_t st)
{
    const int W = c->p.warps_per_leaf;
    const int M = c->p.maxleaf;
    const int T = c->p.targets_per_lane;
    const size_t smem = p32_smem_bytes(c, T);
    void (*kern)(P32Args) = nullptr;
    const bool mixed = c->p.precision == PHOTONS_MIXED;
    const bool ugm = c->ugm;     // equal masses: G m out of the pair core (never DIRECT: build_leaves)
    constexpr bool HAS_UGM = GKIND != GM_DIRECT;
#define PH_SHAPE(TT, HH) (mixed ? (ugm ? p2p_fp32_kernel<TT, HH, true, GKIND, GPAR, HAS_UGM> : p2p_fp32_kernel<TT, HH, true, GKIND, GPAR>) \
                                : (ugm ? p2p_fp32_kernel<TT, HH, false, GKIND, GPAR, HAS_UGM> : p2p_fp32_kernel<TT, HH, false, GKIND, GPAR>))
    switch (M * 8 + T) {   // (MAXLEAF, targets per lane) -> (T, lane groups)
        case 16 * 8 + 1: kern = PH_SHAPE(1, 2); break;
        case 16 * 8 + 2: kern = PH_SHAPE(2, 4); break;
        case 32 * 8 + 1: kern = PH_SHAPE(1, 1); break;
        case 32 * 8 + 2: kern = PH_SHAPE(2, 2); break;
        case 64 * 8 + 2: kern = PH_SHAPE(2, 1); break;
        case 128 * 8 + 4: kern = PH_SHAPE(4, 1); break;
        default: return fail(c, PHOTONS_EINVAL, "targets_per_lane %d is not available for maxleaf %d", T, M);
    }
#undef PH_SHAPE
    PH_CUDA(c, opt_in_smem(c, reinterpret_cast<const void*>(kern), smem));
    kern<<<(unsigned)count, 32 * W, smem, st>>>(a);
    ++c->launches;
    PH_CUDA(c, cudaGetLastError());
    return PHOTONS_OK;
}

int launch_p32_poly(Ctx* c, const P32Args& a, long long count, cudaStream_t st);
template <int DEG>
int launch_p32_poly_deg(Ctx* c, const P32Args& a, long long count, cudaStream_t st);
int launch_p32_table(Ctx* c, const P32Args& a, long long count, cudaStream_t st);
int launch_p32_direct(Ctx* c, const P32Args& a, long long count, cudaStream_t st);
int launch_p32_fused(Ctx* c, const P32Args& a, long long count, cudaStream_t st);

}  // namespace photons
