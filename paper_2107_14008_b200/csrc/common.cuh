// Shared declarations of the photons library (product code; nothing here is used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/photons.h"

namespace photons {

// Interaction-list entry ("chunk"): a run of contiguous source leaves staged as one bulk copy.
//   .x = first particle slot of the run (leaf * maxleaf)
//   .y = bits 0..15 number of slots in the run; bits 16-17, 18-19, 20-21 = sx + 1, sy + 1, sz + 1 with
//        s in {-1, 0, +1} the box lengths added to the source; bit 22 = take the minimum image per pair
//        instead (degenerate geometry, A10)
constexpr unsigned ENTRY_PER_PAIR = 1u << 22;
__host__ __device__ inline unsigned entry_pack(int slots, int sx, int sy, int sz, bool per_pair)
{
    return per_pair ? ((unsigned)slots | (1u << 16) | (1u << 18) | (1u << 20) | ENTRY_PER_PAIR)
                    : ((unsigned)slots | ((unsigned)(sx + 1) << 16) | ((unsigned)(sy + 1) << 18) | ((unsigned)(sz + 1) << 20));
}
// the shift code of include/photons.h: (sx+1) + 3 (sy+1) + 9 (sz+1), or 27 = per pair
__host__ __device__ inline int entry_shift_code(unsigned y)
{
    if (y & ENTRY_PER_PAIR) return 27;
    return (int)((y >> 16) & 3u) + 3 * (int)((y >> 18) & 3u) + 9 * (int)((y >> 20) & 3u);
}
#ifndef PHOTONS_STAGES
#define PHOTONS_STAGES 3
#endif
constexpr int N_STAGES = PHOTONS_STAGES;   // shared-memory ring depth per warp

struct GTable {                 // Eq. 2 table
    int n = 0;                  // intervals over x in [0, 3]; n + 1 nodes
    int level = 2;
    float2* d_TE = nullptr;     // {T_i, E_i} per node (fp32)
    double2* d_TE64 = nullptr;  // fp64 copy for the fp64 path
    double* d_C64 = nullptr;    // coefficient layout (PHOTONS_TABLE_COEF): 5 doubles per node, T^(k)(x_i) h^k / k!
    double* d_Q64 = nullptr;    // PHOTONS_TABLE_QUAD: {T_i, E_i, bracket of T[3], bracket of T[4]} per node
};

constexpr int POLY_MAX_DEG = 20;

// Grow-only device workspace: one buffer per role, allocated on first use and kept until photons_destroy, so
// that repeated set_particles / build_leaves / short_range_acc steps do no cudaMalloc / cudaFree at all.
enum WsSlot {
    WS_POS, WS_MASS, WS_IN_POS, WS_IN_MASS, WS_FLAG, WS_OUT,
    WS_PERM, WS_ORB_P0, WS_ORB_P1, WS_ORB_KEYS, WS_ORB_KEYS2, WS_ORB_VALS, WS_ORB_VALS2, WS_ORB_LO, WS_ORB_HI, WS_CUB_TMP,
    WS_LEAF_CNT, WS_NODE_LO, WS_NODE_HI, WS_NODE_BOX32, WS_LEAF_CTR, WS_SLOT_SRC, WS_P64, WS_P32,
    WS_SEL_NODE, WS_SEL_CNT, WS_SEL_Q0, WS_SEL_C0, WS_SEL_HIST, WS_SEL_NODEVAR, WS_SEL_CNT2, WS_SEL_BASE2, WS_SEL_LO2, WS_SEL_HI2,
    WS_LIST_NCH, WS_LIST_WORK, WS_LIST_TOT, WS_LIST_STASH, WS_LIST_RESUME, WS_CHUNK_PTR, WS_CHUNKS, WS_ORDER, WS_ORDER_KEYS, WS_ORDER_KEYS2, WS_ORDER_VALS,
    WS_COUNT
};
// fp32 coordinate (kernel units, r_cut in [1, 2)) of a padding slot in the equal-mass kernels: r^2 ~ 3e30 stays finite
constexpr float PAD_FAR = 1.0e15f;

struct DevBuf { void* p = nullptr; size_t cap = 0; };

struct Ctx {
    photons_params p{};
    double r_s = 0, r_cut = 0;
    // units of the fp32 / mixed kernels (powers of two, so that rescaling fp32 data is exact): lengths are divided by
    // pscale (the power of two just below r_cut), G m by gmscale (the power of two >= max |G m|); sums are scaled back
    // in fp64 by gmscale / pscale^2 when they are stored
    double pscale = 1.0, gmscale = 1.0;
    double gm_max = 0.0;                 // max |G m_j| of the current particle set
    double gm_uniform = 0.0;             // G m if every particle has the same mass, else 0
    bool ugm = false;                    // the current leaves were packed for the equal-mass fp32 kernels (build_leaves)
    int sm_count = 0;
    std::vector<const void*> smem_opted;  // kernels whose dynamic shared-memory limit has been raised already
    std::vector<cudaStream_t> streams;   // [0] = main stream (the caller's after photons_set_stream)
    cudaStream_t own_stream0 = nullptr;  // the stream created for slot 0 (destroyed with the context)
    long long launches = 0;              // kernels of this library launched so far (cub's are not counted)
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaEvent_t evb0 = nullptr, evb1 = nullptr;   // around the device work of build_leaves
    bool build_ms_pending = false;
    std::vector<cudaEvent_t> stream_done;

    // particles in caller order (wrapped into [0, L))
    long long n = 0;
    double* d_pos = nullptr;   // n x 3
    double* d_mass = nullptr;  // n

    // ORB / leaves
    bool leaves_built = false;
    int depth = 0;              // all leaves at this depth
    long long n_leaves = 0, n_slots = 0;
    uint32_t* d_perm = nullptr;     // sorted position -> caller index
    int* d_slot_src = nullptr;      // slot -> caller index, -1 for padding slots
    int* d_leaf_cnt = nullptr;      // real particles per leaf
    double* d_leaf_ctr = nullptr;   // n_leaves x 3 (mixed: origin of the fp32 offsets)
    double* d_node_lo = nullptr;    // (2 n_leaves - 1) x 3, heap order
    double* d_node_hi = nullptr;
    double4* d_p64 = nullptr;       // n_slots x {x, y, z, G m}   (fp64 path and exact close pairs)
    float* d_p32 = nullptr;         // n_slots/2 x {x0 x1 y0 y1 z0 z1 Gm0 Gm1}  (fp32 / mixed)
    long long* d_chunk_ptr = nullptr;  // n_leaves + 1
    uint2* d_chunks = nullptr;
    int* d_order = nullptr;         // target leaves, heaviest list first
    long long cap_chunks = 0;

    GTable table;
    int poly_deg = 0;
    float poly_c[POLY_MAX_DEG + 1]{};   // Q(s)/(2 r_s)^3 as a polynomial in t = 2 s/s_max - 1, Horner order
    double poly_err = 0;                // max |g_poly - g| over [0, x_cut] in exact arithmetic
    int fused_deg = 0;
    float fused_c[POLY_MAX_DEG + 1]{};  // H(x) = erfcx(x) + 2x/sqrt(pi) as a polynomial in t = 2 x/x_cut - 1, Horner order
    double fused_err = 0;               // max |exp(-x^2) H_poly(x) - g| over [0, x_cut] in exact arithmetic

    DevBuf ws[WS_COUNT];
    // chunk tables of the ORB partition levels (orb_select.cu): they depend on (n, L0) only
    long long sel_n = -1;
    int sel_L0 = -1;
    std::vector<long long> sel_off, sel_noff;

    photons_stats stats{};
    std::string err;
};

// pointer to at least `bytes` of device memory in slot `slot` (contents undefined after growth); nullptr and
// c->err set if the allocation fails
void* workspace(Ctx* c, int slot, size_t bytes);
void workspace_free(Ctx* c);

int fail(Ctx* c, int code, const char* fmt, ...);
// raise a kernel's dynamic shared-memory limit once per context (the size per kernel is fixed by the parameters)
cudaError_t opt_in_smem(Ctx* c, const void* kernel, size_t bytes);
#define PH_CUDA(c, call)                                                                         \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return photons::fail((c), e_ == cudaErrorMemoryAllocation ? PHOTONS_ENOMEM : PHOTONS_ECUDA, \
                                 "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
    } while (0)

// orb_select.cu
int orb_phase_a_select(Ctx* c, int L0, float4*& P_cur, float4*& P_alt, int* lo, int* hi, cudaStream_t st);
// build.cu
int build_leaves_impl(Ctx* c);
void free_leaves(Ctx* c);
// gfunc.cu
int make_table(Ctx* c);
int make_poly(Ctx* c);
int make_fused(Ctx* c);
// p2p_fp64.cu / p2p_fp32.cu: enqueue the kernel for target leaves order[first .. first+count) on a stream;
// out = device buffer in caller order (n x 3, fp64 or fp32 as out_f32 says)
int launch_p2p_fp64(Ctx* c, long long first, long long count, void* out, bool out_f32, cudaStream_t st);
int launch_p2p_fp32(Ctx* c, long long first, long long count, void* out, bool out_f32, cudaStream_t st);

// float <-> int whose signed integer order is the float order (negative coordinates occur with isolated boundaries)
__host__ __device__ inline int f2ord(float f)
{
    int b;
    memcpy(&b, &f, 4);
    return b ^ ((b >> 31) & 0x7fffffff);
}
__host__ __device__ inline float ord2f(int o)
{
    o ^= (o >> 31) & 0x7fffffff;
    float f;
    memcpy(&f, &o, 4);
    return f;
}

// first sorted position of segment k at tree level `level` when n particles are bisected with the
// left child taking floor(size/2) (A13)
__host__ __device__ inline long long seg_start(long long n, int level, long long k)
{
    long long start = 0, size = n;
    for (int b = level - 1; b >= 0; --b) {
        long long left = size >> 1;
        if ((k >> b) & 1) { start += left; size -= left; }
        else size = left;
    }
    return start;
}
// segment that holds sorted position q at `level`
__host__ __device__ inline long long seg_of(long long n, int level, long long q)
{
    long long start = 0, size = n, k = 0;
    for (int b = 0; b < level; ++b) {
        long long left = size >> 1;
        k <<= 1;
        if (q >= start + left) { start += left; size -= left; k |= 1; }
        else size = left;
    }
    return k;
}

}  // namespace photons
