// photons_build_leaves on the device: ORB sort, leaf-sorted packed particle arrays (L69),
// leaf table (L79) and the interaction list grouped by target leaf (the paper's TaskGroup/GroupIdx,
// L83-L85).  FEED steps a1-a3 of SURVEY.md §8(a); readings A10, A11, A13 of DESIGN.md.
#include <cub/cub.cuh>

#include <algorithm>
#include <cmath>

#include "common.cuh"

namespace photons {

// Device buffers live in the context's grow-only workspace (common.cuh): a rebuild with the same particle
// number allocates nothing.  Dropping the leaves therefore only resets the state.
void free_leaves(Ctx* c)
{
    c->d_perm = nullptr; c->d_slot_src = nullptr; c->d_leaf_cnt = nullptr; c->d_leaf_ctr = nullptr;
    c->d_node_lo = c->d_node_hi = nullptr; c->d_p64 = nullptr; c->d_p32 = nullptr;
    c->d_chunk_ptr = nullptr; c->d_chunks = nullptr; c->d_order = nullptr;
    c->leaves_built = false;
    c->n_leaves = c->n_slots = 0;
}

// ---------------------------------------------------------------------------------------------- ORB
// Every tree node is split at its median along the axis of largest extent of its particle bounding box; the
// left child takes floor(size/2) particles (A13).  Two phases:
//   A (levels 0 .. L0-1, nodes larger than ORB_CTA_MAX particles): one stable radix sort per level over the
//     whole array on keys (node, coordinate as a 20-bit fixed-point number inside the node's bbox).  The
//     particles travel with the sort as float4 {x, y, z, caller index} in current order, so every pass reads
//     and writes coalesced; the gather that applies the sorted order also reduces the children's bboxes.
//   B (levels L0 .. depth-1): one CTA per level-L0 node finishes all remaining levels in shared memory
//     (per level a radix select of every sub-node's median key and a stable partition about it).
// Splitting coordinates are the positions rounded to fp32; ties go either way, which never changes `a`.

constexpr int ORB_CTA_MAX = 4096;   // particles a phase-B CTA holds in shared memory
#ifndef PHOTONS_ORB_CTA_THREADS
#define PHOTONS_ORB_CTA_THREADS 1024
#endif
constexpr int ORB_CTA_THREADS = PHOTONS_ORB_CTA_THREADS;
// Phase-A sort key = (node, coordinate quantised to this many bits inside the node's bbox).  20 bits resolve 1e-6 of
// the node's extent — far below the particle spacing of nodes that still hold > 4096 particles — and keep the
// keys within 32 bits (4 radix passes or fewer) down to level 12; ties are split by the stable order.
constexpr int ORB_COORD_BITS = 20;

__global__ void orb_init_kernel(long long n, const double* __restrict__ pos, float4* __restrict__ P)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n) return;
    P[i] = make_float4((float)pos[3 * i], (float)pos[3 * i + 1], (float)pos[3 * i + 2], __int_as_float((int)i));
}

__global__ void fill_int_kernel(long long n, int* p, int v)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// P_out[q] = P_in[src[q]] (src == nullptr: identity), and the bounding boxes of the level-`level` nodes as
// order-preserving integers (f2ord).  Reduced per
// warp and, when the whole block sits in one node (the upper levels), per block, before the global atomics.
__global__ void __launch_bounds__(256) orb_gather_bbox_kernel(long long n, int level, const uint32_t* __restrict__ src,
                                                              const float4* __restrict__ P_in, float4* __restrict__ P_out,
                                                              int* __restrict__ lo, int* __restrict__ hi)
{
    __shared__ int s_lo[8][3], s_hi[8][3];
    long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = q < n;
    const long long qq = live ? q : n - 1;
    const float4 p = src ? P_in[src[qq]] : P_in[qq];
    if (live && P_out) P_out[q] = p;
    if (!lo) return;
    const long long seg = seg_of(n, level, qq);
    const long long q_first = blockIdx.x * (long long)blockDim.x;
    const long long q_last = min(q_first + blockDim.x, n) - 1;
    const bool block_uniform = seg_of(n, level, q_first) == seg_of(n, level, q_last);
    const int v[3] = {f2ord(p.x), f2ord(p.y), f2ord(p.z)};
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long seg0 = __shfl_sync(0xffffffffu, seg, 0);
    const bool warp_uniform = __all_sync(0xffffffffu, seg == seg0);
    if (warp_uniform) {
        for (int a = 0; a < 3; ++a) {
            const int mn = __reduce_min_sync(0xffffffffu, v[a]), mx = __reduce_max_sync(0xffffffffu, v[a]);
            if (lane == 0) {
                if (block_uniform) { s_lo[warp][a] = mn; s_hi[warp][a] = mx; }
                else { atomicMin(&lo[3 * seg + a], mn); atomicMax(&hi[3 * seg + a], mx); }
            }
        }
    } else if (live) {
        for (int a = 0; a < 3; ++a) { atomicMin(&lo[3 * seg + a], v[a]); atomicMax(&hi[3 * seg + a], v[a]); }
    }
    if (block_uniform) {     // then every warp is uniform too
        __syncthreads();
        if (threadIdx.x < 3) {
            int mn = s_lo[0][threadIdx.x], mx = s_hi[0][threadIdx.x];
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { mn = min(mn, s_lo[w][threadIdx.x]); mx = max(mx, s_hi[w][threadIdx.x]); }
            atomicMin(&lo[3 * seg + threadIdx.x], mn);
            atomicMax(&hi[3 * seg + threadIdx.x], mx);
        }
    }
}

__device__ __forceinline__ int widest_axis(const float ext[3])
{
    int axis = 0;                                   // largest extent, ties -> lowest axis
    if (ext[1] > ext[axis]) axis = 1;
    if (ext[2] > ext[axis]) axis = 2;
    return axis;
}

template <typename Key>     // 32-bit keys while node index and coordinate fit (levels 0..8), 64-bit after
__global__ void orb_key_kernel(long long n, int level, const float4* __restrict__ P, const int* __restrict__ lo,
                               const int* __restrict__ hi, Key* __restrict__ keys, uint32_t* __restrict__ vals)
{
    long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (q >= n) return;
    const long long seg = seg_of(n, level, q);
    float l[3], ext[3];
    for (int a = 0; a < 3; ++a) { l[a] = ord2f(lo[3 * seg + a]); ext[a] = ord2f(hi[3 * seg + a]) - l[a]; }
    const int axis = widest_axis(ext);
    const float4 p = P[q];
    const float x = axis == 0 ? p.x : axis == 1 ? p.y : p.z;
    // monotone map of [lo, hi] onto ORB_COORD_BITS-bit integers
    const float u = ext[axis] > 0.f ? (x - l[axis]) / ext[axis] : 0.f;
    const float top = (float)((1u << ORB_COORD_BITS) - 1u);
    const unsigned f = (unsigned)fminf(u * top, top);
    keys[q] = (Key)(((unsigned long long)seg << ORB_COORD_BITS) | f);
    vals[q] = (uint32_t)q;
}

// Phase B: CTA b owns the level-L0 node b, sorted positions [seg_start(L0, b), seg_start(L0, b + 1)), and finishes the
// remaining levels in shared memory.  A level needs every sub-node split at its median along its widest axis - a stable
// partition, not a sort: 24-bit fixed-point keys inside the sub-node's bbox, the median key by radix select (four
// rounds of 6-bit digit histograms, one histogram per sub-node), then a stable partition about it (ballot ranks inside
// a warp, one scan over the warps' totals).  Elements are dealt to the warps in blocks of 128 and to the lanes of a
// warp round-robin, so every shared-memory access is lane-contiguous.
constexpr int ORB_B_WARPS = ORB_CTA_THREADS / 32;
constexpr int ORB_B_ITEMS = ORB_CTA_MAX / ORB_CTA_THREADS;      // 4 elements per thread
constexpr int ORB_B_MAXSUB = 128;                               // sub-nodes of a CTA at its last level (4096 / 32, or / 16 ... / 2^7)
constexpr int ORB_B_DIGIT = 6, ORB_B_BINS = 1 << ORB_B_DIGIT, ORB_B_ROUNDS = 4;   // 4 x 6 = 24 key bits

struct OrbBShared {
    float4 cur[ORB_CTA_MAX];
    unsigned hist[ORB_B_MAXSUB * ORB_B_BINS];
    int blo[3 * ORB_B_MAXSUB], bhi[3 * ORB_B_MAXSUB];
    unsigned prefix[ORB_B_MAXSUB], rank[ORB_B_MAXSUB], below[ORB_B_MAXSUB], ties[ORB_B_MAXSUB];
    unsigned sbase[ORB_B_MAXSUB];            // packed (ties << 16 | less) before the sub-node's first element
    int sstart[2][ORB_B_MAXSUB + 1];         // first element of each sub-node (this level / the next one)
    unsigned wtot[ORB_B_WARPS], wbase[ORB_B_WARPS];
};

__global__ void __launch_bounds__(ORB_CTA_THREADS, ORB_CTA_THREADS >= 1024 ? 1 : 2) orb_cta_kernel(long long n, int L0, int depth, const float4* __restrict__ P,
                                                                  uint32_t* __restrict__ perm)
{
    extern __shared__ __align__(16) unsigned char orb_smem[];
    OrbBShared& S = *reinterpret_cast<OrbBShared*>(orb_smem);
    const long long s0 = seg_start(n, L0, blockIdx.x);
    const long long s1 = blockIdx.x + 1 == (1LL << L0) ? n : seg_start(n, L0, blockIdx.x + 1);
    const int size = (int)(s1 - s0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    // element r of this thread: warp-blocked, lane-striped
    int el[ORB_B_ITEMS];
#pragma unroll
    for (int r = 0; r < ORB_B_ITEMS; ++r) el[r] = warp * (32 * ORB_B_ITEMS) + r * 32 + lane;
#pragma unroll
    for (int r = 0; r < ORB_B_ITEMS; ++r) if (el[r] < size) S.cur[el[r]] = P[s0 + el[r]];
    if (threadIdx.x == 0) { S.sstart[0][0] = 0; S.sstart[0][1] = size; }
    int sub[ORB_B_ITEMS];                            // sub-node of element el[r] at the current level
#pragma unroll
    for (int r = 0; r < ORB_B_ITEMS; ++r) sub[r] = 0;
    __syncthreads();

    for (int level = L0; level < depth; ++level) {
        const int sl = level - L0;                   // sub-nodes of this CTA at this level: 2^sl (<= ORB_B_MAXSUB)
        const int nsub = 1 << sl;
        const int* sstart = S.sstart[sl & 1];
        int* sstart_next = S.sstart[(sl + 1) & 1];
        for (int i = threadIdx.x; i < 3 * nsub; i += blockDim.x) { S.blo[i] = 0x7fffffff; S.bhi[i] = (int)0x80000000; }
        __syncthreads();
        float4 p[ORB_B_ITEMS];
        // bounding boxes of the sub-nodes (whole warps enter: the votes need all lanes)
#pragma unroll
        for (int r = 0; r < ORB_B_ITEMS; ++r) {
            const bool live = el[r] < size;
            p[r] = S.cur[live ? el[r] : size - 1];
            const int v[3] = {f2ord(p[r].x), f2ord(p[r].y), f2ord(p[r].z)};
            const int sub0 = __shfl_sync(0xffffffffu, sub[r], 0);
            if (__all_sync(0xffffffffu, sub[r] == sub0)) {
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int mn = __reduce_min_sync(0xffffffffu, v[a]), mx = __reduce_max_sync(0xffffffffu, v[a]);
                    if (lane == 0) { atomicMin(&S.blo[3 * sub0 + a], mn); atomicMax(&S.bhi[3 * sub0 + a], mx); }
                }
            } else if (live) {
#pragma unroll
                for (int a = 0; a < 3; ++a) { atomicMin(&S.blo[3 * sub[r] + a], v[a]); atomicMax(&S.bhi[3 * sub[r] + a], v[a]); }
            }
        }
        for (int k = threadIdx.x; k < nsub; k += blockDim.x) {
            S.prefix[k] = 0; S.below[k] = 0;
            S.rank[k] = (unsigned)((sstart[k + 1] - sstart[k]) >> 1);    // first element of the right child
        }
        __syncthreads();
        // keys: coordinate along the sub-node's widest axis as a 24-bit fixed-point number inside its bbox
        unsigned key[ORB_B_ITEMS];
#pragma unroll
        for (int r = 0; r < ORB_B_ITEMS; ++r) {
            float lo3[3], ext[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) { lo3[a] = ord2f(S.blo[3 * sub[r] + a]); ext[a] = ord2f(S.bhi[3 * sub[r] + a]) - lo3[a]; }
            const int axis = widest_axis(ext);
            const float x = axis == 0 ? p[r].x : axis == 1 ? p[r].y : p[r].z;
            const float u = ext[axis] > 0.f ? (x - lo3[axis]) / ext[axis] : 0.f;
            key[r] = (unsigned)fminf(u * 16777215.0f, 16777215.0f);
        }
        // median key of every sub-node by radix select
        for (int round = 0; round < ORB_B_ROUNDS; ++round) {
            const int shift = ORB_B_DIGIT * (ORB_B_ROUNDS - 1 - round);
            for (int i = threadIdx.x; i < nsub * ORB_B_BINS; i += blockDim.x) S.hist[i] = 0;
            __syncthreads();
#pragma unroll
            for (int r = 0; r < ORB_B_ITEMS; ++r) {
                if (el[r] < size && (round == 0 || (key[r] >> (shift + ORB_B_DIGIT)) == S.prefix[sub[r]]))
                    atomicAdd(&S.hist[sub[r] * ORB_B_BINS + ((key[r] >> shift) & (ORB_B_BINS - 1))], 1u);
            }
            __syncthreads();
            for (int k = warp; k < nsub; k += ORB_B_WARPS) {       // one warp per sub-node: the bin that holds the rank
                const unsigned v0 = S.hist[k * ORB_B_BINS + 2 * lane], v1 = S.hist[k * ORB_B_BINS + 2 * lane + 1];
                const unsigned s = v0 + v1;
                unsigned inc = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                const unsigned rk = S.rank[k];
                const unsigned cum = inc - s;
                int bin = -1;
                unsigned cb = 0, hb = 0;
                if (rk >= cum && rk < cum + v0) { bin = 2 * lane; cb = cum; hb = v0; }
                else if (rk >= cum + v0 && rk < cum + s) { bin = 2 * lane + 1; cb = cum + v0; hb = v1; }
                const unsigned owner = __ballot_sync(0xffffffffu, bin >= 0);
                if (owner && lane == __ffs(owner) - 1) {           // exactly one lane (rank < size of the sub-node)
                    S.prefix[k] = (S.prefix[k] << ORB_B_DIGIT) | (unsigned)bin;
                    S.rank[k] = rk - cb;
                    S.below[k] += cb;
                    S.ties[k] = hb;
                }
            }
            __syncthreads();
        }
        // stable partition of every sub-node about its median key m: keys < m and the first (left - #less) keys == m
        // go left, the rest right, each side in its old order
        unsigned ex[ORB_B_ITEMS];
        {
            unsigned run = 0;                         // packed (ties << 16 | less) of this warp's elements so far
#pragma unroll
            for (int r = 0; r < ORB_B_ITEMS; ++r) {
                const bool live = el[r] < size;
                const unsigned m = S.prefix[sub[r]];
                const unsigned bl = __ballot_sync(0xffffffffu, live && key[r] < m);
                const unsigned bt = __ballot_sync(0xffffffffu, live && key[r] == m);
                ex[r] = run + (unsigned)__popc(bl & lt_mask) + ((unsigned)__popc(bt & lt_mask) << 16);
                run += (unsigned)__popc(bl) + ((unsigned)__popc(bt) << 16);
            }
            if (lane == 0) S.wtot[warp] = run;
        }
        __syncthreads();
        if (warp == 0) {
            const unsigned v = lane < ORB_B_WARPS ? S.wtot[lane] : 0u;
            unsigned inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane < ORB_B_WARPS) S.wbase[lane] = inc - v;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < ORB_B_ITEMS; ++r) {
            ex[r] += S.wbase[warp];
            if (el[r] < size && el[r] == sstart[sub[r]]) S.sbase[sub[r]] = ex[r];
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < ORB_B_ITEMS; ++r) {
            if (el[r] >= size) { sub[r] = 2 * nsub - 1; continue; }     // padding follows the last element
            const int k = sub[r];
            const int st = sstart[k];
            const unsigned left = (unsigned)((sstart[k + 1] - st) >> 1);
            const unsigned m = S.prefix[k], less_total = S.below[k], tie_total = S.ties[k];
            const unsigned need = left - less_total;                 // ties that still go left
            const unsigned rel = ex[r] - S.sbase[k];                 // both fields are >= the base's: no borrow
            const unsigned lb = rel & 0xffffu, tb = rel >> 16;
            const unsigned idx = (unsigned)(el[r] - st);
            unsigned dst;
            if (key[r] < m) dst = lb;
            else if (key[r] == m) dst = tb < need ? less_total + tb : left + (tb - need);
            else dst = left + (tie_total - need) + (idx - lb - tb);
            S.cur[st + (int)dst] = p[r];
            sub[r] = 2 * k + (el[r] - st >= (int)left);       // the sub-node of POSITION el[r] one level down
        }
        if (level + 1 < depth)       // (the last level may have ORB_B_MAXSUB sub-nodes: nothing follows it)
        for (int k = threadIdx.x; k < nsub; k += blockDim.x) {
            const int st = sstart[k];
            sstart_next[2 * k] = st;
            sstart_next[2 * k + 1] = st + ((sstart[k + 1] - st) >> 1);
            if (k == nsub - 1) sstart_next[2 * nsub] = size;
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < ORB_B_ITEMS; ++r)
        if (el[r] < size) perm[s0 + el[r]] = (uint32_t)__float_as_int(S.cur[el[r]].w);
}

// ------------------------------------------------------------------------------ leaf table + packing

// one thread per leaf: count, tight bbox, origin for the mixed-precision offsets
__global__ void leaf_table_kernel(long long n, int depth, long long n_leaves, const uint32_t* __restrict__ perm,
                                  const double* __restrict__ pos, int* __restrict__ cnt, double* __restrict__ lo,
                                  double* __restrict__ hi, double* __restrict__ ctr)
{
    long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= n_leaves) return;
    const long long s0 = seg_start(n, depth, k);
    const long long s1 = k + 1 == n_leaves ? n : seg_start(n, depth, k + 1);
    double l[3] = {1e300, 1e300, 1e300}, h[3] = {-1e300, -1e300, -1e300};
    for (long long q = s0; q < s1; ++q) {
        const size_t src = perm[q];
        for (int a = 0; a < 3; ++a) {
            const double x = pos[3 * src + a];
            l[a] = fmin(l[a], x);
            h[a] = fmax(h[a], x);
        }
    }
    cnt[k] = (int)(s1 - s0);
    for (int a = 0; a < 3; ++a) {
        lo[3 * k + a] = l[a];
        hi[3 * k + a] = h[a];
        // origin of the fp32 offsets: bbox midpoint rounded to fp32, so that offsets of positions that
        // live on the fp32 grid are (almost always) exact
        ctr[3 * k + a] = (double)(float)(0.5 * (l[a] + h[a]));
    }
}

// one thread per slot: fill the packed arrays.  Padding slots repeat the leaf's first particle with
// zero mass (they add nothing as sources and are never written as targets).  ugm (equal-mass fp32 kernels, which do
// not read G m per pair): the fp32 copy of a padding slot sits far outside the box instead, beyond r_cut of everything.
__global__ void pack_kernel(long long n, int depth, int maxleaf, long long n_slots, double G, int precision, int ugm,
                            double inv_pscale, double inv_gmscale,
                            const uint32_t* __restrict__ perm, const double* __restrict__ pos,
                            const double* __restrict__ mass, const double* __restrict__ ctr,
                            int* __restrict__ slot_src, double4* __restrict__ p64, float* __restrict__ p32)
{
    long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    const long long k = s / maxleaf;
    const int t = (int)(s - k * maxleaf);
    const long long n_leaves = n_slots / maxleaf;
    const long long s0 = seg_start(n, depth, k);
    const long long s1 = k + 1 == n_leaves ? n : seg_start(n, depth, k + 1);
    const bool real = t < s1 - s0;
    const size_t src = perm[real ? s0 + t : s0];
    const double x = pos[3 * src], y = pos[3 * src + 1], z = pos[3 * src + 2];
    const double gm = real ? G * mass[src] : 0.0;
    slot_src[s] = real ? (int)src : -1;
    p64[s] = make_double4(x, y, z, gm);
    if (p32) {
        double ox = 0, oy = 0, oz = 0;
        if (precision == PHOTONS_MIXED) { ox = ctr[3 * k]; oy = ctr[3 * k + 1]; oz = ctr[3 * k + 2]; }
        float* b = p32 + (s >> 1) * 8 + (s & 1);
        // kernel units (powers of two: the rescaling itself is exact)
        const bool away = ugm && !real;
        b[0] = away ? PAD_FAR : (float)((x - ox) * inv_pscale);
        b[2] = away ? PAD_FAR : (float)((y - oy) * inv_pscale);
        b[4] = away ? PAD_FAR : (float)((z - oz) * inv_pscale);
        b[6] = (float)(gm * inv_gmscale);
    }
}

// bounding boxes of the internal tree nodes, one level per launch (heap order: node (l,k) = 2^l - 1 + k)
__global__ void node_bbox_kernel(int level, double* __restrict__ lo, double* __restrict__ hi)
{
    const long long cnt = 1LL << level;
    long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= cnt) return;
    const long long me = cnt - 1 + k, c0 = 2 * cnt - 1 + 2 * k, c1 = c0 + 1;
    for (int a = 0; a < 3; ++a) {
        lo[3 * me + a] = fmin(lo[3 * c0 + a], lo[3 * c1 + a]);
        hi[3 * me + a] = fmax(hi[3 * c0 + a], hi[3 * c1 + a]);
    }
}

// --------------------------------------------------------------------------------- interaction list
// For target leaf i: depth-first walk of the ORB tree, keeping the nodes whose periodic bbox-to-bbox
// distance to leaf i's bbox is below r_cut (A11); accepted leaves come out in ascending order and are
// merged into runs of contiguous leaves with the same image shift, at most chunk_max slots long.
// Pass 1 (chunks == nullptr) counts, pass 2 writes.

constexpr int LIST_STASH = 128;   // list entries per leaf kept from the counting pass

struct ListArgs {
    long long n_leaves;
    int depth, maxleaf, chunk_max, periodic;
    double L, rcut;
    const float4* box;            // 2 per tree node (heap order): {centre, .}, {half-width rounded up, .}
    const int* leaf_cnt;
    const long long* chunk_ptr;   // pass 2
    uint2* chunks;                // pass 2
    uint2* stash;                 // pass 1: the first stash_cap entries of every leaf, stride stash_cap
    int stash_cap;
    long long* n_chunks_of;       // pass 1: per leaf
    unsigned long long* totals;   // pass 1: [0] leaf pairs, [1] pairs evaluated, [2] longest list in source slots
    long long* work_of;           // pass 1: slots in the list of each leaf (for the heaviest-first order)
    int4* resume;                 // per leaf: walk state when the stash filled up {heap index, run_first, run_n, run_code}
};

__global__ void list_kernel(ListArgs a)
{
    const long long i_raw = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = i_raw < a.n_leaves;
    const long long i = live ? i_raw : a.n_leaves - 1;
    const int leaf0 = (int)(a.n_leaves - 1);   // heap index of leaf 0
    // fp32 walk on {centre, half-width} boxes whose half-widths were rounded up (node_box32_kernel) and with a
    // slack of 1e-6 L on every gap: it can only accept more than the exact test would, never less.
    const float4 tc = a.box[2 * (size_t)(leaf0 + i)], thw = a.box[2 * (size_t)(leaf0 + i) + 1];
    const float Lf = (float)a.L, invL = (float)(1.0 / a.L), slack = 1e-6f * Lf;
    const float rc2 = (float)(a.rcut * a.rcut) * (1.0f + 1e-6f);
    const float amb = Lf - 2.0f * (float)a.rcut;      // ambiguous image iff 2 (hw_i + hw_j) >= amb  (A10)
    const int my_cnt = a.leaf_cnt[i];

    int run_first = -1, run_n = 0, run_code = -1, n_chunks = 0, n_pairs = 0;
    long long n_src = 0;          // particles in the accepted source leaves
    // Pass 1 counts and keeps the first stash_cap entries of every leaf, and notes the state of the walk at the moment
    // the stash fills up; pass 2 (only the leaves whose list did not fit; the stashed part is copied by
    // list_copy_kernel) resumes the walk from that state and writes the rest in place.
    const bool pass2 = a.chunks != nullptr;
    const bool skip = !live || (pass2 && a.n_chunks_of[i] <= a.stash_cap);
    uint2* out = pass2 ? a.chunks + a.chunk_ptr[i] : nullptr;
    uint2* stash = pass2 ? nullptr : a.stash + i * a.stash_cap;
    const int max_leaves_per_chunk = a.chunk_max / a.maxleaf;
    unsigned h = skip ? 0u : 1u;
    auto emit = [&]() {
        const uint2 ent = make_uint2((unsigned)(run_first * a.maxleaf), (unsigned)(run_n * a.maxleaf) | (unsigned)run_code);
        if (out) out[n_chunks] = ent;
        else if (n_chunks < a.stash_cap) stash[n_chunks] = ent;
        ++n_chunks;
    };
    if (pass2 && !skip) {      // continue after the leaf that opened run number stash_cap
        const int4 r = a.resume[i];
        h = (unsigned)r.x; run_first = r.y; run_n = r.z; run_code = r.w;
        n_chunks = a.stash_cap;
        const unsigned up = h + 1;
        h = up >> (__ffs(up) - 1);
        if (h == 1) h = 0;
    }

    // Stackless depth-first walk of the complete binary tree: with 1-based heap indices the children of h are 2h and
    // 2h + 1, and the node that follows the subtree of h is (h + 1) >> ctz(h + 1) (up while h is a right child, then
    // on to the sibling); arriving at 1 = back at the root = done.  Left child first: leaves come out in ascending order.
    while (h) {
        const int node = (int)h - 1;
        const float4 nc = __ldg(&a.box[2 * (size_t)node]), nhw = __ldg(&a.box[2 * (size_t)node + 1]);
        // periodic bbox-to-bbox distance (A11): per axis the nearest image of the centre difference, less the half-widths
        const float dcs[3] = {nc.x - tc.x, nc.y - tc.y, nc.z - tc.z};
        const float hws[3] = {nhw.x + thw.x, nhw.y + thw.y, nhw.z + thw.z};
        float img[3];                 // the source is moved by -img box lengths
        float g2 = 0.f;
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            img[x] = a.periodic ? rintf(dcs[x] * invL) : 0.f;
            const float gap = fmaxf(0.f, fabsf(fmaf(-Lf, img[x], dcs[x])) - (hws[x] + slack));
            g2 = fmaf(gap, gap, g2);
        }
        const bool accept = g2 < rc2;
        const bool internal = node < leaf0;
        if (accept && !internal) {
            const int j = node - leaf0;
            // the three shift fields of entry_pack, without the slot count; ambiguous image -> per-pair flag (A10)
            int code = 0x150000;                  // no image shift on any axis: almost every accepted leaf
            if (img[0] != 0.f || img[1] != 0.f || img[2] != 0.f)
                code = ((1 - (int)img[0]) << 16) | ((1 - (int)img[1]) << 18) | ((1 - (int)img[2]) << 20);
            if (a.periodic && 2.0f * fmaxf(hws[0], fmaxf(hws[1], hws[2])) >= amb) code = (int)entry_pack(0, 0, 0, 0, true);
            ++n_pairs;
            n_src += (int)nc.w;          // the leaf's particle count rides in the box record (node_box32_kernel)
            if (run_n > 0 && j == run_first + run_n && code == run_code && run_n < max_leaves_per_chunk) {
                ++run_n;
            } else {
                if (run_n > 0) {
                    emit();
                    if (!pass2 && n_chunks == a.stash_cap) a.resume[i] = make_int4((int)h, j, 1, code);   // state after this leaf
                }
                run_first = j; run_n = 1; run_code = code;
            }
        }
        // accepted internal node: down to the left child; else on to the node after this subtree (one select: the
        // lanes of a warp sit at different nodes, so the two ways on must not be two divergent paths)
        const unsigned up = h + 1;
        const unsigned nxt = up >> (__ffs(up) - 1);
        h = accept && internal ? 2 * h : nxt == 1 ? 0u : nxt;
    }
    const long long n_eval = (long long)my_cnt * n_src;
    if (run_n > 0) emit();
    if (!a.chunks) {       // whole warps arrive here
        const long long work = (long long)n_pairs * a.maxleaf;
        if (live) { a.n_chunks_of[i] = n_chunks; a.work_of[i] = work; }
        unsigned long long tp = (unsigned long long)n_pairs, te = (unsigned long long)n_eval, tw = (unsigned long long)work;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tp += __shfl_xor_sync(0xffffffffu, tp, o);
            te += __shfl_xor_sync(0xffffffffu, te, o);
            tw = max(tw, __shfl_xor_sync(0xffffffffu, tw, o));
        }
        if ((threadIdx.x & 31) == 0) {
            atomicAdd(&a.totals[0], tp);
            atomicAdd(&a.totals[1], te);
            atomicMax(&a.totals[2], tw);
        }
    }
}

// fp32 boxes for the list walk: centre rounded to nearest, half-width rounded up and widened by the centre's rounding
// (.w of the centre record: the particle count of a leaf node, 0 for internal nodes - read by the list walk)
__global__ void node_box32_kernel(long long n_nodes, long long n_leaves, const int* __restrict__ leaf_cnt,
                                  const double* __restrict__ lo, const double* __restrict__ hi, float4* __restrict__ box)
{
    long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= n_nodes) return;
    float c[3], h[3];
    for (int a = 0; a < 3; ++a) {
        const double cd = 0.5 * (lo[3 * k + a] + hi[3 * k + a]);
        c[a] = (float)cd;
        h[a] = __double2float_ru(0.5 * (hi[3 * k + a] - lo[3 * k + a]) + fabs(cd - (double)c[a]));
    }
    const long long leaf = k - (n_leaves - 1);
    box[2 * k] = make_float4(c[0], c[1], c[2], leaf >= 0 ? (float)leaf_cnt[leaf] : 0.f);
    box[2 * k + 1] = make_float4(h[0], h[1], h[2], 0.f);
}

// one warp per leaf: stash -> CSR
__global__ void list_copy_kernel(long long n_leaves, int stash_cap, const long long* __restrict__ chunk_ptr,
                                 const uint2* __restrict__ stash, uint2* __restrict__ chunks)
{
    const long long i = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    if (i >= n_leaves) return;
    const long long c0 = chunk_ptr[i];
    const int cnt = min((int)(chunk_ptr[i + 1] - c0), stash_cap);     // longer lists: list_kernel's second pass writes the rest
    for (int k = threadIdx.x & 31; k < cnt; k += 32) chunks[c0 + k] = stash[i * stash_cap + k];
}

__global__ void order_identity_kernel(long long n_leaves, int* __restrict__ order)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n_leaves) order[i] = (int)i;
}

__global__ void order_keys_kernel(long long n_leaves, const long long* __restrict__ work, unsigned* __restrict__ keys, int* __restrict__ vals)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_leaves) return;
    keys[i] = (unsigned)min(work[i], 0xffffffffLL);
    vals[i] = (int)i;
}

// -------------------------------------------------------------------------------------------- driver

__global__ void orb_perm_kernel(long long n, const float4* __restrict__ P, uint32_t* __restrict__ perm)
{
    long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (q < n) perm[q] = (uint32_t)__float_as_int(P[q].w);
}

#define PH_CUDA_BUILD(call)                                                                                 \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess)                                                                              \
            return fail(c, e_ == cudaErrorMemoryAllocation ? PHOTONS_ENOMEM : PHOTONS_ECUDA, "%s:%d %s: %s", \
                        __FILE__, __LINE__, #call, cudaGetErrorString(e_));                                 \
    } while (0)
#define PH_WS(ptr, type, slot, count)                                                              \
    do {                                                                                           \
        (ptr) = static_cast<type*>(workspace(c, (slot), sizeof(type) * (size_t)(count)));          \
        if (!(ptr)) return PHOTONS_ENOMEM;                                                         \
    } while (0)

static inline unsigned blocks_for(long long n, int tb) { return (unsigned)((n + tb - 1) / tb); }

static int orb_sort(Ctx* c, int depth, cudaStream_t st)
{
    const long long n = c->n;
    const int tb = 256;
    int L0 = 0;
    while (L0 < depth && ((n + (1LL << L0) - 1) >> L0) > ORB_CTA_MAX) ++L0;
    float4 *P_cur = nullptr, *P_alt = nullptr;
    PH_WS(P_cur, float4, WS_ORB_P0, n);
    orb_init_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, c->d_pos, P_cur);
    ++c->launches;
    if (L0 > 0) {
        unsigned long long *keys = nullptr, *keys2 = nullptr;
        uint32_t *vals = nullptr, *vals2 = nullptr;
        int *lo = nullptr, *hi = nullptr;
        PH_WS(P_alt, float4, WS_ORB_P1, n);
        PH_WS(keys, unsigned long long, WS_ORB_KEYS, n);
        PH_WS(keys2, unsigned long long, WS_ORB_KEYS2, n);
        PH_WS(vals, uint32_t, WS_ORB_VALS, n);
        PH_WS(vals2, uint32_t, WS_ORB_VALS2, n);
        PH_WS(lo, int, WS_ORB_LO, 3LL << L0);
        PH_WS(hi, int, WS_ORB_HI, 3LL << L0);
        size_t tmp_bytes = 0;
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, vals, vals2, (int)n, 0, ORB_COORD_BITS + L0, st));
        {
            size_t need32 = 0;
            PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(nullptr, need32, reinterpret_cast<uint32_t*>(keys), reinterpret_cast<uint32_t*>(keys2),
                                                          vals, vals2, (int)n, 0, 32, st));
            tmp_bytes = std::max(tmp_bytes, need32);
        }
        void* tmp = workspace(c, WS_CUB_TMP, tmp_bytes);
        if (!tmp) return PHOTONS_ENOMEM;
        fill_int_kernel<<<1, 32, 0, st>>>(3, lo, 0x7fffffff);
        fill_int_kernel<<<1, 32, 0, st>>>(3, hi, (int)0x80000000);
        orb_gather_bbox_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, 0, nullptr, P_cur, nullptr, lo, hi);
        c->launches += 3;
        if (c->p.orb_method == 0) {
            const int rc = orb_phase_a_select(c, L0, P_cur, P_alt, lo, hi, st);
            if (rc != PHOTONS_OK) return rc;
        } else
        for (int level = 0; level < L0; ++level) {
            if (ORB_COORD_BITS + level <= 32) {
                uint32_t* k32 = reinterpret_cast<uint32_t*>(keys);
                uint32_t* k32b = reinterpret_cast<uint32_t*>(keys2);
                orb_key_kernel<uint32_t><<<blocks_for(n, tb), tb, 0, st>>>(n, level, P_cur, lo, hi, k32, vals);
                PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, k32, k32b, vals, vals2, (int)n, 0, ORB_COORD_BITS + level, st));
            } else {
                orb_key_kernel<unsigned long long><<<blocks_for(n, tb), tb, 0, st>>>(n, level, P_cur, lo, hi, keys, vals);
                PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, vals, vals2, (int)n, 0, ORB_COORD_BITS + level, st));
            }
            ++c->launches;
            const bool more = level + 1 < L0;   // the next level's boxes, reduced while the order is applied
            if (more) {
                const long long nb = 3LL << (level + 1);
                fill_int_kernel<<<blocks_for(nb, tb), tb, 0, st>>>(nb, lo, 0x7fffffff);
                fill_int_kernel<<<blocks_for(nb, tb), tb, 0, st>>>(nb, hi, (int)0x80000000);
                c->launches += 2;
            }
            orb_gather_bbox_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, level + 1, vals2, P_cur, P_alt, more ? lo : nullptr, hi);
            ++c->launches;
            std::swap(P_cur, P_alt);
        }
    }
    if (depth > L0) {
        const size_t smem = sizeof(OrbBShared);
        if (depth - L0 > 8) return fail(c, PHOTONS_EINVAL, "build_leaves: more than 8 ORB levels below a 4096-particle node");
        PH_CUDA_BUILD(cudaFuncSetAttribute(orb_cta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        orb_cta_kernel<<<(unsigned)(1LL << L0), ORB_CTA_THREADS, smem, st>>>(n, L0, depth, P_cur, c->d_perm);
    } else {
        orb_perm_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, P_cur, c->d_perm);
    }
    ++c->launches;
    PH_CUDA_BUILD(cudaGetLastError());
    return PHOTONS_OK;
}

int build_leaves_impl(Ctx* c)
{
    const long long n = c->n;
    const int M = c->p.maxleaf;
    int depth = 0;
    while (((n + (1LL << depth) - 1) >> depth) > M) ++depth;
    const long long n_leaves = 1LL << depth;
    const long long n_slots = n_leaves * M;
    const long long n_nodes = 2 * n_leaves - 1;
    const int tb = 256;
    cudaStream_t st = c->streams[0];
    if (n_slots >= (1LL << 31)) return fail(c, PHOTONS_EINVAL, "build_leaves: more than 2^31 particle slots");
    if (depth - 7 > 24) return fail(c, PHOTONS_EINVAL, "build_leaves: tree too deep");

    PH_WS(c->d_perm, uint32_t, WS_PERM, n);
    int rc = orb_sort(c, depth, st);
    if (rc != PHOTONS_OK) return rc;

    c->depth = depth;
    c->n_leaves = n_leaves;
    c->n_slots = n_slots;
    PH_WS(c->d_leaf_cnt, int, WS_LEAF_CNT, n_leaves);
    PH_WS(c->d_node_lo, double, WS_NODE_LO, 3 * n_nodes);
    PH_WS(c->d_node_hi, double, WS_NODE_HI, 3 * n_nodes);
    PH_WS(c->d_leaf_ctr, double, WS_LEAF_CTR, 3 * n_leaves);
    PH_WS(c->d_slot_src, int, WS_SLOT_SRC, n_slots);
    PH_WS(c->d_p64, double4, WS_P64, n_slots);
    c->d_p32 = nullptr;
    if (c->p.precision != PHOTONS_FP64) PH_WS(c->d_p32, float, WS_P32, 4 * n_slots);
    {
        // the leaves' bboxes are the last n_leaves nodes of the heap arrays
        double* leaf_lo = c->d_node_lo + 3 * (n_leaves - 1);
        double* leaf_hi = c->d_node_hi + 3 * (n_leaves - 1);
        leaf_table_kernel<<<blocks_for(n_leaves, 128), 128, 0, st>>>(n, depth, n_leaves, c->d_perm, c->d_pos, c->d_leaf_cnt, leaf_lo, leaf_hi, c->d_leaf_ctr);
        // equal masses (set_particles) and a kernel that can leave G m out of the pair core (photons_params.mass_path)
        c->ugm = c->gm_uniform != 0.0 && c->p.mass_path == 0 && c->p.precision != PHOTONS_FP64 && c->p.g_mode != PHOTONS_G_DIRECT;
        pack_kernel<<<blocks_for(n_slots, tb), tb, 0, st>>>(n, depth, M, n_slots, c->p.G, c->p.precision, c->ugm ? 1 : 0, 1.0 / c->pscale, 1.0 / c->gmscale,
                                                            c->d_perm, c->d_pos, c->d_mass,
                                                            c->d_leaf_ctr, c->d_slot_src, c->d_p64, c->d_p32);
        c->launches += 2;
        for (int level = depth - 1; level >= 0; --level) {
            node_bbox_kernel<<<blocks_for(1LL << level, tb), tb, 0, st>>>(level, c->d_node_lo, c->d_node_hi);
            ++c->launches;
        }
    }

    // interaction list: count, scan, fill
    long long *d_nch = nullptr, *d_work = nullptr;
    unsigned long long* d_tot = nullptr;
    PH_WS(d_nch, long long, WS_LIST_NCH, n_leaves + 1);
    PH_WS(d_work, long long, WS_LIST_WORK, n_leaves);
    PH_WS(d_tot, unsigned long long, WS_LIST_TOT, 3);
    PH_WS(c->d_chunk_ptr, long long, WS_CHUNK_PTR, n_leaves + 1);
    PH_CUDA_BUILD(cudaMemsetAsync(d_tot, 0, sizeof(unsigned long long) * 3, st));
    PH_CUDA_BUILD(cudaMemsetAsync(d_nch, 0, sizeof(long long) * (n_leaves + 1), st));
    ListArgs la{};
    la.n_leaves = n_leaves; la.depth = depth; la.maxleaf = M; la.chunk_max = c->p.chunk_max;
    la.L = c->p.boxsize; la.rcut = c->r_cut; la.periodic = c->p.periodic;
    {
        float4* box = nullptr;
        PH_WS(box, float4, WS_NODE_BOX32, 2 * n_nodes);
        node_box32_kernel<<<blocks_for(n_nodes, tb), tb, 0, st>>>(n_nodes, n_leaves, c->d_leaf_cnt, c->d_node_lo, c->d_node_hi, box);
        ++c->launches;
        la.box = box;
    }
    la.leaf_cnt = c->d_leaf_cnt;
    la.chunk_ptr = nullptr; la.chunks = nullptr; la.n_chunks_of = d_nch; la.totals = d_tot; la.work_of = d_work;
    la.stash_cap = LIST_STASH;
    PH_WS(la.stash, uint2, WS_LIST_STASH, n_leaves * LIST_STASH);
    PH_WS(la.resume, int4, WS_LIST_RESUME, n_leaves);
    list_kernel<<<blocks_for(n_leaves, 64), 64, 0, st>>>(la);
    ++c->launches;
    {
        size_t scan_bytes = 0;
        PH_CUDA_BUILD(cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, d_nch, c->d_chunk_ptr, (int)(n_leaves + 1), st));
        void* tmp = workspace(c, WS_CUB_TMP, scan_bytes);
        if (!tmp) return PHOTONS_ENOMEM;
        PH_CUDA_BUILD(cub::DeviceScan::ExclusiveSum(tmp, scan_bytes, d_nch, c->d_chunk_ptr, (int)(n_leaves + 1), st));
    }
    unsigned long long h_tot[3] = {0, 0, 0};
    long long h_nchunks = 0;
    PH_CUDA_BUILD(cudaMemcpyAsync(&h_nchunks, c->d_chunk_ptr + n_leaves, sizeof(long long), cudaMemcpyDeviceToHost, st));
    PH_CUDA_BUILD(cudaMemcpyAsync(h_tot, d_tot, sizeof h_tot, cudaMemcpyDeviceToHost, st));
    PH_CUDA_BUILD(cudaStreamSynchronize(st));
    PH_WS(c->d_chunks, uint2, WS_CHUNKS, std::max<long long>(h_nchunks, 1));
    la.chunk_ptr = c->d_chunk_ptr; la.chunks = c->d_chunks;
    list_copy_kernel<<<blocks_for(32 * n_leaves, tb), tb, 0, st>>>(n_leaves, LIST_STASH, c->d_chunk_ptr, la.stash, c->d_chunks);
    list_kernel<<<blocks_for(n_leaves, 64), 64, 0, st>>>(la);
    c->launches += 2;

    // order in which the P2P kernel's CTAs take the target leaves (photons_params.leaf_order)
    PH_WS(c->d_order, int, WS_ORDER, n_leaves);
    if (c->p.leaf_order == 0) {
        // ORB order: neighbouring leaves run at the same time and find each other's source leaves in L2 (1.4 GB of
        // DRAM reads per launch on config 4 against 20 GB in longest-first order, at the same kernel time)
        order_identity_kernel<<<blocks_for(n_leaves, tb), tb, 0, st>>>(n_leaves, c->d_order);
        ++c->launches;
    } else {
        unsigned *d_okeys = nullptr, *d_okeys2 = nullptr;
        int* d_ovals = nullptr;
        PH_WS(d_okeys, unsigned, WS_ORDER_KEYS, n_leaves);
        PH_WS(d_okeys2, unsigned, WS_ORDER_KEYS2, n_leaves);
        PH_WS(d_ovals, int, WS_ORDER_VALS, n_leaves);
        order_keys_kernel<<<blocks_for(n_leaves, tb), tb, 0, st>>>(n_leaves, d_work, d_okeys, d_ovals);
        ++c->launches;
        size_t sort_bytes = 0;
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairsDescending(nullptr, sort_bytes, d_okeys, d_okeys2, d_ovals, c->d_order, (int)n_leaves, 0, 32, st));
        void* tmp = workspace(c, WS_CUB_TMP, sort_bytes);
        if (!tmp) return PHOTONS_ENOMEM;
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairsDescending(tmp, sort_bytes, d_okeys, d_okeys2, d_ovals, c->d_order, (int)n_leaves, 0, 32, st));
    }
    PH_CUDA_BUILD(cudaGetLastError());

    c->stats.n_particles = n;
    c->stats.n_leaves = n_leaves;
    c->stats.n_chunks = h_nchunks;
    c->stats.n_leaf_pairs = (long long)h_tot[0];
    c->stats.pairs_evaluated = (long long)h_tot[1];
    c->stats.max_leaves_per_target = (long long)h_tot[2] / M;
    return PHOTONS_OK;
}

}  // namespace photons
