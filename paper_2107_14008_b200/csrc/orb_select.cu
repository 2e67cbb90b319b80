// ORB phase A by radix-select partition ("the particles belonged to a cell are equally assigned into two
// offspring cells"; A13, §6).
//
// A level of the ORB tree needs every node split at its median along one axis - a partition, not a sort.  Per level:
//   1. key + histogram : 24-bit fixed-point coordinate of every particle inside its node's bounding box along the node's
//                        widest axis (a monotone map), stored; per-node histogram of the top 8 bits
//   2. select x 3      : per node, the bin that holds the element of rank floor(size/2); two more histogram passes over
//                        the keys refine it to the exact 24-bit median key m and the number of keys below it
//   3. count           : per chunk of 2048 particles, how many keys are < m and == m
//   4. scan            : per node, exclusive sums of those counts over its chunks
//   5. scatter         : stable partition: keys < m and the first (floor(size/2) - #less) keys == m go left, the rest
//                        right, every side keeping its order; the children's bounding boxes are reduced on the way
// 64 bytes of HBM traffic per particle and level instead of ~120 for a 3-4 pass radix sort of (node, coordinate) keys
// plus key generation and gather.  Everything is integer counting: the result is deterministic.
#include <cub/cub.cuh>

#include "common.cuh"

namespace photons {

constexpr int SEL_THREADS = 256;
constexpr int SEL_ITEMS = 8;
constexpr int SEL_CHUNK = SEL_THREADS * SEL_ITEMS;   // particles per chunk
constexpr unsigned KEY_MAX = (1u << 24) - 1u;

struct SelLevel {              // device pointers of one level's chunk table
    int level, n_nodes, n_chunks;
    const int* ch_node;        // node of chunk c
    const long long* ch_q0;    // first sorted position of chunk c
    const int* ch_cnt;         // particles in chunk c (<= SEL_CHUNK)
    const int* node_chunk0;    // n_nodes + 1: first chunk of each node
};

__device__ __forceinline__ int sel_axis(const int* lo, const int* hi, long long node, float& l, float& inv_ext)
{
    float lv[3], ext[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { lv[a] = ord2f(lo[3 * node + a]); ext[a] = ord2f(hi[3 * node + a]) - lv[a]; }
    int axis = 0;                                   // largest extent, ties -> lowest axis (A13)
    if (ext[1] > ext[axis]) axis = 1;
    if (ext[2] > ext[axis]) axis = 2;
    l = lv[axis];
    inv_ext = ext[axis] > 0.f ? 1.0f / ext[axis] : 0.f;
    return axis;
}

// 1. keys and the histogram of their top digit
__global__ void __launch_bounds__(SEL_THREADS) sel_key_hist_kernel(SelLevel L, const float4* __restrict__ P, const int* __restrict__ lo,
                                                                   const int* __restrict__ hi, unsigned* __restrict__ keys,
                                                                   unsigned* __restrict__ hist)
{
    __shared__ unsigned sh[256];
    const int c = blockIdx.x, node = L.ch_node[c], cnt = L.ch_cnt[c];
    const long long q0 = L.ch_q0[c];
    sh[threadIdx.x] = 0;
    __syncthreads();
    float l, inv_ext;
    const int axis = sel_axis(lo, hi, node, l, inv_ext);
    for (int e = threadIdx.x; e < cnt; e += SEL_THREADS) {
        const float4 p = P[q0 + e];
        const float x = axis == 0 ? p.x : axis == 1 ? p.y : p.z;
        const unsigned k = (unsigned)fminf((x - l) * inv_ext * (float)KEY_MAX, (float)KEY_MAX);
        keys[q0 + e] = k;
        atomicAdd(&sh[k >> 16], 1u);
    }
    __syncthreads();
    if (sh[threadIdx.x]) atomicAdd(&hist[(size_t)node * 256 + threadIdx.x], sh[threadIdx.x]);
}

// 2. histogram of the next digit among the keys that match the digits chosen so far
__global__ void __launch_bounds__(SEL_THREADS) sel_hist_kernel(SelLevel L, int shift, const unsigned* __restrict__ keys,
                                                               const unsigned* __restrict__ prefix, unsigned* __restrict__ hist)
{
    __shared__ unsigned sh[256];
    const int c = blockIdx.x, node = L.ch_node[c], cnt = L.ch_cnt[c];
    const long long q0 = L.ch_q0[c];
    sh[threadIdx.x] = 0;
    __syncthreads();
    const unsigned want = prefix[node];               // the digits above `shift + 8`
    for (int e = threadIdx.x; e < cnt; e += SEL_THREADS) {
        const unsigned k = keys[q0 + e];
        if ((k >> (shift + 8)) == want) atomicAdd(&sh[(k >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (sh[threadIdx.x]) atomicAdd(&hist[(size_t)node * 256 + threadIdx.x], sh[threadIdx.x]);
}

// one warp per node: the bin that holds rank[node]; rank becomes the rank inside that bin; below[node] += keys below it
__global__ void sel_pick_kernel(int n_nodes, const unsigned* __restrict__ hist, unsigned* __restrict__ prefix,
                                unsigned* __restrict__ rank, unsigned* __restrict__ below, unsigned* __restrict__ ties)
{
    const int node = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (node >= n_nodes) return;
    const unsigned* h = hist + (size_t)node * 256;
    unsigned v[8], s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { v[i] = h[lane * 8 + i]; s += v[i]; }
    unsigned inc = s;                                 // inclusive scan of the lanes' sums
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    const unsigned r = rank[node];
    unsigned cum = inc - s;
    int bin = -1;
    unsigned cb = 0, hb = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        if (bin < 0 && r >= cum && r < cum + v[i]) { bin = lane * 8 + i; cb = cum; hb = v[i]; }
        cum += v[i];
    }
    const unsigned owner = __ballot_sync(0xffffffffu, bin >= 0);
    const int src = __ffs(owner) - 1;                 // exactly one lane holds the bin (rank < total)
    bin = __shfl_sync(0xffffffffu, bin, src);
    cb = __shfl_sync(0xffffffffu, cb, src);
    hb = __shfl_sync(0xffffffffu, hb, src);
    if (lane == 0) {
        prefix[node] = (prefix[node] << 8) | (unsigned)bin;
        rank[node] = r - cb;
        below[node] += cb;
        ties[node] = hb;                              // after the last digit: keys equal to the median key
    }
}

__global__ void sel_init_kernel(long long n, int level, int n_nodes, unsigned* __restrict__ prefix, unsigned* __restrict__ rank,
                                unsigned* __restrict__ below)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_nodes) return;
    const long long s0 = seg_start(n, level, k), s1 = k + 1 == n_nodes ? n : seg_start(n, level, k + 1);
    prefix[k] = 0;
    rank[k] = (unsigned)((s1 - s0) >> 1);             // the first element of the right child (left takes floor(size/2))
    below[k] = 0;
}

// 3. per chunk: keys below / equal to the node's median key
__global__ void __launch_bounds__(SEL_THREADS) sel_count_kernel(SelLevel L, const unsigned* __restrict__ keys, const unsigned* __restrict__ median,
                                                                uint2* __restrict__ ch_cnt2)
{
    __shared__ unsigned s_less, s_tie;
    const int c = blockIdx.x, node = L.ch_node[c], cnt = L.ch_cnt[c];
    const long long q0 = L.ch_q0[c];
    if (threadIdx.x == 0) { s_less = 0; s_tie = 0; }
    __syncthreads();
    const unsigned m = median[node];
    unsigned less = 0, tie = 0;
    for (int e = threadIdx.x; e < cnt; e += SEL_THREADS) {
        const unsigned k = keys[q0 + e];
        less += k < m;
        tie += k == m;
    }
    less = __reduce_add_sync(0xffffffffu, less);
    tie = __reduce_add_sync(0xffffffffu, tie);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_less, less); atomicAdd(&s_tie, tie); }
    __syncthreads();
    if (threadIdx.x == 0) ch_cnt2[c] = make_uint2(s_less, s_tie);
}

// 4. one CTA per node: exclusive sums of (less, tie) over the node's chunks
__global__ void __launch_bounds__(256) sel_scan_kernel(SelLevel L, const uint2* __restrict__ ch_cnt2, uint2* __restrict__ ch_base)
{
    typedef cub::BlockScan<unsigned long long, 256> Scan;
    __shared__ typename Scan::TempStorage tmp;
    __shared__ unsigned long long carry;
    const int node = blockIdx.x, c0 = L.node_chunk0[node], c1 = L.node_chunk0[node + 1];
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b = c0; b < c1; b += 256) {
        const int c = b + threadIdx.x;
        const uint2 v = c < c1 ? ch_cnt2[c] : make_uint2(0u, 0u);
        const unsigned long long packed = ((unsigned long long)v.y << 32) | v.x;     // both sums stay below 2^32
        unsigned long long ex, total;
        Scan(tmp).ExclusiveSum(packed, ex, total);
        ex += carry;
        if (c < c1) ch_base[c] = make_uint2((unsigned)(ex & 0xffffffffu), (unsigned)(ex >> 32));
        __syncthreads();
        if (threadIdx.x == 0) carry += total;
        __syncthreads();
    }
}

// 5. stable partition of every node about its median key; child bounding boxes on the way (lo2 == nullptr: not needed).
// A chunk is dealt to its 8 warps in blocks of 256 elements and to the lanes of a warp round-robin: loads are
// lane-contiguous, ranks inside a warp come from ballots, and the lanes that go to the same side store to consecutive
// addresses.  The boxes are reduced over the whole CTA (a chunk lies inside one node) before the global atomics.
__global__ void __launch_bounds__(SEL_THREADS) sel_scatter_kernel(SelLevel L, long long n, const float4* __restrict__ P,
                                                                  const unsigned* __restrict__ keys, const unsigned* __restrict__ median,
                                                                  const unsigned* __restrict__ below, const unsigned* __restrict__ ties,
                                                                  const uint2* __restrict__ ch_base, float4* __restrict__ P_out,
                                                                  int* __restrict__ lo2, int* __restrict__ hi2)
{
    constexpr int NW = SEL_THREADS / 32;
    __shared__ unsigned wtot[NW];
    __shared__ int s_mn[NW][6], s_mx[NW][6];
    const int c = blockIdx.x, node = L.ch_node[c], cnt = L.ch_cnt[c];
    const long long q0 = L.ch_q0[c];
    const long long s0 = seg_start(n, L.level, node), s1 = node + 1 == L.n_nodes ? n : seg_start(n, L.level, node + 1);
    const unsigned left = (unsigned)((s1 - s0) >> 1);
    const unsigned m = median[node], less_total = below[node], tie_total = ties[node];
    const unsigned need = left - less_total;          // ties that still go left
    const uint2 base = ch_base[c];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int e0 = warp * (32 * SEL_ITEMS) + lane;    // element i of this thread: e0 + 32 i
    unsigned k[SEL_ITEMS], ex[SEL_ITEMS];
    float4 p[SEL_ITEMS];
    unsigned run = 0;                                 // packed (ties << 16 | less) of this warp's elements so far
#pragma unroll
    for (int i = 0; i < SEL_ITEMS; ++i) {
        const int e = e0 + 32 * i;
        const bool live = e < cnt;
        k[i] = live ? keys[q0 + e] : 0xffffffffu;
        if (live) p[i] = P[q0 + e];
        const unsigned bl = __ballot_sync(0xffffffffu, k[i] < m), bt = __ballot_sync(0xffffffffu, k[i] == m);
        ex[i] = run + (unsigned)__popc(bl & lt_mask) + ((unsigned)__popc(bt & lt_mask) << 16);
        run += (unsigned)__popc(bl) + ((unsigned)__popc(bt) << 16);
    }
    if (lane == 0) wtot[warp] = run;
    __syncthreads();
    unsigned wb = 0;
    for (int w = 0; w < warp; ++w) wb += wtot[w];
    int mn[2][3], mx[2][3];
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int a = 0; a < 3; ++a) { mn[s][a] = 0x7fffffff; mx[s][a] = (int)0x80000000; }
#pragma unroll
    for (int i = 0; i < SEL_ITEMS; ++i) {
        const int e = e0 + 32 * i;
        if (e >= cnt) continue;
        const unsigned rel = ex[i] + wb;
        const unsigned lb = base.x + (rel & 0xffffu), tb = base.y + (rel >> 16);   // less / tie elements of this node before mine
        const unsigned idx = (unsigned)(q0 + e - s0);     // position inside the node
        unsigned dst;
        int side;
        if (k[i] < m) { dst = lb; side = 0; }
        else if (k[i] == m) {
            if (tb < need) { dst = less_total + tb; side = 0; }
            else { dst = left + (tb - need); side = 1; }
        } else {
            dst = left + (tie_total - need) + (idx - (lb + tb));      // greater elements before mine
            side = 1;
        }
        P_out[s0 + dst] = p[i];
        const int v[3] = {f2ord(p[i].x), f2ord(p[i].y), f2ord(p[i].z)};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (side == 0) { mn[0][a] = min(mn[0][a], v[a]); mx[0][a] = max(mx[0][a], v[a]); }
            else { mn[1][a] = min(mn[1][a], v[a]); mx[1][a] = max(mx[1][a], v[a]); }
        }
    }
    if (!lo2) return;
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int wmn = __reduce_min_sync(0xffffffffu, mn[s][a]), wmx = __reduce_max_sync(0xffffffffu, mx[s][a]);
            if (lane == 0) { s_mn[warp][3 * s + a] = wmn; s_mx[warp][3 * s + a] = wmx; }
        }
    __syncthreads();
    if (threadIdx.x < 6) {
        int bmn = s_mn[0][threadIdx.x], bmx = s_mx[0][threadIdx.x];
        for (int w = 1; w < NW; ++w) { bmn = min(bmn, s_mn[w][threadIdx.x]); bmx = max(bmx, s_mx[w][threadIdx.x]); }
        if (bmn <= bmx) {                              // threadIdx.x = 3 side + axis
            atomicMin(&lo2[6 * (size_t)node + threadIdx.x], bmn);
            atomicMax(&hi2[6 * (size_t)node + threadIdx.x], bmx);
        }
    }
}

__global__ void sel_fill_kernel(long long n, int* p, int v)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// Chunk tables of all phase-A levels (they depend on n and L0 only): built on the host once, kept on the device.
static int sel_tables(Ctx* c, int L0)
{
    const long long n = c->n;
    if (c->sel_n == n && c->sel_L0 == L0) return PHOTONS_OK;
    std::vector<int> ch_node, ch_cnt, node_c0;
    std::vector<long long> ch_q0;
    c->sel_off.assign(L0 + 1, 0);
    c->sel_noff.assign(L0 + 1, 0);
    for (int l = 0; l < L0; ++l) {
        const long long nodes = 1LL << l;
        for (long long k = 0; k < nodes; ++k) {
            const long long s0 = seg_start(n, l, k), s1 = k + 1 == nodes ? n : seg_start(n, l, k + 1);
            node_c0.push_back((int)(ch_node.size() - c->sel_off[l]));
            for (long long q = s0; q < s1; q += SEL_CHUNK) {
                ch_node.push_back((int)k);
                ch_q0.push_back(q);
                ch_cnt.push_back((int)std::min<long long>(SEL_CHUNK, s1 - q));
            }
        }
        node_c0.push_back((int)(ch_node.size() - c->sel_off[l]));
        c->sel_off[l + 1] = (long long)ch_node.size();
        c->sel_noff[l + 1] = (long long)node_c0.size();
    }
    int *d_node = static_cast<int*>(workspace(c, WS_SEL_NODE, sizeof(int) * ch_node.size()));
    int* d_cnt = static_cast<int*>(workspace(c, WS_SEL_CNT, sizeof(int) * ch_cnt.size()));
    long long* d_q0 = static_cast<long long*>(workspace(c, WS_SEL_Q0, sizeof(long long) * ch_q0.size()));
    int* d_c0 = static_cast<int*>(workspace(c, WS_SEL_C0, sizeof(int) * node_c0.size()));
    if (!d_node || !d_cnt || !d_q0 || !d_c0) return PHOTONS_ENOMEM;
    PH_CUDA(c, cudaMemcpy(d_node, ch_node.data(), sizeof(int) * ch_node.size(), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMemcpy(d_cnt, ch_cnt.data(), sizeof(int) * ch_cnt.size(), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMemcpy(d_q0, ch_q0.data(), sizeof(long long) * ch_q0.size(), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMemcpy(d_c0, node_c0.data(), sizeof(int) * node_c0.size(), cudaMemcpyHostToDevice));
    c->sel_n = n;
    c->sel_L0 = L0;
    return PHOTONS_OK;
}

#define SEL_WS(ptr, type, slot, count)                                                     \
    do {                                                                                   \
        (ptr) = static_cast<type*>(workspace(c, (slot), sizeof(type) * (size_t)(count)));  \
        if (!(ptr)) return PHOTONS_ENOMEM;                                                 \
    } while (0)

// Levels 0 .. L0-1.  In: P_cur in any order, lo/hi = bounding box of the root (ordered ints).  Out: P_cur grouped by
// level-L0 node (P_alt is the other buffer).
int orb_phase_a_select(Ctx* c, int L0, float4*& P_cur, float4*& P_alt, int* lo, int* hi, cudaStream_t st)
{
    const long long n = c->n;
    int rc = sel_tables(c, L0);
    if (rc != PHOTONS_OK) return rc;
    const int* d_node = static_cast<const int*>(c->ws[WS_SEL_NODE].p);
    const int* d_cnt = static_cast<const int*>(c->ws[WS_SEL_CNT].p);
    const long long* d_q0 = static_cast<const long long*>(c->ws[WS_SEL_Q0].p);
    const int* d_c0 = static_cast<const int*>(c->ws[WS_SEL_C0].p);
    const long long max_nodes = 1LL << (L0 - 1);
    long long max_chunks = 0;
    for (int l = 0; l < L0; ++l) max_chunks = std::max(max_chunks, c->sel_off[l + 1] - c->sel_off[l]);
    unsigned *keys = nullptr, *hist = nullptr, *prefix = nullptr, *rank = nullptr, *below = nullptr, *ties = nullptr;
    uint2 *cnt2 = nullptr, *base2 = nullptr;
    int *lo2 = nullptr, *hi2 = nullptr;
    SEL_WS(keys, unsigned, WS_ORB_KEYS, n);
    SEL_WS(hist, unsigned, WS_SEL_HIST, 3 * 256 * max_nodes);
    SEL_WS(prefix, unsigned, WS_SEL_NODEVAR, 4 * max_nodes);
    rank = prefix + max_nodes; below = rank + max_nodes; ties = below + max_nodes;
    SEL_WS(cnt2, uint2, WS_SEL_CNT2, max_chunks);
    SEL_WS(base2, uint2, WS_SEL_BASE2, max_chunks);
    SEL_WS(lo2, int, WS_SEL_LO2, 3LL << L0);
    SEL_WS(hi2, int, WS_SEL_HI2, 3LL << L0);
    for (int level = 0; level < L0; ++level) {
        SelLevel L{};
        L.level = level; L.n_nodes = 1 << level; L.n_chunks = (int)(c->sel_off[level + 1] - c->sel_off[level]);
        L.ch_node = d_node + c->sel_off[level]; L.ch_q0 = d_q0 + c->sel_off[level]; L.ch_cnt = d_cnt + c->sel_off[level];
        L.node_chunk0 = d_c0 + c->sel_noff[level];
        const unsigned nb_nodes = (unsigned)((L.n_nodes + 255) / 256);
        const unsigned nb_warps = (unsigned)((32LL * L.n_nodes + 255) / 256);
        PH_CUDA(c, cudaMemsetAsync(hist, 0, sizeof(unsigned) * 3 * 256 * (size_t)L.n_nodes, st));
        sel_init_kernel<<<nb_nodes, 256, 0, st>>>(n, level, L.n_nodes, prefix, rank, below);
        sel_key_hist_kernel<<<L.n_chunks, SEL_THREADS, 0, st>>>(L, P_cur, lo, hi, keys, hist);
        sel_pick_kernel<<<nb_warps, 256, 0, st>>>(L.n_nodes, hist, prefix, rank, below, ties);
        sel_hist_kernel<<<L.n_chunks, SEL_THREADS, 0, st>>>(L, 8, keys, prefix, hist + 256 * (size_t)L.n_nodes);
        sel_pick_kernel<<<nb_warps, 256, 0, st>>>(L.n_nodes, hist + 256 * (size_t)L.n_nodes, prefix, rank, below, ties);
        sel_hist_kernel<<<L.n_chunks, SEL_THREADS, 0, st>>>(L, 0, keys, prefix, hist + 512 * (size_t)L.n_nodes);
        sel_pick_kernel<<<nb_warps, 256, 0, st>>>(L.n_nodes, hist + 512 * (size_t)L.n_nodes, prefix, rank, below, ties);
        sel_count_kernel<<<L.n_chunks, SEL_THREADS, 0, st>>>(L, keys, prefix, cnt2);
        sel_scan_kernel<<<L.n_nodes, 256, 0, st>>>(L, cnt2, base2);
        const bool more = level + 1 < L0;            // the next level's boxes, reduced while the partition is applied
        if (more) {
            const long long nb = 3LL << (level + 1);
            sel_fill_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, st>>>(nb, lo2, 0x7fffffff);
            sel_fill_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, st>>>(nb, hi2, (int)0x80000000);
            c->launches += 2;
        }
        sel_scatter_kernel<<<L.n_chunks, SEL_THREADS, 0, st>>>(L, n, P_cur, keys, prefix, below, ties, base2, P_alt, more ? lo2 : nullptr, hi2);
        c->launches += 10;
        std::swap(P_cur, P_alt);
        std::swap(lo, lo2);
        std::swap(hi, hi2);
    }
    PH_CUDA(c, cudaGetLastError());
    return PHOTONS_OK;
}

}  // namespace photons
