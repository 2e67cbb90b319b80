// photons_build_leaves on the device: ORB sort, leaf-sorted packed particle arrays (L69),
// leaf table (L79) and the interaction list grouped by target leaf (the paper's TaskGroup/GroupIdx,
// L83-L85).  FEED steps a1-a3 of SURVEY.md §8(a); readings A10, A11, A13 of DESIGN.md.
#include <cub/cub.cuh>

#include <algorithm>
#include <cmath>

#include "common.cuh"

namespace photons {

void free_leaves(Ctx* c)
{
    cudaFree(c->d_perm); c->d_perm = nullptr;
    cudaFree(c->d_slot_src); c->d_slot_src = nullptr;
    cudaFree(c->d_leaf_cnt); c->d_leaf_cnt = nullptr;
    cudaFree(c->d_leaf_lo); c->d_leaf_lo = nullptr;
    cudaFree(c->d_leaf_hi); c->d_leaf_hi = nullptr;
    cudaFree(c->d_leaf_ctr); c->d_leaf_ctr = nullptr;
    cudaFree(c->d_node_lo); c->d_node_lo = nullptr;
    cudaFree(c->d_node_hi); c->d_node_hi = nullptr;
    cudaFree(c->d_p64); c->d_p64 = nullptr;
    cudaFree(c->d_p32); c->d_p32 = nullptr;
    cudaFree(c->d_chunk_ptr); c->d_chunk_ptr = nullptr;
    cudaFree(c->d_chunks); c->d_chunks = nullptr;
    cudaFree(c->d_order); c->d_order = nullptr;
    c->leaves_built = false;
    c->n_leaves = c->n_slots = 0;
}

// ---------------------------------------------------------------------------------------------- ORB
// One tree level: every segment (node) is split at its median along the axis of largest extent of
// its particle bounding box; the left child takes floor(size/2) particles (A13).  Implemented as a
// stable radix sort of (segment, fp32 coordinate) keys over the whole array.

__global__ void iota_kernel(long long n, uint32_t* idx)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) idx[i] = (uint32_t)i;
}

// bounding boxes of the segments of one level, as fp32 bit patterns (positions are >= 0, so the integer
// order of the bits is the float order)
__global__ void seg_bbox_kernel(long long n, int level, const uint32_t* __restrict__ idx,
                                const double* __restrict__ pos, int* __restrict__ lo, int* __restrict__ hi)
{
    long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const bool live = q < n;
    const long long qq = live ? q : n - 1;
    const long long seg = seg_of(n, level, qq);
    const uint32_t src = idx[qq];
    int v[3];
    for (int a = 0; a < 3; ++a) v[a] = __float_as_int((float)pos[3 * (size_t)src + a]);
    // warp-aggregate when the whole warp sits in one segment
    const long long seg0 = __shfl_sync(0xffffffffu, seg, 0);
    const bool uniform = __all_sync(0xffffffffu, seg == seg0);
    if (uniform) {
        for (int a = 0; a < 3; ++a) {
            int mn = v[a], mx = v[a];
            for (int o = 16; o; o >>= 1) {
                mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            }
            if ((threadIdx.x & 31) == 0) {
                atomicMin(&lo[3 * seg + a], mn);
                atomicMax(&hi[3 * seg + a], mx);
            }
        }
    } else if (live) {
        for (int a = 0; a < 3; ++a) {
            atomicMin(&lo[3 * seg + a], v[a]);
            atomicMax(&hi[3 * seg + a], v[a]);
        }
    }
}

__global__ void fill_int_kernel(long long n, int* p, int v)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

__global__ void seg_key_kernel(long long n, int level, const uint32_t* __restrict__ idx,
                               const double* __restrict__ pos, const int* __restrict__ lo,
                               const int* __restrict__ hi, unsigned long long* __restrict__ keys)
{
    long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (q >= n) return;
    const long long seg = seg_of(n, level, q);
    float ext[3];
    for (int a = 0; a < 3; ++a) ext[a] = __int_as_float(hi[3 * seg + a]) - __int_as_float(lo[3 * seg + a]);
    int axis = 0;                                   // largest extent, ties -> lowest axis
    if (ext[1] > ext[axis]) axis = 1;
    if (ext[2] > ext[axis]) axis = 2;
    const float x = (float)pos[3 * (size_t)idx[q] + axis];
    keys[q] = ((unsigned long long)seg << 32) | (unsigned long long)(uint32_t)__float_as_int(x);
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
// zero mass (they add nothing as sources and are never written as targets).
__global__ void pack_kernel(long long n, int depth, int maxleaf, long long n_slots, double G, int precision,
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
        b[0] = (float)(x - ox);
        b[2] = (float)(y - oy);
        b[4] = (float)(z - oz);
        b[6] = (float)gm;
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

struct ListArgs {
    long long n_leaves;
    int depth, maxleaf, chunk_max;
    double L, rcut;
    const double *node_lo, *node_hi;
    const int* leaf_cnt;
    const long long* chunk_ptr;   // pass 2
    uint2* chunks;                // pass 2
    long long* n_chunks_of;       // pass 1: per leaf
    unsigned long long* totals;   // pass 1: [0] leaf pairs, [1] pairs evaluated
    long long* work_of;           // pass 1: slots in the list of each leaf (for the heaviest-first order)
};

__global__ void list_kernel(ListArgs a)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= a.n_leaves) return;
    const long long leaf0 = a.n_leaves - 1;   // heap index of leaf 0
    double tl[3], th[3];
    for (int x = 0; x < 3; ++x) { tl[x] = a.node_lo[3 * (leaf0 + i) + x]; th[x] = a.node_hi[3 * (leaf0 + i) + x]; }
    const double rc2 = a.rcut * a.rcut;
    const int my_cnt = a.leaf_cnt[i];

    long long stack[40];
    int sp = 0;
    stack[sp++] = 0;
    long long run_first = -1, run_n = 0, n_chunks = 0, n_pairs = 0, n_eval = 0, work = 0;
    int run_code = -1;
    uint2* out = a.chunks ? a.chunks + a.chunk_ptr[i] : nullptr;
    const int max_leaves_per_chunk = a.chunk_max / a.maxleaf;

    while (sp) {
        const long long node = stack[--sp];
        double g2 = 0;
        int code = 0, mul = 1;
        bool ambiguous = false;
        for (int x = 0; x < 3; ++x) {
            const double nl = a.node_lo[3 * node + x], nh = a.node_hi[3 * node + x];
            const double hw = 0.5 * ((nh - nl) + (th[x] - tl[x]));
            double dc = 0.5 * ((nl + nh) - (tl[x] + th[x]));
            const double img = rint(dc / a.L);      // source is moved by -img box lengths
            dc -= a.L * img;
            const double gap = fmax(0.0, fabs(dc) - hw);
            g2 += gap * gap;
            code += mul * (1 - (int)img);
            mul *= 3;
            // the image is unique for every pair inside r_cut iff 2 r_cut + extents < L (A10)
            if (2.0 * a.rcut + 2.0 * hw >= a.L) ambiguous = true;
        }
        if (!(g2 < rc2)) continue;
        if (node < leaf0) {               // internal: right child first so the left one is popped first
            stack[sp++] = 2 * node + 2;
            stack[sp++] = 2 * node + 1;
            continue;
        }
        const long long j = node - leaf0;
        if (ambiguous) code = SHIFT_PER_PAIR;
        ++n_pairs;
        n_eval += (long long)my_cnt * a.leaf_cnt[j];
        work += a.maxleaf;
        if (run_n > 0 && j == run_first + run_n && code == run_code && run_n < max_leaves_per_chunk) {
            ++run_n;
        } else {
            if (run_n > 0) {
                if (out) out[n_chunks] = make_uint2((unsigned)(run_first * a.maxleaf), (unsigned)(run_n * a.maxleaf) | ((unsigned)run_code << 16));
                ++n_chunks;
            }
            run_first = j; run_n = 1; run_code = code;
        }
    }
    if (run_n > 0) {
        if (out) out[n_chunks] = make_uint2((unsigned)(run_first * a.maxleaf), (unsigned)(run_n * a.maxleaf) | ((unsigned)run_code << 16));
        ++n_chunks;
    }
    if (!a.chunks) {
        a.n_chunks_of[i] = n_chunks;
        a.work_of[i] = work;
        atomicAdd(&a.totals[0], (unsigned long long)n_pairs);
        atomicAdd(&a.totals[1], (unsigned long long)n_eval);
    }
}

__global__ void order_keys_kernel(long long n_leaves, const long long* __restrict__ work, unsigned* __restrict__ keys, int* __restrict__ vals)
{
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_leaves) return;
    keys[i] = (unsigned)min(work[i], 0xffffffffLL);
    vals[i] = (int)i;
}

// -------------------------------------------------------------------------------------------- driver

#define PH_CUDA_BUILD(call)                                                                                 \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess) {                                                                            \
            rc = fail(c, e_ == cudaErrorMemoryAllocation ? PHOTONS_ENOMEM : PHOTONS_ECUDA, "%s:%d %s: %s", \
                      __FILE__, __LINE__, #call, cudaGetErrorString(e_));                                   \
            goto done;                                                                                      \
        }                                                                                                   \
    } while (0)

static inline unsigned blocks_for(long long n, int tb) { return (unsigned)((n + tb - 1) / tb); }

int build_leaves_impl(Ctx* c)
{
    int rc = PHOTONS_OK;
    const long long n = c->n;
    const int M = c->p.maxleaf;
    int depth = 0;
    while (((n + (1LL << depth) - 1) >> depth) > M) ++depth;
    const long long n_leaves = 1LL << depth;
    const long long n_slots = n_leaves * M;
    const long long n_nodes = 2 * n_leaves - 1;
    const int tb = 256;
    cudaStream_t st = c->streams[0];

    // scratch (freed at the end)
    uint32_t* d_idx2 = nullptr;
    unsigned long long *d_keys = nullptr, *d_keys2 = nullptr;
    int *d_blo = nullptr, *d_bhi = nullptr;
    void* d_tmp = nullptr;
    size_t tmp_bytes = 0;
    long long *d_nch = nullptr, *d_work = nullptr;
    unsigned long long* d_tot = nullptr;
    unsigned *d_okeys = nullptr, *d_okeys2 = nullptr;
    int* d_ovals = nullptr;
    unsigned long long h_tot[2] = {0, 0};
    long long h_nchunks = 0, h_last = 0;
    ListArgs la{};

    if (n_slots >= (1LL << 31)) return fail(c, PHOTONS_EINVAL, "build_leaves: more than 2^31 particle slots");

    PH_CUDA_BUILD(cudaMalloc(&c->d_perm, sizeof(uint32_t) * n));
    iota_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, c->d_perm);
    ++c->launches;
    if (depth > 0) {
        PH_CUDA_BUILD(cudaMalloc(&d_idx2, sizeof(uint32_t) * n));
        PH_CUDA_BUILD(cudaMalloc(&d_keys, sizeof(unsigned long long) * n));
        PH_CUDA_BUILD(cudaMalloc(&d_keys2, sizeof(unsigned long long) * n));
        PH_CUDA_BUILD(cudaMalloc(&d_blo, sizeof(int) * 3 * (n_leaves / 2)));
        PH_CUDA_BUILD(cudaMalloc(&d_bhi, sizeof(int) * 3 * (n_leaves / 2)));
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, d_keys, d_keys2, c->d_perm, d_idx2, (int)n, 0, 64, st));
        PH_CUDA_BUILD(cudaMalloc(&d_tmp, tmp_bytes));
        uint32_t* cur = c->d_perm;
        uint32_t* alt = d_idx2;
        for (int level = 0; level < depth; ++level) {
            const long long nseg = 1LL << level;
            fill_int_kernel<<<blocks_for(3 * nseg, tb), tb, 0, st>>>(3 * nseg, d_blo, 0x7fffffff);
            ++c->launches;
            fill_int_kernel<<<blocks_for(3 * nseg, tb), tb, 0, st>>>(3 * nseg, d_bhi, 0);
            ++c->launches;
            seg_bbox_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, level, cur, c->d_pos, d_blo, d_bhi);
            ++c->launches;
            seg_key_kernel<<<blocks_for(n, tb), tb, 0, st>>>(n, level, cur, c->d_pos, d_blo, d_bhi, d_keys);
            ++c->launches;
            PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairs(d_tmp, tmp_bytes, d_keys, d_keys2, cur, alt, (int)n, 0, 32 + level, st));
            std::swap(cur, alt);
        }
        if (cur != c->d_perm) {   // keep the result in the buffer the context owns
            std::swap(c->d_perm, d_idx2);
        }
    }

    c->depth = depth;
    c->n_leaves = n_leaves;
    c->n_slots = n_slots;
    PH_CUDA_BUILD(cudaMalloc(&c->d_leaf_cnt, sizeof(int) * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&c->d_node_lo, sizeof(double) * 3 * n_nodes));
    PH_CUDA_BUILD(cudaMalloc(&c->d_node_hi, sizeof(double) * 3 * n_nodes));
    PH_CUDA_BUILD(cudaMalloc(&c->d_leaf_ctr, sizeof(double) * 3 * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&c->d_slot_src, sizeof(int) * n_slots));
    PH_CUDA_BUILD(cudaMalloc(&c->d_p64, sizeof(double4) * n_slots));
    if (c->p.precision != PHOTONS_FP64) PH_CUDA_BUILD(cudaMalloc(&c->d_p32, sizeof(float) * 4 * n_slots));
    {
        // the leaves' bboxes are the last n_leaves nodes of the heap arrays
        double* leaf_lo = c->d_node_lo + 3 * (n_leaves - 1);
        double* leaf_hi = c->d_node_hi + 3 * (n_leaves - 1);
        leaf_table_kernel<<<blocks_for(n_leaves, 128), 128, 0, st>>>(n, depth, n_leaves, c->d_perm, c->d_pos, c->d_leaf_cnt, leaf_lo, leaf_hi, c->d_leaf_ctr);
        ++c->launches;
        pack_kernel<<<blocks_for(n_slots, tb), tb, 0, st>>>(n, depth, M, n_slots, c->p.G, c->p.precision, c->d_perm, c->d_pos, c->d_mass,
                                                            c->d_leaf_ctr, c->d_slot_src, c->d_p64, c->d_p32);
        ++c->launches;
        for (int level = depth - 1; level >= 0; --level) {
            node_bbox_kernel<<<blocks_for(1LL << level, tb), tb, 0, st>>>(level, c->d_node_lo, c->d_node_hi);
            ++c->launches;
        }
    }

    // interaction list: count, scan, fill
    PH_CUDA_BUILD(cudaMalloc(&d_nch, sizeof(long long) * (n_leaves + 1)));
    PH_CUDA_BUILD(cudaMalloc(&d_work, sizeof(long long) * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&d_tot, sizeof(unsigned long long) * 2));
    PH_CUDA_BUILD(cudaMemsetAsync(d_tot, 0, sizeof(unsigned long long) * 2, st));
    PH_CUDA_BUILD(cudaMemsetAsync(d_nch, 0, sizeof(long long) * (n_leaves + 1), st));
    PH_CUDA_BUILD(cudaMalloc(&c->d_chunk_ptr, sizeof(long long) * (n_leaves + 1)));
    la.n_leaves = n_leaves; la.depth = depth; la.maxleaf = M; la.chunk_max = c->p.chunk_max;
    la.L = c->p.boxsize; la.rcut = c->r_cut;
    la.node_lo = c->d_node_lo; la.node_hi = c->d_node_hi; la.leaf_cnt = c->d_leaf_cnt;
    la.chunk_ptr = nullptr; la.chunks = nullptr; la.n_chunks_of = d_nch; la.totals = d_tot; la.work_of = d_work;
    list_kernel<<<blocks_for(n_leaves, 64), 64, 0, st>>>(la);
    ++c->launches;
    {
        size_t scan_bytes = 0;
        PH_CUDA_BUILD(cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, d_nch, c->d_chunk_ptr, (int)(n_leaves + 1), st));
        if (scan_bytes > tmp_bytes) {
            cudaFree(d_tmp); d_tmp = nullptr;
            PH_CUDA_BUILD(cudaMalloc(&d_tmp, scan_bytes));
            tmp_bytes = scan_bytes;
        }
        PH_CUDA_BUILD(cub::DeviceScan::ExclusiveSum(d_tmp, scan_bytes, d_nch, c->d_chunk_ptr, (int)(n_leaves + 1), st));
    }
    PH_CUDA_BUILD(cudaMemcpyAsync(&h_nchunks, c->d_chunk_ptr + n_leaves, sizeof(long long), cudaMemcpyDeviceToHost, st));
    PH_CUDA_BUILD(cudaMemcpyAsync(h_tot, d_tot, sizeof h_tot, cudaMemcpyDeviceToHost, st));
    PH_CUDA_BUILD(cudaStreamSynchronize(st));
    PH_CUDA_BUILD(cudaMalloc(&c->d_chunks, sizeof(uint2) * (size_t)std::max<long long>(h_nchunks, 1)));
    la.chunk_ptr = c->d_chunk_ptr; la.chunks = c->d_chunks;
    list_kernel<<<blocks_for(n_leaves, 64), 64, 0, st>>>(la);
    ++c->launches;

    // heaviest-first order of the target leaves
    PH_CUDA_BUILD(cudaMalloc(&c->d_order, sizeof(int) * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&d_okeys, sizeof(unsigned) * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&d_okeys2, sizeof(unsigned) * n_leaves));
    PH_CUDA_BUILD(cudaMalloc(&d_ovals, sizeof(int) * n_leaves));
    order_keys_kernel<<<blocks_for(n_leaves, tb), tb, 0, st>>>(n_leaves, d_work, d_okeys, d_ovals);
    ++c->launches;
    {
        size_t sort_bytes = 0;
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairsDescending(nullptr, sort_bytes, d_okeys, d_okeys2, d_ovals, c->d_order, (int)n_leaves, 0, 32, st));
        if (sort_bytes > tmp_bytes) {
            cudaFree(d_tmp); d_tmp = nullptr;
            PH_CUDA_BUILD(cudaMalloc(&d_tmp, sort_bytes));
            tmp_bytes = sort_bytes;
        }
        PH_CUDA_BUILD(cub::DeviceRadixSort::SortPairsDescending(d_tmp, sort_bytes, d_okeys, d_okeys2, d_ovals, c->d_order, (int)n_leaves, 0, 32, st));
    }
    PH_CUDA_BUILD(cudaMemcpyAsync(&h_last, d_okeys2, sizeof(unsigned), cudaMemcpyDeviceToHost, st));   // largest work
    PH_CUDA_BUILD(cudaStreamSynchronize(st));
    PH_CUDA_BUILD(cudaGetLastError());

    c->stats.n_particles = n;
    c->stats.n_leaves = n_leaves;
    c->stats.n_chunks = h_nchunks;
    c->stats.n_leaf_pairs = (long long)h_tot[0];
    c->stats.pairs_evaluated = (long long)h_tot[1];
    c->stats.max_leaves_per_target = (long long)(unsigned)h_last / M;

done:
    cudaFree(d_idx2); cudaFree(d_keys); cudaFree(d_keys2); cudaFree(d_blo); cudaFree(d_bhi); cudaFree(d_tmp);
    cudaFree(d_nch); cudaFree(d_work); cudaFree(d_tot); cudaFree(d_okeys); cudaFree(d_okeys2); cudaFree(d_ovals);
    return rc;
}

}  // namespace photons
