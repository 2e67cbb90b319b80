/*
 * photons.h — C ABI of the B200-native truncated short-range gravity P2P library.
 *
 * What the library computes (§2, Eq. 1; BASELINE.json north_star):
 *
 *   a_i = G * sum_{j != i, 0 < |d_ij| < r_cut}  m_j * d_ij * g(|d_ij|) / |d_ij|^3
 *   g(r) = erfc(r / 2 r_s) + r / (r_s sqrt(pi)) * exp(-r^2 / 4 r_s^2)              (Eq. 1)
 *   r_s  = rs_over_cell * boxsize / n_pm   (1.2 cells, L33),  r_cut = rcut_over_rs * r_s (6, L53/L143)
 *   d_ij = minimum image of (r_j - r_i) in the periodic cube of side boxsize
 *
 * evaluated the paper's way (§3, Alg. 1/2): particles sorted into the leaves of an ORB tree
 * (<= maxleaf particles each, L35), every target leaf summing over the source leaves whose
 * periodic bounding boxes come within r_cut of its own (the "P2P task list", L65, L77-L85).
 *
 * Conventions for every entry point
 *   - plain C: no C++ types, no exceptions cross this boundary; every call returns a PHOTONS_* status;
 *     out-parameters are untouched on error; photons_last_error() gives the message.
 *   - "host or device" pointers are tagged by a PHOTONS_MEM_* argument.  The caller owns pos, mass and
 *     acc; the library copies inputs inside photons_set_particles and keeps no caller pointer.
 *   - the context owns all device buffers and CUDA streams; a context is not thread-safe; different
 *     contexts are independent.
 *   - call order: create -> set_particles -> build_leaves -> short_range_acc (repeatable);
 *     set_particles invalidates the leaves.  A call out of order returns PHOTONS_ESTATE.
 *   - there is no CPU fallback: without a CUDA device photons_create fails with PHOTONS_ENODEVICE.
 */
#ifndef PHOTONS_H
#define PHOTONS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct photons_ctx photons_ctx; /* opaque; owned by the library */

enum {
    PHOTONS_OK = 0,
    PHOTONS_EINVAL = 1,     /* bad argument or parameter */
    PHOTONS_ESTATE = 2,     /* call out of order */
    PHOTONS_ENOMEM = 3,     /* host or device allocation failed */
    PHOTONS_ECUDA = 4,      /* CUDA runtime error (message in photons_last_error) */
    PHOTONS_ENODEVICE = 5,  /* no usable CUDA device */
    PHOTONS_EBOX = 6,       /* periodic box with r_cut >= boxsize/2: the minimum image is not unique (photons_create).
                               Leaves so large that 2 r_cut + both extents >= boxsize are NOT an error: their list
                               entries take the minimum image per pair instead (shift code 27; A10) */
    PHOTONS_ENONFINITE = 7  /* NaN/Inf in positions or masses */
};

/* precision of the P2P path (SP and DP runs; "mixed": north_star) */
enum {
    PHOTONS_FP64 = 0,   /* fp64 positions, fp64 pair arithmetic */
    PHOTONS_FP32 = 1,   /* absolute positions stored in fp32, fp32 pair arithmetic */
    PHOTONS_MIXED = 2   /* fp32 offsets from the leaf centre (centres and centre differences in fp64),
                           fp32 pair arithmetic */
};

/* how the truncation function g is evaluated inside the pair core (§3.3) */
enum {
    PHOTONS_G_DIRECT = 0, /* erfc/exp special functions per pair (what §3.3 L121 calls expensive) */
    PHOTONS_G_TABLE = 1,  /* Eq. 2 (L127-L143): table {T_i, E_i} in shared memory + Taylor terms T[0..level] */
    PHOTONS_G_POLY = 2,   /* no table, no special function: g/r^3 = 1/r^3 - Q(s)/(2 r_s)^3 with
                             s = (r/2r_s)^2 and Q an FMA-pipe polynomial (fp32 paths only) */
    PHOTONS_G_FUSED = 3   /* Eq. 1 evaluated directly per pair by a hand-fused routine instead of the stock erfcf/expf
                             of G_DIRECT: g = exp(-x^2) H(x), the Gaussian by one ex2.approx (XU pipe), H = erfcx(x) +
                             2x/sqrt(pi) by a polynomial of degree poly_degree (fp32 paths only) */
};

/* what the interpolation table holds per node (PHOTONS_G_TABLE) */
enum {
    PHOTONS_TABLE_PAPER = 0, /* {T_i, E_i} as in the paper (L143); the polynomials of Eq. 2 in x_i are rebuilt per pair */
    PHOTONS_TABLE_COEF = 1,  /* the Taylor coefficients of Eq. 2 themselves, T^(k)(x_i) h^k / k!, k = 0..table_level: the
                                same series about the same node, Horner only (PHOTONS_FP64 only) */
    PHOTONS_TABLE_QUAD = 2   /* {T_i, E_i} plus the two highest node polynomials of Eq. 2, the brackets of T[3] and T[4]
                                (L137-L141), tabulated instead of rebuilt per pair: 32 bytes per node (PHOTONS_FP64 only) */
};

enum { PHOTONS_MEM_HOST = 0, PHOTONS_MEM_DEVICE = 1 };

/* element type of caller arrays (pos, mass, acc) */
enum { PHOTONS_DTYPE_F64 = 0, PHOTONS_DTYPE_F32 = 1 };

typedef struct {
    double boxsize;           /* > 0; period of the cube */
    int n_pm;                 /* PM mesh cells per side (L33); must give r_cut < boxsize/2 */
    double rs_over_cell;      /* split radius in cells: 1.2 (L33) */
    double rcut_over_rs;      /* cut-off in r_s: 6.0 (north_star; the table spans x = r/2r_s in [0,3], L143);
                                 must be <= 6 for g_mode TABLE, POLY and FUSED (their range), any value for DIRECT */
    double G;                 /* gravitational constant */
    int maxleaf;              /* MAXLEAF (L35): 16, 32, 64 or 128 */
    int precision;            /* PHOTONS_FP64 / FP32 / MIXED */
    int g_mode;               /* PHOTONS_G_* */
    int table_nodes;          /* TABLE: number of intervals n over x in [0,3] (n+1 nodes), 64..4096; paper: 512 */
    int table_level;          /* TABLE: highest Taylor term kept (paper: T[2] for SP, T[4] for DP, L149): 0..4 with
                                 PHOTONS_FP64, 0..3 with FP32 / MIXED (T[2] already sits on the fp32 floor) */
    int n_streams;            /* >= 1: target-leaf batches are issued round-robin over this many CUDA streams */
    int device;               /* CUDA device ordinal */
    double close_pair_radius; /* fp32/mixed paths, exact path (A12): a staged run of sources whose fp32 partial
                                 acceleration on a target exceeds max|G m| / close_pair_radius^2 - what one pair at this
                                 separation gives - is re-evaluated in fp64 for that target inside the kernel; 0 = off.
                                 Ignored by PHOTONS_FP64. */
    int chunk_max;            /* largest number of source particle slots staged per shared-memory stage;
                                 0 = default (128); multiple of maxleaf, <= 256 */
    int warps_per_leaf;       /* warps of the CTA that owns one target leaf; they split its source list.
                                 0 = default; 1, 2, 4 or 8 */
    int targets_per_lane;     /* fp32/mixed kernels: targets a lane keeps in registers, 1, 2 or 4 (the warp then splits
                                 into 32 T / maxleaf groups that take alternate source pairs); 0 = default.
                                 Available: maxleaf 16: 1, 2; 32: 1, 2; 64: 2; 128: 4 */
    int poly_degree;          /* POLY: degree of Q in the mapped variable, 10..14; 0 = default (12).
                                 FUSED: degree of H, 9..11; 0 = default (10) */
    int periodic;             /* 1 = periodic cube of side boxsize, minimum image (default; north_star);
                                 0 = isolated boundaries: no images, positions are not wrapped,
                                 boxsize only sets r_s = rs_over_cell * boxsize / n_pm */
    double softening;         /* Plummer softening length eps >= 0 (A23): the pair function is
                                 taken at r_eps = sqrt(r^2 + eps^2), a_i += G m_j d_ij g(r_eps) / r_eps^3 for pairs with
                                 0 < r and r_eps < r_cut.  0 = none (default; north_star's formula) */
    int table_layout;         /* TABLE: PHOTONS_TABLE_PAPER (default), PHOTONS_TABLE_COEF or PHOTONS_TABLE_QUAD */
    int leaf_order;           /* order in which CTAs take the target leaves: 0 = ORB order (default: neighbouring leaves run
                                 together and share their source leaves in L2), 1 = longest source list first */
    int orb_method;           /* upper levels of the ORB build: 0 = radix-select partition of every node about its median
                                 (default), 1 = one full radix sort of (node, coordinate) keys per level (round-1 path) */
    int mass_path;            /* fp32 and mixed kernels with g_mode POLY, FUSED or TABLE: 0 = when photons_set_particles finds every mass
                                 equal (one particle species, the paper's runs; Alg. 2 L177 carries a single GM) the pair core
                                 leaves G m out and applies it once per staged run (default); 1 = always G m_j per pair.
                                 Same sums up to fp32 rounding order. */
} photons_params;

typedef struct {
    long long n_particles;
    long long n_leaves;        /* leaves of the ORB tree (all at the same depth) */
    long long n_chunks;        /* interaction-list entries: runs of contiguous source leaves, <= chunk_max slots */
    long long n_leaf_pairs;    /* (target leaf, source leaf) tasks, the paper's Task list length (L77) */
    long long pairs_evaluated; /* sum over tasks of n_i * n_j, real particles only (paper's count, L218; A18) */
    long long max_leaves_per_target; /* longest source list, in leaves */
    double build_ms;           /* last photons_build_leaves: CUDA-event time of its device work (the call itself returns
                                  once that work is enqueued; the value is read at the next synchronisation) */
    double kernel_ms;          /* last photons_short_range_acc: CUDA-event time of the P2P launches alone */
    double total_ms;           /* last photons_short_range_acc: host wall clock incl. copies and sync */
    long long kernel_launches; /* kernels of this library launched on ctx since photons_create (the CUB sort and
                                  scan launches inside photons_build_leaves are library code and not counted) */
} photons_stats;

/* Fill *p with the paper's defaults: boxsize 1, n_pm 32, rs_over_cell 1.2, rcut_over_rs 6, G 1, maxleaf 32,
 * FP32, G_POLY, table 512/level 2, 1 stream, device 0, close pairs off, chunk_max default, periodic, no softening. */
void photons_default_params(photons_params* p);

/* Validate parameters, select the device, create streams, build the g table (TABLE mode; fp64 on the
 * host, rounded once).  Errors: EINVAL, EBOX (r_cut >= boxsize/2), ENODEVICE, ECUDA, ENOMEM.
 * On error *out is untouched and, if err_buf != NULL, a message is written there (err_len bytes). */
int photons_create(const photons_params* p, photons_ctx** out, char* err_buf, int err_len);

/* Make `cuda_stream` (a cudaStream_t; NULL = back to the context's own stream) the context's main stream:
 * build_leaves and short_range_acc enqueue on it (extra streams of n_streams > 1 fork from it and join it
 * again), so events the caller records on that stream bracket the library's device work.  The stream stays
 * the caller's.  Errors: EINVAL (null ctx). */
int photons_set_stream(photons_ctx* ctx, void* cuda_stream);

/* Copy n particles in.  pos: n x 3 row-major, mass: n values or NULL (= 1/n each), both of element type
 * dtype (PHOTONS_DTYPE_*), both host or both device memory as tagged.  Positions are wrapped into
 * [0, boxsize).  Any units: the fp32 / mixed kernels work on positions divided by a power of two near r_cut and
 * on G m_j divided by a power of two >= max |G m_j| (both exact rescalings, undone in fp64 on output), so
 * neither a large G m nor a large or tiny boxsize can overflow or underflow their fp32 arithmetic.  cuda_stream: a cudaStream_t the device-side copy is enqueued on (NULL = the context's main stream);
 * the call returns after the copy has completed.  Errors: EINVAL (n < 1, or more than 2^31 - 1 particle slots),
 * ENONFINITE, ENOMEM, ECUDA. */
int photons_set_particles(photons_ctx* ctx, long long n, const void* pos, const void* mass, int dtype,
                          int mem_kind, void* cuda_stream);

/* ORB sort (L35) -> leaf-sorted packed particle arrays in the path's precision (SoA by leaf, L69),
 * leaf table (L79: first slot, count; plus tight bounding boxes), interaction list grouped by target leaf
 * with the periodic image shift of every entry (the paper's TaskGroup/GroupIdx, L83-L85).  All on the
 * device.  Errors: ESTATE, EBOX, ENOMEM, ECUDA. */
int photons_build_leaves(photons_ctx* ctx);

/* The P2P kernel (Alg. 1 + Alg. 2): acc[n x 3] row-major in the CALLER's particle order, element type
 * dtype, host or device memory.  stats may be NULL.  Errors: ESTATE, EINVAL, ECUDA. */
int photons_short_range_acc(photons_ctx* ctx, void* acc, int dtype, int mem_kind, photons_stats* stats);

/* Test hooks (host output buffers).  perm[q] = caller index of the particle at leaf-sorted position q
 * (n entries); leaf_start[k] = first sorted position of leaf k (n_leaves + 1 entries).  Either may be NULL. */
int photons_get_leaf_order(photons_ctx* ctx, long long* perm, long long* leaf_start);

/* Interaction list as built: chunk_ptr[n_leaves + 1], then per chunk: first source leaf, number of source
 * leaves, shift code (sx+1) + 3*(sy+1) + 9*(sz+1) with s in {-1,0,+1} box lengths added to the source.
 * Pass NULL pointers to query sizes through stats only. */
int photons_get_interaction_list(photons_ctx* ctx, long long* chunk_ptr, int* first_leaf, int* n_leaf,
                                 int* shift_code);

/* Statistics of the last build / run. */
int photons_get_stats(photons_ctx* ctx, photons_stats* stats);

/* Device throughput micro-benchmarks: the measured roofline denominators next to the nominal
 * SM-count x lanes x clock figure.  kind 0 = FFMA, 1 = FFMA2 (fma.rn.f32x2), 2 = DFMA, 3 = MUFU.RSQ, 4 = MUFU.EX2,
 * 5 = LDS.128 broadcast, 6 = DADD, 7 = MUFU.RSQ64H, 8 = FADD2, 9 = FMUL2;
 * 11..15 = ceiling of the fp32 pair core's own instruction mix per step (two pairs per lane): 24 FFMA2 in two dependent
 * chains (14), plus 2 MUFU.RSQ (11), plus 2 FSETP+FSEL (12), or plus 2 broadcast LDS.128 (13), or plus both (15).
 * kind + 100 b (b = 1..7) runs the probe with only b resident blocks of 8 warps per SM.
 * *out = lane-operations per second summed over the chip (one FMA = 1; an f32x2 instruction counts 2 per lane;
 * multiply FMA rates by 2 for flops).  Errors: EINVAL, ENODEVICE, ENOMEM, ECUDA. */
int photons_peak_probe(int device, int kind, double* out);

/* Host-only (needs no device): the polynomial behind PHOTONS_G_POLY.  With s = (r/2r_s)^2, s_max = (rcut_over_rs/2)^2
 * and t = 2 s/s_max - 1, the kernels use g(r) ~= 1 - s^(3/2) * sum_k coeffs[k] t^k (derived from the
 * integral form of T).  coeffs: degree + 1 doubles (output, lowest power first); max_err_g (may be
 * NULL): largest |approximation - g| over 0 <= r <= r_cut in exact arithmetic.  Errors: EINVAL (degree outside
 * 1..20, rcut_over_rs outside (0, 6], null coeffs). */
int photons_poly_fit(int degree, double rcut_over_rs, double* coeffs, double* max_err_g);

/* Host-only: the polynomial behind PHOTONS_G_FUSED.  With x = r/2r_s, x_cut = rcut_over_rs/2 and t = 2 x/x_cut - 1 the
 * kernels use g(r) ~= exp(-x^2) * sum_k coeffs[k] t^k.  Arguments, output and errors as photons_poly_fit. */
int photons_fused_fit(int degree, double rcut_over_rs, double* coeffs, double* max_err_g);

/* Truncated multipole-to-local operator, fp64 (§2; A24-A26): for every target cell B and
 * every source cell A in its list,
 *     L_n(z_B) += sum_{|m| <= p - |n|} M_m(z_A) D_{n+m}(z_B - z_A - s L),    D_n = grad^n [ erfc(r / 2 r_s) / r ],
 * the derivative tensors assembled from the paper's prefactors f_(k)(x) (L51) with all trace terms (A24).
 * Multi-indices n = (n_x, n_y, n_z), |n| <= p, are ordered by |n|, then n_x descending, then n_y descending; there are
 * NC = (p+1)(p+2)(p+3)/6 of them.  Multipoles carry the Taylor factors, M_m = sum_j m_j (-a_j)^m / m! (A25).
 *   p            expansion order, 0..4 (the paper does not state its order; A26)
 *   centres      n_cells x 3;  multipoles, locals: n_cells x NC, row-major doubles (locals is overwritten)
 *   pair_ptr     n_cells + 1 offsets into pair_src (CSR by target cell);  pair_src: source cell of each pair
 *   pair_shift   3 signed bytes per pair, s in {-1, 0, +1} box lengths added to the source centre, or NULL
 *   mem_kind     all arrays host or all device (PHOTONS_MEM_*); host arrays are copied in and out
 *   cuda_stream  a cudaStream_t (NULL = default stream); the call returns after the work has completed
 *   kernel_ms    (may be NULL) CUDA-event time of the kernel
 * A source at zero separation from its target is not allowed (the list holds well-separated cells).
 * Errors: EINVAL, ENODEVICE, ENOMEM, ECUDA. */
int photons_m2l(int device, int p, double r_s, double boxsize, long long n_cells, const double* centres,
                const double* multipoles, const long long* pair_ptr, const int* pair_src, const signed char* pair_shift,
                double* locals, int mem_kind, void* cuda_stream, double* kernel_ms);

/* photons_m2l for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same operator, arguments and coefficient order as photons_m2l (A24-A26), with
 * DEVICE pointers only (all of them on `device`; pair_shift may be NULL, pair_src may not), and a kernel variant that
 * splits every target cell's source list over several warps and adds their partial L_n in a fixed order - the same sums
 * as photons_m2l up to fp64 rounding order, reproducible from call to call.
 * The partial sums live in a file-scope device array of PHOTONS_M2L_NOALLOC_SCRATCH_BYTES that every GPU which loads the
 * library holds until the process exits.  The call enqueues two kernels on cuda_stream (a cudaStream_t, NULL = default
 * stream) and returns WITHOUT synchronising; it calls no cudaMalloc / cudaFree / allocating library routine, creates no
 * event or stream, and copies nothing.  (The first call on a device looks the array's device address up with
 * cudaGetSymbolAddress: make one call outside any graph capture.)
 * Limit: n_cells * NC(p) * 8 bytes <= PHOTONS_M2L_NOALLOC_SCRATCH_BYTES (29 959 cells at p = 4, 1 048 576 at p = 0);
 * beyond it the call returns PHOTONS_EINVAL, launches nothing and says so in err_buf - use photons_m2l there.
 * All calls on a device share the array: calls that can overlap on the GPU (different streams, different host threads)
 * race on it - serialise them on one stream.  Nothing in it has to be cleared between calls.
 * err_buf (may be NULL): err_len bytes for the message of a failing call.
 * Errors: EINVAL (arguments, the limit), ENODEVICE, ECUDA. */
#define PHOTONS_M2L_NOALLOC_SCRATCH_BYTES (8u << 20)
int photons_m2l_noalloc(int device, int p, double r_s, double boxsize, long long n_cells, const double* centres,
                        const double* multipoles, const long long* pair_ptr, const int* pair_src,
                        const signed char* pair_shift, double* locals, void* cuda_stream, char* err_buf, int err_len);

/* Message of the last failing call on ctx; valid until the next call on ctx. */
const char* photons_last_error(const photons_ctx* ctx);

/* Free everything.  NULL-safe. */
void photons_destroy(photons_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* PHOTONS_H */
