/*
 * ORACLE — test infrastructure, NOT the product.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or constant with the CUDA library.
 *
 * What it computes (plain definition; §2, Eq. 1, and BASELINE.json north_star):
 *
 *   a_i = G * sum_{j != i, 0 < |d_ij| < r_cut}  m_j * d_ij * T(|d_ij|; r_s) / |d_ij|^3
 *
 *   d_ij = minimum image of (r_j - r_i) in the periodic cube of side L     (north_star; A10);
 *          with L <= 0 the boundaries are isolated: d_ij = r_j - r_i
 *   T(r; r_s) = erfc(r / 2 r_s) + r / (r_s sqrt(pi)) * exp(-r^2 / 4 r_s^2)    (Eq. 1)
 *   sign: dx = pos_j - pos_i and a += grav*dx, i.e. attraction towards j     (Alg. 2;
 *         L55 "F_s = -r/r^3 T" with r = r_i - r_j; A3)
 *   pairs with r == 0 (self, coincident) contribute nothing                  (A7)
 *   pairs with r >= r_cut contribute nothing                                 (north_star; A8)
 *   softening ("100 h^-1 kpc softening length"; form not given; A23): with eps > 0
 *          the short-range potential psi(r) = erfc(r/2r_s)/r is taken at r_eps = sqrt(r^2 + eps^2)
 *          (Plummer substitution), whose gradient gives
 *              a_i = G * sum_{j: 0 < |d_ij|, r_eps < r_cut}  m_j * d_ij * T(r_eps; r_s) / r_eps^3 ;
 *          eps = 0 is the unsoftened sum above, bit for bit.
 *
 * The leaf structure, MAXLEAF and the interaction-list criterion do not enter: a pair outside
 * r_cut contributes exactly zero, so the sum over listed leaves equals this all-pairs sum
 * (the paper's own "fiducial" run replaces the tree by direct P2P).
 *
 * No blocking, no cell grid, no reordering: for i, for j, libm erfc/exp/sqrt in double,
 * accumulation of each component in long double (x87 80-bit) so that the oracle is an order of
 * magnitude better than the 1e-12*rms fp64 tolerance it judges.
 *
 * Parity status: pinned (tests/test_oracle_pins.py): closed forms, quadrature of the integral
 * form L125, the long-range complement, two-body closed forms, Newton's third law, lattice
 * symmetry, neighbour count, brute force in mpmath on tiny inputs.
 */
#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Eq. 1 written in x = r / 2 r_s ("x = r/2r_s", L59). */
double oracle_T(double x)
{
    const double two_over_sqrt_pi = 1.1283791670955125738961589031215;
    return erfc(x) + two_over_sqrt_pi * x * exp(-x * x);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Accelerations of the targets tgt[0..nt) (indices into pos) from all n particles.
 * pos: n x 3 row-major doubles, mass: n doubles, acc: nt x 3 doubles (output).
 * counts (may be NULL): counts[0] += pair tests done, counts[1] += pairs inside r_cut.
 * tgt == NULL means targets 0..nt-1 (nt == n gives the full O(N^2) sum).
 * eps: Plummer softening length (A23), 0 = none.
 */
void oracle_p2p(long long n, const double *pos, const double *mass,
                long long nt, const long long *tgt,
                double L, double r_s, double r_cut, double G, double eps,
                double *acc, long long *counts)
{
    const double rcut2 = r_cut * r_cut;
    const double eps2 = eps * eps;                     /* A23; 0 = no softening */
    const double inv2rs = 1.0 / (2.0 * r_s);
    long long n_tests = 0, n_in = 0;

#pragma omp parallel for schedule(dynamic, 16) reduction(+ : n_tests, n_in)
    for (long long t = 0; t < nt; ++t) {
        const long long i = tgt ? tgt[t] : t;
        const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        long double ax = 0.0L, ay = 0.0L, az = 0.0L;
        long long in = 0;
        for (long long j = 0; j < n; ++j) {
            double dx = pos[3 * j] - xi;
            double dy = pos[3 * j + 1] - yi;
            double dz = pos[3 * j + 2] - zi;
            if (L > 0.0) {                             /* L <= 0: isolated boundaries, no images */
                dx -= L * nearbyint(dx / L);           /* minimum image, per axis */
                dy -= L * nearbyint(dy / L);
                dz -= L * nearbyint(dz / L);
            }
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r2e = r2 + eps2;              /* r_eps^2; == r2 when eps == 0 */
            if (r2 > 0.0 && r2e < rcut2) {
                const double r = sqrt(r2e);
                const double grav = G * mass[j] * oracle_T(r * inv2rs) / (r2e * r);
                ax += (long double)(grav * dx);
                ay += (long double)(grav * dy);
                az += (long double)(grav * dz);
                ++in;
            }
        }
        acc[3 * t] = (double)ax;
        acc[3 * t + 1] = (double)ay;
        acc[3 * t + 2] = (double)az;
        n_tests += n;
        n_in += in;
    }
    if (counts) {
        counts[0] += n_tests;
        counts[1] += n_in;
    }
}
