// Host-side generation of what the pair core needs to evaluate the truncation function g (Eq. 1):
//   make_table : the paper's interpolation table {T_i, E_i} (§3.3), built in extended precision
//                and rounded once;
//   make_poly  : coefficients of Q(s) = (1 - g(sqrt s)) / s^(3/2), s = (r / 2 r_s)^2, as a polynomial in the
//                mapped variable t = 2 s / s_max - 1 (Chebyshev interpolation, converted to monomials),
//                so that g(r)/r^3 = 1/r^3 - Q(s)/(2 r_s)^3 needs no special function.
// Nothing here is shared with oracle/.
#include <cmath>
#include <vector>

#include "common.cuh"

namespace photons {

static const long double PI_L = 3.14159265358979323846264338327950288L;

int make_table(Ctx* c)
{
    const int n = c->p.table_nodes;
    std::vector<float2> te(n + 1);
    std::vector<double2> te64(n + 1);
    for (int i = 0; i <= n; ++i) {
        const long double x = 3.0L * i / n;                                  // nodes over x in [0, 3] (L143)
        const long double E = -4.0L * expl(-x * x) / sqrtl(PI_L);            // E_i = -4 exp(-x_i^2)/sqrt(pi)
        const long double T = erfcl(x) - x * E / 2.0L;                       // T_i = erfc(x_i) - x_i E_i / 2
        te[i] = make_float2((float)T, (float)E);
        te64[i] = make_double2((double)T, (double)E);
    }
    c->table.n = n;
    c->table.level = c->p.table_level;
    PH_CUDA(c, cudaMalloc(&c->table.d_TE, sizeof(float2) * (n + 1)));
    PH_CUDA(c, cudaMemcpy(c->table.d_TE, te.data(), sizeof(float2) * (n + 1), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMalloc(&c->table.d_TE64, sizeof(double2) * (n + 1)));
    PH_CUDA(c, cudaMemcpy(c->table.d_TE64, te64.data(), sizeof(double2) * (n + 1), cudaMemcpyHostToDevice));
    return PHOTONS_OK;
}

// Q(s) = (1 - g(x)) / x^3 with x = sqrt(s).  From the integral form T(x) = 4/sqrt(pi) int_x^inf u^2 e^{-u^2} du
// (PAPER.md L125): 1 - T(x) = 4/sqrt(pi) int_0^x u^2 e^{-u^2} du = 4/sqrt(pi) sum_k (-1)^k x^(2k+3) / ((2k+3) k!),
// hence Q(s) = 4/sqrt(pi) sum_k (-s)^k / ((2k+3) k!), an entire function of s.
static long double Q_of_s(long double s)
{
    if (s <= 1.0L) {
        long double term = 1.0L, sum = 0.0L;   // term = (-s)^k / k!
        for (int k = 0; k < 40; ++k) {
            sum += term / (2 * k + 3);
            term *= -s / (k + 1);
        }
        return 4.0L / sqrtl(PI_L) * sum;
    }
    const long double x = sqrtl(s);
    const long double g = erfcl(x) + 2.0L * x / sqrtl(PI_L) * expl(-s);
    return (1.0L - g) / (x * s);
}

int make_poly(Ctx* c)
{
    const int deg = c->p.poly_degree;
    const int N = deg + 1;
    const long double xcut = 0.5L * c->p.rcut_over_rs;
    const long double smax = xcut * xcut;
    // Chebyshev interpolation on N nodes
    std::vector<long double> f(N), cheb(N);
    for (int j = 0; j < N; ++j) {
        const long double t = cosl(PI_L * (j + 0.5L) / N);
        f[j] = Q_of_s(0.5L * smax * (t + 1.0L));
    }
    for (int k = 0; k < N; ++k) {
        long double a = 0;
        for (int j = 0; j < N; ++j) a += f[j] * cosl(PI_L * k * (j + 0.5L) / N);
        cheb[k] = (k == 0 ? 1.0L : 2.0L) * a / N;
    }
    // to monomials in t: T_0 = 1, T_1 = t, T_{k+1} = 2 t T_k - T_{k-1}
    std::vector<long double> mono(N, 0.0L), Tkm1(N, 0.0L), Tk(N, 0.0L), Tkp1(N, 0.0L);
    Tkm1[0] = 1.0L;
    mono[0] += cheb[0];
    if (N > 1) {
        Tk[1] = 1.0L;
        mono[1] += cheb[1];
    }
    for (int k = 1; k + 1 < N; ++k) {
        for (int i = 0; i < N; ++i) Tkp1[i] = -Tkm1[i];
        for (int i = 0; i + 1 < N; ++i) Tkp1[i + 1] += 2.0L * Tk[i];
        for (int i = 0; i < N; ++i) mono[i] += cheb[k + 1] * Tkp1[i];
        Tkm1 = Tk;
        Tk = Tkp1;
    }
    // scale by (1/2r_s)^3 and round once; Horner order (highest degree first)
    const long double k3 = 1.0L / (8.0L * (long double)c->r_s * c->r_s * c->r_s);
    c->poly_deg = deg;
    for (int i = 0; i <= deg; ++i) c->poly_c[i] = (float)(mono[deg - i] * k3);
    // truncation error of the polynomial, expressed as an error of g:  |x^3 (P - Q)|
    long double worst = 0;
    for (int i = 0; i <= 4000; ++i) {
        const long double s = smax * i / 4000.0L;
        const long double t = 2.0L * s / smax - 1.0L;
        long double p = 0;
        for (int k = deg; k >= 0; --k) p = p * t + mono[k];
        const long double e = fabsl(sqrtl(s) * s * (p - Q_of_s(s)));
        if (e > worst) worst = e;
    }
    c->poly_err = (double)worst;
    return PHOTONS_OK;
}

}  // namespace photons
