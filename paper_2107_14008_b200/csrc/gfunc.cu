// Host-side generation of what the pair core needs to evaluate the truncation function g (Eq. 1):
//   make_table : the paper's interpolation table {T_i, E_i} (§3.3), built in extended precision
//                and rounded once;
//   make_poly  : coefficients of Q(s) = (1 - g(sqrt s)) / s^(3/2), s = (r / 2 r_s)^2, as a polynomial in the
//                mapped variable t = 2 s / s_max - 1 (weighted minimax fit, converted to monomials),
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
    std::vector<double> c64((size_t)(n + 1) * 5), q64((size_t)(n + 1) * 4);
    const long double h = 3.0L / n;
    for (int i = 0; i <= n; ++i) {
        const long double x = 3.0L * i / n;                                  // nodes over x in [0, 3] (L143)
        const long double E = -4.0L * expl(-x * x) / sqrtl(PI_L);            // E_i = -4 exp(-x_i^2)/sqrt(pi)
        const long double T = erfcl(x) - x * E / 2.0L;                       // T_i = erfc(x_i) - x_i E_i / 2
        te[i] = make_float2((float)T, (float)E);
        te64[i] = make_double2((double)T, (double)E);
        // coefficient layout: the terms T[k] of Eq. 2 (L129-L141) with eps = e_u h, e_u in node units
        const long double x2 = x * x;
        const long double ck[5] = {T, x2 * E, -x * (x2 - 1.0L) * E, (2.0L / 3.0L * x2 * x2 - 5.0L / 3.0L * x2 + 1.0L / 3.0L) * E,
                                   -x * (x2 * x2 / 3.0L - 1.5L * x2 + 1.0L) * E};
        long double hk = 1.0L;
        for (int k = 0; k < 5; ++k) { c64[(size_t)i * 5 + k] = (double)(ck[k] * hk); hk *= h; }
        // quad layout: the paper's pair and the brackets of T[3] and T[4] (polynomials in x_i, L137-L141)
        q64[(size_t)i * 4] = (double)T; q64[(size_t)i * 4 + 1] = (double)E;
        q64[(size_t)i * 4 + 2] = (double)(2.0L / 3.0L * x2 * x2 - 5.0L / 3.0L * x2 + 1.0L / 3.0L);
        q64[(size_t)i * 4 + 3] = (double)(-x * (x2 * x2 / 3.0L - 1.5L * x2 + 1.0L));
    }
    c->table.n = n;
    c->table.level = c->p.table_level;
    PH_CUDA(c, cudaMalloc(&c->table.d_TE, sizeof(float2) * (n + 1)));
    PH_CUDA(c, cudaMemcpy(c->table.d_TE, te.data(), sizeof(float2) * (n + 1), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMalloc(&c->table.d_TE64, sizeof(double2) * (n + 1)));
    PH_CUDA(c, cudaMemcpy(c->table.d_TE64, te64.data(), sizeof(double2) * (n + 1), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMalloc(&c->table.d_C64, sizeof(double) * c64.size()));
    PH_CUDA(c, cudaMemcpy(c->table.d_C64, c64.data(), sizeof(double) * c64.size(), cudaMemcpyHostToDevice));
    PH_CUDA(c, cudaMalloc(&c->table.d_Q64, sizeof(double) * q64.size()));
    PH_CUDA(c, cudaMemcpy(c->table.d_Q64, q64.data(), sizeof(double) * q64.size(), cudaMemcpyHostToDevice));
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

// Least squares of the M x N system A x = b by Householder QR, in long double (N <= POLY_MAX_DEG + 1).
static void lstsq(std::vector<long double>& A, std::vector<long double>& b, int M, int N, std::vector<long double>& x)
{
    for (int k = 0; k < N; ++k) {
        long double norm = 0;
        for (int i = k; i < M; ++i) norm += A[(size_t)i * N + k] * A[(size_t)i * N + k];
        norm = sqrtl(norm);
        if (norm == 0) continue;
        const long double alpha = A[(size_t)k * N + k] > 0 ? -norm : norm;
        std::vector<long double> v(M - k);
        for (int i = k; i < M; ++i) v[i - k] = A[(size_t)i * N + k];
        v[0] -= alpha;
        long double vv = 0;
        for (long double e : v) vv += e * e;
        if (vv == 0) continue;
        for (int j = k; j < N; ++j) {
            long double dot = 0;
            for (int i = k; i < M; ++i) dot += v[i - k] * A[(size_t)i * N + j];
            const long double f = 2 * dot / vv;
            for (int i = k; i < M; ++i) A[(size_t)i * N + j] -= f * v[i - k];
        }
        long double dot = 0;
        for (int i = k; i < M; ++i) dot += v[i - k] * b[i];
        const long double f = 2 * dot / vv;
        for (int i = k; i < M; ++i) b[i] -= f * v[i - k];
    }
    x.assign(N, 0.0L);
    for (int k = N - 1; k >= 0; --k) {
        long double acc = b[k];
        for (int j = k + 1; j < N; ++j) acc -= A[(size_t)k * N + j] * x[j];
        x[k] = acc / A[(size_t)k * N + k];
    }
}

// Weighted minimax fit on t in [-1, 1] in the Chebyshev basis: Lawson's iteration (repeated weighted least squares,
// weights multiplied by the residual) on a Chebyshev-distributed sample, in long double; one degree cheaper than plain
// Chebyshev interpolation at equal accuracy.  mono[k] = coefficient of t^k (k = 0..deg).
// `target` supplies f(t), the function to fit, and w(t), the weight of the residual.
template <typename Target>
static void lawson_fit(int deg, const Target& target, std::vector<long double>& mono)
{
    const int N = deg + 1;
    const int M = 48 * N;
    std::vector<long double> tt(M), qq(M), wg(M), lw(M, 1.0L), cheb(N, 0.0L);
    for (int i = 0; i < M; ++i) {
        tt[i] = cosl(PI_L * (i + 0.5L) / M);
        qq[i] = target.f(tt[i]);
        wg[i] = target.w(tt[i]);
    }
    std::vector<long double> V((size_t)M * N);
    for (int i = 0; i < M; ++i) {
        V[(size_t)i * N] = 1.0L;
        if (N > 1) V[(size_t)i * N + 1] = tt[i];
        for (int k = 2; k < N; ++k) V[(size_t)i * N + k] = 2.0L * tt[i] * V[(size_t)i * N + k - 1] - V[(size_t)i * N + k - 2];
    }
    for (int it = 0; it < 120; ++it) {
        std::vector<long double> A((size_t)M * N), b(M);
        for (int i = 0; i < M; ++i) {
            const long double w = wg[i] * sqrtl(lw[i]);
            for (int k = 0; k < N; ++k) A[(size_t)i * N + k] = w * V[(size_t)i * N + k];
            b[i] = w * qq[i];
        }
        lstsq(A, b, M, N, cheb);
        long double sum = 0;
        for (int i = 0; i < M; ++i) {
            long double p = 0;
            for (int k = 0; k < N; ++k) p += cheb[k] * V[(size_t)i * N + k];
            lw[i] *= fabsl(wg[i] * (p - qq[i]));
            sum += lw[i];
        }
        if (!(sum > 0)) break;
        for (int i = 0; i < M; ++i) lw[i] = fmaxl(lw[i] / sum, 1e-40L);
    }
    // to monomials in t: T_0 = 1, T_1 = t, T_{k+1} = 2 t T_k - T_{k-1}
    std::vector<long double> Tkm1(N, 0.0L), Tk(N, 0.0L), Tkp1(N, 0.0L);
    mono.assign(N, 0.0L);
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
}

// POLY: Q on [0, s_max] in t = 2 s/s_max - 1, s_max = (rcut_over_rs / 2)^2.  What matters is the error of g = 1 - x^3 Q,
// so the residual carries the weight s^(3/2).  Returns the largest |g_poly - g| over [0, x_cut] in exact arithmetic.
struct PolyTarget {
    long double smax;
    long double s(long double t) const { return 0.5L * smax * (t + 1.0L); }
    long double f(long double t) const { return Q_of_s(s(t)); }
    long double w(long double t) const { return s(t) * sqrtl(s(t)); }
};

static long double fit_poly(int deg, long double rcut_over_rs, std::vector<long double>& mono)
{
    const long double xcut = 0.5L * rcut_over_rs;
    const long double smax = xcut * xcut;
    lawson_fit(deg, PolyTarget{smax}, mono);
    long double worst = 0;
    for (int i = 0; i <= 4000; ++i) {
        const long double s = smax * i / 4000.0L;
        const long double t = 2.0L * s / smax - 1.0L;
        long double p = 0;
        for (int k = deg; k >= 0; --k) p = p * t + mono[k];
        const long double e = fabsl(sqrtl(s) * s * (p - Q_of_s(s)));
        if (e > worst) worst = e;
    }
    return worst;
}

// FUSED: Eq. 1 factorised as g(x) = exp(-x^2) H(x), H(x) = erfcx(x) + 2 x / sqrt(pi) (erfcx = exp(x^2) erfc):
// H is smooth and of order one on [0, x_cut] (H(0) = 1, H' = 2 x erfcx), so a polynomial in t = 2 x/x_cut - 1 of
// degree ~10 reproduces it; the residual carries the weight exp(-x^2), i.e. the fit is minimax in g.
static long double H_of_x(long double x) { return erfcl(x) * expl(x * x) + 2.0L * x / sqrtl(PI_L); }

struct FusedTarget {
    long double xcut;
    long double x(long double t) const { return 0.5L * xcut * (t + 1.0L); }
    long double f(long double t) const { return H_of_x(x(t)); }
    long double w(long double t) const { return expl(-x(t) * x(t)); }
};

static long double fit_fused(int deg, long double rcut_over_rs, std::vector<long double>& mono)
{
    const long double xcut = 0.5L * rcut_over_rs;
    lawson_fit(deg, FusedTarget{xcut}, mono);
    long double worst = 0;
    for (int i = 0; i <= 4000; ++i) {
        const long double x = xcut * i / 4000.0L;
        const long double t = 2.0L * x / xcut - 1.0L;
        long double p = 0;
        for (int k = deg; k >= 0; --k) p = p * t + mono[k];
        const long double e = fabsl(expl(-x * x) * (p - H_of_x(x)));
        if (e > worst) worst = e;
    }
    return worst;
}

int make_fused(Ctx* c)
{
    const int deg = c->p.poly_degree;
    std::vector<long double> mono;
    c->fused_err = (double)fit_fused(deg, c->p.rcut_over_rs, mono);
    c->fused_deg = deg;
    for (int i = 0; i <= deg; ++i) c->fused_c[i] = (float)mono[deg - i];     // Horner order (highest degree first)
    return PHOTONS_OK;
}

int make_poly(Ctx* c)
{
    const int deg = c->p.poly_degree;
    std::vector<long double> mono;
    c->poly_err = (double)fit_poly(deg, c->p.rcut_over_rs, mono);
    // scale by (1/2r_s)^3, r_s in the kernels' length unit (Ctx::pscale), and round once; Horner order (highest
    // degree first)
    const long double rs = (long double)c->r_s / (long double)c->pscale;
    const long double k3 = 1.0L / (8.0L * rs * rs * rs);
    c->poly_deg = deg;
    for (int i = 0; i <= deg; ++i) c->poly_c[i] = (float)(mono[deg - i] * k3);
    return PHOTONS_OK;
}

}  // namespace photons

// Host-only hooks (no device needed): the fitted polynomials themselves, for checks against an independent g.
extern "C" int photons_fused_fit(int degree, double rcut_over_rs, double* coeffs, double* max_err_g)
{
    if (degree < 1 || degree > photons::POLY_MAX_DEG || !(rcut_over_rs > 0) || rcut_over_rs > 6.0 || !coeffs) return PHOTONS_EINVAL;
    std::vector<long double> mono;
    const long double e = photons::fit_fused(degree, rcut_over_rs, mono);
    for (int k = 0; k <= degree; ++k) coeffs[k] = (double)mono[k];
    if (max_err_g) *max_err_g = (double)e;
    return PHOTONS_OK;
}

extern "C" int photons_poly_fit(int degree, double rcut_over_rs, double* coeffs, double* max_err_g)
{
    if (degree < 1 || degree > photons::POLY_MAX_DEG || !(rcut_over_rs > 0) || rcut_over_rs > 6.0 || !coeffs) return PHOTONS_EINVAL;
    std::vector<long double> mono;
    const long double e = photons::fit_poly(degree, rcut_over_rs, mono);
    for (int k = 0; k <= degree; ++k) coeffs[k] = (double)mono[k];
    if (max_err_g) *max_err_g = (double)e;
    return PHOTONS_OK;
}
