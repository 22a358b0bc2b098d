// codebook.cpp -- the library's own TQ-MSE scalar codebooks (reading Q7).
//
// C_b = Lloyd-Max (MSE-optimal) 2^b-level quantiser of N(0,1): each level is the conditional
// mean of its cell, thresholds are midpoints.  This is the scalar quantiser whose
// high-resolution distortion is the paper's C_TQ * 4^-b, C_TQ = sqrt(3)*pi/2.
// Levels are symmetric, ascending, rounded to fp16 ("shared fp16 codebook").
//
// Solver: damped Newton on the centroid equations of the positive half, long double, with a
// tridiagonal (Thomas) solve.  Shares nothing with oracle/codebook.py; tests compare the two
// tables value by value.
#include <cmath>
#include <cstdint>
#include <vector>

namespace bgtq {

namespace {
const long double kInvSqrt2Pi = 0.39894228040143267793994605993438L;
const long double kSqrt2 = 1.41421356237309504880168872420970L;

long double pdf(long double x) { return std::isinf(x) ? 0.0L : kInvSqrt2Pi * expl(-0.5L * x * x); }
// P(a < X < b), 0 <= a < b, through erfc so the tail keeps relative accuracy
long double mass(long double a, long double b)
{
    long double ea = erfcl(a / kSqrt2);
    long double eb = std::isinf(b) ? 0.0L : erfcl(b / kSqrt2);
    return 0.5L * (ea - eb);
}

// positive levels c[0..n) of the symmetric 2n-level quantiser
std::vector<long double> solve_positive(int n)
{
    std::vector<long double> c(n), t(n + 1), F(n), lo(n), di(n), up(n), step(n), cn(n);
    // start: equal-probability cells of the half-normal, level = cell centroid
    {
        // invert the half-normal CDF by bisection
        std::vector<long double> edge(n + 1);
        edge[0] = 0.0L;
        for (int k = 1; k < n; ++k) {
            long double target = (long double)k / n, a = 0.0L, b = 40.0L;
            for (int it = 0; it < 200; ++it) {
                long double mid = 0.5L * (a + b);
                if (1.0L - erfcl(mid / kSqrt2) < target) a = mid; else b = mid;
            }
            edge[k] = 0.5L * (a + b);
        }
        edge[n] = INFINITY;
        for (int k = 0; k < n; ++k) c[k] = (pdf(edge[k]) - pdf(edge[k + 1])) / mass(edge[k], edge[k + 1]);
    }
    for (int iter = 0; iter < 500; ++iter) {
        t[0] = 0.0L;
        for (int k = 1; k < n; ++k) t[k] = 0.5L * (c[k - 1] + c[k]);
        t[n] = INFINITY;
        long double resid = 0.0L;
        for (int k = 0; k < n; ++k) {
            long double a = t[k], b = t[k + 1];
            long double P = mass(a, b);
            long double g = (pdf(a) - pdf(b)) / P;                 // centroid of the cell
            long double dga = pdf(a) * (g - a) / P;                // d g / d a
            long double dgb = std::isinf(b) ? 0.0L : pdf(b) * (b - g) / P;   // d g / d b
            F[k] = c[k] - g;
            lo[k] = 0.0L; up[k] = 0.0L; di[k] = 1.0L;
            if (k > 0) { lo[k] -= 0.5L * dga; di[k] -= 0.5L * dga; }
            if (k + 1 < n) { di[k] -= 0.5L * dgb; up[k] -= 0.5L * dgb; }
            resid = fmaxl(resid, fabsl(F[k]));
        }
        if (resid < 1e-17L) break;
        // Thomas algorithm: J * step = F
        std::vector<long double> cp(n), dp(n);
        cp[0] = up[0] / di[0];
        dp[0] = F[0] / di[0];
        for (int k = 1; k < n; ++k) {
            long double den = di[k] - lo[k] * cp[k - 1];
            cp[k] = up[k] / den;
            dp[k] = (F[k] - lo[k] * dp[k - 1]) / den;
        }
        step[n - 1] = dp[n - 1];
        for (int k = n - 2; k >= 0; --k) step[k] = dp[k] - cp[k] * step[k + 1];
        long double lam = 1.0L;
        for (;;) {
            bool ok = true;
            for (int k = 0; k < n; ++k) cn[k] = c[k] - lam * step[k];
            if (!(cn[0] > 0.0L)) ok = false;
            for (int k = 1; k < n && ok; ++k) if (!(cn[k] > cn[k - 1])) ok = false;
            if (ok || lam < 1e-8L) break;
            lam *= 0.5L;
        }
        c = cn;
    }
    return c;
}

// fp64 -> fp16 round-to-nearest-even (finite, |x| < 65504), returned as the fp16 value in double
double round_to_f16(double x)
{
    if (x == 0.0) return 0.0;
    int e;
    double f = frexp(fabs(x), &e);            // |x| = f * 2^e, f in [0.5, 1)
    int E = e - 1;                            // exponent of the leading bit
    int q = (E < -14) ? -24 : E - 10;         // quantum 2^q (subnormal quantum is 2^-24)
    double scaled = ldexp(fabs(x), -q);       // exact
    double r = nearbyint(scaled);             // default mode: ties-to-even
    (void)f;
    double v = ldexp(r, q);
    return x < 0 ? -v : v;
}
}  // namespace

// levels[0 .. 2^b): ascending, fp16-representable
void codebook_levels(int b, double *levels)
{
    if (b == 0) { levels[0] = 0.0; return; }
    int n = 1 << (b - 1);
    std::vector<long double> pos = solve_positive(n);
    for (int k = 0; k < n; ++k) {
        double v = round_to_f16((double)pos[k]);
        levels[n + k] = v;
        levels[n - 1 - k] = -v;
    }
}


// ---------------------------------------------------------------- e4m3 byte planes (BGTQ-v2 decode path)
// The v2 decode kernel feeds the 5th-generation tensor cores with 8-bit operands: one PRMT byte lookup yields four
// operand bytes.  A codebook level v is therefore represented as (hi + lo) / kappa with hi, lo in the e4m3 grid
// (sign, 4 exponent bits, 3 mantissa bits; finite range +-448), hi = nearest(kappa v), lo = nearest(kappa v - hi).
// kappa is free (it is divided out of q' in fp32): it is searched on [32, 64] for the smallest worst-case relative
// error over the levels of the width -- for b <= 3 there are scales at which every level is (almost) exactly a sum of
// two grid values.
namespace {
double e4m3_value(int byte)
{
    const int s = byte >> 7, e = (byte >> 3) & 15, m = byte & 7;
    const double v = e == 0 ? ldexp((double)m, -9) : ldexp(1.0 + m / 8.0, e - 7);
    return s ? -v : v;
}
// nearest finite e4m3 value (round to nearest, ties to even), returned as its byte
int e4m3_nearest(double x)
{
    const int s = x < 0 ? 0x80 : 0;
    const double a = fabs(x);
    if (a >= 448.0) return s | 0x7E;
    int e;
    (void)frexp(a, &e);                          // a = f * 2^e, f in [0.5, 1): leading bit 2^(e-1)
    int E = a == 0.0 ? -7 : e - 1;
    if (E < -6) E = -6;                          // subnormals share the quantum of the smallest normal binade
    const double q = ldexp(1.0, E - 3);          // quantum: 3 mantissa bits
    const double r = nearbyint(a / q) * q;       // default rounding mode: ties to even
    if (r == 0.0) return s;
    int er;
    const double fr = frexp(r, &er);             // r = fr * 2^er
    int Er = er - 1;
    if (Er < -6) return s | (int)nearbyint(ldexp(r, 9));            // subnormal: m * 2^-9
    return s | ((Er + 7) << 3) | (int)nearbyint((2.0 * fr - 1.0) * 8.0);
}
}  // namespace

static void codebook_planes_search(int b, float *kappa, uint8_t *hi, uint8_t *lo)
{
    const int n = 1 << b;
    double lv[256];
    codebook_levels(b, lv);
    if (b == 1) {                                // {-c, +c}: one plane of +-1, the level itself is the scale
        *kappa = (float)(1.0 / lv[1]);
        hi[0] = 0xB8; hi[1] = 0x38; lo[0] = lo[1] = 0;
        return;
    }
    double best_k = 64.0, best_err = 1e300;
    const int steps = b <= 4 ? 200000 : 20000;
    for (int i = 0; i <= steps; ++i) {
        const float kf = (float)(32.0 + 32.0 * i / steps);          // the kernel divides by the fp32 value
        const double k = (double)kf;
        double worst = 0.0;
        for (int j = n / 2; j < n && worst < best_err; ++j) {       // positive half (the table is symmetric)
            const double v = k * lv[j];
            const double h = e4m3_value(e4m3_nearest(v));
            const double l = e4m3_value(e4m3_nearest(v - h));
            worst = fmax(worst, fabs(v - h - l) / v);
        }
        if (worst < best_err) { best_err = worst; best_k = k; }
    }
    *kappa = (float)best_k;
    for (int j = 0; j < n; ++j) {
        const double v = best_k * lv[j];
        const int hb = e4m3_nearest(v);
        hi[j] = (uint8_t)hb;
        lo[j] = (uint8_t)e4m3_nearest(v - e4m3_value(hb));
    }
}


void codebook_planes(int b, float *kappa, uint8_t *hi, uint8_t *lo)
{
    // searched once per process (the result depends on nothing but b)
    struct Cache { float kappa[9]; uint8_t hi[9][256], lo[9][256]; };
    static const Cache *cache = [] {
        Cache *c = new Cache();
        for (int w = 1; w <= 8; ++w) codebook_planes_search(w, &c->kappa[w], c->hi[w], c->lo[w]);
        return c;
    }();
    *kappa = cache->kappa[b];
    for (int j = 0; j < (1 << b); ++j) { hi[j] = cache->hi[b][j]; lo[j] = cache->lo[b][j]; }
}


// ---------------------------------------------------------------- exact-density codebooks (reading Q7b)
// A coordinate of sqrt(m) * u, u uniform on the unit sphere of R^m (any unit vector after a Haar rotation),
// has the density f_m(x) ~ (1 - x^2/m)^((m-3)/2) on |x| < sqrt(m).  With x = sqrt(m) sin(phi):
//     mass(a, b)  ~  I_n(phi_b) - I_n(phi_a),  I_n(phi) = int_0^phi cos^n,  n = m - 2  (m even: I_0 = phi, then the
//                    recurrence I_n = cos^(n-1) sin / n + (n-1)/n I_(n-2), all terms positive on [0, pi/2])
//     int x f     ~  sqrt(m) (cos^(n+1)(phi_a) - cos^(n+1)(phi_b)) / (n+1)
// C_{b,m} = the Lloyd-Max quantiser of f_m (Newton on the centroid equations, as above), rounded to fp16.  Independent of
// oracle/codebook.py (which uses the incomplete beta function); tests compare the two tables value by value.
namespace {
long double cos_power_integral(int n, long double phi)
{
    const long double c = cosl(phi), s = sinl(phi);
    long double I = phi, cp = c;                  // I_0; cp = cos^(k-1) for the next even k = 2
    for (int k = 2; k <= n; k += 2) {
        I = cp * s / k + (long double)(k - 1) / k * I;
        cp *= c * c;
    }
    return I;
}

std::vector<long double> solve_positive_sphere(int n_pos, int m)
{
    const int n = m - 2;
    const long double rm = sqrtl((long double)m), half_pi = acosl(0.0L);
    std::vector<long double> c = solve_positive(n_pos);
    if (c[n_pos - 1] >= 0.98L * rm) { const long double f = 0.98L * rm / c[n_pos - 1]; for (auto &v : c) v *= f; }
    std::vector<long double> t(n_pos + 1), F(n_pos), lo(n_pos), di(n_pos), up(n_pos), step(n_pos), cn(n_pos), cp(n_pos), dp(n_pos);
    for (int iter = 0; iter < 1000; ++iter) {
        t[0] = 0.0L;
        for (int k = 1; k < n_pos; ++k) t[k] = 0.5L * (c[k - 1] + c[k]);
        long double resid = 0.0L;
        for (int k = 0; k < n_pos; ++k) {
            const long double pa = asinl(t[k] / rm), pb = k + 1 < n_pos ? asinl(t[k + 1] / rm) : half_pi;
            const long double dI = cos_power_integral(n, pb) - cos_power_integral(n, pa);
            const long double g = rm * (powl(cosl(pa), n + 1) - powl(cosl(pb), n + 1)) / ((n + 1) * dI);
            // f(x) / mass = cos^(m-3)(phi) / (sqrt(m) dI)
            const long double fa = powl(cosl(pa), m - 3) / (rm * dI);
            const long double fb = k + 1 < n_pos ? powl(cosl(pb), m - 3) / (rm * dI) : 0.0L;
            const long double dga = fa * (g - t[k]), dgb = k + 1 < n_pos ? fb * (t[k + 1] - g) : 0.0L;
            F[k] = c[k] - g;
            lo[k] = 0.0L; up[k] = 0.0L; di[k] = 1.0L;
            if (k > 0) { lo[k] -= 0.5L * dga; di[k] -= 0.5L * dga; }
            if (k + 1 < n_pos) { di[k] -= 0.5L * dgb; up[k] -= 0.5L * dgb; }
            resid = fmaxl(resid, fabsl(F[k]));
        }
        if (resid < 1e-16L) break;
        cp[0] = up[0] / di[0];
        dp[0] = F[0] / di[0];
        for (int k = 1; k < n_pos; ++k) {
            const long double den = di[k] - lo[k] * cp[k - 1];
            cp[k] = up[k] / den;
            dp[k] = (F[k] - lo[k] * dp[k - 1]) / den;
        }
        step[n_pos - 1] = dp[n_pos - 1];
        for (int k = n_pos - 2; k >= 0; --k) step[k] = dp[k] - cp[k] * step[k + 1];
        long double lam = 1.0L;
        for (;;) {
            bool ok = true;
            for (int k = 0; k < n_pos; ++k) cn[k] = c[k] - lam * step[k];
            if (!(cn[0] > 0.0L) || !(cn[n_pos - 1] < rm)) ok = false;
            for (int k = 1; k < n_pos && ok; ++k) if (!(cn[k] > cn[k - 1])) ok = false;
            if (ok || lam < 1e-10L) break;
            lam *= 0.5L;
        }
        c = cn;
    }
    return c;
}
}  // namespace

// levels[0 .. 2^b) of C_{b,m}: ascending, fp16-representable; m even, 2 <= m
void codebook_levels_sphere(int b, int m, double *levels)
{
    if (b == 0) { levels[0] = 0.0; return; }
    const int n = 1 << (b - 1);
    std::vector<long double> pos = solve_positive_sphere(n, m);
    for (int k = 0; k < n; ++k) {
        const double v = round_to_f16((double)pos[k]);
        levels[n + k] = v;
        levels[n - 1 - k] = -v;
    }
}

}  // namespace bgtq
