// ms_math.cuh -- device-side arithmetic building blocks of the MadSpace hot path (sm_100a, fp64).
//
// Everything here is branch-free per lane (selects, no divergent paths), because a warp of 32 independent
// events takes both sides of every data-dependent branch: the two-branch formulas of DESIGN.md readings
// M-2 / M-3 are evaluated as ONE instruction stream with per-lane selected coefficients.
// Polynomial coefficients come from gen_poly_coeffs.py (Chebyshev fits in 60-digit arithmetic).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ms_params.h"

namespace ms {

// ---------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) and the word-pair -> uniform conversion, readings R-1..R-3.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u = (2*(W>>12)+1) * 2^-53 with W = hi<<32 | lo: the 52 bits are OR-ed into the mantissa of 1.0;
// subtracting 1.0 and adding 2^-53 are both exact, so no int->fp conversion is needed (reading R-3).
__device__ __forceinline__ double uniform_from_words(uint32_t hi, uint32_t lo)
{
    const double one_to_two = __hiloint2double((int)(0x3FF00000u | (hi >> 12)), (int)__funnelshift_r(lo, hi, 12));
    return (one_to_two - 1.0) + 0x1p-53;
}

// Uniforms 2*pair and 2*pair+1 of `event`.
__device__ __forceinline__ void philox_uniform_pair(const PhiloxKey& key, uint64_t event, uint32_t pair, double& a,
                                                    double& b)
{
    uint32_t w[4];
    philox4x32_10((uint32_t)event, (uint32_t)(event >> 32), pair, key.stream, key.k0, key.k1, w);
    a = uniform_from_words(w[0], w[1]);
    b = uniform_from_words(w[2], w[3]);
}

// ---------------------------------------------------------------------------------------------------
// Horner helper, coefficients highest degree first.
// ---------------------------------------------------------------------------------------------------
template <int NC>
__device__ __forceinline__ double horner(const double (&c)[NC], double x)
{
    double r = c[0];
#pragma unroll
    for (int i = 1; i < NC; ++i) r = fma(r, x, c[i]);
    return r;
}

// ---------------------------------------------------------------------------------------------------
// ln(y) for y in (0,1], given also z = 1 - y.  When `z_exact` (the caller obtained z without
// cancellation and y = 1 - z), the reduced argument is taken from z for y >= sqrt(1/2), which is what
// log1p(-z) would do -- but in the same instruction stream as the plain logarithm.
//   y = m 2^e, m in [sqrt(1/2), sqrt(2)), f = m - 1, s = f/(2+f), ln m = f - s (f - s^2 PL(s^2)).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double log_unit(double y, double z, bool z_exact)
{
    const int hi = __double2hiint(y), lo = __double2loint(y);
    int e = (hi >> 20) - 1023;
    int mhi = (hi & 0x000FFFFF) | 0x3FF00000;
    if (mhi >= 0x3FF6A09F) { mhi -= 0x00100000; e += 1; }
    const double m = __hiloint2double(mhi, lo);
    double f = m - 1.0;
    if (z_exact && e == 0) f = -z;
    const double s = f / (2.0 + f);
    const double z2 = s * s;
    const double PL[8] = {0x1.0c97816496c47p-3, 0x1.0fb04d4fa4e54p-3, 0x1.3b1cbf421a439p-3, 0x1.745cf674f6889p-3,
                          0x1.c71c72078b928p-3, 0x1.249249247343fp-2, 0x1.9999999999a4fp-2, 0x1.5555555555555p-1};
    const double R = horner(PL, z2);
    const double lnm = fma(-s, fma(-z2, R, f), f);
    return fma((double)e, 0x1.62e42fefa39efp-1, lnm);
}

// ---------------------------------------------------------------------------------------------------
// exp(h) and expm1(h) for h <= 0 from one range reduction: h = n ln2 + r, |r| <= ln2/2,
// expm1(r) = r + r^2 PE(r);  exp(h) = 2^n (1 + p),  expm1(h) = 2^n p + (2^n - 1)  (no cancellation for n <= 0).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void exp_expm1_neg(double h, double& ex, double& em1)
{
    const int n = __double2int_rn(h * 0x1.71547652b82fep+0);
    const double nd = (double)n;
    double r = fma(-nd, 0x1.62e42fee00000p-1, h);
    r = fma(-nd, 0x1.a39ef35793c76p-33, r);
    const double PE[12] = {0x1.61c2c1ba3877dp-33, 0x1.1f820dbf5e732p-29, 0x1.ae642ad2afd38p-26, 0x1.27e4d2841fc93p-22,
                           0x1.71de3a5af94e9p-19, 0x1.a01a01aa828e2p-16, 0x1.a01a01a0195e6p-13, 0x1.6c16c16c158f5p-10,
                           0x1.1111111111111p-7,  0x1.5555555555557p-5,  0x1.5555555555555p-3,  0x1.0000000000000p-1};
    const double p = fma(r * r, horner(PE, r), r);
    const double sc = __hiloint2double((n + 1023) << 20, 0);
    ex = fma(sc, p, sc);
    em1 = fma(sc, p, sc - 1.0);
}

// exp(h) for any moderate h (|h| < 700).
__device__ __forceinline__ double exp_any(double h)
{
    double ex, em1;
    exp_expm1_neg(h, ex, em1);   // the reduction is sign-agnostic; only em1's conditioning needs h <= 0
    return ex;
}

// ---------------------------------------------------------------------------------------------------
// G_RQF^{-1}(x; c): Eq. 65 for x <= 1/2 and the same quadratic solved for z = 1-y for
// x > 1/2 (reading M-2), merged: with t = min-side variable, g = (c-2) t,
//   low : beta = c - g, alpha = 1 - beta, y = 2t / (beta + sqrt(beta^2 + 4 t alpha))
//   high: beta = g,     alpha = 1 + g,    z = (beta + sqrt(beta^2 + 4 t alpha)) / (2 alpha)
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void rqf_inverse(double x, double c, double& y, double& z, bool& high)
{
    high = x > 0.5;
    const double t = high ? 1.0 - x : x;
    const double g = (c - 2.0) * t;
    const double beta = high ? g : c - g;
    const double alpha = high ? 1.0 + g : 1.0 - beta;
    const double sq = sqrt(fma(beta, beta, 4.0 * t * alpha));
    const double bs = beta + sq;
    const double q = (high ? bs : 2.0 * t) / (high ? 2.0 * alpha : bs);
    y = high ? 1.0 - q : q;
    z = high ? q : 1.0 - q;
}

// Table 1: fitted c_k*, k = 1..7.
__device__ __forceinline__ constexpr double table1_ck(int k)
{
    return k == 1 ? 2.0 : k == 2 ? 2.712001 : k == 3 ? 3.084521 : k == 4 ? 3.313073 : k == 5 ? 3.467512
         : k == 6 ? 3.578833 : 3.662872;
}

// One FastRambo mass step (Eq. 60, 65; weight factor = Eq. 67 / Eq. 63):
//   u = y^{1/(2k)}, omu2 = 1 - u^2 = 1 - y^{1/k}, weight factor (k+1) omu2 / g_RQF(y) = wnum / wden.
template <int K>
__device__ __forceinline__ void fastrambo_mass_step(double x, double& u, double& omu2, double& wnum, double& wden)
{
    constexpr double c = table1_ck(K);
    double y, z;
    bool high;
    rqf_inverse(x, c, y, z, high);
    const double L = log_unit(y, z, high);
    double em1;
    exp_expm1_neg(L * (0.5 / K), u, em1);          // u = exp(L/2k), em1 = u - 1
    omu2 = -em1 * (1.0 + u);                       // 1 - u^2 = (1-u)(1+u)
    const double D = fma((c - 2.0) * y, z, 1.0);
    wnum = (double)(K + 1) * omu2 * (D * D);       // g_RQF = z (2y + c z) / D^2   (Eq. 64 with 1-y = z)
    wden = z * fma(c, z, 2.0 * y);
}

// Binomial coefficient at compile time.
__host__ __device__ constexpr double binom_c(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    double b = 1.0;
    for (int i = 1; i <= k; ++i) b = b * (double)(n - k + i) / (double)i;
    return b;
}

// Exact RamboOnDiet mass step: invert Eq. 62 written for v = u^2 = y^{1/k}:
//   r = (k+1) v^k - k v^{k+1}.
// Reading M-3: for r <= 1/2 solve for w = v, G(w) = (k+1) w^k - k w^{k+1} = r; for r > 1/2 solve for w = t = 1-v,
// G(w) = 1 - (1-w)^k (1+kw) = sum_{j=2}^{k+1} a_j w^j = 1-r.  Both are degree-(k+1) polynomials without constant and
// linear term, so ONE Horner/Newton stream with per-lane selected coefficients serves both sides.
// Start: the FastRambo value (RQF approximates Eq. 62).  Returns false if Newton did not settle.
template <int K>
__device__ __forceinline__ bool rambo_mass_step(double r, double& u, double& omu2)
{
    if constexpr (K == 1) {
        const double t = sqrt(1.0 - r);            // (1-v)^2 = 1-r
        const double v = r / (1.0 + t);
        u = sqrt(v);
        omu2 = t;
        return true;
    } else {
        constexpr double c = table1_ck(K);
        double y, z;
        bool high;
        rqf_inverse(r, c, y, z, high);
        const double L = log_unit(y, z, high);
        double v0, em1;
        exp_expm1_neg(L * (1.0 / K), v0, em1);
        const double tgt = high ? 1.0 - r : r;
        double w = high ? -em1 : v0;
        if (high && tgt < 1e-3) w = sqrt(tgt * (2.0 / (K * (K + 1.0))));
        // per-lane coefficients c_j, j = 2..K+1
        double cj[K + 2];
#pragma unroll
        for (int j = 2; j <= K + 1; ++j) {
            const double sgn = (j % 2 == 0) ? 1.0 : -1.0;
            const double a_hi = -sgn * (binom_c(K, j) - (double)K * binom_c(K, j - 1));
            const double a_lo = (j == K) ? (double)(K + 1) : (j == K + 1) ? -(double)K : 0.0;
            cj[j] = high ? a_hi : a_lo;
        }
        bool done = false;
        bool ok = false;
        for (int it = 0; it < 20; ++it) {
            double G = cj[K + 1], H = (K + 1) * cj[K + 1];
#pragma unroll
            for (int j = K; j >= 2; --j) {
                G = fma(G, w, cj[j]);
                H = fma(H, w, (double)j * cj[j]);
            }
            G = G * w * w;
            H = H * w;
            double wn = w - (G - tgt) / H;
            if (!(wn > 0.0)) wn = 0.5 * w;
            if (!(wn < 1.0)) wn = 0.5 * (w + 1.0);
            const double step = fabs(wn - w);
            if (!done) {
                w = wn;
                if (step <= 0x1p-49 * wn) { done = true; ok = true; }
            }
            if (!__any_sync(0xffffffffu, !done)) break;
        }
        if (!done) ok = false;
        const double v = high ? 1.0 - w : w;
        omu2 = high ? w : 1.0 - w;
        u = sqrt(v);
        return ok;
    }
}

// ---------------------------------------------------------------------------------------------------
// Four-vectors.
// ---------------------------------------------------------------------------------------------------
struct Vec4 {
    double e, x, y, z;
};

// One two-body decay {Q_{i-1}, M} -> p_{i-1} + Q_i (Eq. 54-55; angles Eq. 25):
// massless p of momentum q in the rest frame of Q, boosted by the pure boost taking (M,0) to Q (reading D-3);
// the recoil is Q - p.  `first`: Q = (M,0,0,0), no boost needed.
template <bool FIRST>
__device__ __forceinline__ void two_body_decay(Vec4& Q, double M, double q, double x_cos, double x_phi, Vec4& p)
{
    const double cth = fma(2.0, x_cos, -1.0);
    const double sth = 2.0 * sqrt(x_cos * (1.0 - x_cos));   // sqrt(1 - cth^2) without cancellation
    double sn, cs;
    sincospi(2.0 * x_phi, &sn, &cs);
    const double qs = q * sth;
    const double rx = qs * cs, ry = qs * sn, rz = q * cth;
    if constexpr (FIRST) {
        p.e = q; p.x = rx; p.y = ry; p.z = rz;
        Q.e = M - q; Q.x = -rx; Q.y = -ry; Q.z = -rz;
    } else {
        const double qm = Q.e + M;
        const double inv = 1.0 / (M * qm);
        const double ep = fma(Q.x, rx, fma(Q.y, ry, fma(Q.z, rz, Q.e * q))) * (inv * qm);
        const double f = (q + ep) * (inv * M);
        p.e = ep;
        p.x = fma(Q.x, f, rx);
        p.y = fma(Q.y, f, ry);
        p.z = fma(Q.z, f, rz);
        Q.e -= p.e; Q.x -= p.x; Q.y -= p.y; Q.z -= p.z;
    }
}

// Massless n-body volume at unit energy, Eq. 81: 1/(Gamma(n) Gamma(n-1) pi^(2n-3) 2^(4n-5)).
inline double phi_n_unit(int n)
{
    double g1 = 1.0, g2 = 1.0;                    // Gamma(n) = (n-1)!, Gamma(n-1) = (n-2)!
    for (int i = 2; i <= n - 1; ++i) g1 *= (double)i;
    for (int i = 2; i <= n - 2; ++i) g2 *= (double)i;
    const double pi = 3.14159265358979323846;
    double pw = 1.0;
    for (int i = 0; i < 2 * n - 3; ++i) pw *= pi;
    return 1.0 / (g1 * g2 * pw * ldexp(1.0, 4 * n - 5));
}

}  // namespace ms
