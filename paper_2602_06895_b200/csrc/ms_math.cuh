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

// The same with the round keys given (ms_params.h, PhiloxRoundKeys: launch parameters in the constant bank).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxRoundKeys& rk,
                                              uint32_t (&out)[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ rk.k[2 * round];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ rk.k[2 * round + 1];
        c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u = (2*(W>>12)+1) * 2^-53 with W = hi<<32 | lo: the 52 bits are OR-ed into the mantissa of 1.0 giving
// 1 + m 2^-52; subtracting (1 - 2^-53) leaves (2m+1) 2^-53, which is representable, so the one DADD is exact and
// no int->fp conversion is needed (reading R-3).
__device__ __forceinline__ double uniform_from_words(uint32_t hi, uint32_t lo)
{
    const double one_to_two = __hiloint2double((int)(0x3FF00000u | (hi >> 12)), (int)__funnelshift_r(lo, hi, 12));
    return one_to_two - (1.0 - 0x1p-53);
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

__device__ __forceinline__ void philox_uniform_pair(const PhiloxRoundKeys& rk, uint32_t stream, uint64_t event, uint32_t pair,
                                                    double& a, double& b)
{
    uint32_t w[4];
    philox4x32_10((uint32_t)event, (uint32_t)(event >> 32), pair, stream, rk, w);
    a = uniform_from_words(w[0], w[1]);
    b = uniform_from_words(w[2], w[3]);
}

// Clamp of a non-negative double into [2^-53, 1 - 2^-53] on its bit pattern (non-negative doubles order like
// their high words): same result as fmin(fmax(x, 2^-53), 1 - 2^-53) for 0 <= x <= 1 at half the instructions.
__device__ __forceinline__ double clamp_open_unit(double x)
{
    const int hi = __double2hiint(x), lo = __double2loint(x);
    const int chi = min(max(hi, 0x3CA00000), 0x3FEFFFFF);
    const int clo = hi >= 0x3FF00000 ? -1 : (hi < 0x3CA00000 ? 0 : lo);
    return __hiloint2double(chi, clo);
}

__device__ __forceinline__ double2 lds_double2(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// ---------------------------------------------------------------------------------------------------
// Polynomial coefficients (gen_poly_coeffs.py; highest degree first) live in the constant bank: a DFMA takes them
// as an operand (directly or through a uniform register), so no instruction is spent materialising 64-bit
// immediates (profiles/r01a: 381 of 1848 instructions per event were such moves).
// ---------------------------------------------------------------------------------------------------
static __constant__ double c_PL[8] = {0x1.0c97816496c47p-3, 0x1.0fb04d4fa4e54p-3, 0x1.3b1cbf421a439p-3, 0x1.745cf674f6889p-3,
                                      0x1.c71c72078b928p-3, 0x1.249249247343fp-2, 0x1.9999999999a4fp-2, 0x1.5555555555555p-1};
static __constant__ double c_PE[10] = {0x1.af3ce42b12b24p-26, 0x1.2894f52583578p-22, 0x1.71de0be2b5e96p-19, 0x1.a019b621f9d08p-16,
                                       0x1.a01a01a83ba17p-13, 0x1.6c16c1794e1dcp-10, 0x1.1111111110918p-7,  0x1.5555555553b6cp-5,
                                       0x1.5555555555556p-3,  0x1.0000000000001p-1};
// sin(pi r) = r PS(r^2), cos(pi r) = 1 + r^2 PC(r^2) on |r| <= 1/4 (max rel. error 4.1e-17 / 2.8e-17: seven coefficients
// each are as accurate as eight -- beyond that the rounding of the coefficients themselves is the limit)
static __constant__ double c_PS[7] = {0x1.e3da06a519070p-12, -0x1.e3002ae3c4436p-8, 0x1.50782f90efce4p-4, -0x1.32d2cce2a0bd8p-1,
                                      0x1.466bc67758457p+1,  -0x1.4abbce625be3fp+2, 0x1.921fb54442d18p+1};
static __constant__ double c_PC[7] = {-0x1.b2dfe0c850620p-14, 0x1.f9cdecb2c924fp-10, -0x1.a6d1eebaf8f4cp-6, 0x1.e1f50686529f0p-3,
                                      -0x1.55d3c7e3cb0d4p+0,  0x1.03c1f081b5ac0p+2,  -0x1.3bd3cc9be45dep+2};

// atan(t) / (2 pi) = t PA(t^2) on |t| <= sqrt(2) - 1 (max rel. error 1.1e-16)
static __constant__ double c_PA[11] = {0x1.b5885ec281cd5p-9, -0x1.c422ffbd37433p-8, 0x1.286af929b3851p-7, -0x1.5a412e165d6b3p-7,
                                       0x1.910a4ffc569efp-7, -0x1.da19c30b5077fp-7, 0x1.21bb8b5affe87p-6, -0x1.7483755d2c2f7p-6,
                                       0x1.04c26be36ad85p-5, -0x1.b2995e7b7b135p-5, 0x1.45f306dc9c882p-3};

// Horner, coefficients highest degree first.
template <int NC>
__device__ __forceinline__ double horner(const double* c, double x)
{
    double r = c[0];
#pragma unroll
    for (int i = 1; i < NC; ++i) r = fma(r, x, c[i]);
    return r;
}

// ---------------------------------------------------------------------------------------------------
// Guard-free reciprocal, square root and integer root for arguments known to be positive, normal and far from
// the ends of the exponent range (everything on this path is): one MUFU seed (relative error e <= 2^-22.9) and ONE
// third-order correction on the fp64 pipe, no slow-path branch.  An fp64 instruction occupies the issue port of its
// scheduler for two cycles on sm_100a ("issue model"), so these are counted in instructions:
//   1/a     = r (1 + e + e^2 + O(e^3)),            e = 1 - a r          : 3 instructions, truncation 2^-69
//   sqrt(a) = a r (1 + e/2 + 3 e^2/8 + O(e^3)),    e = 1 - a r^2        : 5 instructions, truncation 2^-70
// (two Newton steps plus a residual correction, as in libdevice, cost 4 and 10).  Results are good to about 1 ulp.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double a)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
    const double e = fma(-a, r, 1.0);
    return fma(r, fma(e, e, e), r);
}

// sqrt(a); `half_rsqrt` receives 1/(2 sqrt(a)) from the same correction (two more instructions when it is used).
__device__ __forceinline__ double sqrt_fast(double a, double& half_rsqrt)
{
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
    const double t = a * r;
    const double e = fma(-t, r, 1.0);
    const double q = fma(e, 0.375, 0.5) * e;
    const double hr = 0.5 * r;
    half_rsqrt = fma(hr, q, hr);
    return fma(t, q, t);
}
__device__ __forceinline__ double sqrt_fast(double a)
{
    double h;
    return sqrt_fast(a, h);
}

// y^(1/R), y in (0,1], R >= 3: fp32 seed exp2(log2(y)/R) from MUFU.LG2/EX2 (relative error e ~ 2^-21), then one
// Halley step u (R-1) u^R + (R+1) y over (R+1) u^R + (R-1) y, whose error is (R^2-1)/12 e^3 < 1e-17 for R <= 14.
template <int R>
__device__ __forceinline__ double root_fast(double y)
{
    const float yf = __double2float_rn(y);
    float l, uf;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(yf));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(uf) : "f"(l * (1.0f / R)));
    const double u = (double)uf;
    double p = u;
    if constexpr (R % 2 == 0) {
        double q = u * u;                        // u^R = (u^2)^(R/2) by squaring
        p = 1.0;
#pragma unroll
        for (int b = R / 2; b > 0; b >>= 1) {
            if (b & 1) p *= q;
            if (b > 1) q *= q;
        }
    } else {
        double q = u;
        p = 1.0;
#pragma unroll
        for (int b = R; b > 0; b >>= 1) {
            if (b & 1) p *= q;
            if (b > 1) q *= q;
        }
    }
    const double num = fma((double)(R - 1), p, (double)(R + 1) * y);
    const double den = fma((double)(R + 1), p, (double)(R - 1) * y);
    return u * num * rcp_fast(den);
}

// sin(2 pi x), cos(2 pi x) for x in (0,1): quarter-turn reduction q = rint(4x), r = 2x - q/2 in [-1/4, 1/4] (exact),
// the two cores above, then the rotation by q quarter turns as one swap and two sign flips.
__device__ __forceinline__ void sincos_2pi(double x, double& sn, double& cs)
{
    const double magic = 0x1.8p52;
    const double qm = fma(4.0, x, magic);                       // low word = q
    const int q = __double2loint(qm);
    const double r = fma(-0.5, qm - magic, 2.0 * x);
    const double r2 = r * r;
    const double s = r * horner<7>(c_PS, r2);
    const double c = fma(r2, horner<7>(c_PC, r2), 1.0);
    const bool odd = q & 1;
    const double a = odd ? c : s;                               // sin(pi r + q pi/2)
    const double b = odd ? s : c;
    const int sa = (int)(((unsigned)q & 2u) << 30), sb = (int)(((unsigned)(q + 1) & 2u) << 30);
    sn = __hiloint2double(__double2hiint(a) ^ sa, __double2loint(a));
    cs = __hiloint2double(__double2hiint(b) ^ sb, __double2loint(b));
}

// atan2(y, x) / (2 pi) folded into [0, 1) (the azimuth uniform of Eq. 25 inverted, reading F-4): first octant
// a = min/max in [0,1]; for a > tan(pi/8) the argument is reduced by atan a = pi/4 + atan((a-1)/(a+1)), which with
// a = mn/mx is (mn-mx)/(mn+mx), so ONE reciprocal serves both cases; then the octant is unfolded by three reflections.
__device__ __forceinline__ double atan2_turns(double y, double x)
{
    const double ax = fabs(x), ay = fabs(y);
    const bool swap = ay > ax;
    const double mx = swap ? ay : ax, mn = swap ? ax : ay;
    const bool big = mn > 0x1.a827999fcef32p-2 * mx;            // tan(pi/8)
    const double num = big ? mn - mx : mn;
    const double den = big ? mn + mx : mx;
    const double t = num * rcp_fast(fmax(den, 0x1p-1000));      // x = y = 0 (no azimuth): turn 0, not NaN
    double turn = fma(t, horner<11>(c_PA, t * t), big ? 0.125 : 0.0);
    if (swap) turn = 0.25 - turn;
    if (x < 0.0) turn = 0.5 - turn;
    if (y < 0.0) turn = 1.0 - turn;
    return turn;
}

// ---------------------------------------------------------------------------------------------------
// ln(y) for positive normal y (callers pass (0,1] or, Chili Eq. 74, [1, 2^511)).  y = m 2^e, m in [sqrt(1/2), sqrt(2)),
// f = m - 1, s = f/(2+f),
// ln m = f - s (f - s^2 PL(s^2)).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double log_unit(double y)
{
    const int hi = __double2hiint(y), lo = __double2loint(y);
    int e = (hi >> 20) - 1023;
    int mhi = (hi & 0x000FFFFF) | 0x3FF00000;
    if (mhi >= 0x3FF6A09F) { mhi -= 0x00100000; e += 1; }
    const double m = __hiloint2double(mhi, lo);
    const double f = m - 1.0;
    const double s = f * rcp_fast(2.0 + f);
    const double z2 = s * s;
    const double R = horner<8>(c_PL, z2);
    const double lnm = fma(-s, fma(-z2, R, f), f);
    return fma((double)e, 0x1.62e42fefa39efp-1, lnm);
}

// ---------------------------------------------------------------------------------------------------
// exp(h) for moderate h (|h| < 700): h = n ln2 + r, |r| <= ln2/2, expm1(r) = r + r^2 PE(r), exp(h) = 2^n (1 + p).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double exp_any(double h)
{
    const double magic = 0x1.8p52;
    const double nm = fma(h, 0x1.71547652b82fep+0, magic);
    const int n = __double2loint(nm);
    const double nd = nm - magic;
    double r = fma(-nd, 0x1.62e42fee00000p-1, h);
    r = fma(-nd, 0x1.a39ef35793c76p-33, r);
    const double p = fma(r * r, horner<10>(c_PE, r), r);
    const double sc = __hiloint2double((n + 1023) << 20, 0);
    return fma(sc, p, sc);
}

// ---------------------------------------------------------------------------------------------------
// G_RQF^{-1}(x; c), both y and z = 1 - y, with no branch and no cancellation.  Eq. 65 is
// y = 2x / (b + sqrt(b^2 - 4x(b-1))), b = c - (c-2)x; the same quadratic written for z (reading M-2) is
// z = (beta + sqrt(beta^2 + 4s(1+beta))) / (2(1+beta)), s = 1-x, beta = (c-2)s.  Since b = 2 + beta the two
// discriminants are the same number, so one square root and one reciprocal give both roots, every term positive.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void rqf_inverse(double x, double c_minus_2, double& y, double& z)
{
    const double s = 1.0 - x;
    const double beta = c_minus_2 * s;
    const double a = 1.0 + beta;
    const double sq = sqrt_fast(fma(beta, beta, 4.0 * s * a));
    const double d1 = (a + 1.0) + sq;
    const double a2 = a + a;
    const double inv = rcp_fast(d1 * a2);
    y = (2.0 * x) * a2 * inv;
    z = (beta + sq) * d1 * inv;
}

// Table 1: fitted c_k*, k = 1..7.
__device__ __forceinline__ constexpr double table1_ck(int k)
{
    return k == 1 ? 2.0 : k == 2 ? 2.712001 : k == 3 ? 3.084521 : k == 4 ? 3.313073 : k == 5 ? 3.467512
         : k == 6 ? 3.578833 : 3.662872;
}
// The same numbers and c_k - 2 in the constant bank (index k): a 64-bit literal costs two moves into uniform registers
// at every use, a constant-bank operand none.
static __constant__ double c_CK[8] = {0.0, table1_ck(1), table1_ck(2), table1_ck(3), table1_ck(4), table1_ck(5), table1_ck(6),
                                      table1_ck(7)};
static __constant__ double c_CKM2[8] = {0.0, table1_ck(1) - 2.0, table1_ck(2) - 2.0, table1_ck(3) - 2.0, table1_ck(4) - 2.0,
                                        table1_ck(5) - 2.0, table1_ck(6) - 2.0, table1_ck(7) - 2.0};

// v = y^(1/K) and u = sqrt(v) = y^(1/(2K)) (Eq. 60), and 1 - v = z / (1 + v + ... + v^(K-1)) from
// z = 1 - y (exact factorisation: no cancellation, no logarithm).  Returns S = 1 + v + ... + v^(K-1).
template <int K>
__device__ __forceinline__ double mass_ratio(double y, double z, double& u, double& omu2)
{
    if constexpr (K == 1) {
        u = sqrt_fast(y);
        omu2 = z;
        return 1.0;
    } else {
        double v;
        if constexpr (K == 2) {
            v = sqrt_fast(y);
            u = sqrt_fast(v);
        } else {
            u = root_fast<2 * K>(y);
            v = u * u;
        }
        double S = 1.0 + v;
#pragma unroll
        for (int j = 2; j < K; ++j) S = fma(S, v, 1.0);
        omu2 = z * rcp_fast(S);
        return S;
    }
}

// One FastRambo mass step (Eq. 60, 65; weight factor = Eq. 67 / Eq. 63):
//   weight factor (k+1)(1 - y^(1/k)) / g_RQF(y) with g_RQF = z (2y + c z) / D^2, D = 1 + (c-2) y z (Eq. 64, 1-y = z)
//   = (k+1) D^2 / ((2y + c z) S) = (k+1) wnum / wden   (the z of 1 - y^(1/k) = z/S cancels).
template <int K>
__device__ __forceinline__ void fastrambo_mass_step(double x, double& u, double& omu2, double& wnum, double& wden)
{
    if constexpr (K == 1) {
        // c_1 = 2 (Table 1): Eq. 64 becomes r = 1 - (1-y)^2, the map coincides with RamboOnDiet's and the
        // weight factor is exactly 1: z = sqrt(1-x), y = x / (1 + z), u = sqrt(y), nothing else
        const double z = sqrt_fast(1.0 - x);
        u = sqrt_fast(x * rcp_fast(1.0 + z));
        omu2 = z;
        wnum = 1.0;
        wden = 1.0;
        return;
    }
    const double c = c_CK[K], cm2 = c_CKM2[K];
    double y, z;
    rqf_inverse(x, cm2, y, z);
    const double S = mass_ratio<K>(y, z, u, omu2);
    const double D = fma(cm2 * y, z, 1.0);
    wnum = D * D;                                  // the factors (k+1) are multiplied in once: fastrambo_chain_factor
    wden = fma(c, z, 2.0 * y) * S;
}

// prod_{k=2}^{n-2} (k+1) = (n-1)!/2: the constant part of the FastRambo weight factors of the steps k >= 2 (the k = 1
// step's factor, (k+1)(1-y)/g_RQF with c_1 = 2, is exactly 1 as a whole)
__host__ __device__ constexpr double fastrambo_chain_factor(int n)
{
    double f = 1.0;
    for (int k = 2; k <= n - 2; ++k) f *= (double)(k + 1);
    return f;
}

// Binomial coefficient at compile time.
__host__ __device__ constexpr double binom_c(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    double b = 1.0;
    for (int i = 1; i <= k; ++i) b = b * (double)(n - k + i) / (double)i;
    return b;
}

// fp32 MUFU helpers (approximate, ~2^-22): the exact-Rambo start value is computed entirely on the otherwise idle
// fp32 / XU pipes.
__device__ __forceinline__ float rcp_f32(float a)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
    return r;
}
__device__ __forceinline__ float sqrt_f32(float a)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
    return r;
}
__device__ __forceinline__ float root_f32(float y, float inv_k)
{
    float l, r;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(y));
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(l * inv_k));
    return r;
}

// Exact RamboOnDiet mass step: invert Eq. 62 written for v = u^2 = y^{1/k}:
//   r = (k+1) v^k - k v^{k+1}.
// Reading M-3: for r <= 1/2 solve for w = v, G(w) = (k+1) w^k - k w^{k+1} = r; for r > 1/2 solve for w = t = 1-v,
// G(w) = 1 - (1-w)^k (1+kw) = sum_{j=2}^{k+1} a_j w^j = 1-r.  Both are degree-(k+1) polynomials without constant and
// linear term (so w keeps full RELATIVE accuracy at either end), and ONE instruction stream with per-lane selected
// coefficients serves both sides.  The paper names no method.  Here, branch-free and vote-free:
//   1. start value in fp32: the FastRambo value (RQF approximates Eq. 62 to a few per cent), or the
//      leading term sqrt(2(1-r)/(k(k+1))) when 1-r < 1e-3;
//   2. three (k <= 3) or four Newton steps in fp32 (-> ~1e-7 relative, measured against 40-digit roots);
//   3. ONE Halley step in fp64 (cubic: 1e-7 -> < 3e-16).
// Returns false (event weight 0, fail counter) if the Halley step moved w by more than 1e-4 relative, i.e. if stage 2
// had not converged.
template <int K>
__device__ __forceinline__ bool rambo_mass_step(double r, double& u, double& omu2)
{
    if constexpr (K == 1) {
        const double t = sqrt_fast(1.0 - r);       // (1-v)^2 = 1-r
        const double v = r * rcp_fast(1.0 + t);
        u = sqrt_fast(v);
        omu2 = t;
        return true;
    } else {
        const bool high = r > 0.5;
        const double s = 1.0 - r;
        const double tgt = high ? s : r;
        // per-lane coefficients c_j, j = 2..K+1
        double cj[K + 2];
        float cf[K + 2];
#pragma unroll
        for (int j = 2; j <= K + 1; ++j) {
            const double sgn = (j % 2 == 0) ? 1.0 : -1.0;
            const double a_hi = -sgn * (binom_c(K, j) - (double)K * binom_c(K, j - 1));
            const double a_lo = (j == K) ? (double)(K + 1) : (j == K + 1) ? -(double)K : 0.0;
            cj[j] = high ? a_hi : a_lo;
            cf[j] = high ? (float)a_hi : (float)a_lo;
        }
        // ---- 1. fp32 start: RQF inverse (Eq. 65 and its z form) and the k-th root
        constexpr float c = (float)table1_ck(K);
        const float xf = __double2float_rn(r), sf = __double2float_rn(s), tf = high ? sf : xf;
        const float beta = (c - 2.0f) * sf, a = 1.0f + beta;
        const float sq = sqrt_f32(fmaf(beta, beta, 4.0f * sf * a));
        float w;
        if (high) {
            const float z = (beta + sq) * rcp_f32(a + a);
            const float y = 1.0f - z;
            const float v = root_f32(fmaxf(y, 1e-30f), 1.0f / K);
            float S = 1.0f + v;
#pragma unroll
            for (int j = 2; j < K; ++j) S = fmaf(S, v, 1.0f);
            w = z * rcp_f32(S);
            if (tf < 1e-3f) w = sqrt_f32(tf * (2.0f / (K * (K + 1.0f))));
        } else {
            const float y = (2.0f * xf) * rcp_f32((a + 1.0f) + sq);
            w = root_f32(y, 1.0f / K);
        }
        // ---- 2. fp32 Newton steps: three reach ~1.5e-7 for k <= 3, four for k <= 7 (40-digit reference roots)
#pragma unroll
        for (int it = 0; it < (K <= 3 ? 3 : 4); ++it) {
            float G = cf[K + 1], H = (K + 1) * cf[K + 1];
#pragma unroll
            for (int j = K; j >= 2; --j) {
                G = fmaf(G, w, cf[j]);
                H = fmaf(H, w, (float)j * cf[j]);
            }
            float wn = fmaf(-(G * w * w - tf), rcp_f32(H * w), w);
            if (!(wn > 0.0f)) wn = 0.5f * w;
            if (!(wn < 1.0f)) wn = 0.5f * (w + 1.0f);
            w = wn;
        }
        // ---- 3. one fp64 Halley step on f(w) = G(w) - tgt
        const double w0 = (double)w;
        double G = cj[K + 1], H = (K + 1) * cj[K + 1], S2 = (double)((K + 1) * K) * cj[K + 1];
#pragma unroll
        for (int j = K; j >= 2; --j) {
            G = fma(G, w0, cj[j]);
            H = fma(H, w0, (double)j * cj[j]);
            S2 = fma(S2, w0, (double)(j * (j - 1)) * cj[j]);
        }
        const double f = fma(G * w0, w0, -tgt);        // G(w0) - tgt
        H *= w0;                                        // G'(w0);  S2 = G''(w0)
        const double dw = (2.0 * f * H) * rcp_fast(fma(2.0 * H, H, -f * S2));
        const double wd = w0 - dw;
        const bool ok = fabs(dw) <= 1e-4 * w0;
        omu2 = high ? wd : 1.0 - wd;
        u = sqrt_fast(high ? 1.0 - wd : wd);
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
// p has energy e_rest and momentum q = q2 / 2 in the rest frame of Q (e_rest = q for a massless particle), and is boosted by the
// pure boost taking (M,0) to Q (reading D-3); the recoil is Q - p.  `first`: Q = (M,0,0,0), no boost needed.
template <bool FIRST>
__device__ __forceinline__ void two_body_decay(Vec4& Q, double M, double e_rest, double q2, double x_cos, double x_phi,
                                               Vec4& p)
{
    // q2 = 2q: cos(theta) = 2x - 1 and sin(theta) = 2 sqrt(x (1 - x)) (no cancellation) hand their factor 2 to q
    double sn, cs;
    sincos_2pi(x_phi, sn, cs);
    const double qs = q2 * sqrt_fast(x_cos * (1.0 - x_cos));
    const double rx = qs * cs, ry = qs * sn, rz = q2 * (x_cos - 0.5);
    if constexpr (FIRST) {
        p.e = e_rest; p.x = rx; p.y = ry; p.z = rz;
        Q.e = M - e_rest; Q.x = -rx; Q.y = -ry; Q.z = -rz;
    } else {
        const double qm = Q.e + M;
        const double inv = rcp_fast(M * qm);
        const double ep = fma(Q.x, rx, fma(Q.y, ry, fma(Q.z, rz, Q.e * e_rest))) * (inv * qm);
        const double f = (e_rest + ep) * (inv * M);
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
