/*
 * oracle/ms_oracle_lit.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Second, *literal* evaluator: the paper's printed equations typed as they stand
 * (Eq. 25, 54-55, 60, 62, 64, 65, 67, 81; Eq. 19, 22 for the x sampling) in
 * __float128 (113-bit, libquadmath), for small event counts.  Its only purpose is
 * to tie the well-conditioned fp64 forms used in ms_oracle.c (DESIGN.md readings
 * M-2, M-3, D-2) back to the text: tests require the fp64 oracle to agree with this
 * evaluator to ~1e-14.  Eq. 62 is inverted by plain bisection on [0,1] -- slow and
 * obviously correct.  Shares nothing with the CUDA path.
 */
#include <quadmath.h>
#include <stdint.h>

typedef __float128 q_t;

static const double LIT_CK[8] = { 0.0, 2.0, 2.712001, 3.084521, 3.313073, 3.467512, 3.578833, 3.662872 };

static q_t lit_pi(void) { return M_PIq; }

static q_t lit_phi_n(int n, q_t E)
{   /* Eq. 81 */
    return powq(E, 2 * n - 4) / (tgammaq((q_t)n) * tgammaq((q_t)(n - 1)) * powq(lit_pi(), 2 * n - 3) * powq(2, 4 * n - 5));
}

static q_t lit_rqf_inverse(q_t r, q_t c)
{   /* Eq. 65 */
    q_t b = c - (c - 2) * r;
    return 2 * r / (b + sqrtq(b * b + 4 * r * (1 - b)));
}
static q_t lit_rqf_density(q_t y, q_t c)
{   /* Eq. 64 */
    q_t D = 1 + (c - 2) * y * (1 - y);
    return (2 * y * (1 - y) + c * (1 - y) * (1 - y)) / (D * D);
}
static q_t lit_diet(q_t y, int k)
{   /* Eq. 62 */
    return (k + 1) * y - k * powq(y, 1 + (q_t)1 / k);
}
static q_t lit_diet_inverse(q_t r, int k)
{
    q_t lo = 0, hi = 1;
    for (int it = 0; it < 130; ++it) {
        q_t mid = (lo + hi) / 2;
        if (lit_diet(mid, k) < r) lo = mid; else hi = mid;
    }
    return (lo + hi) / 2;
}

static void lit_boost(const q_t Q[4], q_t M, const q_t p[4], q_t out[4])
{   /* pure boost taking (M,0) to Q (reading D-3) */
    q_t ep = (Q[0] * p[0] + Q[1] * p[1] + Q[2] * p[2] + Q[3] * p[3]) / M;
    q_t f = (p[0] + ep) / (Q[0] + M);
    out[0] = ep;
    for (int a = 1; a < 4; ++a) out[a] = p[a] + Q[a] * f;
}

/* exact = 0: FastRambo; exact = 1: RamboOnDiet.  Same argument layout as orc_fastrambo. */
void lit_rambo(int exact, int64_t N, int n, double sqrt_s, const double *sqrt_s_arr, const double *x,
               double *p, double *w, int64_t ld)
{
    for (int64_t e = 0; e < N; ++e) {
        q_t E = (sqrt_s > 0.0) ? (q_t)sqrt_s : (q_t)sqrt_s_arr[e];
        q_t M[12], wn = 1;
        M[1] = E;
        M[n] = 0;
        for (int i = 2; i <= n - 1; ++i) {
            int k = n - i;
            q_t r = (q_t)x[(int64_t)(i - 2) * ld + e];
            q_t y;
            if (exact) {
                y = lit_diet_inverse(r, k);
            } else {
                q_t c = (q_t)LIT_CK[k];
                y = lit_rqf_inverse(r, c);
                wn *= (k + 1) * (1 - powq(y, (q_t)1 / k)) / lit_rqf_density(y, c);   /* Eq. 67 / Eq. 63 */
            }
            q_t u = powq(y, (q_t)1 / (2 * k));                                       /* Eq. 60 */
            M[i] = u * M[i - 1];
        }
        q_t Q[4] = { E, 0, 0, 0 };
        for (int i = 2; i <= n; ++i) {
            q_t Mp = M[i - 1], Mi = M[i];
            q_t q = (Mp * Mp - Mi * Mi) / (2 * Mp);                                  /* Eq. 24, m_1 = 0 */
            q_t cth = 2 * (q_t)x[(int64_t)(n - 2 + 2 * (i - 2)) * ld + e] - 1;       /* Eq. 25 */
            q_t phi = 2 * lit_pi() * (q_t)x[(int64_t)(n - 1 + 2 * (i - 2)) * ld + e];
            q_t sth = sqrtq(1 - cth * cth);
            q_t pr[4] = { q, q * sth * cosq(phi), q * sth * sinq(phi), q * cth };
            q_t Qr[4] = { sqrtq(q * q + Mi * Mi), -pr[1], -pr[2], -pr[3] };
            q_t pb[4], Qb[4];
            lit_boost(Q, Mp, pr, pb);
            lit_boost(Q, Mp, Qr, Qb);
            for (int mu = 0; mu < 4; ++mu) {
                p[(int64_t)(4 * i + mu) * ld + e] = (double)pb[mu];                  /* p_{i-1} is particle block i */
                Q[mu] = Qb[mu];
            }
        }
        for (int mu = 0; mu < 4; ++mu) p[(int64_t)(4 * (n + 1) + mu) * ld + e] = (double)Q[mu];
        p[0 * ld + e] = (double)(E / 2); p[1 * ld + e] = 0; p[2 * ld + e] = 0; p[3 * ld + e] = (double)(E / 2);
        p[4 * ld + e] = (double)(E / 2); p[5 * ld + e] = 0; p[6 * ld + e] = 0; p[7 * ld + e] = (double)(-E / 2);
        w[e] = (double)(lit_phi_n(n, E) * wn);
    }
}

/* Eq. 19 (m^2 = 0, x_max = 1, x_min = tau_min; r -> 1-r so that r_0 = 1 is tau_min... see
 * DESIGN.md reading X-1: tau = exp[(1-r_0) ln tau_min]) and Eq. 22, literal. */
void lit_pdf_x_sample(int64_t N, double s_had, double tau_min, const double *r, double *x1x2,
                      double *sqrt_shat, double *jac, int64_t ld)
{
    for (int64_t e = 0; e < N; ++e) {
        q_t r0 = (q_t)r[e], r1 = (q_t)r[ld + e];
        q_t tau = expq(r0 * logq((q_t)1) + (1 - r0) * logq((q_t)tau_min));
        x1x2[e] = (double)powq(tau, r1);
        x1x2[ld + e] = (double)powq(tau, 1 - r1);
        sqrt_shat[e] = (double)sqrtq(tau * (q_t)s_had);
        /* dx1 dx2 = dtau dy, dtau = tau ln(1/tau_min) dr0 (1/g of Eq. 19), dy = ln(1/tau) dr1 (Eq. 23) */
        jac[e] = (double)(tau * (-logq((q_t)tau_min)) * (-logq(tau)));
    }
}

/* Classic RAMBO massive rescale (ref. [64]) with xi found by bisection in quad. */
void lit_massive_rescale(int64_t N, int n, double sqrt_s, const double *masses, double *p, double *w, int64_t ld)
{
    for (int64_t e = 0; e < N; ++e) {
        q_t E[12], lo = 0, hi = 1, W = (q_t)sqrt_s;
        for (int i = 0; i < n; ++i) E[i] = (q_t)p[(int64_t)(4 * (i + 2)) * ld + e];
        for (int it = 0; it < 130; ++it) {
            q_t xi = (lo + hi) / 2, F = -W;
            for (int i = 0; i < n; ++i) F += sqrtq((q_t)masses[i] * masses[i] + xi * xi * E[i] * E[i]);
            if (F < 0) lo = xi; else hi = xi;
        }
        q_t xi = (lo + hi) / 2, prod = 1, sum = 0;
        for (int i = 0; i < n; ++i) {
            q_t kabs = xi * E[i], k0 = sqrtq((q_t)masses[i] * masses[i] + kabs * kabs);
            p[(int64_t)(4 * (i + 2)) * ld + e] = (double)k0;
            for (int mu = 1; mu < 4; ++mu)
                p[(int64_t)(4 * (i + 2) + mu) * ld + e] = (double)(xi * (q_t)p[(int64_t)(4 * (i + 2) + mu) * ld + e]);
            prod *= kabs / k0;
            sum += kabs * kabs / k0;
        }
        w[e] = (double)((q_t)w[e] * powq(xi, 2 * n - 3) * W * prod / sum);
    }
}
