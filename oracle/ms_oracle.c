/*
 * oracle/ms_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, scalar fp64 CPU restatement of the MadSpace phase-space hot path
 * (arXiv 2602.06895), written from /root/reference/PAPER.md only.  One event at a
 * time, no blocking, no fusion, no SIMD intrinsics; OpenMP only splits disjoint
 * event ranges (results do not depend on the thread count because the random
 * numbers are counter based).  It shares NO code with paper_2602_06895_b200/csrc:
 * no header, no table generator, no helper.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 *
 * Every function cites the PAPER.md passage (line : equation) it restates, or the
 * DESIGN.md reading ("reading R-x") where the paper is silent.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors;
 * closed-form massless volume Eq. 81; per-event constant weight for n=2,3 and for
 * exact Rambo; four-momentum conservation; p^2 = m^2; Beta(2,n-2) energy spectrum;
 * unit VEGAS Jacobian / identity on uniform grids; forward o inverse round trips;
 * Table 1 re-fit from Eq. 66; massive two-body closed form and nested-quadrature
 * massive volume; literal __float128 transcription (ms_oracle_lit.c).
 * Parity unpinned: nothing (the toy integrand, not from the paper, is pinned by brute force at every n,
 * by the closed form at n = 2 and by the Dalitz-plot quadrature of its cross-section at n = 3: tests/).
 *
 * Layout convention (an interface, not shared code): structure of arrays,
 * a[row*ld + e] for event e; momentum row = 4*particle + mu, mu = (E,px,py,pz)
 * (Eq. 77 component order); particles 0,1 incoming, 2..n+1 outgoing.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_N 9 /* k = n-2 <= 7: Table 1 */

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------ */
/* R: random inputs.  PAPER.md:585 names "random number generation" as an op */
/* without fixing a generator; BASELINE.json fixes Philox (reading R-1..R-3). */
/* ------------------------------------------------------------------------ */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), as published. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(prod1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)prod1;
        uint32_t n2 = (uint32_t)(prod0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)prod0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Reading R-2 (counter layout) and R-3 (word pair -> uniform in the open interval).
 * key = (seed_lo, seed_hi); ctr = (event_lo, event_hi, j>>1, stream);
 * uniform j uses words (0,1) if j is even, (2,3) if j is odd;
 * W = (w_a << 32) | w_b, m = W >> 12 (52 bits), u = (2m+1) * 2^-53. */
double orc_uniform(uint64_t seed, uint32_t stream, uint64_t event, uint32_t j)
{
    uint32_t ctr[4] = { (uint32_t)event, (uint32_t)(event >> 32), j >> 1, stream };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    orc_philox4x32_10(ctr, key, w);
    uint64_t W = (j & 1u) ? (((uint64_t)w[2] << 32) | w[3]) : (((uint64_t)w[0] << 32) | w[1]);
    uint64_t m = W >> 12;
    return (double)(2u * m + 1u) * 0x1p-53;
}

/* r[j*ld + e] = uniform j of event (event_offset + e). */
void orc_fill_uniforms(int64_t N, int d, uint64_t seed, uint32_t stream, uint64_t event_offset,
                       double *r, int64_t ld)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e)
        for (int j = 0; j < d; ++j)
            r[(int64_t)j * ld + e] = orc_uniform(seed, stream, event_offset + (uint64_t)e, (uint32_t)j);
}

/* ------------------------------------------------------------------------ */
/* V: frozen VEGAS grid map.  PAPER.md:603 ("classic VEGAS"), :746 (grids are */
/* adapted, then frozen); the paper prints no equations -> reading V-1..V-3   */
/* (Lepage's piecewise-linear map).  edges[dim*(n_bins+1) + j].              */
/* ------------------------------------------------------------------------ */
static const double ORC_U_LO = 0x1p-53;            /* reading V-2 guard */
static const double ORC_U_HI = 1.0 - 0x1p-53;

void orc_vegas_forward(int64_t N, int d, int n_bins, const double *edges, const double *r,
                       double *x, double *jac, int64_t ld)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double J = 1.0;
        for (int dim = 0; dim < d; ++dim) {
            const double *xe = edges + (int64_t)dim * (n_bins + 1);
            double t = r[(int64_t)dim * ld + e] * (double)n_bins;
            int j = (int)floor(t);
            if (j > n_bins - 1) j = n_bins - 1;
            if (j < 0) j = 0;
            double delta = t - (double)j;
            double width = xe[j + 1] - xe[j];
            double xv = xe[j] + delta * width;
            if (xv < ORC_U_LO) xv = ORC_U_LO;
            if (xv > ORC_U_HI) xv = ORC_U_HI;
            x[(int64_t)dim * ld + e] = xv;
            J *= (double)n_bins * width;
        }
        if (jac) jac[e] = J;
    }
}

/* Inverse: bin j with x_j <= x < x_{j+1} ("upper bound - 1"), r = (j + (x-x_j)/width)/n_bins,
 * jac_inv = 1 / prod(n_bins * width). */
void orc_vegas_inverse(int64_t N, int d, int n_bins, const double *edges, const double *x,
                       double *r, double *jac_inv, int64_t ld)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double J = 1.0;
        for (int dim = 0; dim < d; ++dim) {
            const double *xe = edges + (int64_t)dim * (n_bins + 1);
            double xv = x[(int64_t)dim * ld + e];
            int j = 0;
            while (j < n_bins - 1 && xe[j + 1] <= xv) ++j; /* linear scan = definition */
            double width = xe[j + 1] - xe[j];
            r[(int64_t)dim * ld + e] = ((double)j + (xv - xe[j]) / width) / (double)n_bins;
            J *= (double)n_bins * width;
        }
        if (jac_inv) jac_inv[e] = 1.0 / J;
    }
}

/* ------------------------------------------------------------------------ */
/* W: massless n-body volume, Eq. 81, including (2pi)^(4-3n)  */
/* (PAPER.md:134, :413).                                                     */
/* ------------------------------------------------------------------------ */
/* V-4: VEGAS adaptation, accumulation pass.  PAPER.md:603 names "the classic  */
/* VEGAS algorithm" and :746 says the grids "are optimized during an initial   */
/* adaptation phase and are then frozen"; no equations are printed, so this is */
/* Lepage's algorithm (refs): every event adds the      */
/* square of its weight w = f J to the bin its uniform r_dim fell into,        */
/* hist[dim][floor(r_dim n_bins)] += w^2.  The uniforms are the event's own    */
/* Philox uniforms (reading R-2), so the pass needs only the weights.          */
/* Sequential, in event order (a reference for sums taken in any order).       */
/* ------------------------------------------------------------------------ */
void orc_vegas_accumulate(int64_t N, int d, int n_bins, const double *w, uint64_t seed, uint32_t stream,
                          uint64_t event_offset, double *hist)
{
    for (int64_t e = 0; e < N; ++e) {
        double w2 = w[e] * w[e];
        for (int dim = 0; dim < d; ++dim) {
            double r = orc_uniform(seed, stream, event_offset + (uint64_t)e, (uint32_t)dim);
            int j = (int)floor(r * (double)n_bins);
            if (j > n_bins - 1) j = n_bins - 1;
            hist[(int64_t)dim * n_bins + j] += w2;
        }
    }
}

/* ------------------------------------------------------------------------ */
double orc_phi_n(int n, double E_cm)
{
    return pow(E_cm, 2 * n - 4) /
           (tgamma((double)n) * tgamma((double)(n - 1)) * pow(M_PI, 2 * n - 3) * pow(2.0, 4 * n - 5));
}

/* ------------------------------------------------------------------------ */
/* M: mass chain.  Table 1 c_k*, k = 1..7.                */
/* ------------------------------------------------------------------------ */
static const double ORC_CK[8] = { 0.0, 2.0, 2.712001, 3.084521, 3.313073, 3.467512, 3.578833, 3.662872 };

double orc_ck(int k) { return (k >= 1 && k <= 7) ? ORC_CK[k] : NAN; }

/* G_RQF and g_RQF, Eq. 64, literal. */
double orc_rqf_forward(double y, double c)
{
    return (y * y + c * y * (1.0 - y)) / (1.0 + (c - 2.0) * y * (1.0 - y));
}
double orc_rqf_density(double y, double c)
{
    double D = 1.0 + (c - 2.0) * y * (1.0 - y);
    return (2.0 * y * (1.0 - y) + c * (1.0 - y) * (1.0 - y)) / (D * D);
}

/* G_RQF^{-1}: Eq. 65 for x <= 1/2; for x > 1/2 the same quadratic
 * solved for z = 1 - y (reading M-2: with s = 1 - x, (1+s(c-2)) z^2 - s(c-2) z - s = 0),
 * so that 1 - y carries no cancellation.  Returns y, writes z = 1 - y. */
static double rqf_inverse_yz(double x, double c, double *z_out)
{
    double y, z;
    if (x <= 0.5) {
        double b = c - (c - 2.0) * x;
        y = 2.0 * x / (b + sqrt(b * b + 4.0 * x * (1.0 - b)));
        z = 1.0 - y;
    } else {
        double s = 1.0 - x;
        double a = s * (c - 2.0);
        double D1 = 1.0 + a;
        z = (a + sqrt(a * a + 4.0 * s * D1)) / (2.0 * D1);
        y = 1.0 - z;
    }
    *z_out = z;
    return y;
}
double orc_rqf_inverse(double x, double c)
{
    double z;
    return rqf_inverse_yz(x, c, &z);
}

/* One FastRambo mass step (PAPER.md:447 M_i = u_i M_{i-1}; Eq. 60 y = u^{2k};
 * Eq. 65; Eq. 67 weight factor (k+1)(1 - y^{1/k})/g_RQF, obtained by dividing
 * Eq. 67 by Eq. 63).  Returns u, writes 1-u^2 and the weight factor. */
static double fastrambo_mass_step(double x, int k, double *one_minus_u2, double *wfac)
{
    double c = ORC_CK[k];
    double z, y = rqf_inverse_yz(x, c, &z);
    double L = (x <= 0.5) ? log(y) : log1p(-z);         /* ln y */
    double u = exp(L / (2.0 * k));                       /* y^{1/(2k)} */
    double omu2 = -expm1(L / (double)k);                 /* 1 - y^{1/k} */
    double D = 1.0 + (c - 2.0) * y * z;
    double g = z * (2.0 * y + c * z) / (D * D);          /* Eq. 64 with 1-y = z */
    *one_minus_u2 = omu2;
    *wfac = (double)(k + 1) * omu2 / g;
    return u;
}

/* Exact RamboOnDiet mass step: invert Eq. 62 for v = u^2 = y^{1/k}:
 * r = (k+1) v^k - k v^{k+1}.  k = 1 closed form; k >= 2 Newton ("numerical methods
 * have to be used"; reading M-3: two branches so that both v and
 * t = 1-v are obtained without cancellation).  Returns u, writes t = 1-u^2. */
static double binom(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    double b = 1.0;
    for (int i = 1; i <= k; ++i) b = b * (double)(n - k + i) / (double)i;
    return b;
}

int orc_rambo_mass_step(double r, int k, double *u_out, double *one_minus_u2)
{
    double v, t;
    int iters = 0;
    if (k == 1) {
        t = sqrt(1.0 - r);                 /* (1-v)^2 = 1-r */
        v = r / (1.0 + t);
    } else {
        /* start: FastRambo value */
        double z0, y0 = rqf_inverse_yz(r, ORC_CK[k], &z0);
        double L0 = (r <= 0.5) ? log(y0) : log1p(-z0);
        if (r <= 0.5) {
            v = exp(L0 / (double)k);
            for (iters = 0; iters < 60; ++iters) {
                double vk1 = pow(v, k - 1);
                double f = vk1 * v * ((double)(k + 1) - (double)k * v) - r;
                double fp = (double)k * (double)(k + 1) * vk1 * (1.0 - v);
                double dv = f / fp;
                double vn = v - dv;
                if (!(vn > 0.0)) vn = 0.5 * v;
                if (!(vn < 1.0)) vn = 0.5 * (v + 1.0);
                double step = fabs(vn - v);
                v = vn;
                if (step <= 4.0 * 0x1p-52 * v) { ++iters; break; }
            }
            t = 1.0 - v;
        } else {
            /* P(t) = 1 - (1-t)^k (1+kt) = sum_{j=2}^{k+1} a_j t^j = 1 - r */
            double a[ORC_MAX_N + 2];
            for (int j = 2; j <= k + 1; ++j) {
                double sgn = (j % 2 == 0) ? 1.0 : -1.0;
                a[j] = -sgn * (binom(k, j) - (double)k * binom(k, j - 1));
            }
            double s = 1.0 - r;
            t = -expm1(L0 / (double)k);
            if (s < 1e-3) t = sqrt(2.0 * s / ((double)k * (double)(k + 1)));
            for (iters = 0; iters < 60; ++iters) {
                double P = 0.0;
                for (int j = k + 1; j >= 2; --j) P = P * t + a[j];
                P = P * t * t;                            /* Horner, lowest power t^2 */
                double Pp = (double)k * (double)(k + 1) * t * pow(1.0 - t, k - 1);
                double dt = (P - s) / Pp;
                double tn = t - dt;
                if (!(tn > 0.0)) tn = 0.5 * t;
                if (!(tn < 1.0)) tn = 0.5 * (t + 1.0);
                double step = fabs(tn - t);
                t = tn;
                if (step <= 4.0 * 0x1p-52 * t) { ++iters; break; }
            }
            v = 1.0 - t;
        }
    }
    *u_out = sqrt(v);
    *one_minus_u2 = t;
    return iters;
}

/* ------------------------------------------------------------------------ */
/* D: decay chain, Eq. 53-55, angles Eq. 25 */
/* ------------------------------------------------------------------------ */

/* Pure boost taking (M,0,0,0) to Q (reading D-3): e' = (Q0 e + Q.p)/M,
 * p' = p + Q (e + e')/(Q0 + M). */
static void boost_to(const double Q[4], double M, const double p[4], double out[4])
{
    double e = p[0];
    double ep = (Q[0] * e + Q[1] * p[1] + Q[2] * p[2] + Q[3] * p[3]) / M;
    double f = (e + ep) / (Q[0] + M);
    out[0] = ep;
    out[1] = p[1] + Q[1] * f;
    out[2] = p[2] + Q[2] * f;
    out[3] = p[3] + Q[3] * f;
}
/* Its inverse: the boost taking Q to rest, applied to p. */
static void boost_from(const double Q[4], double M, const double p[4], double out[4])
{
    double e = p[0];
    double ep = (Q[0] * e - Q[1] * p[1] - Q[2] * p[2] - Q[3] * p[3]) / M;
    double f = (e + ep) / (Q[0] + M);
    out[0] = ep;
    out[1] = p[1] - Q[1] * f;
    out[2] = p[2] - Q[2] * f;
    out[3] = p[3] - Q[3] * f;
}

/* M[1..n] intermediate masses (M[1] = sqrt_s, M[n] = 0), omu2[2..n-1] = 1-u_i^2,
 * xang[2(i-2)] -> cos theta_{i-1}, xang[2(i-2)+1] -> phi_{i-1} (reading D-1).
 * Output pout[j][4], j = 0..n-1 = p_1..p_n of Eq. 53, in the frame where Q_1 rests. */
static void decay_chain(int n, const double *M, const double *omu2, const double *xang,
                        double pout[][4])
{
    double Q[4] = { M[1], 0.0, 0.0, 0.0 };
    for (int i = 2; i <= n; ++i) {
        double Mp = M[i - 1];
        /* Eq. 24 with m_1 = 0, m_2 = M_i: |p| = (M_{i-1}^2 - M_i^2)/(2 M_{i-1}) = M_{i-1}(1-u_i^2)/2 */
        double q = (i < n) ? 0.5 * Mp * omu2[i] : 0.5 * Mp;
        double xc = xang[2 * (i - 2)], xp = xang[2 * (i - 2) + 1];
        double cth = 2.0 * xc - 1.0;                       /* Eq. 25 */
        double sth = 2.0 * sqrt(xc * (1.0 - xc));          /* sqrt(1 - cth^2), no cancellation */
        double phi = 2.0 * M_PI * xp;                      /* Eq. 25 */
        double pr[4] = { q, q * sth * cos(phi), q * sth * sin(phi), q * cth };
        double Qr[4] = { Mp - q, -pr[1], -pr[2], -pr[3] }; /* recoil in the rest frame of Q_{i-1} */
        if (i == 2) {
            memcpy(pout[i - 2], pr, sizeof pr);
            memcpy(Q, Qr, sizeof Qr);
        } else {
            double Qn[4];
            boost_to(Q, Mp, pr, pout[i - 2]);
            boost_to(Q, Mp, Qr, Qn);
            memcpy(Q, Qn, sizeof Qn);
        }
    }
    memcpy(pout[n - 1], Q, sizeof Q);                      /* {Q_n, M_n} = {p_n, m_n} */
}

/* Generic driver for FastRambo (exact = 0) and RamboOnDiet (exact = 1).
 * x rows: [0..n-3] mass steps i = 2..n-1, then (cos theta, phi) pairs (reading D-1).
 * sqrt_s > 0: fixed; else per-event sqrt_s_arr[e].  Writes all (n+2)*4 momentum rows
 * (incoming rows per reading D-4) and w = Phi_n(sqrt_s) * w_n (reading W-1). */
static void rambo_generic(int exact, int64_t N, int n, double sqrt_s, const double *sqrt_s_arr,
                          const double *x, double *p, double *w, int64_t ld)
{
    double phi1 = orc_phi_n(n, 1.0);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double E = (sqrt_s > 0.0) ? sqrt_s : sqrt_s_arr[e];
        double M[ORC_MAX_N + 2], omu2[ORC_MAX_N + 2], xang[2 * ORC_MAX_N];
        double pout[ORC_MAX_N][4];
        double wn = 1.0;
        M[1] = E;
        M[n] = 0.0;
        for (int i = 2; i <= n - 1; ++i) {
            int k = n - i;                                 /* Eq. 62 */
            double xi = x[(int64_t)(i - 2) * ld + e];
            double u, wf = 1.0;
            if (exact) orc_rambo_mass_step(xi, k, &u, &omu2[i]);
            else u = fastrambo_mass_step(xi, k, &omu2[i], &wf);
            wn *= wf;
            M[i] = u * M[i - 1];
        }
        for (int a = 0; a < 2 * (n - 1); ++a) xang[a] = x[(int64_t)(n - 2 + a) * ld + e];
        decay_chain(n, M, omu2, xang, pout);
        /* incoming, partonic frame (reading D-4) */
        double in_a[4] = { 0.5 * E, 0.0, 0.0, 0.5 * E }, in_b[4] = { 0.5 * E, 0.0, 0.0, -0.5 * E };
        for (int mu = 0; mu < 4; ++mu) {
            p[(int64_t)(0 + mu) * ld + e] = in_a[mu];
            p[(int64_t)(4 + mu) * ld + e] = in_b[mu];
        }
        for (int j = 0; j < n; ++j)
            for (int mu = 0; mu < 4; ++mu) p[(int64_t)(4 * (j + 2) + mu) * ld + e] = pout[j][mu];
        w[e] = phi1 * pow(E, 2 * n - 4) * wn;
    }
}

void orc_fastrambo(int64_t N, int n, double sqrt_s, const double *sqrt_s_arr, const double *x,
                   double *p, double *w, int64_t ld)
{
    rambo_generic(0, N, n, sqrt_s, sqrt_s_arr, x, p, w, ld);
}
void orc_rambo_massless(int64_t N, int n, double sqrt_s, const double *sqrt_s_arr, const double *x,
                        double *p, double *w, int64_t ld)
{
    rambo_generic(1, N, n, sqrt_s, sqrt_s_arr, x, p, w, ld);
}

/* ------------------------------------------------------------------------ */
/* K-4: massive extension, strategy (ii) of PAPER.md:510-522 -- the one the  */
/* paper adopts: "mass effects are incorporated through a reweighting of     */
/* massless phase-space points" (Eq. 68-69).  Step by step:                  */
/*   K_1 = M_1 - sum_j m_j; K_i = u_2..u_i K_1 with the u_i of the MASSLESS  */
/*   FastRambo (or exact Rambo) map; M_i = K_i + sum_{j>=i} m_j (Eq. 69, with */
/*   the sum read as j = i..n: as printed, j = 1..n, K_i would go negative    */
/*   and contradict the line's own K_n = 0 -- DESIGN.md reading K-4a);       */
/*   n-1 two-body decays {Q_{i-1}, M_{i-1}} -> {p_{i-1}, m_{i-1}} + {Q_i, M_i}  */
/*   (Eq. 53-55; two-body momentum Eq. 24);                                   */
/*   weight = Phi_n(K_1) w_n  prod_{i=2}^{n} rho(M_{i-1},M_i,m_{i-1}) /       */
/*            rho(K_{i-1},K_i,0)  prod_{i=2}^{n-1} M_i/K_i  (Eq. 68, with the  */
/*   printed prefactor 1/8 dropped: under the paper's own rho, Eq. 55, the   */
/*   i = n term rho(K_{n-1},0,0) = 1/8 already sits in the denominator and    */
/*   the printed form gives 1/8 of the exact volume for n = 2 -- reading K-4b;*/
/*   pinned by the closed-form two-body volume and the nested-quadrature      */
/*   massive 4-body volume in tests/test_oracle_massive_rw.py).               */
/* Returns the number of events with sum m >= sqrt_s (weight 0).              */
/* ------------------------------------------------------------------------ */
/* sqrt(lambda(M^2, m1^2, m2^2)) through the textbook factorisation
 *   lambda = (M - m1 - m2)(M + m1 + m2)(M - m1 + m2)(M + m1 - m2),
 * with the first factor d = M - m1 - m2 supplied by the caller, who knows it without cancellation:
 * here M_{i-1} - m_{i-1} - M_i = K_{i-1} - K_i (Eq. 69).  The expanded form a^2+b^2+c^2-2ab-2ac-2bc loses
 * eps M^4/lambda and would make soft emissions (u_i -> 1) the accuracy limit of the whole oracle. */
static double sqrt_kallen(double M, double m1, double m2, double d)
{
    double lam = d * (M + m1 + m2) * (M - m1 + m2) * (M + m1 - m2);
    return sqrt(lam > 0.0 ? lam : 0.0);
}

int64_t orc_rambo_massive_reweight(int exact, int64_t N, int n, double sqrt_s, const double *masses,
                                   const double *x, double *p, double *w, int64_t ld)
{
    double phi1 = orc_phi_n(n, 1.0);
    double msum[ORC_MAX_N + 2];                            /* msum[i] = sum_{j>=i} m_j, i = 1..n */
    msum[n + 1] = 0.0;
    for (int i = n; i >= 1; --i) msum[i] = msum[i + 1] + masses[i - 1];
    int64_t nbad = 0;
#pragma omp parallel for schedule(static) reduction(+ : nbad)
    for (int64_t e = 0; e < N; ++e) {
        double K[ORC_MAX_N + 2], M[ORC_MAX_N + 2], u[ORC_MAX_N + 2], omu2[ORC_MAX_N + 2];
        double pout[ORC_MAX_N][4];
        double wn = 1.0, wm = 1.0;
        K[1] = sqrt_s - msum[1];
        if (!(K[1] > 0.0)) { w[e] = 0.0; nbad += 1; continue; }
        M[1] = sqrt_s;
        for (int i = 2; i <= n - 1; ++i) {
            int k = n - i;
            double xi = x[(int64_t)(i - 2) * ld + e];
            double wf = 1.0;
            if (exact) orc_rambo_mass_step(xi, k, &u[i], &omu2[i]);
            else u[i] = fastrambo_mass_step(xi, k, &omu2[i], &wf);
            wn *= wf;
            K[i] = u[i] * K[i - 1];
            M[i] = K[i] + msum[i];                         /* Eq. 69 (reading K-4a) */
            wm *= M[i] / K[i];                             /* second product of Eq. 68 */
        }
        K[n] = 0.0;
        M[n] = masses[n - 1];
        /* decay chain, Eq. 53-55 with masses; first product of Eq. 68 alongside */
        double Q[4] = { M[1], 0.0, 0.0, 0.0 };
        for (int i = 2; i <= n; ++i) {
            double Mp = M[i - 1], m1 = masses[i - 2], m2 = M[i];
            /* K_{i-1} - K_i = K_{i-1} (1 - u_i) = K_{i-1} (1 - u_i^2)/(1 + u_i);  K_n = 0 */
            double d = (i < n) ? K[i - 1] * omu2[i] / (1.0 + u[i]) : K[i - 1];
            double sl = sqrt_kallen(Mp, m1, m2, d);
            double q = sl / (2.0 * Mp);                    /* Eq. 24 */
            double rho_M = sl / (8.0 * Mp * Mp);           /* Eq. 55 */
            double rho_K = (i < n) ? omu2[i] / 8.0 : 1.0 / 8.0;   /* Eq. 55 at m = 0: (K_{i-1}^2 - K_i^2)/(8 K_{i-1}^2) */
            wm *= rho_M / rho_K;
            double e1 = (Mp * Mp + m1 * m1 - m2 * m2) / (2.0 * Mp);
            double xc = x[(int64_t)(n - 2 + 2 * (i - 2)) * ld + e], xp = x[(int64_t)(n - 1 + 2 * (i - 2)) * ld + e];
            double cth = 2.0 * xc - 1.0, sth = 2.0 * sqrt(xc * (1.0 - xc)), phi = 2.0 * M_PI * xp;   /* Eq. 25 */
            double pr[4] = { e1, q * sth * cos(phi), q * sth * sin(phi), q * cth };
            double Qr[4] = { Mp - e1, -pr[1], -pr[2], -pr[3] };
            if (i == 2) {
                memcpy(pout[0], pr, sizeof pr);
                memcpy(Q, Qr, sizeof Qr);
            } else {
                double Qn[4];
                boost_to(Q, Mp, pr, pout[i - 2]);
                boost_to(Q, Mp, Qr, Qn);
                memcpy(Q, Qn, sizeof Qn);
            }
        }
        memcpy(pout[n - 1], Q, sizeof Q);
        double in_a[4] = { 0.5 * sqrt_s, 0.0, 0.0, 0.5 * sqrt_s }, in_b[4] = { 0.5 * sqrt_s, 0.0, 0.0, -0.5 * sqrt_s };
        for (int mu = 0; mu < 4; ++mu) {
            p[(int64_t)(0 + mu) * ld + e] = in_a[mu];
            p[(int64_t)(4 + mu) * ld + e] = in_b[mu];
        }
        for (int j = 0; j < n; ++j)
            for (int mu = 0; mu < 4; ++mu) p[(int64_t)(4 * (j + 2) + mu) * ld + e] = pout[j][mu];
        w[e] = phi1 * pow(K[1], 2 * n - 4) * wn * wm;
    }
    return nbad;
}

/* ------------------------------------------------------------------------ */
/* F: FastRambo inverse.  Eq. 64 for the masses; angles by */
/* undoing Eq. 25 in the rest frame of Q_{i-1} (reading F-1..F-5).           */
/* p: outgoing momenta are rows 8.. ; frame: any frame (Q_1 = sum of p).     */
/* ------------------------------------------------------------------------ */
void orc_fastrambo_inverse(int64_t N, int n, const double *p, double *x, double *w, int64_t ld)
{
    double phi1 = orc_phi_n(n, 1.0);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double pj[ORC_MAX_N + 1][4], Q[ORC_MAX_N + 2][4], M[ORC_MAX_N + 2];
        for (int j = 1; j <= n; ++j)
            for (int mu = 0; mu < 4; ++mu) pj[j][mu] = p[(int64_t)(4 * (j + 1) + mu) * ld + e];
        for (int mu = 0; mu < 4; ++mu) Q[n][mu] = pj[n][mu];
        for (int i = n - 1; i >= 1; --i)
            for (int mu = 0; mu < 4; ++mu) Q[i][mu] = Q[i + 1][mu] + pj[i][mu];
        for (int i = 1; i <= n - 1; ++i) {
            double m2 = Q[i][0] * Q[i][0] - Q[i][1] * Q[i][1] - Q[i][2] * Q[i][2] - Q[i][3] * Q[i][3];
            M[i] = sqrt(m2 > 0.0 ? m2 : 0.0);
        }
        M[n] = 0.0;
        double wn = 1.0;
        for (int i = 2; i <= n - 1; ++i) {
            int k = n - i;
            double c = ORC_CK[k];
            double u = M[i] / M[i - 1];
            double y = pow(u, 2 * k);                      /* Eq. 60 */
            x[(int64_t)(i - 2) * ld + e] = orc_rqf_forward(y, c);
            double omu2 = 1.0 - u * u;
            wn *= (double)(k + 1) * omu2 / orc_rqf_density(y, c);
        }
        for (int i = 2; i <= n; ++i) {
            double pr[4];
            boost_from(Q[i - 1], M[i - 1], pj[i - 1], pr);
            double pm = sqrt(pr[1] * pr[1] + pr[2] * pr[2] + pr[3] * pr[3]);
            double cth = pr[3] / pm;
            double phi = atan2(pr[2], pr[1]);
            if (phi < 0.0) phi += 2.0 * M_PI;
            x[(int64_t)(n - 2 + 2 * (i - 2)) * ld + e] = 0.5 * (cth + 1.0);
            x[(int64_t)(n - 1 + 2 * (i - 2)) * ld + e] = phi / (2.0 * M_PI);
        }
        if (w) w[e] = phi1 * pow(M[1], 2 * n - 4) * wn;
    }
}

/* ------------------------------------------------------------------------ */
/* Inverse of orc_rambo_massive_reweight with the FastRambo u_i (the paper's   */
/* invertibility check uses massive gg -> t tbar g g kinematics). */
/* Undo the steps in reverse: Q_i = sum_{j>=i} p_j, M_i = sqrt(Q_i^2) (i < n),  */
/* K_i = M_i - sum_{j>=i} m_j (Eq. 69, reading K-4a), u_i = K_i / K_{i-1},     */
/* r_i = G_RQF(u_i^{2k}; c_k) (Eq. 64); angles from p_{i-1} boosted to the rest */
/* frame of Q_{i-1} (Eq. 25 inverted).  w (optional): the forward weight,      */
/* Eq. 68 evaluated from the recovered masses and the rest-frame momenta.      */
/* ------------------------------------------------------------------------ */
void orc_rambo_massive_reweight_inverse(int64_t N, int n, const double *masses, const double *p, double *x,
                                        double *w, int64_t ld)
{
    double phi1 = orc_phi_n(n, 1.0);
    double msum[ORC_MAX_N + 2];
    msum[n + 1] = 0.0;
    for (int i = n; i >= 1; --i) msum[i] = msum[i + 1] + masses[i - 1];
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double pj[ORC_MAX_N + 1][4], Q[ORC_MAX_N + 2][4], M[ORC_MAX_N + 2], K[ORC_MAX_N + 2];
        for (int j = 1; j <= n; ++j)
            for (int mu = 0; mu < 4; ++mu) pj[j][mu] = p[(int64_t)(4 * (j + 1) + mu) * ld + e];
        for (int mu = 0; mu < 4; ++mu) Q[n][mu] = pj[n][mu];
        for (int i = n - 1; i >= 1; --i)
            for (int mu = 0; mu < 4; ++mu) Q[i][mu] = Q[i + 1][mu] + pj[i][mu];
        for (int i = 1; i <= n - 1; ++i) {
            double m2 = Q[i][0] * Q[i][0] - Q[i][1] * Q[i][1] - Q[i][2] * Q[i][2] - Q[i][3] * Q[i][3];
            M[i] = sqrt(m2 > 0.0 ? m2 : 0.0);
            K[i] = M[i] - msum[i];                         /* Eq. 69 */
        }
        M[n] = masses[n - 1];
        K[n] = 0.0;
        double wn = 1.0, wm = 1.0;
        for (int i = 2; i <= n - 1; ++i) {
            int k = n - i;
            double c = ORC_CK[k];
            double u = K[i] / K[i - 1];
            double y = pow(u, 2 * k);                      /* Eq. 60 */
            x[(int64_t)(i - 2) * ld + e] = orc_rqf_forward(y, c);
            wn *= (double)(k + 1) * (1.0 - u * u) / orc_rqf_density(y, c);
            wm *= M[i] / K[i];
        }
        for (int i = 2; i <= n; ++i) {
            double pr[4];
            boost_from(Q[i - 1], M[i - 1], pj[i - 1], pr);
            double q = sqrt(pr[1] * pr[1] + pr[2] * pr[2] + pr[3] * pr[3]);
            double cth = pr[3] / q;
            double phi = atan2(pr[2], pr[1]);
            if (phi < 0.0) phi += 2.0 * M_PI;
            x[(int64_t)(n - 2 + 2 * (i - 2)) * ld + e] = 0.5 * (cth + 1.0);
            x[(int64_t)(n - 1 + 2 * (i - 2)) * ld + e] = phi / (2.0 * M_PI);
            /* Eq. 55: rho(M_{i-1}, M_i, m_{i-1}) = sqrt(lambda)/(8 M^2) = q/(4 M);  rho(K_{i-1}, K_i, 0) = (1 - u_i^2)/8 */
            double uK = K[i] / K[i - 1];
            wm *= (q / (4.0 * M[i - 1])) / ((1.0 - uK * uK) / 8.0);
        }
        if (w) w[e] = phi1 * pow(K[1], 2 * n - 4) * wn * wm;
    }
}

/* ------------------------------------------------------------------------ */
/* K: massive extension, strategy (i) of PAPER.md:510 -- momentum rescaling  */
/* of classic RAMBO (ref. [64]); formulas restated in reading   */
/* K-1..K-3 because the paper prints none.  p rows 8.. are read (massless,   */
/* CM frame) and overwritten; w[e] is multiplied by w_m.  Returns the number */
/* of events whose Newton iteration hit max_iter (their weight is set to 0). */
/* ------------------------------------------------------------------------ */
int64_t orc_massive_rescale(int64_t N, int n, double sqrt_s, const double *masses, double rel_tol,
                            int max_iter, double *p, double *w, int64_t ld)
{
    double msum = 0.0;
    for (int i = 0; i < n; ++i) msum += masses[i];
    int64_t nfail = 0;
#pragma omp parallel for schedule(static) reduction(+ : nfail)
    for (int64_t e = 0; e < N; ++e) {
        double E[ORC_MAX_N];
        for (int i = 0; i < n; ++i) E[i] = p[(int64_t)(4 * (i + 2)) * ld + e];
        double xi = sqrt(1.0 - (msum / sqrt_s) * (msum / sqrt_s));
        int ok = 0;
        for (int it = 0; it <= max_iter; ++it) {
            double F = -sqrt_s, Fp = 0.0;
            for (int i = 0; i < n; ++i) {
                double k0 = sqrt(masses[i] * masses[i] + xi * xi * E[i] * E[i]);
                F += k0;
                Fp += xi * E[i] * E[i] / k0;
            }
            if (fabs(F) <= rel_tol * sqrt_s) { ok = 1; break; }
            if (it == max_iter) break;
            xi -= F / Fp;
        }
        double prod = 1.0, sum = 0.0;
        for (int i = 0; i < n; ++i) {
            double kabs = xi * E[i];
            double k0 = sqrt(masses[i] * masses[i] + kabs * kabs);
            p[(int64_t)(4 * (i + 2) + 0) * ld + e] = k0;
            for (int mu = 1; mu < 4; ++mu) p[(int64_t)(4 * (i + 2) + mu) * ld + e] *= xi;
            prod *= kabs / k0;
            sum += kabs * kabs / k0;
        }
        double wm = pow(xi, 2 * n - 3) * sqrt_s * prod / sum;
        if (!ok || !isfinite(wm)) { wm = 0.0; ++nfail; }
        w[e] *= wm;
    }
    return nfail;
}

/* ------------------------------------------------------------------------ */
/* X: Bjorken-x sampling and lab boost.  Eq. 19 with m^2 = 0, */
/* Eq. 21-23, boost_beam; reading X-1, X-2. */
/* ------------------------------------------------------------------------ */
void orc_pdf_x_sample(int64_t N, double s_had, double tau_min, const double *r, double *x1x2,
                      double *sqrt_shat, double *jac, int64_t ld)
{
    double lmin = log(tau_min);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double r0 = r[e], r1 = r[ld + e];
        double ltau = (1.0 - r0) * lmin;                   /* Eq. 19: tau = exp[r log 1 + (1-r) log tau_min] */
        double tau = exp(ltau);
        x1x2[e] = exp(r1 * ltau);                          /* Eq. 22 */
        x1x2[ld + e] = exp((1.0 - r1) * ltau);
        sqrt_shat[e] = sqrt(tau * s_had);
        jac[e] = tau * (-lmin) * (-ltau);                  /* 1/g_{nu=1} times |log tau| of Eq. 23 */
    }
}

/* Boost rows 8.. from the partonic CM frame to the lab along z with rapidity
 * (1/2) ln(x1/x2), and fill the incoming rows 0..7 (lab frame). */
void orc_pdf_boost(int64_t N, int n, double s_had, const double *x1x2, double *p, int64_t ld)
{
    double Eb = 0.5 * sqrt(s_had);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double x1 = x1x2[e], x2 = x1x2[ld + e];
        double rt = sqrt(x1 * x2);
        double ch = (x1 + x2) / (2.0 * rt), sh = (x1 - x2) / (2.0 * rt);
        for (int j = 2; j < n + 2; ++j) {
            double E = p[(int64_t)(4 * j) * ld + e], pz = p[(int64_t)(4 * j + 3) * ld + e];
            p[(int64_t)(4 * j) * ld + e] = E * ch + pz * sh;
            p[(int64_t)(4 * j + 3) * ld + e] = pz * ch + E * sh;
        }
        double a[4] = { x1 * Eb, 0.0, 0.0, x1 * Eb }, b[4] = { x2 * Eb, 0.0, 0.0, -x2 * Eb };
        for (int mu = 0; mu < 4; ++mu) {
            p[(int64_t)mu * ld + e] = a[mu];
            p[(int64_t)(4 + mu) * ld + e] = b[mu];
        }
    }
}

/* ------------------------------------------------------------------------ */
/* T: toy integrand of BASELINE.json (not from the paper; reading T):        */
/* f = prod_{i=1}^{n-1} 1/(s_{i,i+1} + reg), open chain over outgoing        */
/* neighbours, s_ij := E_i E_j |n_i - n_j|^2 with n = p/E.                   */
/* ------------------------------------------------------------------------ */
void orc_toy_integrand(int64_t N, int n, double reg, const double *p, double *f, int64_t ld)
{
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < N; ++e) {
        double prod = 1.0;
        for (int i = 0; i < n - 1; ++i) {
            const double *pa = p + (int64_t)(4 * (i + 2)) * ld + e;
            const double *pb = p + (int64_t)(4 * (i + 3)) * ld + e;
            double Ea = pa[0], Eb = pb[0];
            double dx = pa[ld] / Ea - pb[ld] / Eb;
            double dy = pa[2 * ld] / Ea - pb[2 * ld] / Eb;
            double dz = pa[3 * ld] / Ea - pb[3 * ld] / Eb;
            double sij = Ea * Eb * (dx * dx + dy * dy + dz * dz);
            prod *= 1.0 / (sij + reg);
        }
        f[e] = prod;
    }
}

/* ------------------------------------------------------------------------ */
/* U: hit-or-miss unweighting against a fixed w_max (reading U) */
/* accept <=> u * w_max < w, u = uniform 0 of stream `stream`; accepted       */
/* indices in increasing order; w_out = max(1, w / w_max).  Sequential on     */
/* purpose.  Returns the number accepted (idx/w_out hold min(n_acc, cap)).    */
/* ------------------------------------------------------------------------ */
int64_t orc_unweight(int64_t N, const double *w, double w_max, uint64_t seed, uint32_t stream,
                     uint64_t event_offset, int64_t cap, int64_t *idx, double *w_out)
{
    int64_t n_acc = 0;
    for (int64_t e = 0; e < N; ++e) {
        double u = orc_uniform(seed, stream, event_offset + (uint64_t)e, 0u);
        if (u * w_max < w[e]) {
            if (n_acc < cap) {
                idx[n_acc] = e;
                double ratio = w[e] / w_max;
                w_out[n_acc] = ratio > 1.0 ? ratio : 1.0;
            }
            ++n_acc;
        }
    }
    return n_acc;
}

double orc_max(int64_t N, const double *w)
{
    double m = -INFINITY;
    for (int64_t e = 0; e < N; ++e)
        if (w[e] > m) m = w[e];
    return m;
}
