/*
 * madspace_b200.h -- C ABI of the B200-native MadSpace phase-space hot path (arXiv 2602.06895).
 *
 * The library maps uniforms r in (0,1)^d to phase-space points x = G(r) with density g and
 * returns the Monte Carlo weight 1/g [* f] (Eq. 1-5; forward Jacobian = 1/g,
 * PAPER.md:112, Eq. 12).  Conventions follow the paper's own C interface style (UMAMI,
 * PAPER.md:656-677): C-callable functions with fixed signatures, batched over events,
 * device-resident pointers with a defined layout, no host<->device copies inside a call.
 *
 * COMMON CONVENTIONS
 *  - Every pointer named d_* is a DEVICE pointer owned by the caller (torch tensors); h_* is a HOST
 *    pointer.  The library allocates nothing, keeps no global state (except the last CUDA error
 *    code) and never synchronises: each call validates its arguments on the host, enqueues its
 *    kernel(s) on `stream` (a cudaStream_t passed as void*) and returns.
 *  - Layout: structure of arrays, fp64.  A "row" is N consecutive doubles; a[row*ld + e] is the
 *    value of event e, ld >= N the row stride in elements.  Base pointers must be 16-byte aligned.
 *    Momentum rows: row = 4*particle + mu with mu = (E,px,py,pz) (Eq. 77 component
 *    order); particles 0,1 are the incoming partons a,b, particles 2..n+1 the outgoing p_1..p_n
 *    of Eq. 53.  A momentum block therefore has 4*(n+2) rows.
 *  - Random numbers: Philox4x32-10, counter = (event_lo, event_hi, j>>1, stream), key = seed, where
 *    event = rng.event_offset + e is the GLOBAL event index and j the uniform's dimension index;
 *    uniform j takes output words (0,1) if j is even, (2,3) if odd: W = w_a<<32 | w_b,
 *    u = (2*(W>>12)+1) * 2^-53, in the open interval (0,1) (readings R-1..R-3).
 *    Wherever a uniform-row pointer may be NULL, NULL means "draw the uniforms in-kernel".
 *  - N <= MS_MAX_EVENTS = 2^31 events per call of the phase-space entry points (MS_EINVAL beyond).
 *  - Return value: MS_OK, or a negative code detected on the host BEFORE any launch (nothing was
 *    enqueued), or MS_ECUDA when a launch failed (raw cudaError_t: ms_last_cuda_error()).
 *  - Per-event failures (Newton cap hit, non-finite weight) do not fail the call: the event gets
 *    weight 0 and, if d_fail != NULL, *d_fail (a device uint32 the caller zeroed) is incremented.
 *  - n = number of outgoing particles, 2 <= n <= MS_MAX_N (k = n-2 <= 7: Table 1).
 */
#ifndef MADSPACE_B200_H
#define MADSPACE_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MS_MAX_N 9
#define MS_MAX_DIMS 32      /* VEGAS grid dimensions */
#define MS_MAX_EVENTS ((int64_t)1 << 31) /* events per call of the per-multiplicity kernels (ms_generate, ms_fastrambo,
                                            ms_rambo_*, ms_fastrambo_inverse, ms_chili): 32-bit local event index;
                                            longer batches are split by the caller (advance rng.event_offset) */
#define MS_MAX_LD ((int64_t)0xFFFFFFFF)     /* row stride of those calls: a 32-bit element count */
#define MS_MAX_BINS 1024    /* VEGAS bins per dimension; d*(n_bins+1)*16 B must fit 200 KB of shared memory */

enum {
    MS_OK = 0,
    MS_EINVAL = -1,   /* null / misaligned pointer, N <= 0, n out of range, ld < N, bad flag */
    MS_EGRID = -2,    /* reported by ms_check_grid: edges not strictly increasing, x_0 != 0 or x_nb != 1 */
    MS_EKIN = -3,     /* sum of masses >= sqrt_s, tau_min outside (0,1), sqrt_s <= 0 with no per-event array */
    MS_ECUDA = -4,    /* kernel launch failed */
    MS_ELIMIT = -5    /* size beyond the fixed capacity of an entry point that allocates nothing (ms_unweight_static) */
};

/* Counter-based RNG coordinates, passed by value (reading R-2). */
typedef struct ms_rng {
    uint64_t seed;          /* Philox key */
    uint32_t stream;        /* 0: phase-space uniforms, 1: unweighting uniform */
    uint32_t reserved;      /* must be 0 */
    uint64_t event_offset;  /* global index of event 0 of this call */
} ms_rng;

const char* ms_version(void);
/* Raw cudaError_t of the last MS_ECUDA returned to the CALLING THREAD (thread-local; 0 if none). The library keeps no
 * other state: every call is re-entrant and may be issued from several host threads on different streams -- with the one
 * exception of ms_unweight_static, whose scratch is a device array shared by all its calls (see there). */
int ms_last_cuda_error(void);

/* Host-side validation of a VEGAS edge table h_edges[d][n_bins+1] (reading V-1):
 * MS_OK, or MS_EGRID if any row is not 0 = x_0 < x_1 < ... < x_nb = 1, MS_EINVAL on bad sizes. */
int ms_check_grid(int d, int n_bins, const double* h_edges);

/* ms_vegas_map -- frozen VEGAS grid map (PAPER.md:603 "classic VEGAS", :746 grids adapted then
 * frozen; the paper prints no equations: Lepage's piecewise-linear map, readings V-1..V-3).
 *   direction 0 (forward):  t = r*n_bins, j = min(floor t, n_bins-1), x = x_j + (t-j)(x_{j+1}-x_j),
 *       clamped into [2^-53, 1-2^-53]; d_jac[e] = prod_dims n_bins (x_{j+1}-x_j).
 *       d_in = r rows [d][ld], or NULL -> Philox uniforms j = 0..d-1 of stream rng.stream.
 *   direction 1 (inverse):  j = bin with x_j <= x < x_{j+1} (binary search, every lane of a warp descending its
 *       own path through a breadth-first edge tree in shared memory), r = (j + (x-x_j)/(x_{j+1}-x_j))/n_bins;
 *       d_jac[e] = 1/prod(...).
 *       d_in = x rows (must not be NULL).
 *       The quotient is the IEEE-754 correctly rounded one (the divisor-only part of div.rn.f64 is tabulated per
 *       bin; inputs outside its fast path go through div.rn.f64 itself): results are bit-identical to a / b on the host.
 * d_edges: device table [d][n_bins+1], validated by the caller with ms_check_grid.
 * d_out: [d][ld].  d_jac: [N] or NULL.  d_in and d_out may be the same buffer (in place) or disjoint; a partial
 * overlap is rejected (MS_EINVAL).
 * Errors: MS_EINVAL on bad sizes or pointers, or if the tables exceed 200 KB of shared memory
 * (forward: 16 d n_bins bytes; inverse: 16 d (n_bins+1) + 4 d 2^ceil(log2 n_bins) bytes). */
int ms_vegas_map(int64_t N, int d, int n_bins, const double* d_edges, int direction,
                 const double* d_in, ms_rng rng, double* d_out, double* d_jac, int64_t ld, void* stream);

/* ms_vegas_accumulate / ms_vegas_refine -- adaptation of the grid before it is frozen ("classic VEGAS",
 * :746 "optimized during an initial adaptation phase"; no equations printed: Lepage's algorithm, reading V-4).
 *   accumulate (device): d_hist[dim*n_bins + floor(r_dim n_bins)] += d_w[e]^2 for dim < d, where r_dim is uniform
 *       `dim` of event rng.event_offset + e (seed / stream as in the generating call); d_hist [d][n_bins] is ADDED to
 *       (zero it before the first batch of an iteration).  Summation order is unspecified (fp64 atomics).
 *   refine (host only, no CUDA call): per dimension smooth (d_{j-1} + 6 d_j + d_{j+1})/8, normalise, damp
 *       ((1-d)/ln(1/d))^alpha, and re-split h_edges so that every new bin receives an equal share; a dimension with an
 *       all-zero histogram is copied unchanged.  Returns MS_EGRID if h_edges is not a valid grid. */
int ms_vegas_accumulate(int64_t N, int d, int n_bins, const double* d_w, ms_rng rng, double* d_hist, void* stream);
int ms_vegas_refine(int d, int n_bins, const double* h_hist, double alpha, const double* h_edges, double* h_edges_out);

/* ms_rambo_massless -- exact flat massless n-body phase space, RamboOnDiet (PAPER.md:405-474,
 * Eq. 52-63): intermediate masses M_i = u_i M_{i-1} with u_i solving Eq. 62 (Newton, reading
 * M-3), then n-1 two-body decays (Eq. 54-55, angles Eq. 25).  Weight is flat: d_w[e] = Phi_n(sqrt_s)
 * of Eq. 81 (incl. (2 pi)^(4-3n)).
 *   sqrt_s > 0: fixed CM energy; sqrt_s <= 0: per-event energies d_sqrt_s[N] (must be non-NULL).
 *   d_x: [3n-4][ld] uniforms (rows 0..n-3 -> mass steps i=2..n-1; then (cos theta, phi) pairs per
 *        decay, reading D-1), or NULL -> Philox j = 0..3n-5.
 *   d_p: [4(n+2)][ld] out, frame = CM frame of Q_1; incoming rows = (sqrt_s/2)(1,0,0,+-1).
 *   d_w: [N] out. */
int ms_rambo_massless(int64_t N, int n, double sqrt_s, const double* d_sqrt_s, const double* d_x, ms_rng rng,
                      double* d_p, double* d_w, int64_t ld, uint32_t* d_fail, void* stream);

/* ms_fastrambo -- FastRambo (Eq. 64-67, Table 1): as above with Eq. 62 replaced by
 * the rational-quadratic map, y_i = G_RQF^{-1}(x; c_k) (Eq. 65), u_i = y_i^{1/(2k)}, k = n-i; weight
 * d_w[e] = Phi_n(sqrt_s) * prod_i (k+1)(1-y_i^{1/k})/g_RQF(y_i; c_k) (Eq. 67 / Eq. 63). */
int ms_fastrambo(int64_t N, int n, double sqrt_s, const double* d_sqrt_s, const double* d_x, ms_rng rng,
                 double* d_p, double* d_w, int64_t ld, uint32_t* d_fail, void* stream);

/* ms_fastrambo_inverse -- analytic inverse of ms_fastrambo (Eq. 64; readings F-1..F-5).
 * Reads the outgoing rows 8.. of d_p (any frame in which they were generated from Q_1 = sum p),
 * writes d_x [3n-4][ld] and, if d_w != NULL, the same weight the forward map returns.
 * Degenerate input (no inverse exists): a subsystem Q_i with Q_i^2 <= 0 after rounding (an exactly collinear massless
 * pair) is given the mass 2^-500 Q_i^0, so every output stays finite and inside [0,1] (its mass uniform is below 1e-290, its
 * angles arbitrary), and the event's d_w is 0; a particle with zero momentum gets cos theta uniform 1/2, azimuth 0. */
int ms_fastrambo_inverse(int64_t N, int n, const double* d_p, double* d_x, double* d_w, int64_t ld, void* stream);

/* ms_fastrambo_inverse_vegas -- ms_fastrambo_inverse followed by the inverse direction of ms_vegas_map, in one kernel: the
 * momenta are mapped straight to the uniforms r of a fused generation (Eq. 64, then :603), and the 3n-4
 * phase-space variables never travel through HBM (the two calls write and re-read 16 B per variable and event).
 *   d_edges: [grid_dims][grid_bins + 1], grid_dims == 3n-4 exactly, grid_bins 64 or 128 (the grids of the BASELINE.json
 *            configs; any other grid: MS_EINVAL -- use the two calls).
 *   d_r: [3n-4][ld] out.  Bit for bit what ms_vegas_map(direction 1) returns on the d_x of ms_fastrambo_inverse: same
 *        search, same quotient.
 *   d_w: [N] out or NULL: the weight of ms_fastrambo_inverse times the grid's Jacobian prod_j grid_bins * w_j, i.e. the
 *        weight ms_generate returns for these uniforms (no PDF, no integrand). */
int ms_fastrambo_inverse_vegas(int64_t N, int n, const double* d_p, const double* d_edges, int grid_dims, int grid_bins,
                               double* d_r, double* d_w, int64_t ld, void* stream);

/* ms_massive_rescale -- massive extension, strategy (i) of PAPER.md:510 (momentum rescaling of classic
 * RAMBO, ref. [64]; readings K-1..K-3): solve sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt_s for xi by Newton
 * in registers (the first two steps are Halley's third-order variant of the Newton step, the rest plain Newton) until
 * |F| <= rel_tol*sqrt_s (at most max_iter steps), k_i = (sqrt(m_i^2+xi^2 E_i^2), xi p_i),
 * w_m = xi^(2n-3) sqrt_s prod(|k_i|/k_i^0) / sum(|k_i|^2/k_i^0).
 * d_p: outgoing rows 8.. are read (massless, CM frame) and overwritten; incoming rows untouched.
 * d_w: [N] multiplied in place by w_m.  h_masses: n doubles on the HOST. */
int ms_massive_rescale(int64_t N, int n, double sqrt_s, const double* h_masses, double rel_tol, int max_iter,
                       double* d_p, double* d_w, int64_t ld, uint32_t* d_fail, void* stream);

/* ms_rambo_massive_reweight -- massive extension, strategy (ii) of PAPER.md:510-522 (the one MadSpace adopts): the
 * massless mass chain runs at K_1 = sqrt_s - sum m_j, M_i = K_i + sum_{j>=i} m_j (Eq. 69, reading K-4a), the
 * n-1 two-body decays use the massive two-body momentum (Eq. 24) and the weight is
 *   Phi_n(K_1) w_n prod_{i=2..n} rho(M_{i-1},M_i,m_{i-1})/rho(K_{i-1},K_i,0) prod_{i=2..n-1} M_i/K_i   (Eq. 68, reading K-4b).
 * mapping 0: FastRambo u_i, 1: exact Rambo u_i.  d_x: [3n-4][ld] uniforms or NULL -> Philox.  h_masses: n doubles on
 * the HOST, sum < sqrt_s (else MS_EKIN).  d_p: [4(n+2)][ld] out, CM frame; d_w: [N] out. */
int ms_rambo_massive_reweight(int64_t N, int n, int mapping, double sqrt_s, const double* h_masses, const double* d_x,
                              ms_rng rng, double* d_p, double* d_w, int64_t ld, uint32_t* d_fail, void* stream);

/* ms_rambo_massive_reweight_inverse -- analytic inverse of ms_rambo_massive_reweight with mapping 0 (PAPER.md:740 checks
 * the invertibility on massive gg -> t tbar g g kinematics): Q_i = sum_{j>=i} p_j, M_i = sqrt(Q_i^2),
 * K_i = M_i - sum_{j>=i} m_j (Eq. 69), u_i = K_i/K_{i-1}, r_i = G_RQF(u_i^{2k}; c_k) (Eq. 64), angles in the rest frame of
 * Q_{i-1}.  Reads the outgoing rows 8.. of d_p, writes d_x [3n-4][ld] and, if d_w != NULL, the forward weight. */
int ms_rambo_massive_reweight_inverse(int64_t N, int n, const double* h_masses, const double* d_p, double* d_x,
                                      double* d_w, int64_t ld, void* stream);

/* ms_chili -- the Chili mapping (Eq. 70-77; readings C-1..C-5): particles 1..n-1 in
 * (pT, y, phi) -- pT by Eq. 72 if h_pt_min[i] > 0, else Eq. 73 with lambda_C = m_i or 1 GeV; |y| <= y_max(m_T) of Eq. 74,
 * further limited by h_y_cut[i] > 0; phi from the current recoil direction (Eq. 75) --, particle n by transverse recoil
 * (Eq. 76) and a rapidity in |y| <= y_max(m_T,n), incoming momenta from E+- (Eq. 77).  3n-2 uniforms per event:
 * (r_pT, r_y, r_phi) per generated particle, then r_y of the last one.
 *   d_w[e] = density of dPhi_n dx1 dx2 (incl. (2 pi)^(4-3n); no flux, no PDFs), 0 outside the technical cut
 *            E+- <= sqrt(s_lab) or where Eq. 74 has no solution;  d_x1x2 (optional) = E+-/sqrt(s_lab).
 *   h_masses, h_pt_min, h_y_cut: n doubles on the HOST each, or NULL (all zero).  d_x: [3n-2][ld] or NULL -> Philox.
 *   d_p: [4(n+2)][ld] out, lab frame. */
int ms_chili(int64_t N, int n, double s_lab, const double* h_masses, const double* h_pt_min, const double* h_y_cut,
             const double* d_x, ms_rng rng, double* d_p, double* d_w, double* d_x1x2, int64_t ld, void* stream);

/* ms_pdf_x_boost -- Bjorken-x sampling and lab boost (Eq. 19 with m^2=0, Eq. 21-23;
 * ops r_to_x1x2 and boost_beam; readings X-1, X-2).
 *   phase 0 (sample): tau = tau_min^(1-r_0), x1 = tau^r_1, x2 = tau^(1-r_1);
 *       d_x1x2 [2][ld], d_sqrt_shat[N] = sqrt(tau s_had), d_jac[N] = tau ln(1/tau_min) ln(1/tau).
 *       d_r = rows r_0, r_1 [2][ld] or NULL -> Philox j = 0,1.  d_p unused.
 *   phase 1 (boost): outgoing rows of d_p are boosted along z from the partonic CM frame by
 *       rapidity (1/2) ln(x1/x2); incoming rows are set to x_{1,2} (sqrt(s_had)/2)(1,0,0,+-1).
 *       Reads d_x1x2; d_r, d_sqrt_shat, d_jac unused. */
int ms_pdf_x_boost(int64_t N, int n, double s_had, double tau_min, int phase, const double* d_r, ms_rng rng,
                   double* d_x1x2, double* d_sqrt_shat, double* d_jac, double* d_p, int64_t ld, void* stream);

/* ms_toy_integrand -- BASELINE.json's matrix-element stand-in (not from the paper; reading T):
 * f = prod_{i=1}^{n-1} 1/(s_{i,i+1} + reg), s_ij := E_i E_j |p_i/E_i - p_j/E_j|^2 over outgoing neighbours.
 * d_f[e] = f, or d_f[e] *= f when accumulate != 0. */
int ms_toy_integrand(int64_t N, int n, double reg, const double* d_p, double* d_f, int accumulate, int64_t ld,
                     void* stream);

/* ms_reduce_max -- *d_out = max(d_w[0..N-1]) (w_max of the pre-run, reading U).  d_out must be
 * zero-initialised or hold a lower bound; weights are non-negative. */
int ms_reduce_max(int64_t N, const double* d_w, double* d_out, void* stream);

/* ms_unweight -- single-pass hit-or-miss unweighting against a fixed w_max (reading U)
 * with stable stream compaction (warp ballots per 512-event tile, then a scatter that scans the tile counts: two
 * kernels on `stream`, neither of which waits on another block's progress).
 *   accept_e <=> u_e * w_max < w_e, u_e = Philox uniform j=0 of (rng.seed, rng.stream, event);
 *   accepted events are written in increasing event order: d_idx[k] = e, d_w_out[k] = max(1, w_e/w_max),
 *   d_rows_out[r*cap + k] = d_rows_in[r*ld + e] for r < n_rows (skipped if either pointer is NULL).
 *   *d_n_accepted = true number accepted; only the first `cap` are stored.
 * d_wmax: device scalar; precondition 0 < w_max < inf.  If it is violated (every pre-run weight 0 under tight cuts, a
 * non-finite maximum) NOTHING is accepted: *d_n_accepted = 0 and no output is written -- the caller sees an empty sample
 * instead of infinite output weights.  d_scratch: ms_unweight_scratch_bytes(N) bytes (68 B per 512 events + 64 KB), any content, 16-byte
 * aligned; overwritten. */
size_t ms_unweight_scratch_bytes(int64_t N);
int ms_unweight(int64_t N, const double* d_w, const double* d_wmax, ms_rng rng, int n_rows, const double* d_rows_in,
                int64_t cap, int64_t* d_idx, double* d_w_out, double* d_rows_out, int64_t* d_n_accepted,
                void* d_scratch, size_t scratch_bytes, int64_t ld, void* stream);

/* ms_unweight_static -- ms_unweight for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments without d_scratch / scratch_bytes, same kernels, same results bit for
 * bit.  The scratch is a static device array inside the library, MS_UNWEIGHT_STATIC_SCRATCH_BYTES = 2 293 760 B (2.2 MiB),
 * which every GPU that loads the library holds until the process exits; it serves N <= MS_UNWEIGHT_STATIC_MAX_EVENTS = 2^24
 * events per call (the largest unweighting batch of the BASELINE.json configs).  N beyond that: MS_ELIMIT, nothing is
 * enqueued -- split the batch or use ms_unweight.  The call makes no cudaMalloc / cudaFree and calls no allocating
 * library routine; the first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device,
 * with the caller's current device) and returns MS_ECUDA if that fails -- under stream capture make one call (N = 0
 * suffices) before the capture begins.
 * EVERY call on a device shares the one array: two calls whose kernels can overlap on the GPU (different streams, or
 * different host threads) race on it and corrupt each other's result -- serialise them on one stream, or give all but one
 * of them ms_unweight with its own scratch.  The array keeps the previous call's contents; nothing in it has to start at
 * zero (the decide kernel writes every word the scatter kernel reads), so no clearing is done. */
#define MS_UNWEIGHT_STATIC_MAX_EVENTS ((int64_t)1 << 24)
#define MS_UNWEIGHT_STATIC_SCRATCH_BYTES 2293760
int ms_unweight_static(int64_t N, const double* d_w, const double* d_wmax, ms_rng rng, int n_rows, const double* d_rows_in,
                       int64_t cap, int64_t* d_idx, double* d_w_out, double* d_rows_out, int64_t* d_n_accepted, int64_t ld,
                       void* stream);

/* ms_invariant_map -- analytic 1-D mappings for invariants (Eq. 15-20): flat (Eq. 20), power law with
 * exponent nu = par (Eq. 18; par == 1 selects the logarithmic limit Eq. 19; m2 may be the negative auxiliary mass of
 * PAPER.md:185) and Breit-Wigner with par = m * Gamma (Eq. 16-17).  direction 0: d_out = G(d_in), d_in in [0,1];
 * direction 1: d_out = G^-1(d_in).  d_g (optional) = density g of Eq. 15 at x.  Bounds: scalars x_min, x_max, or per-event
 * arrays d_x_min / d_x_max [N] when non-NULL.  MS_EKIN if x_max <= x_min, m Gamma <= 0 or x_min - m2 <= 0 (power law). */
enum { MS_MAP_FLAT = 0, MS_MAP_POWER = 1, MS_MAP_BW = 2 };
int ms_invariant_map(int64_t N, int kind, int direction, double x_min, double x_max, const double* d_x_min,
                     const double* d_x_max, double m2, double par, const double* d_in, double* d_out, double* d_g, void* stream);

/* Observables, cuts and weighted histograms (Sec. 3.2.4-3.2.5; scales Eq. 79-80; the paper names the
 * observables without formulas: DESIGN.md reading O-1).  Particle indices a, b count row blocks: 0, 1 incoming,
 * 2.. outgoing.  phi in (-pi, pi], theta in [0, pi], dphi folded into [0, pi], deta = |eta_a - eta_b|,
 * dR = sqrt(deta^2 + dphi^2), mass = sqrt(max((p_a + p_b)^2, 0)); event level: sqrt(s-hat) from the incoming rows,
 * E_T^tot = sum E pT/|p| (Eq. 79) and H_T = sum sqrt(m^2 + pT^2) (Eq. 80, m^2 = max(E^2 - |p|^2, 0)) over the first n_out
 * outgoing particles.
 *   ms_observable:     d_obs[e] = observable `kind` of event e.
 *   ms_cut:            d_w[e] = 0 unless lo <= d_obs[e] <= hi (+-infinity allowed; a NaN observable fails the cut).
 *   ms_histogram_fill: d_sum_w / d_sum_w2 [n_bins + 2] += sum of w / w^2 per slot; slot 0 = underflow, 1..n_bins the
 *                      uniform bins of [lo, hi), n_bins + 1 = overflow; NaN observables are skipped.  Summation order
 *                      is unspecified (fp64 atomics). */
enum {
    MS_OBS_E = 0, MS_OBS_PX, MS_OBS_PY, MS_OBS_PZ, MS_OBS_PT, MS_OBS_PABS, MS_OBS_PHI, MS_OBS_THETA, MS_OBS_Y, MS_OBS_ABSY,
    MS_OBS_ETA, MS_OBS_ABSETA, MS_OBS_DPHI, MS_OBS_DETA, MS_OBS_DR, MS_OBS_MASS, MS_OBS_SQRT_SHAT, MS_OBS_ET_TOT, MS_OBS_HT,
    MS_OBS_COUNT
};
int ms_observable(int64_t N, int kind, int a, int b, int n_out, const double* d_p, double* d_obs, int64_t ld, void* stream);
int ms_cut(int64_t N, const double* d_obs, double lo, double hi, double* d_w, void* stream);
int ms_histogram_fill(int64_t N, const double* d_obs, const double* d_w, double lo, double hi, int n_bins, double* d_sum_w,
                      double* d_sum_w2, void* stream);

/* Running-maximum unweighting with an overweight allowance ("We estimate the maximum event weight on the
 * fly, allowing for a user-defined amount of overweight events relative to the total cross section ... a final
 * unweighting with respect to the final maximum weight is performed"; no formulas printed: DESIGN.md reading U-2).
 *   ms_weight_histogram (device): d_counts[k] += number of weights whose IEEE-754 bits 62..48 equal k (MS_HIST_BINS =
 *       32768 bins, 16 per octave); weights that are not positive finite numbers are not counted.  Exact integers, so
 *       the statistic does not depend on the order or batching of the events.  d_counts is ADDED to.
 *   ms_wmax_from_histogram (host only): *h_wmax = the smallest bin edge lo_k with
 *       sum_{j>=k} count_j (lo_{j+1} - lo_k) <= fraction * sum_j count_j lo_j, which guarantees
 *       sum_{w > w_max} (w - w_max) <= fraction * sum w;  0 for an empty histogram, +inf if no finite edge qualifies.
 *   Each batch is then unweighted with ms_unweight against the running maximum; the kept events are finally
 *   unweighted against the final maximum w_f by ms_unweight applied to max(w, w_old) (ms_elementwise_max) with a
 *   fresh uniform stream: an event kept with probability min(1, w/w_old) survives with min(1, max(w, w_old)/w_f). */
#define MS_HIST_BINS 32768
/* ms_gather (bookkeeping of the kept events, no arithmetic on the data): d_out[r*ld_out + k] = d_in[r*ld_in + d_idx[k]] for
 * r < n_rows, k < K (8-byte words copied bit for bit: doubles, or int64 viewed as such), and, if d_idx_out != NULL,
 * d_idx_out[k] = d_idx[k] + idx_add (local -> global event index).  Pointers 8-byte aligned; d_out must not overlap d_in. */
int ms_gather(int64_t K, const int64_t* d_idx, int n_rows, const double* d_in, int64_t ld_in, double* d_out, int64_t ld_out,
              int64_t idx_add, int64_t* d_idx_out, void* stream);
int ms_weight_histogram(int64_t N, const double* d_w, uint64_t* d_counts, void* stream);
int ms_wmax_from_histogram(const uint64_t* h_counts, double fraction, double* h_wmax);
int ms_elementwise_max(int64_t N, const double* d_a, const double* d_b, double* d_out, void* stream);

/* ms_generate -- the fused hot path: Philox -> VEGAS -> [x1,x2] -> Rambo/FastRambo -> [massive rescale]
 * -> [lab boost] -> [toy integrand] -> weight, one thread per event, everything in registers, only the
 * momenta and the weight are written.  Computes exactly what the chain
 * ms_vegas_map, ms_pdf_x_boost(0), ms_rambo_massless|ms_fastrambo, ms_massive_rescale, ms_pdf_x_boost(1),
 * ms_toy_integrand computes; d_w[e] = jac_VEGAS * w_PS [* J_x] [* w_m] [* f]. */
typedef struct ms_gen_config {
    int32_t n;             /* outgoing particles */
    int32_t mapping;       /* 0 FastRambo, 1 exact Rambo */
    int32_t grid_dims;     /* 0: no grid (uniforms used directly); else >= uniforms consumed */
    int32_t grid_bins;
    int32_t pdf;           /* 1: dims 0,1 -> (tau, y); phase space at sqrt(tau s_had); boost to lab */
    int32_t massive;       /* 0: massless; 1: Newton rescale to `masses` (strategy i); 2: reweighting (strategy ii, Eq. 68-69) */
    int32_t toy;           /* 1: multiply the weight by the toy integrand */
    int32_t max_iter;      /* Newton cap of the rescale */
    int32_t tail_unit_jacobian; /* 1: the caller asserts that every grid dimension the phase-space map does not consume
                              (index >= 3n-4 [+2 with pdf]) has n_bins*(x_{j+1}-x_j) == 1.0 exactly in every bin (e.g. a
                              uniform grid with a power-of-two bin count), so its Jacobian factor is exactly 1 and the
                              kernel skips it; 0: those dimensions are drawn and looked up like the others */
    int32_t reserved;      /* must be 0 */
    double sqrt_s;         /* partonic (pdf=0) or hadronic (pdf=1) CM energy */
    double tau_min;
    double rel_tol;        /* rescale tolerance */
    double toy_reg;
    double masses[MS_MAX_N];
} ms_gen_config;

/* d_edges: [grid_dims][grid_bins+1] or NULL when grid_dims = 0.  d_p: [4(n+2)][ld].  d_w: [N].
 * d_x1x2: [2][ld] or NULL (pdf only). */
int ms_generate(const ms_gen_config* cfg, int64_t N, ms_rng rng, const double* d_edges, double* d_p, double* d_w,
                double* d_x1x2, int64_t ld, uint32_t* d_fail, void* stream);

/* ms_generate_unweight -- ms_generate with the hit-or-miss decision of ms_unweight taken in the same kernel (
 * reading U): possible whenever w_max is known before the launch, i.e. for every batch after the pre-run.  Beside everything
 * ms_generate writes, bit (e & 31) of d_accept_bits[e >> 5] is set iff u_e * w_max < w_e, with u_e = Philox uniform j = 0 of
 * (rng_unweight.seed, rng_unweight.stream, rng_unweight.event_offset + e) -- the decision ms_unweight takes, bit for bit.
 * d_accept_bits: ms_accept_bits_words(N) = 8 ceil(N/256) uint32, 16-byte aligned, every word is written.  d_wmax: device
 * scalar, read at kernel start (precondition 0 < w_max < inf, else nothing is accepted).
 * ms_unweight_compact -- the compaction half of ms_unweight for decisions that already exist as such a bit array: same
 * outputs (d_idx, d_w_out = max(1, w/w_max), d_rows_out, *d_n_accepted; stable order, `cap` as in ms_unweight), same
 * scratch (ms_unweight_scratch_bytes(N)); reads 4 bytes per 32 events instead of drawing a uniform per event. */
size_t ms_accept_bits_words(int64_t N);
int ms_generate_unweight(const ms_gen_config* cfg, int64_t N, ms_rng rng, const double* d_edges, double* d_p, double* d_w,
                         double* d_x1x2, int64_t ld, uint32_t* d_fail, const double* d_wmax, ms_rng rng_unweight,
                         uint32_t* d_accept_bits, void* stream);
int ms_unweight_compact(int64_t N, const double* d_w, const double* d_wmax, const uint32_t* d_accept_bits, int n_rows,
                        const double* d_rows_in, int64_t cap, int64_t* d_idx, double* d_w_out, double* d_rows_out,
                        int64_t* d_n_accepted, void* d_scratch, size_t scratch_bytes, int64_t ld, void* stream);

/* ms_fill_uniforms -- materialise Philox uniforms j = 0..d-1 as rows d_r[d][ld] (step S0 on its own). */
int ms_fill_uniforms(int64_t N, int d, ms_rng rng, double* d_r, int64_t ld, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MADSPACE_B200_H */
