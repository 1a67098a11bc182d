// ms_params.h -- plain-data launch parameters shared by the host API (ms_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ms {

constexpr int kBlock = 256;
constexpr int kMaxN = 9;

struct PhiloxKey {
    uint32_t k0, k1, stream;
    uint64_t event_offset;
};

// The ten round keys of a Philox4x32-10 call, (k0 + r W0, k1 + r W1) for r = 0..9 (Weyl sequence of the key, reading R-1):
// they depend on the seed alone, so the host works them out once and the generation kernels read them as constant-bank
// operands of the XORs (in the kernel the additions were re-done per 256-event tile: 18 instructions per event).
struct PhiloxRoundKeys {
    uint32_t k[20];
};
inline PhiloxRoundKeys philox_round_keys(uint32_t k0, uint32_t k1)
{
    PhiloxRoundKeys rk;
    for (int r = 0; r < 10; ++r) {
        rk.k[2 * r] = k0 + (uint32_t)r * 0x9E3779B9u;
        rk.k[2 * r + 1] = k1 + (uint32_t)r * 0xBB67AE85u;
    }
    return rk;
}

// ---------------------------------------------------------------------------------------------------
// Launch parameters (plain data, passed by value as a __grid_constant__).
// ---------------------------------------------------------------------------------------------------
struct GenParams {
    int64_t N, ld;
    PhiloxKey key;
    const double* x_rows;      // [d][ld] uniforms, or nullptr -> Philox in-kernel
    const double* sqrt_s_arr;  // per-event CM energy, or nullptr
    const double* edges;       // VEGAS edges [grid_dims][grid_bins+1], or nullptr
    int grid_dims, grid_bins;
    int pdf, toy, max_iter, _pad;
    double sqrt_s;             // fixed CM energy (partonic), or hadronic sqrt(s_had) when pdf
    double phi_unit;           // Phi_n(1), Eq. 81
    double phi_fixed;          // Phi_n(sqrt_s) when the energy is fixed
    double ln_tau_min, rel_tol, toy_reg;
    double grid_bins_f;        // (double)grid_bins
    double jac_scale;          // grid_bins^grid_dims: the VEGAS Jacobian is jac_scale * prod of bin widths
    double masses[kMaxN];
    double msuf[kMaxN + 1];    // msuf[i] = sum_{j >= i} masses[j] (0-based), msuf[n] = 0: Eq. 69
    int massmode, _pad2;       // 0 massless, 1 Newton rescale (strategy i), 2 reweighting (strategy ii)
    double* p;                 // [4(n+2)][ld]
    double* w;                 // [N]
    double* x1x2;              // [2][ld] or nullptr
    uint32_t* fail;
    // fused unweighting decision (ms_generate_unweight), or accept_bits == nullptr
    const double* wmax;        // device scalar
    uint32_t* accept_bits;     // [8 ceil(N/256)]: bit (e & 31) of word e >> 5 <=> event e accepted
    PhiloxKey ukey;            // unweighting stream
    PhiloxRoundKeys rk, urk;   // round keys of key / ukey (filled by the dispatcher)
};

struct InvParams {
    int64_t N, ld;
    const double* p;
    double* x;
    double* w;                 // or nullptr
    double phi_unit;
    const double* edges;       // ms_fastrambo_inverse_vegas: [3n-4][grid_bins + 1], else nullptr (x = the phase-space variables)
    int grid_bins;             // 64 or 128
    double jac_scale;          // grid_bins^(3n-4)
    double masses[kMaxN];      // massive inverse only
    double msuf[kMaxN + 1];    // msuf[i] = sum_{j >= i} masses[j]
};

struct ChiliParams {
    int64_t N, ld;
    PhiloxKey key;
    PhiloxRoundKeys rk;        // round keys of `key`
    const double* x_rows;      // [3n-2][ld] uniforms, or nullptr -> Philox in-kernel
    double s_lab, sqrt_s, half_sqrt_s, inv_half_sqrt_s;
    double weight_unit;        // (2 pi)^(4-3n) * 2 / s_lab * pi^(n-1) * prod_{i<n-1} (constant factor of dpT^2/dr: Eq. 72
                               // 1/pTmin^2 - 1/pTmax^2, Eq. 73 2 (2 lambda + pTmax))
    double inv_ptmax2;         // 1 / pT_max^2, pT_max = sqrt(s_lab)/2 (Eq. 71)
    double masses[kMaxN];
    double inv_ptmin2[kMaxN];  // 1 / pT_min^2 (Eq. 72) or 0 -> Eq. 73
    double lambda_c[kMaxN];    // regulator of Eq. 73: the mass, or 1 for a massless particle
    double y_cut[kMaxN];       // > 0: |y| <= y_cut; else no rapidity cut
    double* p;                 // [4(n+2)][ld]
    double* w;                 // [N]
    double* x1x2;              // [2][ld] or nullptr
};

struct RescaleParams {
    int64_t N, ld;
    double sqrt_s, rel_tol;
    int max_iter, _pad;
    double masses[kMaxN];
    double* p;
    double* w;
    uint32_t* fail;
};

}  // namespace ms
