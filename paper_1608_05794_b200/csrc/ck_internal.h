// Internal declarations shared by the libck translation units (product path; no oracle code).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/ck.h"

namespace ck {

constexpr double R_U = 8.31446261815324e7;  // erg/(mol K)
constexpr double R_CAL = 1.98720425864083;  // cal/(mol K)
constexpr double P_0 = 1.01325e6;           // dyn/cm^2 ("one atmosphere")
constexpr int MAX_TINT = 8;
constexpr int RPH = 6;   // header doubles of an rpack row
constexpr int SPS = 28;  // doubles per species row of spack
constexpr double T_SAFE_LO = 250.0, T_SAFE_HI = 4500.0;  // window in which the fast rows need no exp range checks                 // temperature intervals (distinct t_mid values + 1)

// Device view of the packed mechanism (all pointers into one device arena; passed by value to kernels).
// Reactions are regrouped by type: [0,r_22) A+B<=>C+D (four distinct species), [r_22,r_dup) other plain rows with distinct slot species (both groups: exp arguments bounded, see ck_mech.cu), [r_dup,r_tb) plain with a
// repeated species (nu >= 2 or a species on both sides), [r_tb,r_lind) three-body, [r_lind,r_troe) Lindemann,
// [r_troe,R) Troe.  Every per-reaction array is SoA over the regrouped index.
// Stoichiometry is stored as SLOTS: each side of a reaction is expanded to exactly three species indices,
// nu copies of each participant, padded with the dummy index K (the kernels keep C[K] = 1 and a sink
// accumulator at K), so rate products and the omega scatter are branch-free.
struct MechDev {
  int K, R, nT;
  int cv;                     // 1: constant-volume reactors: the batch argument `p` holds the density rho
  int r_22;                   // leading rows of the plain group with at most two reactants and two products, all
                              //   distinct (A + B <=> C + D; a missing partner is the dummy species K)
  int r_dup, r_tb, r_lind, r_troe;
  int r_tbf;                  // [r_tb, r_tbf): three-body rows with distinct slot species, bounded exponents, <= 6 efficiencies
  double t_safe_lo, t_safe_hi;  // see ck_mech.cu `bounded`
  double tedge[MAX_TINT];     // interval t holds tedge[t-1] < T <= tedge[t]; nT-1 finite edges
  const double* W;            // [K]
  const double* invW;         // [K]
  const double* nlo;          // [7][K] NASA-7, T <= t_mid
  const double* nhi;          // [7][K]
  const double* tmid;         // [K]
  const double* spack;        // [K][SPS] AoS for smem staging: W, 1/W, t_mid, 0; cp/R coefficients a1..a5 (low range,
                              //   high range); H/RT coefficients a1, a2/2, a3/3, a4/4, a5/5, a6 (low, high); 2 pad
  const double* lnA;          // [R]  Eq. 15: ln k_f = lnA + beta lnT - Ta/T
  const double* beta;         // [R]
  const double* Ta;           // [R]  Ea / R_cal
  const double* krc;          // [nT][7][R]  ln k_r = c0 + c1 lnT + c2/T + c3 T + c4 T^2 + c5 T^3 + c6 T^4
  const int* slot;            // [6][R]  slots 0-2 reactants, 3-5 products (species index or K)
  const int* rflag;           // [R]  bit 0: a species sits in two slots of the reaction
  const double* rpack;        // [R][rstride] AoS for smem staging: lnA, beta, Ta, slots (6 x 10 bit in the
                              //   low/high 32-bit words), slots 0, 1, 3, 4 once more as 32-bit words holding
                              //   slot << 12 (byte offset of the C column in a 512-thread CTA; >> 11 is the
                              //   tensor-memory column), then per interval 8 doubles: c0..c6, 0
  int rstride;                // = RPH + 8 nT
  const double* xpack;        // [R - r_tb][16] AoS for smem staging of third-body / falloff rows: lnA0, beta0, Ta0,
                              //   Troe a, 1/T***, 1/T*, T**, packed (n_eff | 6 x 10-bit species), 6 x (alpha-1), 0, 0
                              //   (n_eff field 15: more than 6 efficiencies, read them from eptr/espec/eval1)
  const int* eptr;            // [R - r_tb + 1] CSR of non-unit efficiencies, rows = reactions r_tb..R-1
  const int* espec;
  const double* eval1;        // alpha - 1
  const double* lnA0;         // [R - r_lind] low-pressure limit of falloff rows
  const double* beta0;
  const double* Ta0;
  const double* troe;         // [4][R - r_troe]  a, 1/T***, 1/T*, T** (T** < 0: absent)
  // transposed stoichiometry (gather form for cooperative kernels): species k <- sum nu_ki q_i
  const int* tptr;            // [K+1]
  const int* tent;            // (reaction << 8) | (net nu + 128)
  int n_tent;                 // entries of tent
  const int* perm;            // [R] regrouped index -> caller's reaction index
};

void set_error(const char* fmt, ...);
int32_t cuda_fail(cudaError_t e, const char* what);

}  // namespace ck

struct ck_mech {
  int device = 0;
  int sms = 148;              // SM count of `device` (grid sizing)
  ck::MechDev dev;            // device view
  void* arena = nullptr;      // device allocation backing `dev`
  size_t arena_bytes = 0;
  // host copies used by the launch logic / roofline accounting
  int K = 0, R = 0;
  int n_tb = 0, n_lind = 0, n_troe = 0, n_rev = 0;
  long long n_part = 0, n_eff = 0;
  // cached device staging buffers of the *_host entry points
  void* stage = nullptr;
  size_t stage_bytes = 0;
  cudaStream_t hstream = nullptr;
  cudaStream_t pstream[3] = {nullptr, nullptr, nullptr};   // column-block pipeline of ck_rhs_host
};

#define CK_CUDA(call)                                                    \
  do {                                                                   \
    cudaError_t e_ = (call);                                             \
    if (e_ != cudaSuccess) return ck::cuda_fail(e_, #call);              \
  } while (0)
