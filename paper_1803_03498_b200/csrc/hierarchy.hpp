// hierarchy.hpp -- host-side hierarchy and coefficient builder of the CUDA library.
//
// Index set (Eq. 9), +/- link graph, mode map (Eq. 10-11),
// Matsubara coefficients (Eq. 19-20), terminator (Eq. 14) and
// the rescaled coupling factors (Eq. 35-36).  Integer tables come
// from closed-form combinatorial ranks, not from searching an enumeration.
// Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace heom {

constexpr double kHbar = 5308.8;      // cm^-1 fs (BASELINE.json config 1)
constexpr double kBoltz = 0.6950348;  // cm^-1 / K (R3)

struct Hierarchy {
  int N = 0, K = 0, M = 0, W = 0, D = 0;
  int64_t nodes = 0;
  // PINNED order (R1)
  std::vector<uint8_t> tuples;  // [nodes][W]
  std::vector<int32_t> plus;    // [nodes][W], -1 invalid
  std::vector<int32_t> minus;   // [nodes][W], -1 invalid
  // storage slot of pinned node u in the chosen device order, and its inverse
  std::vector<int32_t> slot_of;  // [nodes]
  std::vector<int32_t> node_at;  // [nodes]
};

struct Coefficients {
  double beta_hbar = 0;            // fs
  std::vector<double> gamma;       // [W]   Eq. 19
  std::vector<double> c_re, c_im;  // [W]   Eq. 20 / V^o part of Eq. 17, divided by hbar (R2)
  std::vector<double> delta;       // [N]   Eq. 14 bracket
  // coupling factors for occupation n = 0..D (Eq. 35-36 in the division-free form, R5)
  std::vector<double> a_plus;      // [W][D+1]  sqrt((n+1) s_l)
  std::vector<double> a_minus_x;   // [W][D+1]  sgn(Re c_l) sqrt(n s_l)
  std::vector<double> a_minus_o;   // [W][D+1]  delta_{k0} sqrt(n/s_l) (lambda_b/hbar) nu_b
};

// order: 0 = pinned, 1 = plain lexicographic on (n_0..n_{W-1}), n_0 slowest.
// Returns false (err filled) on overflow / invalid sizes.
bool build_hierarchy(int N, int K, int D, int order, Hierarchy& h, std::string& err);

// Returns false on a singular coefficient (cot pole, gamma_k == nu_b) or bad input.
// pade = 0: Matsubara poles (Eq. 19-20); pade = 1: Pade poles (Eq. 27-33, R11).
bool build_coefficients(int N, int K, int D, const double* lambda_cm, const double* nu_per_fs,
                        double T_kelvin, int pade, Coefficients& c, std::string& err);

// Poles xi_j (increasing) and weights eta_j, j = 1..K, of the [K-1/K] Pade decomposition of the Bose function
// (Eq. 27-31): eigenvalues of the two symmetric tridiagonal matrices by Sturm-sequence bisection.
void pade_poles(int K, std::vector<double>& xi, std::vector<double>& eta);

}  // namespace heom
