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

// One rank's part of a hierarchy split over `world` ranks (the paper's partitions + halo regions,
// P:501): the rank owns a contiguous range of the lexicographic storage order; its ghosts are the neighbours of
// owned nodes that live elsewhere.  Local node order: owned nodes by global lexicographic slot, then ghosts by
// global slot (hence grouped by owning rank, in the order the owner sends them).
struct Partition {
  int rank = 0, world = 1;
  int64_t n_owned = 0, n_ghost = 0;
  std::vector<int64_t> global_id;    // [n_owned + n_ghost] pinned-order id of each local node
  std::vector<int64_t> send_counts;  // [world] owned nodes peer p needs
  std::vector<int64_t> recv_counts;  // [world] ghosts owned by peer p (contiguous in the ghost region)
  std::vector<int32_t> send_idx;     // [sum send_counts] local indices, grouped by peer, ascending
  int64_t root = -1;                 // local index of the hierarchy's root node (n = 0), -1 if not local
  // Slice halo: a gather reads of a ghost only row s (and, for states that are not Hermitian, column s) of the
  // states s = state of the bath through which the ghost is reached (Eq. 23, 25).  (node, state) pairs, unique,
  // sorted by (peer, global slot, state): the same order on the sending and on the receiving side.
  std::vector<int64_t> send_pair_counts, recv_pair_counts;   // [world]
  std::vector<int32_t> send_pair_node, send_pair_state;      // local OWNED index, state; grouped by peer
  std::vector<int32_t> recv_pair_node, recv_pair_state;      // local GHOST index (>= n_owned), state; grouped by peer
};

// Replaces `h` (a full hierarchy built with order = 1) by the rank's local hierarchy: tuples and link tables of the
// n_owned + n_ghost local nodes with local indices (ghost rows: every link invalid; they are never the result of
// a computation, only copies), slot_of = node_at = identity.
// state_of_bath: [B] state bath b couples to (tuple position l belongs to bath l / M).
bool restrict_hierarchy(Hierarchy& h, int rank, int world, const std::vector<int>& state_of_bath, Partition& part,
                        std::string& err);

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
