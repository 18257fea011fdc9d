// hierarchy.cpp -- see hierarchy.hpp.  Host only, integer + a little fp64.
#include "hierarchy.hpp"

#include <algorithm>
#include <cmath>
#include <limits>
#include <utility>

namespace heom {
namespace {

// Pascal triangle choose(a, b) for a <= amax, b <= bmax, saturating at INT64_MAX.
struct Binomials {
  int amax, bmax;
  std::vector<int64_t> v;
  Binomials(int amax_, int bmax_) : amax(amax_), bmax(bmax_), v((size_t)(amax_ + 1) * (bmax_ + 1), 0) {
    const int64_t SAT = std::numeric_limits<int64_t>::max();
    for (int a = 0; a <= amax; ++a) {
      at(a, 0) = 1;
      for (int b = 1; b <= bmax && b <= a; ++b) {
        const int64_t x = at(a - 1, b - 1), y = (b <= a - 1) ? at(a - 1, b) : 0;
        at(a, b) = (x > SAT - y) ? SAT : x + y;
      }
    }
  }
  int64_t& at(int a, int b) { return v[(size_t)a * (bmax + 1) + b]; }
  // C(a, b) with b possibly > a or negative a
  int64_t operator()(int a, int b) const {
    if (a < 0 || b < 0 || b > a) return 0;
    return v[(size_t)a * (bmax + 1) + b];
  }
};

// Rank of tuple n (level L) in the pinned order:
//   u = C(L-1+W, W) + sum_{l=0}^{W-2} C(t_{l+1} - 1 + m_l, m_l),  m_l = W-l-1,
//   t_{l+1} = sum_{l' > l} n_{l'};  C(x-1+m, m) evaluated as C(x-1+m, x-1), x <= D.
inline int64_t pinned_rank(const uint8_t* n, int W, int L, const Binomials& C) {
  int64_t u = (L >= 1) ? C(L - 1 + W, L - 1) : 0;
  int t = L;  // suffix sum starting at l
  for (int l = 0; l + 1 < W; ++l) {
    t -= n[l];  // now t = t_{l+1}
    if (t == 0) break;
    u += C(t - 1 + (W - l - 1), t - 1);
  }
  return u;
}

// Rank in plain ascending lexicographic order over all tuples with sum <= D:
//   slot = sum_l sum_{v < n_l} C(R_l - v + m_l, m_l),  R_l = D - sum_{l'<l} n_{l'}.
inline int64_t lex_rank(const uint8_t* n, int W, int D, const Binomials& C) {
  int64_t s = 0;
  int R = D;
  for (int l = 0; l < W; ++l) {
    const int m = W - l - 1;
    for (int v = 0; v < n[l]; ++v) s += C(R - v + m, R - v);
    R -= n[l];
  }
  return s;
}

}  // namespace

bool build_hierarchy(int N, int K, int D, int order, Hierarchy& h, std::string& err) {
  if (N < 1 || K < 0 || D < 0 || D > 255) { err = "invalid N, K or D"; return false; }
  if (order != 0 && order != 1) { err = "unknown storage order"; return false; }
  const int M = K + 1;
  if ((int64_t)N * M > 100000) { err = "tuple length too large"; return false; }
  const int W = N * M;
  Binomials C(W + D + 1, D + 1);
  const int64_t nodes = C(W + D, D);
  if (nodes <= 0 || nodes > 2147483647LL) { err = "hierarchy has more than 2^31-1 nodes"; return false; }
  h.N = N; h.K = K; h.M = M; h.W = W; h.D = D; h.nodes = nodes;
  try {
    h.tuples.assign((size_t)nodes * W, 0);
    h.plus.assign((size_t)nodes * W, -1);
    h.minus.assign((size_t)nodes * W, -1);
    h.slot_of.assign((size_t)nodes, 0);
    h.node_at.assign((size_t)nodes, 0);
  } catch (const std::bad_alloc&) { err = "out of host memory for the hierarchy tables"; return false; }

  // Enumerate in the pinned order with the descending-lexicographic successor:
  // rightmost p < W-1 with n_p > 0: n_p -= 1, n_{p+1} = n_{W-1} + 1, n_{W-1} = 0 (if p+1 != W-1).
  {
    std::vector<uint8_t> n((size_t)W, 0);
    int64_t u = 0;
    for (int L = 0; L <= D; ++L) {
      for (int l = 0; l < W; ++l) n[l] = 0;
      n[0] = (uint8_t)L;
      for (;;) {
        uint8_t* dst = &h.tuples[(size_t)u * W];
        for (int l = 0; l < W; ++l) dst[l] = n[l];
        ++u;
        int p = W - 2;
        while (p >= 0 && n[p] == 0) --p;
        if (p < 0) break;
        const int r = n[W - 1];
        n[W - 1] = 0;
        n[p] -= 1;
        n[p + 1] = (uint8_t)(r + 1);
      }
    }
    if (u != nodes) { err = "internal error: enumeration count mismatch"; return false; }
  }

  // Links through the closed-form rank of n +- e_l (P:90 validity rules).
#pragma omp parallel
  {
    std::vector<uint8_t> n((size_t)W);
#pragma omp for schedule(static)
    for (int64_t u = 0; u < nodes; ++u) {
      int L = 0;
      for (int l = 0; l < W; ++l) { n[l] = h.tuples[(size_t)u * W + l]; L += n[l]; }
      for (int l = 0; l < W; ++l) {
        if (L < D) {
          n[l] += 1;
          h.plus[(size_t)u * W + l] = (int32_t)pinned_rank(n.data(), W, L + 1, C);
          n[l] -= 1;
        }
        if (n[l] > 0) {
          n[l] -= 1;
          h.minus[(size_t)u * W + l] = (int32_t)pinned_rank(n.data(), W, L - 1, C);
          n[l] += 1;
        }
      }
      h.slot_of[(size_t)u] = (order == 0) ? (int32_t)u : (int32_t)lex_rank(n.data(), W, D, C);
    }
  }
  for (int64_t u = 0; u < nodes; ++u) h.node_at[(size_t)h.slot_of[(size_t)u]] = (int32_t)u;
  return true;
}

bool restrict_hierarchy(Hierarchy& h, int rank, int world, const std::vector<int>& state_of_bath, Partition& part,
                        std::string& err) {
  if (world < 1 || rank < 0 || rank >= world) { err = "invalid rank/world"; return false; }
  const int64_t nodes = h.nodes;
  const int W = h.W;
  if (world > nodes) { err = "more ranks than nodes"; return false; }
  std::vector<int64_t> lo((size_t)world + 1);
  for (int r = 0; r <= world; ++r) lo[(size_t)r] = nodes * r / world;
  auto owner_of = [&](int64_t slot) {
    int a = 0, b = world;                       // largest r with lo[r] <= slot
    while (b - a > 1) { const int m = (a + b) / 2; if (lo[(size_t)m] <= slot) a = m; else b = m; }
    return a;
  };
  const int64_t s0 = lo[(size_t)rank], s1 = lo[(size_t)rank + 1], n_owned = s1 - s0;
  // ghosts (by global slot) and, by the symmetry of the link graph (u -> a by +e_l iff a -> u by -e_l), the owned
  // nodes every peer needs: those with a neighbour in the peer's range
  std::vector<uint8_t> is_ghost((size_t)nodes, 0);
  std::vector<std::vector<int32_t>> send((size_t)world);
  // slice halo pairs as (peer, global slot, state) keys: what I receive (ghost t read through a bath on state st)
  // and what I send (my node s read by a node of peer p through a bath on state st; link symmetry)
  struct PairKey { int peer; int64_t slot; int state; };
  std::vector<PairKey> rpairs, spairs;
  for (int64_t s = s0; s < s1; ++s) {
    const int64_t u = h.node_at[(size_t)s];
    int last_peer = -1;
    std::vector<int> peers;
    for (int l = 0; l < W; ++l)
      for (int dir = 0; dir < 2; ++dir) {
        const int32_t v = dir ? h.minus[(size_t)u * W + l] : h.plus[(size_t)u * W + l];
        if (v < 0) continue;
        const int64_t t = h.slot_of[(size_t)v];
        if (t >= s0 && t < s1) continue;
        is_ghost[(size_t)t] = 1;
        const int p = owner_of(t);
        const int st = state_of_bath[(size_t)(l / h.M)];
        rpairs.push_back({p, t, st});
        spairs.push_back({p, s, st});
        if (p != last_peer) {
          bool seen = false;
          for (int q : peers) seen = seen || q == p;
          if (!seen) peers.push_back(p);
          last_peer = p;
        }
      }
    for (int p : peers) send[(size_t)p].push_back((int32_t)(s - s0));
  }
  std::vector<int64_t> ghost_slots;
  for (int64_t t = 0; t < nodes; ++t) if (is_ghost[(size_t)t]) ghost_slots.push_back(t);
  const int64_t n_ghost = (int64_t)ghost_slots.size(), n_local = n_owned + n_ghost;
  if (n_local > 2147483647LL) { err = "partition too large"; return false; }
  std::vector<int32_t> local_of((size_t)nodes, -1);     // global slot -> local index
  for (int64_t s = s0; s < s1; ++s) local_of[(size_t)s] = (int32_t)(s - s0);
  for (int64_t q = 0; q < n_ghost; ++q) local_of[(size_t)ghost_slots[(size_t)q]] = (int32_t)(n_owned + q);

  part.rank = rank; part.world = world; part.n_owned = n_owned; part.n_ghost = n_ghost;
  part.global_id.assign((size_t)n_local, 0);
  part.send_counts.assign((size_t)world, 0); part.recv_counts.assign((size_t)world, 0);
  part.send_idx.clear();
  for (int p = 0; p < world; ++p) {
    part.send_counts[(size_t)p] = (int64_t)send[(size_t)p].size();
    part.send_idx.insert(part.send_idx.end(), send[(size_t)p].begin(), send[(size_t)p].end());
  }
  for (int64_t q = 0; q < n_ghost; ++q) part.recv_counts[(size_t)owner_of(ghost_slots[(size_t)q])] += 1;

  Hierarchy loc;
  loc.N = h.N; loc.K = h.K; loc.M = h.M; loc.W = W; loc.D = h.D; loc.nodes = n_local;
  loc.tuples.assign((size_t)n_local * W, 0);
  loc.plus.assign((size_t)n_local * W, -1);
  loc.minus.assign((size_t)n_local * W, -1);
  loc.slot_of.resize((size_t)n_local); loc.node_at.resize((size_t)n_local);
  for (int64_t i = 0; i < n_local; ++i) {
    const int64_t slot = i < n_owned ? s0 + i : ghost_slots[(size_t)(i - n_owned)];
    const int64_t u = h.node_at[(size_t)slot];
    part.global_id[(size_t)i] = u;
    loc.slot_of[(size_t)i] = (int32_t)i; loc.node_at[(size_t)i] = (int32_t)i;
    for (int l = 0; l < W; ++l) {
      loc.tuples[(size_t)i * W + l] = h.tuples[(size_t)u * W + l];
      if (i >= n_owned) continue;                   // ghost rows: copies only, no links
      const int32_t a = h.plus[(size_t)u * W + l], b = h.minus[(size_t)u * W + l];
      loc.plus[(size_t)i * W + l] = a < 0 ? -1 : local_of[(size_t)h.slot_of[(size_t)a]];
      loc.minus[(size_t)i * W + l] = b < 0 ? -1 : local_of[(size_t)h.slot_of[(size_t)b]];
    }
  }
  part.root = local_of[(size_t)h.slot_of[0]];
  auto finish = [&](std::vector<PairKey>& v, std::vector<int64_t>& counts, std::vector<int32_t>& node,
                    std::vector<int32_t>& state) {
    std::sort(v.begin(), v.end(), [](const PairKey& a, const PairKey& b) {
      return a.peer != b.peer ? a.peer < b.peer : (a.slot != b.slot ? a.slot < b.slot : a.state < b.state);
    });
    v.erase(std::unique(v.begin(), v.end(), [](const PairKey& a, const PairKey& b) {
              return a.peer == b.peer && a.slot == b.slot && a.state == b.state; }), v.end());
    counts.assign((size_t)world, 0);
    node.clear(); state.clear();
    for (const PairKey& k : v) {
      counts[(size_t)k.peer] += 1;
      node.push_back(local_of[(size_t)k.slot]);
      state.push_back(k.state);
    }
  };
  finish(spairs, part.send_pair_counts, part.send_pair_node, part.send_pair_state);
  finish(rpairs, part.recv_pair_counts, part.recv_pair_node, part.recv_pair_state);
  h = std::move(loc);
  return true;
}

namespace {

// The K largest eigenvalues (decreasing) of the symmetric tridiagonal matrix with zero diagonal and
// off-diagonal entries off[0..n-2], by bisection on the Sturm count (eigenvalues below x).
std::vector<double> largest_eigenvalues(const std::vector<double>& off, int n, int count) {
  auto below = [&](double x) {            // number of eigenvalues < x
    int neg = 0;
    double d = 1.0;
    for (int i = 0; i < n; ++i) {
      const double b2 = (i == 0) ? 0.0 : off[(size_t)i - 1] * off[(size_t)i - 1];
      d = -x - (i == 0 ? 0.0 : b2 / d);
      if (d == 0.0) d = -1e-300;
      if (d < 0.0) ++neg;
    }
    return neg;
  };
  double bound = 0.0;                      // Gershgorin
  for (int i = 0; i < n; ++i) {
    const double r = (i > 0 ? std::fabs(off[(size_t)i - 1]) : 0.0) + (i + 1 < n ? std::fabs(off[(size_t)i]) : 0.0);
    if (r > bound) bound = r;
  }
  std::vector<double> ev((size_t)count);
  for (int k = 0; k < count; ++k) {        // k-th largest: n - k - 1 eigenvalues lie below it
    double lo = 0.0, hi = bound;
    for (int iter = 0; iter < 200; ++iter) {
      const double mid = 0.5 * (lo + hi);
      if (mid == lo || mid == hi) break;
      if (below(mid) <= n - k - 1) lo = mid; else hi = mid;
    }
    ev[(size_t)k] = 0.5 * (lo + hi);
  }
  return ev;
}

}  // namespace

void pade_poles(int K, std::vector<double>& xi, std::vector<double>& eta) {
  xi.assign((size_t)K, 0.0); eta.assign((size_t)K, 0.0);
  if (K <= 0) return;
  auto offdiag = [](int size, int shift) {  // (m, m+1) entry, m = 1..size-1: 1/sqrt((2m+shift)(2m+2+shift))
    std::vector<double> o((size_t)(size > 1 ? size - 1 : 0));
    for (int m = 1; m < size; ++m) o[(size_t)m - 1] = 1.0 / std::sqrt((2.0 * m + shift) * (2.0 * m + 2.0 + shift));
    return o;
  };
  const std::vector<double> ev = largest_eigenvalues(offdiag(2 * K, 1), 2 * K, K);           // Eq. 27, 30
  for (int j = 0; j < K; ++j) xi[(size_t)j] = 2.0 / ev[(size_t)j];
  std::vector<double> zeta;
  if (K > 1) {
    const std::vector<double> evp = largest_eigenvalues(offdiag(2 * K - 1, 3), 2 * K - 1, K - 1);   // Eq. 28, 31
    for (int j = 0; j < K - 1; ++j) zeta.push_back(2.0 / evp[(size_t)j]);
  }
  for (int j = 0; j < K; ++j) {                                                                  // Eq. 29 (R11)
    double num = 1.0, den = 1.0;
    for (double z : zeta) num *= z * z - xi[(size_t)j] * xi[(size_t)j];
    for (int k = 0; k < K; ++k) if (k != j) den *= xi[(size_t)k] * xi[(size_t)k] - xi[(size_t)j] * xi[(size_t)j];
    eta[(size_t)j] = ((double)K * K + 1.5 * K) * num / den;
  }
}

bool build_coefficients(int N, int K, int D, const double* lambda_cm, const double* nu_per_fs,
                        double T_kelvin, int pade, Coefficients& c, std::string& err) {
  if (!(T_kelvin > 0.0) || !std::isfinite(T_kelvin)) { err = "T_kelvin must be > 0"; return false; }
  const int M = K + 1, W = N * M;
  const double two_pi = 6.283185307179586476925286766559;
  c.beta_hbar = kHbar / (kBoltz * T_kelvin);
  c.gamma.assign(W, 0.0); c.c_re.assign(W, 0.0); c.c_im.assign(W, 0.0); c.delta.assign(N, 0.0);
  c.a_plus.assign((size_t)W * (D + 1), 0.0);
  c.a_minus_x.assign((size_t)W * (D + 1), 0.0);
  c.a_minus_o.assign((size_t)W * (D + 1), 0.0);
  std::vector<double> pxi, peta;
  if (pade) pade_poles(K, pxi, peta);
  for (int b = 0; b < N; ++b) {
    const double lam = lambda_cm[b], nu = nu_per_fs[b];
    if (!(lam >= 0.0) || !std::isfinite(lam)) { err = "lambda_cm must be >= 0"; return false; }
    if (!(nu > 0.0) || !std::isfinite(nu)) { err = "nu_per_fs must be > 0"; return false; }
    const double lh = lam / kHbar;  // lambda_b / hbar
    double series = 0.0;            // sum_k Re c(b,k) / gamma(b,k)
    for (int k = 0; k < M; ++k) {
      const int l = b * M + k;
      double g, cre, cim = 0.0;
      if (k == 0) {
        g = nu;
        if (!pade) {
          const double x = 0.5 * c.beta_hbar * nu;
          const double sn = std::sin(x), cs = std::cos(x);
          if (lh != 0.0 && sn == 0.0) { err = "cot(beta hbar nu/2) is singular"; return false; }
          cre = (lh == 0.0) ? 0.0 : lh * nu * (cs / sn);
        } else {                            // Eq. 33, k = 0
          double sum = 0.0;
          for (int q = 0; q < K; ++q) {
            const double gq = pxi[(size_t)q] / c.beta_hbar, dq = gq * gq - nu * nu;
            if (lh != 0.0 && dq == 0.0) { err = "Pade pole equals the Drude rate"; return false; }
            sum += 2.0 * peta[(size_t)q] * nu * nu / dq;
          }
          cre = (lh == 0.0) ? 0.0 : 2.0 * lh / c.beta_hbar * (1.0 - sum);
        }
        cim = -lh * nu;
      } else {
        const double weight = pade ? peta[(size_t)k - 1] : 1.0;          // Eq. 33, k > 0 / Eq. 20
        g = pade ? pxi[(size_t)k - 1] / c.beta_hbar : two_pi * (double)k / c.beta_hbar;   // Eq. 32 / Eq. 19
        const double den = c.beta_hbar * (g * g - nu * nu);
        if (lh != 0.0 && den == 0.0) { err = "pole frequency equals the Drude rate"; return false; }
        cre = (lh == 0.0) ? 0.0 : 4.0 * lh * nu * weight * g / den;
      }
      if (!std::isfinite(cre)) { err = "non-finite coefficient"; return false; }
      c.gamma[l] = g; c.c_re[l] = cre; c.c_im[l] = cim;
      series += cre / g;
      const double s = std::fabs(cre);
      const double sgn = (cre > 0.0) ? 1.0 : ((cre < 0.0) ? -1.0 : 0.0);
      for (int n = 0; n <= D; ++n) {
        c.a_plus[(size_t)l * (D + 1) + n] = std::sqrt(((double)n + 1.0) * s);
        c.a_minus_x[(size_t)l * (D + 1) + n] = sgn * std::sqrt((double)n * s);
        c.a_minus_o[(size_t)l * (D + 1) + n] =
            (k == 0 && s > 0.0) ? std::sqrt((double)n / s) * (lh * nu) : 0.0;
      }
    }
    c.delta[b] = 2.0 * lh / (c.beta_hbar * nu) - series;
  }
  return true;
}

}  // namespace heom
