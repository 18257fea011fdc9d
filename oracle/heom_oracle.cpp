/*
 * heom_oracle.cpp -- plain, slow, obviously-correct CPU ORACLE of the HEOM
 * right-hand side (hierarchical Liouvillian) and the RK4 propagator of
 * arXiv 1803.03498 (DM-HEOM), written from the paper's equations.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (see heom_oracle.h).  No blocking, no
 * fusion, no table or code shared with the CUDA path.  Everything is fp64.
 *
 * "P:n" = line n of /root/reference/PAPER.md.  "R*" = a reading listed in
 * DESIGN.md section 3.
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   tables        : Eq. 9 closed form incl. the paper's printed 12 271 512
 *                    and the 3.3 GiB figure; link-count closed
 *                   form; minus[plus[u][l]][l]==u; brute force for small W, D.
 *   coefficients  : Mittag-Leffler series of cot (Delta_b -> 0+ as K -> inf).
 *   commutator,
 *   hbar, RK4     : lambda=0 -> closed-form two-level Rabi oscillation; dt^4.
 *   +/- couplings,
 *   V^x, V^o, c_0,
 *   terminator    : pure-dephasing closed form (line-shape function g(t));
 *                   trace and Hermiticity invariants; relaxation towards
 *                   Boltzmann populations; independence of sigma_0 from the
 *                   rescaling of Eq. 35-36; dense-Liouvillian expm comparison.
 *   bath -> state
 *   map           : two-level absorber cumulant closed form; lambda = 0 per-site
 *                   equivalence; Eq. 48 block structure (tests/test_oracle_sites.py).
 *   S(b) > 1, several baths per state, complex / time-dependent H
 *   (oracle_create_general, oracle_set_hamiltonian, oracle_rk4_step_td;
 *   tests/test_oracle_general.py): two-exciton coherences at J = 0 against the
 *   product of one-exciton line shapes; a bath shared by two states (the shared
 *   coupling cancels in their coherence; the printed and the operator form of the
 *   Eq. 14 sum, R12, differ by exactly exp(-2 Delta t) there); gauge transform
 *   H -> U H U^dagger with a diagonal unitary against the pinned real-H path;
 *   lambda = 0 against scipy expm; resonantly driven two-level system (RWA) against
 *   the rotating-frame Rabi formula.
 *   Parity unpinned: nothing in this file is without a pin, but configs 2-5 of
 *   BASELINE.json have no printed values anywhere (the paper prints none);
 *   they rest on the pins above evaluated at those shapes.
 */
#include "heom_oracle.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cplx;

/* BASELINE.json config 1 fixes hbar; k_B is reading R3. */
const double HBAR_CM_FS = 5308.8;      /* cm^-1 fs */
const double KB_CM_PER_K = 0.6950348;  /* cm^-1 / K */
const double PI = 3.14159265358979323846;

}  // namespace

struct oracle_ctx {
  int N = 0;       /* system states (rows of every sigma_u)                   */
  int B = 0;       /* baths; bath b couples through the projectors |s><s| on the
                      S(b) = bptr[b+1] - bptr[b] states bst[bptr[b]..] (P:84, P:119
                      Eq. 18, Eq. 21).  oracle_create: B = N, one state each,
                      bs(b) = b; oracle_create_sites: one state each, any injective
                      map (a ground state without a bath);
                      oracle_create_general: any lists ("multiple states can share
                      one bath, or multiple baths can couple to the same state",
                      P:84: the two-exciton manifold of Eq. 54)                */
  std::vector<int> bptr;        /* [B+1] offsets into bst                       */
  std::vector<int> bst;         /* states of every bath, bath after bath       */
  int terminator_form = 0;      /* Eq. 14's sum over s: 0 = as printed,
                                   sum_s V_s^x V_s^x; 1 = (sum_s V_s^x)^2 (R12)  */
  int K = 0;       /* Matsubara terms beyond the Drude pole                   */
  int M = 0;       /* modes per bath = K+1 = the paper's K             */
  int W = 0;       /* tuple length W = B*K_paper                        */
  int D = 0;       /* truncation depth                                        */
  int64_t nodes = 0;
  int scaling = 1;
  int terminator = 1;
  int threads = 0;
  int pade = 0;      /* 0 = Matsubara poles (Eq. 19-20), 1 = Pade poles (Eq. 27-33) */
  double T_kelvin = 0;
  std::vector<double> H;        /* [N][N] cm^-1, real part (symmetric)         */
  std::vector<double> Him;      /* [N][N] cm^-1, imaginary part (antisymmetric;
                                   zero unless oracle_create_general /
                                   oracle_set_hamiltonian gave one: RWA field
                                   coupling, Eq. 51)                            */
  std::vector<double> lambda;   /* [B] cm^-1                                  */
  std::vector<double> nu;       /* [B] fs^-1                                  */
  double beta_hbar = 0;         /* beta*hbar = hbar/(k_B T), fs               */
  std::vector<double> gamma;    /* [W] Eq. 19, fs^-1                          */
  std::vector<double> c_re;     /* [W] Re c(b,k)/hbar, Eq. 20, fs^-2          */
  std::vector<double> c_im;     /* [W] Im part carried by Eq. 17's V^o term   */
  std::vector<double> delta;    /* [B] Eq. 14 bracket, fs^-1                  */
  std::vector<uint8_t> tuples;  /* [nodes][W]                                 */
  std::vector<int32_t> plus;    /* [nodes][W]                                 */
  std::vector<int32_t> minus;   /* [nodes][W]                                 */
  std::vector<cplx> y;          /* state [nodes][N][N]                        */
  bool have_state = false;
};

namespace {

/* ---------------------------------------------------------------- index set
 * all tuples n in N^W with sum <= D.  The paper leaves the linear
 * numbering open; reading R1 pins it: level L = 0..D, and inside a
 * level  for n_0 = L..0: for n_1 = (L-n_0)..0: ... ; n_{W-1} = remainder.   */
void enumerate_level(int W, int pos, int remaining, std::vector<uint8_t>& cur,
                     std::vector<uint8_t>& out) {
  if (pos == W - 1) {
    cur[pos] = (uint8_t)remaining;
    out.insert(out.end(), cur.begin(), cur.end());
    return;
  }
  for (int v = remaining; v >= 0; --v) {
    cur[pos] = (uint8_t)v;
    enumerate_level(W, pos + 1, remaining - v, cur, out);
  }
}

int level_of(const uint8_t* t, int W) {
  int s = 0;
  for (int l = 0; l < W; ++l) s += t[l];
  return s;
}

/* Ordering predicate of the enumeration above: lower level first; inside a
 * level the tuple that is lexicographically LARGER comes first. */
bool comes_before(const uint8_t* a, const uint8_t* b, int W) {
  int la = level_of(a, W), lb = level_of(b, W);
  if (la != lb) return la < lb;
  for (int l = 0; l < W; ++l)
    if (a[l] != b[l]) return a[l] > b[l];
  return false;
}

/* Look a tuple up in the enumerated list by bisection (the list is sorted by
 * comes_before by construction).  Returns -1 if absent. */
int64_t find_tuple(const std::vector<uint8_t>& tuples, int64_t nodes, int W,
                   const uint8_t* key) {
  int64_t lo = 0, hi = nodes;
  while (lo < hi) {
    int64_t mid = lo + (hi - lo) / 2;
    if (comes_before(&tuples[(size_t)mid * W], key, W)) lo = mid + 1;
    else hi = mid;
  }
  if (lo < nodes && std::memcmp(&tuples[(size_t)lo * W], key, (size_t)W) == 0) return lo;
  return -1;
}

int nthreads(const oracle_ctx* c) {
#ifdef _OPENMP
  return c->threads > 0 ? c->threads : omp_get_max_threads();
#else
  (void)c;
  return 1;
#endif
}

/* "+" link valid iff sum(n + e_l) <= D; "-" link valid iff n_l - 1 >= 0. */
void build_links(oracle_ctx* c) {
  const int W = c->W;
  c->plus.assign((size_t)c->nodes * W, -1);
  c->minus.assign((size_t)c->nodes * W, -1);
#pragma omp parallel for schedule(static) num_threads(nthreads(c))
  for (int64_t u = 0; u < c->nodes; ++u) {
    std::vector<uint8_t> t(&c->tuples[(size_t)u * W], &c->tuples[(size_t)u * W] + W);
    const int L = level_of(t.data(), W);
    for (int l = 0; l < W; ++l) {
      if (L + 1 <= c->D) {
        t[l] += 1;
        c->plus[(size_t)u * W + l] = (int32_t)find_tuple(c->tuples, c->nodes, W, t.data());
        t[l] -= 1;
      }
      if (t[l] >= 1) {
        t[l] -= 1;
        c->minus[(size_t)u * W + l] = (int32_t)find_tuple(c->tuples, c->nodes, W, t.data());
        t[l] += 1;
      }
    }
  }
}

/* -------------------------------------------------------------- coefficients
 * P:121 Eq. 19, Eq. 20, Eq. 14 bracket.  Mode index (0-based)
 * l = b*M + k (Eq. 10 rewritten 0-based), k = 0 the Drude pole.
 * Reading R2: every c of Eq. 16-17 and 35-36 enters as c-hat = c/hbar so that
 * all terms of the RHS are rates.                                            */
/* ------------------------------------------------------- Pade decomposition
 * P:148-176 Eq. 27-33 ([K-1/K] Pade spectrum decomposition of the Bose function, the paper's ref. 31):
 *   1/(1 - exp(-x)) ~ 1/x + 1/2 + sum_{j=1..K} 2 eta_j x / (x^2 + xi_j^2).
 * xi_j = 2/eigenvalue_j(Lambda) for the K positive eigenvalues of the 2K x 2K matrix Eq. 27, zeta_j the same
 * for the (2K-1) x (2K-1) matrix Eq. 28 (K-1 positive eigenvalues), and Eq. 29 read as (R11: the
 * printed indices are garbled)
 *   eta_j = (K^2 + 3K/2) prod_{k=1..K-1} (zeta_k^2 - xi_j^2) / prod_{k != j} (xi_k^2 - xi_j^2).
 * Eigenvalues by the cyclic Jacobi rotation method on the dense symmetric matrix: slow, short, hard to get
 * wrong. */
std::vector<double> jacobi_eigenvalues(std::vector<double> a, int n) {
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0.0;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) off += a[(size_t)p * n + q] * a[(size_t)p * n + q];
    if (off < 1e-300) break;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = a[(size_t)p * n + q];
        if (apq == 0.0) continue;
        const double theta = (a[(size_t)q * n + q] - a[(size_t)p * n + p]) / (2.0 * apq);
        const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double cs = 1.0 / std::sqrt(t * t + 1.0), sn = t * cs;
        for (int k = 0; k < n; ++k) {   /* A <- A J */
          const double akp = a[(size_t)k * n + p], akq = a[(size_t)k * n + q];
          a[(size_t)k * n + p] = cs * akp - sn * akq;
          a[(size_t)k * n + q] = sn * akp + cs * akq;
        }
        for (int k = 0; k < n; ++k) {   /* A <- J^T A */
          const double apk = a[(size_t)p * n + k], aqk = a[(size_t)q * n + k];
          a[(size_t)p * n + k] = cs * apk - sn * aqk;
          a[(size_t)q * n + k] = sn * apk + cs * aqk;
        }
      }
  }
  std::vector<double> ev(n);
  for (int i = 0; i < n; ++i) ev[i] = a[(size_t)i * n + i];
  std::sort(ev.begin(), ev.end(), [](double x, double y) { return x > y; });   /* decreasing */
  return ev;
}

/* Eq. 27 (shift = 1) and Eq. 28 (shift = 3): (M)_{m,n} = delta_{m,n+-1} / sqrt((2m+shift)(2n+shift)), m,n = 1..size */
std::vector<double> pade_matrix(int size, int shift) {
  std::vector<double> a((size_t)size * size, 0.0);
  for (int m = 1; m <= size; ++m)
    for (int n = 1; n <= size; ++n)
      if (m == n - 1 || m == n + 1)
        a[(size_t)(m - 1) * size + (n - 1)] = 1.0 / std::sqrt((2.0 * m + shift) * (2.0 * n + shift));
  return a;
}

void pade_poles(int K, std::vector<double>& xi, std::vector<double>& eta) {
  xi.assign((size_t)K, 0.0); eta.assign((size_t)K, 0.0);
  if (K == 0) return;
  const std::vector<double> ev = jacobi_eigenvalues(pade_matrix(2 * K, 1), 2 * K);
  for (int i = 0; i < K; ++i) xi[i] = 2.0 / ev[i];                                   /* Eq. 30 */
  std::vector<double> zeta((size_t)(K > 1 ? K - 1 : 0));
  if (K > 1) {
    const std::vector<double> evp = jacobi_eigenvalues(pade_matrix(2 * K - 1, 3), 2 * K - 1);
    for (int i = 0; i < K - 1; ++i) zeta[i] = 2.0 / evp[i];                          /* Eq. 31 */
  }
  for (int j = 0; j < K; ++j) {                                                      /* Eq. 29 */
    double num = 1.0, den = 1.0;
    for (int k = 0; k < K - 1; ++k) num *= zeta[k] * zeta[k] - xi[j] * xi[j];
    for (int k = 0; k < K; ++k) if (k != j) den *= xi[k] * xi[k] - xi[j] * xi[j];
    eta[j] = ((double)K * K + 1.5 * K) * num / den;
  }
}

int build_coefficients(oracle_ctx* c, double T_kelvin) {
  const int N = c->B, M = c->M;   /* loop over baths */
  c->beta_hbar = HBAR_CM_FS / (KB_CM_PER_K * T_kelvin);
  c->gamma.assign((size_t)c->W, 0.0);
  c->c_re.assign((size_t)c->W, 0.0);
  c->c_im.assign((size_t)c->W, 0.0);
  c->delta.assign((size_t)N, 0.0);
  std::vector<double> pxi, peta;
  if (c->pade) pade_poles(M - 1, pxi, peta);
  for (int b = 0; b < N; ++b) {
    const double lam = c->lambda[b] / HBAR_CM_FS; /* lambda_b / hbar, fs^-1 */
    const double nu = c->nu[b];
    for (int k = 0; k < M; ++k) {
      const int l = b * M + k;
      if (k == 0) {
        c->gamma[l] = nu;                                           /* Eq. 19 */
        if (!c->pade) {
          const double x = c->beta_hbar * nu / 2.0;
          const double t = std::tan(x);
          if (lam != 0.0 && (t == 0.0 || !std::isfinite(1.0 / t))) return -1;
          c->c_re[l] = (lam == 0.0) ? 0.0 : nu * lam / t;           /* Eq. 20 */
        } else {
          /* Eq. 33, k = 0:  (2 lambda/(beta hbar)) (1 - sum_j 2 eta_j nu^2 / ((xi_j/(beta hbar))^2 - nu^2)) */
          double sum = 0.0;
          for (int jj = 0; jj < M - 1; ++jj) {
            const double gj = pxi[(size_t)jj] / c->beta_hbar;
            if (lam != 0.0 && gj * gj - nu * nu == 0.0) return -1;
            sum += 2.0 * peta[(size_t)jj] * nu * nu / (gj * gj - nu * nu);
          }
          c->c_re[l] = (lam == 0.0) ? 0.0 : 2.0 * lam / c->beta_hbar * (1.0 - sum);
        }
        c->c_im[l] = -lam * nu;           /* the V^o term of Eq. 17 (R4)     */
      } else if (!c->pade) {
        const double g = 2.0 * PI * k / c->beta_hbar;               /* Eq. 19 */
        c->gamma[l] = g;
        if (lam != 0.0 && g * g - nu * nu == 0.0) return -1;
        c->c_re[l] = (lam == 0.0) ? 0.0
                     : 4.0 * lam * nu / c->beta_hbar * g / (g * g - nu * nu); /* Eq. 20 */
      } else {
        const double g = pxi[(size_t)k - 1] / c->beta_hbar;          /* Eq. 32 */
        c->gamma[l] = g;
        if (lam != 0.0 && g * g - nu * nu == 0.0) return -1;
        c->c_re[l] = (lam == 0.0) ? 0.0
                     : 4.0 * lam * nu / c->beta_hbar * peta[(size_t)k - 1] * g / (g * g - nu * nu); /* Eq. 33, k > 0 */
      }
    }
    /* Eq. 14:  2 lambda_b/(beta hbar^2 nu_b) - sum_k c(b,k)/(hbar gamma(b,k)) */
    double d = 2.0 * lam / (c->beta_hbar * nu);
    for (int k = 0; k < M; ++k) d -= c->c_re[b * M + k] / c->gamma[b * M + k];
    c->delta[b] = d;
  }
  return 0;
}

/* ------------------------------------------------------- site superoperators
 * P:136-140 Eq. 23-25 (Eq. 23's printed left subscript "ii" read as "ij").   */
inline double Vx(int s, int i, int j) { return (double)(i == s) - (double)(s == j); }
inline double VxVx(int s, int i, int j) {
  return (double)(i != j) * ((double)(i == s) + (double)(s == j));
}
inline double Vo(int s, int i, int j) { return (double)(i == s) + (double)(s == j); }

/* |c(b,k)| of Eq. 35-36 under the chosen reading (R5). */
inline double abs_c(const oracle_ctx* c, int l) {
  if (c->scaling == 2) return std::sqrt(c->c_re[l] * c->c_re[l] + c->c_im[l] * c->c_im[l]);
  return std::fabs(c->c_re[l]);
}

/* ------------------------------------------------------------ right-hand side
 * d sigma_u / dt, Eq. 12-17, for one node u of the state `st`.  The sums over
 * the S(b) states of a bath are written out as the paper prints them.        */
void rhs_node(const oracle_ctx* c, const cplx* st, int64_t u, cplx* out) {
  const int N = c->N, M = c->M, W = c->W;
  const size_t NN = (size_t)N * N;
  const cplx I(0.0, 1.0);
  const cplx* s = st + (size_t)u * NN;
  const uint8_t* n = &c->tuples[(size_t)u * W];

  /* Eq. 12:  -(i/hbar) [H, sigma_u],  H = H_re + i H_im Hermitian */
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      cplx comm(0.0, 0.0);
      for (int m = 0; m < N; ++m)
        comm += cplx(c->H[(size_t)i * N + m], c->Him[(size_t)i * N + m]) * s[(size_t)m * N + j] -
                s[(size_t)i * N + m] * cplx(c->H[(size_t)m * N + j], c->Him[(size_t)m * N + j]);
      out[(size_t)i * N + j] = -(I / HBAR_CM_FS) * comm;
    }

  /* Eq. 13:  - sigma_u sum_{b,k} n_{u,(b,k)} gamma(b,k) */
  double damp = 0.0;
  for (int l = 0; l < W; ++l) damp += (double)n[l] * c->gamma[l];
  for (size_t e = 0; e < NN; ++e) out[e] -= damp * s[e];

  /* Eq. 14:  - sum_b sum_{s=1..S(b)} [ ... ] V_s^x V_s^x sigma_u  as printed (terminator_form 0), or with the
   * operator of the bath squared, (sum_s V_s^x)^2 (terminator_form 1, R12); the same thing when S(b) = 1 */
  if (c->terminator)
    for (int b = 0; b < c->B; ++b)
      for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
          double mask = 0.0;
          if (c->terminator_form == 0) {
            for (int q = c->bptr[b]; q < c->bptr[b + 1]; ++q) mask += VxVx(c->bst[q], i, j);
          } else {
            double v = 0.0;
            for (int q = c->bptr[b]; q < c->bptr[b + 1]; ++q) v += Vx(c->bst[q], i, j);
            mask = v * v;
          }
          out[(size_t)i * N + j] -= c->delta[b] * mask * s[(size_t)i * N + j];
        }

  /* Eq. 15 -> Eq. 35:  + sum_b sum_s sum_k i sqrt((n+1)|c|) V_s^x sigma^+_{(u,b,k)} */
  for (int l = 0; l < W; ++l) {
    const int32_t up = c->plus[(size_t)u * W + l];
    if (up < 0) continue; /* invalid link contributes nothing */
    const int b = l / M;  /* Eq. 11 */
    const cplx* sp = st + (size_t)up * NN;
    const double f = c->scaling ? std::sqrt(((double)n[l] + 1.0) * abs_c(c, l)) : 1.0;
    for (int q = c->bptr[b]; q < c->bptr[b + 1]; ++q)
      for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
          out[(size_t)i * N + j] += I * (f * Vx(c->bst[q], i, j)) * sp[(size_t)i * N + j];
  }

  /* Eq. 16-17 -> Eq. 36:  + sum_b sum_s sum_k sqrt(n/|c|) theta_MA(b,k) sigma^-_{(u,b,k)},
   * theta_MA = i c V_s^x + delta_{k,0} (lambda_b nu_b / hbar) V_s^o.
   * Unscaled (Eq. 16) the prefactor is n.  |c| = 0 (lambda_b = 0): the bath is
   * decoupled and the term is dropped (limit of the printed 0/0). */
  for (int l = 0; l < W; ++l) {
    const int32_t um = c->minus[(size_t)u * W + l];
    if (um < 0) continue;
    const int b = l / M, k = l % M;
    const cplx* sm = st + (size_t)um * NN;
    double f;
    if (c->scaling) {
      const double a = abs_c(c, l);
      f = (a > 0.0) ? std::sqrt((double)n[l] / a) : 0.0;
    } else {
      f = (double)n[l];
    }
    const double lam_nu = (k == 0) ? -c->c_im[l] : 0.0; /* lambda_b nu_b / hbar */
    for (int q = c->bptr[b]; q < c->bptr[b + 1]; ++q)
      for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
          const cplx theta = I * (c->c_re[l] * Vx(c->bst[q], i, j)) + lam_nu * Vo(c->bst[q], i, j);
          out[(size_t)i * N + j] += f * theta * sm[(size_t)i * N + j];
        }
  }
}

void rhs_all(const oracle_ctx* c, const cplx* st, cplx* out) {
  const size_t NN = (size_t)c->N * c->N;
#pragma omp parallel for schedule(static) num_threads(nthreads(c))
  for (int64_t u = 0; u < c->nodes; ++u) rhs_node(c, st, u, out + (size_t)u * NN);
}

}  // namespace

extern "C" {

int oracle_create_general(oracle_ctx** out, int n_states, const double* H_re_cm, const double* H_im_cm,
                          int n_baths, const int* bath_ptr, const int* bath_states, const double* lambda_cm,
                          const double* nu_per_fs, double T_kelvin, int K, int D) {
  if (!out || !H_re_cm || !lambda_cm || !nu_per_fs || !bath_ptr || !bath_states) return -1;
  if (n_states < 1 || n_baths < 1 || K < 0 || D < 0 || D > 255 || !(T_kelvin > 0.0)) return -1;
  if (bath_ptr[0] != 0) return -1;
  for (int b = 0; b < n_baths; ++b) {
    if (!(lambda_cm[b] >= 0.0) || !(nu_per_fs[b] > 0.0)) return -1;
    if (bath_ptr[b + 1] <= bath_ptr[b]) return -1;                       /* S(b) >= 1 */
    for (int q = bath_ptr[b]; q < bath_ptr[b + 1]; ++q) {
      if (bath_states[q] < 0 || bath_states[q] >= n_states) return -1;
      for (int q2 = bath_ptr[b]; q2 < q; ++q2) if (bath_states[q2] == bath_states[q]) return -1;   /* a state once per bath */
    }
  }
  for (int i = 0; i < n_states; ++i)
    for (int j = 0; j < n_states; ++j) {
      if (!std::isfinite(H_re_cm[i * n_states + j])) return -1;
      if (H_re_cm[i * n_states + j] != H_re_cm[j * n_states + i]) return -1;
      if (H_im_cm) {
        if (!std::isfinite(H_im_cm[i * n_states + j])) return -1;
        if (H_im_cm[i * n_states + j] != -H_im_cm[j * n_states + i]) return -1;   /* Hermitian */
      }
    }
  oracle_ctx* c = new (std::nothrow) oracle_ctx();
  if (!c) return -2;
  try {
    c->N = n_states; c->B = n_baths; c->K = K; c->M = K + 1; c->W = n_baths * (K + 1); c->D = D;
    c->bptr.assign(bath_ptr, bath_ptr + n_baths + 1);
    c->bst.assign(bath_states, bath_states + bath_ptr[n_baths]);
    c->H.assign(H_re_cm, H_re_cm + (size_t)n_states * n_states);
    c->Him.assign((size_t)n_states * n_states, 0.0);
    if (H_im_cm) c->Him.assign(H_im_cm, H_im_cm + (size_t)n_states * n_states);
    c->lambda.assign(lambda_cm, lambda_cm + n_baths);
    c->nu.assign(nu_per_fs, nu_per_fs + n_baths);
    c->T_kelvin = T_kelvin;
    if (build_coefficients(c, T_kelvin) != 0) { delete c; return -1; }
    std::vector<uint8_t> cur((size_t)c->W, 0);
    for (int L = 0; L <= D; ++L) enumerate_level(c->W, 0, L, cur, c->tuples);
    c->nodes = (int64_t)(c->tuples.size() / (size_t)c->W);
    if (c->nodes > 2147483647LL) { delete c; return -1; }
    build_links(c);
  } catch (const std::bad_alloc&) {
    delete c;
    return -2;
  }
  *out = c;
  return 0;
}

/* One state per bath, all different: the S(b) = 1 special case of oracle_create_general. */
int oracle_create_sites(oracle_ctx** out, int n_states, const double* H_cm, int n_baths,
                        const int* bath_state, const double* lambda_cm, const double* nu_per_fs,
                        double T_kelvin, int K, int D) {
  if (!bath_state || n_baths < 1 || n_baths > n_states) return -1;
  std::vector<int> ptr((size_t)n_baths + 1);
  for (int b = 0; b <= n_baths; ++b) ptr[(size_t)b] = b;
  for (int b = 0; b < n_baths; ++b)
    for (int b2 = 0; b2 < b; ++b2) if (bath_state[b2] == bath_state[b]) return -1;   /* one bath per state */
  return oracle_create_general(out, n_states, H_cm, nullptr, n_baths, ptr.data(), bath_state, lambda_cm,
                               nu_per_fs, T_kelvin, K, D);
}

/* Per-site baths: one bath per state, bath b on state b (BASELINE.json's five configurations). */
int oracle_create(oracle_ctx** out, int n_sites, const double* H_cm, const double* lambda_cm,
                  const double* nu_per_fs, double T_kelvin, int K, int D) {
  if (n_sites < 1) return -1;
  std::vector<int> ident((size_t)n_sites);
  for (int b = 0; b < n_sites; ++b) ident[(size_t)b] = b;
  return oracle_create_sites(out, n_sites, H_cm, n_sites, ident.data(), lambda_cm, nu_per_fs, T_kelvin, K, D);
}

void oracle_destroy(oracle_ctx* c) { delete c; }

int oracle_set_option(oracle_ctx* c, const char* name, int value) {
  if (!c || !name) return -1;
  const std::string s(name);
  if (s == "scaling") { if (value < 0 || value > 2) return -1; c->scaling = value; return 0; }
  if (s == "terminator") { c->terminator = value ? 1 : 0; return 0; }
  if (s == "terminator_form") { if (value < 0 || value > 1) return -1; c->terminator_form = value; return 0; }
  if (s == "threads") { if (value < 0) return -1; c->threads = value; return 0; }
  if (s == "pade") { c->pade = value ? 1 : 0; return build_coefficients(c, c->T_kelvin); }
  return -1;
}

int oracle_pade_poles(int K, double* xi, double* eta) {
  if (K < 0 || K > 64 || (K > 0 && (!xi || !eta))) return -1;
  std::vector<double> x, e;
  pade_poles(K, x, e);
  for (int i = 0; i < K; ++i) { xi[i] = x[(size_t)i]; eta[i] = e[(size_t)i]; }
  return 0;
}

int64_t oracle_num_nodes(const oracle_ctx* c) { return c ? c->nodes : -1; }
int oracle_num_modes(const oracle_ctx* c) { return c ? c->W : -1; }
int oracle_num_baths(const oracle_ctx* c) { return c ? c->B : -1; }
int oracle_num_threads(const oracle_ctx* c) { return c ? nthreads(c) : -1; }

int oracle_get_tables(const oracle_ctx* c, uint8_t* tuples, int32_t* plus, int32_t* minus) {
  if (!c) return -1;
  if (tuples) std::memcpy(tuples, c->tuples.data(), c->tuples.size());
  if (plus) std::memcpy(plus, c->plus.data(), c->plus.size() * sizeof(int32_t));
  if (minus) std::memcpy(minus, c->minus.data(), c->minus.size() * sizeof(int32_t));
  return 0;
}

int oracle_get_coefficients(const oracle_ctx* c, double* gamma, double* c_re, double* c_im,
                            double* delta) {
  if (!c) return -1;
  if (gamma) std::memcpy(gamma, c->gamma.data(), c->gamma.size() * sizeof(double));
  if (c_re) std::memcpy(c_re, c->c_re.data(), c->c_re.size() * sizeof(double));
  if (c_im) std::memcpy(c_im, c->c_im.data(), c->c_im.size() * sizeof(double));
  if (delta) std::memcpy(delta, c->delta.data(), c->delta.size() * sizeof(double));
  return 0;
}

int oracle_set_state(oracle_ctx* c, const double* sigma0) {
  if (!c || !sigma0) return -1;
  const size_t NN = (size_t)c->N * c->N;
  try { c->y.assign((size_t)c->nodes * NN, cplx(0.0, 0.0)); }
  catch (const std::bad_alloc&) { return -2; }
  for (size_t e = 0; e < NN; ++e) c->y[e] = cplx(sigma0[2 * e], sigma0[2 * e + 1]);
  c->have_state = true;
  return 0;
}

int oracle_set_full_state(oracle_ctx* c, const double* sigma) {
  if (!c || !sigma) return -1;
  const size_t total = (size_t)c->nodes * c->N * c->N;
  try { c->y.resize(total); } catch (const std::bad_alloc&) { return -2; }
  for (size_t e = 0; e < total; ++e) c->y[e] = cplx(sigma[2 * e], sigma[2 * e + 1]);
  c->have_state = true;
  return 0;
}

int oracle_get_full_state(const oracle_ctx* c, double* sigma) {
  if (!c || !sigma) return -1;
  if (!c->have_state) return -4;
  for (size_t e = 0; e < c->y.size(); ++e) { sigma[2 * e] = c->y[e].real(); sigma[2 * e + 1] = c->y[e].imag(); }
  return 0;
}

int oracle_rhs(oracle_ctx* c, double* dsigma) {
  if (!c || !dsigma) return -1;
  if (!c->have_state) return -4;
  rhs_all(c, c->y.data(), reinterpret_cast<cplx*>(dsigma));
  return 0;
}

int oracle_rhs_nodes(oracle_ctx* c, const int64_t* ids, int64_t count, double* out) {
  if (!c || !ids || !out || count < 0) return -1;
  if (!c->have_state) return -4;
  const size_t NN = (size_t)c->N * c->N;
  for (int64_t q = 0; q < count; ++q)
    if (ids[q] < 0 || ids[q] >= c->nodes) return -1;
#pragma omp parallel for schedule(static) num_threads(nthreads(c))
  for (int64_t q = 0; q < count; ++q)
    rhs_node(c, c->y.data(), ids[q], reinterpret_cast<cplx*>(out) + (size_t)q * NN);
  return 0;
}

/* Classical fourth-order Runge-Kutta ("Runge-Kutta integration", P:503
 * "4 intermediate results", "4 copies of the ADOs"; reading R6):
 *   k1 = f(y); k2 = f(y + dt/2 k1); k3 = f(y + dt/2 k2); k4 = f(y + dt k3);
 *   y <- y + dt/6 (k1 + 2 k2 + 2 k3 + k4).
 * Four state-sized arrays (y, stage input, k, running sum), like the paper. */
int oracle_rk4_steps(oracle_ctx* c, double dt, int nsteps) {
  if (!c || nsteps < 0 || !std::isfinite(dt)) return -1;
  if (!c->have_state) return -4;
  const size_t total = c->y.size();
  std::vector<cplx> x, k, sum;
  try { x.resize(total); k.resize(total); sum.resize(total); }
  catch (const std::bad_alloc&) { return -2; }
  cplx* y = c->y.data();
  const int nt = nthreads(c);
  for (int step = 0; step < nsteps; ++step) {
    rhs_all(c, y, k.data());                                   /* k1 */
#pragma omp parallel for schedule(static) num_threads(nt)
    for (size_t e = 0; e < total; ++e) { sum[e] = k[e]; x[e] = y[e] + (dt / 2.0) * k[e]; }
    rhs_all(c, x.data(), k.data());                            /* k2 */
#pragma omp parallel for schedule(static) num_threads(nt)
    for (size_t e = 0; e < total; ++e) { sum[e] += 2.0 * k[e]; x[e] = y[e] + (dt / 2.0) * k[e]; }
    rhs_all(c, x.data(), k.data());                            /* k3 */
#pragma omp parallel for schedule(static) num_threads(nt)
    for (size_t e = 0; e < total; ++e) { sum[e] += 2.0 * k[e]; x[e] = y[e] + dt * k[e]; }
    rhs_all(c, x.data(), k.data());                            /* k4 */
#pragma omp parallel for schedule(static) num_threads(nt)
    for (size_t e = 0; e < total; ++e) { sum[e] += k[e]; y[e] += (dt / 6.0) * sum[e]; }
  }
  return 0;
}

/* Replace the Hamiltonian (time-dependent H(t), Eq. 47-51: the caller evaluates the field). */
int oracle_set_hamiltonian(oracle_ctx* c, const double* H_re_cm, const double* H_im_cm) {
  if (!c || !H_re_cm) return -1;
  const int N = c->N;
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      if (!std::isfinite(H_re_cm[i * N + j]) || H_re_cm[i * N + j] != H_re_cm[j * N + i]) return -1;
      if (H_im_cm && (!std::isfinite(H_im_cm[i * N + j]) || H_im_cm[i * N + j] != -H_im_cm[j * N + i])) return -1;
    }
  c->H.assign(H_re_cm, H_re_cm + (size_t)N * N);
  c->Him.assign((size_t)N * N, 0.0);
  if (H_im_cm) c->Him.assign(H_im_cm, H_im_cm + (size_t)N * N);
  return 0;
}

/* One classical RK4 step of the NON-autonomous system d sigma/dt = L(H(t)) sigma:
 *   k1 = f(t, y); k2 = f(t + dt/2, y + dt/2 k1); k3 = f(t + dt/2, y + dt/2 k2); k4 = f(t + dt, y + dt k3),
 * with H(t), H(t + dt/2), H(t + dt) handed in (each as real and imaginary part; imaginary parts may be NULL).
 * Leaves H(t + dt) set. */
int oracle_rk4_step_td(oracle_ctx* c, double dt, const double* H0_re, const double* H0_im,
                       const double* Hm_re, const double* Hm_im, const double* H1_re, const double* H1_im) {
  if (!c || !std::isfinite(dt)) return -1;
  if (!c->have_state) return -4;
  const size_t total = c->y.size();
  std::vector<cplx> x, k, sum;
  try { x.resize(total); k.resize(total); sum.resize(total); }
  catch (const std::bad_alloc&) { return -2; }
  cplx* y = c->y.data();
  int rc;
  if ((rc = oracle_set_hamiltonian(c, H0_re, H0_im)) != 0) return rc;
  rhs_all(c, y, k.data());                                     /* k1 */
  for (size_t e = 0; e < total; ++e) { sum[e] = k[e]; x[e] = y[e] + (dt / 2.0) * k[e]; }
  if ((rc = oracle_set_hamiltonian(c, Hm_re, Hm_im)) != 0) return rc;
  rhs_all(c, x.data(), k.data());                              /* k2 */
  for (size_t e = 0; e < total; ++e) { sum[e] += 2.0 * k[e]; x[e] = y[e] + (dt / 2.0) * k[e]; }
  rhs_all(c, x.data(), k.data());                              /* k3 */
  for (size_t e = 0; e < total; ++e) { sum[e] += 2.0 * k[e]; x[e] = y[e] + dt * k[e]; }
  if ((rc = oracle_set_hamiltonian(c, H1_re, H1_im)) != 0) return rc;
  rhs_all(c, x.data(), k.data());                              /* k4 */
  for (size_t e = 0; e < total; ++e) { sum[e] += k[e]; y[e] += (dt / 6.0) * sum[e]; }
  return 0;
}

/* P:144 Eq. 26: rho = sigma_0. */
int oracle_populations(const oracle_ctx* c, double* pop, double* tr_re, double* tr_im) {
  if (!c) return -1;
  if (!c->have_state) return -4;
  cplx tr(0.0, 0.0);
  for (int i = 0; i < c->N; ++i) {
    const cplx d = c->y[(size_t)i * c->N + i];
    if (pop) pop[i] = d.real();
    tr += d;
  }
  if (tr_re) *tr_re = tr.real();
  if (tr_im) *tr_im = tr.imag();
  return 0;
}

}  // extern "C"
