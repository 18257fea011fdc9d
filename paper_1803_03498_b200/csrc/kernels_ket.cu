// kernels_ket.cu -- column-sparse states: the HEOM right-hand side on one COLUMN of every sigma_u.
//
// Linear absorption (Eq. 56) propagates sigma_0(0) = mu_p |0><0|.  With the ground state |0>
// uncoupled in H (Eq. 48: H[0][m] = 0 for m != 0) and without a bath, every term of Eq. 12-17 maps column c
// of sigma_u to column c and leaves the other columns zero:
//   (H sigma)[i][c]      = sum_m H[i][m] sigma[m][c]
//   (sigma H)[i][c]      = sigma[i][c] H[c][c]                       (row c of H is diagonal)
//   Eq. 13-14            = -(d_u + (1 - delta_ic)(Delta_i + Delta_c)) sigma[i][c]
//   Eq. 15-17, row part  = V_b acts on row b = i through the bath of state i
//   Eq. 15-17, col part  = V_b acts on column b = c: state c has no bath -> absent
// so the state is one N-vector v_u = sigma_u[:, c] per node: N times less memory and traffic than the matrix
// kernels, and (for the paper's FMO sizes) a state that stays resident in the 126 MB L2.  api.cu selects this
// kernel in heom_set_state only after checking those conditions exactly; everything host-visible (heom_rhs,
// heom_get_full_state, heom_populations, heom_expectation) still speaks full matrices.
//
// Mapping: LP = 2, 4, 8 or 16 lanes per node (a power of two >= N), 32/LP nodes per warp; lane i holds v_u[i], the
// commutator H v is N warp shuffles + FMAs with row i of H/hbar from shared memory, lane i gathers the 2M
// neighbour elements of its own bath (16-byte loads, L2-resident), and the Horner-form RK4 epilogue (DESIGN.md
// R6) is fused: out_x = y + ax k (y may alias x, out_x may alias y).  The meta rows are the pipelined kernel's
// (hpipe_pack_links): neighbour offsets are slot*N*N, so the ket offset is off/N.
#include "kernels.cuh"

namespace heom {
namespace {

constexpr int kKetMaxModes = 64;
constexpr int kKetMaxSqrt = 64;
constexpr int kKetThreads = 256;

template <int N>
struct KetParams {
  const double2* x;        // [nodes][N] stage input (gathered)
  const double2* y;        // [nodes][N] step-start state (may alias x)
  double2* out_x;          // y + ax * k
  double2* out_acc;        // k itself when rhs_only
  const int32_t* links;    // hpipe meta rows [nodes][lrow]
  int lrow, nodes, M, col, rhs_only;
  double ax;
  double hcc;              // H[c][c] / hbar
  double H[N * N];         // H / hbar
  double tdamp[N];         // (1 - delta_ic)(Delta_i + Delta_c)      Eq. 14 with Eq. 24
  double cP[kKetMaxModes], cX[kKetMaxModes], cO[kKetMaxModes];   // as in kernels_hpipe.cu
};

template <int N>
__global__ void __launch_bounds__(kKetThreads) rhs_ket_kernel(const __grid_constant__ KetParams<N> P) {
  constexpr int LP = (N <= 2) ? 2 : (N <= 4) ? 4 : (N <= 8) ? 8 : 16;
  constexpr int G = 32 / LP;
  constexpr int NP4 = (N + 3) / 4 * 4, NB8 = (N + 7) / 8 * 8, GROUP = (2 * NP4 + NB8 / 2 + 3) / 4 * 4;
  __shared__ double sH[N * N];
  __shared__ double sCoef[3 * kKetMaxModes];
  __shared__ double2 sSQ[2 * kKetMaxSqrt];          // [2 n + up] = (sqrt(n), up ? sqrt(n+1) : 0)
  for (int e = threadIdx.x; e < N * N; e += blockDim.x) sH[e] = P.H[e];
  for (int e = threadIdx.x; e < kKetMaxModes; e += blockDim.x) {
    sCoef[e] = P.cP[e]; sCoef[kKetMaxModes + e] = P.cX[e]; sCoef[2 * kKetMaxModes + e] = P.cO[e];
  }
  for (int e = threadIdx.x; e < 2 * kKetMaxSqrt; e += blockDim.x)
    sSQ[e] = make_double2(sqrt((double)(e >> 1)), (e & 1) ? sqrt((double)((e >> 1) + 1)) : 0.0);
  __syncthreads();

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int i = lane % LP, g = lane / LP;
  const bool lane_used = i < N;
  const int ii = lane_used ? i : 0;
  const int M = P.M;
  const int wpb = blockDim.x >> 5;
  const int npass = (P.nodes + G - 1) / G;
  for (int q = blockIdx.x * wpb + warp; q < npass; q += gridDim.x * wpb) {
    const int u = q * G + g;
    const bool active = lane_used && u < P.nodes;
    const size_t e = (size_t)(active ? u : 0) * N + ii;
    double2 v = make_double2(0.0, 0.0);
    if (active) v = P.x[e];
    const int32_t* lk = P.links + (size_t)(active ? u : 0) * P.lrow;

    // ---- couplings of the lane's own bath: element i of v_{u +- e_l}, l = i*M + kk (Eq. 15-17 / 35-36) ----
    double kr = 0.0, ki = 0.0;
#pragma unroll 2
    for (int kk = 0; kk < M; ++kk) {
      const int32_t* grp = lk + kk * GROUP;
      int up = -1, dn = -1;
      unsigned rec = 0;
      if (active) {
        up = grp[ii]; dn = grp[NP4 + ii];
        rec = reinterpret_cast<const unsigned short*>(grp + 2 * NP4)[ii];
      }
      double2 wu = make_double2(0.0, 0.0), wd = make_double2(0.0, 0.0);
      if (up >= 0) wu = __ldg(P.x + (up / N + ii));
      if (dn >= 0) wd = __ldg(P.x + (dn / N + ii));
      const double2 sq = sSQ[rec >> 4];
      const int l = ii * M + kk;
      const double a = sq.y * sCoef[l], ax = sq.x * sCoef[kKetMaxModes + l], ao = sq.x * sCoef[2 * kKetMaxModes + l];
      kr = fma(-a, wu.y, kr); ki = fma(a, wu.x, ki);                        // i a+ v^+
      kr = fma(-ax, wd.y, kr); ki = fma(ax, wd.x, ki);                      // i a-x v^-
      kr = fma(ao, wd.x, kr); ki = fma(ao, wd.y, ki);                       // a-o v^-   (zero for k != 0)
    }

    // ---- -(i/hbar)(H v - v H_cc) - (d_u + T_ic) v   (Eq. 12-14) ----
    double cr = -P.hcc * v.x, ci = -P.hcc * v.y;
#pragma unroll
    for (int m = 0; m < N; ++m) {
      const double vr = __shfl_sync(0xffffffffu, v.x, m, LP), vi = __shfl_sync(0xffffffffu, v.y, m, LP);
      const double h = sH[ii * N + m];
      cr = fma(h, vr, cr); ci = fma(h, vi, ci);
    }
    if (!active) continue;
    const double dmp = *reinterpret_cast<const double*>(lk + M * GROUP);   // d_u (Eq. 13)
    const double hd = -(dmp + (ii == P.col ? 0.0 : P.tdamp[ii]));
    kr += fma(hd, v.x, ci);                                                  // -i (cr + i ci) = ci - i cr
    ki += fma(hd, v.y, -cr);

    // ---- fused Horner-form RK4 epilogue (R6): w' = y + ax k ----
    if (P.rhs_only) {
      P.out_acc[e] = make_double2(kr, ki);
    } else {
      const double2 yv = (P.y == P.x) ? v : P.y[e];
      P.out_x[e] = make_double2(fma(P.ax, kr, yv.x), fma(P.ax, ki, yv.y));
    }
  }
}

// dst[slot][i][j] = (j == col) ? ket[slot][i] : 0
__global__ void ket_expand_kernel(const double2* __restrict__ ket, double2* __restrict__ dst, long long total,
                                  int N, int col) {
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(t % N);
    dst[t] = (j == col) ? ket[t / N] : make_double2(0.0, 0.0);
  }
}

template <int N>
cudaError_t launch_ket_t(const RhsParams& p, const int32_t* links, int lrow, int col, const double* a_plus,
                         const double* a_minus_x, const double* a_minus_o, const double* H_host,
                         const double* delta_host, int sms, cudaStream_t s) {
  KetParams<N> P;
  P.x = p.x; P.y = p.y; P.out_x = p.out_x; P.out_acc = p.out_acc;
  P.links = links; P.lrow = lrow; P.nodes = p.nodes; P.M = p.M; P.col = col; P.rhs_only = p.rhs_only;
  P.ax = p.ax;
  P.hcc = H_host[col * N + col] * p.inv_hbar;
  for (int e = 0; e < N * N; ++e) P.H[e] = H_host[e] * p.inv_hbar;
  for (int e = 0; e < N; ++e) P.tdamp[e] = (e == col) ? 0.0 : delta_host[e] + delta_host[col];
  const int D1 = p.D + 1;
  for (int l = 0; l < kKetMaxModes; ++l) {
    const bool on = l < p.W && p.D >= 1;
    P.cP[l] = on ? a_plus[(size_t)l * D1] : 0.0;
    P.cX[l] = on ? a_minus_x[(size_t)l * D1 + 1] : 0.0;
    P.cO[l] = on ? a_minus_o[(size_t)l * D1 + 1] : 0.0;
  }
  constexpr int LP = (N <= 2) ? 2 : (N <= 4) ? 4 : (N <= 8) ? 8 : 16;
  const int per_block = (kKetThreads / 32) * (32 / LP);
  int grid = (p.nodes + per_block - 1) / per_block;
  if (grid > sms * 8) grid = sms * 8;      // 8 CTAs of 256 threads per SM, grid-stride beyond that
  if (grid < 1) grid = 1;
  rhs_ket_kernel<N><<<grid, kKetThreads, 0, s>>>(P);
  return cudaGetLastError();
}

}  // namespace

#define HEOM_KET_ALL(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

bool ket_supported(int N, int W, int D) {
  return N >= 2 && N <= 16 && W <= kKetMaxModes && D + 2 <= kKetMaxSqrt;
}

cudaError_t launch_rhs_ket(const RhsParams& p, const int32_t* links, int lrow, int col, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, const double* H_host,
                           const double* delta_host, int sms, cudaStream_t s) {
  switch (p.N) {
#define HEOM_KET_CASE(n) \
  case n: return launch_ket_t<n>(p, links, lrow, col, a_plus, a_minus_x, a_minus_o, H_host, delta_host, sms, s);
    HEOM_KET_ALL(HEOM_KET_CASE)
#undef HEOM_KET_CASE
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t launch_ket_expand(const double2* ket, double2* dst, long long nodes, int N, int col, cudaStream_t s) {
  const long long total = nodes * N * N;
  long long blocks = (total + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (blocks < 1) blocks = 1;
  ket_expand_kernel<<<(int)blocks, 256, 0, s>>>(ket, dst, total, N, col);
  return cudaGetLastError();
}

}  // namespace heom
