// kernels_rows.cu -- small-N (2 <= N <= 16) sm_100a kernel for the HEOM right-hand side with the
// RK4 stage combination fused into its epilogue.
//
// Mapping: one thread per matrix ROW.  A warp owns G = 32/N consecutive nodes; lane (g,i) keeps
// row i and column i of sigma_u in registers and forms
//     (sigma H)[i,:] = sum_m sigma[i,m] H[m,:]        (from its row)
//     (H sigma)[:,i] = sum_m H[:,m] sigma[m,i]        (from its column)
// with H read as warp-uniform constant-bank operands (H travels in the kernel parameters).  The
// column results are transposed through a warp-private shared-memory tile so that every lane ends
// with row i of the commutator (Eq. 12).  A CTA owns a tile of T consecutive storage slots whose
// sigma matrices are staged once in shared memory; the +/- couplings (Eq. 15-17 with the masks of
// Eq. 23-25) read a neighbour from that tile when it lies inside it and from global memory (L2)
// otherwise.  The "row part" of a coupling (bath b = i) reads the neighbour's row i (contiguous),
// the "column part" (every bath b) reads element [i][b]; both include the diagonal, where the
// V^x contributions cancel and the V^o contributions add up to 2 (Eq. 23, 25).
// The k rows go back to the warp-private tile and the warp streams the fused RK4 update
// (y, acc -> next stage input, acc) with fully coalesced 16-byte accesses.
#include "kernels.cuh"
#ifdef HEOM_DEBUG
#include <cassert>
#define DBG(c) assert(c)
#else
#define DBG(c) ((void)0)
#endif

namespace heom {
namespace {

constexpr int kWarps = 8;
constexpr int kThreadsRows = kWarps * 32;

template <int N>
struct RowCfg {
  static constexpr int NN = N * N;
  static constexpr int G = 32 / N;                    // nodes per warp pass
  static constexpr int T = (N <= 8) ? 64 : 32;        // nodes per CTA tile
  static constexpr int PASSES = (T + G * kWarps - 1) / (G * kWarps);
};

template <int N>
struct RowParams {
  RhsParams p;
  const int32_t* links;  // [nodes][lrow]: plus[W], minus[W], tuple bytes packed 4 per int32
  int lrow;              // int32 entries per links row (multiple of 4)
  double H[N * N];
};

template <int N>
__global__ void __launch_bounds__(kThreadsRows, (N <= 8) ? 2 : 1)
rhs_rows_kernel(const __grid_constant__ RowParams<N> P) {
  using C = RowCfg<N>;
  constexpr int NN = C::NN, G = C::G, T = C::T;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int W = p.W, M = p.M, D1 = p.D + 1;
  double2* sX = reinterpret_cast<double2*>(smem_raw);        // [T][NN] stage-input tile
  double2* sK = sX + T * NN;                                 // [kWarps][G][NN] warp-private
  double* sA = reinterpret_cast<double*>(sK + kWarps * G * NN);  // a_plus, a_minus_x, a_minus_o

  const int t0 = blockIdx.x * T;
  const int tcount = min(T, p.nodes - t0);
  // stage the tile (coalesced 16 B) and the coupling-factor tables
  {
    const double2* src = p.x + (size_t)t0 * p.stride;
    for (int e = threadIdx.x; e < tcount * NN; e += kThreadsRows) sX[e] = src[e];
    const int na = W * D1;
    for (int e = threadIdx.x; e < na; e += kThreadsRows) {
      sA[e] = p.a_plus[e]; sA[na + e] = p.a_minus_x[e]; sA[2 * na + e] = p.a_minus_o[e];
    }
  }
  __syncthreads();
  const double* sAp = sA;
  const double* sAx = sA + W * D1;
  const double* sAo = sA + 2 * W * D1;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane / N, i = lane - g * N;
  double2* myK = sK + warp * (G * NN);

  for (int pass = 0; pass < C::PASSES; ++pass) {
    const int first = (pass * kWarps + warp) * G;   // first tile-local node of this warp pass
    if (first >= tcount) break;                     // warp-uniform
    const int ncnt = min(G, tcount - first);
    const int tl = first + g;                       // tile-local node of this lane
    const bool active = (lane < G * N) && (g < ncnt);
    const int s = t0 + (active ? tl : first);       // storage slot (clamped for idle lanes)
    const double2* sig = sX + (size_t)(s - t0) * NN;
    DBG(s >= t0 && s - t0 < tcount && i < N && first + ncnt <= tcount);

    double2 k[N];
    {
      // ---- Eq. 12: commutator ------------------------------------------------------------
      double2 v[N];
#pragma unroll
      for (int m = 0; m < N; ++m) v[m] = sig[m * N + i];          // column i
      double2 b[N];
#pragma unroll
      for (int j = 0; j < N; ++j) {
        double br = 0.0, bi = 0.0;
#pragma unroll
        for (int m = 0; m < N; ++m) { br = fma(P.H[j * N + m], v[m].x, br); bi = fma(P.H[j * N + m], v[m].y, bi); }
        b[j] = make_double2(br, bi);
      }
      __syncwarp();
      if (active) {
#pragma unroll
        for (int j = 0; j < N; ++j) myK[g * NN + j * N + i] = b[j];  // (H sigma)[j][i]
      }
      __syncwarp();
#pragma unroll
      for (int m = 0; m < N; ++m) v[m] = sig[i * N + m];          // row i
      const double dd = p.damp[s];
#pragma unroll
      for (int j = 0; j < N; ++j) {
        double ar = 0.0, ai = 0.0;
#pragma unroll
        for (int m = 0; m < N; ++m) { ar = fma(v[m].x, P.H[m * N + j], ar); ai = fma(v[m].y, P.H[m * N + j], ai); }
        const double2 hs = myK[(active ? g : 0) * NN + i * N + j];  // (H sigma)[i][j]; idle lanes stay in range
        const double cr = hs.x - ar, ci = hs.y - ai;
        // -(i/hbar)(cr + i ci) = (ci - i cr)/hbar ; Eq. 13 + Eq. 14 on top
        const double dt = dd + p.Tterm[i * N + j];
        k[j].x = fma(-dt, v[j].x, ci * p.inv_hbar);
        k[j].y = fma(-dt, v[j].y, -cr * p.inv_hbar);
      }
    }

    // ---- Eq. 15-17 / 35-36: couplings to sigma_{n +- e_l} -------------------------------------
    const int32_t* lk = P.links + (size_t)s * P.lrow;
    const unsigned char* tup = reinterpret_cast<const unsigned char*>(lk + 2 * W);
    // row part: bath b = i, modes l = i*M + kk; V^x = +1, V^o = 1 on the whole row
    for (int kk = 0; kk < M; ++kk) {
      const int l = i * M + kk;
      const int up = lk[l], dn = lk[W + l], n = tup[l];
      DBG(l < W && n <= p.D && up < p.nodes && dn < p.nodes && s < p.nodes);
      if (up >= 0) {
        const double a = sAp[l * D1 + n];
        const unsigned loc = (unsigned)(up - t0);
        const double2* src = (loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)up * p.stride) + i * N;
#pragma unroll
        for (int j = 0; j < N; ++j) {
          const double2 w = src[j];
          k[j].x = fma(-a, w.y, k[j].x); k[j].y = fma(a, w.x, k[j].y);
        }
      }
      if (dn >= 0) {
        const double ax = sAx[l * D1 + n], ao = sAo[l * D1 + n];
        const unsigned loc = (unsigned)(dn - t0);
        const double2* src = (loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)dn * p.stride) + i * N;
#pragma unroll
        for (int j = 0; j < N; ++j) {
          const double2 w = src[j];
          k[j].x = fma(ao, w.x, fma(-ax, w.y, k[j].x));
          k[j].y = fma(ao, w.y, fma(ax, w.x, k[j].y));
        }
      }
    }
    // column part: every bath b, element [i][b]; V^x = -1, V^o = 1
#pragma unroll
    for (int b = 0; b < N; ++b) {
      for (int kk = 0; kk < M; ++kk) {
        const int l = b * M + kk;
        const int up = lk[l], dn = lk[W + l], n = tup[l];
        DBG(l < W && n <= p.D && up < p.nodes && dn < p.nodes);
        if (up >= 0) {
          const double a = sAp[l * D1 + n];
          const unsigned loc = (unsigned)(up - t0);
          const double2 w = (loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)up * p.stride)[i * N + b];
          k[b].x = fma(a, w.y, k[b].x); k[b].y = fma(-a, w.x, k[b].y);
        }
        if (dn >= 0) {
          const double ax = sAx[l * D1 + n], ao = sAo[l * D1 + n];
          const unsigned loc = (unsigned)(dn - t0);
          const double2 w = (loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)dn * p.stride)[i * N + b];
          k[b].x = fma(ao, w.x, fma(ax, w.y, k[b].x));
          k[b].y = fma(ao, w.y, fma(-ax, w.x, k[b].y));
        }
      }
    }

    // ---- k rows -> warp tile, then the fused RK4 stage epilogue, coalesced ---------------------
    __syncwarp();
    if (active) {
#pragma unroll
      for (int j = 0; j < N; ++j) myK[g * NN + i * N + j] = k[j];
    }
    __syncwarp();
    const size_t base = (size_t)(t0 + first) * p.stride;
    const int nel = ncnt * NN;
    if (p.rhs_only) {
      for (int e = lane; e < nel; e += 32) p.out_acc[base + e] = myK[e];
    } else if (p.out_x) {
      for (int e = lane; e < nel; e += 32) {
        const double2 kv = myK[e];
        const double2 yv = p.y[base + e];
        const double2 av = p.acc_in[base + e];
        p.out_x[base + e] = make_double2(fma(p.ax, kv.x, yv.x), fma(p.ax, kv.y, yv.y));
        p.out_acc[base + e] = make_double2(fma(p.bx, kv.x, av.x), fma(p.bx, kv.y, av.y));
      }
    } else {
      for (int e = lane; e < nel; e += 32) {
        const double2 kv = myK[e];
        const double2 av = p.acc_in[base + e];
        p.out_acc[base + e] = make_double2(fma(p.bx, kv.x, av.x), fma(p.bx, kv.y, av.y));
      }
    }
  }
}

template <int N>
size_t rows_smem(int W, int D) {
  using C = RowCfg<N>;
  return (size_t)(C::T + kWarps * C::G) * C::NN * sizeof(double2) + (size_t)3 * W * (D + 1) * sizeof(double);
}

template <int N>
cudaError_t launch_rows_t(const RhsParams& p, const int32_t* links, int lrow, const double* H_host,
                          cudaStream_t s) {
  using C = RowCfg<N>;
  RowParams<N> P;
  P.p = p; P.links = links; P.lrow = lrow;
  for (int e = 0; e < N * N; ++e) P.H[e] = H_host[e];
  const size_t smem = rows_smem<N>(p.W, p.D);
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_rows_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  const int grid = (p.nodes + C::T - 1) / C::T;
  rhs_rows_kernel<N><<<grid, kThreadsRows, smem, s>>>(P);
  return cudaGetLastError();
}

}  // namespace

bool rows_supported(int N, int W, int D) {
  if (N < 2 || N > 16) return false;
  return (size_t)3 * W * (D + 1) * 8 <= 32 * 1024;
}

cudaError_t launch_rhs_rows(const RhsParams& p, const int32_t* links, int lrow, const double* H_host,
                            cudaStream_t s) {
  switch (p.N) {
#define HEOM_ROWS_CASE(n) case n: return launch_rows_t<n>(p, links, lrow, H_host, s);
    HEOM_ROWS_CASE(2) HEOM_ROWS_CASE(3) HEOM_ROWS_CASE(4) HEOM_ROWS_CASE(5) HEOM_ROWS_CASE(6)
    HEOM_ROWS_CASE(7) HEOM_ROWS_CASE(8) HEOM_ROWS_CASE(9) HEOM_ROWS_CASE(10) HEOM_ROWS_CASE(11)
    HEOM_ROWS_CASE(12) HEOM_ROWS_CASE(13) HEOM_ROWS_CASE(14) HEOM_ROWS_CASE(15) HEOM_ROWS_CASE(16)
#undef HEOM_ROWS_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace heom
