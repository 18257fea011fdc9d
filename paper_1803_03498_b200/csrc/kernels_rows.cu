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

template <int N>
struct RowCfg {
  static constexpr int NN = N * N;
  static constexpr int G = 32 / N;                    // nodes per warp pass
  static constexpr int WARPS = 8;
  static constexpr int THREADS = WARPS * 32;
  static constexpr int T = (N <= 8) ? 64 : 32;        // nodes per CTA tile
  static constexpr int MINB = (N <= 8) ? 2 : 1;       // CTAs per SM the register budget is cut for
  static constexpr int PASSES = (T + G * WARPS - 1) / (G * WARPS);
  static constexpr int EPI = (G * NN + 31) / 32;      // 16-byte elements per lane in the epilogue
};

template <int N>
struct RowParams {
  RhsParams p;
  const int32_t* links;  // [nodes][lrow]: plus[W], minus[W], tuple bytes packed 4 per int32
  int lrow;              // int32 entries per links row (multiple of 4)
  double H[N * N];
};

__device__ __forceinline__ void prefetch_l2(const void* ptr) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
}

template <int N>
__global__ void __launch_bounds__(RowCfg<N>::THREADS, RowCfg<N>::MINB)
rhs_rows_kernel(const __grid_constant__ RowParams<N> P) {
  using C = RowCfg<N>;
  constexpr int NN = C::NN, G = C::G, T = C::T, WARPS = C::WARPS, THREADS = C::THREADS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int W = p.W, M = p.M, D1 = p.D + 1, lrow = P.lrow;
  double2* sX = reinterpret_cast<double2*>(smem_raw);            // [T][NN] stage-input tile
  double2* sK = sX + T * NN;                                     // [WARPS][G][NN] warp-private
  double* sA = reinterpret_cast<double*>(sK + WARPS * G * NN);   // a_plus, a_minus_x, a_minus_o
  int32_t* sL = reinterpret_cast<int32_t*>(sA + ((3 * W * D1 + 1) & ~1));     // [T][lrow] link rows of the tile

  const int t0 = blockIdx.x * T;
  const int tcount = min(T, p.nodes - t0);
  // stage the sigma tile and its link rows (coalesced 16 B), the coupling-factor tables, and pull
  // the y / acc lines the epilogue will need into L2 while the arithmetic runs
  {
    const double2* src = p.x + (size_t)t0 * p.stride;
    for (int e = threadIdx.x; e < tcount * NN; e += THREADS) sX[e] = src[e];
    const int4* lsrc = reinterpret_cast<const int4*>(P.links + (size_t)t0 * lrow);
    int4* ldst = reinterpret_cast<int4*>(sL);
    for (int e = threadIdx.x; e < tcount * (lrow >> 2); e += THREADS) ldst[e] = lsrc[e];
    const int na = W * D1;
    for (int e = threadIdx.x; e < na; e += THREADS) {
      sA[e] = p.a_plus[e]; sA[na + e] = p.a_minus_x[e]; sA[2 * na + e] = p.a_minus_o[e];
    }
    if (!p.rhs_only) {
      const size_t off = (size_t)t0 * p.stride;
      const int lines = (tcount * NN * 16 + 127) >> 7;
      for (int e = threadIdx.x; e < lines; e += THREADS) {
        prefetch_l2(reinterpret_cast<const char*>(p.acc_in + off) + ((size_t)e << 7));
        if (p.out_x) prefetch_l2(reinterpret_cast<const char*>(p.y + off) + ((size_t)e << 7));
      }
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
    const int first = (pass * WARPS + warp) * G;    // first tile-local node of this warp pass
    if (first >= tcount) break;                     // warp-uniform
    const int ncnt = min(G, tcount - first);
    const bool active = (lane < G * N) && (g < ncnt);
    const int gg = active ? g : 0;                  // idle lanes shadow the pass's first node
    const int tl = first + gg;                      // tile-local node of this lane
    const int s = t0 + tl;                          // storage slot
    const double2* sig = sX + (size_t)tl * NN;
    DBG(tl < tcount && i < N && first + ncnt <= tcount);

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
        const double2 hs = myK[gg * NN + i * N + j];               // (H sigma)[i][j]
        const double cr = hs.x - ar, ci = hs.y - ai;
        // -(i/hbar)(cr + i ci) = (ci - i cr)/hbar ; Eq. 13 + Eq. 14 on top
        const double dt = dd + p.Tterm[i * N + j];
        k[j].x = fma(-dt, v[j].x, ci * p.inv_hbar);
        k[j].y = fma(-dt, v[j].y, -cr * p.inv_hbar);
      }
    }

    // ---- Eq. 15-17 / 35-36: couplings to sigma_{n +- e_l} -------------------------------------
    // Branch-free loads: an invalid link reads the lane's own node from the tile with a
    // zero factor, so every batch of neighbour loads is issued back to back (the L2 round trips
    // overlap instead of queueing behind per-link branches).
    const int32_t* lk = sL + tl * lrow;
    const unsigned char* tup = reinterpret_cast<const unsigned char*>(lk + 2 * W);
    auto nb = [&](int idx) -> const double2* {
      const int c = idx >= 0 ? idx : s;
      const unsigned loc = (unsigned)(c - t0);
      return loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)c * p.stride;
    };
    for (int kk = 0; kk < M; ++kk) {
      // row part: bath b = i, mode l = i*M + kk; V^x = +1, V^o = 1 on the whole row i
      {
        const int l = i * M + kk;
        const int up = lk[l], dn = lk[W + l], n = tup[l];
        DBG(l < W && n <= p.D && up < p.nodes && dn < p.nodes);
        const double a = up >= 0 ? sAp[l * D1 + n] : 0.0;
        const double ax = dn >= 0 ? sAx[l * D1 + n] : 0.0;
        const double ao = dn >= 0 ? sAo[l * D1 + n] : 0.0;
        const double2* pu = nb(up) + i * N;
        const double2* pd = nb(dn) + i * N;
        double2 wu[N], wd[N];
#pragma unroll
        for (int j = 0; j < N; ++j) { wu[j] = pu[j]; wd[j] = pd[j]; }
#pragma unroll
        for (int j = 0; j < N; ++j) {
          k[j].x = fma(-a, wu[j].y, k[j].x); k[j].y = fma(a, wu[j].x, k[j].y);
          k[j].x = fma(ao, wd[j].x, fma(-ax, wd[j].y, k[j].x));
          k[j].y = fma(ao, wd[j].y, fma(ax, wd[j].x, k[j].y));
        }
      }
      // column part: every bath b, mode l = b*M + kk, element [i][b]; V^x = -1, V^o = 1
      {
        double2 wu[N], wd[N];
        double a[N], ax[N], ao[N];
#pragma unroll
        for (int b = 0; b < N; ++b) {
          const int l = b * M + kk;
          const int up = lk[l], dn = lk[W + l], n = tup[l];
          a[b] = up >= 0 ? sAp[l * D1 + n] : 0.0;
          ax[b] = dn >= 0 ? sAx[l * D1 + n] : 0.0;
          ao[b] = dn >= 0 ? sAo[l * D1 + n] : 0.0;
          wu[b] = nb(up)[i * N + b];
          wd[b] = nb(dn)[i * N + b];
        }
#pragma unroll
        for (int b = 0; b < N; ++b) {
          k[b].x = fma(a[b], wu[b].y, k[b].x); k[b].y = fma(-a[b], wu[b].x, k[b].y);
          k[b].x = fma(ao[b], wd[b].x, fma(ax[b], wd[b].y, k[b].x));
          k[b].y = fma(ao[b], wd[b].y, fma(-ax[b], wd[b].x, k[b].y));
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
    } else {
      constexpr int CH = 4;   // loads in flight per lane and array
      for (int c0 = 0; c0 < C::EPI; c0 += CH) {
        double2 yv[CH], av[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) {
          const int e = lane + 32 * (c0 + c);
          if (e < nel) {
            av[c] = p.acc_in[base + e];
            if (p.out_x) yv[c] = p.y[base + e];
          }
        }
#pragma unroll
        for (int c = 0; c < CH; ++c) {
          const int e = lane + 32 * (c0 + c);
          if (e < nel) {
            const double2 kv = myK[e];
            if (p.out_x) p.out_x[base + e] = make_double2(fma(p.ax, kv.x, yv[c].x), fma(p.ax, kv.y, yv[c].y));
            p.out_acc[base + e] = make_double2(fma(p.bx, kv.x, av[c].x), fma(p.bx, kv.y, av[c].y));
          }
        }
      }
    }
  }
}

template <int N>
size_t rows_smem(int W, int D, int lrow) {
  using C = RowCfg<N>;
  return (size_t)(C::T + C::WARPS * C::G) * C::NN * sizeof(double2) + (((size_t)3 * W * (D + 1) + 1) & ~(size_t)1) * sizeof(double) +
         (size_t)C::T * lrow * sizeof(int32_t);
}

template <int N>
cudaError_t launch_rows_t(const RhsParams& p, const int32_t* links, int lrow, const double* H_host,
                          cudaStream_t s) {
  using C = RowCfg<N>;
  RowParams<N> P;
  P.p = p; P.links = links; P.lrow = lrow;
  for (int e = 0; e < N * N; ++e) P.H[e] = H_host[e];
  const size_t smem = rows_smem<N>(p.W, p.D, lrow);
  static size_t configured_on[64] = {};   // per device: the attribute belongs to the device's context
  int dev_ = 0;
  cudaGetDevice(&dev_);
  size_t& configured = configured_on[dev_ & 63];
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_rows_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  const int grid = (p.nodes + C::T - 1) / C::T;
  rhs_rows_kernel<N><<<grid, C::THREADS, smem, s>>>(P);
  return cudaGetLastError();
}

template <int N>
bool rows_fit(int W, int D, int lrow) { return rows_smem<N>(W, D, lrow) <= 200 * 1024; }

}  // namespace

#define HEOM_ROWS_ALL(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

bool rows_supported(int N, int W, int D, int lrow) {
  switch (N) {
#define HEOM_ROWS_CASE(n) case n: return rows_fit<n>(W, D, lrow);
    HEOM_ROWS_ALL(HEOM_ROWS_CASE)
#undef HEOM_ROWS_CASE
    default: return false;
  }
}

cudaError_t launch_rhs_rows(const RhsParams& p, const int32_t* links, int lrow, const double* H_host,
                            cudaStream_t s) {
  switch (p.N) {
#define HEOM_ROWS_CASE(n) case n: return launch_rows_t<n>(p, links, lrow, H_host, s);
    HEOM_ROWS_ALL(HEOM_ROWS_CASE)
#undef HEOM_ROWS_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace heom
