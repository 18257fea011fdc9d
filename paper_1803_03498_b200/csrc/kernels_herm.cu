// kernels_herm.cu -- small-N (2 <= N <= 16) sm_100a kernel for HERMITIAN hierarchy states.
//
// The hierarchical Liouvillian (Eq. 12-17) maps Hermitian ADOs to Hermitian ADOs (gamma and
// Re c real), so for a Hermitian state the column b of a neighbour is the conjugate of its row b
// and the whole right-hand side can be written with ROW reads only:
//     Z   = -(i/hbar) H sigma_u + sum_l [ i a+ P_b sigma_{u+e_l} + (i a-x + a-o) P_b sigma_{u-e_l} ]
//     k_u = Z + Z^dagger - (d_u + T) o sigma_u          (P_b keeps row b; b = l div M; Eq. 23-25)
// Row b of a neighbour is 16N contiguous bytes, read by the N lanes of a node with one coalesced
// request -- the strided column gathers of the general kernel (kernels_rows.cu) disappear.
//
// Mapping: lane (g, j) owns COLUMN j of node g of the warp (G = 32/N nodes per warp pass); H and
// the terminator constants are warp-uniform constant-bank operands.  A CTA stages its tile of T
// consecutive storage slots (sigma matrices + link rows) in shared memory; neighbours inside
// the tile are read from there.  Z is transposed through a warp-private tile; k goes back to it
// and the warp streams the fused RK4 update with coalesced 16-byte accesses.
// Element (j,i) is produced by exactly the conjugate operations of element (i,j), so the state
// stays bit-exactly Hermitian from stage to stage.
#include "kernels.cuh"

namespace heom {
namespace {

template <int N>
struct HermCfg {
  static constexpr int NN = N * N;
  static constexpr int G = 32 / N;                    // nodes per warp pass
  static constexpr int WARPS = 8;
  static constexpr int THREADS = WARPS * 32;
  static constexpr int T = (N <= 8) ? 64 : 32;        // nodes per CTA tile
  static constexpr int MINB = (N <= 8) ? 2 : 1;
  static constexpr int PASSES = (T + G * WARPS - 1) / (G * WARPS);
  static constexpr int EPI = (G * NN + 31) / 32;
  static constexpr int NP4 = (N + 3) / 4 * 4;         // ints per index group
  static constexpr int NB8 = (N + 7) / 8 * 8;         // tuple bytes per group
  static constexpr int GROUP = (2 * NP4 + NB8 / 4 + 3) / 4 * 4;  // ints per mode group kk: plus, minus, n bytes (16 B multiple)
};

template <int N>
struct HermParams {
  RhsParams p;
  const int32_t* links;   // [nodes][lrow] in the grouped layout of herm_links_row()
  const double* coef;     // [W][D+1][4] = a+, a-x, a-o, 0
  int lrow;               // ints per links row (multiple of 4)
  double H[N * N];
  double delta[N];
};

__device__ __forceinline__ void prefetch_l2h(const void* ptr) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
}

template <int N>
__global__ void __launch_bounds__(HermCfg<N>::THREADS, HermCfg<N>::MINB)
rhs_herm_kernel(const __grid_constant__ HermParams<N> P) {
  using C = HermCfg<N>;
  constexpr int NN = C::NN, G = C::G, T = C::T, WARPS = C::WARPS, THREADS = C::THREADS;
  constexpr int NP4 = C::NP4, NB8 = C::NB8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int W = p.W, M = p.M, D1 = p.D + 1, lrow = P.lrow;
  double2* sX = reinterpret_cast<double2*>(smem_raw);            // [T][NN]
  double2* sK = sX + T * NN;                                     // [WARPS][G][NN]
  double2* sC = sK + WARPS * G * NN;                             // [W*D1][2] double2 = 4 doubles
  int32_t* sL = reinterpret_cast<int32_t*>(sC + 2 * W * D1);     // [T][lrow]

  const int t0 = blockIdx.x * T;
  const int tcount = min(T, p.nodes - t0);
  {
    const double2* src = p.x + (size_t)t0 * p.stride;
    for (int e = threadIdx.x; e < tcount * NN; e += THREADS) sX[e] = src[e];
    const int4* lsrc = reinterpret_cast<const int4*>(P.links + (size_t)t0 * lrow);
    int4* ldst = reinterpret_cast<int4*>(sL);
    for (int e = threadIdx.x; e < tcount * (lrow >> 2); e += THREADS) ldst[e] = lsrc[e];
    const double2* csrc = reinterpret_cast<const double2*>(P.coef);
    for (int e = threadIdx.x; e < 2 * W * D1; e += THREADS) sC[e] = csrc[e];
    if (!p.rhs_only) {
      const size_t off = (size_t)t0 * p.stride;
      const int lines = (tcount * NN * 16 + 127) >> 7;
      for (int e = threadIdx.x; e < lines; e += THREADS) {
        prefetch_l2h(reinterpret_cast<const char*>(p.acc_in + off) + ((size_t)e << 7));
        if (p.out_x) prefetch_l2h(reinterpret_cast<const char*>(p.y + off) + ((size_t)e << 7));
      }
    }
  }
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane / N, j = lane - g * N;
  double2* myK = sK + warp * (G * NN);
  const double my_delta = P.delta[j];

  for (int pass = 0; pass < C::PASSES; ++pass) {
    const int first = (pass * WARPS + warp) * G;
    if (first >= tcount) break;                     // warp-uniform
    const int ncnt = min(G, tcount - first);
    const bool active = (lane < G * N) && (g < ncnt);
    const int gg = active ? g : 0;                  // idle lanes shadow the pass's first node
    const int tl = first + gg;
    const int s = t0 + tl;
    const double2* sig = sX + (size_t)tl * NN;

    // ---- Z = -(i/hbar) H sigma, column j ------------------------------------------------------
    double2 col[N], z[N];
#pragma unroll
    for (int m = 0; m < N; ++m) col[m] = sig[m * N + j];
#pragma unroll
    for (int b = 0; b < N; ++b) {
      double zr = 0.0, zi = 0.0;
#pragma unroll
      for (int m = 0; m < N; ++m) { zr = fma(P.H[b * N + m], col[m].x, zr); zi = fma(P.H[b * N + m], col[m].y, zi); }
      z[b] = make_double2(zi * p.inv_hbar, -zr * p.inv_hbar);
    }

    // ---- couplings: row b of sigma_{u +- e_l}, element j (Eq. 15-17 / 35-36, Eq. 23, 25) -------
    auto nb = [&](int idx) -> const double2* {
      const unsigned loc = (unsigned)(idx - t0);
      return loc < (unsigned)tcount ? sX + (size_t)loc * NN : p.x + (size_t)idx * p.stride;
    };
    for (int kk = 0; kk < M; ++kk) {
      const int32_t* grp = sL + tl * lrow + kk * C::GROUP;
      int up[NP4], dn[NP4];
      unsigned nbytes[NB8 / 4];
#pragma unroll
      for (int q = 0; q < NP4 / 4; ++q) {
        const int4 a = reinterpret_cast<const int4*>(grp)[q];
        const int4 c = reinterpret_cast<const int4*>(grp + NP4)[q];
        up[4 * q] = a.x; up[4 * q + 1] = a.y; up[4 * q + 2] = a.z; up[4 * q + 3] = a.w;
        dn[4 * q] = c.x; dn[4 * q + 1] = c.y; dn[4 * q + 2] = c.z; dn[4 * q + 3] = c.w;
      }
#pragma unroll
      for (int q = 0; q < NB8 / 8; ++q) {
        const uint2 t = reinterpret_cast<const uint2*>(grp + 2 * NP4)[q];
        nbytes[2 * q] = t.x; nbytes[2 * q + 1] = t.y;
      }
      double2 wu[N], wd[N], c01[N], c23[N];
#pragma unroll
      for (int b = 0; b < N; ++b) {
        const int n = (nbytes[b >> 2] >> (8 * (b & 3))) & 0xff;
        const double2* rec = sC + 2 * ((b * M + kk) * D1 + n);
        c01[b] = rec[0];   // a+, a-x
        c23[b] = rec[1];   // a-o, 0
        wu[b] = make_double2(0.0, 0.0);
        wd[b] = make_double2(0.0, 0.0);
        if (up[b] >= 0) wu[b] = nb(up[b])[b * N + j];
        if (dn[b] >= 0) wd[b] = nb(dn[b])[b * N + j];
      }
#pragma unroll
      for (int b = 0; b < N; ++b) {
        const double a = c01[b].x, ax = c01[b].y, ao = c23[b].x;
        z[b].x = fma(-a, wu[b].y, z[b].x); z[b].y = fma(a, wu[b].x, z[b].y);
        z[b].x = fma(ao, wd[b].x, fma(-ax, wd[b].y, z[b].x));
        z[b].y = fma(ao, wd[b].y, fma(ax, wd[b].x, z[b].y));
      }
    }

    // ---- k = Z + Z^dagger - (d_u + T) o sigma, column j ------------------------------------------
    __syncwarp();
    if (active) {
#pragma unroll
      for (int b = 0; b < N; ++b) myK[g * NN + b * N + j] = z[b];
    }
    __syncwarp();
    const double dd = p.damp[s];
    double2 k[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const double2 zt = myK[gg * NN + j * N + i];               // Z[j][i]
      const double dt = dd + ((i == j) ? 0.0 : P.delta[i] + my_delta);   // Eq. 13 + Eq. 14/24
      k[i].x = fma(-dt, col[i].x, z[i].x + zt.x);
      k[i].y = fma(-dt, col[i].y, z[i].y - zt.y);
    }
    __syncwarp();
    if (active) {
#pragma unroll
      for (int i = 0; i < N; ++i) myK[g * NN + i * N + j] = k[i];
    }
    __syncwarp();

    // ---- fused RK4 stage epilogue, coalesced over the warp's nodes --------------------------------
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
size_t herm_smem(int W, int D, int lrow) {
  using C = HermCfg<N>;
  return (size_t)(C::T + C::WARPS * C::G) * C::NN * sizeof(double2) + (size_t)W * (D + 1) * 32 +
         (size_t)C::T * lrow * sizeof(int32_t);
}

template <int N>
cudaError_t launch_herm_t(const RhsParams& p, const int32_t* links, int lrow, const double* coef,
                          const double* H_host, const double* delta_host, cudaStream_t s) {
  using C = HermCfg<N>;
  HermParams<N> P;
  P.p = p; P.links = links; P.coef = coef; P.lrow = lrow;
  for (int e = 0; e < N * N; ++e) P.H[e] = H_host[e];
  for (int e = 0; e < N; ++e) P.delta[e] = delta_host[e];
  const size_t smem = herm_smem<N>(p.W, p.D, lrow);
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_herm_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  const int grid = (p.nodes + C::T - 1) / C::T;
  rhs_herm_kernel<N><<<grid, C::THREADS, smem, s>>>(P);
  return cudaGetLastError();
}

}  // namespace

#define HEOM_HERM_ALL(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

int herm_links_row(int N, int M) {
  if (N < 2 || N > 16) return 0;
  const int np4 = (N + 3) / 4 * 4, nb8 = (N + 7) / 8 * 8;
  return M * ((2 * np4 + nb8 / 4 + 3) / 4 * 4);
}

bool herm_supported(int N, int W, int D) {
  const int M = W / (N > 0 ? N : 1);
  const int lrow = herm_links_row(N, M);
  if (lrow == 0) return false;
  switch (N) {
#define HEOM_HERM_CASE(n) case n: return herm_smem<n>(W, D, lrow) <= 200 * 1024;
    HEOM_HERM_ALL(HEOM_HERM_CASE)
#undef HEOM_HERM_CASE
    default: return false;
  }
}

void herm_pack_links(int N, int M, const int32_t* plus, const int32_t* minus, const uint8_t* tuple,
                     int32_t* row) {
  const int np4 = (N + 3) / 4 * 4, nb8 = (N + 7) / 8 * 8, group = (2 * np4 + nb8 / 4 + 3) / 4 * 4;
  for (int kk = 0; kk < M; ++kk) {
    int32_t* grp = row + kk * group;
    unsigned char* nby = reinterpret_cast<unsigned char*>(grp + 2 * np4);
    for (int b = 0; b < np4; ++b) {
      grp[b] = (b < N) ? plus[b * M + kk] : -1;
      grp[np4 + b] = (b < N) ? minus[b * M + kk] : -1;
    }
    for (int b = 0; b < nb8; ++b) nby[b] = (b < N) ? tuple[b * M + kk] : 0;
  }
}

cudaError_t launch_rhs_herm(const RhsParams& p, const int32_t* links, int lrow, const double* coef,
                            const double* H_host, const double* delta_host, cudaStream_t s) {
  switch (p.N) {
#define HEOM_HERM_CASE(n) case n: return launch_herm_t<n>(p, links, lrow, coef, H_host, delta_host, s);
    HEOM_HERM_ALL(HEOM_HERM_CASE)
#undef HEOM_HERM_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace heom
