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

// ---- TMA bulk copy (global -> shared, completion on an mbarrier) and friends ------------------
__device__ __forceinline__ unsigned smem_u32(const void* ptr) {
  return (unsigned)__cvta_generic_to_shared(ptr);
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes,
                                         unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
// 16-byte load from a generic address (shared tile or global state), executed only when `on`;
// returns 0 otherwise.  Keeps the gather loop straight-line so the loads of a batch overlap.
__device__ __forceinline__ double2 ld_if(const double2* ptr, bool on) {
  double2 r;
  asm("{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %3, 0;\n"
      "mov.f64 %0, 0d0000000000000000;\n"
      "mov.f64 %1, 0d0000000000000000;\n"
      "@p ld.v2.f64 {%0, %1}, [%2];\n"
      "}\n" : "=d"(r.x), "=d"(r.y) : "l"(ptr), "r"((int)on));
  return r;
}

template <int N>
__global__ void __launch_bounds__(HermCfg<N>::THREADS, HermCfg<N>::MINB)
rhs_herm_kernel(const __grid_constant__ HermParams<N> P) {
  using C = HermCfg<N>;
  constexpr int NN = C::NN, G = C::G, T = C::T, WARPS = C::WARPS;
  constexpr int NP4 = C::NP4, NB8 = C::NB8;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int W = p.W, M = p.M, D1 = p.D + 1, lrow = P.lrow;
  double2* sX = reinterpret_cast<double2*>(smem_raw);            // [T][NN]
  double2* sK = sX + T * NN;                                     // [WARPS][G][NN]
  double2* sC = sK + WARPS * G * NN;                             // [W*D1][2] double2 = 4 doubles
  int32_t* sL = reinterpret_cast<int32_t*>(sC + 2 * W * D1);     // [T][lrow]
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(sL + T * lrow);

  const int t0 = blockIdx.x * T;
  const int tcount = min(T, p.nodes - t0);
  // One thread arms the mbarrier and issues three bulk copies (sigma tile, link rows, coupling
  // factors) plus L2 prefetches of the y / acc ranges the epilogue will stream.
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned bx = (unsigned)tcount * NN * 16, bl = (unsigned)tcount * lrow * 4, bc = (unsigned)W * D1 * 32;
    mbar_expect_tx(bar, bx + bl + bc);
    bulk_g2s(sX, p.x + (size_t)t0 * p.stride, bx, bar);
    bulk_g2s(sL, P.links + (size_t)t0 * lrow, bl, bar);
    bulk_g2s(sC, P.coef, bc, bar);
    if (!p.rhs_only) {
      bulk_prefetch_l2(p.acc_in + (size_t)t0 * p.stride, bx);
      if (p.out_x) bulk_prefetch_l2(p.y + (size_t)t0 * p.stride, bx);
    }
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int g = lane / N, j = lane - g * N;
  double2* myK = sK + warp * (G * NN);
  const double my_delta = P.delta[j];
  mbar_wait(bar, 0);

  for (int pass = 0; pass < C::PASSES; ++pass) {
    const int first = (pass * WARPS + warp) * G;
    if (first >= tcount) break;                     // warp-uniform
    const int ncnt = min(G, tcount - first);
    const bool active = (lane < G * N) && (g < ncnt);
    const int gg = active ? g : 0;                  // idle lanes shadow the pass's first node
    const int tl = first + gg;
    const int s = t0 + tl;
    const double2* sig = sX + (size_t)tl * NN;

    // ---- Z = -(i/hbar) H sigma - (d_u + T)/2 o sigma, column j ------------------------------------
    // (Z + Z^dagger then carries the full damping/terminator term, Eq. 13-14, exactly symmetrically)
    double2 z[N];
    {
      double2 col[N];
#pragma unroll
      for (int m = 0; m < N; ++m) col[m] = sig[m * N + j];
      const double dd = p.damp[s];
#pragma unroll
      for (int b = 0; b < N; ++b) {
        double zr = 0.0, zi = 0.0;
#pragma unroll
        for (int m = 0; m < N; ++m) { zr = fma(P.H[b * N + m], col[m].x, zr); zi = fma(P.H[b * N + m], col[m].y, zi); }
        const double hd = -0.5 * (dd + ((b == j) ? 0.0 : P.delta[b] + my_delta));
        z[b].x = fma(hd, col[b].x, zi * p.inv_hbar);
        z[b].y = fma(hd, col[b].y, -zr * p.inv_hbar);
      }
    }

    // ---- couplings: row b of sigma_{u +- e_l}, element j (Eq. 15-17 / 35-36, Eq. 23, 25) -------
    const double2* xg = p.x;
    const int stride = p.stride;
    auto nb = [&](int idx, int off) -> const double2* {
      const unsigned loc = (unsigned)(idx - t0);
      return (loc < (unsigned)tcount ? sX + (size_t)loc * NN : xg + (size_t)idx * stride) + off;
    };
    for (int kk = 0; kk < M; ++kk) {
      const int32_t* grp = sL + tl * lrow + kk * C::GROUP;
      unsigned nbytes[NB8 / 4];
#pragma unroll
      for (int q = 0; q < NB8 / 8; ++q) {
        const uint2 t = reinterpret_cast<const uint2*>(grp + 2 * NP4)[q];
        nbytes[2 * q] = t.x; nbytes[2 * q + 1] = t.y;
      }
      {  // "+" links: i a+ sigma^+[b][j]
        int up[NP4];
#pragma unroll
        for (int q = 0; q < NP4 / 4; ++q) {
          const int4 a = reinterpret_cast<const int4*>(grp)[q];
          up[4 * q] = a.x; up[4 * q + 1] = a.y; up[4 * q + 2] = a.z; up[4 * q + 3] = a.w;
        }
        double2 w[N];
#pragma unroll
        for (int b = 0; b < N; ++b) w[b] = ld_if(nb(up[b], b * N + j), up[b] >= 0);
#pragma unroll
        for (int b = 0; b < N; ++b) {
          const int n = (nbytes[b >> 2] >> (8 * (b & 3))) & 0xff;
          const double a = sC[2 * ((b * M + kk) * D1 + n)].x;
          z[b].x = fma(-a, w[b].y, z[b].x); z[b].y = fma(a, w[b].x, z[b].y);
        }
      }
      {  // "-" links: (i a-x + a-o) sigma^-[b][j]
        int dn[NP4];
#pragma unroll
        for (int q = 0; q < NP4 / 4; ++q) {
          const int4 c = reinterpret_cast<const int4*>(grp + NP4)[q];
          dn[4 * q] = c.x; dn[4 * q + 1] = c.y; dn[4 * q + 2] = c.z; dn[4 * q + 3] = c.w;
        }
        double2 w[N];
#pragma unroll
        for (int b = 0; b < N; ++b) w[b] = ld_if(nb(dn[b], b * N + j), dn[b] >= 0);
#pragma unroll
        for (int b = 0; b < N; ++b) {
          const int n = (nbytes[b >> 2] >> (8 * (b & 3))) & 0xff;
          const double2* rec = sC + 2 * ((b * M + kk) * D1 + n);
          const double ax = rec[0].y, ao = rec[1].x;
          z[b].x = fma(ao, w[b].x, fma(-ax, w[b].y, z[b].x));
          z[b].y = fma(ao, w[b].y, fma(ax, w[b].x, z[b].y));
        }
      }
    }

    // ---- k = Z + Z^dagger, column j -------------------------------------------------------------
    __syncwarp();
    if (active) {
#pragma unroll
      for (int b = 0; b < N; ++b) myK[g * NN + b * N + j] = z[b];
    }
    __syncwarp();
    double2 k[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const double2 zt = myK[gg * NN + j * N + i];               // Z[j][i]
      k[i].x = z[i].x + zt.x;
      k[i].y = z[i].y - zt.y;
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
         (size_t)C::T * lrow * sizeof(int32_t) + 16;
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
  static size_t configured_on[64] = {};   // per device: the attribute belongs to the device's context
  int dev_ = 0;
  cudaGetDevice(&dev_);
  size_t& configured = configured_on[dev_ & 63];
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
