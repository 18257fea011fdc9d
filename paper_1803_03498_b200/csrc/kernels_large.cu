// kernels_large.cu -- sm_100a kernel for LARGE system sizes (N a multiple of 32 up to 96; BASELINE config
// 5: N = 96), where the commutator of Eq. 12 is a real dense contraction: the HEOM right-hand side
// (Eq. 12-17 with Eq. 23-25, 35-36) with the RK4 stage combination fused into its epilogue.
//
// One persistent CTA per SM works on one node at a time (nodes are drawn from a global ticket counter).
//   * H/hbar (real, N x N) stays in shared memory for the whole launch; the node's sigma (complex N x N)
//     is streamed into shared memory by the TMA (cp.async.bulk, one copy per matrix row into a padded
//     row, completion on an mbarrier) while the previous node's epilogue is still running.
//   * C = (H/hbar) sigma - sigma (H/hbar) runs on the FP64 tensor cores (mma.sync.m8n8k4.f64, SASS
//     DMMA.8x8x4 -- tcgen05 has no FP64 kind).  The CTA's warps tile the N x N complex result WR x WC; each
//     warp keeps its tile in registers for both products:
//       P1 = H sigma      A = H[i][m],           B = sigma[m][(j,c)]  (sigma as an N x 2N real matrix)
//       P2 = sigma H      A = -sigma[i][(m,c)],  B = H[m][j]          (one DMMA for c = re, one for c = im)
//     Fragment rows, P1's k order and P2's column order are permuted (below) so that every lane ends up
//     with whole complex elements, both products accumulate into the SAME registers, and the shared-
//     memory fragment loads are (almost) free of bank conflicts with plain padded rows.
//   * k = -i C - (d_u + T) o sigma (Eq. 13-14) is formed in the fragment layout; the couplings to
//     sigma_{u +- e_l} (Eq. 15-17 / 35-36) are added from a compact per-node link list with predicated
//     global loads of the neighbour's row b and column b (Eq. 23, 25); the RK4 update reads y / acc and
//     writes the next stage input / running sum straight from the fragment layout (64-byte segments).
//   * HERM = true (the state is exactly Hermitian, checked in api.cu, never assumed): the hierarchical Liouvillian
//     maps Hermitian ADOs to Hermitian ADOs, so k_u = Z + Z^dagger with
//       Z = -(i/hbar) H sigma_u - (d_u + T)/2 o sigma_u + sum_l (a-o + i a) P_b sigma_{u +- e_l}   (P_b keeps row b)
//     as in kernels_hpipe.cu: only P1 = H sigma runs on the tensor cores (4 N^3 instead of 8 N^3 flop), only ROWS
//     of the neighbours are gathered (contiguous), and Z is transposed through the sigma tile's shared memory
//     once the contraction is done with it.  Element (j,i) is produced by exactly the conjugate operations of
//     (i,j): the state stays bit-exactly Hermitian.  The rows are gathered ROW-WISE: a lane looks the links of the
//     rows it owns up in the node's dense link row {plus[W], minus[W], n[W]} (bath b <-> row b in these contexts) and
//     issues their loads independently of one another; all neighbour rows of the node are bulk-prefetched into L2 at
//     the top of the node, behind the contraction.  (General states walk the compact link list.)
#include "kernels.cuh"

#include <cmath>

namespace heom {
namespace {

constexpr int kLargeMaxModes = 288;   // W of the constant-bank coupling tables (N = 96, K = 2)

template <int N>
struct LargeCfg {
  static constexpr int WR = N / 32;                   // warp grid: WR x WC warps
  static constexpr int WC = 4;
  static constexpr int WARPS = WR * WC;
  static constexpr int THREADS = WARPS * 32;
  static constexpr int RW = N / WR;                   // rows per warp (32)
  static constexpr int CWc = N / WC;                  // complex columns per warp
  static constexpr int RG = RW / 8;                   // 8-row groups per warp
  static constexpr int CT = CWc / 4;                  // 4-complex-column tiles per warp (P1 n-tiles)
  static constexpr int CG = CWc / 8;                  // 8-complex-column groups per warp (P2 n-tiles)
  static constexpr int HS = N + 2;                    // H row stride in doubles  (row bytes == 16 mod 128)
  static constexpr int SS = N + 1;                    // sigma row stride in double2 (row bytes == 16 mod 128)
  static_assert(N % 32 == 0 && CWc % 8 == 0, "unsupported N");
  static_assert((HS * 8) % 128 == 16 && (SS * 16) % 128 == 16, "row padding");
};

template <int N>
struct LargeParams {
  RhsParams p;
  const int64_t* lptr;     // [nodes+1] CSR offsets into lent
  const int4* lent;        // link entries: x = neighbour slot, y = mode l, z = 0 ("+") or 1 ("-"), w = n_l
  const int32_t* mrows;    // [nodes][mrow] dense link rows {plus[W], minus[W], n[W], d_u}, as in kernels_mma.cu
  int mrow;                // ints per dense row
  const double* Hs;        // DEVICE [N][N]: H / hbar
  const double* delta;     // DEVICE [N]
  unsigned long long* tickets;
  unsigned long long ticket_base;
  double cP[kLargeMaxModes], cX[kLargeMaxModes], cO[kLargeMaxModes];   // as in kernels_hpipe.cu
};

__device__ __forceinline__ unsigned lsmem_u32(const void* ptr) {
  return (unsigned)__cvta_generic_to_shared(ptr);
}
__device__ __forceinline__ void lmbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lsmem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void lmbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lsmem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void lmbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LWAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra LWAIT_DONE;\n"
      "bra LWAIT_LOOP;\n"
      "LWAIT_DONE:\n"
      "}\n" ::"r"(lsmem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void lbulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes,
                                          unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(lsmem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(lsmem_u32(bar)) : "memory");
}
__device__ __forceinline__ void lbulk_prefetch_l2(const void* src_gmem, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
// D(8x8) += A(8x4) B(4x8), fp64 tensor core.  a: A[lane/4][lane%4]; b: B[lane%4][lane/4];
// c0, c1: C[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double neg(double v) { return -v; }
// 16-byte read-only load of *ptr, executed only if ok; otherwise the destination keeps its contents
__device__ __forceinline__ void ldg_if(double2& r, const double2* ptr, bool ok) {
  asm volatile("{\n"
      ".reg .pred p;\n"
      "setp.ne.s32 p, %3, 0;\n"
      "@p ld.global.nc.v2.f64 {%0, %1}, [%2];\n"
      "}\n" : "+d"(r.x), "+d"(r.y) : "l"(ptr), "r"((int)ok));
}

template <int N, bool HERM>
__global__ void __launch_bounds__(LargeCfg<N>::THREADS, 1)
rhs_large_kernel(const __grid_constant__ LargeParams<N> P) {
  using C = LargeCfg<N>;
  constexpr int NN = N * N, HS = C::HS, SS = C::SS, RG = C::RG, CT = C::CT, CG = C::CG;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  double* sH = reinterpret_cast<double*>(smem_raw);                           // [N][HS]  H / hbar
  double2* sS = reinterpret_cast<double2*>(sH + N * HS);                      // [N][SS]  sigma of the node
  double* sDelta = reinterpret_cast<double*>(sS + N * SS);                    // [N]
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(sDelta + N);
  int* sNode = reinterpret_cast<int*>(bar + 1);
  double* sSqrt = reinterpret_cast<double*>(sNode + 2);                       // [258] sqrt(n), n = 0..D+1 <= 256
  for (int e = threadIdx.x; e < 258; e += C::THREADS) sSqrt[e] = sqrt((double)e);

  for (int e = threadIdx.x; e < NN; e += C::THREADS) sH[(e / N) * HS + (e % N)] = P.Hs[e];
  for (int e = threadIdx.x; e < N; e += C::THREADS) sDelta[e] = P.delta[e];
  if (threadIdx.x == 0) {
    lmbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = lane >> 2, t = lane & 3;
  const int rho = (r >> 1) + 4 * (r & 1);             // fragment row r <-> matrix row offset {0,4,1,5,2,6,3,7}
  const int i0w = (warp / C::WC) * C::RW, j0w = (warp % C::WC) * C::CWc;
  const int nodes = p.nodes;

  // the node's sigma -> padded shared-memory rows; issued by warp 0 (lane 0 arms the mbarrier).  With no
  // node left lane 0 still completes the phase so that the waiting warps wake up and leave.
  auto load_sigma = [&](int node) {
    if (lane == 0) lmbar_expect_tx(bar, node < nodes ? (unsigned)NN * 16 : 0u);
    __syncwarp();
    if (node < nodes)
      for (int row = lane; row < N; row += 32)
        lbulk_g2s(sS + row * SS, p.x + (size_t)node * NN + (size_t)row * N, N * 16, bar);
  };
  auto draw = [&]() -> int {
    const unsigned long long tk = atomicAdd(P.tickets, 1ULL) - P.ticket_base;
    return tk < (unsigned long long)nodes ? (int)tk : nodes;
  };
  // Nodes are drawn TWO ahead: the ticket for the node after the next one is requested at the top of an iteration
  // and its value looked at only at the bottom, so that the atomic's round trip never stalls warp 0 (and, through
  // the CTA barrier, everyone else).  Every CTA ends with two failing draws.
  int next = nodes;                                   // the node after the one in flight (warp 0)
  if (warp == 0) {
    int first = 0;
    if (lane == 0) { first = draw(); next = draw(); *sNode = first; }
    first = __shfl_sync(0xffffffffu, first, 0);
    next = __shfl_sync(0xffffffffu, next, 0);
    load_sigma(first);
  }

  unsigned ph = 0;
  for (;;) {
    lmbar_wait(bar, ph);                              // sigma of the node has landed (or there is no node)
    ph ^= 1u;
    const int node = *reinterpret_cast<volatile int*>(sNode);
    if (node >= nodes) break;
    // warp 0 pulls the next node's sigma into L2 behind this node's arithmetic and requests a ticket
    unsigned long long traw = 0ULL;
    if (warp == 0 && lane == 0) {
      if (next < nodes) lbulk_prefetch_l2(p.x + (size_t)next * NN, (unsigned)NN * 16);
      traw = atomicAdd(P.tickets, 1ULL);
    }

    if (HERM) {
      // the NEXT node's dense link row -> L2; THIS node's neighbour rows (row b of sigma_{u +- e_l}, b the bath of
      // mode l) -> L2 behind the contraction, so that the coupling phase pays L2 round trips only
      if (warp == 2 && lane == 0 && next < nodes)
        lbulk_prefetch_l2(P.mrows + (size_t)next * P.mrow, (unsigned)P.mrow * 4);
      const int32_t* lr0 = P.mrows + (size_t)node * P.mrow;
      for (int q = threadIdx.x; q < 2 * p.W; q += C::THREADS) {
        const int idx = __ldg(lr0 + q);
        const int l = q < p.W ? q : q - p.W;
        if (idx >= 0) lbulk_prefetch_l2(p.x + (size_t)idx * NN + (size_t)(l / p.M) * N, (unsigned)N * 16);
      }
    }

    // ---- C = (H/hbar) sigma - sigma (H/hbar) on the FP64 tensor cores (Eq. 12) --------------------
    double2 acc[RG][CT];
#pragma unroll
    for (int rg = 0; rg < RG; ++rg)
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) acc[rg][ct] = make_double2(0.0, 0.0);

    const double* hArow = sH + (i0w + rho) * HS + 2 * t;                // P1 A: H[row][m0 + 2t, +1]
    const double* sBcol = reinterpret_cast<const double*>(sS + (2 * t) * SS + j0w + (r >> 1)) + (r & 1);   // P1 B
    const double2* sArow = sS + (i0w + rho) * SS + t;                    // P2 A: sigma[row][mm + t]
    const double* hBrow = sH + (j0w + rho) * HS + t;                     // P2 B: H[col pi(n)][mm + t]
#pragma unroll 1
    for (int m0 = 0; m0 < N; m0 += 8) {
      {  // P1: k-half 0 = rows m0+{0,2,4,6}, k-half 1 = rows m0+{1,3,5,7}
        double2 hA[RG];
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) hA[rg] = *reinterpret_cast<const double2*>(hArow + rg * 8 * HS + m0);
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const double b0 = sBcol[(size_t)(m0 * SS + 4 * ct) * 2];
          const double b1 = sBcol[(size_t)((m0 + 1) * SS + 4 * ct) * 2];
          // the two k-halves update the same accumulators: keep RG independent DMMAs between them
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) dmma(acc[rg][ct].x, acc[rg][ct].y, hA[rg].x, b0);
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) dmma(acc[rg][ct].x, acc[rg][ct].y, hA[rg].y, b1);
        }
      }
      if (!HERM)
#pragma unroll
      for (int h = 0; h < 2; ++h) {  // P2: natural k, two sub-steps of 4
        const int mm = m0 + 4 * h;
        double2 sA[RG];
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
          const double2 v = sArow[rg * 8 * SS + mm];
          sA[rg] = make_double2(neg(v.x), neg(v.y));
        }
#pragma unroll
        for (int cg = 0; cg < CG; ++cg) {
          const double hB = hBrow[cg * 8 * HS + mm];
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) {
            dmma(acc[rg][2 * cg].x, acc[rg][2 * cg + 1].x, sA[rg].x, hB);
            dmma(acc[rg][2 * cg].y, acc[rg][2 * cg + 1].y, sA[rg].y, hB);
          }
        }
      }
    }

    // Horner stage: this node's y is needed by the epilogue -- pull it into L2 now (prefetching it a whole node
    // ahead made it compete with the sigma tiles for L2: 1.5x the DRAM reads, profiles/r2_cfg5_large.md)
    if (warp == 1 && lane == 0 && p.horner && p.y != p.x) lbulk_prefetch_l2(p.y + (size_t)node * NN, (unsigned)NN * 16);

    // ---- k = -i C - (d_u + T) o sigma (Eq. 13-14, mask Eq. 24), in the fragment layout ------------
    //      (HERM: Z = -i P1 - (d_u + T)/2 o sigma)
    const double dd = p.damp[node];
#pragma unroll
    for (int rg = 0; rg < RG; ++rg) {
      const int row = i0w + 8 * rg + rho;
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) {
        const int col = j0w + 4 * ct + t;
        const double2 sv = sS[row * SS + col];
        double dt = dd + (row == col ? 0.0 : sDelta[row] + sDelta[col]);
        if (HERM) dt *= 0.5;
        const double2 c = acc[rg][ct];
        acc[rg][ct] = make_double2(fma(-dt, sv.x, c.y), fma(-dt, sv.y, -c.x));
      }
    }
    if (!HERM) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();                                // every warp is done with the node's sigma
      // ---- next node: start its TMA load (from L2) behind the rest of this node's work ------------
      if (warp == 0) {
        if (lane == 0) *sNode = next;
        load_sigma(next);
      }
    }

    // ---- couplings to sigma_{u +- e_l}: row b and column b of the neighbour (Eq. 15-17, 23, 25, 35-36) --
    //      (HERM: the row part only, added to Z; Z^dagger supplies the column part)
    if (HERM) {
      // Row-wise: a lane owns rows b = i0w + 8 rg + rho; row b is touched by the links of the modes of bath b only
      // (site map: bath b <-> state b), which it looks up in the node's dense link row and gathers all at once --
      // 2 M CT independent 16-byte loads per row, predicated on the link's existence.  (Walking the node's link list
      // instead made every warp step through ~W links one after the other: 5.2 of 28.0 ms per launch on config 5.)
      const int32_t* lr = P.mrows + (size_t)node * P.mrow;
      const int W = p.W, M = p.M;
      for (int kk = 0; kk < M; ++kk) {
        int up[RG], dn[RG], nn[RG];
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
          const int l = (i0w + 8 * rg + rho) * M + kk;
          up[rg] = __ldg(lr + l); dn[rg] = __ldg(lr + W + l); nn[rg] = __ldg(lr + 2 * W + l);
        }
        // "+" links (one per row below the top level): two rows' loads in flight at a time
#pragma unroll
        for (int r2 = 0; r2 < RG; r2 += 2) {
          double2 wu[2][CT];
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (r2 + h < RG) {
              const int b = i0w + 8 * (r2 + h) + rho;
              const double2* nu = p.x + (size_t)(up[r2 + h] < 0 ? 0 : up[r2 + h]) * NN + (size_t)b * N + j0w + t;
#pragma unroll
              for (int ct = 0; ct < CT; ++ct) { wu[h][ct] = make_double2(0.0, 0.0); ldg_if(wu[h][ct], nu + 4 * ct, up[r2 + h] >= 0); }
            }
          }
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (r2 + h < RG) {
              const int rg = r2 + h;
              const double a = sSqrt[nn[rg] + 1] * P.cP[(i0w + 8 * rg + rho) * M + kk];      // i a+
#pragma unroll
              for (int ct = 0; ct < CT; ++ct) {
                acc[rg][ct].x = fma(-a, wu[h][ct].y, acc[rg][ct].x);
                acc[rg][ct].y = fma(a, wu[h][ct].x, acc[rg][ct].y);
              }
            }
          }
        }
        // "-" links exist only where n_l > 0 (at most D per node): skipped when no lane of the warp has one
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
          if (__any_sync(0xffffffffu, dn[rg] >= 0)) {
            const int b = i0w + 8 * rg + rho, l = b * M + kk;
            const double2* nd = p.x + (size_t)(dn[rg] < 0 ? 0 : dn[rg]) * NN + (size_t)b * N + j0w + t;
            double2 wd[CT];
#pragma unroll
            for (int ct = 0; ct < CT; ++ct) { wd[ct] = make_double2(0.0, 0.0); ldg_if(wd[ct], nd + 4 * ct, dn[rg] >= 0); }
            const double sn = sSqrt[nn[rg]], fx = sn * P.cX[l], fo = sn * P.cO[l];              // i a-x + a-o
#pragma unroll
            for (int ct = 0; ct < CT; ++ct) {
              acc[rg][ct].x = fma(fo, wd[ct].x, fma(-fx, wd[ct].y, acc[rg][ct].x));
              acc[rg][ct].y = fma(fo, wd[ct].y, fma(fx, wd[ct].x, acc[rg][ct].y));
            }
          }
        }
      }
    } else {
      const int64_t e0 = P.lptr[node], e1 = P.lptr[node + 1];
      for (int64_t e = e0; e < e1; ++e) {
        const int4 ent = P.lent[e];
        const int l = ent.y, b = l / p.M;
        // row factor fr (elements (b, j)) and column factor fc (elements (i, b)) of this link
        double frx, fry, fcy;
        if (ent.z == 0) {                             // "+":  i a+ (delta_ib - delta_bj)
          const double a = sSqrt[ent.w + 1] * P.cP[l];
          frx = 0.0; fry = a; fcy = -a;
        } else {                                      // "-":  i a-x (delta_ib - delta_bj) + a-o (delta_ib + delta_bj)
          const double sn = sSqrt[ent.w];
          frx = sn * P.cO[l]; fry = sn * P.cX[l]; fcy = -fry;
        }
        const double2* nb = p.x + (size_t)ent.x * NN;
        if (b >= i0w && b < i0w + C::RW) {            // warp-uniform: this warp owns part of row b
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) {
            if (i0w + 8 * rg + rho == b) {
#pragma unroll
              for (int ct = 0; ct < CT; ++ct) {
                const double2 w = __ldg(nb + (size_t)b * N + (j0w + 4 * ct + t));
                acc[rg][ct].x = fma(frx, w.x, fma(-fry, w.y, acc[rg][ct].x));
                acc[rg][ct].y = fma(frx, w.y, fma(fry, w.x, acc[rg][ct].y));
              }
            }
          }
        }
        if (!HERM && b >= j0w && b < j0w + C::CWc) {  // warp-uniform: this warp owns part of column b
#pragma unroll
          for (int ct = 0; ct < CT; ++ct) {
            if (j0w + 4 * ct + t == b) {
#pragma unroll
              for (int rg = 0; rg < RG; ++rg) {
                const double2 w = __ldg(nb + (size_t)(i0w + 8 * rg + rho) * N + b);
                acc[rg][ct].x = fma(frx, w.x, fma(-fcy, w.y, acc[rg][ct].x));
                acc[rg][ct].y = fma(frx, w.y, fma(fcy, w.x, acc[rg][ct].y));
              }
            }
          }
        }
      }
    }

    if (HERM) {
      // ---- k = Z + Z^dagger through the sigma tile's shared memory (the contraction is done with it) ----
      __syncthreads();                                // every warp is done with the node's sigma
#pragma unroll
      for (int rg = 0; rg < RG; ++rg)
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) sS[(i0w + 8 * rg + rho) * SS + j0w + 4 * ct + t] = acc[rg][ct];
      __syncthreads();
#pragma unroll
      for (int rg = 0; rg < RG; ++rg)
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const double2 zt = sS[(j0w + 4 * ct + t) * SS + i0w + 8 * rg + rho];     // Z[col][row]
          acc[rg][ct].x += zt.x;
          acc[rg][ct].y -= zt.y;
        }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();                                // the tile may be overwritten
      if (warp == 0) {
        if (lane == 0) *sNode = next;
        load_sigma(next);
      }
    }

    // ---- fused RK4 stage epilogue straight from the fragment layout ------------------------------------
    const size_t nbase = (size_t)node * NN;
#pragma unroll
    for (int rg = 0; rg < RG; ++rg) {
      const size_t rbase = nbase + (size_t)(i0w + 8 * rg + rho) * N + j0w + t;
      if (p.rhs_only) {
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) p.out_acc[rbase + 4 * ct] = acc[rg][ct];
      } else if (p.horner) {
        // Horner stage (R6): w' = y + ax k; no running sum, nothing but y is loaded
        double2 yv[CT];
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) yv[ct] = p.y[rbase + 4 * ct];
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const double2 kv = acc[rg][ct];
          p.out_x[rbase + 4 * ct] = make_double2(fma(p.ax, kv.x, yv[ct].x), fma(p.ax, kv.y, yv[ct].y));
        }
      } else {
        double2 yv[CT], av[CT];
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          av[ct] = p.acc_in[rbase + 4 * ct];
          if (p.out_x) yv[ct] = p.y[rbase + 4 * ct];
        }
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const double2 kv = acc[rg][ct];
          if (p.out_x) p.out_x[rbase + 4 * ct] = make_double2(fma(p.ax, kv.x, yv[ct].x), fma(p.ax, kv.y, yv[ct].y));
          p.out_acc[rbase + 4 * ct] = make_double2(fma(p.bx, kv.x, av[ct].x), fma(p.bx, kv.y, av[ct].y));
        }
      }
    }
    if (warp == 0) {                                  // the ticket requested at the top has long arrived
      const unsigned long long tk = traw - P.ticket_base;
      next = __shfl_sync(0xffffffffu, tk < (unsigned long long)nodes ? (int)tk : nodes, 0);
    }
  }
}

template <int N>
size_t large_smem() {
  using C = LargeCfg<N>;
  return (size_t)N * C::HS * 8 + (size_t)N * C::SS * 16 + (size_t)N * 8 + 8 + 16 + 258 * 8;
}

template <int N, bool HERM>
cudaError_t launch_large_t(const RhsParams& p, const int64_t* lptr, const int4* lent, const int32_t* mrows, int mrow,
                           const double* Hs_dev,
                           const double* delta_dev, const double* a_plus, const double* a_minus_x,
                           const double* a_minus_o, int sms, unsigned long long* tickets,
                           unsigned long long* ticket_base, cudaStream_t s) {
  using C = LargeCfg<N>;
  if (p.W > kLargeMaxModes) return cudaErrorInvalidValue;
  LargeParams<N> P;
  P.p = p; P.lptr = lptr; P.lent = lent; P.mrows = mrows; P.mrow = mrow; P.Hs = Hs_dev; P.delta = delta_dev;
  const int D1 = p.D + 1;
  for (int l = 0; l < kLargeMaxModes; ++l) {
    const bool on = l < p.W && p.D >= 1;
    P.cP[l] = on ? a_plus[(size_t)l * D1] : 0.0;
    P.cX[l] = on ? a_minus_x[(size_t)l * D1 + 1] : 0.0;
    P.cO[l] = on ? a_minus_o[(size_t)l * D1 + 1] : 0.0;
  }
  const size_t smem = large_smem<N>();
  static bool configured_on[64] = {};     // per device: the attribute belongs to the device's context (one flag per instantiation)
  int dev_ = 0;
  cudaGetDevice(&dev_);
  bool& configured = configured_on[dev_ & 63];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_large_kernel<N, HERM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  int grid = sms < p.nodes ? sms : p.nodes;
  if (grid < 1) grid = 1;
  P.tickets = tickets;
  P.ticket_base = *ticket_base;
  rhs_large_kernel<N, HERM><<<grid, C::THREADS, smem, s>>>(P);
  const cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    *ticket_base += (unsigned long long)p.nodes + 2ULL * (unsigned long long)grid;   // two failing draws per CTA
  } else {                                 // nothing ran: keep host base and device counter in step
    cudaMemsetAsync(tickets, 0, sizeof(unsigned long long), s);
    *ticket_base = 0;
  }
  return e;
}

}  // namespace

bool large_supported(int N, int W) { return (N == 32 || N == 64 || N == 96) && W <= kLargeMaxModes; }

cudaError_t launch_rhs_large(const RhsParams& p, const int64_t* lptr, const void* lent, const int32_t* mrows, int mrow,
                             const double* Hs_dev,
                             const double* delta_dev, const double* a_plus, const double* a_minus_x,
                             const double* a_minus_o, int hermitian, int sms, unsigned long long* tickets,
                             unsigned long long* ticket_base, cudaStream_t s) {
  const int4* le = reinterpret_cast<const int4*>(lent);
#define HEOM_LARGE_CASE(n)                                                                                              \
  case n:                                                                                                               \
    return hermitian ? launch_large_t<n, true>(p, lptr, le, mrows, mrow, Hs_dev, delta_dev, a_plus, a_minus_x, a_minus_o, sms,       \
                                               tickets, ticket_base, s)                                                 \
                     : launch_large_t<n, false>(p, lptr, le, mrows, mrow, Hs_dev, delta_dev, a_plus, a_minus_x, a_minus_o, sms,      \
                                                tickets, ticket_base, s);
  switch (p.N) {
    HEOM_LARGE_CASE(32) HEOM_LARGE_CASE(64) HEOM_LARGE_CASE(96)
    default: return cudaErrorInvalidValue;
  }
#undef HEOM_LARGE_CASE
}

}  // namespace heom
