// kernels_mma.cu -- sm_100a FP64 tensor-core kernel for MID-SIZE and GENERAL systems: 17 <= N <= 96 states
// (padded to NP = 32, 48, 64, 80 or 96), any system-bath operator of the paper's form (bath b couples through
// the projectors on a SET of states, several baths may share a state: P:84, the sums over s of Eq. 14-17;
// the two-exciton manifold of Eq. 54 with N = 29 for FMO), real or complex Hermitian H (the RWA
// field coupling of Eq. 51).  The HEOM right-hand side (Eq. 12-17 with Eq. 23-25, 35-36) with the RK4 stage
// combination fused into its epilogue.
//
// One CTA works on one node at a time (nodes drawn from a global ticket counter); several CTAs share an SM
// (as many as shared memory allows, up to 4), so that one CTA's link gathers and epilogue overlap another's
// contraction.
//   * H/hbar (real part, and imaginary part when CPLX) stays in shared memory, zero-padded to NP x NP; the
//     node's sigma is streamed into zero-padded shared-memory rows by the TMA (cp.async.bulk, one copy per
//     matrix row, completion on an mbarrier).
//   * C = (H/hbar) sigma - sigma (H/hbar) runs on the FP64 tensor cores (mma.sync.m8n8k4.f64, SASS
//     DMMA.8x8x4 -- tcgen05 has no FP64 kind).  Fragment layout as in kernels_large.cu: rows permuted
//     {0,4,1,5,2,6,3,7}, P1 = H sigma over sigma as an NP x 2NP real matrix with the k index split into even
//     and odd rows, P2 = sigma H with its column order permuted the same way, so that every lane owns whole
//     complex elements and both products accumulate into the same registers.  CPLX adds the two products
//     with Im H: (i Hi) sigma uses the operand (-Im sigma, Re sigma), sigma (i Hi) the operand swap with
//     -Hi^T = Hi (antisymmetric).
//   * k = -i C - (d_u + T) o sigma with the Eq. 14 table T read through the read-only cache; the couplings
//     to sigma_{u +- e_l} are gathered ELEMENT-wise: element (i,j) is touched by the links of the baths whose
//     state set contains i or j (state -> baths lists and membership bits in shared memory), factor
//     i a (q_i - q_j) + a_o (q_i + q_j)  (Eq. 23, 25 summed over the bath's states).  A thread therefore
//     looks its rows' and columns' baths up in the node's dense link row {plus[W], minus[W], n[W], d_u}
//     (staged in shared memory two nodes ahead with cp.async) and issues all its gathers independently of
//     one another -- walking the node's links one after the other cost one L2 round trip per link;
//   * fused epilogue straight from the fragment layout: Horner form w' = y + ax k (R6), the
//     classical form with a running sum, or the bare right-hand side.
#include "kernels.cuh"

#include <cmath>
#include <cstring>

namespace heom {
namespace {

constexpr int kMmaMaxModes = 288;   // W of the constant-bank coupling tables
constexpr int kMmaMaxBaths = 96;
constexpr int kMmaMaxMember = 256;  // total (state, bath) memberships in the state -> baths lists

template <int NP>
struct MmaCfg {
#ifndef HEOM_MMA_ROWS
#define HEOM_MMA_ROWS 16
#endif
  static constexpr int WR = (NP == 96) ? 3 : NP / HEOM_MMA_ROWS;   // warp grid WR x WC (16-row warp tiles; 8-row tiles measured 1.4x slower: no A-fragment reuse)
  static constexpr int WC = (NP == 96) ? 4 : 2;
  static constexpr int WARPS = WR * WC;
  static constexpr int THREADS = WARPS * 32;
  static constexpr int RW = NP / WR;                  // rows per warp (16, or 32 for NP = 96)
  static constexpr int CWc = NP / WC;                 // complex columns per warp
  static constexpr int RG = RW / 8;                   // 8-row groups per warp
  static constexpr int CT = CWc / 4;                  // 4-complex-column tiles per warp (P1 n-tiles)
  static constexpr int CG = CWc / 8;                  // 8-complex-column groups per warp (P2 n-tiles)
  static constexpr int HS = NP + 2;                   // H row stride in doubles  (row bytes == 16 mod 128)
  static constexpr int SS = NP + 1;                   // sigma row stride in double2 (row bytes == 16 mod 128)
  // small problems leave shared memory free: a second sigma tile lets the next node's TMA load run behind this
  // node's contraction instead of behind its gathers and epilogue only
  static constexpr bool DB = NP <= 48;
  static_assert(NP % 16 == 0 && RW % 8 == 0 && CWc % 8 == 0, "unsupported NP");
  static_assert((HS * 8) % 128 == 16 && (SS * 16) % 128 == 16, "row padding");
};

template <int NP, bool CPLX>
constexpr size_t mma_smem_bytes() {
  using C = MmaCfg<NP>;
  // without the three staged link rows (3 * mrow * 4 bytes, added at launch)
  return (size_t)NP * C::HS * 8 * (CPLX ? 2 : 1) + (size_t)NP * C::SS * 16 * (C::DB ? 2 : 1) + (size_t)kMmaMaxBaths * 16 +
         (size_t)(NP + 4 + kMmaMaxMember) * 4 + 16 + 16 + 258 * 8;
}
template <int NP, bool CPLX>
constexpr int mma_ctas_per_sm() {
  constexpr size_t per = mma_smem_bytes<NP, CPLX>() + 1024 + 1024;     // + link rows, the runtime's per-CTA reservation
  constexpr int by_smem = (int)((size_t)227 * 1024 / per);
  constexpr int by_threads = 512 / MmaCfg<NP>::THREADS;              // >= 128 registers per thread
  constexpr int m = by_smem < by_threads ? by_smem : by_threads;
  return m < 1 ? 1 : (m > 4 ? 4 : m);
}

struct MmaParams {
  RhsParams p;
  const int32_t* mrows;    // [nodes][mrow] dense link rows: plus[W], minus[W], n[W] (int32), d_u (double), padding
  int mrow;                // ints per row (multiple of 4)
  unsigned long long* tickets;
  unsigned long long ticket_base;
  double cP[kMmaMaxModes], cX[kMmaMaxModes], cO[kMmaMaxModes];   // as in kernels_hpipe.cu
};

__device__ __forceinline__ unsigned msmem_u32(const void* ptr) { return (unsigned)__cvta_generic_to_shared(ptr); }
__device__ __forceinline__ void mmbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(msmem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mmbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(msmem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mmbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MWAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MWAIT_DONE;\n"
      "bra MWAIT_LOOP;\n"
      "MWAIT_DONE:\n"
      "}\n" ::"r"(msmem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(msmem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(msmem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbulk_prefetch_l2(const void* src_gmem, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
// D(8x8) += A(8x4) B(4x8), fp64 tensor core.  a: A[lane/4][lane%4]; b: B[lane%4][lane/4];
// c0, c1: C[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void mdmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NP, bool CPLX, bool HERM>
__global__ void __launch_bounds__(MmaCfg<NP>::THREADS, mma_ctas_per_sm<NP, CPLX>())
rhs_mma_kernel(const __grid_constant__ MmaParams P) {
  using C = MmaCfg<NP>;
  constexpr int HS = C::HS, SS = C::SS, RG = C::RG, CT = C::CT, CG = C::CG;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int N = p.N, NN = N * N;
  double* sH = reinterpret_cast<double*>(smem_raw);                           // [NP][HS]  Re H / hbar
  double* sHi = sH + (CPLX ? NP * HS : 0);                                    // [NP][HS]  Im H / hbar (CPLX)
  constexpr bool DB = C::DB;
  double2* sS0 = reinterpret_cast<double2*>(sHi + NP * HS);                   // [DB ? 2 : 1][NP][SS]  sigma tile(s)
  unsigned* sMask = reinterpret_cast<unsigned*>(sS0 + (DB ? 2 : 1) * NP * SS);   // [kMmaMaxBaths][4] membership bits
  int* sSptr = reinterpret_cast<int*>(sMask + 4 * kMmaMaxBaths);               // [NP + 4] state -> baths CSR offsets
  int* sSbl = sSptr + NP + 4;                                                  // [kMmaMaxMember] bath indices
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(sSbl + kMmaMaxMember);   // [2]
  int* sNode = reinterpret_cast<int*>(bar + 2);                                                  // [2] (+ padding)
  double* sSqrt = reinterpret_cast<double*>(sNode + 4);                       // [258] sqrt(n), n = 0..D+1 <= 256
  int32_t* sRows = reinterpret_cast<int32_t*>(sSqrt + 258);                   // [3][mrow] staged link rows
  const int mrow = P.mrow, W = p.W;
  for (int e = threadIdx.x; e < 258; e += C::THREADS) sSqrt[e] = sqrt((double)e);
  for (int e = threadIdx.x; e < NP + 4; e += C::THREADS) sSptr[e] = p.sptr[e < N ? e : N];
  for (int e = threadIdx.x; e < kMmaMaxMember; e += C::THREADS) sSbl[e] = e < p.sptr[N] ? p.sbl[e] : 0;

  for (int e = threadIdx.x; e < NP * HS; e += C::THREADS) {
    const int i = e / HS, j = e % HS;
    const bool in = i < N && j < N;
    sH[e] = in ? p.H[i * N + j] * p.inv_hbar : 0.0;
    if (CPLX) sHi[e] = (in && p.Him) ? p.Him[i * N + j] * p.inv_hbar : 0.0;
  }
  for (int e = threadIdx.x; e < (DB ? 2 : 1) * NP * SS; e += C::THREADS) sS0[e] = make_double2(0.0, 0.0);   // padding stays zero
  for (int e = threadIdx.x; e < 4 * kMmaMaxBaths; e += C::THREADS) sMask[e] = e < 4 * p.B ? p.bmask[e] : 0u;
  if (threadIdx.x == 0) {
    mmbar_init(bar, 1);
    mmbar_init(bar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zero fill precedes the bulk copies
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = lane >> 2, t = lane & 3;
  const int rho = (r >> 1) + 4 * (r & 1);             // fragment row r <-> matrix row offset {0,4,1,5,2,6,3,7}
  const int i0w = (warp / C::WC) * C::RW, j0w = (warp % C::WC) * C::CWc;
  const int nodes = p.nodes;

  auto load_sigma = [&](int node, int buf) {
    if (lane == 0) mmbar_expect_tx(bar + buf, node < nodes ? (unsigned)NN * 16 : 0u);
    __syncwarp();
    if (node < nodes)
      for (int row = lane; row < N; row += 32)
        mbulk_g2s(sS0 + buf * NP * SS + row * SS, p.x + (size_t)node * NN + (size_t)row * N, (unsigned)N * 16, bar + buf);
  };
  auto draw = [&]() -> int {
    const unsigned long long tk = atomicAdd(P.tickets, 1ULL) - P.ticket_base;
    return tk < (unsigned long long)nodes ? (int)tk : nodes;
  };
  // warp 0 stages a node's link row with 16-byte cp.async copies into one of THREE buffers: the next node's row is
  // requested at the top of an iteration (its buffer was last read two iterations ago, which every warp had left
  // before the barrier warp 0 has passed since) and waited for before this iteration's barrier
  auto stage_row = [&](int node, int buf) {
    if (node < nodes) {
      const int32_t* src = P.mrows + (size_t)node * mrow;
      const unsigned dst = msmem_u32(sRows + buf * mrow);
      for (int c = lane; c < mrow / 4; c += 32)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * c), "l"(src + 4 * c) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // Nodes are drawn TWO ahead (as in kernels_large.cu): the ticket requested at the top of an iteration is looked at
  // at its bottom, so the atomic's round trip never stalls warp 0.  Every CTA ends with two failing draws.
  int next = nodes;                                   // the node after the one in flight (warp 0)
  if (warp == 0) {
    int first = 0;
    if (lane == 0) { first = draw(); next = draw(); sNode[0] = first; }
    first = __shfl_sync(0xffffffffu, first, 0);
    next = __shfl_sync(0xffffffffu, next, 0);
    load_sigma(first, 0);
    stage_row(first, 0);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  }
  __syncthreads();

  // Eq. 14 table values of this thread's elements are the same for every node: hoisted when the tile is small
  constexpr bool T_IN_REGS = RG * CT <= 12;
  double tt[T_IN_REGS ? RG * CT : 1];
  if (T_IN_REGS) {
#pragma unroll
    for (int rg = 0; rg < RG; ++rg)
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) {
        const int row = i0w + 8 * rg + rho, col = j0w + 4 * ct + t;
        tt[rg * CT + ct] = (row < N && col < N) ? __ldg(p.Tterm + row * N + col) : 0.0;
      }
  }

  unsigned ph = 0;                                    // bit b: phase of bar[b]
  int lbuf = 0;                                       // link-row buffer (of three) of the node in flight
  int cur = 0;                                        // sigma tile / mbarrier / sNode slot of the node in flight
  for (;;) {
    mmbar_wait(bar + cur, (ph >> cur) & 1u);          // sigma of the node has landed (or there is no node)
    ph ^= 1u << cur;
    const int node = *reinterpret_cast<volatile int*>(sNode + cur);
    if (node >= nodes) break;
    const double2* sS = sS0 + cur * NP * SS;
    unsigned long long traw = 0ULL;
    if (warp == 0) {
      if (DB) {
        // the other tile was last read before the previous node's CTA barrier: the next node's sigma streams into
        // it behind this node's contraction
        if (lane == 0) sNode[cur ^ 1] = next;
        load_sigma(next, cur ^ 1);
      }
      if (lane == 0) {
        if (next < nodes) {
          mbulk_prefetch_l2(p.x + (size_t)next * NN, (unsigned)NN * 16);
          if (p.horner && p.y != p.x) mbulk_prefetch_l2(p.y + (size_t)next * NN, (unsigned)NN * 16);
        }
        traw = atomicAdd(P.tickets, 1ULL);
      }
      stage_row(next, lbuf == 2 ? 0 : lbuf + 1);      // in flight behind this node's contraction
    }

    // ---- C = (H/hbar) sigma - sigma (H/hbar) on the FP64 tensor cores (Eq. 12) --------------------
    double2 acc[RG][CT];
#pragma unroll
    for (int rg = 0; rg < RG; ++rg)
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) acc[rg][ct] = make_double2(0.0, 0.0);

    const int hA_off = (i0w + rho) * HS + 2 * t;                         // P1 A: H[row][m0 + 2t, +1]
    const double* sBcol = reinterpret_cast<const double*>(sS + (2 * t) * SS + j0w + (r >> 1)) + (r & 1);   // P1 B
    const double2* sArow = sS + (i0w + rho) * SS + t;                    // P2 A: sigma[row][mm + t]
    const int hB_off = (j0w + rho) * HS + t;                             // P2 B: H[col pi(n)][mm + t]
#pragma unroll 1
    for (int m0 = 0; m0 < NP; m0 += 8) {
      {  // P1: k-half 0 = rows m0+{0,2,4,6}, k-half 1 = rows m0+{1,3,5,7}
        double2 hA[RG], gA[CPLX ? RG : 1];
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
          hA[rg] = *reinterpret_cast<const double2*>(sH + hA_off + rg * 8 * HS + m0);
          if (CPLX) gA[rg] = *reinterpret_cast<const double2*>(sHi + hA_off + rg * 8 * HS + m0);
        }
        // all B fragments first, then the two k-halves one after the other: RG*CT independent DMMAs lie between two
        // updates of the same accumulator
        double b0[CT], b1[CT];
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          b0[ct] = sBcol[(size_t)(m0 * SS + 4 * ct) * 2];
          b1[ct] = sBcol[(size_t)((m0 + 1) * SS + 4 * ct) * 2];
        }
#pragma unroll
        for (int ct = 0; ct < CT; ++ct)
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) mdmma(acc[rg][ct].x, acc[rg][ct].y, hA[rg].x, b0[ct]);
#pragma unroll
        for (int ct = 0; ct < CT; ++ct)
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) mdmma(acc[rg][ct].x, acc[rg][ct].y, hA[rg].y, b1[ct]);
        if (CPLX) {
          // (i Hi) sigma: operand (-Im sigma, Re sigma) = the lane's OTHER component, sign by parity
          const double* other = (r & 1) ? sBcol - 1 : sBcol + 1;
          const double sg = (r & 1) ? 1.0 : -1.0;
#pragma unroll
          for (int ct = 0; ct < CT; ++ct) {
            b0[ct] = sg * other[(size_t)(m0 * SS + 4 * ct) * 2];
            b1[ct] = sg * other[(size_t)((m0 + 1) * SS + 4 * ct) * 2];
          }
#pragma unroll
          for (int ct = 0; ct < CT; ++ct)
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) mdmma(acc[rg][ct].x, acc[rg][ct].y, gA[rg].x, b0[ct]);
#pragma unroll
          for (int ct = 0; ct < CT; ++ct)
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) mdmma(acc[rg][ct].x, acc[rg][ct].y, gA[rg].y, b1[ct]);
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
          sA[rg] = make_double2(-v.x, -v.y);
        }
#pragma unroll
        for (int cg = 0; cg < CG; ++cg) {
          const double hB = sH[hB_off + cg * 8 * HS + mm];             // Hr[mm+t][col] = Hr[col][mm+t]
#pragma unroll
          for (int rg = 0; rg < RG; ++rg) {
            mdmma(acc[rg][2 * cg].x, acc[rg][2 * cg + 1].x, sA[rg].x, hB);
            mdmma(acc[rg][2 * cg].y, acc[rg][2 * cg + 1].y, sA[rg].y, hB);
          }
          if (CPLX) {
            // -sigma (i Hi): Re -= -(s.y Hi) ... with Hi[mm+t][col] = -Hi[col][mm+t] =: gB
            //   Re(-s i g) = +s.y g,  Im(-s i g) = -s.x g;  sA holds -s, so Re = -sA.y g, Im = sA.x g
            const double gB = -sHi[hB_off + cg * 8 * HS + mm];
#pragma unroll
            for (int rg = 0; rg < RG; ++rg) {
              mdmma(acc[rg][2 * cg].x, acc[rg][2 * cg + 1].x, -sA[rg].y, gB);
              mdmma(acc[rg][2 * cg].y, acc[rg][2 * cg + 1].y, sA[rg].x, gB);
            }
          }
        }
      }
    }

    // ---- k = -i C - (d_u + T) o sigma (Eq. 13-14), in the fragment layout ---------------------------
    const int32_t* srow = sRows + lbuf * mrow;       // this node's plus[W], minus[W], n[W], d_u
    const double dd = *reinterpret_cast<const double*>(srow + 3 * W + (W & 1));
#pragma unroll
    for (int rg = 0; rg < RG; ++rg) {
      const int row = i0w + 8 * rg + rho;
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) {
        const int col = j0w + 4 * ct + t;
        const double2 sv = sS[row * SS + col];
        const double tv = T_IN_REGS ? tt[rg * CT + ct] : ((row < N && col < N) ? __ldg(p.Tterm + row * N + col) : 0.0);
        const double dt = HERM ? 0.5 * (dd + tv) : dd + tv;   // HERM: Z = -i P1 - (d_u + T)/2 o sigma
        const double2 c = acc[rg][ct];
        acc[rg][ct] = make_double2(fma(-dt, sv.x, c.y), fma(-dt, sv.y, -c.x));
      }
    }
    if (warp == 0) asm volatile("cp.async.wait_group 0;" ::: "memory");   // the next node's link row has landed
    if (!HERM) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();                                // every warp is done with the node's sigma
      // ---- next node: start its TMA load behind the rest of this node's work -------------------------
      if (!DB && warp == 0) {
        if (lane == 0) sNode[0] = next;
        load_sigma(next, 0);
      }
    }

    // ---- couplings to sigma_{u +- e_l} (Eq. 15-17, 23, 25, 35-36, summed over the bath's states) ------
    // Element (i,j) takes, from every link of a bath b, the factor i fx (q_i - q_j) + fo (q_i + q_j), q = membership
    // of b's state set.  Row part: the baths that contain the thread's row i act on all its columns (q_i = 1);
    // column part: the baths that contain its column j and not the row (q_i = 0, q_j = 1).  HERM: the row part with
    // (fo + i fx) only -- Z^dagger supplies the rest.  Every gather depends on the staged link row alone.
    {
      const int32_t* spl = srow;
      const int32_t* smi = srow + W;
      const int32_t* snn = srow + 2 * W;
      const int M = p.M;
#pragma unroll
      for (int rg = 0; rg < RG; ++rg) {
        const int row = i0w + 8 * rg + rho;
        if (row >= N) continue;
        for (int e = sSptr[row]; e < sSptr[row + 1]; ++e) {
          const int b = sSbl[e];
          const unsigned long long cbits =
              (((unsigned long long)sMask[b * 4 + (j0w >> 5) + 1] << 32) | sMask[b * 4 + (j0w >> 5)]) >> (j0w & 31);
          for (int k2 = 0; k2 < 2 * M; ++k2) {       // the bath's modes, "+" then "-" link of each
            const int l = b * M + (k2 >> 1);
            const int slot = (k2 & 1) ? smi[l] : spl[l];
            if (slot < 0) continue;
            const int n = snn[l];
            double fx, fo;
            if (k2 & 1) { const double sn = sSqrt[n]; fx = sn * P.cX[l]; fo = sn * P.cO[l]; }   // "-"
            else { fx = sSqrt[n + 1] * P.cP[l]; fo = 0.0; }                                     // "+"
            const double2* nbrow = p.x + (size_t)slot * NN + (size_t)row * N;
#pragma unroll
            for (int ct = 0; ct < CT; ++ct) {
              const int col = j0w + 4 * ct + t;
              if (col < N) {
                const bool qj = !HERM && ((cbits >> (4 * ct + t)) & 1ULL);
                const double fr = qj ? 2.0 * fo : fo, fi = qj ? 0.0 : fx;
                const double2 w = __ldg(nbrow + col);
                acc[rg][ct].x = fma(fr, w.x, fma(-fi, w.y, acc[rg][ct].x));
                acc[rg][ct].y = fma(fr, w.y, fma(fi, w.x, acc[rg][ct].y));
              }
            }
          }
        }
      }
      if (!HERM) {
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const int col = j0w + 4 * ct + t;
          if (col >= N) continue;
          for (int e = sSptr[col]; e < sSptr[col + 1]; ++e) {
            const int b = sSbl[e];
            const unsigned rbits = sMask[b * 4 + (i0w >> 5)] >> (i0w & 31);
            for (int k2 = 0; k2 < 2 * M; ++k2) {
              const int l = b * M + (k2 >> 1);
              const int slot = (k2 & 1) ? smi[l] : spl[l];
              if (slot < 0) continue;
              const int n = snn[l];
              double fx, fo;
              if (k2 & 1) { const double sn = sSqrt[n]; fx = sn * P.cX[l]; fo = sn * P.cO[l]; }
              else { fx = sSqrt[n + 1] * P.cP[l]; fo = 0.0; }
              const double2* nbcol = p.x + (size_t)slot * NN + col;
#pragma unroll
              for (int rg = 0; rg < RG; ++rg) {
                const int row = i0w + 8 * rg + rho;
                if (row < N && !((rbits >> (8 * rg + rho)) & 1u)) {   // rows inside the set were done above
                  const double2 w = __ldg(nbcol + (size_t)row * N);
                  acc[rg][ct].x = fma(fo, w.x, fma(fx, w.y, acc[rg][ct].x));      // (fo - i fx) w
                  acc[rg][ct].y = fma(fo, w.y, fma(-fx, w.x, acc[rg][ct].y));
                }
              }
            }
          }
        }
      }
    }

    if (HERM) {
      // ---- k = Z + Z^dagger through the sigma tile (every warp is done with it after the first barrier) ----
      double2* sZ = sS0 + cur * NP * SS;
      __syncthreads();
#pragma unroll
      for (int rg = 0; rg < RG; ++rg)
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) sZ[(i0w + 8 * rg + rho) * SS + j0w + 4 * ct + t] = acc[rg][ct];
      __syncthreads();
#pragma unroll
      for (int rg = 0; rg < RG; ++rg)
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const double2 zt = sZ[(j0w + 4 * ct + t) * SS + i0w + 8 * rg + rho];     // Z[col][row]
          acc[rg][ct].x += zt.x;
          acc[rg][ct].y -= zt.y;
        }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncthreads();                                // the tile may be overwritten by a TMA load
      if (!DB && warp == 0) {
        if (lane == 0) sNode[0] = next;
        load_sigma(next, 0);
      }
    }
    lbuf = lbuf == 2 ? 0 : lbuf + 1;
    if (DB) cur ^= 1;

    // ---- fused RK4 stage epilogue straight from the fragment layout ------------------------------------
    const size_t nbase = (size_t)node * NN;
#pragma unroll
    for (int rg = 0; rg < RG; ++rg) {
      const int row = i0w + 8 * rg + rho;
      if (row >= N) continue;
      const size_t rbase = nbase + (size_t)row * N;
      if (p.rhs_only) {
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {
          const int col = j0w + 4 * ct + t;
          if (col < N) p.out_acc[rbase + col] = acc[rg][ct];
        }
      } else if (p.horner) {
        constexpr int CH = CT % 4 == 0 ? 4 : (CT % 3 == 0 ? 3 : 2);   // tiles per batch of loads
#pragma unroll
        for (int c0 = 0; c0 < CT; c0 += CH) {
          double2 yv[CH];
#pragma unroll
          for (int c = 0; c < CH; ++c) {
            const int col = j0w + 4 * (c0 + c) + t;
            yv[c] = col < N ? p.y[rbase + col] : make_double2(0.0, 0.0);
          }
#pragma unroll
          for (int c = 0; c < CH; ++c) {
            const int col = j0w + 4 * (c0 + c) + t;
            const double2 kv = acc[rg][c0 + c];
            if (col < N) p.out_x[rbase + col] = make_double2(fma(p.ax, kv.x, yv[c].x), fma(p.ax, kv.y, yv[c].y));
          }
        }
      } else {
#pragma unroll
        for (int ct = 0; ct < CT; ++ct) {       // classical form: not the fast path, one element at a time
          const int col = j0w + 4 * ct + t;
          const double2 kv = acc[rg][ct];
          if (col < N) {
            const double2 av = p.acc_in[rbase + col];
            if (p.out_x) {
              const double2 yv = p.y[rbase + col];
              p.out_x[rbase + col] = make_double2(fma(p.ax, kv.x, yv.x), fma(p.ax, kv.y, yv.y));
            }
            p.out_acc[rbase + col] = make_double2(fma(p.bx, kv.x, av.x), fma(p.bx, kv.y, av.y));
          }
        }
      }
    }
    if (warp == 0) {                                  // the ticket requested at the top has long arrived
      const unsigned long long tk = traw - P.ticket_base;
      next = __shfl_sync(0xffffffffu, tk < (unsigned long long)nodes ? (int)tk : nodes, 0);
    }
  }
}

template <int NP, bool CPLX, bool HERM>
cudaError_t launch_mma_t(const RhsParams& p, const int32_t* mrows, int mrow, const double* a_plus,
                         const double* a_minus_x, const double* a_minus_o, int sms, unsigned long long* tickets,
                         unsigned long long* ticket_base, cudaStream_t s) {
  using C = MmaCfg<NP>;
  if (p.W > kMmaMaxModes || p.B > kMmaMaxBaths) return cudaErrorInvalidValue;
  MmaParams P;
  P.p = p; P.mrows = mrows; P.mrow = mrow;
  const int D1 = p.D + 1;
  for (int l = 0; l < kMmaMaxModes; ++l) {
    const bool on = l < p.W && p.D >= 1;
    P.cP[l] = on ? a_plus[(size_t)l * D1] : 0.0;
    P.cX[l] = on ? a_minus_x[(size_t)l * D1 + 1] : 0.0;
    P.cO[l] = on ? a_minus_o[(size_t)l * D1 + 1] : 0.0;
  }
  const size_t smem = mma_smem_bytes<NP, CPLX>() + 3 * (size_t)mrow * 4;
  static size_t configured_on[64] = {};
  int dev_ = 0;
  cudaGetDevice(&dev_);
  size_t& configured = configured_on[dev_ & 63];
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_mma_kernel<NP, CPLX, HERM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  int grid = sms * mma_ctas_per_sm<NP, CPLX>();
  if (grid > p.nodes) grid = p.nodes;
  if (grid < 1) grid = 1;
  P.tickets = tickets;
  P.ticket_base = *ticket_base;
  rhs_mma_kernel<NP, CPLX, HERM><<<grid, C::THREADS, smem, s>>>(P);
  const cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    *ticket_base += (unsigned long long)p.nodes + 2ULL * (unsigned long long)grid;   // two failing draws per CTA
  } else {
    cudaMemsetAsync(tickets, 0, sizeof(unsigned long long), s);
    *ticket_base = 0;
  }
  return e;
}

int mma_padded(int N) { return N <= 32 ? 32 : (N + 15) / 16 * 16; }

}  // namespace

int mma_link_row(int W) { return (3 * W + (W & 1) + 2 + 3) / 4 * 4; }   // ints: plus, minus, n, (pad), d_u; 16-byte multiple

void mma_pack_row(int W, const int32_t* plus, const int32_t* minus, const uint8_t* tuple, double damp, int32_t* row) {
  for (int l = 0; l < W; ++l) { row[l] = plus[l]; row[W + l] = minus[l]; row[2 * W + l] = tuple[l]; }
  const int off = 3 * W + (W & 1);                    // 8-byte aligned
  double d = damp;
  std::memcpy(row + off, &d, 8);
  for (int e = off + 2; e < mma_link_row(W); ++e) row[e] = 0;
  if (W & 1) row[3 * W] = 0;
}

bool mma_supported(int N, int W, int B, int memberships, bool cplx) {
  if (N < 17 || N > 96 || W > kMmaMaxModes || B > kMmaMaxBaths || memberships > kMmaMaxMember) return false;
  if (mma_padded(N) == 96 && mma_smem_bytes<96, false>() + 3 * (size_t)mma_link_row(W) * 4 > (size_t)227 * 1024)
    return false;                                     // H, sigma and the staged link rows must fit one SM
  return !(cplx && mma_padded(N) == 96);              // Re H, Im H and sigma do not fit one SM's shared memory
}

cudaError_t launch_rhs_mma(const RhsParams& p, const int32_t* mrows, int mrow, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, int hermitian, int sms,
                           unsigned long long* tickets, unsigned long long* ticket_base, cudaStream_t s) {
  const bool cplx = p.Him != nullptr;
#define HEOM_MMA_ARGS p, mrows, mrow, a_plus, a_minus_x, a_minus_o, sms, tickets, ticket_base, s
#define HEOM_MMA_CASE(np)                                                                              \
  case np:                                                                                             \
    if (cplx) return hermitian ? launch_mma_t<np, true, true>(HEOM_MMA_ARGS) : launch_mma_t<np, true, false>(HEOM_MMA_ARGS);   \
    return hermitian ? launch_mma_t<np, false, true>(HEOM_MMA_ARGS) : launch_mma_t<np, false, false>(HEOM_MMA_ARGS);
  switch (mma_padded(p.N)) {
    HEOM_MMA_CASE(32) HEOM_MMA_CASE(48) HEOM_MMA_CASE(64) HEOM_MMA_CASE(80)
    case 96:
      if (cplx) return cudaErrorInvalidValue;
      return hermitian ? launch_mma_t<96, false, true>(HEOM_MMA_ARGS) : launch_mma_t<96, false, false>(HEOM_MMA_ARGS);
    default: return cudaErrorInvalidValue;
  }
#undef HEOM_MMA_CASE
#undef HEOM_MMA_ARGS
}

}  // namespace heom
