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
//     to sigma_{u +- e_l} walk the node's CSR link list: a link of bath b touches the elements (i,j) with
//     i or j in the bath's state set (membership bits in shared memory), factor
//     i a (q_i - q_j) + a_o (q_i + q_j)  (Eq. 23, 25 summed over the bath's states);
//   * fused epilogue straight from the fragment layout: Horner form w' = y + ax k (R6), the
//     classical form with a running sum, or the bare right-hand side.
#include "kernels.cuh"

#include <cmath>

namespace heom {
namespace {

constexpr int kMmaMaxModes = 288;   // W of the constant-bank coupling tables
constexpr int kMmaMaxBaths = 96;
constexpr int kMmaStaged = 64;      // link entries of a node staged in shared memory (the rest is read from global)

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
  return (size_t)NP * C::HS * 8 * (CPLX ? 2 : 1) + (size_t)NP * C::SS * 16 * (C::DB ? 2 : 1) + (size_t)kMmaMaxBaths * 16 +
         2 * ((size_t)kMmaStaged * 16 + 32) + 16 + 16 + 258 * 8;
}
template <int NP, bool CPLX>
constexpr int mma_ctas_per_sm() {
  constexpr size_t per = mma_smem_bytes<NP, CPLX>() + 1024;            // + the runtime's per-CTA reservation
  constexpr int by_smem = (int)((size_t)227 * 1024 / per);
  constexpr int by_threads = 512 / MmaCfg<NP>::THREADS;              // >= 128 registers per thread
  constexpr int m = by_smem < by_threads ? by_smem : by_threads;
  return m < 1 ? 1 : (m > 4 ? 4 : m);
}

struct MmaParams {
  RhsParams p;
  const int64_t* lptr;     // [nodes+1] CSR offsets into lent
  const int4* lent;        // link entries: x = neighbour slot, y = mode l, z = 0 ("+") or 1 ("-"), w = n_l
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

template <int NP, bool CPLX>
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
  // per node parity: {damping rate d_u, first entry e0, entry count} and the first kMmaStaged link entries
  unsigned char* sLinkBase = reinterpret_cast<unsigned char*>(sMask + 4 * kMmaMaxBaths);
  constexpr int kLinkBuf = kMmaStaged * 16 + 32;
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(sLinkBase + 2 * kLinkBuf);   // [2]
  int* sNode = reinterpret_cast<int*>(bar + 2);                                                  // [2] (+ padding)
  double* sSqrt = reinterpret_cast<double*>(sNode + 4);                       // [258] sqrt(n), n = 0..D+1 <= 256
  for (int e = threadIdx.x; e < 258; e += C::THREADS) sSqrt[e] = sqrt((double)e);

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
  // warp 0 stages a node's header and link entries: fetch() early (registers), publish() behind a CTA barrier
  struct Staged { double dd; long long e0; int cnt; int4 ent[2]; };
  auto fetch = [&](int node) {
    Staged st;
    st.dd = 0.0; st.e0 = 0; st.cnt = 0;
    st.ent[0] = make_int4(0, 0, 0, 0); st.ent[1] = make_int4(0, 0, 0, 0);
    if (node < nodes) {
      st.e0 = P.lptr[node];
      st.cnt = (int)(P.lptr[node + 1] - st.e0);
      st.dd = p.damp[node];
      if (lane < st.cnt && lane < kMmaStaged) st.ent[0] = __ldg(P.lent + st.e0 + lane);
      if (lane + 32 < st.cnt && lane + 32 < kMmaStaged) st.ent[1] = __ldg(P.lent + st.e0 + lane + 32);
    }
    return st;
  };
  auto publish = [&](const Staged& st, int buf) {
    unsigned char* base = sLinkBase + buf * kLinkBuf;
    if (lane == 0) {
      *reinterpret_cast<double*>(base) = st.dd;
      *reinterpret_cast<long long*>(base + 8) = st.e0;
      *reinterpret_cast<int*>(base + 16) = st.cnt;
    }
    int4* ents = reinterpret_cast<int4*>(base + 32);
    ents[lane] = st.ent[0];
    ents[lane + 32] = st.ent[1];
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
    publish(fetch(first), 0);
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
  int lbuf = 0;                                       // link-staging buffer of the node in flight
  int cur = 0;                                        // sigma tile / mbarrier / sNode slot of the node in flight
  for (;;) {
    mmbar_wait(bar + cur, (ph >> cur) & 1u);          // sigma of the node has landed (or there is no node)
    ph ^= 1u << cur;
    const int node = *reinterpret_cast<volatile int*>(sNode + cur);
    if (node >= nodes) break;
    const double2* sS = sS0 + cur * NP * SS;
    Staged nst;
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
      nst = fetch(next);                              // in flight behind this node's contraction
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
    const unsigned char* lhead = sLinkBase + lbuf * kLinkBuf;
    const double dd = *reinterpret_cast<const double*>(lhead);
#pragma unroll
    for (int rg = 0; rg < RG; ++rg) {
      const int row = i0w + 8 * rg + rho;
#pragma unroll
      for (int ct = 0; ct < CT; ++ct) {
        const int col = j0w + 4 * ct + t;
        const double2 sv = sS[row * SS + col];
        const double tv = T_IN_REGS ? tt[rg * CT + ct] : ((row < N && col < N) ? __ldg(p.Tterm + row * N + col) : 0.0);
        const double dt = dd + tv;
        const double2 c = acc[rg][ct];
        acc[rg][ct] = make_double2(fma(-dt, sv.x, c.y), fma(-dt, sv.y, -c.x));
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();                                  // every warp is done with the node's sigma

    // ---- next node: start its TMA load behind the rest of this node's work ---------------------------
    if (warp == 0) {
      if (!DB) {
        if (lane == 0) sNode[0] = next;
        load_sigma(next, 0);
      }
      publish(nst, lbuf ^ 1);                         // read after the next node's barrier
    }

    // ---- couplings to sigma_{u +- e_l} (Eq. 15-17, 23, 25, 35-36, summed over the bath's states) ------
    {
      const long long e0 = *reinterpret_cast<const long long*>(lhead + 8);
      const int cnt = *reinterpret_cast<const int*>(lhead + 16);
      const int4* staged = reinterpret_cast<const int4*>(lhead + 32);
      // Small tiles (DENSE_LINKS), branch-free per link: every thread loads all RG*CT of its elements (an inactive one
      // reads element 0 of the neighbour, warp-wide the same address, and gets a zero factor), so that the loads of a
      // link -- and, with the loop unrolled by two, of two links -- are in flight together.  Membership bits exist only for real states,
      // so padded rows and columns are inactive by construction.
      constexpr bool DENSE_LINKS = RG * CT <= 12;
      const unsigned rsel = ((C::RW == 32) ? 0xffffffffu : ((1u << C::RW) - 1u));
      const unsigned long long csel = (1ULL << C::CWc) - 1ULL;
#pragma unroll 2
      for (int q = 0; q < cnt; ++q) {
        const int4 ent = q < kMmaStaged ? staged[q] : __ldg(P.lent + e0 + q);
        const int l = ent.y, b = l / p.M;
        const unsigned rbits = (sMask[b * 4 + (i0w >> 5)] >> (i0w & 31)) & rsel;
        const unsigned long long cbits =
            ((((unsigned long long)sMask[b * 4 + (j0w >> 5) + 1] << 32) | sMask[b * 4 + (j0w >> 5)]) >> (j0w & 31)) & csel;
        if (rbits == 0u && cbits == 0ULL) continue;   // warp-uniform: the link does not touch this warp's tile
        // element factor = i fx (q_i - q_j) + fo (q_i + q_j), q in {0, 1}
        double fx, fo;
        if (ent.z == 0) { fx = sSqrt[ent.w + 1] * P.cP[l]; fo = 0.0; }                         // "+"
        else { const double sn = sSqrt[ent.w]; fx = sn * P.cX[l]; fo = sn * P.cO[l]; }           // "-"
        const double2* nb = p.x + (size_t)ent.x * NN;
#pragma unroll
        for (int rg = 0; rg < RG; ++rg) {
          const int row = i0w + 8 * rg + rho;
          const bool qr = (rbits >> (8 * rg + rho)) & 1u;
          // (re, im) factor of the element for q_j = 0 and for q_j = 1
          const double a0r = qr ? fo : 0.0, a0i = qr ? fx : 0.0;
          const double a1r = qr ? 2.0 * fo : fo, a1i = qr ? 0.0 : -fx;
#pragma unroll
          for (int ct = 0; ct < CT; ++ct) {
            const int col = j0w + 4 * ct + t;
            const bool qj = (cbits >> (4 * ct + t)) & 1ULL;
            const double fr = qj ? a1r : a0r, fi = qj ? a1i : a0i;
            if (DENSE_LINKS) {
              const int off = (qr | qj) ? row * N + col : 0;
              const double2 w = __ldg(nb + off);
              acc[rg][ct].x = fma(fr, w.x, fma(-fi, w.y, acc[rg][ct].x));
              acc[rg][ct].y = fma(fr, w.y, fma(fi, w.x, acc[rg][ct].y));
            } else if (qr | qj) {                     // large tiles: few of a thread's elements are touched
              const double2 w = __ldg(nb + row * N + col);
              acc[rg][ct].x = fma(fr, w.x, fma(-fi, w.y, acc[rg][ct].x));
              acc[rg][ct].y = fma(fr, w.y, fma(fi, w.x, acc[rg][ct].y));
            }
          }
        }
      }
    }

    lbuf ^= 1;
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

template <int NP, bool CPLX>
cudaError_t launch_mma_t(const RhsParams& p, const int64_t* lptr, const int4* lent, const double* a_plus,
                         const double* a_minus_x, const double* a_minus_o, int sms, unsigned long long* tickets,
                         unsigned long long* ticket_base, cudaStream_t s) {
  using C = MmaCfg<NP>;
  if (p.W > kMmaMaxModes || p.B > kMmaMaxBaths) return cudaErrorInvalidValue;
  MmaParams P;
  P.p = p; P.lptr = lptr; P.lent = lent;
  const int D1 = p.D + 1;
  for (int l = 0; l < kMmaMaxModes; ++l) {
    const bool on = l < p.W && p.D >= 1;
    P.cP[l] = on ? a_plus[(size_t)l * D1] : 0.0;
    P.cX[l] = on ? a_minus_x[(size_t)l * D1 + 1] : 0.0;
    P.cO[l] = on ? a_minus_o[(size_t)l * D1 + 1] : 0.0;
  }
  constexpr size_t smem = mma_smem_bytes<NP, CPLX>();
  static bool configured_on[64] = {};
  int dev_ = 0;
  cudaGetDevice(&dev_);
  bool& configured = configured_on[dev_ & 63];
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_mma_kernel<NP, CPLX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  int grid = sms * mma_ctas_per_sm<NP, CPLX>();
  if (grid > p.nodes) grid = p.nodes;
  if (grid < 1) grid = 1;
  P.tickets = tickets;
  P.ticket_base = *ticket_base;
  rhs_mma_kernel<NP, CPLX><<<grid, C::THREADS, smem, s>>>(P);
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

bool mma_supported(int N, int W, int B, bool cplx) {
  if (N < 17 || N > 96 || W > kMmaMaxModes || B > kMmaMaxBaths) return false;
  return !(cplx && mma_padded(N) == 96);              // Re H, Im H and sigma do not fit one SM's shared memory
}

cudaError_t launch_rhs_mma(const RhsParams& p, const int64_t* lptr, const void* lent, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, int sms, unsigned long long* tickets,
                           unsigned long long* ticket_base, cudaStream_t s) {
  const int4* le = reinterpret_cast<const int4*>(lent);
  const bool cplx = p.Him != nullptr;
#define HEOM_MMA_CASE(np)                                                                                          \
  case np:                                                                                                         \
    return cplx ? launch_mma_t<np, true>(p, lptr, le, a_plus, a_minus_x, a_minus_o, sms, tickets, ticket_base, s)  \
                : launch_mma_t<np, false>(p, lptr, le, a_plus, a_minus_x, a_minus_o, sms, tickets, ticket_base, s);
  switch (mma_padded(p.N)) {
    HEOM_MMA_CASE(32) HEOM_MMA_CASE(48) HEOM_MMA_CASE(64) HEOM_MMA_CASE(80)
    case 96:
      if (cplx) return cudaErrorInvalidValue;
      return launch_mma_t<96, false>(p, lptr, le, a_plus, a_minus_x, a_minus_o, sms, tickets, ticket_base, s);
    default: return cudaErrorInvalidValue;
  }
#undef HEOM_MMA_CASE
}

}  // namespace heom
