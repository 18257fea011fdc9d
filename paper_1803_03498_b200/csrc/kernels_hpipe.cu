// kernels_hpipe.cu -- persistent, software-pipelined sm_100a kernel for HERMITIAN hierarchy states,
// 2 <= N <= 16: the HEOM right-hand side (Eq. 12-17 with Eq. 23-25, 35-36) with the RK4 stage
// combination fused into its epilogue.
//
// Arithmetic (as kernels_herm.cu): the hierarchical Liouvillian maps Hermitian ADOs to Hermitian ADOs,
// so with   Z = -(i/hbar) H sigma_u - (d_u + T)/2 o sigma_u
//               + sum_l [ i a+ P_b sigma_{u+e_l} + (i a-x + a-o) P_b sigma_{u-e_l} ]      (P_b keeps row b)
// the right-hand side is k_u = Z + Z^dagger and only ROWS of neighbours are read.  Lane (g,j) owns
// column j of node g of its warp; a node takes LP = 2, 4, 8 or 16 lanes (the power of two >= N), so a
// warp pass covers G = 32/LP nodes.  Element (j,i) is produced by exactly
// the conjugate operations of element (i,j): the state stays bit-exactly Hermitian.
// The coupling factors of Eq. 35-36 are formed as sqrt(n) * c_l: (sqrt(n), sqrt(n+1)) from a small
// shared-memory table (one 16-byte load per link pair) and the per-mode constants c_l from the
// constant bank.
//
// Machine mapping -- every byte that streams goes through the TMA, only the gathers are plain loads:
//   * one CTA per SM; every WARP is an independent worker that draws groups of G consecutive storage
//     slots from a global ticket counter (so the groups in flight always form one compact window of
//     the state, which is what keeps the neighbour gathers in L2), with a private ring of S = 2
//     shared-memory slots {XA, ML} and two AC buffers (the one not holding this pass's running sum is
//     the transposition scratch);
//   * lane 0 is the warp's producer: cp.async.bulk (global -> shared, completion on the slot's
//     mbarrier) brings the stage input x and the nodes' meta rows (neighbour element offsets,
//     occupation records, damping rate) one pass ahead; the running sum acc follows half a pass ahead
//     (bulk-prefetched into L2 before that); once a pass has its sigma columns in registers the XA
//     region is dead and the step-start state y is bulk-loaded into it;
//   * a quarter-warp never spans two nodes (LP lanes per node) and the scratch uses a row stride == 1
//     (mod 8) elements, so the column reads, the transposition and the epilogue are free of bank
//     conflicts -- the LSU data pipe, not DRAM, limits this kernel otherwise;
//   * all 2*M*N neighbour-row loads of a pass are issued back to back (one L2/DRAM round trip per
//     pass), predicated, from pre-multiplied element offsets (one IMAD.WIDE + one LDG per link);
//   * the epilogue updates XA (next stage input) and AC (running sum) in place in shared memory and
//     lane 0 writes them back with cp.async.bulk (shared -> global, bulk async-group).
//
// GENERAL (non-Hermitian) states, e.g. the mu rho(0) of linear absorption, use the same
// pipeline with HERM = false: lane (g,j) forms column j of k_u directly,
//     k[:,j] = -i (H sigma)[:,j] + i sigma H[:,j] - (d_u + T[:,j]) o sigma[:,j]
//              + sum_l f_l (row part: element (b,j) of the neighbour's row b -- the same loads as above)
//              + sum_{l in bath j} f'_l sigma_{u +- e_l}[:,j]     (column part: the lane's own bath, a strided
//                                                                 column of the neighbour, Eq. 23, 25)
// with sigma H from the whole sigma tile (broadcast shared-memory reads) and no transposition.
#include "kernels.cuh"

#include <cmath>
#include <type_traits>

namespace heom {
namespace {

constexpr int kMaxModes = 64;   // W of the constant-bank coupling tables
constexpr int kMaxSqrt = 64;    // occupation numbers 0..D+1 < kMaxSqrt

template <int N>
struct PipeCfg {
  static constexpr int NN = N * N;
  static constexpr int LP = (N <= 2) ? 2 : (N <= 4) ? 4 : (N <= 8) ? 8 : 16;   // lanes per node
  static constexpr int G = 32 / LP;                   // nodes per warp pass
  static constexpr int S = 2;                         // ring slots per warp
  // warps per CTA (fewer if shared memory is short).  N > 8: 8 warps of 254 registers -- measured on config 4
  // (N = 14): 6 warps 2.556, 7 warps 2.425, 8 warps 2.338 ms per step; 10 warps (168 registers, spills) 3.07.
  // N <= 8: 12 warps of 168 registers; 16 warps of 128 registers with one mode index per gather batch: the same time.
  static constexpr int MAXW = (N <= 8) ? 12 : 8;
  // general states need more registers per thread (up to 251); N > 8, config 4 with hermitian=0: 6 warps 4.37, 7 warps 4.22,
  // 8 warps 4.39 ms per step
  static constexpr int MAXW_GENERAL = (N <= 8) ? 8 : 7;
  static constexpr int SMEM_BUDGET = 224 * 1024;
  static constexpr int KB = (16 / N) > 0 ? (16 / N) : 1;   // mode indices kk per gather batch (<= 32 loads)
  static constexpr int NP4 = (N + 3) / 4 * 4;         // ints per index group
  static constexpr int NB8 = (N + 7) / 8 * 8;         // occupation records (uint16) per group
  static constexpr int GROUP = (2 * NP4 + NB8 / 2 + 3) / 4 * 4;
  static constexpr int PS = NN;                       // shared-memory node stride (double2 elements): dense
  // transposition scratch: row stride == 1 (mod 8) elements
  static constexpr int RS = (N >= 5) ? ((N - 1 + 7) / 8 * 8 + 1) : N;
  static constexpr int SZ = (N - 1) * RS + N;
  static constexpr int XB = G * PS * 16;              // bytes of an XA region
  static constexpr int AB = G * SZ * 16;              // bytes of an AC buffer (also the scratch)
};

template <int N>
struct PipeParams {
  RhsParams p;
  const int32_t* links;   // [nodes][lrow]: per mode index kk: plus offsets[NP4], minus offsets[NP4], uint16
                          // occupation records [NB8] = 16 (2 n_l + [the "+" link exists]), the byte offset
                          // into the sqrt table; then d_u (double), padding
  int lrow;               // ints per links row (multiple of 4)
  int npass;              // groups of G nodes
  int nwarps;             // warps per CTA
  unsigned long long* tickets;   // DEVICE ticket counter; pass index = ticket - ticket_base
  unsigned long long ticket_base;
  double H[N * N];        // H / hbar, fs^-1
  double delta[N];
  double cP[kMaxModes];   // sqrt(s_l)                      a+(l,n)  = sqrt(n+1) cP[l]     (Eq. 35)
  double cX[kMaxModes];   // sgn(Re c_l) sqrt(s_l)          a-x(l,n) = sqrt(n) cX[l]       (Eq. 36, V^x part)
  double cO[kMaxModes];   // delta_k0 (lambda nu/hbar)/sqrt(s_l)   a-o(l,n) = sqrt(n) cO[l] (Eq. 36, V^o part)
};

__device__ __forceinline__ unsigned smem_u32(const void* ptr) {
  return (unsigned)__cvta_generic_to_shared(ptr);
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
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
// L2 eviction priorities: the streams (y, acc, the written buffers) are read or written once per launch
// -> evict_first; the stage input x is re-read by the neighbour gathers -> evict_last.
__device__ __forceinline__ unsigned long long policy_evict_first() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_last() {
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes,
                                         unsigned long long* bar, unsigned long long pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, unsigned bytes, unsigned long long pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, unsigned bytes, unsigned long long pol) {
  asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(src_gmem), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 16-byte read-only global load of base[off], executed only for off >= 0 (a valid link); otherwise the
// destination keeps its old contents.
__device__ __forceinline__ void ldg_link(double2& r, const double2* base, int off, unsigned long long pol) {
  asm volatile("{\n"
      ".reg .pred p;\n"
      ".reg .b64 a;\n"
      "setp.ge.s32 p, %3, 0;\n"
      "mad.wide.s32 a, %3, 16, %2;\n"
      "@p ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [a], %4;\n"
      "}\n" : "+d"(r.x), "+d"(r.y) : "l"(base), "r"(off), "l"(pol));
}

// One ticket.  Inline PTX on purpose: for a plain atomicAdd under `if (lane == 0)` the compiler emits its
// warp-aggregation sequence (vote, leader atomic, SHFL of the result), and that SHFL waits for the atomic's round
// trip on the spot (7.5 % of the stall samples on config 2) although the value is only needed a pass later.
__device__ __forceinline__ unsigned long long ticket_add(unsigned long long* ctr) {
  unsigned long long old;
  asm volatile("atom.global.add.u64 %0, [%1], 1;" : "=l"(old) : "l"(ctr) : "memory");
  return old;
}

template <int N, bool HERM>
__global__ void __launch_bounds__((HERM ? PipeCfg<N>::MAXW : PipeCfg<N>::MAXW_GENERAL) * 32, 1)
rhs_hpipe_kernel(const __grid_constant__ PipeParams<N> P) {
  using C = PipeCfg<N>;
  constexpr int NN = C::NN, G = C::G, S = C::S, KB = C::KB, PS = C::PS, RS = C::RS, SZ = C::SZ;
  constexpr int NP4 = C::NP4, NB8 = C::NB8, GROUP = C::GROUP, XB = C::XB, AB = C::AB;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const RhsParams& p = P.p;
  const int M = p.M, lrow = P.lrow, CW = P.nwarps;
  // shared memory per warp: S slots of {XA [G][PS] double2, ML [G][lrow] int32} and 2 AC buffers; then a
  // null meta row, the sqrt table [n][up] = (sqrt(n), up ? sqrt(n+1) : 0) and the mbarriers
  // (Horner stages keep no running sum: one AC buffer, the transposition scratch, is enough -- more warps fit)
  const int slot_bytes = XB + G * lrow * 4;
  const int nab = (p.horner != 0 && p.rhs_only == 0) ? 1 : 2;
  const int warp_bytes = S * slot_bytes + nab * AB;
  int32_t* sNull = reinterpret_cast<int32_t*>(smem_raw + CW * warp_bytes);    // [lrow]
  double2* sSQ = reinterpret_cast<double2*>(sNull + lrow);                    // [kMaxSqrt][2]
  double* sCoef = reinterpret_cast<double*>(sSQ + 2 * kMaxSqrt);              // [3][kMaxModes]: cP, cX, cO (lane-indexed)
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(sCoef + 3 * kMaxModes);
  for (int e = threadIdx.x; e < 2 * kMaxSqrt; e += blockDim.x)
    sSQ[e] = make_double2(sqrt((double)(e >> 1)), (e & 1) ? sqrt((double)((e >> 1) + 1)) : 0.0);
  for (int e = threadIdx.x; e < kMaxModes; e += blockDim.x) {
    sCoef[e] = P.cP[e]; sCoef[kMaxModes + e] = P.cX[e]; sCoef[2 * kMaxModes + e] = P.cO[e];
  }

  // a null meta row: every link invalid, every occupation record 0 (all coupling factors vanish)
  for (int e = threadIdx.x; e < lrow; e += blockDim.x) sNull[e] = (e < M * GROUP && (e % GROUP) < 2 * NP4) ? -1 : 0;
  constexpr int NBAR = 2 * S + 2;                     // per warp: barX[S], barY[S], barA[2]
  if (threadIdx.x == 0) {
    for (int q = 0; q < CW * NBAR; ++q) mbar_init(bars + q, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned char* ring = smem_raw + warp * warp_bytes;
  unsigned char* acbuf = ring + S * slot_bytes;       // 2 AC buffers
  unsigned long long* barX = bars + warp * NBAR;      // x + meta rows landed
  unsigned long long* barY = barX + S;                // y landed (in the XA region)
  unsigned long long* barA = barY + S;                // acc landed (in an AC buffer)
  const int npass = P.npass;

  const bool rhs_only = p.rhs_only != 0;
  const bool horner = p.horner != 0;                  // out_x = y + ax*k, no running sum (R6)
  const bool y_is_x = (p.y == p.x), acc_is_x = (p.acc_in == p.x);
  const bool need_A = !rhs_only && !horner && !acc_is_x;
  const bool need_Y = !rhs_only && p.out_x != nullptr && !y_is_x;
  const bool write_x = !rhs_only && p.out_x != nullptr;
  const bool producer = lane == 0;
  const unsigned long long pol_stream = policy_evict_first(), pol_keep = policy_evict_last();

  // ---- producer side (lane 0 only) -------------------------------------------------------------
  auto issue_x = [&](int q, int slot) {               // stage input + meta rows of pass q -> ring slot
    const int n0 = q * G;
    const int ncnt = min(G, p.nodes - n0);
    unsigned char* dst = ring + slot * slot_bytes;
    const unsigned bx = (unsigned)ncnt * NN * 16, bl = (unsigned)ncnt * lrow * 4;
    mbar_expect_tx(barX + slot, bx + bl);
    bulk_g2s(dst, p.x + (size_t)n0 * NN, bx, barX + slot, pol_keep);
    bulk_g2s(dst + XB, P.links + (size_t)n0 * lrow, bl, barX + slot, pol_stream);
    if (need_A) bulk_prefetch_l2(p.acc_in + (size_t)n0 * NN, bx, pol_stream);
    if (need_Y) bulk_prefetch_l2(p.y + (size_t)n0 * NN, bx, pol_stream);
  };
  auto issue_a = [&](int q, int buf) {                // running sum of pass q -> AC buffer
    const int n0 = q * G;
    const unsigned bx = (unsigned)min(G, p.nodes - n0) * NN * 16;
    mbar_expect_tx(barA + buf, bx);
    bulk_g2s(acbuf + buf * AB, p.acc_in + (size_t)n0 * NN, bx, barA + buf, pol_stream);
  };
  // Groups of this warp: one ticket per pass, drawn by lane 0 TWO passes ahead (the atomic's round trip under
  // contention is microseconds; values >= npass: no more work).  Every warp ends with exactly two such tickets.
  auto draw = [&]() -> int {
    const unsigned long long t = ticket_add(P.tickets) - P.ticket_base;
    return t < (unsigned long long)npass ? (int)t : npass;
  };
  int q = 0, qn = 0;                                  // this pass, the pass after it
  if (producer) {
    q = draw();
    qn = draw();
    if (q < npass) {
      issue_x(q, 0);
      if (need_A) issue_a(q, 0);
    }
  }
  q = __shfl_sync(0xffffffffu, q, 0);
  qn = __shfl_sync(0xffffffffu, qn, 0);

  constexpr int LP = C::LP;
  const int g = lane / LP;
  const bool lane_used = (lane % LP) < N;
  const int j = lane_used ? lane % LP : 0;            // idle lanes shadow column 0 of their node
  const double my_delta = P.delta[j];
  const double2* xj = p.x + j;
  double hcol[HERM ? 1 : N];                          // general states: column j of H / hbar
  if (!HERM) {
#pragma unroll
    for (int m = 0; m < N; ++m) hcol[m] = P.H[m * N + j];
  }

  int s = 0, ab = 0;                                  // ring slot and AC buffer of this pass
  unsigned ph = 0, pha = 0;                           // their mbarrier phases
  while (q < npass) {
    // the pass after the next one: the ticket is drawn now and its value looked at only at the end of this pass,
    // so that the atomic's round trip (microseconds under contention: 13 % of the stall samples when the value was
    // consumed at once, profiles/r2_cfg2_hpipe.md) hides behind the pass.  Always drawn: tickets per launch are fixed.
    unsigned long long traw = 0ULL;
    if (producer) traw = ticket_add(P.tickets);
    const int n0 = q * G;
    const int ncnt = min(G, p.nodes - n0);
    unsigned char* slot = ring + s * slot_bytes;
    double2* sXA = reinterpret_cast<double2*>(slot);
    double2* sAC = reinterpret_cast<double2*>(acbuf + (nab == 2 ? ab * AB : 0));   // unused when nab == 1
    double2* scr = reinterpret_cast<double2*>(acbuf + (nab == 2 ? (ab ^ 1) * AB : 0));
    const int32_t* sL = reinterpret_cast<const int32_t*>(slot + XB);
    mbar_wait(barX + s, ph);

    const bool active = lane_used && (g < ncnt);
    const int tl = active ? g : 0;                  // idle lanes shadow the pass's first node
    const double2* sig = sXA + tl * PS;
    const int32_t* lk = active ? sL + tl * lrow : sNull;

    // ---- Z = -(i/hbar) H sigma - (d_u + T)/2 o sigma, column j (Eq. 12-14) ----------------------
    // (general states: z = column j of -(i/hbar)[H, sigma] - (d_u + T) o sigma, the whole term)
    double2 z[N];
    {
      double2 col[N];
#pragma unroll
      for (int m = 0; m < N; ++m) col[m] = sig[m * N + j];
      double2 sh[HERM ? 1 : N];                     // general states: (sigma H / hbar)[i][j]
      if (!HERM) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
          double ar = 0.0, ai = 0.0;
#pragma unroll
          for (int m = 0; m < N; ++m) {
            const double2 v = sig[i * N + m];       // broadcast within the node
            ar = fma(v.x, hcol[m], ar); ai = fma(v.y, hcol[m], ai);
          }
          sh[i] = make_double2(ar, ai);
        }
      }
      if (need_Y) {
        // the sigma columns are in registers: XA is dead, stream the step-start state y into it
        fence_async_smem();
        __syncwarp();
        if (lane == 0) {
          const unsigned bx = (unsigned)ncnt * NN * 16;
          mbar_expect_tx(barY + s, bx);
          bulk_g2s(sXA, p.y + (size_t)n0 * NN, bx, barY + s, pol_stream);
        }
      }
      const double mhd = -0.5 * *reinterpret_cast<const double*>(lk + M * GROUP);   // -d_u/2 (Eq. 13)
#pragma unroll
      for (int b = 0; b < N; ++b) {
        double zr = 0.0, zi = 0.0;                  // (H/hbar) sigma, element (b, j)
#pragma unroll
        for (int m = 0; m < N; ++m) { zr = fma(P.H[b * N + m], col[m].x, zr); zi = fma(P.H[b * N + m], col[m].y, zi); }
        const double hd = (b == j) ? mhd : fma(-0.5, P.delta[b] + my_delta, mhd);   // Eq. 14 with Eq. 24
        if (HERM) {
          z[b].x = fma(hd, col[b].x, zi);           // -i (zr + i zi) = zi - i zr
          z[b].y = fma(hd, col[b].y, -zr);
        } else {                                    // -i (H sigma - sigma H) - (d_u + T) sigma
          z[b].x = fma(2.0 * hd, col[b].x, zi - sh[b].y);
          z[b].y = fma(2.0 * hd, col[b].y, sh[b].x - zr);
        }
      }
    }

    // ---- couplings: row b of sigma_{u +- e_l}, element j (Eq. 15-17 / 35-36, Eq. 23, 25) -------
    // An invalid "-" link has n_l = 0, an invalid "+" link (top level) carries the record byte 0:
    // both give a zero factor, so a skipped load contributes nothing.
    // One batch = KBN mode indices kk0..kk0+KBN-1: all 2*KBN*N loads are issued before the first is used.
    // FIRST marks the batch that starts at kk = 0, the only mode index with a V^o factor (delta_k0).
    auto gather = [&](auto kbn_tag, auto first_tag, int kk0) {
      constexpr int KBN = decltype(kbn_tag)::value;
      constexpr bool FIRST = decltype(first_tag)::value;
      double2 w[2 * KBN * N];
#pragma unroll
      for (int b = 0; b < 2 * KBN * N; ++b) w[b] = make_double2(0.0, 0.0);
#pragma unroll
      for (int kb = 0; kb < KBN; ++kb) {
        const int32_t* grp = lk + (kk0 + kb) * GROUP;
        int up[NP4], dn[NP4];
#pragma unroll
        for (int t = 0; t < NP4 / 4; ++t) {
          const int4 a = reinterpret_cast<const int4*>(grp)[t];
          up[4 * t] = a.x; up[4 * t + 1] = a.y; up[4 * t + 2] = a.z; up[4 * t + 3] = a.w;
          const int4 c = reinterpret_cast<const int4*>(grp + NP4)[t];
          dn[4 * t] = c.x; dn[4 * t + 1] = c.y; dn[4 * t + 2] = c.z; dn[4 * t + 3] = c.w;
        }
#pragma unroll
        for (int b = 0; b < N; ++b) {
          ldg_link(w[(2 * kb) * N + b], xj + b * N, up[b], pol_keep);
          ldg_link(w[(2 * kb + 1) * N + b], xj + b * N, dn[b], pol_keep);
        }
      }
      if (FIRST) {
        // with the gathers in flight: the write-back of the previous pass has left shared memory, so
        // its ring slot can take the next pass
        if (producer) {
          bulk_wait_read0();
          if (qn < npass) issue_x(qn, s ^ 1);
        }
      }
#pragma unroll
      for (int kb = 0; kb < KBN; ++kb) {
        const int kk = kk0 + kb;
        const int32_t* grp = lk + kk * GROUP;
        unsigned rw[NB8 / 2];
#pragma unroll
        for (int t = 0; t < NB8 / 8; ++t) {
          const uint4 v = reinterpret_cast<const uint4*>(grp + 2 * NP4)[t];
          rw[4 * t] = v.x; rw[4 * t + 1] = v.y; rw[4 * t + 2] = v.z; rw[4 * t + 3] = v.w;
        }
#pragma unroll
        for (int b = 0; b < N; ++b) {
          const unsigned rec = (b & 1) ? (rw[b >> 1] >> 16) : (rw[b >> 1] & 0xffffu);
          const double2 sq = *reinterpret_cast<const double2*>(reinterpret_cast<const unsigned char*>(sSQ) + rec);
          const int l = b * M + kk;
          const double a = sq.y * P.cP[l], ax = sq.x * P.cX[l];     // sqrt(n+1)|0, sqrt(n)
          const double2 wu = w[(2 * kb) * N + b], wd = w[(2 * kb + 1) * N + b];
          z[b].x = fma(-a, wu.y, z[b].x); z[b].y = fma(a, wu.x, z[b].y);                       // i a+ sigma^+
          z[b].x = fma(-ax, wd.y, z[b].x); z[b].y = fma(ax, wd.x, z[b].y);                     // i a-x sigma^-
          if (FIRST && kb == 0) {                                                              // a-o sigma^-, k = 0 only
            const double ao = sq.x * P.cO[l];
            z[b].x = fma(ao, wd.x, z[b].x); z[b].y = fma(ao, wd.y, z[b].y);
          }
        }
      }
    };
    {
      using std::integral_constant;
      int kk0 = 0;
      if (M >= KB) { gather(integral_constant<int, KB>{}, integral_constant<bool, true>{}, 0); kk0 = KB; }
      for (; kk0 + KB <= M; kk0 += KB) gather(integral_constant<int, KB>{}, integral_constant<bool, false>{}, kk0);
      if (kk0 < M) {                                  // remainder batch of 1..KB-1 mode indices
        const int rem = M - kk0;
        if (kk0 == 0) {
          if (KB > 1 && rem == 1) gather(integral_constant<int, 1>{}, integral_constant<bool, true>{}, 0);
          else if (KB > 2 && rem == 2) gather(integral_constant<int, (KB > 2 ? 2 : 1)>{}, integral_constant<bool, true>{}, 0);
          else if (KB > 3 && rem == 3) gather(integral_constant<int, (KB > 3 ? 3 : 1)>{}, integral_constant<bool, true>{}, 0);
          else {
            gather(integral_constant<int, 1>{}, integral_constant<bool, true>{}, 0);
            for (int kk = 1; kk < M; ++kk) gather(integral_constant<int, 1>{}, integral_constant<bool, false>{}, kk);
          }
        } else {
          for (int kk = kk0; kk < M; ++kk) gather(integral_constant<int, 1>{}, integral_constant<bool, false>{}, kk);
        }
      }
    }

    double2 k[N];
    if (HERM) {
      // ---- k = Z + Z^dagger, column j, through the scratch (conflict-free row stride RS) ---------
      __syncwarp();
      if (active) {
#pragma unroll
        for (int b = 0; b < N; ++b) scr[g * SZ + b * RS + j] = z[b];
      }
      __syncwarp();
#pragma unroll
      for (int i = 0; i < N; ++i) {
        const double2 zt = scr[tl * SZ + j * RS + i];              // Z[j][i]
        k[i].x = z[i].x + zt.x;
        k[i].y = z[i].y - zt.y;
      }
    } else {
      // ---- general states: column part of the couplings (Eq. 15-17 with Eq. 23, 25): the modes of the
      //      lane's OWN bath b = j act on column j, elements (i, j) of the neighbour, i = 0..N-1 ----------
      for (int kk = 0; kk < M; ++kk) {
        const int32_t* grp = lk + kk * GROUP;
        const int up = grp[j], dn = grp[NP4 + j];
        double2 wu[N], wd[N];
#pragma unroll
        for (int i = 0; i < N; ++i) { wu[i] = make_double2(0.0, 0.0); wd[i] = make_double2(0.0, 0.0); }
#pragma unroll
        for (int i = 0; i < N; ++i) {
          ldg_link(wu[i], xj + i * N, up, pol_keep);
          ldg_link(wd[i], xj + i * N, dn, pol_keep);
        }
        const unsigned rec = reinterpret_cast<const unsigned short*>(grp + 2 * NP4)[j];
        const double2 sq = *reinterpret_cast<const double2*>(reinterpret_cast<const unsigned char*>(sSQ) + rec);
        const int l = j * M + kk;
        const double a = sq.y * sCoef[l], ax = sq.x * sCoef[kMaxModes + l], ao = sq.x * sCoef[2 * kMaxModes + l];
#pragma unroll
        for (int i = 0; i < N; ++i) {               // V^x = -1, V^o = +1 on column b
          z[i].x = fma(a, wu[i].y, z[i].x); z[i].y = fma(-a, wu[i].x, z[i].y);                 // -i a+ sigma^+
          z[i].x = fma(ao, wd[i].x, fma(ax, wd[i].y, z[i].x));                                 // (-i a-x + a-o) sigma^-
          z[i].y = fma(ao, wd[i].y, fma(-ax, wd[i].x, z[i].y));
        }
      }
#pragma unroll
      for (int i = 0; i < N; ++i) k[i] = z[i];
      __syncwarp();
    }
    if (need_A && qn < npass) {
      // the scratch is free again: bring the next pass's running sum (already in L2) into it
      fence_async_smem();
      __syncwarp();
      if (producer) issue_a(qn, ab ^ 1);
    }

    // ---- fused RK4 stage epilogue, in place in shared memory ------------------------------------
    if (need_Y) mbar_wait(barY + s, ph);
    if (need_A) mbar_wait(barA + ab, pha);
    if (active) {
      double2* xa = sXA + g * PS + j;
      double2* ac = sAC + g * PS + j;
      // one straight-line loop per stage kind (uniform branches), so nothing is selected per element
      if (rhs_only) {
#pragma unroll
        for (int i = 0; i < N; ++i) ac[i * N] = k[i];
      } else if (horner) {                          // Horner stage: XA holds y (first stage: y = x); w' = y + ax k
#pragma unroll
        for (int i = 0; i < N; ++i) {
          const double2 yv = xa[i * N];
          xa[i * N] = make_double2(fma(p.ax, k[i].x, yv.x), fma(p.ax, k[i].y, yv.y));
        }
      } else if (acc_is_x) {                        // stage 1: y = acc_in = x, still in XA
#pragma unroll
        for (int i = 0; i < N; ++i) {
          const double2 yv = xa[i * N];
          xa[i * N] = make_double2(fma(p.ax, k[i].x, yv.x), fma(p.ax, k[i].y, yv.y));
          ac[i * N] = make_double2(fma(p.bx, k[i].x, yv.x), fma(p.bx, k[i].y, yv.y));
        }
      } else if (!write_x) {                        // stage 4: running sum only
#pragma unroll
        for (int i = 0; i < N; ++i) {
          const double2 av = ac[i * N];
          ac[i * N] = make_double2(fma(p.bx, k[i].x, av.x), fma(p.bx, k[i].y, av.y));
        }
      } else {                                      // classical stages 2, 3: y is in XA
#pragma unroll
        for (int i = 0; i < N; ++i) {
          const double2 yv = xa[i * N], av = ac[i * N];
          xa[i * N] = make_double2(fma(p.ax, k[i].x, yv.x), fma(p.ax, k[i].y, yv.y));
          ac[i * N] = make_double2(fma(p.bx, k[i].x, av.x), fma(p.bx, k[i].y, av.y));
        }
      }
    }
    fence_async_smem();
    __syncwarp();
    if (lane == 0) {
      const unsigned bx = (unsigned)ncnt * NN * 16;
      if (write_x) bulk_s2g(p.out_x + (size_t)n0 * NN, sXA, bx, pol_stream);
      if (!horner) bulk_s2g(p.out_acc + (size_t)n0 * NN, sAC, bx, pol_stream);
      bulk_commit();
    }
    if ((s ^= 1) == 0) ph ^= 1u;
    if ((ab ^= 1) == 0) pha ^= 1u;
    int qnn = 0;
    if (producer) {
      const unsigned long long t = traw - P.ticket_base;
      qnn = t < (unsigned long long)npass ? (int)t : npass;
    }
    q = qn;
    qn = __shfl_sync(0xffffffffu, qnn, 0);
  }
  if (producer) bulk_wait_all();
}

template <int N>
size_t hpipe_smem(int lrow, int warps, int nab = 2) {
  using C = PipeCfg<N>;
  return (size_t)warps * (C::S * ((size_t)C::XB + (size_t)C::G * lrow * 4) + nab * (size_t)C::AB) +
         (size_t)lrow * 4 + 2 * kMaxSqrt * 16 + 3 * kMaxModes * 8 + (size_t)warps * (2 * C::S + 2) * 8;
}
// warps per CTA: as many as fit into the shared-memory budget (0 if not even one fits)
template <int N>
int hpipe_warps(int lrow, bool herm = true, int nab = 2) {
  using C = PipeCfg<N>;
  int w = herm ? C::MAXW : C::MAXW_GENERAL;
  while (w >= 1 && hpipe_smem<N>(lrow, w, nab) > (size_t)C::SMEM_BUDGET) --w;
  return w;
}

template <int N, bool HERM>
cudaError_t launch_hpipe_t(const RhsParams& p, const int32_t* links, int lrow, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, const double* H_host,
                           const double* delta_host, int warps, int sms, unsigned long long* tickets,
                           unsigned long long* ticket_base, cudaStream_t s) {
  using C = PipeCfg<N>;
  PipeParams<N> P;
  P.p = p; P.links = links; P.lrow = lrow;
  P.npass = (p.nodes + C::G - 1) / C::G;
  const int nab = (p.horner != 0 && p.rhs_only == 0) ? 1 : 2;
  const int wmax = hpipe_warps<N>(lrow, HERM, nab);
  if (wmax < 1) return cudaErrorInvalidValue;
  P.nwarps = (warps > 0 && warps < wmax) ? warps : wmax;
  for (int e = 0; e < N * N; ++e) P.H[e] = H_host[e] * p.inv_hbar;
  for (int e = 0; e < N; ++e) P.delta[e] = delta_host[e];
  const int D1 = p.D + 1;
  for (int l = 0; l < kMaxModes; ++l) {
    const bool on = l < p.W && p.D >= 1;
    P.cP[l] = on ? a_plus[(size_t)l * D1] : 0.0;            // sqrt(1 * s_l)
    P.cX[l] = on ? a_minus_x[(size_t)l * D1 + 1] : 0.0;     // sgn sqrt(1 * s_l)
    P.cO[l] = on ? a_minus_o[(size_t)l * D1 + 1] : 0.0;     // sqrt(1 / s_l) lambda nu / hbar
  }
  const size_t smem = hpipe_smem<N>(lrow, P.nwarps, nab);
  static size_t configured_on[64] = {};   // per device: the attribute belongs to the device's context
  int dev_ = 0;
  cudaGetDevice(&dev_);
  size_t& configured = configured_on[dev_ & 63];
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_hpipe_kernel<N, HERM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  int grid = sms;
  if (grid > (P.npass + P.nwarps - 1) / P.nwarps) grid = (P.npass + P.nwarps - 1) / P.nwarps;
  if (grid < 1) grid = 1;
  P.tickets = tickets;
  P.ticket_base = *ticket_base;
  rhs_hpipe_kernel<N, HERM><<<grid, P.nwarps * 32, smem, s>>>(P);
  const cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    *ticket_base += (unsigned long long)P.npass + 2ULL * grid * P.nwarps;   // two failing draws per warp
  } else {                                 // nothing ran: keep host base and device counter in step
    cudaMemsetAsync(tickets, 0, sizeof(unsigned long long), s);
    *ticket_base = 0;
  }
  return e;
}

}  // namespace

#define HEOM_HPIPE_ALL(X) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)

int hpipe_links_row(int N, int M) {
  if (N < 2 || N > 16) return 0;
  const int np4 = (N + 3) / 4 * 4, nb8 = (N + 7) / 8 * 8;
  return M * ((2 * np4 + nb8 / 2 + 3) / 4 * 4) + 4;
}

bool hpipe_supported(int N, int W, int D, long long nodes) {
  const int M = W / (N > 0 ? N : 1);
  const int lrow = hpipe_links_row(N, M);
  if (lrow == 0) return false;
  if (nodes * (long long)N * N >= 2147483647LL) return false;   // element offsets are int32
  if (W > kMaxModes || D + 2 > kMaxSqrt) return false;          // constant-bank tables
  switch (N) {
#define HEOM_HPIPE_CASE(n) case n: return hpipe_warps<n>(lrow) >= 2;
    HEOM_HPIPE_ALL(HEOM_HPIPE_CASE)
#undef HEOM_HPIPE_CASE
    default: return false;
  }
}

void hpipe_pack_links(int N, int M, int D, const int32_t* plus, const int32_t* minus, const uint8_t* tuple,
                      double damp, int32_t* row) {
  const int np4 = (N + 3) / 4 * 4, nb8 = (N + 7) / 8 * 8, group = (2 * np4 + nb8 / 2 + 3) / 4 * 4;
  const int NN = N * N;
  (void)D;
  for (int kk = 0; kk < M; ++kk) {
    int32_t* grp = row + kk * group;
    uint16_t* rec = reinterpret_cast<uint16_t*>(grp + 2 * np4);   // 16 (2 n_l + ["+" link exists])
    for (int b = 0; b < np4; ++b) {
      const int32_t up = (b < N) ? plus[b * M + kk] : -1, dn = (b < N) ? minus[b * M + kk] : -1;
      grp[b] = up < 0 ? -1 : up * NN;               // pre-multiplied element offset of the neighbour
      grp[np4 + b] = dn < 0 ? -1 : dn * NN;
    }
    for (int b = 0; b < nb8; ++b) {
      if (b < N) {
        const unsigned n = tuple[b * M + kk];
        rec[b] = (uint16_t)(16u * (2u * n + (plus[b * M + kk] >= 0 ? 1u : 0u)));
      } else {
        rec[b] = 0;
      }
    }
  }
  double* tail = reinterpret_cast<double*>(row + M * group);    // 16-byte tail: d_u (Eq. 13), padding
  tail[0] = damp; tail[1] = 0.0;
}

cudaError_t launch_rhs_hpipe(const RhsParams& p, const int32_t* links, int lrow, const double* a_plus,
                             const double* a_minus_x, const double* a_minus_o, const double* H_host,
                             const double* delta_host, int hermitian, int warps, int sms,
                             unsigned long long* tickets, unsigned long long* ticket_base, cudaStream_t s) {
  switch (p.N) {
#define HEOM_HPIPE_CASE(n)                                                                                          \
  case n:                                                                                                           \
    return hermitian ? launch_hpipe_t<n, true>(p, links, lrow, a_plus, a_minus_x, a_minus_o, H_host, delta_host,  \
                                               warps, sms, tickets, ticket_base, s)                                \
                     : launch_hpipe_t<n, false>(p, links, lrow, a_plus, a_minus_x, a_minus_o, H_host, delta_host, \
                                                warps, sms, tickets, ticket_base, s);
    HEOM_HPIPE_ALL(HEOM_HPIPE_CASE)
#undef HEOM_HPIPE_CASE
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace heom
