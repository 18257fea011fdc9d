// kernels.cuh -- launch interface between the C ABI (api.cu) and the sm_100a kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace heom {

// Everything one RHS evaluation needs.  All pointers DEVICE.  Node index = storage slot.
struct RhsParams {
  int N;            // sites
  int M;            // modes per bath (K+1)
  int W;            // N*M
  int D;            // depth
  int nodes;        // number of nodes
  int stride;       // complex elements per node in a state buffer (>= N*N)
  double inv_hbar;  // 1/hbar, fs^-1 per cm^-1
  const double* H;          // [N][N] cm^-1
  const double* Tterm;      // [N][N]  (1-delta_ij)(Delta_i+Delta_j)            Eq. 14 + 24
  const double* damp;       // [nodes] sum_l n_l gamma_l                         Eq. 13
  const int32_t* plus;      // [nodes][W] slot of n+e_l or -1
  const int32_t* minus;     // [nodes][W] slot of n-e_l or -1
  const uint8_t* tuples;    // [nodes][W]
  const double* a_plus;     // [W][D+1]                                          Eq. 35
  const double* a_minus_x;  // [W][D+1]                                          Eq. 36, V^x part
  const double* a_minus_o;  // [W][D+1]                                          Eq. 36, V^o part
  // state buffers (complex128 as double2)
  const double2* x;       // stage input: the state the Liouvillian is applied to (gathered)
  const double2* y;       // step-start state (may be null when not needed)
  const double2* acc_in;  // running RK4 sum to extend (may alias y)
  double2* out_x;         // next stage input  = y + ax*k      (null: not written)
  double2* out_acc;       // acc_in + bx*k     (or, in RHS-only mode, k itself)
  double ax, bx;
  int rhs_only;           // 1: out_acc = k, nothing else read or written
  // Horner form of RK4 for a linear autonomous right-hand side (R6): w <- y + (dt/s) L w, s = 4, 3, 2, 1.
  // No running sum: acc_in / out_acc / bx are unused, out_x = y + ax*k (y may alias x: first stage; out_x may alias
  // y: last stage, in place).  Honoured by the pipelined small-N, the tensor-core and the column kernels.
  int horner;
  // General system-bath operators (heom_create_general; generic and mma kernels): modes are indexed l = b*M + k
  // over the B baths (W = B*M), bath b couples through the projectors on the states whose bit is set in
  // bmask[b][0..3] (sums over s of Eq. 14-17), and H = H + i Him may be complex Hermitian (Eq. 51).
  int gen;                  // 1: general context
  int B;                    // baths
  const int32_t* sptr;      // [N+1] CSR offsets: baths that state s belongs to
  const int32_t* sbl;       // bath indices
  const uint32_t* bmask;    // [B][4]
  const double* Him;        // [N][N] cm^-1 or null (real H)
};

// Generic kernel: any N <= 96, one thread per matrix element.
cudaError_t launch_rhs_generic(const RhsParams& p, cudaStream_t s);
// Shared-memory bytes the generic kernel needs (0 if N is unsupported).
size_t rhs_generic_smem(int N);

// Persistent TMA-pipelined kernel for 2 <= N <= 16 (kernels_hpipe.cu); hermitian = 1: the state is exactly
// Hermitian (row-only gathers, exact Hermiticity preserved), 0: general state (row and column gathers).  links: DEVICE
// [nodes][lrow] int32 written by hpipe_pack_links (neighbour entries are element offsets slot*N*N, uint16
// occupation records, and the row ends with the node's damping rate).  a_plus, a_minus_x, a_minus_o,
// H_host, delta_host: HOST (the per-mode constants travel in the kernel parameters).  warps <= 0: as
// many warps per CTA as shared memory allows; grid = one CTA per SM.  tickets: DEVICE counter (zeroed once);
// *ticket_base: HOST running total of the tickets drawn by earlier launches (updated here).
int hpipe_links_row(int N, int M);
bool hpipe_supported(int N, int W, int D, long long nodes);
void hpipe_pack_links(int N, int M, int D, const int32_t* plus, const int32_t* minus, const uint8_t* tuple,
                      double damp, int32_t* row);
cudaError_t launch_rhs_hpipe(const RhsParams& p, const int32_t* links, int lrow, const double* a_plus,
                             const double* a_minus_x, const double* a_minus_o, const double* H_host,
                             const double* delta_host, int hermitian, int warps, int sms,
                             unsigned long long* tickets, unsigned long long* ticket_base, cudaStream_t s);

// Tensor-core (DMMA) kernel for N = 32, 64, 96 (kernels_large.cu), any state; hermitian = 1: the state is exactly
// Hermitian (one product H sigma instead of two, row-only gathers, exact Hermiticity preserved).  lptr: DEVICE [nodes+1] CSR
// offsets; lent: DEVICE int4 link entries {neighbour slot, mode l, 0 "+" | 1 "-", n_l}; Hs_dev: DEVICE
// [N][N] = H/hbar; delta_dev: DEVICE [N]; a_*: HOST coupling tables [W][D+1]; tickets as for hpipe.
bool large_supported(int N, int W);
// mrows: dense link rows [nodes][mrow] in the format of mma_link_row / mma_pack_row (read by the Hermitian variant)
cudaError_t launch_rhs_large(const RhsParams& p, const int64_t* lptr, const void* lent, const int32_t* mrows, int mrow,
                             const double* Hs_dev, const double* delta_dev, const double* a_plus, const double* a_minus_x,
                             const double* a_minus_o, int hermitian, int sms, unsigned long long* tickets,
                             unsigned long long* ticket_base, cudaStream_t s);

// Tensor-core kernel for 17 <= N <= 96 and general system-bath operators (kernels_mma.cu): p.gen = 1 with the bath
// membership bits and the state -> baths lists, p.Him != null selects the complex-H instantiation.  mrows: DEVICE
// [nodes][mrow] dense link rows written by mma_pack_row (plus[W], minus[W], n[W] as int32 with mode indices
// l = b*M + k, then d_u); a_*: HOST [W][D+1]; tickets as for hpipe.  hermitian = 1: the state is exactly Hermitian
// (one product H sigma, row-only gathers, k = Z + Z^dagger; exact Hermiticity preserved).
bool mma_supported(int N, int W, int B, int memberships, bool cplx);
int mma_link_row(int W);   // int32 entries per row (multiple of 4)
void mma_pack_row(int W, const int32_t* plus, const int32_t* minus, const uint8_t* tuple, double damp, int32_t* row);
cudaError_t launch_rhs_mma(const RhsParams& p, const int32_t* mrows, int mrow, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, int hermitian, int sms,
                           unsigned long long* tickets, unsigned long long* ticket_base, cudaStream_t s);

// Whole-propagation kernel for tiny hierarchies (kernels_tiny.cu): nsteps classical RK4 steps of the state p.x
// (DEVICE, storage-slot order, updated in place) inside ONE launch of one CTA; tables as for the generic kernel.
bool tiny_supported(int N, int W, int D, long long nodes);
cudaError_t launch_rk4_tiny(const RhsParams& p, double dt, int nsteps, cudaStream_t s);

// dst[slot_of[u]*dst_stride + e] = src[u*NN + e]  (to_device=1) or the inverse (to_device=0)
cudaError_t launch_permute(const double2* src, double2* dst, const int32_t* slot_of, int nodes,
                           int NN, int stride, int to_device, cudaStream_t s);
// out[0..N-1] = Re sigma_0[i][i]; out[N], out[N+1] = trace (re, im)
cudaError_t launch_populations(const double2* node0, int N, double* out, cudaStream_t s);

// Column-sparse states (kernels_ket.cu): sigma_u = v_u e_col^T for every node, state `col` without a bath and
// uncoupled in H (linear absorption).  p.x, p.acc_in, p.out_x, p.out_acc are KET buffers [nodes][N];
// p.rhs_only / p.ax / p.bx as for the matrix kernels (Taylor form: out_x = ax k, out_acc = acc_in + bx k).
// links / lrow: the rows written by hpipe_pack_links; a_*, H_host, delta_host: HOST.
bool ket_supported(int N, int W, int D);
cudaError_t launch_rhs_ket(const RhsParams& p, const int32_t* links, int lrow, int col, const double* a_plus,
                           const double* a_minus_x, const double* a_minus_o, const double* H_host,
                           const double* delta_host, int sms, cudaStream_t s);
// dst[slot][i][j] = (j == col) ? ket[slot][i] : 0   (full matrices for the host-visible getters)
cudaError_t launch_ket_expand(const double2* ket, double2* dst, long long nodes, int N, int col, cudaStream_t s);

// dst[q][0..NN) = src[idx[q]*stride + 0..NN): the send buffer of a halo exchange
cudaError_t launch_pack_rows(const double2* src, double2* dst, const int32_t* idx, long long rows, int NN, int stride,
                             cudaStream_t s);

// slice halo: pair q = (node[q], st[q]) <-> packed[q][0..per), per = N (row st) or 2N (row st, then column st);
// to_packed = 1 gathers from the state buffer, 0 scatters into it
cudaError_t launch_halo_slices(double2* state, double2* packed, const int32_t* node, const int32_t* st, long long pairs,
                               int N, int with_cols, int to_packed, cudaStream_t s);

// out[L] = max over the nodes of level L of max(|re|, |im|) of their elements, as the bit pattern of the double
// (out must be zeroed; 256 entries); level: DEVICE uint8 per storage slot; per = complex elements per node
cudaError_t launch_level_max(const double2* state, const uint8_t* level, long long nodes, int per,
                             unsigned long long* out, cudaStream_t s);

// out[0], out[1] = Tr(A sigma_0) (re, im); A: DEVICE [N][N] complex128
cudaError_t launch_expectation(const double2* node0, const double2* A, int N, double* out, cudaStream_t s);

}  // namespace heom
