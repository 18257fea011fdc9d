// api.cu -- the C ABI of include/heom.h: argument checking, workspace layout, stream-ordered
// launches.  Every step of the hot path runs in the kernels; nothing here computes on the host
// beyond the one-time hierarchy/coefficient build.
#include "../../include/heom.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "hierarchy.hpp"
#include "kernels.cuh"

using namespace heom;

struct heom_ctx {
  Hierarchy h;                      // h.N = system states; h.W = B*M modes (tuple length, host tables)
  Coefficients c;                   // per bath: [B*M] / [B]; what heom_get_coefficients returns
  // Bath -> state map (heom_create_sites; identity for heom_create).  The kernels index modes per STATE
  // (l_dev = state*M + k, Wd = N*M): a state without a bath gets M mode columns whose links are all invalid
  // and whose coupling constants are zero, so no kernel knows about the map.
  int B = 0;                        // baths
  std::vector<int> site;            // [B] state of bath b
  std::vector<int> bath_of;         // [N] bath of state s, -1 = none
  Coefficients cd;                  // the same coefficients in the kernels' per-state mode indexing [Wd] / [N]
  // General system-bath operators (heom_create_general): bath b couples through the projectors on the states
  // bst[bptr[b]..bptr[b+1]) (the sums over s of Eq. 14-17), H may be complex Hermitian (Eq. 51).  Such a
  // context keeps the HOST mode indexing on the device (l = b*M + k, Wd = B*M) and runs the general kernels.
  bool general = false;             // = need_general || (mma_opt == 1 && eligible)
  bool need_general = false;        // the lists or a complex H ask for it
  int mma_opt = -1;                 // option "mma": -1 auto, 0 never for site-map contexts, 1 whenever eligible
  std::vector<int> bptr, bst;       // bath -> states (always filled)
  std::vector<int> sptr, sbl;       // state -> baths (CSR)
  std::vector<uint32_t> bmask;      // [B][4] membership bits of the bath's states
  bool use_mma = false;
  std::vector<double> Him;          // [N][N] imaginary part of H (general contexts created with one; else empty)
  int terminator_form = 0;          // option "terminator_form" (R12)
  std::vector<double> lambda, nu;   // bath parameters (kept for the "pade" option)
  double T_kelvin = 0;
  int pade = 0;
  std::vector<double> H;      // [N][N]
  std::vector<double> Tterm;  // [N][N]
  int device = 0;
  int order = 1;
  int kernel = 1;
  int timing = 0;
  bool hierarchy_built = false;
  int built_order = -1;
  std::string err;
  // workspace
  bool bound = false;
  bool have_state = false;
  cudaStream_t stream = nullptr;
  int stride = 0;  // complex elements per node
  size_t state_bytes = 0;
  double2 *y = nullptr, *acc = nullptr, *xa = nullptr, *xb = nullptr;
  int32_t *d_plus = nullptr, *d_minus = nullptr, *d_slot = nullptr;
  // Hermitian fast path of the pipelined kernel
  int herm_opt = 1;          // option "hermitian": 1 = use it when the state is exactly Hermitian
  bool state_hermitian = false;
  // persistent pipelined kernel (kernels_hpipe.cu)
  bool use_hpipe = false;
  int32_t* d_linksP = nullptr;
  int lrowP = 0;
  int warps_per_cta = 0;     // option "warps_per_cta": 0 = as many as fit
  // tensor-core kernel for large N (kernels_large.cu)
  bool use_tiny = false;     // whole-propagation kernel for tiny hierarchies (kernels_tiny.cu)
  bool use_large = false;
  int64_t* d_lptr = nullptr;
  void* d_lent = nullptr;
  int32_t* d_mrows = nullptr;        // large kernel: dense link rows (mma_pack_row format)
  double *d_Hs = nullptr, *d_delta = nullptr;
  double* d_Him = nullptr;          // general contexts: imaginary part of H (cm^-1)
  int32_t *d_sptr = nullptr, *d_sbl = nullptr;
  uint32_t* d_bmask = nullptr;
  double2* d_A = nullptr;    // operator of heom_expectation
  // column-sparse states (kernels_ket.cu): sigma_u = v_u e_col^T, selected by heom_set_state after an exact check
  int ket_opt = 1;           // option "ket": 1 = use the column kernel when the conditions hold, 0 = never
  int ket_col = -1;          // >= 0: the state is held as kets [nodes][N] (ky, kacc in the y region; kxa, kxb in acc's)
  double2* d_S0 = nullptr;   // sigma_0 expanded to a full matrix for the observables
  // one rank's part of a hierarchy sharded over several GPUs (heom_create_partition)
  bool partitioned = false;
  int part_rank = 0, part_world = 1;
  Partition part;
  uint8_t* d_level = nullptr;         // hierarchy level of every storage slot (heom_level_max)
  unsigned long long* d_lmax = nullptr;   // [256] scratch of heom_level_max
  int32_t* d_send = nullptr; // DEVICE copy of part.send_idx
  int32_t *d_spn = nullptr, *d_sps = nullptr, *d_rpn = nullptr, *d_rps = nullptr;   // slice-halo pair lists
  size_t n_links = 0;
  unsigned long long* d_tickets = nullptr;   // work counter of the persistent kernel
  unsigned long long ticket_base = 0;
  int rk4_form = -1;         // option "rk4_form": 0 classical stages, 1 Horner form (where the kernel supports it), -1 auto
  int l2_fetch = 0;          // option "l2_fetch": cudaLimitMaxL2FetchGranularity in bytes, 0 = leave the default
  int l2_persist = 0;        // option "l2_persist": percent of the device's maximum persisting-L2 carve-out to request
  int sms = 148;
  uint8_t* d_tuples = nullptr;
  double *d_damp = nullptr, *d_H = nullptr, *d_T = nullptr, *d_ap = nullptr, *d_amx = nullptr,
         *d_amo = nullptr, *d_scratch = nullptr;
  double* h_pinned = nullptr;  // small pinned staging (sigma_0 / populations)
  int64_t launches = 0;
  // per-launch timing
  std::vector<cudaEvent_t> ev;  // pairs
  size_t ev_used = 0;
};

namespace {

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

heom_status fail(heom_ctx* c, heom_status s, const std::string& msg) {
  if (c) c->err = msg;
  return s;
}
heom_status cuda_fail(heom_ctx* c, cudaError_t e, const char* where) {
  return fail(c, HEOM_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                                   \
  do {                                                             \
    cudaError_t e_ = (call);                                       \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);       \
  } while (0)

int dev_modes(const heom_ctx* c) { return c->general ? c->h.W : c->h.N * c->h.M; }
// storage slot of the hierarchy's root node sigma_0 (-1: a partition that does not hold it)
int64_t root_slot(const heom_ctx* c) { return c->partitioned ? c->part.root : (int64_t)c->h.slot_of[0]; }   // Wd: mode columns of the device tables

// c->cd, c->Tterm from c->c and the bath -> state map
void expand_coefficients(heom_ctx* c) {
  const int N = c->h.N, M = c->h.M, D1 = c->h.D + 1, Wd = N * M;
  if (c->general) {
    // host mode indexing on the device; Eq. 14's mask from the membership q_b of every bath: as printed
    // sum_s V_s^x V_s^x = (1 - delta_ij)(q_b(i) + q_b(j)), or (sum_s V_s^x)^2 = (q_b(i) - q_b(j))^2 (R12)
    c->cd = c->c;
    c->Tterm.assign((size_t)N * N, 0.0);
    for (int b = 0; b < c->B; ++b) {
      std::vector<int> q((size_t)N, 0);
      for (int e = c->bptr[(size_t)b]; e < c->bptr[(size_t)b + 1]; ++e) q[(size_t)c->bst[(size_t)e]] = 1;
      for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
          const int m = c->terminator_form ? (q[i] - q[j]) * (q[i] - q[j]) : (i != j) * (q[i] + q[j]);
          c->Tterm[(size_t)i * N + j] += c->c.delta[(size_t)b] * m;
        }
    }
    return;
  }
  Coefficients& d = c->cd;
  d.beta_hbar = c->c.beta_hbar;
  d.gamma.assign((size_t)Wd, 0.0); d.c_re.assign((size_t)Wd, 0.0); d.c_im.assign((size_t)Wd, 0.0);
  d.delta.assign((size_t)N, 0.0);
  d.a_plus.assign((size_t)Wd * D1, 0.0); d.a_minus_x.assign((size_t)Wd * D1, 0.0); d.a_minus_o.assign((size_t)Wd * D1, 0.0);
  for (int s = 0; s < N; ++s) {
    const int b = c->bath_of[(size_t)s];
    if (b < 0) continue;
    d.delta[(size_t)s] = c->c.delta[(size_t)b];
    for (int k = 0; k < M; ++k) {
      const size_t ld = (size_t)s * M + k, lh = (size_t)b * M + k;
      d.gamma[ld] = c->c.gamma[lh]; d.c_re[ld] = c->c.c_re[lh]; d.c_im[ld] = c->c.c_im[lh];
      for (int n = 0; n < D1; ++n) {
        d.a_plus[ld * D1 + n] = c->c.a_plus[lh * D1 + n];
        d.a_minus_x[ld * D1 + n] = c->c.a_minus_x[lh * D1 + n];
        d.a_minus_o[ld * D1 + n] = c->c.a_minus_o[lh * D1 + n];
      }
    }
  }
  c->Tterm.assign((size_t)N * N, 0.0);
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j)
      if (i != j) c->Tterm[(size_t)i * N + j] = d.delta[(size_t)i] + d.delta[(size_t)j];  // Eq. 14 + 24
}

// site-map contexts may run in the general representation (host mode indexing, membership bits) to reach the
// tensor-core kernel of kernels_mma.cu; partitions keep the per-state representation
void update_general(heom_ctx* c) {
  const int N = c->h.N;
  const bool eligible = !c->partitioned && N >= 17 && N <= 96 && !c->bmask.empty();
  const bool want = c->mma_opt == 1 || (c->mma_opt == -1 && !large_supported(N, N * c->h.M));
  c->general = c->need_general || (eligible && want);
  expand_coefficients(c);
}

bool ensure_hierarchy(heom_ctx* c) {
  if (c->hierarchy_built && c->built_order == c->order) return true;
  std::string err;
  const int n_states = c->h.N;
  bool ok = build_hierarchy(c->B, c->h.K, c->h.D, c->partitioned ? 1 : c->order, c->h, err);   // tuples over the B*M modes
  if (ok && c->partitioned) ok = restrict_hierarchy(c->h, c->part_rank, c->part_world, c->site, c->part, err);
  c->h.N = n_states;
  if (!ok) { c->err = err; return false; }
  c->hierarchy_built = true;
  c->built_order = c->order;
  return true;
}

int node_stride(int N) { return N * N; }

struct Layout {
  size_t state, off_y, off_acc, off_xa, off_xb, off_plus, off_minus, off_slot, off_tuples, off_damp,
      off_H, off_T, off_ap, off_amx, off_amo, off_scratch, off_linksP, off_Hs, off_delta, off_Him, off_gen, off_A, off_S0, off_level, off_send, off_pairs, off_lptr, off_lent, off_mrows, total;
};

// Which kernel family the bound configuration will run (fixed by the shape and the "kernel" option), so that the
// workspace holds the link tables of that family only (config 3: 1.1 GB of plain tables against 1.7 GB of meta rows).
struct KernelChoice { bool hpipe, large, tiny, mma, plain_tables; };
KernelChoice kernel_choice(const heom_ctx* c) {
  KernelChoice k{};
  const int N = c->h.N, Wd = dev_modes(c), D = c->h.D;
  const long long nodes = (long long)c->h.nodes;
  k.large = c->kernel >= 1 && !c->general && large_supported(N, Wd);
  k.hpipe = c->kernel >= 1 && !c->general && hpipe_supported(N, Wd, D, nodes);
  k.tiny = c->kernel == 1 && !c->general && !c->partitioned && tiny_supported(N, Wd, D, nodes);
  k.mma = c->kernel >= 1 && c->general && mma_supported(N, Wd, c->B, (int)c->sbl.size(), !c->Him.empty());
  k.plain_tables = k.tiny || !(k.large || k.hpipe || k.mma);   // plus/minus/tuples [nodes][W]: generic and tiny kernels
  return k;
}

Layout layout_of(const heom_ctx* c) {
  Layout L{};
  const size_t nodes = (size_t)c->h.nodes, W = (size_t)dev_modes(c), N = (size_t)c->h.N, D1 = (size_t)c->h.D + 1;
  const KernelChoice kc = kernel_choice(c);
  const size_t tab = kc.plain_tables ? nodes * W : 0;
  L.state = align_up(nodes * (size_t)node_stride((int)N) * sizeof(double2));
  size_t o = 0;
  L.off_y = o; o += L.state;
  L.off_acc = o; o += L.state;
  L.off_xa = o; o += L.state;
  L.off_xb = o; o += L.state;
  L.off_plus = o; o += align_up(tab * 4);
  L.off_minus = o; o += align_up(tab * 4);
  L.off_slot = o; o += align_up(nodes * 4);
  L.off_tuples = o; o += align_up(tab);
  L.off_damp = o; o += align_up((nodes + 1) * 8);
  L.off_H = o; o += align_up(N * N * 8);
  L.off_T = o; o += align_up(N * N * 8);
  L.off_ap = o; o += align_up(W * D1 * 8);
  L.off_amx = o; o += align_up(W * D1 * 8);
  L.off_amo = o; o += align_up(W * D1 * 8);
  L.off_scratch = o; o += align_up((N + 2) * 8 + 128);
  L.off_linksP = o; o += align_up(kc.hpipe ? nodes * (size_t)hpipe_links_row((int)N, c->h.M) * 4 : 0);
  L.off_Hs = o; o += align_up(N * N * 8);
  L.off_delta = o; o += align_up(N * 8);
  L.off_Him = o; o += align_up(N * N * 8);
  L.off_gen = o; o += align_up((N + 1) * 4) + align_up(c->sbl.size() * 4 + 16) + align_up((size_t)c->B * 16 + 16);
  L.off_A = o; o += align_up(N * N * 16);
  L.off_S0 = o; o += align_up(N * N * 16);
  L.off_level = o; o += align_up(nodes + 16) + align_up(256 * 8);
  L.off_send = o; o += align_up(c->part.send_idx.size() * 4 + 16);
  L.off_pairs = o; o += 2 * align_up(c->part.send_pair_node.size() * 4 + 16) + 2 * align_up(c->part.recv_pair_node.size() * 4 + 16);
  if (kc.mma) { L.off_lptr = o; L.off_lent = o; o += align_up(nodes * (size_t)mma_link_row((int)W) * 4); }
  if (kc.large) {
    // CSR link list: one 16-byte entry per valid "+" and per valid "-" link (a partition's table has links for its
    // owned rows only, so the two counts differ there)
    size_t links = 0;
    for (size_t q = 0; q < c->h.minus.size(); ++q) links += (c->h.minus[q] >= 0) + (c->h.plus[q] >= 0);
    L.off_lptr = o; o += align_up((nodes + 1) * 8);
    L.off_lent = o; o += align_up(links * 16 + 16);
    // dense link rows for the Hermitian variant's row-wise gathers
    L.off_mrows = o; o += align_up(nodes * (size_t)mma_link_row((int)W) * 4);
  }
  L.total = o;
  return L;
}

RhsParams base_params(const heom_ctx* c) {
  RhsParams p{};
  p.N = c->h.N; p.M = c->h.M; p.W = dev_modes(c); p.D = c->h.D;
  // a partition computes its OWNED rows only (the first n_owned local nodes); the ghost rows behind them are
  // read by the gathers and written by the halo exchange, never by a kernel
  p.nodes = c->partitioned ? (int)c->part.n_owned : (int)c->h.nodes;
  p.stride = c->stride;
  p.inv_hbar = 1.0 / kHbar;
  p.H = c->d_H; p.Tterm = c->d_T; p.damp = c->d_damp;
  p.plus = c->d_plus; p.minus = c->d_minus; p.tuples = c->d_tuples;
  p.a_plus = c->d_ap; p.a_minus_x = c->d_amx; p.a_minus_o = c->d_amo;
  if (c->general) {
    p.gen = 1; p.B = c->B; p.sptr = c->d_sptr; p.sbl = c->d_sbl; p.bmask = c->d_bmask;
    p.Him = c->Him.empty() ? nullptr : c->d_Him;
  }
  return p;
}

heom_status launch_rhs(heom_ctx* ctx, const RhsParams& p) {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (ctx->timing) {
    if (ctx->ev_used + 2 > ctx->ev.size()) {
      for (int q = 0; q < 2; ++q) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        ctx->ev.push_back(e);
      }
    }
    e0 = ctx->ev[ctx->ev_used]; e1 = ctx->ev[ctx->ev_used + 1];
    ctx->ev_used += 2;
    CU(cudaEventRecord(e0, ctx->stream));
  }
  if (ctx->ket_col >= 0)
    CU(launch_rhs_ket(p, ctx->d_linksP, ctx->lrowP, ctx->ket_col, ctx->cd.a_plus.data(), ctx->cd.a_minus_x.data(),
                      ctx->cd.a_minus_o.data(), ctx->H.data(), ctx->cd.delta.data(), ctx->sms, ctx->stream));
  else if (ctx->use_mma)
    CU(launch_rhs_mma(p, (const int32_t*)ctx->d_lent, mma_link_row(p.W), ctx->cd.a_plus.data(), ctx->cd.a_minus_x.data(),
                      ctx->cd.a_minus_o.data(), ctx->herm_opt && ctx->state_hermitian, ctx->sms, ctx->d_tickets,
                      &ctx->ticket_base, ctx->stream));
  else if (ctx->use_large)
    CU(launch_rhs_large(p, ctx->d_lptr, ctx->d_lent, ctx->d_mrows, mma_link_row(p.W), ctx->d_Hs, ctx->d_delta, ctx->cd.a_plus.data(),
                        ctx->cd.a_minus_x.data(), ctx->cd.a_minus_o.data(), ctx->herm_opt && ctx->state_hermitian,
                        ctx->sms, ctx->d_tickets, &ctx->ticket_base, ctx->stream));
  else if (ctx->use_hpipe)
    CU(launch_rhs_hpipe(p, ctx->d_linksP, ctx->lrowP, ctx->cd.a_plus.data(), ctx->cd.a_minus_x.data(),
                        ctx->cd.a_minus_o.data(), ctx->H.data(), ctx->cd.delta.data(),
                        ctx->herm_opt && ctx->state_hermitian, ctx->warps_per_cta, ctx->sms, ctx->d_tickets,
                        &ctx->ticket_base, ctx->stream));
  else CU(launch_rhs_generic(p, ctx->stream));
  ctx->launches += 1;
  if (ctx->timing) CU(cudaEventRecord(e1, ctx->stream));
  return HEOM_OK;
}

// ket buffers: two in the y region, two in the acc region (each region holds nodes*N*N >= 2*nodes*N elements)
double2* ket_buf(const heom_ctx* c, int which) {
  const size_t n = (size_t)c->h.nodes * c->h.N;
  double2* base = (which < 2) ? c->y : c->acc;
  return base + (size_t)(which & 1) * n;
}
enum { KET_Y = 0, KET_ACC = 1, KET_XA = 2, KET_XB = 3 };

// DEVICE pointer to sigma_0 as a full N x N matrix (ket mode: expanded into d_S0 first)
heom_status sigma0_matrix(heom_ctx* ctx, const double2** out) {
  if (root_slot(ctx) < 0) return fail(ctx, HEOM_ESTATE, "sigma_0 is not held by this partition");
  if (ctx->ket_col < 0) { *out = ctx->y + (size_t)root_slot(ctx) * ctx->stride; return HEOM_OK; }
  CU(launch_ket_expand(ket_buf(ctx, KET_Y) + (size_t)ctx->h.slot_of[0] * ctx->h.N, ctx->d_S0, 1, ctx->h.N,
                       ctx->ket_col, ctx->stream));
  ctx->launches += 1;
  *out = ctx->d_S0;
  return HEOM_OK;
}

// One fused RHS + RK4-stage launch (stage = 0..3) of the matrix kernels, in the form the kernel in use takes (R6):
//  - Horner (pipelined small-N and tensor-core kernels unless rk4_form = 0): w <- y + (dt/s) f(w), s = 4, 3, 2, 1,
//      xa = y + dt/4 f(y) | xb = y + dt/3 f(xa) | xa = y + dt/2 f(xb) | y = y + dt f(xa)  (in place)
//      no running sum: 2 + 3 + 3 + 3 = 11 state sizes of traffic per step, three buffers
//  - classical: k1 = f(y); xa = y + dt/2 k1; acc = y + dt/6 k1 | k2 = f(xa); xb = y + dt/2 k2; acc += dt/3 k2 |
//               k3 = f(xb); xa = y + dt k3; acc += dt/3 k3     | k4 = f(xa); y = acc + dt/6 k4     (16 state sizes)
// After the stage the next stage's input is xa (stages 0, 2), xb (stage 1) or y (stage 3): heom_stage_output.
heom_status launch_stage(heom_ctx* ctx, double dt, int stage) {
  RhsParams p = base_params(ctx);
  p.rhs_only = 0;
  const bool horner = (ctx->use_large || ctx->use_hpipe || ctx->use_mma) && ctx->rk4_form != 0;
  p.x = stage == 0 ? ctx->y : (stage == 2 ? ctx->xb : ctx->xa);
  p.y = ctx->y;
  if (horner) {
    p.horner = 1;
    p.out_x = stage == 3 ? ctx->y : (stage == 1 ? ctx->xb : ctx->xa);
    p.acc_in = nullptr; p.out_acc = nullptr;
    p.ax = dt / (double)(4 - stage);
    p.bx = 0.0;
    return launch_rhs(ctx, p);
  }
  p.out_x = stage == 3 ? nullptr : (stage == 1 ? ctx->xb : ctx->xa);
  p.acc_in = stage == 0 ? ctx->y : ctx->acc;
  p.out_acc = stage == 3 ? ctx->y : ctx->acc;
  p.ax = stage == 2 ? dt : dt / 2.0;
  p.bx = (stage == 0 || stage == 3) ? dt / 6.0 : dt / 3.0;
  return launch_rhs(ctx, p);
}

}  // namespace

extern "C" {

static heom_status create_impl(heom_ctx** out, int n_states, const double* H_cm, const double* H_im_cm, int n_baths,
                               const int* bath_ptr, const int* bath_states, const double* lambda_cm,
                               const double* nu_per_fs, double T_kelvin, int K, int D, int device, int rank, int world) {
  if (!out) return HEOM_EINVAL;
  *out = nullptr;
  if (world < 0 || (world > 0 && (rank < 0 || rank >= world))) return HEOM_EINVAL;
  if (!H_cm || !lambda_cm || !nu_per_fs || !bath_ptr || !bath_states || n_states < 1 || n_baths < 1 ||
      K < 0 || D < 0 || D > 255 || device < 0)
    return HEOM_EINVAL;
  for (int i = 0; i < n_states; ++i)
    for (int j = 0; j < n_states; ++j) {
      const double a = H_cm[(size_t)i * n_states + j], b = H_cm[(size_t)j * n_states + i];
      if (!std::isfinite(a) || a != b) return HEOM_EINVAL;
      if (H_im_cm) {
        const double c = H_im_cm[(size_t)i * n_states + j], d = H_im_cm[(size_t)j * n_states + i];
        if (!std::isfinite(c) || c != -d) return HEOM_EINVAL;                      // Hermitian
      }
    }
  if (bath_ptr[0] != 0) return HEOM_EINVAL;
  std::vector<int> bath_of((size_t)n_states, -1);
  bool general = H_im_cm != nullptr;
  for (int b = 0; b < n_baths; ++b) {
    if (bath_ptr[b + 1] <= bath_ptr[b]) return HEOM_EINVAL;                        // S(b) >= 1
    if (bath_ptr[b + 1] - bath_ptr[b] > 1) general = true;
    for (int e = bath_ptr[b]; e < bath_ptr[b + 1]; ++e) {
      const int s = bath_states[e];
      if (s < 0 || s >= n_states) return HEOM_EINVAL;
      for (int e2 = bath_ptr[b]; e2 < e; ++e2) if (bath_states[e2] == s) return HEOM_EINVAL;   // a state once per bath
      if (bath_of[(size_t)s] >= 0) general = true;                                 // several baths on one state
      bath_of[(size_t)s] = b;
    }
  }
  if (general && (world > 0 || n_states > 128)) return HEOM_EINVAL;   // general contexts: one GPU, 128 membership bits
  heom_ctx* c = new (std::nothrow) heom_ctx();
  if (!c) return HEOM_ENOMEM;
  c->device = device;
  c->partitioned = world > 0;
  c->part_rank = rank; c->part_world = world > 0 ? world : 1;
  c->B = n_baths;
  c->general = c->need_general = general;
  c->bptr.assign(bath_ptr, bath_ptr + n_baths + 1);
  c->bst.assign(bath_states, bath_states + bath_ptr[n_baths]);
  if (!general) {
    c->site.assign(bath_states, bath_states + n_baths);
    c->bath_of = bath_of;
  }
  if (n_states <= 128) {
    std::vector<std::vector<int>> of((size_t)n_states);
    c->bmask.assign((size_t)n_baths * 4, 0u);
    for (int b = 0; b < n_baths; ++b)
      for (int e = bath_ptr[b]; e < bath_ptr[b + 1]; ++e) {
        const int s = bath_states[e];
        of[(size_t)s].push_back(b);
        c->bmask[(size_t)b * 4 + (s >> 5)] |= 1u << (s & 31);
      }
    c->sptr.assign(1, 0);
    for (int s = 0; s < n_states; ++s) {
      c->sbl.insert(c->sbl.end(), of[(size_t)s].begin(), of[(size_t)s].end());
      c->sptr.push_back((int)c->sbl.size());
    }
    if (H_im_cm) c->Him.assign(H_im_cm, H_im_cm + (size_t)n_states * n_states);
  }
  c->h.N = n_states; c->h.K = K; c->h.M = K + 1; c->h.W = n_baths * (K + 1); c->h.D = D;
  std::string err;
  if (!build_coefficients(n_baths, K, D, lambda_cm, nu_per_fs, T_kelvin, 0, c->c, err)) {
    delete c;
    return HEOM_EINVAL;
  }
  c->lambda.assign(lambda_cm, lambda_cm + n_baths);
  c->nu.assign(nu_per_fs, nu_per_fs + n_baths);
  c->T_kelvin = T_kelvin;
  c->H.assign(H_cm, H_cm + (size_t)n_states * n_states);
  update_general(c);
  if (!ensure_hierarchy(c)) {
    const bool oom = c->err.find("memory") != std::string::npos;
    delete c;
    return oom ? HEOM_ENOMEM : HEOM_EINVAL;
  }
  *out = c;
  return HEOM_OK;
}

static heom_status create_sites_impl(heom_ctx** out, int n_states, const double* H_cm, int n_baths,
                                     const int* bath_state, const double* lambda_cm, const double* nu_per_fs,
                                     double T_kelvin, int K, int D, int device, int rank, int world) {
  if (out) *out = nullptr;
  if (!bath_state || n_baths < 1 || n_baths > n_states) return HEOM_EINVAL;
  std::vector<int> ptr((size_t)n_baths + 1);
  for (int b = 0; b <= n_baths; ++b) ptr[(size_t)b] = b;
  for (int b = 0; b < n_baths; ++b)
    for (int b2 = 0; b2 < b; ++b2) if (bath_state[b2] == bath_state[b]) return HEOM_EINVAL;   // one bath per state at most
  return create_impl(out, n_states, H_cm, nullptr, n_baths, ptr.data(), bath_state, lambda_cm, nu_per_fs, T_kelvin, K, D,
                     device, rank, world);
}

heom_status heom_create_sites(heom_ctx** out, int n_states, const double* H_cm, int n_baths, const int* bath_state,
                              const double* lambda_cm, const double* nu_per_fs, double T_kelvin, int K, int D,
                              int device) {
  return create_sites_impl(out, n_states, H_cm, n_baths, bath_state, lambda_cm, nu_per_fs, T_kelvin, K, D, device, 0, 0);
}

heom_status heom_create_general(heom_ctx** out, int n_states, const double* H_re_cm, const double* H_im_cm, int n_baths,
                                const int* bath_ptr, const int* bath_states, const double* lambda_cm,
                                const double* nu_per_fs, double T_kelvin, int K, int D, int device) {
  return create_impl(out, n_states, H_re_cm, H_im_cm, n_baths, bath_ptr, bath_states, lambda_cm, nu_per_fs, T_kelvin, K, D,
                     device, 0, 0);
}

heom_status heom_create_partition(heom_ctx** out, int n_states, const double* H_cm, int n_baths, const int* bath_state,
                                  const double* lambda_cm, const double* nu_per_fs, double T_kelvin, int K, int D,
                                  int device, int rank, int world) {
  if (world < 1) return HEOM_EINVAL;
  return create_sites_impl(out, n_states, H_cm, n_baths, bath_state, lambda_cm, nu_per_fs, T_kelvin, K, D, device, rank, world);
}

int64_t heom_partition_owned(const heom_ctx* c) { return !c ? -1 : (c->partitioned ? c->part.n_owned : c->h.nodes); }

heom_status heom_partition_plan(const heom_ctx* c, int64_t* global_ids, int64_t* send_counts, int64_t* recv_counts,
                                int32_t* send_idx) {
  if (!c || !c->partitioned) return HEOM_EINVAL;
  const Partition& q = c->part;
  if (global_ids) std::memcpy(global_ids, q.global_id.data(), q.global_id.size() * 8);
  if (send_counts) std::memcpy(send_counts, q.send_counts.data(), q.send_counts.size() * 8);
  if (recv_counts) std::memcpy(recv_counts, q.recv_counts.data(), q.recv_counts.size() * 8);
  if (send_idx && !q.send_idx.empty()) std::memcpy(send_idx, q.send_idx.data(), q.send_idx.size() * 4);
  return HEOM_OK;
}

heom_status heom_create(heom_ctx** out, int n_sites, const double* H_cm, const double* lambda_cm,
                        const double* nu_per_fs, double T_kelvin, int K, int D, int device) {
  if (!out) return HEOM_EINVAL;
  *out = nullptr;
  if (n_sites < 1) return HEOM_EINVAL;
  std::vector<int> ident((size_t)n_sites);
  for (int b = 0; b < n_sites; ++b) ident[(size_t)b] = b;
  return heom_create_sites(out, n_sites, H_cm, n_sites, ident.data(), lambda_cm, nu_per_fs, T_kelvin, K, D, device);
}

void heom_destroy(heom_ctx* c) {
  if (!c) return;
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  delete c;
}

heom_status heom_set_option(heom_ctx* ctx, const char* name, int value) {
  if (!ctx || !name) return HEOM_EINVAL;
  const std::string s(name);
  if (s == "timing") { ctx->timing = value ? 1 : 0; return HEOM_OK; }
  if (s == "hermitian") { ctx->herm_opt = value ? 1 : 0; return HEOM_OK; }
  if (s == "l2_persist") {
    if (value < 0 || value > 100) return fail(ctx, HEOM_EINVAL, "l2_persist must be 0..100 (percent of the maximum)");
    ctx->l2_persist = value;
    return HEOM_OK;
  }
  if (s == "l2_fetch") {
    if (value != 0 && value != 32 && value != 64 && value != 128) return fail(ctx, HEOM_EINVAL, "l2_fetch must be 0, 32, 64 or 128");
    ctx->l2_fetch = value;
    return HEOM_OK;
  }
  if (s == "ket") { ctx->ket_opt = value ? 1 : 0; return HEOM_OK; }   // takes effect at the next heom_set_state
  if (s == "rk4_form") {
    if (value < -1 || value > 1) return fail(ctx, HEOM_EINVAL, "rk4_form must be -1, 0 or 1");
    ctx->rk4_form = value;
    return HEOM_OK;
  }
  if (s == "warps_per_cta") {
    if (value < 0 || value > 32) return fail(ctx, HEOM_EINVAL, "warps_per_cta must be 0..32");
    ctx->warps_per_cta = value;
    return HEOM_OK;
  }
  if (ctx->bound) return fail(ctx, HEOM_ESTATE, "option must be set before heom_bind_workspace");
  if (s == "mma") {
    // site-map contexts (one state per bath, real H) on the general tensor-core kernel: -1 = where no other
    // specialised kernel exists (17 <= N <= 96 except 32, 64, 96), 0 = never, 1 = whenever 17 <= N <= 96
    if (value < -1 || value > 1) return fail(ctx, HEOM_EINVAL, "mma must be -1, 0 or 1");
    ctx->mma_opt = value;
    update_general(ctx);
    return HEOM_OK;
  }
  if (s == "terminator_form") {
    if (value != 0 && value != 1) return fail(ctx, HEOM_EINVAL, "terminator_form must be 0 or 1");
    ctx->terminator_form = value;
    expand_coefficients(ctx);
    return HEOM_OK;
  }
  if (s == "pade") {
    Coefficients nc;
    std::string err;
    if (!build_coefficients(ctx->B, ctx->h.K, ctx->h.D, ctx->lambda.data(), ctx->nu.data(), ctx->T_kelvin,
                            value ? 1 : 0, nc, err))
      return fail(ctx, HEOM_EINVAL, err);
    ctx->c = nc;
    ctx->pade = value ? 1 : 0;
    expand_coefficients(ctx);
    return HEOM_OK;
  }
  if (s == "order") {
    if (value != 0 && value != 1) return fail(ctx, HEOM_EINVAL, "order must be 0 or 1");
    if (ctx->partitioned) return fail(ctx, HEOM_EINVAL, "a partition keeps its own node order");
    ctx->order = value;
    return HEOM_OK;
  }
  if (s == "kernel") {
    if (value < 0 || value > 2) return fail(ctx, HEOM_EINVAL, "unknown kernel variant");
    ctx->kernel = value;
    return HEOM_OK;
  }
  return fail(ctx, HEOM_EINVAL, "unknown option");
}

int64_t heom_num_nodes(const heom_ctx* c) { return c ? c->h.nodes : -1; }
int heom_num_modes(const heom_ctx* c) { return c ? c->h.W : -1; }
int heom_num_baths(const heom_ctx* c) { return c ? c->B : -1; }

heom_status heom_get_tables(const heom_ctx* c, uint8_t* tuples, int32_t* plus, int32_t* minus) {
  if (!c) return HEOM_EINVAL;
  if (tuples) std::memcpy(tuples, c->h.tuples.data(), c->h.tuples.size());
  if (plus) std::memcpy(plus, c->h.plus.data(), c->h.plus.size() * sizeof(int32_t));
  if (minus) std::memcpy(minus, c->h.minus.data(), c->h.minus.size() * sizeof(int32_t));
  return HEOM_OK;
}

heom_status heom_get_coefficients(const heom_ctx* c, double* gamma, double* c_re, double* c_im,
                                  double* delta) {
  if (!c) return HEOM_EINVAL;
  const size_t W = (size_t)c->h.W;
  if (gamma) std::memcpy(gamma, c->c.gamma.data(), W * 8);
  if (c_re) std::memcpy(c_re, c->c.c_re.data(), W * 8);
  if (c_im) std::memcpy(c_im, c->c.c_im.data(), W * 8);
  if (delta) std::memcpy(delta, c->c.delta.data(), (size_t)c->B * 8);
  return HEOM_OK;
}

size_t heom_workspace_bytes(const heom_ctx* c) { return c ? layout_of(c).total : 0; }

}  // extern "C"

extern "C" {

heom_status heom_bind_workspace(heom_ctx* ctx, void* dev_ptr, size_t bytes, void* cuda_stream) {
  if (!ctx || !dev_ptr) return HEOM_EINVAL;
  if (((uintptr_t)dev_ptr & 255u) != 0) return fail(ctx, HEOM_EINVAL, "workspace must be 256-byte aligned");
  if (rhs_generic_smem(ctx->h.N) == 0)
    return fail(ctx, HEOM_EINVAL, "n_sites > 96 is not supported by this build");
  if (!ensure_hierarchy(ctx)) return HEOM_EINVAL;
  const Layout L = layout_of(ctx);
  if (bytes < L.total) return fail(ctx, HEOM_ENOMEM, "workspace smaller than heom_workspace_bytes()");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= ctx->device)
    return fail(ctx, HEOM_ECUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(e));
  CU(cudaSetDevice(ctx->device));
  if (ctx->l2_fetch) CU(cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, (size_t)ctx->l2_fetch));
  if (ctx->l2_persist) {
    cudaDeviceProp pr;
    CU(cudaGetDeviceProperties(&pr, ctx->device));
    CU(cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)pr.persistingL2CacheMaxSize / 100 * (size_t)ctx->l2_persist));
  }
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->stride = node_stride(ctx->h.N);
  ctx->state_bytes = L.state;
  char* base = (char*)dev_ptr;
  ctx->y = (double2*)(base + L.off_y);
  ctx->acc = (double2*)(base + L.off_acc);
  ctx->xa = (double2*)(base + L.off_xa);
  ctx->xb = (double2*)(base + L.off_xb);
  ctx->d_plus = (int32_t*)(base + L.off_plus);
  ctx->d_minus = (int32_t*)(base + L.off_minus);
  ctx->d_slot = (int32_t*)(base + L.off_slot);
  ctx->d_tuples = (uint8_t*)(base + L.off_tuples);
  ctx->d_damp = (double*)(base + L.off_damp);
  ctx->d_H = (double*)(base + L.off_H);
  ctx->d_T = (double*)(base + L.off_T);
  ctx->d_ap = (double*)(base + L.off_ap);
  ctx->d_amx = (double*)(base + L.off_amx);
  ctx->d_amo = (double*)(base + L.off_amo);
  ctx->d_scratch = (double*)(base + L.off_scratch);
  ctx->d_tickets = (unsigned long long*)(base + L.off_scratch + (((size_t)ctx->h.N + 2) * 8 + 63) / 64 * 64);
  ctx->ticket_base = 0;
  CU(cudaMemset(ctx->d_tickets, 0, 8));
  const int Wd = dev_modes(ctx);
  const KernelChoice kc = kernel_choice(ctx);
  ctx->use_large = kc.large;
  ctx->use_mma = kc.mma;
  ctx->use_tiny = kc.tiny;
  ctx->d_Hs = (double*)(base + L.off_Hs);
  ctx->d_delta = (double*)(base + L.off_delta);
  ctx->d_Him = (double*)(base + L.off_Him);
  ctx->d_sptr = (int32_t*)(base + L.off_gen);
  ctx->d_sbl = (int32_t*)(base + L.off_gen + align_up(((size_t)ctx->h.N + 1) * 4));
  ctx->d_bmask = (uint32_t*)((char*)ctx->d_sbl + align_up(ctx->sbl.size() * 4 + 16));
  if (ctx->general) {
    CU(cudaMemcpy(ctx->d_sptr, ctx->sptr.data(), ctx->sptr.size() * 4, cudaMemcpyHostToDevice));
    if (!ctx->sbl.empty()) CU(cudaMemcpy(ctx->d_sbl, ctx->sbl.data(), ctx->sbl.size() * 4, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_bmask, ctx->bmask.data(), ctx->bmask.size() * 4, cudaMemcpyHostToDevice));
    if (!ctx->Him.empty()) CU(cudaMemcpy(ctx->d_Him, ctx->Him.data(), ctx->Him.size() * 8, cudaMemcpyHostToDevice));
  }
  ctx->d_A = (double2*)(base + L.off_A);
  ctx->d_S0 = (double2*)(base + L.off_S0);
  ctx->d_level = (uint8_t*)(base + L.off_level);
  ctx->d_lmax = (unsigned long long*)(base + L.off_level + align_up((size_t)ctx->h.nodes + 16));
  {
    std::vector<uint8_t> lev((size_t)ctx->h.nodes, 0);
    for (int64_t u = 0; u < ctx->h.nodes; ++u) {
      int Ls = 0;
      for (int l = 0; l < ctx->h.W; ++l) Ls += ctx->h.tuples[(size_t)u * ctx->h.W + l];
      lev[(size_t)ctx->h.slot_of[(size_t)u]] = (uint8_t)Ls;
    }
    CU(cudaMemcpy(ctx->d_level, lev.data(), lev.size(), cudaMemcpyHostToDevice));
  }
  ctx->d_send = (int32_t*)(base + L.off_send);
  if (!ctx->part.send_idx.empty())
    CU(cudaMemcpy(ctx->d_send, ctx->part.send_idx.data(), ctx->part.send_idx.size() * 4, cudaMemcpyHostToDevice));
  {
    const Partition& q = ctx->part;
    const size_t ns = align_up(q.send_pair_node.size() * 4 + 16), nr = align_up(q.recv_pair_node.size() * 4 + 16);
    ctx->d_spn = (int32_t*)(base + L.off_pairs); ctx->d_sps = (int32_t*)(base + L.off_pairs + ns);
    ctx->d_rpn = (int32_t*)(base + L.off_pairs + 2 * ns); ctx->d_rps = (int32_t*)(base + L.off_pairs + 2 * ns + nr);
    if (!q.send_pair_node.empty()) {
      CU(cudaMemcpy(ctx->d_spn, q.send_pair_node.data(), q.send_pair_node.size() * 4, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_sps, q.send_pair_state.data(), q.send_pair_state.size() * 4, cudaMemcpyHostToDevice));
    }
    if (!q.recv_pair_node.empty()) {
      CU(cudaMemcpy(ctx->d_rpn, q.recv_pair_node.data(), q.recv_pair_node.size() * 4, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_rps, q.recv_pair_state.data(), q.recv_pair_state.size() * 4, cudaMemcpyHostToDevice));
    }
  }
  ctx->ket_col = -1;
  ctx->d_lptr = (int64_t*)(base + L.off_lptr);
  ctx->d_lent = (void*)(base + L.off_lent);
  ctx->d_mrows = (int32_t*)(base + L.off_mrows);
  ctx->d_linksP = (int32_t*)(base + L.off_linksP);
  ctx->lrowP = hpipe_links_row(ctx->h.N, ctx->h.M);
  ctx->use_hpipe = kc.hpipe && !kc.large;
  {
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, ctx->device));
    ctx->sms = prop.multiProcessorCount;
  }
  if (!ctx->h_pinned) CU(cudaMallocHost((void**)&ctx->h_pinned, ((size_t)ctx->h.N * ctx->h.N * 2 + 8) * 8));

  // Device tables in STORAGE-slot order: row slot_of[u] holds the slots of u's neighbours.
  const Hierarchy& h = ctx->h;
  const size_t nodes = (size_t)h.nodes, W = (size_t)Wd, Wh = (size_t)h.W, Mm = (size_t)h.M;
  try {
    std::vector<int32_t> tp(nodes * W), tm(nodes * W);
    std::vector<uint8_t> tt(nodes * W);
    std::vector<double> damp(nodes);
#pragma omp parallel for schedule(static)
    for (int64_t u = 0; u < (int64_t)nodes; ++u) {
      const size_t s = (size_t)h.slot_of[(size_t)u];
      double d = 0.0;
      for (size_t l = 0; l < W; ++l) {      // device mode column l = state*M + k (general contexts: l = b*M + k)
        const int bath = ctx->general ? (int)(l / Mm) : ctx->bath_of[l / Mm];
        if (bath < 0) { tp[s * W + l] = -1; tm[s * W + l] = -1; tt[s * W + l] = 0; continue; }
        const size_t lh = (size_t)bath * Mm + l % Mm;   // host mode index (Eq. 10)
        const int32_t a = h.plus[(size_t)u * Wh + lh], b = h.minus[(size_t)u * Wh + lh];
        tp[s * W + l] = a < 0 ? -1 : h.slot_of[(size_t)a];
        tm[s * W + l] = b < 0 ? -1 : h.slot_of[(size_t)b];
        const uint8_t n = h.tuples[(size_t)u * Wh + lh];
        tt[s * W + l] = n;
        d += (double)n * ctx->cd.gamma[l];  // Eq. 13
      }
      damp[s] = d;
    }
    if (kc.plain_tables) {
      CU(cudaMemcpy(ctx->d_plus, tp.data(), nodes * W * 4, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_minus, tm.data(), nodes * W * 4, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_tuples, tt.data(), nodes * W, cudaMemcpyHostToDevice));
    }
    CU(cudaMemset(ctx->d_damp + nodes, 0, 8));
    CU(cudaMemcpy(ctx->d_damp, damp.data(), nodes * 8, cudaMemcpyHostToDevice));
    if (ctx->use_mma) {
      const size_t mrow = (size_t)mma_link_row((int)W);
      std::vector<int32_t> rows(nodes * mrow, 0);
#pragma omp parallel for schedule(static)
      for (int64_t s = 0; s < (int64_t)nodes; ++s)
        mma_pack_row((int)W, &tp[(size_t)s * W], &tm[(size_t)s * W], &tt[(size_t)s * W], damp[(size_t)s], &rows[(size_t)s * mrow]);
      CU(cudaMemcpy(ctx->d_lent, rows.data(), nodes * mrow * 4, cudaMemcpyHostToDevice));
    }
    if (ctx->use_large) {
      // CSR link list in storage-slot order: "+" links first, then "-" links, of every node
      std::vector<int64_t> lptr(nodes + 1, 0);
      for (size_t s = 0; s < nodes; ++s) {
        int64_t cnt = 0;
        for (size_t l = 0; l < W; ++l) cnt += (tp[s * W + l] >= 0) + (tm[s * W + l] >= 0);
        lptr[s + 1] = lptr[s] + cnt;
      }
      std::vector<int32_t> lent((size_t)lptr[nodes] * 4 + 4, 0);
#pragma omp parallel for schedule(static)
      for (int64_t s = 0; s < (int64_t)nodes; ++s) {
        int32_t* e = &lent[(size_t)lptr[(size_t)s] * 4];
        for (size_t l = 0; l < W; ++l)
          if (tp[(size_t)s * W + l] >= 0) { e[0] = tp[(size_t)s * W + l]; e[1] = (int32_t)l; e[2] = 0; e[3] = tt[(size_t)s * W + l]; e += 4; }
        for (size_t l = 0; l < W; ++l)
          if (tm[(size_t)s * W + l] >= 0) { e[0] = tm[(size_t)s * W + l]; e[1] = (int32_t)l; e[2] = 1; e[3] = tt[(size_t)s * W + l]; e += 4; }
      }
      ctx->n_links = (size_t)lptr[nodes];
      {
        const size_t mrow = (size_t)mma_link_row((int)W);
        std::vector<int32_t> rows(nodes * mrow, 0);
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < (int64_t)nodes; ++s)
          mma_pack_row((int)W, &tp[(size_t)s * W], &tm[(size_t)s * W], &tt[(size_t)s * W], damp[(size_t)s], &rows[(size_t)s * mrow]);
        CU(cudaMemcpy(ctx->d_mrows, rows.data(), nodes * mrow * 4, cudaMemcpyHostToDevice));
      }
      CU(cudaMemcpy(ctx->d_lptr, lptr.data(), (nodes + 1) * 8, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_lent, lent.data(), (size_t)lptr[nodes] * 16 + 16, cudaMemcpyHostToDevice));
      std::vector<double> Hs(ctx->H);
      for (double& v : Hs) v *= 1.0 / kHbar;
      CU(cudaMemcpy(ctx->d_Hs, Hs.data(), Hs.size() * 8, cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_delta, ctx->cd.delta.data(), (size_t)h.N * 8, cudaMemcpyHostToDevice));
    }
    if (ctx->use_hpipe) {
      const size_t lrow = (size_t)ctx->lrowP;
      std::vector<int32_t> lk(nodes * lrow, 0);
#pragma omp parallel for schedule(static)
      for (int64_t s = 0; s < (int64_t)nodes; ++s)
        hpipe_pack_links(h.N, h.M, h.D, &tp[(size_t)s * W], &tm[(size_t)s * W], &tt[(size_t)s * W], damp[(size_t)s], &lk[(size_t)s * lrow]);
      CU(cudaMemcpy(ctx->d_linksP, lk.data(), nodes * lrow * 4, cudaMemcpyHostToDevice));
    }
  } catch (const std::bad_alloc&) {
    return fail(ctx, HEOM_ENOMEM, "out of host memory while staging the device tables");
  }
  const size_t NN = (size_t)h.N * h.N, WD = W * ((size_t)h.D + 1);
  CU(cudaMemcpy(ctx->d_slot, h.slot_of.data(), nodes * 4, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_H, ctx->H.data(), NN * 8, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_T, ctx->Tterm.data(), NN * 8, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_ap, ctx->cd.a_plus.data(), WD * 8, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_amx, ctx->cd.a_minus_x.data(), WD * 8, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_amo, ctx->cd.a_minus_o.data(), WD * 8, cudaMemcpyHostToDevice));
  // the uploads above are pageable-memory copies on the legacy stream: they may return before the DMA has landed,
  // and ctx->stream does not synchronise with the legacy stream -- wait for the device once, here
  CU(cudaDeviceSynchronize());
  ctx->bound = true;
  ctx->have_state = false;
  return HEOM_OK;
}

heom_status heom_set_state(heom_ctx* ctx, const double* sigma0) {
  if (!ctx || !sigma0) return HEOM_EINVAL;
  if (!ctx->bound) return fail(ctx, HEOM_ESTATE, "no workspace bound");
  const size_t NN = (size_t)ctx->h.N * ctx->h.N;
  for (size_t e = 0; e < 2 * NN; ++e)
    if (!std::isfinite(sigma0[e])) return fail(ctx, HEOM_EINVAL, "sigma0 has a non-finite entry");
  {
    const int N = ctx->h.N;
    bool herm = true;
    for (int i = 0; i < N && herm; ++i)
      for (int j = i; j < N; ++j) {
        const double ar = sigma0[2 * (i * N + j)], ai = sigma0[2 * (i * N + j) + 1];
        const double br = sigma0[2 * (j * N + i)], bi = sigma0[2 * (j * N + i) + 1];
        if (ar != br || ai != -bi) { herm = false; break; }
      }
    ctx->state_hermitian = herm;
  }
  ctx->ket_col = -1;
  if (ctx->ket_opt && !ctx->general && ctx->use_hpipe && !ctx->use_tiny && !ctx->partitioned && ket_supported(ctx->h.N, dev_modes(ctx), ctx->h.D)) {
    // column-sparse state?  exactly one non-zero column c, state c without a bath and uncoupled in H
    const int N = ctx->h.N;
    int col = -1, ncols = 0;
    for (int j = 0; j < N; ++j) {
      bool nz = false;
      for (int i = 0; i < N; ++i) nz = nz || sigma0[2 * (i * N + j)] != 0.0 || sigma0[2 * (i * N + j) + 1] != 0.0;
      if (nz) { col = j; ++ncols; }
    }
    bool ok = ncols == 1 && ctx->bath_of[(size_t)col] < 0;
    for (int j = 0; ok && j < N; ++j)
      if (j != col && ctx->H[(size_t)col * N + j] != 0.0) ok = false;
    if (ok) ctx->ket_col = col;
  }
  CU(cudaStreamSynchronize(ctx->stream));  // the pinned staging buffer may still be in flight
  if (ctx->ket_col >= 0) {
    const int N = ctx->h.N;
    for (int i = 0; i < N; ++i) {
      ctx->h_pinned[2 * i] = sigma0[2 * (i * N + ctx->ket_col)];
      ctx->h_pinned[2 * i + 1] = sigma0[2 * (i * N + ctx->ket_col) + 1];
    }
    double2* ky = ket_buf(ctx, KET_Y);
    CU(cudaMemsetAsync(ky, 0, (size_t)ctx->h.nodes * N * 16, ctx->stream));
    CU(cudaMemcpyAsync(ky + (size_t)ctx->h.slot_of[0] * N, ctx->h_pinned, (size_t)N * 16, cudaMemcpyHostToDevice,
                       ctx->stream));
    ctx->state_hermitian = false;
    ctx->have_state = true;
    return HEOM_OK;
  }
  std::memcpy(ctx->h_pinned, sigma0, NN * 16);
  CU(cudaMemsetAsync(ctx->y, 0, ctx->state_bytes, ctx->stream));
  if (root_slot(ctx) >= 0)   // a partition sets its copy of sigma_0 (owned or ghost) if it holds one
    CU(cudaMemcpyAsync(ctx->y + (size_t)root_slot(ctx) * ctx->stride, ctx->h_pinned, NN * 16,
                       cudaMemcpyHostToDevice, ctx->stream));
  ctx->have_state = true;
  return HEOM_OK;
}

heom_status heom_set_full_state(heom_ctx* ctx, const double* sigma) {
  if (!ctx || !sigma) return HEOM_EINVAL;
  if (!ctx->bound) return fail(ctx, HEOM_ESTATE, "no workspace bound");
  const size_t NN = (size_t)ctx->h.N * ctx->h.N, nodes = (size_t)ctx->h.nodes;
  ctx->ket_col = -1;
  {
    // exact Hermiticity of every node selects the row-gather kernel (checked, never assumed)
    const int N = ctx->h.N;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(| : bad)
    for (int64_t u = 0; u < (int64_t)nodes; ++u) {
      const double* a = sigma + (size_t)u * NN * 2;
      for (int i = 0; i < N; ++i)
        for (int j = i; j < N; ++j)
          if (a[2 * (i * N + j)] != a[2 * (j * N + i)] || a[2 * (i * N + j) + 1] != -a[2 * (j * N + i) + 1]) bad |= 1;
    }
    ctx->state_hermitian = !bad;
  }
  // stage in xa (pinned order, unpadded), then permute into y on the device
  CU(cudaMemcpyAsync(ctx->xa, sigma, nodes * NN * 16, cudaMemcpyHostToDevice, ctx->stream));
  CU(launch_permute(ctx->xa, ctx->y, ctx->d_slot, (int)nodes, (int)NN, ctx->stride, 1, ctx->stream));
  ctx->launches += 1;
  CU(cudaStreamSynchronize(ctx->stream));
  ctx->have_state = true;
  return HEOM_OK;
}

static heom_status read_back(heom_ctx* ctx, const double2* dev_state, double2* scratch, double* host) {
  const size_t NN = (size_t)ctx->h.N * ctx->h.N, nodes = (size_t)ctx->h.nodes;
  CU(launch_permute(dev_state, scratch, ctx->d_slot, (int)nodes, (int)NN, ctx->stride, 0, ctx->stream));
  ctx->launches += 1;
  CU(cudaMemcpyAsync(host, scratch, nodes * NN * 16, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return HEOM_OK;
}

heom_status heom_get_full_state(heom_ctx* ctx, double* sigma) {
  if (!ctx || !sigma) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  if (ctx->ket_col >= 0) {
    CU(launch_ket_expand(ket_buf(ctx, KET_Y), ctx->xa, ctx->h.nodes, ctx->h.N, ctx->ket_col, ctx->stream));
    ctx->launches += 1;
    return read_back(ctx, ctx->xa, ctx->xb, sigma);
  }
  return read_back(ctx, ctx->y, ctx->xa, sigma);
}

heom_status heom_rhs(heom_ctx* ctx, double* dsigma) {
  if (!ctx || !dsigma) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  RhsParams p = base_params(ctx);
  if (ctx->ket_col >= 0) {
    p.x = ket_buf(ctx, KET_Y); p.rhs_only = 1; p.out_acc = ket_buf(ctx, KET_XA);
    heom_status s = launch_rhs(ctx, p);
    if (s != HEOM_OK) return s;
    CU(launch_ket_expand(ket_buf(ctx, KET_XA), ctx->xa, ctx->h.nodes, ctx->h.N, ctx->ket_col, ctx->stream));
    ctx->launches += 1;
    return read_back(ctx, ctx->xa, ctx->xb, dsigma);
  }
  p.x = ctx->y; p.rhs_only = 1; p.out_acc = ctx->xa;
  heom_status s = launch_rhs(ctx, p);
  if (s != HEOM_OK) return s;
  return read_back(ctx, ctx->xa, ctx->xb, dsigma);
}

/* nsteps RK4 steps, four fused RHS + stage launches each (launch_stage above: Horner or classical form, R6). */
heom_status heom_rk4_steps(heom_ctx* ctx, double dt, int nsteps) {
  if (!ctx || nsteps < 0 || !std::isfinite(dt)) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  RhsParams p = base_params(ctx);
  p.rhs_only = 0;
  if (ctx->ket_col >= 0) {
    /* column-sparse state: Horner form (R6) on the kets, 4 launches per step, three ket buffers */
    double2 *ky = ket_buf(ctx, KET_Y), *kxa = ket_buf(ctx, KET_XA), *kxb = ket_buf(ctx, KET_XB);
    p.horner = 1; p.y = ky;
    for (int step = 0; step < nsteps; ++step) {
      heom_status s;
      p.x = ky; p.out_x = kxa; p.ax = dt / 4.0;
      if ((s = launch_rhs(ctx, p)) != HEOM_OK) return s;
      p.x = kxa; p.out_x = kxb; p.ax = dt / 3.0;
      if ((s = launch_rhs(ctx, p)) != HEOM_OK) return s;
      p.x = kxb; p.out_x = kxa; p.ax = dt / 2.0;
      if ((s = launch_rhs(ctx, p)) != HEOM_OK) return s;
      p.x = kxa; p.out_x = ky; p.ax = dt;                /* in place: only node u reads y_u */
      if ((s = launch_rhs(ctx, p)) != HEOM_OK) return s;
    }
    return HEOM_OK;
  }
  if (ctx->use_tiny && nsteps > 0) {
    /* launch-latency-bound hierarchies: all nsteps classical RK4 steps in one launch of one CTA */
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->timing) {
      while (ctx->ev_used + 2 > ctx->ev.size()) { cudaEvent_t e; CU(cudaEventCreate(&e)); ctx->ev.push_back(e); }
      e0 = ctx->ev[ctx->ev_used]; e1 = ctx->ev[ctx->ev_used + 1];
      ctx->ev_used += 2;
      CU(cudaEventRecord(e0, ctx->stream));
    }
    p.x = ctx->y;
    CU(launch_rk4_tiny(p, dt, nsteps, ctx->stream));
    ctx->launches += 1;
    if (ctx->timing) CU(cudaEventRecord(e1, ctx->stream));
    return HEOM_OK;
  }
  if (nsteps == 0) return HEOM_OK;
  if (ctx->partitioned && ctx->part_world > 1)
    return fail(ctx, HEOM_ESTATE, "a partition advances stage by stage (heom_rk4_stage + halo exchange)");
  for (int step = 0; step < nsteps; ++step)
    for (int stage = 0; stage < 4; ++stage) {
      heom_status s = launch_stage(ctx, dt, stage);
      if (s != HEOM_OK) return s;
    }
  return HEOM_OK;
}

heom_status heom_rk4_stage(heom_ctx* ctx, double dt, int stage) {
  if (!ctx || stage < 0 || stage > 3 || !std::isfinite(dt)) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  if (ctx->ket_col >= 0 || ctx->use_tiny)
    return fail(ctx, HEOM_ESTATE, "stage-wise stepping is for the matrix kernels (set options ket=0 and kernel=2)");
  return launch_stage(ctx, dt, stage);
}

heom_status heom_stage_output(heom_ctx* ctx, int stage, void** dev_ptr) {
  if (!ctx || !dev_ptr || stage < 0 || stage > 3) return HEOM_EINVAL;
  if (!ctx->bound) return fail(ctx, HEOM_ESTATE, "no workspace bound");
  *dev_ptr = (stage == 3) ? ctx->y : (stage == 1 ? ctx->xb : ctx->xa);
  return HEOM_OK;
}

heom_status heom_pack_halo(heom_ctx* ctx, const void* src_dev, void* dst_dev) {
  if (!ctx || !src_dev || !dst_dev) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->partitioned) return fail(ctx, HEOM_ESTATE, "not a bound partition");
  const long long rows = (long long)ctx->part.send_idx.size();
  if (rows == 0) return HEOM_OK;
  CU(launch_pack_rows((const double2*)src_dev, (double2*)dst_dev, ctx->d_send, rows, ctx->h.N * ctx->h.N, ctx->stride,
                      ctx->stream));
  ctx->launches += 1;
  return HEOM_OK;
}

heom_status heom_partition_plan_slices(const heom_ctx* c, int64_t* send_counts, int64_t* recv_counts,
                                       int32_t* send_node, int32_t* send_state, int32_t* recv_node, int32_t* recv_state) {
  if (!c || !c->partitioned) return HEOM_EINVAL;
  const Partition& q = c->part;
  if (send_counts) std::memcpy(send_counts, q.send_pair_counts.data(), q.send_pair_counts.size() * 8);
  if (recv_counts) std::memcpy(recv_counts, q.recv_pair_counts.data(), q.recv_pair_counts.size() * 8);
  if (send_node && !q.send_pair_node.empty()) std::memcpy(send_node, q.send_pair_node.data(), q.send_pair_node.size() * 4);
  if (send_state && !q.send_pair_state.empty()) std::memcpy(send_state, q.send_pair_state.data(), q.send_pair_state.size() * 4);
  if (recv_node && !q.recv_pair_node.empty()) std::memcpy(recv_node, q.recv_pair_node.data(), q.recv_pair_node.size() * 4);
  if (recv_state && !q.recv_pair_state.empty()) std::memcpy(recv_state, q.recv_pair_state.data(), q.recv_pair_state.size() * 4);
  return HEOM_OK;
}

int heom_halo_slice_elements(const heom_ctx* c) {
  if (!c) return -1;
  /* rows only while the state is exactly Hermitian and the row-gather kernels run, rows + columns otherwise */
  return (c->herm_opt && c->state_hermitian && (c->use_hpipe || c->use_large)) ? c->h.N : 2 * c->h.N;   // (mma: single GPU)
}

heom_status heom_pack_halo_slices(heom_ctx* ctx, const void* src_dev, void* dst_dev) {
  if (!ctx || !src_dev || !dst_dev) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->partitioned) return fail(ctx, HEOM_ESTATE, "not a bound partition");
  const long long pairs = (long long)ctx->part.send_pair_node.size();
  if (pairs == 0) return HEOM_OK;
  CU(launch_halo_slices((double2*)src_dev, (double2*)dst_dev, ctx->d_spn, ctx->d_sps, pairs, ctx->h.N,
                        heom_halo_slice_elements(ctx) == 2 * ctx->h.N, 1, ctx->stream));
  ctx->launches += 1;
  return HEOM_OK;
}

heom_status heom_unpack_halo_slices(heom_ctx* ctx, const void* src_dev, void* state_dev) {
  if (!ctx || !src_dev || !state_dev) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->partitioned) return fail(ctx, HEOM_ESTATE, "not a bound partition");
  const long long pairs = (long long)ctx->part.recv_pair_node.size();
  if (pairs == 0) return HEOM_OK;
  CU(launch_halo_slices((double2*)state_dev, (double2*)src_dev, ctx->d_rpn, ctx->d_rps, pairs, ctx->h.N,
                        heom_halo_slice_elements(ctx) == 2 * ctx->h.N, 0, ctx->stream));
  ctx->launches += 1;
  return HEOM_OK;
}

heom_status heom_sync(heom_ctx* ctx) {
  if (!ctx) return HEOM_EINVAL;
  if (!ctx->bound) return fail(ctx, HEOM_ESTATE, "no workspace bound");
  CU(cudaStreamSynchronize(ctx->stream));
  return HEOM_OK;
}

heom_status heom_set_hamiltonian(heom_ctx* ctx, const double* H_re_cm, const double* H_im_cm) {
  if (!ctx || !H_re_cm) return HEOM_EINVAL;
  const int N = ctx->h.N;
  if (H_im_cm && ctx->Him.empty())
    return fail(ctx, HEOM_EINVAL, "a complex H needs a context created by heom_create_general with H_im_cm != NULL");
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      const double a = H_re_cm[(size_t)i * N + j], b = H_re_cm[(size_t)j * N + i];
      if (!std::isfinite(a) || a != b) return fail(ctx, HEOM_EINVAL, "H_re must be finite and symmetric");
      if (H_im_cm) {
        const double c = H_im_cm[(size_t)i * N + j], d = H_im_cm[(size_t)j * N + i];
        if (!std::isfinite(c) || c != -d) return fail(ctx, HEOM_EINVAL, "H_im must be finite and antisymmetric");
      }
    }
  if (ctx->ket_col >= 0) {
    for (int j = 0; j < N; ++j)
      if (j != ctx->ket_col && H_re_cm[(size_t)ctx->ket_col * N + j] != 0.0)
        return fail(ctx, HEOM_ESTATE, "the column-sparse state needs its state uncoupled in H (set option ket=0)");
  }
  ctx->H.assign(H_re_cm, H_re_cm + (size_t)N * N);
  if (!ctx->Him.empty()) {
    if (H_im_cm) ctx->Him.assign(H_im_cm, H_im_cm + (size_t)N * N);
    else std::fill(ctx->Him.begin(), ctx->Him.end(), 0.0);
  }
  if (ctx->bound) {
    // stream-ordered: launches already enqueued keep the old H, later ones see the new one
    CU(cudaMemcpyAsync(ctx->d_H, ctx->H.data(), (size_t)N * N * 8, cudaMemcpyHostToDevice, ctx->stream));
    if (!ctx->Him.empty())
      CU(cudaMemcpyAsync(ctx->d_Him, ctx->Him.data(), (size_t)N * N * 8, cudaMemcpyHostToDevice, ctx->stream));
    if (ctx->use_large) {
      std::vector<double> Hs(ctx->H);
      for (double& v : Hs) v *= 1.0 / kHbar;
      CU(cudaMemcpyAsync(ctx->d_Hs, Hs.data(), Hs.size() * 8, cudaMemcpyHostToDevice, ctx->stream));
    }
  }
  return HEOM_OK;
}

heom_status heom_populations(heom_ctx* ctx, double* pop, double* trace_re, double* trace_im) {
  if (!ctx) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  const int N = ctx->h.N;
  const double2* s0 = nullptr;
  { heom_status st = sigma0_matrix(ctx, &s0); if (st != HEOM_OK) return st; }
  CU(launch_populations(s0, N, ctx->d_scratch, ctx->stream));
  ctx->launches += 1;
  CU(cudaMemcpyAsync(ctx->h_pinned, ctx->d_scratch, (size_t)(N + 2) * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (pop) std::memcpy(pop, ctx->h_pinned, (size_t)N * 8);
  if (trace_re) *trace_re = ctx->h_pinned[N];
  if (trace_im) *trace_im = ctx->h_pinned[N + 1];
  return HEOM_OK;
}

heom_status heom_level_max(heom_ctx* ctx, double* max_abs) {
  if (!ctx || !max_abs) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  const bool ket = ctx->ket_col >= 0;
  // a partition reports its owned nodes (ghost rows are copies)
  const long long n = ctx->partitioned ? (long long)ctx->part.n_owned : (long long)ctx->h.nodes;
  CU(cudaMemsetAsync(ctx->d_lmax, 0, 256 * 8, ctx->stream));
  CU(launch_level_max(ket ? ket_buf(ctx, KET_Y) : ctx->y, ctx->d_level, n, ket ? ctx->h.N : ctx->h.N * ctx->h.N,
                      ctx->d_lmax, ctx->stream));
  ctx->launches += 1;
  unsigned long long bits[256];
  CU(cudaMemcpyAsync(bits, ctx->d_lmax, 256 * 8, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int L = 0; L <= ctx->h.D; ++L) std::memcpy(&max_abs[L], &bits[L], 8);
  return HEOM_OK;
}

heom_status heom_expectation(heom_ctx* ctx, const double* A, double* re, double* im) {
  if (!ctx || !A) return HEOM_EINVAL;
  if (!ctx->bound || !ctx->have_state) return fail(ctx, HEOM_ESTATE, "no state set");
  const int N = ctx->h.N;
  const size_t NN = (size_t)N * N;
  for (size_t e = 0; e < 2 * NN; ++e)
    if (!std::isfinite(A[e])) return fail(ctx, HEOM_EINVAL, "operator has a non-finite entry");
  CU(cudaStreamSynchronize(ctx->stream));  // the pinned staging buffer may still be in flight
  std::memcpy(ctx->h_pinned, A, NN * 16);
  CU(cudaMemcpyAsync(ctx->d_A, ctx->h_pinned, NN * 16, cudaMemcpyHostToDevice, ctx->stream));
  const double2* s0 = nullptr;
  { heom_status st = sigma0_matrix(ctx, &s0); if (st != HEOM_OK) return st; }
  CU(launch_expectation(s0, ctx->d_A, N, ctx->d_scratch, ctx->stream));
  ctx->launches += 1;
  CU(cudaMemcpyAsync(ctx->h_pinned, ctx->d_scratch, 16, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (re) *re = ctx->h_pinned[0];
  if (im) *im = ctx->h_pinned[1];
  return HEOM_OK;
}

int64_t heom_launch_count(const heom_ctx* c) { return c ? c->launches : -1; }

heom_status heom_kernel_time(heom_ctx* ctx, double* total_ms, int64_t* launches) {
  if (!ctx) return HEOM_EINVAL;
  if (!ctx->bound) return fail(ctx, HEOM_ESTATE, "no workspace bound");
  CU(cudaStreamSynchronize(ctx->stream));
  double tot = 0.0;
  for (size_t q = 0; q + 1 < ctx->ev_used; q += 2) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ctx->ev[q], ctx->ev[q + 1]));
    tot += ms;
  }
  if (total_ms) *total_ms = tot;
  if (launches) *launches = (int64_t)(ctx->ev_used / 2);
  ctx->ev_used = 0;
  return HEOM_OK;
}

const char* heom_kernel_name(const heom_ctx* c) {
  if (!c) return "none";
  if (c->ket_col >= 0) return "rhs_ket_kernel";
  if (c->use_mma) return (c->herm_opt && c->state_hermitian) ? "rhs_mma_herm_kernel" : "rhs_mma_kernel";
  if (c->use_large) return (c->herm_opt && c->state_hermitian) ? "rhs_large_herm_kernel" : "rhs_large_kernel";
  if (c->use_hpipe) return (c->herm_opt && c->state_hermitian) ? "rhs_hpipe_kernel" : "rhs_hpipe_general_kernel";
  return "rhs_generic_kernel";
}

const char* heom_last_error(const heom_ctx* c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"
