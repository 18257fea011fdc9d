/*
 * heom.h -- C ABI of the B200-native HEOM right-hand side + RK4 propagator.
 *
 * The hot path of DM-HEOM (arXiv 1803.03498): the hierarchical Liouvillian
 * (Eq. 12-17 with the site superoperators Eq. 23-25 and the ADO rescaling
 * Eq. 35-36) applied to every auxiliary density matrix sigma_n of a
 * depth-truncated hierarchy (Eq. 9), inside a fixed-step classical RK4
 * propagator whose stage combinations are fused into the
 * right-hand-side kernel.  "P:n" = line n of the paper text PAPER.md; "R*" = a
 * reading of the paper listed in DESIGN.md section 3.
 *
 * Plain C: opaque handle, plain pointers, sizes.  No torch types.  Every
 * pointer argument says HOST or DEVICE.  Errors are integer statuses; nothing
 * throws or aborts.  There is NO CPU fallback: without a CUDA device every
 * compute entry point returns HEOM_ECUDA.
 *
 * Units: energies cm^-1, time fs, hbar = 5308.8 cm^-1 fs (BASELINE.json),
 * k_B = 0.6950348 cm^-1/K (R3).  Matrices row-major; complex numbers are
 * interleaved (re, im) doubles ("complex128").
 *
 * Node order of every HOST-visible table or state: the PINNED order (R1):
 * level-major (L = sum n = 0..D), inside a level descending lexicographic on
 * (n_0..n_{W-1}).  The device-side storage order is internal.
 *
 * Threading: one context per stream; calls on one context are not re-entrant.
 */
#ifndef HEOM_H
#define HEOM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct heom_ctx heom_ctx; /* opaque; owns host tables, coefficients, H copy */

typedef enum {
  HEOM_OK = 0,
  HEOM_EINVAL = -1, /* bad argument (NULL, NaN, non-symmetric H, singular coefficient) */
  HEOM_ENOMEM = -2, /* host allocation failed or workspace too small                   */
  HEOM_ECUDA = -3,  /* CUDA error or no device; heom_last_error() has the text         */
  HEOM_ESTATE = -4  /* call order: no workspace bound / no state set                   */
} heom_status;

/* Build the hierarchy (index set Eq. 9, +/- link graph P:90, mode map Eq. 10-11)
 * and the coefficients (Eq. 14, 19, 20, 35, 36) on the host.  No CUDA call.
 *   H_cm        HOST  n_sites*n_sites doubles, real symmetric (checked exactly), cm^-1
 *   lambda_cm   HOST  [n_sites] reorganisation energies >= 0 of the per-site
 *                     Drude-Lorentz baths (Eq. 6 with Omega = 0; S(b)=1, bs(b)=b)
 *   nu_per_fs   HOST  [n_sites] Drude rates nu_b > 0 in fs^-1 (BASELINE's "gamma")
 *   T_kelvin    > 0
 *   K           >= 0 Matsubara terms beyond the Drude pole: modes per bath M = K+1
 *               (= the paper's "K"); tuple length W = n_sites*M
 *   D           >= 0 truncation depth (sum n <= D)
 *   device      CUDA ordinal used by heom_bind_workspace
 * The caller keeps ownership of all input arrays (they are copied). */
heom_status heom_create(heom_ctx** out, int n_sites, const double* H_cm,
                        const double* lambda_cm, const double* nu_per_fs,
                        double T_kelvin, int K, int D, int device);
/* The same for a system in which not every state carries a bath: the electronic
 * ground state |0> of linear absorption (Eq. 48, 53, 56), which no bath couples to (P:128:
 * each bath b couples through the projector on ONE state, S(b) = 1).
 *   n_states    system states = rows of every sigma_u; H_cm is n_states*n_states
 *   n_baths     1 <= n_baths <= n_states
 *   bath_state  HOST [n_baths] 0-based state bath b couples to, all different (else HEOM_EINVAL)
 *   lambda_cm, nu_per_fs  HOST [n_baths]
 * Tuple length W = n_baths*(K+1); mode l = b*(K+1) + k belongs to bath b (Eq. 10-11).
 * heom_create(n, ...) == heom_create_sites(n, ..., n, {0..n-1}, ...). */
heom_status heom_create_sites(heom_ctx** out, int n_states, const double* H_cm, int n_baths,
                              const int* bath_state, const double* lambda_cm, const double* nu_per_fs,
                              double T_kelvin, int K, int D, int device);
/* General system-bath operators and complex H.  P:84: "Multiple states can share one bath,
 * or multiple baths can couple to the same state (for instance a two-exciton state is coupled to two sites ...)":
 * the sums over s = 1..S(b) of Eq. 14-17; the two-exciton manifold of Eq. 54 (P:279-281,
 * N_states = 1 + N + N(N-1)/2); the RWA field coupling of Eq. 51, which makes H complex Hermitian.
 *   bath_ptr    HOST [n_baths+1], bath_ptr[0] = 0, increasing: bath b couples through the projectors on the
 *               S(b) = bath_ptr[b+1] - bath_ptr[b] >= 1 states bath_states[bath_ptr[b] .. bath_ptr[b+1])
 *   bath_states HOST, 0-based; a state at most once per bath; a state may be listed by several baths
 *   H_re_cm     HOST [n_states][n_states] symmetric; H_im_cm HOST antisymmetric or NULL (real H).  A context
 *               created with H_im_cm != NULL accepts complex Hamiltonians in heom_set_hamiltonian later.
 * n_states <= 96.  With one state per bath, all different, and H_im_cm = NULL this IS heom_create_sites (same
 * kernels); otherwise the general kernels run (kernels_mma.cu for 17 <= n_states <= 96, else the generic kernel),
 * one GPU.  Option "terminator_form" (below) selects how Eq. 14 sums over the states of a bath (R12).
 * Errors: bad lists, non-Hermitian H -> HEOM_EINVAL. */
heom_status heom_create_general(heom_ctx** out, int n_states, const double* H_re_cm, const double* H_im_cm,
                                int n_baths, const int* bath_ptr, const int* bath_states, const double* lambda_cm,
                                const double* nu_per_fs, double T_kelvin, int K, int D, int device);
/* Replace the Hamiltonian: time-dependent H(t) (Eq. 47-51; the caller evaluates the field).  HOST arrays as
 * above; H_im_cm != NULL needs a context created by heom_create_general with H_im_cm != NULL.  Stream-ordered:
 * launches enqueued before the call use the old H.  A time-dependent RK4 step is heom_set_hamiltonian(H(t));
 * heom_rk4_stage(dt, 0); heom_set_hamiltonian(H(t + dt/2)); stages 1, 2; heom_set_hamiltonian(H(t + dt)); stage 3,
 * with option "rk4_form" = 0 (the Horner form holds for a time-independent H only). */
heom_status heom_set_hamiltonian(heom_ctx* ctx, const double* H_re_cm, const double* H_im_cm);
void heom_destroy(heom_ctx* ctx); /* NULL-safe; does not free the workspace */

/* Options, to be set before heom_bind_workspace:
 *   "order"   device storage order of the nodes: 0 = pinned order, 1 = plain
 *             lexicographic (default 1)
 *   "kernel"  0 = generic element-per-thread kernel, 1 = auto (specialised
 *             kernels where available; default), 2 = as 1 without the
 *             whole-propagation kernel for tiny hierarchies (always 4 launches per step)
 *   "pade"    0 (default) = Matsubara poles and coefficients (Eq. 19-20); 1 = Pade poles (P:148-176
 *             Eq. 27-33, R11): the K poles beyond the Drude pole become xi_k/(beta hbar) with weights eta_k.
 *             Rebuilds the coefficients (heom_get_coefficients reports them)
 *   "terminator_form" how Eq. 14 sums over the S(b) states of a bath (R12; no effect when S(b) = 1):
 *             0 (default) = as printed, sum_s V_s^x V_s^x, i.e. the mask (1 - delta_ij)(q_b(i) + q_b(j)) with q_b the
 *             0/1 membership of the bath's state set; 1 = the bath's operator squared, (sum_s V_s^x)^2, i.e. the mask
 *             (q_b(i) - q_b(j))^2
 *   "l2_fetch" cudaLimitMaxL2FetchGranularity to request (32, 64, 128), 0 = leave it
 * and at any time:
 *   "rk4_form" how heom_rk4_steps groups the classical RK4 step (R6): 0 = the four
 *             classical stages with a running sum (16 state sizes of traffic per step); 1 or -1
 *             (default) = the Horner form w <- y + (dt/s) L w for s = 4, 3, 2, 1, y' = the last w --
 *             the same polynomial in dt L for this linear autonomous right-hand side, equal up to
 *             rounding, no running sum, 11 state sizes of traffic -- where the kernel in use
 *             supports it (the pipelined small-N, the tensor-core and the column kernels)
 *   "warps_per_cta" warps per CTA of the pipelined small-N kernel, 0 = as many as fit (default)
 *   "timing"  1 = bracket every RHS launch with CUDA events (heom_kernel_time)
 *   "hermitian" 1 (default) = when heom_set_state / heom_set_full_state find the state
 *             EXACTLY Hermitian (every node equals its conjugate transpose bit for bit), use
 *             the row-gather kernel that keeps it exactly Hermitian; 0 = always the general
 *             kernel.  "timing" and "hermitian" may be changed at any time.
 *   "ket"     1 (default) = when heom_set_state finds sigma_0 with exactly ONE non-zero column c, state c
 *             without a bath (heom_create_sites) and uncoupled in H (H[c][j] = 0 for j != c) -- the
 *             mu_p|0><0| state of linear absorption, P:301 -- every sigma_u keeps that shape, and the state is
 *             held and propagated as one N-vector per node (kernels_ket.cu; Horner form of RK4).
 *             All getters still return full matrices.  0 = always full matrices.  Takes effect at the next
 *             heom_set_state; heom_set_full_state always selects full matrices. */
heom_status heom_set_option(heom_ctx* ctx, const char* name, int value);

int64_t heom_num_nodes(const heom_ctx* ctx); /* Eq. 9: C(W+D, D) */
int heom_num_modes(const heom_ctx* ctx);     /* W = n_baths*(K+1) */
int heom_num_baths(const heom_ctx* ctx);

/* Copies the host tables in the PINNED order.  Any pointer may be NULL.
 *   tuples HOST uint8 [nodes][W]; plus, minus HOST int32 [nodes][W]:
 *   index of n + e_l / n - e_l, or -1 where the link is invalid. */
heom_status heom_get_tables(const heom_ctx* ctx, uint8_t* tuples, int32_t* plus,
                            int32_t* minus);
/* gamma[W] (Eq. 19, fs^-1); c_re[W], c_im[W] = c(b,k)/hbar (Eq. 20 and the V^o
 * part of Eq. 17, fs^-2); delta[n_baths] = Eq. 14 bracket (fs^-1).  All HOST. */
heom_status heom_get_coefficients(const heom_ctx* ctx, double* gamma, double* c_re,
                                  double* c_im, double* delta);

/* The state lives in caller-owned DEVICE memory (e.g. a torch tensor): the
 * library never allocates state memory.  heom_workspace_bytes = 4 padded state
 * buffers ("4 copies") + device tables.  dev_ptr must be 256-byte
 * aligned and stay valid until heom_destroy or the next bind.  cuda_stream is
 * a cudaStream_t (NULL = default stream); all work is enqueued on it.
 * Uploads the tables (synchronous). */
size_t heom_workspace_bytes(const heom_ctx* ctx);
heom_status heom_bind_workspace(heom_ctx* ctx, void* dev_ptr, size_t bytes,
                                void* cuda_stream);

/* sigma_0 = the given matrix, every ADO zero.
 *   sigma0 HOST n_sites*n_sites complex128, row-major. */
heom_status heom_set_state(heom_ctx* ctx, const double* sigma0);
/* Full-state I/O, PINNED node order, unpadded [nodes][N][N] complex128, HOST.
 * These are also the checkpoint/resume path. */
heom_status heom_set_full_state(heom_ctx* ctx, const double* sigma);
heom_status heom_get_full_state(heom_ctx* ctx, double* sigma);

/* dsigma = L(current state): one evaluation of Eq. 12-17 on every node; the
 * state is not changed.  dsigma HOST, same layout as heom_get_full_state. */
heom_status heom_rhs(heom_ctx* ctx, double* dsigma);
/* Advance the state by nsteps classical RK4 steps of dt_fs (R6; option "rk4_form" selects how
 * the step is grouped).  Enqueues 4*nsteps fused kernels on the bound stream and returns;
 * heom_sync or any HOST getter synchronises. */
heom_status heom_rk4_steps(heom_ctx* ctx, double dt_fs, int nsteps);
heom_status heom_sync(heom_ctx* ctx);
/* Eq. 26: pop[i] = Re sigma_0[i][i] (HOST [n_sites]); trace = sum_i sigma_0[i][i].
 * Computed by a device reduction kernel; output pointers may be NULL. */
heom_status heom_populations(heom_ctx* ctx, double* pop, double* trace_re,
                             double* trace_im);

/* Growth monitor (Eq. 38: dt << 1/gamma_k; config 3 at dt = 1 fs lies outside RK4's
 * stability region): max_abs[L] = max over the nodes of hierarchy level L (sum n = L) and their elements of
 * max(|Re|, |Im|), L = 0..D (HOST [D+1]); +inf if a NaN or Inf is present.  Device reduction; synchronises. */
heom_status heom_level_max(heom_ctx* ctx, double* max_abs);

/* Tr(A sigma_0) = sum_ij A[i][j] sigma_0[j][i]: the integrand of the dipole correlation function of
 * Eq. 56 with A = mu_p.  A HOST [N][N] complex128 row-major; re, im HOST (may be NULL).
 * Computed by a device reduction kernel; synchronises. */
heom_status heom_expectation(heom_ctx* ctx, const double* A, double* re, double* im);

/* ---- One hierarchy sharded over several GPUs (the paper's partitions + halo regions) ----
 * One process per GPU; rank r of `world` owns a contiguous range of the lexicographic node order and keeps ghost
 * copies of the neighbours of its nodes that live on other ranks.  A partition context behaves like a context
 * whose hierarchy is the n_owned + n_ghost LOCAL nodes (heom_num_nodes, heom_get_tables with local indices,
 * heom_set_full_state / heom_get_full_state / heom_rhs over the local nodes; ghost rows of a result are not
 * meaningful).  Local order: owned nodes, then ghosts grouped by owning rank in the order the owner sends them,
 * so the ghost rows of a state buffer ARE the receive buffer of the exchange.  The caller moves the halos
 * (torch.distributed / NCCL all_to_all_single in paper_1803_03498_b200/sharded.py): per RK4 step
 *   for stage in 0..3: heom_rk4_stage; heom_stage_output -> buf; heom_pack_halo(buf -> send);
 *                      all-to-all: send rows -> the peers' ghost rows of buf
 * heom_set_state sets the rank's copy of sigma_0 (owned or ghost) if it holds one; heom_populations and
 * heom_expectation return HEOM_ESTATE on a rank that holds none; heom_rk4_steps returns HEOM_ESTATE on a
 * partition with world > 1 (it cannot exchange).  Kernels launch over the owned rows only.  Errors: rank/world out
 * of range or world > number of nodes -> HEOM_EINVAL. */
heom_status heom_create_partition(heom_ctx** out, int n_states, const double* H_cm, int n_baths,
                                  const int* bath_state, const double* lambda_cm, const double* nu_per_fs,
                                  double T_kelvin, int K, int D, int device, int rank, int world);
int64_t heom_partition_owned(const heom_ctx* ctx); /* n_owned (the first n_owned local nodes) */
/* global_ids HOST int64 [local nodes]: pinned-order id (R1) of every local node; send_counts, recv_counts HOST
 * int64 [world]: nodes sent to / ghosts received from every peer; send_idx HOST int32 [sum send_counts]: local
 * indices of the nodes to send, grouped by peer.  Any pointer may be NULL. */
heom_status heom_partition_plan(const heom_ctx* ctx, int64_t* global_ids, int64_t* send_counts,
                                int64_t* recv_counts, int32_t* send_idx);
/* One fused RHS + RK4-stage launch, stage = 0..3 of the current step (matrix kernels only). */
heom_status heom_rk4_stage(heom_ctx* ctx, double dt_fs, int stage);
/* DEVICE pointer (complex128 [local nodes][N][N], local order) of the buffer the NEXT stage reads, i.e. the one
 * whose ghost rows must be refreshed after `stage` (after stage 3: the new state y). */
heom_status heom_stage_output(heom_ctx* ctx, int stage, void** dev_ptr);
/* dst_dev[q] = node send_idx[q] of src_dev (device kernel on the bound stream); dst_dev DEVICE, sum(send_counts)
 * nodes of N*N complex128. */
heom_status heom_pack_halo(heom_ctx* ctx, const void* src_dev, void* dst_dev);

/* Slice halo: a neighbour gather reads of a ghost only row s -- and, unless the state is exactly Hermitian and a
 * row-gather kernel runs, column s -- where s is the state of the bath through which the ghost is reached (the masks
 * of Eq. 23, 25): 16 N (or 32 N) bytes per (ghost, state) pair instead of 16 N^2 per ghost.  The (node, state) pairs
 * are unique and sorted by (peer, global node order, state) on both sides, so sender and receiver agree without
 * communication.  Per stage: heom_rk4_stage; heom_stage_output -> buf; heom_pack_halo_slices(buf -> send);
 * all-to-all of the packed pairs (heom_halo_slice_elements() complex128 each) ; heom_unpack_halo_slices(recv -> buf).
 *   send_counts, recv_counts HOST int64 [world]: pairs per peer; send_node / send_state HOST int32 [sum send_counts]:
 *   local OWNED node index and state; recv_node / recv_state HOST int32 [sum recv_counts]: local GHOST node index
 *   and state.  Any pointer may be NULL. */
heom_status heom_partition_plan_slices(const heom_ctx* ctx, int64_t* send_counts, int64_t* recv_counts,
                                       int32_t* send_node, int32_t* send_state, int32_t* recv_node, int32_t* recv_state);
int heom_halo_slice_elements(const heom_ctx* ctx);   /* N (row) or 2N (row, then column) complex128 per pair, now */
/* dst_dev[q] = the slices of pair q of src_dev (a state buffer); DEVICE pointers; kernel on the bound stream. */
heom_status heom_pack_halo_slices(heom_ctx* ctx, const void* src_dev, void* dst_dev);
/* scatter the received pairs (DEVICE, in recv order) into the ghost nodes of state_dev. */
heom_status heom_unpack_halo_slices(heom_ctx* ctx, const void* src_dev, void* state_dev);

/* Introspection for the harness. */
int64_t heom_launch_count(const heom_ctx* ctx); /* kernels launched so far */
/* With option "timing"=1: sum of CUDA-event durations of the RHS/stage kernels
 * launched since the last call, and their number.  Synchronises. */
heom_status heom_kernel_time(heom_ctx* ctx, double* total_ms, int64_t* launches);
/* Name of the RHS kernel variant the bound configuration uses (static string). */
const char* heom_kernel_name(const heom_ctx* ctx);
/* Measured peak of `device` for the harness' roofline (no context needed; synchronises; allocates
 * and frees its own scratch): kind 0 = FP64 FMA (register-resident DFMA chains), 1 = FP64 tensor core
 * (mma.sync.m8n8k4.f64, SASS DMMA.8x8x4) -- *value in TFLOP/s; 2 = HBM copy bandwidth (read + write bytes of a
 * 1 GiB device-to-device copy kernel) -- *value in GB/s.  Best of 5 timed repetitions after one warm-up. */
heom_status heom_probe_peak(int device, int kind, double* value);
/* The growth monitor of heom_level_max for callers that may not allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): no context, no workspace, nothing allocated or
 * freed.  Its scratch (the per-level running maxima and a finished-blocks counter, 768 bytes) is a file-scope
 * __device__ array that every GPU loading the library holds until the process exits, hence the limit
 * depth <= HEOM_STATIC_MAX_DEPTH; a larger depth is rejected with HEOM_EINVAL (use heom_level_max).
 *   device          CUDA ordinal the pointers belong to (made current for the call, then restored)
 *   state_dev       DEVICE complex128 [nodes][elems_per_node], any node order (e.g. heom_stage_output's buffer)
 *   level_dev       DEVICE uint8 [nodes]: hierarchy level sum(n) of every node, same order; levels > depth are ignored
 *   max_abs_dev     DEVICE double [depth+1]: max over the nodes of level L and their elements of max(|Re|, |Im|);
 *                   +inf if a NaN or Inf is present; 0 for a level without nodes
 *   cuda_stream     cudaStream_t; the call enqueues a clear of the scratch and one kernel on it and returns
 *                   (no synchronisation: max_abs_dev is valid once the stream reaches that point)
 * All calls on a device share the scratch: each clears it first, so nothing of an earlier call survives, but calls
 * that overlap on the GPU (different streams without an ordering between them) race and give wrong maxima.
 * The first call on a device looks the scratch address up (cudaGetSymbolAddress); make it outside a graph capture. */
#define HEOM_STATIC_MAX_DEPTH 63
heom_status heom_level_max_static(int device, const void* state_dev, const uint8_t* level_dev, int64_t nodes,
                                  int elems_per_node, int depth, double* max_abs_dev, void* cuda_stream);
/* Text of the last error heom_level_max_static returned on the calling thread (static storage, "" if none). */
const char* heom_static_last_error(void);

/* Human-readable text of the last error on this context (ctx-owned). */
const char* heom_last_error(const heom_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
