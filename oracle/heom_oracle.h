/*
 * heom_oracle.h -- C ABI of the CPU ORACLE for the HEOM right-hand side + RK4.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1803_03498_b200/csrc/ and neither includes the other.
 *
 * Citations "P:n" are line numbers of /root/reference/PAPER.md (arXiv
 * 1803.03498, Kramer et al., DM-HEOM).  Readings of the paper where it is
 * silent or garbled are listed in DESIGN.md section 3 ("R1".."R9").
 *
 * Units: energies cm^-1, time fs, hbar = 5308.8 cm^-1 fs, k_B = 0.6950348
 * cm^-1/K; rates in fs^-1.  All matrices row-major, complex numbers as
 * interleaved (re, im) doubles.  Node order: the pinned order of DESIGN.md R1
 * (level-major, descending lexicographic inside a level).
 *
 * Every function returns 0 on success, negative on error (-1 bad argument,
 * -2 out of memory, -4 no state set).
 */
#ifndef HEOM_ORACLE_H
#define HEOM_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_ctx oracle_ctx;

/* P:84-97 (index set), Eq. 19-20 (Matsubara coefficients).
 * H_cm: n_sites*n_sites doubles, real symmetric.  One Drude-Lorentz bath per
 * site (S(b)=1, bs(b)=b): lambda_cm[b], nu_per_fs[b] (Drude rate
 * nu_b, Eq. 6 with Omega=0).  K = number of Matsubara terms beyond the Drude
 * pole, i.e. modes per bath M = K+1 = the paper's "K".  D = truncation depth. */
int  oracle_create(oracle_ctx** out, int n_sites, const double* H_cm,
                   const double* lambda_cm, const double* nu_per_fs,
                   double T_kelvin, int K, int D);
/* Same, for a system whose states do not all carry a bath (the ground state |0> of
 * linear absorption, Eq. 53, 56; "each bath couples to one state"): n_states system states,
 * n_baths <= n_states baths, bath b couples through the projector on state bath_state[b] (0-based, all
 * different).  lambda_cm, nu_per_fs have n_baths entries; W = n_baths*(K+1); delta has n_baths entries.
 * oracle_create(n) == oracle_create_sites(n, n, {0..n-1}). */
int  oracle_create_sites(oracle_ctx** out, int n_states, const double* H_cm, int n_baths,
                         const int* bath_state, const double* lambda_cm, const double* nu_per_fs,
                         double T_kelvin, int K, int D);
/* General system-bath operators ("Multiple states can share one bath, or multiple
 * baths can couple to the same state (for instance a two-exciton state is coupled to two sites ...)"; the sums
 * over s = 1..S(b) in Eq. 14-17; the two-exciton manifold of Eq. 54) and a complex Hermitian H (the
 * RWA field coupling of Eq. 51):
 *   bath b couples through the projectors on the S(b) = bath_ptr[b+1] - bath_ptr[b] >= 1 states
 *   bath_states[bath_ptr[b] .. bath_ptr[b+1]) (0-based, a state at most once per bath; a state may appear in the
 *   lists of several baths; bath_ptr[0] = 0);  H = H_re_cm + i H_im_cm, H_re symmetric, H_im antisymmetric
 *   (H_im_cm may be NULL = real H).
 * oracle_create_sites(...) == oracle_create_general with one state per bath. */
int  oracle_create_general(oracle_ctx** out, int n_states, const double* H_re_cm, const double* H_im_cm,
                           int n_baths, const int* bath_ptr, const int* bath_states, const double* lambda_cm,
                           const double* nu_per_fs, double T_kelvin, int K, int D);
void oracle_destroy(oracle_ctx* ctx);

/* Options (set before any rhs/rk4 call; defaults in brackets):
 *   "scaling"    0 = Eq. 15-16 as printed (no rescaling)
 *               [1] = Eq. 35-36 with |c| = |Re c(b,k)|      (R5)
 *                2 = Eq. 35-36 with |c| = complex modulus of c(b,0)
 *   "terminator" [1] = Eq. 14 on, 0 = off
 *   "terminator_form" the sum over the S(b) states of a bath in Eq. 14 (R12; no effect when S(b) = 1):
 *               [0] = as printed, sum_s V_s^x V_s^x, mask (1 - delta_ij)(m_b(i) + m_b(j)), m_b = membership
 *                1 = the bath's operator squared, (sum_s V_s^x)^2, mask (m_b(i) - m_b(j))^2
 *   "pade"       [0] = Matsubara poles and coefficients (Eq. 19-20), 1 = Pade (Eq. 27-33); rebuilds the
 *                coefficients, K keeps its meaning (number of poles beyond the Drude pole)
 *   "threads"    OpenMP threads for the loop over nodes [0 = runtime default];
 *                results are bit-identical for any thread count (no reductions). */
int  oracle_set_option(oracle_ctx* ctx, const char* name, int value);

/* P:148-176 Eq. 27-31: poles xi_j and weights eta_j (j = 1..K, xi increasing) of the [K-1/K] Pade
 * decomposition of the Bose function, 1/(1-exp(-x)) ~ 1/x + 1/2 + sum_j 2 eta_j x/(x^2 + xi_j^2). */
int  oracle_pade_poles(int K, double* xi, double* eta);

int64_t oracle_num_nodes(const oracle_ctx* ctx);   /* Eq. 9: C(W+D, W)        */
int     oracle_num_modes(const oracle_ctx* ctx);   /* W = n_baths*(K+1)       */
int     oracle_num_baths(const oracle_ctx* ctx);
int     oracle_num_threads(const oracle_ctx* ctx); /* threads the loops use   */

/* tuples uint8 [nodes][W]; plus/minus int32 [nodes][W], -1 = invalid link
 * (P:90).  Any pointer may be NULL. */
int  oracle_get_tables(const oracle_ctx* ctx, uint8_t* tuples,
                       int32_t* plus, int32_t* minus);
/* gamma[W], c_re[W], c_im[W] (c-hat = c/hbar in fs^-2; c_im is non-zero for
 * k=0 only and equals -(lambda_b/hbar) nu_b), delta[n_baths] (Eq. 14 bracket,
 * fs^-1). */
int  oracle_get_coefficients(const oracle_ctx* ctx, double* gamma, double* c_re,
                             double* c_im, double* delta);

/* sigma_0 = given N x N matrix, all ADOs zero. */
int  oracle_set_state(oracle_ctx* ctx, const double* sigma0);
/* full state [nodes][N][N] complex128 in the pinned order */
int  oracle_set_full_state(oracle_ctx* ctx, const double* sigma);
int  oracle_get_full_state(const oracle_ctx* ctx, double* sigma);

/* Eq. 12-17 (with 23-25, 35-36) applied to the current state, all nodes. */
int  oracle_rhs(oracle_ctx* ctx, double* dsigma);
/* Same for a list of nodes only: out is [count][N][N] complex128. */
int  oracle_rhs_nodes(oracle_ctx* ctx, const int64_t* node_ids, int64_t count,
                      double* out);
/* Classical RK4, nsteps steps of dt_fs, in place. */
int  oracle_rk4_steps(oracle_ctx* ctx, double dt_fs, int nsteps);
/* Time-dependent H(t) (Eq. 47-51): replace the Hamiltonian (H_im_cm may be NULL) ... */
int  oracle_set_hamiltonian(oracle_ctx* ctx, const double* H_re_cm, const double* H_im_cm);
/* ... and one classical RK4 step of the non-autonomous system with H(t), H(t + dt/2), H(t + dt) handed in. */
int  oracle_rk4_step_td(oracle_ctx* ctx, double dt_fs, const double* H0_re, const double* H0_im,
                        const double* Hm_re, const double* Hm_im, const double* H1_re, const double* H1_im);
/* Eq. 26: p_i = Re sigma_0[i][i], trace = sum_i sigma_0[i][i]. */
int  oracle_populations(const oracle_ctx* ctx, double* pop, double* trace_re,
                        double* trace_im);

#ifdef __cplusplus
}
#endif
#endif
