// kernels_generic.cu -- generic sm_100a kernel for the HEOM right-hand side with the
// RK4 stage combination fused into its epilogue, plus the small helper kernels.
//
// One thread per matrix element (i,j) of a node; a CTA owns G consecutive nodes
// whose sigma tiles it stages in shared memory (coalesced 16 B loads) together
// with H, so the commutator (Eq. 12) runs out of shared memory.  The couplings to
// sigma_{n +- e_l} (Eq. 15-17 with the masks Eq. 23-25) touch element (i,j) only
// through the modes of bath i (row part) and bath j (column part), so each thread
// walks 2M links instead of W.
#include "kernels.cuh"

namespace heom {
namespace {

constexpr int kThreads = 256;

__host__ __device__ inline int nodes_per_cta(int N) {
  const int NN = N * N;
  return NN >= kThreads ? 1 : (kThreads + NN - 1) / NN;
}

__device__ __forceinline__ double2 ldg2(const double2* p) { return __ldg(p); }

__global__ void __launch_bounds__(kThreads)
rhs_generic_kernel(const RhsParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int N = p.N, NN = N * N, M = p.M, W = p.W, D1 = p.D + 1;
  const int G = nodes_per_cta(N);
  double* sH = reinterpret_cast<double*>(smem_raw);                 // [N][N]
  double2* sS = reinterpret_cast<double2*>(sH + ((NN + 1) & ~1));   // [G][NN]

  const int s0 = blockIdx.x * G;
  const int g_here = min(G, p.nodes - s0);
  for (int e = threadIdx.x; e < NN; e += kThreads) sH[e] = p.H[e];
  for (int e = threadIdx.x; e < g_here * NN; e += kThreads) {
    const int g = e / NN, q = e - g * NN;
    sS[e] = p.x[(size_t)(s0 + g) * p.stride + q];
  }
  __syncthreads();

  for (int e = threadIdx.x; e < g_here * NN; e += kThreads) {
    const int g = e / NN, q = e - g * NN;
    const int i = q / N, j = q - i * N;
    const int s = s0 + g;
    const double2* sig = sS + g * NN;

    // Eq. 12: -(i/hbar)(H sigma - sigma H), H real symmetric (+ i Him, antisymmetric, for general contexts)
    double cr = 0.0, ci = 0.0;
    for (int m = 0; m < N; ++m) {
      const double him = sH[i * N + m], hmj = sH[m * N + j];
      const double2 a = sig[m * N + j], b = sig[i * N + m];
      cr = fma(him, a.x, cr); ci = fma(him, a.y, ci);
      cr = fma(-hmj, b.x, cr); ci = fma(-hmj, b.y, ci);
    }
    if (p.Him) {
      for (int m = 0; m < N; ++m) {
        const double gim = __ldg(p.Him + i * N + m), gmj = __ldg(p.Him + m * N + j);
        const double2 a = sig[m * N + j], b = sig[i * N + m];
        cr = fma(-gim, a.y, cr); ci = fma(gim, a.x, ci);      // i g (a.x + i a.y)
        cr = fma(gmj, b.y, cr); ci = fma(-gmj, b.x, ci);
      }
    }
    double kr = ci * p.inv_hbar, ki = -cr * p.inv_hbar;

    // Eq. 13 + Eq. 14 (mask Eq. 24; general contexts: the table holds the sum over the baths' states, R12)
    const double2 own = sig[q];
    const double dd = p.damp[s] + p.Tterm[q];
    kr = fma(-dd, own.x, kr); ki = fma(-dd, own.y, ki);

    const int32_t* pl = p.plus + (size_t)s * W;
    const int32_t* mi = p.minus + (size_t)s * W;
    const uint8_t* tu = p.tuples + (size_t)s * W;
    // the M modes of one bath (mode columns c*M .. c*M + M - 1) acting on element (i,j) with the mask values
    // vx = V^x (Eq. 23) and vo = V^o (Eq. 25) summed over the bath's states
    auto couple = [&](int c, double vx, double vo) {
      for (int k = 0; k < M; ++k) {
        const int l = c * M + k;
        const int n = tu[l];
        const int up = pl[l], dn = mi[l];
        if (up >= 0 && vx != 0.0) {  // Eq. 15/35: + i a+ V^x sigma^+
          const double a = vx * p.a_plus[l * D1 + n];
          const double2 v = ldg2(p.x + (size_t)up * p.stride + q);
          kr = fma(-a, v.y, kr); ki = fma(a, v.x, ki);
        }
        if (dn >= 0) {  // Eq. 16-17/36: (i a-x V^x + a-o V^o) sigma^-
          const double ax = vx * p.a_minus_x[l * D1 + n], ao = vo * p.a_minus_o[l * D1 + n];
          const double2 v = ldg2(p.x + (size_t)dn * p.stride + q);
          kr = fma(ao, v.x, kr); kr = fma(-ax, v.y, kr);
          ki = fma(ao, v.y, ki); ki = fma(ax, v.x, ki);
        }
      }
    };
    if (p.gen) {
      // baths whose state set contains i: q_i = 1, V^x = 1 - q_j, V^o = 1 + q_j; then those that contain j only
      for (int e = p.sptr[i]; e < p.sptr[i + 1]; ++e) {
        const int b = p.sbl[e];
        const double qj = (double)((p.bmask[b * 4 + (j >> 5)] >> (j & 31)) & 1u);
        couple(b, 1.0 - qj, 1.0 + qj);
      }
      for (int e = p.sptr[j]; e < p.sptr[j + 1]; ++e) {
        const int b = p.sbl[e];
        if (!((p.bmask[b * 4 + (i >> 5)] >> (i & 31)) & 1u)) couple(b, -1.0, 1.0);
      }
    } else if (i != j) {
      couple(i, 1.0, 1.0);    // the bath of state i acts on row i
      couple(j, -1.0, 1.0);   // the bath of state j on column j
    } else {
      couple(i, 0.0, 2.0);    // diagonal: V^x = 0, V^o = 2
    }

    // fused RK4 stage epilogue
    const size_t off = (size_t)s * p.stride + q;
    if (p.rhs_only) {
      p.out_acc[off] = make_double2(kr, ki);
    } else {
      if (p.out_x) {
        const double2 yv = p.y[off];
        p.out_x[off] = make_double2(fma(p.ax, kr, yv.x), fma(p.ax, ki, yv.y));
      }
      const double2 av = p.acc_in[off];
      p.out_acc[off] = make_double2(fma(p.bx, kr, av.x), fma(p.bx, ki, av.y));
    }
  }
}

__global__ void permute_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                               const int32_t* __restrict__ slot_of, int nodes, int NN, int stride,
                               int to_device) {
  const size_t total = (size_t)nodes * NN;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total;
       e += (size_t)gridDim.x * blockDim.x) {
    const int u = (int)(e / NN), q = (int)(e - (size_t)u * NN);
    const size_t dev = (size_t)slot_of[u] * stride + q;
    if (to_device) dst[dev] = src[e];
    else dst[e] = src[dev];
  }
}

__global__ void populations_kernel(const double2* __restrict__ node0, int N, double* __restrict__ out) {
  // one warp; lanes stride over the diagonal, shuffle-reduce the trace (Eq. 26)
  double tr = 0.0, ti = 0.0;
  for (int i = threadIdx.x; i < N; i += 32) {
    const double2 d = node0[(size_t)i * N + i];
    out[i] = d.x;
    tr += d.x; ti += d.y;
  }
  for (int o = 16; o > 0; o >>= 1) {
    tr += __shfl_xor_sync(0xffffffffu, tr, o);
    ti += __shfl_xor_sync(0xffffffffu, ti, o);
  }
  if (threadIdx.x == 0) { out[N] = tr; out[N + 1] = ti; }
}

// halo send buffer: dst[q][e] = src[idx[q]][e], one node (NN complex elements) per row
__global__ void pack_rows_kernel(const double2* __restrict__ src, double2* __restrict__ dst,
                                 const int32_t* __restrict__ idx, long long rows, int NN, int stride) {
  const long long total = rows * NN;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
    const long long q = t / NN;
    const int e = (int)(t - q * NN);
    dst[t] = src[(size_t)idx[q] * stride + e];
  }
}

// Tr(A sigma_0) = sum_ij A[i][j] sigma_0[j][i] (the dipole correlation function of Eq. 56); one warp, fixed order
__global__ void expectation_kernel(const double2* __restrict__ node0, const double2* __restrict__ A, int N,
                                   double* __restrict__ out) {
  double tr = 0.0, ti = 0.0;
  for (int e = threadIdx.x; e < N * N; e += 32) {
    const int i = e / N, j = e - i * N;
    const double2 a = A[e], s = node0[(size_t)j * N + i];
    tr += a.x * s.x - a.y * s.y;
    ti += a.x * s.y + a.y * s.x;
  }
  for (int o = 16; o > 0; o >>= 1) {
    tr += __shfl_xor_sync(0xffffffffu, tr, o);
    ti += __shfl_xor_sync(0xffffffffu, ti, o);
  }
  if (threadIdx.x == 0) { out[0] = tr; out[1] = ti; }
}

}  // namespace

size_t rhs_generic_smem(int N) {
  if (N < 1 || N > 96) return 0;
  const size_t NN = (size_t)N * N;
  return ((NN + 1) & ~(size_t)1) * sizeof(double) + (size_t)nodes_per_cta(N) * NN * sizeof(double2);
}

cudaError_t launch_rhs_generic(const RhsParams& p, cudaStream_t s) {
  const size_t smem = rhs_generic_smem(p.N);
  if (smem == 0) return cudaErrorInvalidValue;
  static size_t configured_on[64] = {};   // per device: the attribute belongs to the device's context
  int dev_ = 0;
  cudaGetDevice(&dev_);
  size_t& configured = configured_on[dev_ & 63];
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(rhs_generic_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  const int G = nodes_per_cta(p.N);
  const int grid = (p.nodes + G - 1) / G;
  rhs_generic_kernel<<<grid, kThreads, smem, s>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_permute(const double2* src, double2* dst, const int32_t* slot_of, int nodes,
                           int NN, int stride, int to_device, cudaStream_t s) {
  const size_t total = (size_t)nodes * NN;
  int grid = (int)((total + 255) / 256);
  if (grid > 148 * 16) grid = 148 * 16;
  if (grid < 1) grid = 1;
  permute_kernel<<<grid, 256, 0, s>>>(src, dst, slot_of, nodes, NN, stride, to_device);
  return cudaGetLastError();
}

cudaError_t launch_populations(const double2* node0, int N, double* out, cudaStream_t s) {
  populations_kernel<<<1, 32, 0, s>>>(node0, N, out);
  return cudaGetLastError();
}

cudaError_t launch_pack_rows(const double2* src, double2* dst, const int32_t* idx, long long rows, int NN, int stride,
                             cudaStream_t s) {
  long long blocks = (rows * NN + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (blocks < 1) blocks = 1;
  pack_rows_kernel<<<(int)blocks, 256, 0, s>>>(src, dst, idx, rows, NN, stride);
  return cudaGetLastError();
}

// slice halo: pair q = (node, state st) moves row st of the node -- and, with_cols, column st
// behind it -- between the state buffer and a packed buffer of `per` = N or 2N elements per pair
__global__ void halo_slices_kernel(double2* __restrict__ state, double2* __restrict__ packed,
                                   const int32_t* __restrict__ node, const int32_t* __restrict__ st, long long pairs,
                                   int N, int per, int to_packed) {
  const long long total = pairs * per;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const long long q = t / per;
    const int e = (int)(t - q * per);
    const size_t base = (size_t)node[q] * N * N;
    const size_t el = e < N ? base + (size_t)st[q] * N + e : base + (size_t)(e - N) * N + st[q];
    if (to_packed) packed[t] = state[el];
    else state[el] = packed[t];
  }
}

cudaError_t launch_halo_slices(double2* state, double2* packed, const int32_t* node, const int32_t* st, long long pairs,
                               int N, int with_cols, int to_packed, cudaStream_t s) {
  const int per = with_cols ? 2 * N : N;
  long long blocks = (pairs * per + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  if (blocks < 1) blocks = 1;
  halo_slices_kernel<<<(int)blocks, 256, 0, s>>>(state, packed, node, st, pairs, N, per, to_packed);
  return cudaGetLastError();
}

// max |element| over the nodes of every hierarchy level: out[L] (bit pattern of a non-negative double, compared as
// an integer) for L = 0..D; per is the number of complex elements per node
__global__ void level_max_kernel(const double2* __restrict__ state, const uint8_t* __restrict__ level, long long nodes,
                                 int per, unsigned long long* __restrict__ out) {
  __shared__ unsigned long long smax[256];
  for (int e = threadIdx.x; e < 256; e += blockDim.x) smax[e] = 0ULL;
  __syncthreads();
  const long long total = nodes * per;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const double2 v = state[t];
    const double a = fmax(fabs(v.x), fabs(v.y));          // max-norm of the element: |re|, |im|
    // NaN counts as +inf (fmax drops a NaN operand: test the parts themselves)
    const double m = (v.x == v.x && v.y == v.y) ? a : __longlong_as_double(0x7ff0000000000000LL);
    atomicMax(&smax[level[t / per]], (unsigned long long)__double_as_longlong(m));
  }
  __syncthreads();
  for (int e = threadIdx.x; e < 256; e += blockDim.x)
    if (smax[e]) atomicMax(&out[e], smax[e]);
}

cudaError_t launch_level_max(const double2* state, const uint8_t* level, long long nodes, int per,
                             unsigned long long* out, cudaStream_t s) {
  long long blocks = (nodes * per + 255) / 256;
  if (blocks > 148 * 8) blocks = 148 * 8;
  if (blocks < 1) blocks = 1;
  level_max_kernel<<<(int)blocks, 256, 0, s>>>(state, level, nodes, per, out);
  return cudaGetLastError();
}

cudaError_t launch_expectation(const double2* node0, const double2* A, int N, double* out, cudaStream_t s) {
  expectation_kernel<<<1, 32, 0, s>>>(node0, A, N, out);
  return cudaGetLastError();
}

}  // namespace heom
