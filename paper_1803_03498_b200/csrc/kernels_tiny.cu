// kernels_tiny.cu -- whole-propagation kernel for TINY hierarchies (BASELINE config 1: the dimer, 70 nodes of
// 2 x 2): nodes * N^2 <= 2048 matrix elements.  Such a hierarchy is launch-latency-bound when every RK4 stage is
// its own kernel, so ONE CTA keeps the four state buffers (y, acc, x_a, x_b -- the paper's "4 copies"), the
// link tables and all coefficient tables in shared memory and runs nsteps classical RK4 steps (the four
// stages as in api.cu) inside one launch, one __syncthreads per stage.  One thread per matrix element evaluates
// Eq. 12-17 (masks Eq. 23-25, factors Eq. 35-36) exactly like the generic kernel, from shared memory.
#include "kernels.cuh"

namespace heom {
namespace {

constexpr int kTinyThreads = 512;
constexpr int kTinyMaxElems = 2048;    // nodes * N * N
constexpr int kTinyMaxLinks = 4096;    // nodes * W
constexpr int kTinyFastLinks = 16;     // links per matrix element the fast path keeps in registers: 4 M <= 16

struct TinyParams {
  RhsParams p;          // tables as for the generic kernel; p.x = the state y (DEVICE), read and written
  double dt;
  int nsteps;
};

__global__ void __launch_bounds__(kTinyThreads, 1)
rk4_tiny_kernel(const TinyParams T) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const RhsParams& p = T.p;
  const int N = p.N, NN = N * N, M = p.M, W = p.W, D1 = p.D + 1, nodes = p.nodes;
  const int total = nodes * NN;
  double2* sY = reinterpret_cast<double2*>(smem_raw);
  double2* sAcc = sY + total;
  double2* sXa = sAcc + total;
  double2* sXb = sXa + total;
  double* sH = reinterpret_cast<double*>(sXb + total);        // [N][N]
  double* sT = sH + NN;                                       // [N][N] terminator mask table
  double* sDamp = sT + NN;                                    // [nodes]
  double* sAp = sDamp + nodes;                                // [W][D1] x 3
  double* sAx = sAp + W * D1;
  double* sAo = sAx + W * D1;
  int32_t* sPlus = reinterpret_cast<int32_t*>(sAo + W * D1);  // [nodes][W]
  int32_t* sMinus = sPlus + nodes * W;
  uint8_t* sTup = reinterpret_cast<uint8_t*>(sMinus + nodes * W);

  double2* gy = const_cast<double2*>(p.x);
  for (int e = threadIdx.x; e < total; e += kTinyThreads) sY[e] = gy[e];
  for (int e = threadIdx.x; e < NN; e += kTinyThreads) { sH[e] = p.H[e]; sT[e] = p.Tterm[e]; }
  for (int e = threadIdx.x; e < nodes; e += kTinyThreads) sDamp[e] = p.damp[e];
  for (int e = threadIdx.x; e < W * D1; e += kTinyThreads) { sAp[e] = p.a_plus[e]; sAx[e] = p.a_minus_x[e]; sAo[e] = p.a_minus_o[e]; }
  for (int e = threadIdx.x; e < nodes * W; e += kTinyThreads) { sPlus[e] = p.plus[e]; sMinus[e] = p.minus[e]; sTup[e] = p.tuples[e]; }
  __syncthreads();

  // k(e) = (L x)[e] for matrix element e = node * NN + i * N + j, x in shared memory
  auto rhs = [&](const double2* x, int e) -> double2 {
    const int s = e / NN, q = e - s * NN, i = q / N, j = q - i * N;
    const double2* sig = x + s * NN;
    double cr = 0.0, ci = 0.0;                               // Eq. 12: -(i/hbar)(H sigma - sigma H), H real
    for (int m = 0; m < N; ++m) {
      const double him = sH[i * N + m], hmj = sH[m * N + j];
      const double2 a = sig[m * N + j], b = sig[i * N + m];
      cr = fma(him, a.x, cr); ci = fma(him, a.y, ci);
      cr = fma(-hmj, b.x, cr); ci = fma(-hmj, b.y, ci);
    }
    double kr = ci * p.inv_hbar, ki = -cr * p.inv_hbar;
    const double2 own = sig[q];
    const double dd = sDamp[s] + sT[q];                      // Eq. 13 + Eq. 14 (mask Eq. 24)
    kr = fma(-dd, own.x, kr); ki = fma(-dd, own.y, ki);
    const int32_t* pl = sPlus + s * W;
    const int32_t* mi = sMinus + s * W;
    const uint8_t* tu = sTup + s * W;
    // Eq. 15-17 / 35-36 with the masks of Eq. 23, 25: bath i acts on row i (V^x = +1, V^o = 1), bath j on
    // column j (V^x = -1, V^o = 1); on the diagonal the V^x parts cancel and V^o counts twice
    if (i != j) {
      for (int side = 0; side < 2; ++side) {
        const int b = side == 0 ? i : j;
        const double sx = side == 0 ? 1.0 : -1.0;
        for (int k = 0; k < M; ++k) {
          const int l = b * M + k, n = tu[l];
          const int up = pl[l], dn = mi[l];
          if (up >= 0) {
            const double a = sx * sAp[l * D1 + n];
            const double2 v = x[up * NN + q];
            kr = fma(-a, v.y, kr); ki = fma(a, v.x, ki);
          }
          if (dn >= 0) {
            const double ax = sx * sAx[l * D1 + n], ao = sAo[l * D1 + n];
            const double2 v = x[dn * NN + q];
            kr = fma(ao, v.x, fma(-ax, v.y, kr));
            ki = fma(ao, v.y, fma(ax, v.x, ki));
          }
        }
      }
    } else {
      for (int k = 0; k < M; ++k) {                           // diagonal: V^x = 0, V^o = 2
        const int l = i * M + k, dn = mi[l];
        if (dn >= 0) {
          const double ao = 2.0 * sAo[l * D1 + tu[l]];
          const double2 v = x[dn * NN + q];
          kr = fma(ao, v.x, kr); ki = fma(ao, v.y, ki);
        }
      }
    }
    return make_double2(kr, ki);
  };

  const double dt = T.dt;
  if (total <= kTinyThreads && 4 * M <= kTinyFastLinks) {
    // ---- fast path: one matrix element per thread for the whole propagation.  Everything that does not change from
    //      stage to stage -- the element's indices, its damping rate, and for every link that touches it the
    //      neighbour's element index and the complex factor (Eq. 35-36 with the signs of Eq. 23, 25) -- is worked
    //      out ONCE into registers; a stage is then the commutator, one FMA pair per link and the RK4 update.
    //      (The generic loop below redoes two integer divisions, the table walks and the validity branches per
    //      element and stage: 1.5 us per stage on the dimer, against the few hundred cycles the arithmetic needs.)
    const int e = threadIdx.x;
    const bool on = e < total;
    const int s = on ? e / NN : 0, q = on ? e - s * NN : 0, i = q / N, j = q - i * N;
    const int sig = s * NN;
    const double dd = sDamp[s] + sT[q];
    int lidx[kTinyFastLinks];
    double lre[kTinyFastLinks], lim[kTinyFastLinks];
    int cnt = 0;
    auto add = [&](int idx, double re, double im) {
#pragma unroll
      for (int t = 0; t < kTinyFastLinks; ++t)
        if (t == cnt) { lidx[t] = idx; lre[t] = re; lim[t] = im; }
      ++cnt;
    };
#pragma unroll
    for (int t = 0; t < kTinyFastLinks; ++t) { lidx[t] = 0; lre[t] = 0.0; lim[t] = 0.0; }
    if (on) {
      const int32_t* pl = sPlus + s * W;
      const int32_t* mi = sMinus + s * W;
      const uint8_t* tu = sTup + s * W;
      if (i != j) {
        for (int side = 0; side < 2; ++side) {
          const int b = side == 0 ? i : j;
          const double sx = side == 0 ? 1.0 : -1.0;
          for (int k = 0; k < M; ++k) {
            const int l = b * M + k, n = tu[l];
            if (pl[l] >= 0) add(pl[l] * NN + q, 0.0, sx * sAp[l * D1 + n]);                       // i a+
            if (mi[l] >= 0) add(mi[l] * NN + q, sAo[l * D1 + n], sx * sAx[l * D1 + n]);           // a-o + i a-x
          }
        }
      } else {
        for (int k = 0; k < M; ++k) {                         // diagonal: V^x = 0, V^o = 2
          const int l = i * M + k;
          if (mi[l] >= 0) add(mi[l] * NN + q, 2.0 * sAo[l * D1 + tu[l]], 0.0);
        }
      }
    }
    auto rhs_fast = [&](const double2* x) -> double2 {
      double cr = 0.0, ci = 0.0;                             // Eq. 12
      for (int m = 0; m < N; ++m) {
        const double him = sH[i * N + m], hmj = sH[m * N + j];
        const double2 a = x[sig + m * N + j], b = x[sig + i * N + m];
        cr = fma(him, a.x, cr); ci = fma(him, a.y, ci);
        cr = fma(-hmj, b.x, cr); ci = fma(-hmj, b.y, ci);
      }
      double kr = ci * p.inv_hbar, ki = -cr * p.inv_hbar;
      const double2 own = x[sig + q];
      kr = fma(-dd, own.x, kr); ki = fma(-dd, own.y, ki);   // Eq. 13-14
#pragma unroll
      for (int t = 0; t < kTinyFastLinks; ++t) {
        if (t < cnt) {                                       // Eq. 15-17
          const double2 v = x[lidx[t]];
          kr = fma(lre[t], v.x, fma(-lim[t], v.y, kr));
          ki = fma(lre[t], v.y, fma(lim[t], v.x, ki));
        }
      }
      return make_double2(kr, ki);
    };
    for (int step = 0; step < T.nsteps; ++step) {
      double2 y = make_double2(0.0, 0.0), a = y;
      if (on) {                                              // k1 = f(y)
        const double2 k = rhs_fast(sY);
        y = sY[e];
        sXa[e] = make_double2(fma(dt / 2.0, k.x, y.x), fma(dt / 2.0, k.y, y.y));
        a = make_double2(fma(dt / 6.0, k.x, y.x), fma(dt / 6.0, k.y, y.y));
      }
      __syncthreads();
      if (on) {                                              // k2 = f(y + dt/2 k1)
        const double2 k = rhs_fast(sXa);
        sXb[e] = make_double2(fma(dt / 2.0, k.x, y.x), fma(dt / 2.0, k.y, y.y));
        a = make_double2(fma(dt / 3.0, k.x, a.x), fma(dt / 3.0, k.y, a.y));
      }
      __syncthreads();
      if (on) {                                              // k3 = f(y + dt/2 k2)
        const double2 k = rhs_fast(sXb);
        sXa[e] = make_double2(fma(dt, k.x, y.x), fma(dt, k.y, y.y));
        a = make_double2(fma(dt / 3.0, k.x, a.x), fma(dt / 3.0, k.y, a.y));
      }
      __syncthreads();
      if (on) {                                              // k4 = f(y + dt k3)
        const double2 k = rhs_fast(sXa);
        sY[e] = make_double2(fma(dt / 6.0, k.x, a.x), fma(dt / 6.0, k.y, a.y));
      }
      __syncthreads();
    }
    if (on) gy[e] = sY[e];
    return;
  }
  for (int step = 0; step < T.nsteps; ++step) {
    for (int e = threadIdx.x; e < total; e += kTinyThreads) {          // k1 = f(y)
      const double2 k = rhs(sY, e), y = sY[e];
      sXa[e] = make_double2(fma(dt / 2.0, k.x, y.x), fma(dt / 2.0, k.y, y.y));
      sAcc[e] = make_double2(fma(dt / 6.0, k.x, y.x), fma(dt / 6.0, k.y, y.y));
    }
    __syncthreads();
    for (int e = threadIdx.x; e < total; e += kTinyThreads) {          // k2 = f(y + dt/2 k1)
      const double2 k = rhs(sXa, e), y = sY[e], a = sAcc[e];
      sXb[e] = make_double2(fma(dt / 2.0, k.x, y.x), fma(dt / 2.0, k.y, y.y));
      sAcc[e] = make_double2(fma(dt / 3.0, k.x, a.x), fma(dt / 3.0, k.y, a.y));
    }
    __syncthreads();
    for (int e = threadIdx.x; e < total; e += kTinyThreads) {          // k3 = f(y + dt/2 k2)
      const double2 k = rhs(sXb, e), y = sY[e], a = sAcc[e];
      sXa[e] = make_double2(fma(dt, k.x, y.x), fma(dt, k.y, y.y));
      sAcc[e] = make_double2(fma(dt / 3.0, k.x, a.x), fma(dt / 3.0, k.y, a.y));
    }
    __syncthreads();
    for (int e = threadIdx.x; e < total; e += kTinyThreads) {          // k4 = f(y + dt k3)
      const double2 k = rhs(sXa, e), a = sAcc[e];
      sY[e] = make_double2(fma(dt / 6.0, k.x, a.x), fma(dt / 6.0, k.y, a.y));
    }
    __syncthreads();
  }
  for (int e = threadIdx.x; e < total; e += kTinyThreads) gy[e] = sY[e];
}

size_t tiny_smem(int N, int W, int D, int nodes) {
  const size_t total = (size_t)nodes * N * N;
  size_t b = 4 * total * 16 + 2 * (size_t)N * N * 8 + (size_t)nodes * 8 + 3 * (size_t)W * (D + 1) * 8 +
             2 * (size_t)nodes * W * 4 + (size_t)nodes * W;
  return (b + 15) / 16 * 16;
}

}  // namespace

bool tiny_supported(int N, int W, int D, long long nodes) {
  if (nodes * N * N > kTinyMaxElems || nodes * W > kTinyMaxLinks) return false;
  return tiny_smem(N, W, D, (int)nodes) <= 200 * 1024;
}

cudaError_t launch_rk4_tiny(const RhsParams& p, double dt, int nsteps, cudaStream_t s) {
  TinyParams T;
  T.p = p; T.dt = dt; T.nsteps = nsteps;
  const size_t smem = tiny_smem(p.N, p.W, p.D, p.nodes);
  cudaError_t e = cudaFuncSetAttribute(rk4_tiny_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  rk4_tiny_kernel<<<1, kTinyThreads, smem, s>>>(T);
  return cudaGetLastError();
}

}  // namespace heom
