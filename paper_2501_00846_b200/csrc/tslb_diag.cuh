// tslb_diag.cuh -- on-device diagnostics: the box reductions behind what
// the paper plots (centre-of-mass velocity of a rising bubble, Fig. 4) and what
// BASELINE.json checks (conservation of sum(phi), Laplace's law on configs[1]), without reading
// whole fields back to the host.
//
// Two launches, deterministic (no atomics, fixed reduction order, so two runs and two scratch
// buffers give bit-identical results):
//   k_diag_partial : block b reduces the DIAG_NODES consecutive nodes [b, b+1) * DIAG_NODES to
//                    one row of NDIAG doubles in the scratch array (row b);
//   k_diag_final   : one block reduces the rows to out[NDIAG].
// Reads 5 scalars per node (p*, u, phi): HBM-bound, accumulation in fp64 in both precisions.
#pragma once
#include "tslb_device.cuh"

namespace tslb {

constexpr int NDIAG = 16;
constexpr int DIAG_THREADS = 256, DIAG_PER_THREAD = 32;
constexpr int DIAG_NODES = DIAG_THREADS * DIAG_PER_THREAD;   // nodes per block / scratch row

inline long long diag_rows(long long nodes) { return (nodes + DIAG_NODES - 1) / DIAG_NODES; }

__device__ __forceinline__ void load_pu(const double* __restrict__ S, long long N, long long idx,
                                        double& ps, double& ux, double& uy, double& uz) {
  const double2* g = reinterpret_cast<const double2*>(S);
  const double2 a = __ldg(g + idx), b = __ldg(g + N + idx);
  ps = a.x; ux = a.y; uy = b.x; uz = b.y;
}
__device__ __forceinline__ void load_pu(const float* __restrict__ S, long long N, long long idx,
                                        float& ps, float& ux, float& uy, float& uz) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(S) + idx);
  ps = a.x; ux = a.y; uy = a.z; uz = a.w;
}

template <typename T>
__global__ void __launch_bounds__(DIAG_THREADS)
k_diag_partial(DevParams<T> P, long long nodes, const T* __restrict__ S,
               double* __restrict__ partial) {
  __shared__ double red[DIAG_THREADS / 32][NDIAG];
  double s[NDIAG];
#pragma unroll
  for (int k = 0; k < NDIAG; ++k) s[k] = 0.0;
  const long long base = (long long)blockIdx.x * DIAG_NODES;
  const T* phi = S + F_PHI * P.N;
#pragma unroll 4
  for (int i = 0; i < DIAG_PER_THREAD; ++i) {
    const long long idx = base + i * DIAG_THREADS + threadIdx.x;
    if (idx >= nodes) break;
    const unsigned u32 = unsigned(idx);                         // nodes < 2^31 (tslb_create)
    const unsigned row = u32 / unsigned(P.nx);
    const int ix = int(u32 - row * unsigned(P.nx));
    const int iz = int(row / unsigned(P.ny));
    const int iy = int(row - unsigned(iz) * unsigned(P.ny));
    T ps, ux, uy, uz;
    load_pu(S, P.N, idx, ps, ux, uy, uz);
    const T ph = __ldg(phi + idx);
    // p = p* rho cs^2 with the clamped mixture density, as tslb_get returns it (R15)
    const T p = ps * fma(clamp01(ph), P.drho, P.rho_g) * T(1.0 / 3.0);
    const double f = double(ph), x = double(ux), y = double(uy), z = double(uz);
    s[0] += f;
    s[1] += double(ps);
    s[2] = fmax(s[2], sqrt(x * x + y * y + z * z));
    s[3] += f * ix; s[4] += f * iy; s[5] += f * iz;
    s[6] += f * x; s[7] += f * y; s[8] += f * z;
    s[9] += x; s[10] += y; s[11] += z;
    if (ph > T(0.99)) { s[12] += double(p); s[13] += 1.0; }
    if (ph < T(0.01)) { s[14] += double(p); s[15] += 1.0; }
  }
#pragma unroll
  for (int k = 0; k < NDIAG; ++k) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const double v = __shfl_xor_sync(0xffffffffu, s[k], o);
      s[k] = k == 2 ? fmax(s[k], v) : s[k] + v;
    }
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NDIAG; ++k) red[warp][k] = s[k];
  }
  __syncthreads();
  if (threadIdx.x < NDIAG) {
    const int k = threadIdx.x;
    double v = red[0][k];
    for (int w = 1; w < DIAG_THREADS / 32; ++w) v = k == 2 ? fmax(v, red[w][k]) : v + red[w][k];
    partial[(long long)blockIdx.x * NDIAG + k] = v;             // every row is fully overwritten
  }
}

// one block: thread t folds rows t, t + 256, ... in order, then a fixed tree over the threads
__global__ void __launch_bounds__(DIAG_THREADS)
k_diag_final(const double* __restrict__ partial, long long rows, double* __restrict__ out) {
  __shared__ double red[DIAG_THREADS][NDIAG + 1];
  double s[NDIAG];
#pragma unroll
  for (int k = 0; k < NDIAG; ++k) s[k] = 0.0;
  for (long long r = threadIdx.x; r < rows; r += DIAG_THREADS) {
#pragma unroll
    for (int k = 0; k < NDIAG; ++k) {
      const double v = partial[r * NDIAG + k];
      s[k] = k == 2 ? fmax(s[k], v) : s[k] + v;
    }
  }
#pragma unroll
  for (int k = 0; k < NDIAG; ++k) red[threadIdx.x][k] = s[k];
  __syncthreads();
  for (int half = DIAG_THREADS / 2; half > 0; half >>= 1) {
    if (threadIdx.x < half) {
#pragma unroll
      for (int k = 0; k < NDIAG; ++k) {
        const double v = red[threadIdx.x + half][k];
        red[threadIdx.x][k] = k == 2 ? fmax(red[threadIdx.x][k], v) : red[threadIdx.x][k] + v;
      }
    }
    __syncthreads();
  }
  // fmax drops NaNs: a non-finite velocity field must not read as max|u| = 0
  if (threadIdx.x < NDIAG) {
    double v = red[0][threadIdx.x];
    const double su = red[0][9] + red[0][10] + red[0][11];
    if (threadIdx.x == 2 && su != su) v = su;
    out[threadIdx.x] = v;
  }
}

}  // namespace tslb
