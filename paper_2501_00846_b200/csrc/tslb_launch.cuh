// tslb_launch.cuh -- launch of one time step: kernel selection, grid sizing, attributes.
#pragma once
#include "tslb_fast.cuh"
#include "tslb_flux.cuh"
#include "tslb_flux_row.cuh"
#include "tslb_stag.cuh"
#include "tslb_tiled.cuh"

namespace tslb {

constexpr int ZCHUNK = 32;   // planes marched by one block (2 extra source planes per chunk)

template <typename K>
inline cudaError_t prepare(K kernel, size_t smem) {
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       int(smem));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout,
                              cudaSharedmemCarveoutMaxShared);
}

template <typename T, int TY, int MINB, bool PREFETCH, int ABL = 0, int NSTAGE = 0, int TX = 32>
cudaError_t launch_fast(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream) {
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_fast<T, TX, TY, MINB, PREFETCH, ABL, NSTAGE>;
  const size_t smem = sizeof(K2FastSmem<T, M::CELLS>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D, Q, ZCHUNK);
  return cudaGetLastError();
}

template <typename T, int TY, int MINB, int NSTAGE = 0>
cudaError_t launch_stag(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream) {
  constexpr int TX = 32;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_stag<T, TX, TY, MINB, NSTAGE>;
  const size_t smem = sizeof(K2FastSmem<T, M::CELLS>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D, Q, ZCHUNK);
  return cudaGetLastError();
}

template <typename T, bool WALLS, int NSTAGE = 1>
cudaError_t launch_generic(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream) {
  constexpr int TX = 32, TY = 8;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_tiled<T, TX, TY, WALLS, 1, NSTAGE>;
  const size_t smem = sizeof(K2Smem<T, TX, TY>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D, ZCHUNK);
  return cudaGetLastError();
}

template <typename T, int TY, int MINB, int NSTAGE>
cudaError_t launch_k1_flux(const DevParams<T>& P, const T* S, const T* Q, T* D, cudaStream_t stream) {
  constexpr int TX = 32;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_allen_cahn_flux<T, TX, TY, MINB, NSTAGE>;
  const size_t smem = 2 * sizeof(FluxBuf<T, M::CELLS>) + NSTAGE * sizeof(FluxStage<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, Q, D + F_PHI * P.N, ZCHUNK);
  return cudaGetLastError();
}

// row kernel: V = 128 bit / sizeof(T) nodes per thread, zc planes per block
template <typename T, int TY, int MINB, int NSTAGE>
cudaError_t launch_k1_row(const DevParams<T>& P, const T* S, const T* Q, T* D, int zc,
                          cudaStream_t stream) {
  static_assert(TY + 2 <= 16, "one extra warp owns the 2 (TY + 2) side columns");
  constexpr int V = RowVec<T>::V;
  auto kernel = k_allen_cahn_row<T, TY, MINB, NSTAGE>;
  const size_t smem = sizeof(RowSmem<T, TY, NSTAGE>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + 32 * V - 1) / (32 * V), (P.ny + TY - 1) / TY, (P.nz + zc - 1) / zc);
  kernel<<<grid, (TY + 3) * 32, smem, stream>>>(P, S, Q, D + F_PHI * P.N, zc);
  return cudaGetLastError();
}

template <typename T, int TY, int MINB, bool WALLS>
cudaError_t launch_k1w(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream) {
  constexpr int TX = 32;
  using M = TileMap<TX, TY, 2>;
  auto kernel = k_allen_cahn_tiled<T, TX, TY, MINB, WALLS>;
  const size_t smem = 2 * sizeof(K1Buf<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D + F_PHI * P.N, ZCHUNK);
  return cudaGetLastError();
}

template <typename T, int TY, int MINB>
cudaError_t launch_k1(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream) {
  return (P.bcx || P.bcy || P.bcz) ? launch_k1w<T, TY, MINB, true>(P, S, D, stream)
                                   : launch_k1w<T, TY, MINB, false>(P, S, D, stream);
}

// variant = (flags >> 8) & 0xff : tuning selector, 0 = production choice.
template <typename T>
int launch_step_tiled(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                      long long* launches, const Marker& mk, int flags) {
  const bool walls = P.bcx || P.bcy || P.bcz;
  const bool generic = walls || (flags & 2);
  const int variant = (flags >> 8) & 0xff;
  cudaError_t e;
  int k1v = (flags >> 16) & 0xff;   // bits 16-23: tuning variant of the Allen-Cahn kernel
  const bool flux_form = !(P.bcx || P.bcy || P.bcz) && !(flags & 2) && (k1v == 0 || k1v >= 5);
  const bool row_ok = P.nx % RowVec<T>::V == 0;          // vector alignment of every row
  if (flux_form && k1v == 0) k1v = row_ok ? 20 : 12;     // production choice, periodic
  if (flux_form && k1v >= 20 && !row_ok) k1v = 12;
  switch (flux_form ? 100 + k1v : k1v) {
    case 112: e = launch_k1_flux<T, 8, 2, 3>(P, S, Q, D, stream); break;   // one node per thread
    case 120: e = launch_k1_row<T, 8, 2, 3>(P, S, Q, D, 32, stream); break;   // row kernel
    case 121: e = launch_k1_row<T, 8, 2, 3>(P, S, Q, D, 16, stream); break;
    case 122: e = launch_k1_row<T, 8, 2, 3>(P, S, Q, D, 64, stream); break;
    case 123: e = launch_k1_row<T, 8, 3, 2>(P, S, Q, D, 32, stream); break;
    case 124: e = launch_k1_row<T, 8, 3, 2>(P, S, Q, D, 16, stream); break;
    case 125: e = launch_k1_row<T, 12, 2, 2>(P, S, Q, D, 32, stream); break;
    case 126: e = launch_k1_row<T, 12, 1, 4>(P, S, Q, D, 32, stream); break;
    case 127: e = launch_k1_row<T, 14, 1, 4>(P, S, Q, D, 32, stream); break;
    case 128: e = launch_k1_row<T, 4, 4, 3>(P, S, Q, D, 32, stream); break;
    case 129: e = launch_k1_row<T, 8, 2, 4>(P, S, Q, D, 24, stream); break;
    case 105: e = launch_k1_flux<T, 8, 3, 2>(P, S, Q, D, stream); break;
    case 106: e = launch_k1_flux<T, 8, 3, 4>(P, S, Q, D, stream); break;
    case 107: e = launch_k1_flux<T, 16, 2, 3>(P, S, Q, D, stream); break;
    case 108: e = launch_k1_flux<T, 8, 2, 0>(P, S, Q, D, stream); break;   // register prefetch x2
    case 110: e = launch_k1_flux<T, 8, 3, 0>(P, S, Q, D, stream); break;
    case 111: e = launch_k1_flux<T, 16, 2, 0>(P, S, Q, D, stream); break;
    case 109: e = launch_k1_flux<T, 8, 4, 4>(P, S, Q, D, stream); break;
    default:
    case 0: case 4: e = launch_k1<T, 8, 2>(P, S, D, stream); break;
    case 1: e = launch_k1<T, 16, 1>(P, S, D, stream); break;
    case 2: e = launch_k1<T, 8, 1>(P, S, D, stream); break;
    case 3: e = launch_k1<T, 4, 3>(P, S, D, stream); break;
  }
  if (e != cudaSuccess) return int(e);
  mk.mark(1);
  if (generic) {
    // cp.async staging pays in fp32 (0.75 vs 1.16 ms on 256^3) but not in fp64 (1.91 vs 1.83 ms)
    constexpr int NS = sizeof(T) == 8 ? 0 : 1;
    if (variant == 1)       // the other choice, kept for comparison
      e = walls ? launch_generic<T, true, 1 - NS>(P, S, D, stream) : launch_generic<T, false, 1 - NS>(P, S, D, stream);
    else
      e = walls ? launch_generic<T, true, NS>(P, S, D, stream) : launch_generic<T, false, NS>(P, S, D, stream);
  } else {
    switch (variant) {
      default:   // production choice: fp64 one block/SM, fp32 two blocks/SM
      case 0:
        e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream)
                           : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream);
        break;
      case 6: e = launch_fast<T, 8, 1, false>(P, S, D, Q, stream); break;
      case 7: e = launch_fast<T, 4, 2, false>(P, S, D, Q, stream); break;
      case 21: e = launch_fast<T, 8, 1, false, 4, 1>(P, S, D, Q, stream); break;    // timing ablations
      case 22: e = launch_fast<T, 8, 1, false, 8, 1>(P, S, D, Q, stream); break;
      case 23: e = launch_fast<T, 8, 1, false, 12, 1>(P, S, D, Q, stream); break;
      case 24: e = launch_fast<T, 8, 1, false, 16, 1>(P, S, D, Q, stream); break;
      case 25: e = launch_fast<T, 8, 1, false, 1 + 2 + 32, 1>(P, S, D, Q, stream); break;
      case 26: e = launch_fast<T, 8, 1, false, 1 + 2 + 16 + 32, 1>(P, S, D, Q, stream); break;
      case 27: e = launch_fast<T, 8, 1, false, 1, 1>(P, S, D, Q, stream); break;
      case 28: e = launch_fast<T, 8, 1, false, 2, 1>(P, S, D, Q, stream); break;
      case 29: e = launch_fast<T, 8, 1, false, 32, 1>(P, S, D, Q, stream); break;
      case 30: e = launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream); break;   // cp.async staging
      case 31: e = launch_fast<T, 8, 1, false, 0, 2>(P, S, D, Q, stream); break;
      case 32: e = launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream); break;
      case 36: e = launch_fast<T, 4, 2, false, 0, 1>(P, S, D, Q, stream); break;
      case 37: e = launch_fast<T, sizeof(T) == 8 ? 8 : 16, 1, false, 0, 1>(P, S, D, Q, stream); break;
      case 38: e = launch_fast<T, 4, 3, false, 0, 1>(P, S, D, Q, stream); break;
      case 39: e = launch_fast<T, sizeof(T) == 8 ? 8 : 16, 1, false, 0, 2>(P, S, D, Q, stream); break;
      case 40: e = launch_fast<T, 4, 1, false, 0, 1, 64>(P, S, D, Q, stream); break;   // 64 x 4 tiles
      case 43: e = launch_fast<T, 8, 1, false, 1 + 2 + 16 + 32, 2>(P, S, D, Q, stream); break;  // memory only, 2 stages
      case 45: e = launch_fast<T, 9, 1, false, 0, 1>(P, S, D, Q, stream); break;
      case 46: e = launch_fast<T, 6, 1, false, 0, 2>(P, S, D, Q, stream); break;
      case 10: e = launch_stag<T, 8, 1>(P, S, D, Q, stream); break;
      case 11: e = launch_stag<T, 8, 2>(P, S, D, Q, stream); break;
      case 12: e = launch_stag<T, 4, 2>(P, S, D, Q, stream); break;
      case 8: e = launch_fast<T, 4, 2, true>(P, S, D, Q, stream); break;
      case 9: e = launch_fast<T, 4, 3, false>(P, S, D, Q, stream); break;
      case 1: e = launch_fast<T, 8, 1, true>(P, S, D, Q, stream); break;
      case 2: e = launch_fast<T, 8, 2, false>(P, S, D, Q, stream); break;
      case 3: e = launch_fast<T, sizeof(T) == 8 ? 8 : 16, 1, false>(P, S, D, Q, stream); break;
      case 4: e = launch_fast<T, sizeof(T) == 8 ? 8 : 16, 1, true>(P, S, D, Q, stream); break;
      case 5: e = launch_fast<T, 8, 2, true>(P, S, D, Q, stream); break;
    }
  }
  mk.mark(2);
  *launches += 2;
  return int(e);
}

}  // namespace tslb
