// tslb_launch.cuh -- launch of one time step: kernel selection, grid sizing, attributes.
#pragma once
#include <cuda.h>

#include "tslb_fast.cuh"
#include "tslb_fast_tma.cuh"
#include "tslb_ws.cuh"
#include "tslb_flux.cuh"
#include "tslb_flux_row.cuh"
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
cudaError_t launch_fast(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                        int zc = ZCHUNK) {
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_fast<T, TX, TY, MINB, PREFETCH, ABL, NSTAGE>;
  const size_t smem = sizeof(K2FastSmem<T, M::CELLS, M::NMAIN>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + zc - 1) / zc);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D, Q, zc);
  return cudaGetLastError();
}

// ---- TMA-staged lean kernel (tslb_fast_tma.cuh) ---------------------------------------------
// Tensor maps are encoded through the driver entry point (no link-time dependency on libcuda:
// the library must load on a machine without a GPU) and cached per source buffer in the handle.
struct TmaCache {
  const void* key[2] = {nullptr, nullptr};
  TmaMaps maps[2];
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline EncodeTiledFn tma_encoder() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult st;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &st) == cudaSuccess &&
        st == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}
inline bool tma_encode(TmaMap* out, CUtensorMapDataType dt, int rank, const void* base,
                       const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box) {
  static_assert(sizeof(TmaMap) == sizeof(CUtensorMap), "CUtensorMap is a 128-byte blob");
  EncodeTiledFn enc = tma_encoder();
  if (!enc) return false;
  const cuuint32_t ones[4] = {1, 1, 1, 1};
  return enc(reinterpret_cast<CUtensorMap*>(out), dt, cuuint32_t(rank), const_cast<void*>(base),
             dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename T, int TX, int TY>
bool tma_build_maps(const DevParams<T>& P, const T* S, const T* D, TmaMaps* m) {
  using STG = TmaStage<T, TX, TY>;
  using M = TileMap<TX, TY, 1>;
  constexpr int Wel = VecOf<T>::W;
  const CUtensorMapDataType dt = sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64
                                                : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  const cuuint64_t nx = P.nx, ny = P.ny, nz = P.nz, es = sizeof(T);
  const cuuint64_t vdims[4] = {nx * Wel, ny, nz, cuuint64_t(STG::KV)};
  const cuuint64_t vstr[3] = {nx * 16, nx * ny * 16, cuuint64_t(P.N) * 16};
  const cuuint64_t sdims[3] = {nx, ny, nz};
  const cuuint64_t sstr[2] = {nx * es, nx * ny * es};
  for (int kind = 0; kind < 4; ++kind) {
    const bool colw = kind == 1 || kind == 3, roww = kind == 2 || kind == 3;
    const cuuint32_t vbox[4] = {cuuint32_t((colw ? 1 : M::W) * Wel), cuuint32_t(roww ? 1 : M::HT), 1,
                                cuuint32_t(STG::KV)};
    const cuuint32_t sbox[3] = {cuuint32_t(colw ? STG::PAD : STG::PITCH),
                                cuuint32_t(roww ? 1 : M::HT), 1};
    if (!tma_encode(&m->vec[kind], dt, 4, S, vdims, vstr, vbox)) return false;
    if (!tma_encode(&m->az[kind], dt, 3, S + 12 * P.N, sdims, sstr, sbox)) return false;
    if (!tma_encode(&m->ph[kind], dt, 3, D + F_PHI * P.N, sdims, sstr, sbox)) return false;
  }
  const cuuint32_t fbox[4] = {cuuint32_t(M::W * Wel), cuuint32_t(M::HT), 1, 1};
  if (!tma_encode(&m->vecf, dt, 4, S, vdims, vstr, fbox)) return false;
  return true;
}

template <typename T> inline bool tma_usable(const DevParams<T>& P) {
  return P.nx % 32 == 0 && P.nx >= 64 && P.ny > 8;
}

template <typename T, int TY, int MINB, int NSTAGE, int ABL = 0, int PF = 0, bool SPLIT = false>
cudaError_t launch_tma(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream, int zc,
                       TmaCache* tc) {
  constexpr int TX = 32;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_tma<T, TX, TY, MINB, NSTAGE, ABL, PF, SPLIT>;
  constexpr size_t smem = sizeof(K2FastSmem<T, M::CELLS, M::NMAIN>) +
                          NSTAGE * sizeof(TmaStage<T, TX, TY, SPLIT>) +
                          NSTAGE * sizeof(unsigned long long);
  static_assert(smem <= 227 * 1024, "staging depth does not fit in shared memory");
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  int slot = tc->key[0] == S ? 0 : (tc->key[1] == S ? 1 : -1);
  if (slot < 0) {
    slot = tc->key[0] == nullptr ? 0 : 1;
    if (!tma_build_maps<T, TX, TY>(P, S, D, &tc->maps[slot])) return cudaErrorNotSupported;
    tc->key[slot] = S;
  }
  const dim3 grid(P.nx / TX, (P.ny + TY - 1) / TY, (P.nz + zc - 1) / zc);
  kernel<<<grid, M::NTHREADS + 32, smem, stream>>>(P, tc->maps[slot], D, Q, zc);
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

// Planes per block such that the grid fills whole waves of `slots` resident blocks: among the
// chunk counts that give between 16 and 64 planes per block, the one with the best last wave.
inline int balanced_zchunk(long long tiles_xy, int nz, int slots) {
  int best = 32;
  double best_eff = -1.0;
  for (int nch = (nz + 63) / 64; nch <= (nz + 15) / 16; ++nch) {
    const int zc = (nz + nch - 1) / nch;
    const long long blocks = tiles_xy * ((nz + zc - 1) / zc);
    const double waves = double(blocks) / slots;
    const double eff = waves / double((long long)(waves + 0.999999)) * (double(zc) / (zc + 2));
    if (eff > best_eff + 1e-9) { best_eff = eff; best = zc; }
  }
  return best;
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

// warp-specialised kernel (tslb_ws.cuh): 8 source warps + 8 receiver warps, TMA staging
template <typename T, int NSTAGE>
cudaError_t launch_ws(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream, int zc,
                      TmaCache* tc) {
  constexpr int TX = 32, TY = 8;
  auto kernel = k_stream_collide_ws<T, TX, TY, NSTAGE>;
  constexpr size_t smem = sizeof(WsSmem<T, TX, TY, NSTAGE>);
  static_assert(smem <= 227 * 1024, "staging depth does not fit in shared memory");
  static bool ready = false;
  if (!ready) {
    cudaError_t e = prepare(kernel, smem);
    if (e != cudaSuccess) return e;
    ready = true;
  }
  int slot = tc->key[0] == S ? 0 : (tc->key[1] == S ? 1 : -1);
  if (slot < 0) {
    slot = tc->key[0] == nullptr ? 0 : 1;
    if (!tma_build_maps<T, TX, TY>(P, S, D, &tc->maps[slot])) return cudaErrorNotSupported;
    tc->key[slot] = S;
  }
  const dim3 grid(P.nx / TX, (P.ny + TY - 1) / TY, (P.nz + zc - 1) / zc);
  kernel<<<grid, 512, smem, stream>>>(P, tc->maps[slot], D, Q, zc);
  return cudaGetLastError();
}

// variant = (flags >> 8) & 0xff : tuning selector, 0 = production choice.
template <typename T>
int launch_step_tiled(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                      long long* launches, const Marker& mk, int flags, TmaCache* tc = nullptr) {
  const bool walls = P.bcx || P.bcy || P.bcz;
  const bool generic = walls || (flags & 2);
  const int variant = (flags >> 8) & 0xff;
  cudaError_t e;
  int k1v = (flags >> 16) & 0xff;   // bits 16-23: tuning variant of the Allen-Cahn kernel
  const bool flux_form = !(P.bcx || P.bcy || P.bcz) && !(flags & 2) && (k1v == 0 || k1v >= 5);
  const bool row_ok = P.nx % RowVec<T>::V == 0;          // vector alignment of every row
  if (flux_form && k1v == 0) k1v = row_ok ? 35 : 12;     // production choice, periodic
  if (flux_form && k1v >= 20 && !row_ok) k1v = 12;
  switch (flux_form ? 100 + k1v : k1v) {
    case 112: e = launch_k1_flux<T, 8, 2, 3>(P, S, Q, D, stream); break;   // one node per thread
    case 120: e = launch_k1_row<T, 8, 2, 3>(P, S, Q, D, 32, stream); break;   // row kernel
    case 135: {   // planes per block chosen for whole waves (2 blocks per SM, 148 SMs)
      constexpr int V = RowVec<T>::V;
      const long long txy = (long long)((P.nx + 32 * V - 1) / (32 * V)) * ((P.ny + 7) / 8);
      e = launch_k1_row<T, 8, 2, 3>(P, S, Q, D, balanced_zchunk(txy, P.nz, 2 * 148), stream);
      break;
    }
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
    int v2 = variant;
    if (v2 >= 57 && v2 < 80 && !(tc && tma_usable(P))) v2 = 0;    // TMA staging needs full tile rows
    switch (v2) {
      case 70: e = launch_ws<T, 2>(P, S, D, Q, stream, 64, tc); break;
      case 71: e = launch_ws<T, 2>(P, S, D, Q, stream, 32, tc); break;
      case 72:
        if constexpr (sizeof(T) == 8) e = launch_ws<T, 2>(P, S, D, Q, stream, 128, tc);
        else e = launch_ws<T, 4>(P, S, D, Q, stream, 64, tc);
        break;
      case 60:
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2>(P, S, D, Q, stream, 64, tc);
        break;
      case 66:   // + L2 prefetch one plane beyond the staging depth (0.817 against 0.829 ms in fp64)
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 0, 1>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 0, 1>(P, S, D, Q, stream, 64, tc);
        break;
      case 57:   // loads only, one box per field plane
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 3, 0, true>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 3, 0, true>(P, S, D, Q, stream, 64, tc);
        break;
      case 58:   // loads only, fp32: one block per SM, four slots
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 3>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 1, 4, 3>(P, S, D, Q, stream, 64, tc);
        break;
      case 59:   // production + one box per field plane
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 0, 0, true>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 0, 0, true>(P, S, D, Q, stream, 64, tc);
        break;
      case 73:   // one box per field plane + L2 prefetch of the next plane
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 0, 1, true>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 0, 1, true>(P, S, D, Q, stream, 64, tc);
        break;
      case 74:   // one box per field plane, 32 planes per block
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 0, 0, true>(P, S, D, Q, stream, 32, tc);
        else e = launch_tma<T, 8, 2, 2, 0, 0, true>(P, S, D, Q, stream, 32, tc);
        break;
      case 63:   // timing ablation: loads only
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 3>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 3>(P, S, D, Q, stream, 64, tc);
        break;
      case 64:   // timing ablation: stores only
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 5>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 5>(P, S, D, Q, stream, 64, tc);
        break;
      case 65:   // timing ablation: memory only (wrong results on purpose)
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2, 1>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 2, 2, 1>(P, S, D, Q, stream, 64, tc);
        break;
      case 61:
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 1>(P, S, D, Q, stream, 64, tc);
        else e = launch_tma<T, 8, 1, 4>(P, S, D, Q, stream, 64, tc);
        break;
      case 62:
        if constexpr (sizeof(T) == 8) e = launch_tma<T, 8, 1, 2>(P, S, D, Q, stream, 32, tc);
        else e = launch_tma<T, 8, 2, 2>(P, S, D, Q, stream, 32, tc);
        break;
      case 55:
        if constexpr (sizeof(T) == 8) e = launch_fast<T, 8, 1, false, 0, 2>(P, S, D, Q, stream, 64);
        else e = launch_fast<T, 8, 2, false, 0, 3>(P, S, D, Q, stream, 64);
        break;
      default:   // production choice: fp64 one block/SM, fp32 two blocks/SM
      case 0: {
        // 64 planes per block (2 priming planes per chunk instead of 2 per 32) when the grid
        // still fills the machine about three times over; fp32 then stages two planes ahead
        constexpr int minb = sizeof(T) == 8 ? 1 : 2;
        const long long tiles = (long long)((P.nx + 31) / 32) * ((P.ny + 7) / 8);
        const bool deep = tiles * ((P.nz + 63) / 64) >= 3LL * 148 * minb;
        if constexpr (sizeof(T) == 8) {
          // fp64: TMA tensor staging two planes ahead where the tile rows are full (0.79 ms on
          // 256^3 against 0.85 ms with cp.async); it needs the depth, so only on deep grids
          if (deep && tc && tma_usable(P))
            e = launch_tma<T, 8, 1, 2, 0, 0, true>(P, S, D, Q, stream, 64, tc);   // one box per field plane
          else e = launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, deep ? 64 : 32);
        } else
          e = deep ? launch_fast<T, 8, 2, false, 0, 2>(P, S, D, Q, stream, 64)
                   : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream, 32);
        break;
      }
      case 56: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, 64)
                                  : launch_fast<T, 8, 2, false, 0, 2>(P, S, D, Q, stream, 64);
        break;
      case 54: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, 32)
                                  : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream, 32);
        break;
      case 50: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, 64)
                                  : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream, 64);
        break;
      case 51: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 2>(P, S, D, Q, stream, 64)
                                  : launch_fast<T, 8, 2, false, 0, 2>(P, S, D, Q, stream, 64);
        break;
      case 52: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, 128)
                                  : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream, 128);
        break;
      case 53: e = sizeof(T) == 8 ? launch_fast<T, 8, 1, false, 0, 1>(P, S, D, Q, stream, 43)
                                  : launch_fast<T, 8, 2, false, 0, 1>(P, S, D, Q, stream, 43);
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
