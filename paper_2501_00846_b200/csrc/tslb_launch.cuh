// tslb_launch.cuh -- launch of one time step: kernel selection, grid sizing, attributes.
//
// Only kernels that compute the step correctly live here.  Which one runs is decided from the
// lattice (walls, size, alignment); flags can only force another CORRECT kernel of the product
// (validation selectors, include/tslb.h), never a tuning or timing variant.
#pragma once
#include <cuda.h>

#include "tslb_fast.cuh"
#include "tslb_fast_tma.cuh"
#include "tslb_flux.cuh"
#include "tslb_flux_row.cuh"
#include "tslb_tiled.cuh"

namespace tslb {

constexpr int ZCHUNK = 32;   // planes marched by one block (2 extra source planes per chunk)
constexpr int kMaxDev = 64;  // device ordinals the per-device set-up caches cover

// Opt-in to more than 48 KB of dynamic shared memory: a per-DEVICE attribute of the kernel, so
// it is cached per device ordinal (a second solver on another GPU of the same process sets it
// again there).
template <typename K>
inline cudaError_t prepare(K kernel, size_t smem, bool (&ready)[kMaxDev]) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < kMaxDev && ready[dev]) return cudaSuccess;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout,
                           cudaSharedmemCarveoutMaxShared);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < kMaxDev) ready[dev] = true;
  return cudaSuccess;
}

// ---- lean periodic stream-collide kernel, cp.async staging NSTAGE planes ahead ---------------
template <typename T, int TY, int MINB, int NSTAGE, bool WXY = false, int TX = 32>
cudaError_t launch_fast(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                        int zc = ZCHUNK) {
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_fast<T, TX, TY, MINB, NSTAGE, WXY>;
  const size_t smem = sizeof(K2FastSmem<T, M::CELLS, M::NMAIN>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.zend - P.zbeg + zc - 1) / zc);
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

// returns cudaErrorNotSupported when the tensor maps cannot be encoded (the caller falls back
// to the cp.async kernel)
template <typename T, int TY, int MINB, int NSTAGE>
cudaError_t launch_tma(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream, int zc,
                       TmaCache* tc) {
  constexpr int TX = 32;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_tma<T, TX, TY, MINB, NSTAGE>;
  constexpr size_t smem = sizeof(K2FastSmem<T, M::CELLS, M::NMAIN>) +
                          NSTAGE * sizeof(TmaStage<T, TX, TY>) +
                          NSTAGE * sizeof(unsigned long long);
  static_assert(smem <= 227 * 1024, "staging depth does not fit in shared memory");
  int slot = tc->key[0] == S ? 0 : (tc->key[1] == S ? 1 : -1);
  if (slot < 0) {
    slot = tc->key[0] == nullptr ? 0 : 1;
    if (!tma_build_maps<T, TX, TY>(P, S, D, &tc->maps[slot])) return cudaErrorNotSupported;
    tc->key[slot] = S;
  }
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  const dim3 grid(P.nx / TX, (P.ny + TY - 1) / TY, (P.zend - P.zbeg + zc - 1) / zc);
  kernel<<<grid, M::NTHREADS + 32, smem, stream>>>(P, tc->maps[slot], D, Q, zc);
  return cudaGetLastError();
}

// ---- wall-capable pair (tslb_tiled.cuh) -----------------------------------------------------
template <typename T, bool WALLS, int NSTAGE>
cudaError_t launch_generic(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream) {
  constexpr int TX = 32, TY = 8;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_stream_collide_tiled<T, TX, TY, WALLS, 1, NSTAGE>;
  const size_t smem = sizeof(K2Smem<T, TX, TY>) + NSTAGE * sizeof(StageBuf<T, M::CELLS>);
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D, ZCHUNK);
  return cudaGetLastError();
}

template <typename T, bool WALLS>
cudaError_t launch_k1w(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream) {
  constexpr int TX = 32, TY = 8, MINB = 2;
  using M = TileMap<TX, TY, 2>;
  auto kernel = k_allen_cahn_tiled<T, TX, TY, MINB, WALLS>;
  const size_t smem = 2 * sizeof(K1Buf<T, M::CELLS>);
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, D + F_PHI * P.N, ZCHUNK);
  return cudaGetLastError();
}

// ---- flux-form interface kernels (periodic) -------------------------------------------------
// one node per thread: the fallback when nx is not a multiple of the 128-bit vector width
template <typename T>
cudaError_t launch_k1_flux(const DevParams<T>& P, const T* S, const T* Q, T* D, cudaStream_t stream) {
  constexpr int TX = 32, TY = 8, MINB = 2, NSTAGE = 3;
  using M = TileMap<TX, TY, 1>;
  auto kernel = k_allen_cahn_flux<T, TX, TY, MINB, NSTAGE>;
  const size_t smem = 2 * sizeof(FluxBuf<T, M::CELLS>) + NSTAGE * sizeof(FluxStage<T, M::CELLS>);
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZCHUNK - 1) / ZCHUNK);
  kernel<<<grid, M::NTHREADS, smem, stream>>>(P, S, Q, D + F_PHI * P.N, ZCHUNK);
  return cudaGetLastError();
}

// Planes per block such that the grid fills whole waves of `slots` resident blocks: among the
// chunk counts that give between 4 and 64 planes per block, the one with the best product of
// last-wave efficiency and priming efficiency (2 extra source planes per chunk).  Small lattices
// (fewer blocks than slots) thereby get short chunks: their step time is the latency of one
// block's march, not throughput.
inline int balanced_zchunk(long long tiles_xy, int nz, int slots) {
  int best = 32;
  double best_eff = -1.0;
  for (int nch = (nz + 63) / 64; nch <= (nz + 3) / 4; ++nch) {
    const int zc = (nz + nch - 1) / nch;
    const long long blocks = tiles_xy * ((nz + zc - 1) / zc);
    const double waves = double(blocks) / slots;
    const double eff = waves / double((long long)(waves + 0.999999)) * (double(zc) / (zc + 2));
    if (eff > best_eff + 1e-9) { best_eff = eff; best = zc; }
  }
  return best;
}

// row kernel: V = 128 bit / sizeof(T) nodes per thread, 8 rows per block, cp.async 3 planes
// ahead, planes per block chosen for whole waves (2 blocks per SM)
template <typename T, bool WXY = false>
cudaError_t launch_k1_row(const DevParams<T>& P, const T* S, const T* Q, T* D, cudaStream_t stream) {
  constexpr int TY = 8, MINB = 2, NSTAGE = 3;
  static_assert(TY + 2 <= 16, "one extra warp owns the 2 (TY + 2) side columns");
  constexpr int V = RowVec<T>::V;
  auto kernel = k_allen_cahn_row<T, TY, MINB, NSTAGE, WXY>;
  const size_t smem = sizeof(RowSmem<T, TY, NSTAGE>);
  static bool ready[kMaxDev] = {};
  cudaError_t e = prepare(kernel, smem, ready);
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const long long txy = (long long)((P.nx + 32 * V - 1) / (32 * V)) * ((P.ny + TY - 1) / TY);
  const int nzr = P.zend - P.zbeg;
  const int zc = balanced_zchunk(txy, nzr, MINB * sms);
  const dim3 grid((P.nx + 32 * V - 1) / (32 * V), (P.ny + TY - 1) / TY, (nzr + zc - 1) / zc);
  kernel<<<grid, (TY + 3) * 32, smem, stream>>>(P, S, Q, D + F_PHI * P.N, zc);
  return cudaGetLastError();
}

// Validation selectors (include/tslb.h TSLB_FLAG_*): every choice is a correct kernel.
enum { SEL_GENERIC = 2, SEL_K2_CPASYNC = 4, SEL_K2_TMA = 8, SEL_K1_FLUX = 16 };

// One time step of the split pair: K1 (interface tracking, Eq. 20) then K2 (stream-collide-
// moments-forces, Eq. 7-17), each over the output planes [P.zbeg, P.zend) (the whole lattice for
// tslb_step; pieces for a slab's split step, lean pair only).  They return a cudaError_t.
template <typename T> inline bool k1_is_tiled(const DevParams<T>& P, int flags) {
  const bool row_ok = P.nx % RowVec<T>::V == 0;
  return (flags & SEL_GENERIC) != 0 || ((P.bcx || P.bcy || P.bcz) && !row_ok);
}

// ---- K1 (interface tracking).  The row kernel serves periodic axes and walls (ghost positions
// rebuild the mirrored flux from Q, phi and u); rows it cannot vectorise fall back to the
// one-node flux kernel on all-periodic boxes and to the wall-capable kernel (normals recomputed
// on a ring of depth 2) on boxes with walls, which hands no flux over: K2 then writes none.
template <typename T>
cudaError_t launch_k1_stage(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                            int flags) {
  const bool side_walls = P.bcx || P.bcy;
  const bool row_ok = P.nx % RowVec<T>::V == 0;
  if (k1_is_tiled(P, flags)) {
    const bool walls = side_walls || P.bcz;
    return walls ? launch_k1w<T, true>(P, S, D, stream) : launch_k1w<T, false>(P, S, D, stream);
  }
  if (row_ok && (side_walls || P.bcz || !(flags & SEL_K1_FLUX)))
    return side_walls ? launch_k1_row<T, true>(P, S, Q, D, stream)
                      : launch_k1_row<T, false>(P, S, Q, D, stream);
  return launch_k1_flux<T>(P, S, Q, D, stream);
}

// ---- K2 (stream-collide-moments-forces): the lean kernel unless the wall-capable one is
// forced; walls on z cost it two ghost planes per column (publish()), walls on x or y the
// bounce accounting of the wall-adjacent receivers (wall_bounce, cp.async staging only)
template <typename T>
cudaError_t launch_k2_stage(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                            int flags, TmaCache* tc) {
  const bool side_walls = P.bcx || P.bcy;
  const bool forced = (flags & SEL_GENERIC) != 0;
  cudaError_t e;
  T* Qk2 = k1_is_tiled(P, flags) ? nullptr : Q;
  if (forced) {
    const bool walls = side_walls || P.bcz;
    // cp.async staging pays in fp32 (0.75 vs 1.16 ms on 256^3) but not in fp64 (1.91 vs 1.83 ms)
    constexpr int NS = sizeof(T) == 8 ? 0 : 1;
    e = walls ? launch_generic<T, true, NS>(P, S, D, stream)
              : launch_generic<T, false, NS>(P, S, D, stream);
  } else {
    // fp64 one block per SM, fp32 two.  64 planes per block (2 priming planes per chunk instead
    // of 2 per 32) when the grid still fills the machine about three times over ("deep").
    constexpr int minb = sizeof(T) == 8 ? 1 : 2;
    const long long tiles = (long long)((P.nx + 31) / 32) * ((P.ny + 7) / 8);
    const int nzr = P.zend - P.zbeg;
    const bool deep = tiles * ((nzr + 63) / 64) >= 3LL * 148 * minb;
    const int zc = deep ? 64 : balanced_zchunk(tiles, nzr, 148 * minb);
    // TMA tensor staging two planes ahead: fp64 production wherever the tile rows are full
    // (256^3: 0.79 against 0.85 ms with cp.async; 192^3, 128^3, 96^3, 64^3: +10, +8, +5, +4 % in
    // GLUPS); in fp32 (two blocks per SM) only when asked for (it loses 4 %)
    bool want_tma = tc && tma_usable(P) && !side_walls && !(flags & SEL_K2_CPASYNC) &&
                    ((flags & SEL_K2_TMA) || sizeof(T) == 8);
    e = cudaErrorNotSupported;
    if (want_tma) e = launch_tma<T, 8, minb, 2>(P, S, D, Qk2, stream, zc, tc);
    if (e == cudaErrorNotSupported) {          // not wanted, or no tensor-map encoder: cp.async
      if (side_walls) {
        if constexpr (sizeof(T) == 8) e = launch_fast<T, 8, 1, 1, true>(P, S, D, Qk2, stream, zc);
        else e = launch_fast<T, 8, 2, 2, true>(P, S, D, Qk2, stream, zc);
      } else if constexpr (sizeof(T) == 8) {
        e = launch_fast<T, 8, 1, 1>(P, S, D, Qk2, stream, zc);
      } else {      // fp32: two planes ahead on every grid (one ahead: -9 % at 128^3 / 192^3)
        e = launch_fast<T, 8, 2, 2>(P, S, D, Qk2, stream, zc);
      }
    }
  }
  return e;
}

template <typename T>
int launch_step_tiled(const DevParams<T>& P, const T* S, T* D, T* Q, cudaStream_t stream,
                      long long* launches, const Marker& mk, int flags, TmaCache* tc = nullptr) {
  cudaError_t e = launch_k1_stage<T>(P, S, D, Q, stream, flags);
  if (e != cudaSuccess) return int(e);
  mk.mark(1);
  e = launch_k2_stage<T>(P, S, D, Q, stream, flags, tc);
  mk.mark(2);
  *launches += 2;
  return int(e);
}

}  // namespace tslb
