// tslb_flux.cuh -- interface tracking (Eq. 20) in FLUX FORM for all-periodic boxes.
//
//   phi^{n+1} = phi - div Q + D lap(phi),   Q = phi u + kappa_AC phi (1-phi) n   (R13, R16)
//
// The normal n needs grad(phi^n), which the stream-collide kernel of the PREVIOUS step already
// computed for the forces (phi^n is that step's phi^{n+1}).  So that kernel (and tslb_init for
// the first step) stores Q, and this kernel is left with one radius-1 stencil pass: no ring of
// depth 2, no normalisation, no second barrier.  Per node and plane:
//   * z-combinations of the own column (Eq. 18/19 are separable):
//       X = Qx(k-1) + 4 Qx(k) + Qx(k+1),  Y likewise,  Z = Qz(k+1) - Qz(k-1),
//       pz = phi(k-1) + 4 phi(k) + phi(k+1);
//   * with A = c1 Z + c2 pz, Bx = c1 X, By = c1 Y  (c1 = -3/216, c2 = 6 D/216) the node SCATTERS
//     w(dx) w(dy) (A - dx Bx - dy By) to its 8 in-plane neighbours (integer weights (1,4,1));
//   * the receiver adds its 8 arrivals, its own 16 A and (1 - 6 D) phi(k).
// Walls use k_allen_cahn_tiled (ghost rules differ for the two parts of Q, R19).
#pragma once
#include "tslb_fast.cuh"
#include "tslb_tiled.cuh"

namespace tslb {

template <typename T, int CELLS>
struct FluxBuf { T dv[8][CELLS]; };   // 8 direction scalars (separate arrays: conflict-free reads)
// cp.async staging slot of one plane: (Qx,Qy), Qz, phi of the thread's own node
template <typename T, int CELLS>
struct FluxStage { T qx[CELLS]; T qy[CELLS]; T qz[CELLS]; T ph[CELLS]; };

// NSTAGE planes are kept in flight per thread through cp.async (the kernel moves 40 / 20 bytes
// per update: without a deep memory pipeline it is bound by latency, not bandwidth).
template <typename T, int TX, int TY, int MINB, int NSTAGE>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS), MINB)
k_allen_cahn_flux(DevParams<T> P, const T* __restrict__ S, const T* __restrict__ Q,
                  T* __restrict__ phin, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  extern __shared__ __align__(16) unsigned char flux_smem_raw[];
  FluxBuf<T, M::CELLS>* sm = reinterpret_cast<FluxBuf<T, M::CELLS>*>(flux_smem_raw);
  FluxStage<T, M::CELLS>* stg = reinterpret_cast<FluxStage<T, M::CELLS>*>(
      flux_smem_raw + 2 * sizeof(FluxBuf<T, M::CELLS>));

  const int tid = threadIdx.x;
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = blockIdx.x * TX + lx, gy = blockIdx.y * TY + ly;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(P.nz, z0 + zchunk);
  const int c = M::cell(lx, ly);
  const bool in_ring = mapped && gx >= -1 && gx <= P.nx && gy >= -1 && gy <= P.ny;
  const bool is_out = tid < M::NMAIN && gx < P.nx && gy < P.ny;
  const int sx = gx < 0 ? gx + P.nx : (gx >= P.nx ? gx - P.nx : gx);
  const int sy = gy < 0 ? gy + P.ny : (gy >= P.ny ? gy - P.ny : gy);
  const int plane = P.nx * P.ny;
  const int col = in_ring ? sx + P.nx * sy : 0;
  const T* phi = S + F_PHI * P.N;
  const T c1 = T(-3.0 / 216.0), c2 = P.c2;

  auto load = [&](int z, T (&q)[3], T& f) {
    const int jz = z < 0 ? z + P.nz : (z >= P.nz ? z - P.nz : z);
    const int s = col + plane * jz;
    load_q(Q, P.N, s, q);
    f = __ldg(phi + s);
  };

  auto stage_issue = [&](int z, int slot) {
    if (in_ring && z <= z1) {
      const int jz = z < 0 ? z + P.nz : (z >= P.nz ? z - P.nz : z);
      const int s = col + plane * jz;
      cp_async_small(&stg[slot].qx[c], Q + s);
      cp_async_small(&stg[slot].qy[c], Q + P.N + s);
      cp_async_small(&stg[slot].qz[c], Q + 2 * P.N + s);
      cp_async_small(&stg[slot].ph[c], phi + s);
    }
    cp_async_commit();
  };

  // own column at planes k-1 (a), k (b), k+1 (c)
  T qa[3] = {}, qb[3] = {}, qc[3] = {}, fa = 0, fb = 0, fc = 0;
  if (in_ring) {
    load(z0 - 1, qb, fb);
    load(z0, qc, fc);
  }
  if (NSTAGE > 0) {
#pragma unroll
    for (int d = 0; d < NSTAGE; ++d) stage_issue(z0 + 1 + d, d);
  }
  // NSTAGE == 0: planes k+1 and k+2 wait in two register sets that alternate (loop unrolled by 2)
  T r0q[3] = {}, r1q[3] = {}, r0f = 0, r1f = 0;
  if (NSTAGE == 0 && in_ring) {
    load(z0 + 1, r0q, r0f);
    load(z0 + 2, r1q, r1f);
  }

  int slot = 0;
  auto step = [&](const int k, FluxBuf<T, M::CELLS>& w, T (&rq)[3], T& rf) {
    T a0 = 0, g0 = 0;
#pragma unroll
    for (int i = 0; i < 3; ++i) { qa[i] = qb[i]; qb[i] = qc[i]; }
    fa = fb; fb = fc;
    if (NSTAGE > 0) {
      cp_async_wait<(NSTAGE > 0 ? NSTAGE - 1 : 0)>();   // plane k+1 of the own column has landed
      if (in_ring) {
        qc[0] = stg[slot].qx[c]; qc[1] = stg[slot].qy[c]; qc[2] = stg[slot].qz[c];
        fc = stg[slot].ph[c];
      }
      stage_issue(k + 1 + NSTAGE, slot);
      slot = (slot + 1 == NSTAGE) ? 0 : slot + 1;
    } else if (in_ring) {
      qc[0] = rq[0]; qc[1] = rq[1]; qc[2] = rq[2]; fc = rf;
      if (k + 3 <= z1) load(k + 3, rq, rf);
    }
    if (in_ring) {
      const T X = fma(T(4), qb[0], qa[0] + qc[0]);
      const T Y = fma(T(4), qb[1], qa[1] + qc[1]);
      const T Z = qc[2] - qa[2];
      // phi along z in difference form (see tslb_flux_row.cuh): A carries 6 c2 phi and is only
      // ever used in differences, g0 is the node's own small part
      const T d2z = (fa - fb) + (fc - fb);
      const T pz = fma(T(6), fb, d2z);
      const T A = fma(c1, Z, c2 * pz), Bx = c1 * X, By = c1 * Y;
      a0 = A;
      g0 = fma(c1, Z, c2 * d2z);
      const T apx = A + Bx, amx = A - Bx;
      // direction d = (dx,dy): slots 0..7 = (-1,-1) (0,-1) (1,-1) (-1,0) (1,0) (-1,1) (0,1) (1,1)
      w.dv[0][c] = apx + By;            w.dv[1][c] = T(4) * (A + By);
      w.dv[2][c] = amx + By;            w.dv[3][c] = T(4) * apx;
      w.dv[4][c] = T(4) * amx;          w.dv[5][c] = apx - By;
      w.dv[6][c] = T(4) * (A - By);     w.dv[7][c] = amx - By;
    }
    __syncthreads();
    if (is_out) {
      // the value sent in direction d arrives from the source at -d
      // every arrival minus its weight times the own A: a sum of small differences, so that
      // phi' = phi + 36 g0 + (...) is an increment on top of phi (the 36 A + c0 phi of the plain
      // flux form cancel symbolically: c0 + 216 c2 = 1)
      const T a4 = T(4) * a0;
      T s = ((w.dv[0][c + M::W + 1] - a0) + (w.dv[7][c - M::W - 1] - a0))          // (-1,-1) , (1,1)
          + ((w.dv[2][c + M::W - 1] - a0) + (w.dv[5][c - M::W + 1] - a0));         // (1,-1)  , (-1,1)
      s += ((w.dv[1][c + M::W] - a4) + (w.dv[6][c - M::W] - a4))                   // (0,-1)  , (0,1)
         + ((w.dv[3][c + 1] - a4) + (w.dv[4][c - 1] - a4));                        // (-1,0)  , (1,0)
      phin[gx + P.nx * gy + plane * k] = fb + fma(T(36), g0, s);
    }
  };
  for (int k = z0; k < z1; k += 2) {
    step(k, sm[0], r0q, r0f);
    if (k + 1 < z1) step(k + 1, sm[1], r1q, r1f);
  }
  if (NSTAGE > 0) cp_async_wait<0>();
}

}  // namespace tslb
