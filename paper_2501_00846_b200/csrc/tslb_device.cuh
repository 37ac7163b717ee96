// tslb_device.cuh -- per-node device arithmetic of the TSLB step (sm_100a).
//
// Product code.  Shares nothing with oracle/.  Citations: "P:<line>" = PAPER.md, "Rk" =
// DESIGN.md readings.  Everything is templated on the scalar type T (float / double).
#pragma once
#include <cuda_runtime.h>

#include <vector>

namespace tslb {

// Optional per-kernel timing (tslb_step_timed): an event after every launch, tagged by kind.
struct Marker {
  std::vector<cudaEvent_t>* events = nullptr;
  std::vector<int>* kinds = nullptr;
  cudaStream_t stream = nullptr;
  void mark(int kind) const {
    if (!events) return;
    cudaEvent_t e;
    cudaEventCreate(&e);
    cudaEventRecord(e, stream);
    events->push_back(e);
    kinds->push_back(kind);
  }
};

// Stored state per node: 14 scalars, indexed in this order everywhere in the code:
//   0 p*   1-3 u   4-9 Ahat = (1 - omega(phi)) a2_neq (xx,yy,zz,xy,xz,yz)   10-12 a = F/rho   13 phi
enum { F_P = 0, F_UX = 1, F_UY = 2, F_UZ = 3, F_AXX = 4, F_AYY = 5, F_AZZ = 6, F_AXY = 7,
       F_AXZ = 8, F_AYZ = 9, F_AX = 10, F_AY = 11, F_AZ = 12, F_PHI = 13, NFIELD = 14 };

// HBM layout: one buffer = 14 N scalars (N = padded node count).
// Fields 0..11 are interleaved per node in 128-bit vectors so that a thread moves them with
// 128-bit loads/stores and a warp touches 512 contiguous bytes per instruction:
//   fp64: 6 planes of double2  (p*,ux) (uy,uz) (Axx,Ayy) (Azz,Axy) (Axz,Ayz) (ax,ay)
//   fp32: 3 planes of float4   (p*,ux,uy,uz) (Axx,Ayy,Azz,Axy) (Axz,Ayz,ax,ay)
// followed by the scalar plane az (offset 12 N) and the scalar plane phi (offset 13 N), which
// the Allen-Cahn kernel writes on its own.
template <typename T> struct VecOf;
template <> struct VecOf<double> { using type = double2; static constexpr int W = 2; };
template <> struct VecOf<float> { using type = float4; static constexpr int W = 4; };

__device__ __forceinline__ void unpack(const double2& v, double* m) { m[0] = v.x; m[1] = v.y; }
__device__ __forceinline__ void unpack(const float4& v, float* m) {
  m[0] = v.x; m[1] = v.y; m[2] = v.z; m[3] = v.w;
}
__device__ __forceinline__ double2 pack(const double* m) { return make_double2(m[0], m[1]); }
__device__ __forceinline__ float4 pack(const float* m) { return make_float4(m[0], m[1], m[2], m[3]); }

// the 13 moment scalars (fields 0..12) of node idx
template <typename T>
__device__ __forceinline__ void load13(const T* __restrict__ S, long long N, long long idx,
                                       T (&m)[13]) {
  using V = typename VecOf<T>::type;
  constexpr int W = VecOf<T>::W;
  const V* g = reinterpret_cast<const V*>(S);
#pragma unroll
  for (int k = 0; k < 12 / W; ++k) unpack(__ldg(g + k * N + idx), &m[k * W]);
  m[12] = __ldg(S + 12 * N + idx);
}
template <typename T>
__device__ __forceinline__ void store13(T* __restrict__ D, long long N, long long idx,
                                        const T (&m)[13]) {
  using V = typename VecOf<T>::type;
  constexpr int W = VecOf<T>::W;
  V* g = reinterpret_cast<V*>(D);
#pragma unroll
  for (int k = 0; k < 12 / W; ++k) g[k * N + idx] = pack(&m[k * W]);
  D[12 * N + idx] = m[12];
}
// velocity only (Allen-Cahn stage): 2 x 128 bit in fp64, 1 x 128 bit in fp32
__device__ __forceinline__ void load_u(const double* __restrict__ S, long long N, long long idx,
                                       double& ux, double& uy, double& uz) {
  const double2* g = reinterpret_cast<const double2*>(S);
  const double2 a = __ldg(g + idx), b = __ldg(g + N + idx);
  ux = a.y; uy = b.x; uz = b.y;
}
__device__ __forceinline__ void load_u(const float* __restrict__ S, long long N, long long idx,
                                       float& ux, float& uy, float& uz) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(S) + idx);
  ux = a.y; uy = a.z; uz = a.w;
}
// element offset of one scalar field of node idx (slow path: init / get / naive kernels)
template <typename T>
__device__ __forceinline__ long long field_off(long long N, long long idx, int f) {
  constexpr int W = VecOf<T>::W;
  return f < 12 ? (long long)(f / W) * W * N + idx * W + (f % W) : (long long)f * N + idx;
}

template <typename T>
struct DevParams {
  int nx, ny, nz;
  int bcx, bcy, bcz;          // 0 periodic, 1 wall
  int zbeg, zend;             // output planes [zbeg, zend) of a launch of the lean pair: the whole
                              // lattice, or one piece of a slab's split step (tslb_slab_step_*)
  long long N;
  T rho_l, rho_g, drho;       // drho = rho_l - rho_g
  T mu_g, dmu;                // mu = mu_g + phi_c dmu                      (R14)
  T beta4, kappa_mu;          // 4 beta = 48 sigma/delta ; 3 sigma delta/2
  T mob, kappa_ac;            // D ; 4 D/delta
  T c2;                       // D 6/216 rounded to T: weight of the (1,4,1)^3 Laplacian sums in the
                              // flux-form interface kernels (the centre weight 1 - 216 c2 is never
                              // formed: the kernels add an increment of differences to phi)
  T gx, gy, gz;               // body acceleration                          (R20)
  T rho_b;                    // force density (rho - rho_b) g: rho_l or rho_g (R20b)
};

template <typename T> __device__ __forceinline__ T rsqrt_t(T x);
template <> __device__ __forceinline__ float rsqrt_t<float>(float x) { return rsqrtf(x); }
template <> __device__ __forceinline__ double rsqrt_t<double>(double x) { return rsqrt(x); }

template <typename T> __device__ __forceinline__ T clamp01(T x) {
  return x < T(0) ? T(0) : (x > T(1) ? T(1) : x);
}

// Mixture rules (R14, R15).  One division: r = 1/(rho (3 mu + rho/2)) gives
//   1/rho = r (3 mu + rho/2),  omega = 1/(3 nu + 1/2) = rho^2 r,  nu omega / cs^2 = 3 mu rho r.
template <typename T> struct Mix { T rho, inv_rho, omega, nuom3; };
template <typename T>
__device__ __forceinline__ Mix<T> mixture(const DevParams<T>& P, T phi) {
  T pc = clamp01(phi);
  T rho = fma(pc, P.drho, P.rho_g);
  T mu = fma(pc, P.dmu, P.mu_g);
  T d = fma(T(3), mu, T(0.5) * rho);
  T r = T(1) / (rho * d);
  Mix<T> m;
  m.rho = rho;
  m.inv_rho = r * d;
  m.omega = rho * rho * r;
  m.nuom3 = T(3) * mu * rho * r;
  return m;
}

// One-dimensional lattice weights (R1) and second Hermite polynomial on c in {-1,0,1}.
template <typename T> __device__ __forceinline__ constexpr T w1(int c) {
  return c == 0 ? T(2.0 / 3.0) : T(1.0 / 6.0);
}
template <typename T> __device__ __forceinline__ constexpr T h2(int c) {
  return c == 0 ? T(-1.0 / 3.0) : T(2.0 / 3.0);
}

// The 17 Hermite coefficients of the post-collision population of one node:
//   f_post(c) = w(c) [ C0 + c.C1/cs^2 + H2(c):C2/(2cs^4) + H3(c):C3/(6cs^6) ]
// with f_post = f_eq + (1-omega) f_neq + S/2 (Eq. 7, 9, 10, 14; R2, R3, R5):
//   C0 = p*, C1 = u + a/2, C2 = uu + Ahat + (ua + au)/2, C3 = uuu + sym(u Ahat)  (7 live comps).
template <typename T>
struct Coef {
  T c0, c1x, c1y, c1z, xx, yy, zz, xy, xz, yz, xxy, xyy, xxz, xzz, yyz, yzz, xyz;
};

template <typename T>
__device__ __forceinline__ Coef<T> coefficients(T p, T ux, T uy, T uz, T axx, T ayy, T azz, T axy,
                                                T axz, T ayz, T ax, T ay, T az) {
  Coef<T> c;
  const T h = T(0.5);
  c.c0 = p;
  c.c1x = fma(h, ax, ux);
  c.c1y = fma(h, ay, uy);
  c.c1z = fma(h, az, uz);
  // second order: u_a u_b + Ahat_ab + (u_a a_b + a_a u_b)/2 = u_a (u_b + a_b/2) + a_a u_b/2 + Ahat
  c.xx = fma(ux, ux + ax, axx);
  c.yy = fma(uy, uy + ay, ayy);
  c.zz = fma(uz, uz + az, azz);
  c.xy = fma(ux, c.c1y, fma(h * ax, uy, axy));
  c.xz = fma(ux, c.c1z, fma(h * ax, uz, axz));
  c.yz = fma(uy, c.c1z, fma(h * ay, uz, ayz));
  // third order (recursive relation P:106): u_a u_b u_g + u_a Ahat_bg + u_b Ahat_ag + u_g Ahat_ab
  T uxx = fma(ux, ux, axx), uyy = fma(uy, uy, ayy), uzz = fma(uz, uz, azz);
  c.xxy = fma(uy, uxx, T(2) * ux * axy);
  c.xyy = fma(ux, uyy, T(2) * uy * axy);
  c.xxz = fma(uz, uxx, T(2) * ux * axz);
  c.xzz = fma(ux, uzz, T(2) * uz * axz);
  c.yyz = fma(uz, uyy, T(2) * uy * ayz);
  c.yzz = fma(uy, uzz, T(2) * uz * ayz);
  c.xyz = fma(ux, fma(uy, uz, ayz), fma(uy, axz, uz * axy));
  return c;
}

// Post-collision population in the compile-time direction (CX,CY,CZ).
template <typename T, int CX, int CY, int CZ>
__device__ __forceinline__ T fpost_dir(const Coef<T>& c) {
  const T hx = h2<T>(CX), hy = h2<T>(CY), hz = h2<T>(CZ);
  T s = c.c0;
  s += T(3) * (T(CX) * c.c1x + T(CY) * c.c1y + T(CZ) * c.c1z);
  s += T(4.5) * (hx * c.xx + hy * c.yy + hz * c.zz)
     + T(9) * (T(CX * CY) * c.xy + T(CX * CZ) * c.xz + T(CY * CZ) * c.yz);
  s += T(13.5) * (hx * (T(CY) * c.xxy + T(CZ) * c.xxz) + hy * (T(CX) * c.xyy + T(CZ) * c.yyz)
                  + hz * (T(CX) * c.xzz + T(CY) * c.yzz))
     + T(27) * T(CX * CY * CZ) * c.xyz;
  return w1<T>(CX) * w1<T>(CY) * w1<T>(CZ) * s;
}

// Raw moments of the 27 streamed populations (Eq. 11-13): p*, m, Pi.
template <typename T> struct Mom { T p, mx, my, mz, xx, yy, zz, xy, xz, yz; };

template <typename T, int CX, int CY, int CZ>
__device__ __forceinline__ void accumulate(Mom<T>& m, T f) {
  m.p += f;
  if (CX) m.mx += T(CX) * f;
  if (CY) m.my += T(CY) * f;
  if (CZ) m.mz += T(CZ) * f;
  if (CX) m.xx += f;
  if (CY) m.yy += f;
  if (CZ) m.zz += f;
  if (CX * CY) m.xy += T(CX * CY) * f;
  if (CX * CZ) m.xz += T(CX * CZ) * f;
  if (CY * CZ) m.yz += T(CY * CZ) * f;
}

// Closing stage of a node (DESIGN.md a6-a9): forces from phi^{n+1} (R8), velocity, Ahat.
//   gphi = grad(phi^{n+1}), lap = laplacian(phi^{n+1}), phi = phi^{n+1}(x), (uox,uoy,uoz) = u^n(x).
template <typename T> struct NodeOut { T p, ux, uy, uz, axx, ayy, azz, axy, axz, ayz, ax, ay, az; };

template <typename T>
__device__ __forceinline__ NodeOut<T> close_node(const DevParams<T>& P, const Mom<T>& m, T phi,
                                                 T gx, T gy, T gz, T lap, T uox, T uoy, T uoz) {
  const T cs2 = T(1.0 / 3.0);
  Mix<T> mx = mixture(P, phi);
  // chemical potential, phi_l = 1, phi_g = 0, phi_0 = 1/2
  T mu_phi = P.beta4 * phi * (phi - T(1)) * (phi - T(0.5)) - P.kappa_mu * lap;
  // Pi^neq = Pi - p* cs^2 delta - u^n u^n  (R7)
  T pc = m.p * cs2;
  T nxx = m.xx - pc - uox * uox, nyy = m.yy - pc - uoy * uoy, nzz = m.zz - pc - uoz * uoz;
  T nxy = m.xy - uox * uoy, nxz = m.xz - uox * uoz, nyz = m.yz - uoy * uoz;
  // F = mu_phi grad(phi) - p* cs^2 grad(rho) - (nu omega/cs^2) Pi^neq . grad(rho) + (rho - rho_b) g
  // with grad(rho) = drho grad(phi) (R18):  F = k1 grad(phi) - k2 Pi^neq.grad(phi) + (rho-rho_b) g
  T k1 = mu_phi - pc * P.drho;
  T k2 = mx.nuom3 * P.drho;
  T fx = k1 * gx - k2 * (nxx * gx + nxy * gy + nxz * gz);
  T fy = k1 * gy - k2 * (nxy * gx + nyy * gy + nyz * gz);
  T fz = k1 * gz - k2 * (nxz * gx + nyz * gy + nzz * gz);
  T db = mx.rho - P.rho_b;
  NodeOut<T> o;
  o.ax = fma(db, P.gx, fx) * mx.inv_rho;
  o.ay = fma(db, P.gy, fy) * mx.inv_rho;
  o.az = fma(db, P.gz, fz) * mx.inv_rho;
  o.p = m.p;
  const T h = T(0.5);
  o.ux = fma(h, o.ax, m.mx);                                   // Eq. 12, R4
  o.uy = fma(h, o.ay, m.my);
  o.uz = fma(h, o.az, m.mz);
  // Eq. 13 in closed form (R6): A = Pi - p* cs^2 d - uu + (ua + au)/2 ; stored times (1 - omega)
  T om1 = T(1) - mx.omega;
  o.axx = om1 * (m.xx - pc - o.ux * (o.ux - o.ax));
  o.ayy = om1 * (m.yy - pc - o.uy * (o.uy - o.ay));
  o.azz = om1 * (m.zz - pc - o.uz * (o.uz - o.az));
  o.axy = om1 * (m.xy - o.ux * o.uy + h * (o.ux * o.ay + o.ax * o.uy));
  o.axz = om1 * (m.xz - o.ux * o.uz + h * (o.ux * o.az + o.ax * o.uz));
  o.ayz = om1 * (m.yz - o.uy * o.uz + h * (o.uy * o.az + o.ay * o.uz));
  return o;
}

template <typename T>
__device__ __forceinline__ void store_out(T* __restrict__ D, long long N, long long idx,
                                          const NodeOut<T>& o) {
  const T m[13] = {o.p, o.ux, o.uy, o.uz, o.axx, o.ayy, o.azz, o.axy, o.axz, o.ayz, o.ax, o.ay, o.az};
  store13(D, N, idx, m);
}
template <typename T>
__device__ __forceinline__ Coef<T> coef_from13(const T (&m)[13]) {
  return coefficients<T>(m[F_P], m[F_UX], m[F_UY], m[F_UZ], m[F_AXX], m[F_AYY], m[F_AZZ], m[F_AXY],
                         m[F_AXZ], m[F_AYZ], m[F_AX], m[F_AY], m[F_AZ]);
}

// Total Allen-Cahn flux of Eq. 20 at one node (R13, R16):  Q = phi u + kappa_AC phi (1-phi) n,
// n = grad(phi)/sqrt(|grad(phi)|^2 + eps^2).  The periodic path evaluates it where grad(phi^{n+1})
// is already known (closing stage of the stream-collide kernel) and stores it for the next
// step's interface update; layout: three scalar planes Qx, Qy, Qz at offsets 0, N, 2N (so the
// interface kernel reads each of them with 128-bit loads, several nodes per thread).
template <typename T>
__device__ __forceinline__ void flux_q(const DevParams<T>& P, T phi, T gx, T gy, T gz, T ux, T uy,
                                       T uz, T (&q)[3]) {
  const T s = P.kappa_ac * phi * (T(1) - phi) * rsqrt_t(gx * gx + gy * gy + gz * gz + T(1e-24));
  q[0] = fma(phi, ux, s * gx);
  q[1] = fma(phi, uy, s * gy);
  q[2] = fma(phi, uz, s * gz);
}
template <typename T>
__device__ __forceinline__ void store_q(T* Q, long long N, long long idx, const T (&q)[3]) {
  Q[idx] = q[0];
  Q[N + idx] = q[1];
  Q[2 * N + idx] = q[2];
}
template <typename T>
__device__ __forceinline__ void load_q(const T* Q, long long N, long long idx, T (&q)[3]) {
  q[0] = __ldg(Q + idx);
  q[1] = __ldg(Q + N + idx);
  q[2] = __ldg(Q + 2 * N + idx);
}

// ---- cp.async staging of the next source planes (memory pipeline without registers) ---------
// The kernel is bound by global-memory latency unless several planes per SM are in flight
// (profiles/r1_tuning_evidence.md), and fp64 has no registers to spare for a deeper prefetch.  Each
// thread therefore copies the 14 scalars of ITS OWN node for plane j+NSTAGE straight into a
// private shared-memory slot (cp.async, no register staging) and picks them up NSTAGE iterations
// later; only cp.async.wait_group is needed, no block barrier, because nobody else reads the slot.
template <typename T, int CELLS>
struct StageBuf {
  typename VecOf<T>::type vec[12 / VecOf<T>::W][CELLS];
  T az[CELLS];
  T ph[CELLS];
};
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst)), "l"(src));
}
__device__ __forceinline__ void cp_async_small(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst)), "l"(src));
}
__device__ __forceinline__ void cp_async_small(float* dst, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst)), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// Ghost rule along one axis (R19): periodic wrap or even mirror about a wall half a cell outside
// the first/last node.  Valid for -n <= i < 2n.  crossed = 1 if mirrored.
__device__ __forceinline__ int ghost_index(int i, int n, int bc, int& crossed) {
  crossed = 0;
  if (i < 0) {
    if (bc) { crossed = 1; return -1 - i; }
    return i + n;
  }
  if (i >= n) {
    if (bc) { crossed = 1; return 2 * n - 1 - i; }
    return i - n;
  }
  return i;
}

}  // namespace tslb
