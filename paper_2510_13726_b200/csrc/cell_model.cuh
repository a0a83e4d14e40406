// cell_model.cuh -- cell model of the HHRRLBM in fp32 on population deviations f_i - w_i, on the velocity set
// HHRR_Q: D3Q27 (BASELINE.json's configs, the default build) or D3Q19 (the paper's own, Fig. 2 :107;
// the library built with -DHHRR_Q=19).
//
// PAPER.md:98 (Eq. 6), :102 (Eq. 7), :113-122 (Eq. 8-10), :126-129 (Eq. 11), :133 (Eq. 12),
// :144 (Eq. 14); readings R1-R6, R23 of DESIGN.md.  The sums over the directions are written through the
// structure of the set:
//   * D3Q27 moments: three separable passes (x, then y, then z) over c in {-1,0,1}^3          ~70 adds
//   * D3Q19 moments: sums and differences of the 9 opposite pairs, then per-axis sums           ~54 adds
//   * reconstruction: f_i = w_i (E_i + O_i), f_ibar = w_i (E_i - O_i) with E the even and
//     O the odd polynomial in c; the same Hermite algebra for both sets, only the third-order
//     coefficients differ (R3 / R23)                                                           ~220 / ~170 flops
// CUDA path only; shares nothing with oracle/.
#pragma once
#include "lattice.h"

namespace hhrr {

static_assert(Q == 27 || Q == 19, "velocity set: D3Q27 or D3Q19");

// Direction i of the set sits at slot (cx+1) + 3(cy+1) + 9(cz+1) of the 27-point cube; D3Q19 = the slots with
// |c|^2 <= 2 in the same order, so that for both sets rest = (Q-1)/2 and opposite = Q-1-i.
__host__ __device__ constexpr int dir_slot(int i) {
  if (Q == 27) return i;
  constexpr int s19[19] = {1, 3, 4, 5, 7, 9, 10, 11, 12, 13, 14, 15, 16, 17, 19, 21, 22, 23, 25};
  return s19[i < 19 ? i : 0];
}
__host__ __device__ constexpr int dir_cx(int i) { return dir_slot(i) % 3 - 1; }
__host__ __device__ constexpr int dir_cy(int i) { return (dir_slot(i) / 3) % 3 - 1; }
__host__ __device__ constexpr int dir_cz(int i) { return dir_slot(i) / 9 - 1; }
constexpr int REST = (Q - 1) / 2;
__host__ __device__ constexpr int dir_opp(int i) { return Q - 1 - i; }
// index of direction (cx, cy, cz); -1 if the set does not hold it (cube corners on D3Q19)
__host__ __device__ constexpr int dir_index(int cx, int cy, int cz) {
  const int slot = (cx + 1) + 3 * (cy + 1) + 9 * (cz + 1);
  if (Q == 27) return slot;
  // D3Q19: slot minus the number of cube-corner slots below it (arithmetic: cheap with run-time arguments too)
  constexpr unsigned corners = (1u << 0) | (1u << 2) | (1u << 6) | (1u << 8) | (1u << 18) | (1u << 20) | (1u << 24) | (1u << 26);
  if ((corners >> slot) & 1u) return -1;
  unsigned v = corners & ((1u << slot) - 1u);
  v = v - ((v >> 1) & 0x55555555u);
  v = (v & 0x33333333u) + ((v >> 2) & 0x33333333u);
  v = (v + (v >> 4)) & 0x0f0f0f0fu;
  return slot - (int)((v * 0x01010101u) >> 24);
}
// direction i with the marked components reversed (a population reflected at MIRROR planes, R12)
__host__ __device__ constexpr int dir_flip(int i, bool fx, bool fy, bool fz) {
  return dir_index(fx ? -dir_cx(i) : dir_cx(i), fy ? -dir_cy(i) : dir_cy(i), fz ? -dir_cz(i) : dir_cz(i));
}
__host__ __device__ constexpr double dir_wd(int i) {
  if (Q == 27)
    return (dir_cx(i) ? 1.0 / 6.0 : 2.0 / 3.0) * (dir_cy(i) ? 1.0 / 6.0 : 2.0 / 3.0) * (dir_cz(i) ? 1.0 / 6.0 : 2.0 / 3.0);
  const int nn = dir_cx(i) * dir_cx(i) + dir_cy(i) * dir_cy(i) + dir_cz(i) * dir_cz(i);
  return nn == 0 ? 1.0 / 3.0 : (nn == 1 ? 1.0 / 18.0 : 1.0 / 36.0);
}
__host__ __device__ constexpr float dir_w(int i) { return (float)dir_wd(i); }
__host__ __device__ constexpr double dir_wd_of(int cx, int cy, int cz) {  // weight of direction (cx, cy, cz)
  if (Q == 27) return (cx ? 1.0 / 6.0 : 2.0 / 3.0) * (cy ? 1.0 / 6.0 : 2.0 / 3.0) * (cz ? 1.0 / 6.0 : 2.0 / 3.0);
  const int nn = cx * cx + cy * cy + cz * cz;
  return nn == 0 ? 1.0 / 3.0 : (nn == 1 ? 1.0 / 18.0 : 1.0 / 36.0);
}

// MUFU reciprocal + one Newton step (<= 1 ulp, branch-free) and MUFU square root (2^-23 rel.)
__device__ __forceinline__ float rcp_nr(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return fmaf(r, fmaf(-x, r, 1.f), r);
}
__device__ __forceinline__ float sqrt_fast(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// Two x-adjacent cells in one register pair (.x: cell x, .y: cell x + 1): sm_100's packed fp32 arithmetic
// (FADD2 / FMUL2 / FFMA2) runs the same instruction stream on both -- half the issue slots of the scalar code.
// Every arithmetic routine below is a template over T = float (one cell) or T = f2 (a cell pair).
struct f2 {
  float2 v;
};
__device__ __forceinline__ f2 mk2(float a, float b) { return f2{make_float2(a, b)}; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return f2{__fadd2_rn(a.v, b.v)}; }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return f2{__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))}; }
__device__ __forceinline__ f2 operator-(f2 a) { return f2{make_float2(-a.v.x, -a.v.y)}; }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return f2{__fmul2_rn(a.v, b.v)}; }
__device__ __forceinline__ f2 operator*(float s, f2 b) { return f2{__fmul2_rn(make_float2(s, s), b.v)}; }
__device__ __forceinline__ f2 operator*(f2 a, float s) { return f2{__fmul2_rn(a.v, make_float2(s, s))}; }
__device__ __forceinline__ f2 operator+(f2 a, float s) { return f2{__fadd2_rn(a.v, make_float2(s, s))}; }
__device__ __forceinline__ f2 operator+(float s, f2 a) { return f2{__fadd2_rn(a.v, make_float2(s, s))}; }
__device__ __forceinline__ f2 operator-(f2 a, float s) { return f2{__fadd2_rn(a.v, make_float2(-s, -s))}; }
__device__ __forceinline__ f2 operator-(float s, f2 a) { return f2{__fadd2_rn(make_float2(s, s), make_float2(-a.v.x, -a.v.y))}; }
__device__ __forceinline__ f2 fma_t(f2 a, f2 b, f2 c) { return f2{__ffma2_rn(a.v, b.v, c.v)}; }
__device__ __forceinline__ f2 fma_t(float a, f2 b, f2 c) { return f2{__ffma2_rn(make_float2(a, a), b.v, c.v)}; }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ f2 rcp_nr(f2 x) { return mk2(rcp_nr(x.v.x), rcp_nr(x.v.y)); }
__device__ __forceinline__ f2 sqrt_fast(f2 x) { return mk2(sqrt_fast(x.v.x), sqrt_fast(x.v.y)); }
template <class T> __device__ __forceinline__ T bcast(float s);
template <> __device__ __forceinline__ float bcast<float>(float s) { return s; }
template <> __device__ __forceinline__ f2 bcast<f2>(float s) { return mk2(s, s); }

template <class T>
struct MomentsT {  // of the deviations: drho = rho - 1, j, M_ab = sum c_a c_b (f - w)
  T drho, jx, jy, jz, mxx, myy, mzz, mxy, mxz, myz;
};
using Moments = MomentsT<float>;

// Sums over the directions, per velocity set.
template <class T, int NQ>
struct CellSums;

// D3Q27: three separable passes (x, then y, then z)
template <class T>
struct CellSums<T, 27> {
  // rho and j only (halo cells, moments pass, read-back)
  static __device__ __forceinline__ void rho_j(const T (&f)[27], T& drho, T& jx, T& jy, T& jz) {
  T s0[9], s1[9];
#pragma unroll
  for (int m = 0; m < 9; ++m) {
    T fm = f[3 * m], f0 = f[3 * m + 1], fp = f[3 * m + 2];
    s0[m] = (fp + fm) + f0;
    s1[m] = fp - fm;
  }
  T t00[3], t01[3], t10[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    t00[k] = (s0[3 * k + 2] + s0[3 * k]) + s0[3 * k + 1];
    t01[k] = s0[3 * k + 2] - s0[3 * k];
    t10[k] = (s1[3 * k + 2] + s1[3 * k]) + s1[3 * k + 1];
  }
  drho = (t00[2] + t00[0]) + t00[1];
  jz = t00[2] - t00[0];
  jy = (t01[2] + t01[0]) + t01[1];
  jx = (t10[2] + t10[0]) + t10[1];
}

  static __device__ __forceinline__ MomentsT<T> all(const T (&f)[27]) {
  T s0[9], s1[9], s2[9];
#pragma unroll
  for (int m = 0; m < 9; ++m) {
    T fm = f[3 * m], f0 = f[3 * m + 1], fp = f[3 * m + 2];
    s2[m] = fp + fm;
    s0[m] = s2[m] + f0;
    s1[m] = fp - fm;
  }
  T t00[3], t01[3], t02[3], t10[3], t11[3], t20[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    t02[k] = s0[3 * k + 2] + s0[3 * k];
    t00[k] = t02[k] + s0[3 * k + 1];
    t01[k] = s0[3 * k + 2] - s0[3 * k];
    t10[k] = (s1[3 * k + 2] + s1[3 * k]) + s1[3 * k + 1];
    t11[k] = s1[3 * k + 2] - s1[3 * k];
    t20[k] = (s2[3 * k + 2] + s2[3 * k]) + s2[3 * k + 1];
  }
  MomentsT<T> m;
  m.mzz = t00[2] + t00[0];
  m.drho = m.mzz + t00[1];
  m.jz = t00[2] - t00[0];
  m.jy = (t01[2] + t01[0]) + t01[1];
  m.myz = t01[2] - t01[0];
  m.myy = (t02[2] + t02[0]) + t02[1];
  m.jx = (t10[2] + t10[0]) + t10[1];
  m.mxz = t10[2] - t10[0];
  m.mxy = (t11[2] + t11[0]) + t11[1];
  m.mxx = (t20[2] + t20[0]) + t20[1];
  return m;
}

};

// D3Q19: sum s and difference d of each opposite pair (direction j > REST minus direction Q-1-j), then the
// per-axis sums; the compile-time direction components pick the terms
template <class T>
struct CellSums<T, 19> {
  struct Acc {  // sum of signed terms without a leading zero
    T v;
    bool any = false;
    __device__ __forceinline__ void add(const T& t, int sgn) {
      if (!any) v = sgn > 0 ? t : -t;
      else v = sgn > 0 ? v + t : v - t;
      any = true;
    }
  };
  // rho and j in EXACTLY the summation order of all(): a plane's uhat must not depend on which of the two a block
  // uses for it (overlap planes of a z-chunk take rho_j, the neighbouring chunk takes all())
  static __device__ __forceinline__ void rho_j(const T (&f)[19], T& drho, T& jx, T& jy, T& jz) {
    Acc x, y, z, zz;
    T sd = f[9];
#pragma unroll
    for (int j = 10; j < 19; ++j) {
      const T s = f[j] + f[18 - j], d = f[j] - f[18 - j];
      if (dir_cx(j)) x.add(d, dir_cx(j));
      if (dir_cy(j)) y.add(d, dir_cy(j));
      if (dir_cz(j)) z.add(d, dir_cz(j));
      if (dir_cz(j)) zz.add(s, 1);
      else sd = sd + s;
    }
    drho = sd + zz.v; jx = x.v; jy = y.v; jz = z.v;
  }
  static __device__ __forceinline__ MomentsT<T> all(const T (&f)[19]) {
    Acc x, y, z, xx, yy, zz, xy, xz, yz, ax;  // ax: the axis pairs (one non-zero component)
    T sd = f[9];                              // rest + face-diagonal pairs not counted in mzz
#pragma unroll
    for (int j = 10; j < 19; ++j) {
      const int cx = dir_cx(j), cy = dir_cy(j), cz = dir_cz(j);
      const T s = f[j] + f[18 - j], d = f[j] - f[18 - j];
      if (cx) x.add(d, cx);
      if (cy) y.add(d, cy);
      if (cz) z.add(d, cz);
      if (cx) xx.add(s, 1);
      if (cy) yy.add(s, 1);
      if (cz) zz.add(s, 1);
      if (cx * cy) xy.add(s, cx * cy);
      if (cx * cz) xz.add(s, cx * cz);
      if (cy * cz) yz.add(s, cy * cz);
      if (!cz) sd = sd + s;
    }
    MomentsT<T> m;
    m.drho = sd + zz.v;
    m.jx = x.v; m.jy = y.v; m.jz = z.v;
    m.mxx = xx.v; m.myy = yy.v; m.mzz = zz.v;
    m.mxy = xy.v; m.mxz = xz.v; m.myz = yz.v;
    return m;
  }
};

template <class T>
__device__ __forceinline__ void moments_rho_j(const T (&f)[Q], T& drho, T& jx, T& jy, T& jz) {
  CellSums<T, Q>::rho_j(f, drho, jx, jy, jz);
}
template <class T>
__device__ __forceinline__ MomentsT<T> moments_all(const T (&f)[Q]) {
  return CellSums<T, Q>::all(f);
}

// u^B of a cell (fringe R12), without the wall-model slip
__device__ __forceinline__ void solid_velocity(const PhysF& ph, const BodiesF& bo, uint8_t flags, int x,
                                               int y, int z, float uB[3]) {
  int type = flags & TYPE_MASK;
  uB[0] = uB[1] = uB[2] = 0.f;
  if (type == HHRR_FRINGE) {
    uB[0] = ph.fr_u[0];
    uB[1] = ph.fr_u[1];
    uB[2] = ph.fr_u[2];
  } else if (type == HHRR_SOLID || type == HHRR_FRONTIER || type == T_FRONTIER_W) {
    int k = (flags >> TAG_SHIFT) & TAG_MASK;
    float rx = (float)x - bo.c[k][0], ry = (float)y - bo.c[k][1], rz = (float)z - bo.c[k][2];
    uB[0] = bo.v[k][0] + (bo.w[k][1] * rz - bo.w[k][2] * ry);
    uB[1] = bo.v[k][1] + (bo.w[k][2] * rx - bo.w[k][0] * rz);
    uB[2] = bo.v[k][2] + (bo.w[k][0] * ry - bo.w[k][1] * rx);
  }
}

// hybrid factor of a cell: bulk cells run Listing 2's model, Eq. 7 at sigma = 1 (R20)
__device__ __forceinline__ float cell_sigma(const PhysF& ph, uint8_t flags) {
  return (flags & TYPE_MASK) == HHRR_BULK ? 1.f : ph.sigma;
}
__device__ __forceinline__ bool type_has_solid_state(int type) {  // FRONTIER (in W or not), SOLID, FRINGE: d < 1, u^B
  return (type >= HHRR_FRONTIER && type <= HHRR_FRINGE) || type == T_FRONTIER_W;
}
__device__ __forceinline__ bool type_is_frontier(int type) { return type == HHRR_FRONTIER || type == T_FRONTIER_W; }

// Eq. 12 with reading R1 (d = 1 fluid): uhat = d u + (1-d) u^B, u = (j + g)/rho  (R11)
template <class T>
__device__ __forceinline__ void homogenised_velocity(const PhysF& ph, T drho, T jx, T jy, T jz, T d, const T uB[3],
                                                     T& rho, T uh[3]) {
  rho = 1.f + drho;
  T ir = rcp_nr(rho);
  T ux = (jx + ph.g[0]) * ir, uy = (jy + ph.g[1]) * ir, uz = (jz + ph.g[2]) * ir;
  T e = 1.f - d;
  uh[0] = d * ux + e * uB[0];
  uh[1] = d * uy + e * uB[1];
  uh[2] = d * uz + e * uB[2];
}

// One collision.  m: moments of the deviations; rho, uh: from homogenised_velocity;
// S: strain handed to the hybrid term (xx yy zz xy xz yz); sigma: this cell's hybrid factor.
// Output: post-collision deviations f*_i - w_i.
template <class T>
__device__ __forceinline__ void collide(const PhysF& ph, const MomentsT<T>& m, T rho, const T uh[3], const T S[6],
                                        T sigma, T (&out)[Q]) {
  const float third = 1.f / 3.f;
  T ux = uh[0], uy = uh[1], uz = uh[2];
  T rux = rho * ux, ruy = rho * uy, ruz = rho * uz;
  // Pi^neq = sum H2 f - rho uh uh  (R4)
  T dr3 = third * m.drho;
  T pxx = m.mxx - dr3 - rux * ux, pyy = m.myy - dr3 - ruy * uy, pzz = m.mzz - dr3 - ruz * uz;
  T pxy = m.mxy - rux * uy, pxz = m.mxz - rux * uz, pyz = m.myz - ruy * uz;
  // Smagorinsky closed form (Eq. 3-5, 14; R6)
  T pp = pxx * pxx + pyy * pyy + pzz * pzz + 2.f * (pxy * pxy + pxz * pxz + pyz * pyz);
  T Qn = sqrt_fast(2.f * pp);
  T tau = 0.5f * (ph.tau0 + sqrt_fast(ph.tau0 * ph.tau0 + ph.smag18 * (Qn * rcp_nr(rho))));
  T k = 1.f - rcp_nr(tau);
  // hybrid a1^(2) (Eq. 7 + Eq. 10; R2), already scaled by k = 1 - 1/tau_eff (Eq. 6)
  T ks = k * sigma, kh = k * ((1.f - sigma) * ((2.f * third) * (rho * tau)));
  T axx = ks * pxx - kh * S[0], ayy = ks * pyy - kh * S[1], azz = ks * pzz - kh * S[2];
  T axy = ks * pxy - kh * S[3], axz = ks * pxz - kh * S[4], ayz = ks * pyz - kh * S[5];
  // second order: T = 4.5 (rho uh uh + k a2)
  T Txx = 4.5f * (rux * ux + axx), Tyy = 4.5f * (ruy * uy + ayy), Tzz = 4.5f * (ruz * uz + azz);
  T Txy = 9.f * (rux * uy + axy), Txz = 9.f * (rux * uz + axz), Tyz = 9.f * (ruy * uz + ayz);
  // third order: A3_aab = rho ua ua ub + k (2 ua a_ab + ub a_aa) (recursion of R3); G_ab = coefficient of H_aab.
  // D3Q27 (R3): G_ab = 13.5 A3_aab, Gxyz = 27 A3_xyz.  D3Q19 (R23, basis of the paper's ref. [43]): per group
  // (H1, H2) in {(xxy, yzz), (xzz, xyy), (yyz, xxz)} the term is 13.5 (H1 + H2)(A1 + A2) + 4.5 (H1 - H2)(A1 - A2),
  // i.e. coefficient 18 A1 + 9 A2 of H1 and 9 A1 + 18 A2 of H2; H_xyz is not supported.
  T ux2 = ux + ux, uy2 = uy + uy, uz2 = uz + uz;
  T Axy = (rux * ux) * uy + (ux2 * axy + uy * axx);  // xx y
  T Axz = (rux * ux) * uz + (ux2 * axz + uz * axx);  // xx z
  T Ayx = (ruy * uy) * ux + (uy2 * axy + ux * ayy);  // yy x
  T Ayz = (ruy * uy) * uz + (uy2 * ayz + uz * ayy);  // yy z
  T Azx = (ruz * uz) * ux + (uz2 * axz + ux * azz);  // zz x
  T Azy = (ruz * uz) * uy + (uz2 * ayz + uy * azz);  // zz y
  T Gxy, Gxz, Gyx, Gyz, Gzx, Gzy, Gxyz = bcast<T>(0.f);
  if (Q == 27) {
    Gxy = 13.5f * Axy; Gxz = 13.5f * Axz; Gyx = 13.5f * Ayx; Gyz = 13.5f * Ayz; Gzx = 13.5f * Azx; Gzy = 13.5f * Azy;
    Gxyz = 27.f * ((rux * uy) * uz + (ux * ayz + uy * axz + uz * axy));
  } else {
    Gxy = 18.f * Axy + 9.f * Azy; Gzy = 9.f * Axy + 18.f * Azy;  // (xxy, yzz)
    Gzx = 18.f * Azx + 9.f * Ayx; Gyx = 9.f * Azx + 18.f * Ayx;  // (xzz, xyy)
    Gyz = 18.f * Ayz + 9.f * Axz; Gxz = 9.f * Ayz + 18.f * Axz;  // (yyz, xxz)
  }
  // even part tables: q(c) = c^2 - 1/3
  T Ex[2] = {-third * Txx, (2.f * third) * Txx};
  T Ey[2] = {-third * Tyy, (2.f * third) * Tyy};
  T Ez[2] = {m.drho - third * Tzz, m.drho + (2.f * third) * Tzz};
  // odd part: coefficient of c_b is m_b + sum_{a != b} q(c_a) G_ab
  T mx = 3.f * rux, my = 3.f * ruy, mz = 3.f * ruz;
  T OX[2][2], OY[2][2], OZ[2][2];  // [other axis 1 squared][other axis 2 squared]
#pragma unroll
  for (int p = 0; p < 2; ++p)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      float qp = p ? 2.f * third : -third, qq = q ? 2.f * third : -third;
      OX[p][q] = mx + qp * Gyx + qq * Gzx;  // p: cy^2, q: cz^2
      OY[p][q] = my + qp * Gxy + qq * Gzy;  // p: cx^2, q: cz^2
      OZ[p][q] = mz + qp * Gxz + qq * Gyz;  // p: cx^2, q: cy^2
    }
#pragma unroll
  for (int i = 0; i <= REST; ++i) {
    const int cx = dir_cx(i), cy = dir_cy(i), cz = dir_cz(i);
    const int x2 = cx * cx, y2 = cy * cy, z2 = cz * cz;
    T E = Ex[x2] + Ey[y2] + Ez[z2];
    if (cx * cy == 1) E = E + Txy;
    if (cx * cy == -1) E = E - Txy;
    if (cx * cz == 1) E = E + Txz;
    if (cx * cz == -1) E = E - Txz;
    if (cy * cz == 1) E = E + Tyz;
    if (cy * cz == -1) E = E - Tyz;
    const float w = dir_w(i);
    if (i == REST) {
      out[REST] = w * E;
    } else {
      T O = bcast<T>(0.f);
      bool first = true;
      auto acc = [&](const T& v, int sgn) {
        if (first) { O = sgn > 0 ? v : -v; first = false; }
        else O = sgn > 0 ? O + v : O - v;
      };
      if (cx) acc(OX[y2][z2], cx);
      if (cy) acc(OY[x2][z2], cy);
      if (cz) acc(OZ[x2][y2], cz);
      if (Q == 27 && cx * cy * cz) acc(Gxyz, cx * cy * cz);
      const T wE = w * E;
      out[i] = fma_t(w, O, wE);
      out[dir_opp(i)] = fma_t(-w, O, wE);
    }
  }
}

// where population i of the post-stream state of cell (x,y,z) is stored (see Dom::xs)
// (cx = c_x of direction i, passed by callers that know it at compile time while i is a run-time value)
__device__ __forceinline__ int64_t pop_index_cx(const Dom& dm, int i, int cx, int x, int y, int z) {
  int xs = x - dm.xs * cx;
  if (xs < 0) xs += dm.nx;
  else if (xs >= dm.nx) xs -= dm.nx;
  return (int64_t)i * dm.n + xs + (int64_t)dm.nx * (y + (int64_t)dm.ny * z);
}
__device__ __forceinline__ int64_t pop_index(const Dom& dm, int i, int x, int y, int z) {
  int xs = x - dm.xs * dir_cx(i);
  if (xs < 0) xs += dm.nx;
  else if (xs >= dm.nx) xs -= dm.nx;
  return (int64_t)i * dm.n + xs + (int64_t)dm.nx * (y + (int64_t)dm.ny * z);
}

// neighbour index along one axis with the outer-boundary rule R12.
// Returns the wrapped / reflected coordinate; flip = true if it was reflected.
__device__ __forceinline__ int wrap_axis(int v, int n, int mode, bool& flip) {
  flip = false;
  if (v >= 0 && v < n) return v;
  if (mode == HHRR_PERIODIC) return v < 0 ? v + n : v - n;
  flip = true;
  return v < 0 ? -1 - v : 2 * n - 1 - v;
}

// push-store of the 27 post-collision values with the outer-boundary rule R12
__device__ __forceinline__ void push_store(const Dom& dm, float* __restrict__ fout, int x, int y, int z,
                                           const float (&o)[Q]) {
  bool fxm, fxp, fym, fyp, fzm, fzp;
  int xm = wrap_axis(x - 1, dm.nx, dm.mode[0], fxm), xp = wrap_axis(x + 1, dm.nx, dm.mode[0], fxp);
  int ym = wrap_axis(y - 1, dm.ny, dm.mode[1], fym), yp = wrap_axis(y + 1, dm.ny, dm.mode[1], fyp);
  int zm = wrap_axis(z - 1, dm.nz, dm.mode[2], fzm), zp = wrap_axis(z + 1, dm.nz, dm.mode[2], fzp);
  const int64_t nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  if (!(fxm | fxp | fym | fyp | fzm | fzp)) {
    int xs[3] = {xm, x, xp};
    int64_t ys[3] = {ym * nx, y * nx, yp * nx};
    int64_t zs[3] = {zm * nxy, z * nxy, zp * nxy};
#pragma unroll
    for (int i = 0; i < Q; ++i)
      fout[(int64_t)i * dm.n + zs[dir_cz(i) + 1] + ys[dir_cy(i) + 1] + xs[dir_cx(i) + 1]] = o[i];
  } else {
    // a population leaving through a mirror plane returns to the same cell, component reversed
#pragma unroll
    for (int i = 0; i < Q; ++i) {
      int cx = dir_cx(i), cy = dir_cy(i), cz = dir_cz(i);
      int tx = cx < 0 ? xm : (cx > 0 ? xp : x);
      int ty = cy < 0 ? ym : (cy > 0 ? yp : y);
      int tz = cz < 0 ? zm : (cz > 0 ? zp : z);
      if ((cx < 0 && fxm) || (cx > 0 && fxp)) { tx = x; cx = -cx; }
      if ((cy < 0 && fym) || (cy > 0 && fyp)) { ty = y; cy = -cy; }
      if ((cz < 0 && fzm) || (cz > 0 && fzp)) { tz = z; cz = -cz; }
      int io = dir_index(cx, cy, cz);
      fout[(int64_t)io * dm.n + tz * nxy + ty * nx + tx] = o[i];
    }
  }
}

}  // namespace hhrr
