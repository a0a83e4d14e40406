// wallmodel.cu -- K3: WallModelO (Listing 3 line 4; Eq. 15-20 :159-184; :186;
// :324) on the compact wall-cell list, and K4: boundary force collection + per-element
// integration (Listing 3 lines 5-6, :315-317; Eq. 23 :211; :267).
//
// Both kernels touch 1e4-1e5 cells, so they run in fp64 on the fp32 populations: the Newton
// stop rule (:184) decides an iteration count, and it is taken in the same precision as the
// oracle takes it.  Forces accumulate in fp64.  K3 is ONE launch on the critical path between two
// collide-stream kernels (its output feeds the next collision); K4 only reads the streamed populations
// and runs on the side stream beside the next collide-stream kernel.
// CUDA path only; shares nothing with oracle/.
#include <algorithm>

#include "cell_model.cuh"

namespace hhrr {

struct WmArgs {
  Dom dm;
  double g[3];
  double nu, kappa, E, tol, hs;
  int max_iter;
  int wall_function;  // 0 truncated Spalding, 1 Musker
  int wm_slip;        // 0: u_wm = u_tau e_t; 1: wall-function velocity at y1 (hhrr_set_wall_model_variant)
  int wm_shear;       // 0: one-sided difference; 1: analytic slope of the wall function
  BodiesD bo;
  const float* f;  // post-stream populations (deviations)
  uint8_t* flags;
  const int32_t* wall_idx;
  const double* wall_y1n;
  const Counters* cnt;
  int cap_list;
  double* samp;  // [cap_list][6]: sampled velocity v_s and the cell's own velocity v(x_w), sampling kernel -> Newton kernel
  double* wm_utau;
  float* wm_u;
  float* wm_s;
};

__device__ __forceinline__ int wrap_far(int v, int n, int mode, bool& flip) {
  flip = false;
  if (v >= 0 && v < n) return v;
  if (mode == HHRR_PERIODIC) return ((v % n) + n) % n;
  flip = true;
  return v < 0 ? -1 - v : 2 * n - 1 - v;
}

// reported velocity moment v = (j + g/2)/rho of a cell (R11)
__device__ __forceinline__ void cell_velocity_d(const float* __restrict__ f, const Dom& dm, int x, int y, int z,
                                                const double g[3], double v[3]) {
  double drho = 0, j0 = 0, j1 = 0, j2 = 0;
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    double fi = (double)__ldg(f + pop_index(dm, i, x, y, z));
    drho += fi;
    j0 += dir_cx(i) * fi;
    j1 += dir_cy(i) * fi;
    j2 += dir_cz(i) * fi;
  }
  double ir = 1.0 / (1.0 + drho);
  v[0] = (j0 + 0.5 * g[0]) * ir;
  v[1] = (j1 + 0.5 * g[1]) * ir;
  v[2] = (j2 + 0.5 * g[2]) * ir;
}

__device__ __forceinline__ void body_velocity_d(const BodiesD& bo, int k, int x, int y, int z, double us[3]) {
  double r0 = x - bo.c[k][0], r1 = y - bo.c[k][1], r2 = z - bo.c[k][2];
  us[0] = bo.v[k][0] + (bo.w[k][1] * r2 - bo.w[k][2] * r1);
  us[1] = bo.v[k][1] + (bo.w[k][2] * r0 - bo.w[k][0] * r2);
  us[2] = bo.v[k][2] + (bo.w[k][0] * r1 - bo.w[k][1] * r0);
}

// truncated Spalding law (Eq. 18) and its u_tau derivative (R9)
__device__ __forceinline__ double spalding_f(double ut, double U, double y, double nu, double kap, double E) {
  double up = U / ut, k = kap * up;
  return up + (exp(k) - 1.0 - k - 0.5 * k * k - k * k * k / 6.0) / E - y * ut / nu;
}
__device__ __forceinline__ double spalding_df(double ut, double U, double y, double nu, double kap, double E) {
  double up = U / ut, k = kap * up;
  return -(U / (ut * ut)) * (1.0 + (kap / E) * (exp(k) - 1.0 - k - 0.5 * k * k)) - y / nu;
}

// fp64 value of another lane
__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_down_d(double v, int delta) { return __shfl_down_sync(0xffffffffu, v, delta); }

// K3 = two launches on the critical path between two collide-stream kernels.
// wall_sample_kernel: a WARP takes a batch of WM_BATCH wall-model cells.  Phase 1: for every cell of the batch, lane
// 3k + g (k = 0..8, g = 0..2) issues the loads of up to nine populations of cell k -- k = 0..7 the corners of the
// trilinear stencil around x_w + h_s n (R15), k = 8 the wall cell itself -- so the 243 gathered loads
// of ALL cells of the batch are in flight before any is used (the kernel is bound by the latency of these gathers:
// 27 planes, one page each).  Phase 2: per cell the partial sums meet by shuffles; lane j stores v_s and v(x_w).
// wall_model_kernel: one THREAD per cell (32 Newton solves per fp64 instruction): tangential speed, Newton iteration
// on Eq. 18 (Eq. 19; fp64 exp), slip velocity and wall strain.  (Both in one launch, with the Newton solves on a few
// lanes of the sampling warps, was measured slower: 148 vs 87 us -- the fp64 pipe then runs a quarter full.)

// what a lane needs to finish its part of one wall cell's sample once its nine loads have landed
// neighbour coordinate with the outer-boundary rule R12 for SMALL offsets (a few cells beyond the lattice): no integer
// division; the loops run at most once unless the lattice is only a few cells wide
__device__ __forceinline__ int wrap_near(int v, int n, int mode, bool& flip) {
  flip = false;
  if (mode == HHRR_PERIODIC) {
    while (v < 0) v += n;
    while (v >= n) v -= n;
    return v;
  }
  while (v < 0 || v >= n) {  // reflections at the two planes alternate
    v = v < 0 ? -1 - v : 2 * n - 1 - v;
    flip = !flip;
  }
  return v;
}

// Per wall cell, computed ONCE by the lane that owns the list entry and handed to the warp by shuffles: the cell, the
// base corner of the trilinear stencil around x_w + h_s n (R15) and the three weights.
struct SamplePoint {
  int x, y, z;        // the wall cell
  int ix, iy, iz;     // base corner of the stencil
  double tx, ty, tz;  // interpolation weights
};
__device__ __forceinline__ SamplePoint sample_point(const WmArgs& a, int c, const double y1v[3]) {
  SamplePoint p;
  const unsigned cu = (unsigned)c, nx = (unsigned)a.dm.nx, ny = (unsigned)a.dm.ny;  // cells are int32 list entries
  const unsigned row = cu / nx;
  p.x = (int)(cu - row * nx);
  p.z = (int)(row / ny);
  p.y = (int)(row - (unsigned)p.z * ny);
  double y1 = sqrt(y1v[0] * y1v[0] + y1v[1] * y1v[1] + y1v[2] * y1v[2]);
  double nrm[3] = {y1v[0] / y1, y1v[1] / y1, y1v[2] / y1};
  double px = p.x + a.hs * nrm[0], py = p.y + a.hs * nrm[1], pz = p.z + a.hs * nrm[2];
  double fx = floor(px), fy = floor(py), fz = floor(pz);
  p.tx = px - fx;
  p.ty = py - fy;
  p.tz = pz - fz;
  p.ix = (int)fx;
  p.iy = (int)fy;
  p.iz = (int)fz;
  return p;
}
__device__ __forceinline__ SamplePoint shfl_point(const SamplePoint& p, int src) {
  SamplePoint q;
  q.x = __shfl_sync(0xffffffffu, p.x, src);
  q.y = __shfl_sync(0xffffffffu, p.y, src);
  q.z = __shfl_sync(0xffffffffu, p.z, src);
  q.ix = __shfl_sync(0xffffffffu, p.ix, src);
  q.iy = __shfl_sync(0xffffffffu, p.iy, src);
  q.iz = __shfl_sync(0xffffffffu, p.iz, src);
  q.tx = shfl_d(p.tx, src);
  q.ty = shfl_d(p.ty, src);
  q.tz = shfl_d(p.tz, src);
  return q;
}

struct SampleLane {
  float fv[9];    // populations with cz = g - 1 of stencil cell kc (zeros where the set has no such direction)
  double w;       // trilinear weight of stencil cell kc (0 for the wall cell itself, kc = 8)
  bool flx, fly, flz;
};

// phase 1: addresses and loads of this lane (lane 3k + g: stencil cell k, population group g; lanes 27-31 idle)
__device__ __forceinline__ void wall_sample_issue(const WmArgs& a, const SamplePoint& p, int lane, SampleLane& sl) {
  const int kc = lane / 3, g = lane - 3 * kc;
  int xx = p.x, yy = p.y, zz = p.z;
  sl.flx = sl.fly = sl.flz = false;
  sl.w = 0.0;
  if (kc < 8) {
    int ox = kc & 1, oy = (kc >> 1) & 1, oz = (kc >> 2) & 1;
    sl.w = (ox ? p.tx : 1.0 - p.tx) * (oy ? p.ty : 1.0 - p.ty) * (oz ? p.tz : 1.0 - p.tz);
    xx = wrap_near(p.ix + ox, a.dm.nx, a.dm.mode[0], sl.flx);
    yy = wrap_near(p.iy + oy, a.dm.ny, a.dm.mode[1], sl.fly);
    zz = wrap_near(p.iz + oz, a.dm.nz, a.dm.mode[2], sl.flz);
  }
  const int64_t yz = (int64_t)a.dm.nx * (yy + (int64_t)a.dm.ny * zz);
#pragma unroll
  for (int q = 0; q < 9; ++q) {  // cx = q % 3 - 1, cy = q / 3 - 1, cz = g - 1
    const int i = dir_index(q % 3 - 1, q / 3 - 1, g - 1);  // -1: the set has no such direction (D3Q19 corners)
    int xs = xx - a.dm.xs * (q % 3 - 1);                   // population storage, as pop_index
    if (xs < 0) xs += a.dm.nx;
    else if (xs >= a.dm.nx) xs -= a.dm.nx;
    sl.fv[q] = (kc < 9 && i >= 0) ? __ldg(a.f + (int64_t)i * a.dm.n + yz + xs) : 0.f;
  }
}

// phase 2: v = (j + g/2)/rho of the nine cells (R11); v_s = weighted sum over the stencil as a tree over lanes 0, 3, ..,
// 21 (valid on lane 0), v_w = the wall cell's own (every lane)
__device__ __forceinline__ void wall_sample_reduce(const WmArgs& a, const SampleLane& sl, int lane, double vs[3],
                                                   double vw[3]) {
  const int g = lane % 3;
  double drho = 0, j0 = 0, j1 = 0, j2 = 0;
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    double fi = (double)sl.fv[q];
    drho += fi;
    j0 += (q % 3 - 1) * fi;
    j1 += (q / 3 - 1) * fi;
  }
  j2 = (g - 1) * drho;
  // the three groups of a cell: lanes 3k, 3k+1, 3k+2
  drho += shfl_down_d(drho, 1) + shfl_down_d(drho, 2);
  j0 += shfl_down_d(j0, 1) + shfl_down_d(j0, 2);
  j1 += shfl_down_d(j1, 1) + shfl_down_d(j1, 2);
  j2 += shfl_down_d(j2, 1) + shfl_down_d(j2, 2);
  double ir = 1.0 / (1.0 + drho);  // valid on lanes 3k
  double v[3] = {(j0 + 0.5 * a.g[0]) * ir, (j1 + 0.5 * a.g[1]) * ir, (j2 + 0.5 * a.g[2]) * ir};
  if (sl.flx) v[0] = -v[0];
  if (sl.fly) v[1] = -v[1];
  if (sl.flz) v[2] = -v[2];
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    vw[q] = shfl_d(v[q], 24);
    double t = sl.w * v[q];    // lanes 3k + 1, 3k + 2 and the wall cell's carry values nobody reads (w = 0 on lane 24)
    t += shfl_down_d(t, 12);   // stencil cell k + 4
    t += shfl_down_d(t, 6);    // k + 2
    t += shfl_down_d(t, 3);    // k + 1
    vs[q] = t;
  }
}

// Musker's explicit profile and its slope (include/hhrr.h: hhrr_set_wall_function); residual U/u_tau - u+(y u_tau/nu)
__device__ __forceinline__ double musker_uplus(double yp) {
  double q = yp * yp - 8.15 * yp + 86.0;
  return 5.424 * atan((2.0 * yp - 8.15) / 16.7) + log10(pow(yp + 10.6, 9.6) / (q * q)) - 3.52;
}
__device__ __forceinline__ double musker_duplus(double yp) {
  double a = (2.0 * yp - 8.15) / 16.7;
  return 5.424 * (2.0 / 16.7) / (1.0 + a * a) +
         (9.6 / (yp + 10.6) - 2.0 * (2.0 * yp - 8.15) / (yp * yp - 8.15 * yp + 86.0)) / log(10.0);
}
__device__ __forceinline__ double wall_f(int kind, double ut, double U, double y, double nu, double kap, double E) {
  return kind == 1 ? U / ut - musker_uplus(y * ut / nu) : spalding_f(ut, U, y, nu, kap, E);
}
__device__ __forceinline__ double wall_df(int kind, double ut, double U, double y, double nu, double kap, double E) {
  return kind == 1 ? -U / (ut * ut) - musker_duplus(y * ut / nu) * y / nu : spalding_df(ut, U, y, nu, kap, E);
}

// Second readings (include/hhrr.h: hhrr_set_wall_model_variant).  u+(y+) of the truncated Spalding law: Newton on
// Eq. 17 read as h(u+) = 0, h increasing and convex; started at min(y+, 60/kappa) >= root.
__device__ __forceinline__ double spalding_uplus(double yp, double kap, double E) {
  if (!(yp > 0.0)) return 0.0;
  double u = yp < 60.0 / kap ? yp : 60.0 / kap;
  for (int it = 0; it < 200; ++it) {
    double k = kap * u, ek = exp(k);
    double h = u + (ek - 1.0 - k - 0.5 * k * k - k * k * k / 6.0) / E - yp;
    double dh = 1.0 + (kap / E) * (ek - 1.0 - k - 0.5 * k * k);
    double un = u - h / dh;
    bool done = !(fabs(un - u) > 1e-15 * fabs(un));
    u = un;
    if (done) break;
  }
  return u;
}
// du/dy = (u_tau^2/nu) du+/dy+ of the wall function at the sampling point
__device__ __forceinline__ double wall_shear(int kind, double ut, double U, double y, double nu, double kap, double E) {
  double slope;
  if (kind == 1) {
    slope = musker_duplus(y * ut / nu);
  } else {
    double k = kap * (U / ut);
    slope = 1.0 / (1.0 + (kap / E) * (exp(k) - 1.0 - k - 0.5 * k * k));
  }
  return ut * ut / nu * slope;
}

// Outputs of the allocation-free entry point (hhrr_wall_model_noalloc, end of this file): per list entry e instead
// of per cell, in caller-owned device arrays; the lattice's own wall-model state is neither read nor written.
struct WmDirect {
  const double* start;  // [count] warm-start u_tau per entry (<= 0: none, Eq. 20's cold start), or NULL
  double* utau;         // [count]
  float* u;             // [count][3]
  float* s;             // [count][6]
};

// one wall-model cell: tangential speed relative to the wall, u_tau, slip velocity, wall strain, state valid.
// DIRECT = false (every existing caller): warm start from, and results into, the lattice's per-cell state.
template <bool DIRECT = false>
__device__ __forceinline__ void wall_finish_cell(const WmArgs& a, int64_t c, const double y1v[3], const double vs[3],
                                                 const double vw[3], const WmDirect* o = nullptr, int e = 0) {
  const int64_t n = a.dm.n, nx = a.dm.nx, nxy = (int64_t)a.dm.nx * a.dm.ny;
  {
    int x = (int)(c % nx), y = (int)((c / nx) % a.dm.ny), z = (int)(c / nxy);
    double y1 = sqrt(y1v[0] * y1v[0] + y1v[1] * y1v[1] + y1v[2] * y1v[2]);
    double nrm[3] = {y1v[0] / y1, y1v[1] / y1, y1v[2] / y1};
    double us[3];
    uint8_t fl = a.flags[c];
    body_velocity_d(a.bo, (fl >> TAG_SHIFT) & TAG_MASK, x, y, z, us);
    double r[3], rn = 0.0;
    for (int q = 0; q < 3; ++q) {
      r[q] = vs[q] - us[q];
      rn += r[q] * nrm[q];
    }
    double ut[3], U = 0.0;
    for (int q = 0; q < 3; ++q) {
      ut[q] = r[q] - rn * nrm[q];
      U += ut[q] * ut[q];
    }
    U = sqrt(U);
    double utau = 0.0;
    double uw[3] = {0, 0, 0}, sw[6] = {0, 0, 0, 0, 0, 0};
    if (!(U < 1e-14)) {
      double yy = y1 + a.hs;
      double prev;
      bool have_prev;
      if (DIRECT) {
        prev = o->start ? o->start[e] : 0.0;
        have_prev = true;
      } else {
        prev = a.wm_utau[c];
        have_prev = (fl & WM_VALID) != 0;
      }
      double ua = (have_prev && prev > 0.0) ? prev : sqrt(a.nu * U / yy);  // Eq. 20
      // Newton-Raphson (Eq. 19), stop rule of PAPER.md:184
      double fa = wall_f(a.wall_function, ua, U, yy, a.nu, a.kappa, a.E), ub = ua;
      for (int it = 0; it < a.max_iter; ++it) {
        ub = ua - fa / wall_df(a.wall_function, ua, U, yy, a.nu, a.kappa, a.E);
        if (!(ub > 0.0)) ub = 0.5 * ua;
        double fb = wall_f(a.wall_function, ub, U, yy, a.nu, a.kappa, a.E);
        double df = fabs(fb - fa);
        ua = ub;
        fa = fb;
        if (df < a.tol) break;
      }
      utau = ub;
      double upl = 1.0;  // R8: the friction velocity itself; R22: the wall-function velocity at y1
      if (a.wm_slip == 1) {
        double yp1 = y1 * utau / a.nu;
        upl = a.wall_function == 1 ? musker_uplus(yp1) : spalding_uplus(yp1, a.kappa, a.E);
      }
      for (int q = 0; q < 3; ++q) uw[q] = utau * upl * ut[q] / U;
      double G[3][3];
      if (a.wm_shear == 1) {  // R22
        double dudy = wall_shear(a.wall_function, utau, U, yy, a.nu, a.kappa, a.E);
        for (int p = 0; p < 3; ++p)
          for (int q = 0; q < 3; ++q) G[p][q] = dudy * (ut[p] / U) * nrm[q];
      } else {
        for (int p = 0; p < 3; ++p)
          for (int q = 0; q < 3; ++q) G[p][q] = (vs[p] - vw[p]) * nrm[q] / a.hs;  // R10
      }
      sw[0] = G[0][0];
      sw[1] = G[1][1];
      sw[2] = G[2][2];
      sw[3] = 0.5 * (G[0][1] + G[1][0]);
      sw[4] = 0.5 * (G[0][2] + G[2][0]);
      sw[5] = 0.5 * (G[1][2] + G[2][1]);
    }
    if (DIRECT) {
      o->utau[e] = utau;
      for (int q = 0; q < 3; ++q) o->u[3 * (int64_t)e + q] = (float)uw[q];
      for (int q = 0; q < 6; ++q) o->s[6 * (int64_t)e + q] = (float)sw[q];
      return;
    }
    a.wm_utau[c] = utau;
    for (int q = 0; q < 3; ++q) a.wm_u[(int64_t)q * n + c] = (float)uw[q];
    for (int q = 0; q < 6; ++q) a.wm_s[(int64_t)q * n + c] = (float)sw[q];
    a.flags[c] = fl | WM_VALID;
  }
}

template <int WM_BATCH, int BLOCKS_PER_SM>
__global__ void __launch_bounds__(128, BLOCKS_PER_SM) wall_sample_kernel(const __grid_constant__ WmArgs a) {
  const int count = min(a.cnt->wall_count, a.cap_list);
  const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
  const int nw = gridDim.x * wpb;
  for (int base = (blockIdx.x * wpb + (threadIdx.x >> 5)) * WM_BATCH; base < count; base += nw * WM_BATCH) {
    // lanes 0..WM_BATCH-1 hold the list entries of the batch
    const int e_l = base + lane;
    const bool mine = lane < WM_BATCH && e_l < count;
    int c_l = 0;
    double y_l[3] = {1.0, 0.0, 0.0};
    if (mine) {
      c_l = a.wall_idx[e_l];
#pragma unroll
      for (int q = 0; q < 3; ++q) y_l[q] = a.wall_y1n[3 * (int64_t)e_l + q];
    }
    const SamplePoint mine_p = sample_point(a, c_l, y_l);  // lanes >= WM_BATCH: a dummy cell, never used
    SampleLane sl[WM_BATCH];
#pragma unroll
    for (int j = 0; j < WM_BATCH; ++j) {  // a batch's tail repeats its last cell (never out of range, no branch)
      const int src = min(j, count - 1 - base);
      wall_sample_issue(a, shfl_point(mine_p, src), lane, sl[j]);
    }
    double my_vs[3] = {0, 0, 0}, my_vw[3] = {0, 0, 0};
#pragma unroll
    for (int j = 0; j < WM_BATCH; ++j) {
      double vs[3], vw[3];
      wall_sample_reduce(a, sl[j], lane, vs, vw);  // vs valid on lane 0, vw on every lane
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const double s0 = shfl_d(vs[q], 0);
        if (lane == j) {
          my_vs[q] = s0;
          my_vw[q] = vw[q];
        }
      }
    }
    if (mine) {
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        a.samp[6 * (int64_t)e_l + q] = my_vs[q];
        a.samp[6 * (int64_t)e_l + 3 + q] = my_vw[q];
      }
    }
  }
}

__global__ void __launch_bounds__(128) wall_model_kernel(const __grid_constant__ WmArgs a) {
  const int count = min(a.cnt->wall_count, a.cap_list);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
    const int64_t c = a.wall_idx[e];
    double y1v[3], vs[3], vw[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      y1v[q] = a.wall_y1n[3 * (int64_t)e + q];
      vs[q] = a.samp[6 * (int64_t)e + q];
      vw[q] = a.samp[6 * (int64_t)e + 3 + q];
    }
    wall_finish_cell(a, c, y1v, vs, vw);
  }
}

// ---------------------------------------------------------------------------- K4 forces
struct ForceArgs {
  Dom dm;
  BodiesD bo;
  const float* f;
  const uint8_t* flags;
  const int32_t* force_idx;
  const Counters* cnt;
  int cap_list;
  double* out;    // [MAX_TAGS][3] of this step (zeroed by the kernel launched before)
  double* out_m;  // [MAX_TAGS][3]: torque of the same per-cell forces about the body centre
};

__global__ void zero_force_kernel(double* out, double* out_m) {
  if (threadIdx.x < MAX_TAGS * 3) out[threadIdx.x] = out_m[threadIdx.x] = 0.0;
}

// F_k = - sum_{x: d<1, tag=k} sum_{i != rest} [(c_i - u^s) f_i(x + c_i) + (c_i + u^s) f_ibar(x)]
// (Eq. 23 with reading R7), fp64 accumulation.  One LANE per cell, a warp takes 32 consecutive list entries:
// geometry pass 2 appends a warp's cells in x order, so the entries are runs of x-neighbours and each of the
// 52 loads of the warp touches a few sectors instead of 32.  Warp shuffle sum (when the 32 cells belong to one
// element, the usual case; per-lane atomics otherwise) -> shared per-tag bins -> one global atomic per block,
// tag and component.  The torque M_k = sum_x (x - x_c) x F(x) about the centre of the element's rigid body
// takes the same path through a second set of bins.
__device__ __forceinline__ void force_block(const ForceArgs& a, int block, int nblocks) {
  __shared__ double bins[MAX_TAGS * 3];
  __shared__ double bins_m[MAX_TAGS * 3];
  for (int t = threadIdx.x; t < MAX_TAGS * 3; t += blockDim.x) bins[t] = bins_m[t] = 0.0;
  __syncthreads();
  const int count = min(a.cnt->force_count, a.cap_list);
  const int64_t nx = a.dm.nx, nxy = (int64_t)a.dm.nx * a.dm.ny;
  const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
  for (int base = (block * wpb + (threadIdx.x >> 5)) * 32; base < count; base += nblocks * wpb * 32) {
    const int e = base + lane;
    const bool act = e < count;
    int k = -1;
    double v[6] = {0, 0, 0, 0, 0, 0};  // force, torque of this lane's cell
    if (act) {
      const int64_t c = a.force_idx[e];
      const int x = (int)(c % nx), y = (int)((c / nx) % a.dm.ny), z = (int)(c / nxy);
      k = (a.flags[c] >> TAG_SHIFT) & TAG_MASK;
      double us[3];
      body_velocity_d(a.bo, k, x, y, z, us);
      double acc[3] = {0, 0, 0};
#pragma unroll 1
      for (int pz = 0; pz < 3; ++pz) {  // one z-plane of links at a time keeps the kernel at 8 blocks per SM
        const int cz = pz - 1;
        bool flx, fly, flz;
        const int zz = wrap_far(z + cz, a.dm.nz, a.dm.mode[2], flz);
#pragma unroll
        for (int j = 0; j < 9; ++j) {
          const int cx = j % 3 - 1, cy = j / 3 - 1;
          if ((Q == 19 && cx * cy * cz != 0) || (cx == 0 && cy == 0 && cz == 0)) continue;  // not in the set / rest
          const int i = dir_index(cx, cy, cz);
          const int xx = wrap_far(x + cx, a.dm.nx, a.dm.mode[0], flx);
          const int yy = wrap_far(y + cy, a.dm.ny, a.dm.mode[1], fly);
          // R12: the cell behind a MIRROR plane is the reflected image of the lattice -- f_i there is the population
          // of the reflected cell with the normal velocity component reversed (what push_store does to a
          // population that leaves through the plane)
          const int ir = dir_index(flx ? -cx : cx, fly ? -cy : cy, flz ? -cz : cz);
          // stored values are deviations: f = w + dev, and w_i = w_ibar = w of the reflected direction
          const double w = dir_wd_of(cx, cy, cz);
          const double fa = w + (double)__ldg(a.f + pop_index_cx(a.dm, ir, flx ? -cx : cx, xx, yy, zz));
          const double fb = w + (double)__ldg(a.f + pop_index_cx(a.dm, dir_opp(i), -cx, x, y, z));
          const double ci[3] = {(double)cx, (double)cy, (double)cz};
#pragma unroll
          for (int q = 0; q < 3; ++q) acc[q] += (ci[q] - us[q]) * fa + (ci[q] + us[q]) * fb;
        }
      }
      const double r0 = x - a.bo.c[k][0], r1 = y - a.bo.c[k][1], r2 = z - a.bo.c[k][2];
      v[0] = -acc[0];
      v[1] = -acc[1];
      v[2] = -acc[2];
      v[3] = r1 * v[2] - r2 * v[1];
      v[4] = r2 * v[0] - r0 * v[2];
      v[5] = r0 * v[1] - r1 * v[0];
    }
    const int k0 = __shfl_sync(0xffffffffu, k, 0);  // lane 0 is active whenever the warp is here
    if (__all_sync(0xffffffffu, !act || k == k0)) {
#pragma unroll
      for (int off = 16; off > 0; off >>= 1)
#pragma unroll
        for (int q = 0; q < 6; ++q) v[q] += __shfl_down_sync(0xffffffffu, v[q], off);
      if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          atomicAdd(&bins[k0 * 3 + q], v[q]);
          atomicAdd(&bins_m[k0 * 3 + q], v[3 + q]);
        }
      }
    } else if (act) {
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        atomicAdd(&bins[k * 3 + q], v[q]);
        atomicAdd(&bins_m[k * 3 + q], v[3 + q]);
      }
    }
  }
  __syncthreads();
  for (int t = threadIdx.x; t < MAX_TAGS * 3; t += blockDim.x) {
    if (bins[t] != 0.0) atomicAdd(&a.out[t], bins[t]);
    if (bins_m[t] != 0.0) atomicAdd(&a.out_m[t], bins_m[t]);
  }
}

// 64 threads x 64 registers: fits beside a resident block of the collide-stream kernel (see geometry.cu: geo_grid)
__global__ void __launch_bounds__(64, 16) force_kernel(const __grid_constant__ ForceArgs f) {
  force_block(f, blockIdx.x, gridDim.x);
}

// ---------------------------------------------------------------------------- launchers
static void fill_bodies(const hhrr_lattice* L, BodiesD& b) { b = L->bodies; }

static void fill_wm(const hhrr_lattice* L, WmArgs& a) {
  a.dm = L->dom;
  for (int q = 0; q < 3; ++q) a.g[q] = L->p.body_force[q];
  a.nu = (L->p.tau0 - 0.5) / 3.0;
  a.kappa = L->p.kappa;
  a.E = L->p.E;
  a.tol = L->p.newton_tol;
  a.hs = L->p.sampling_distance;
  a.max_iter = L->p.newton_max_iter;
  a.wall_function = L->wall_function;
  a.wm_slip = L->wm_slip;
  a.wm_shear = L->wm_shear;
  fill_bodies(L, a.bo);
  a.f = L->fA;
  a.flags = L->flags;
  a.wall_idx = L->wall_idx;
  a.wall_y1n = L->wall_y1n;
  a.cnt = L->counters;
  a.cap_list = (int)L->cap_list;
  a.samp = L->wall_samp;
  a.wm_utau = L->wm_utau;
  a.wm_u = L->wm_u;
  a.wm_s = L->wm_s;
}

// The next step's geometry was written ahead into the alternate set with WM_VALID clear (geometry.cu).  Its collision
// consumes the wall-model state of a cell iff the cell is in W there AND holds state now, i.e. was in W of this step
// (O1: the state of cells that leave W is dropped): one pass over the alternate wall list after the wall model.
__global__ void merge_valid_kernel(const int32_t* __restrict__ alt_wall_idx, const Counters* alt_cnt, int cap,
                                   const uint8_t* __restrict__ flags, uint8_t* __restrict__ alt_flags) {
  const int count = min(alt_cnt->wall_count, cap);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
    const int64_t c = alt_wall_idx[e];
    if (flags[c] & WM_VALID) alt_flags[c] |= WM_VALID;
  }
}

// Listing 3 line 4: WallModelO
cudaError_t launch_wall_model(hhrr_lattice* L) {
  if (!L->wm_enabled) return cudaSuccess;
  WmArgs w;
  fill_wm(L, w);
  // two cells per warp and sweep, 8 blocks per SM (64 registers); measured against 1, 4 and 8 cells per warp
  wall_sample_kernel<2, 8><<<4736, 128, 0, L->stream>>>(w);
  wall_model_kernel<<<592, 128, 0, L->stream>>>(w);
  L->launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_merge_valid(hhrr_lattice* L) {
  merge_valid_kernel<<<148, 256, 0, L->stream>>>(L->alt_wall_idx, L->alt_counters, (int)L->cap_list, L->flags, L->alt_flags);
  L->launches++;
  return cudaGetLastError();
}

// Listing 3 lines 5-6: force collection and per-element integration into the ring slot of
// this step.  Reads the streamed populations, the flag bytes (tags) and the force list of the current geometry.
cudaError_t launch_forces(hhrr_lattice* L, cudaStream_t s) {
  ForceArgs a;
  a.dm = L->dom;
  fill_bodies(L, a.bo);
  a.f = L->fA;
  a.flags = L->flags;
  a.force_idx = L->force_idx;
  a.cnt = L->counters;
  a.cap_list = (int)L->cap_list;
  a.out = L->force + (L->step % FORCE_HISTORY) * MAX_TAGS * 3;
  a.out_m = L->torque + (L->step % FORCE_HISTORY) * MAX_TAGS * 3;
  zero_force_kernel<<<1, 64, 0, s>>>(a.out, a.out_m);
  force_kernel<<<4736, 64, 0, s>>>(a);
  L->launches += 2;
  return cudaGetLastError();
}

}  // namespace hhrr

// ---------------------------------------------------------------------------- allocation-free wall model
// hhrr_wall_model_noalloc (include/hhrr.h): WallModelO (K3) on the lattice's current populations and wall list for
// callers that may not allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  K3 is two kernels with scratch between them (v_s and v(x_w) per wall cell, 48 B); the regular path keeps
// that scratch in the caller's workspace, this one in the file-scope array below: HHRR_NOALLOC_MAX_WALL_CELLS cells x 6
// doubles = 3 MiB, held by every GPU that loads the library until the process exits.
//   * The array's NAME is a host-side stand-in in host code, not a device address: its address on a device comes from
//     cudaGetSymbolAddress, asked once per device with that device current (scratch_address below).
//   * All calls share the array.  The sampling kernel overwrites entries [0, count) before the Newton kernel reads
//     them and nothing reads beyond: no entry has to start at zero, a shorter list after a longer one reads nothing
//     stale.  Two calls that OVERLAP on the GPU (different streams, or lattices on different streams of one device) race
//     on it; calls on one stream, or on different devices, do not.
//   * No cudaMalloc / cudaFree / allocating library routine on this path: two kernel launches on the lattice's stream.
namespace hhrr {

static __device__ __align__(256) double g_noalloc_scratch[(size_t)HHRR_NOALLOC_MAX_WALL_CELLS * 6];

constexpr int MAX_DEVICES = 64;
static double* g_noalloc_ptr[MAX_DEVICES] = {};

// device address of the scratch array on the CURRENT device (the caller has made `device` current)
static cudaError_t scratch_address(int device, double** out) {
  if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
  if (!g_noalloc_ptr[device]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[device] = p;  // benign if two threads get here together: both write the same address
  }
  *out = g_noalloc_ptr[device];
  return cudaSuccess;
}

// Newton kernel of the allocation-free path: one thread per list entry, outputs per entry into the caller's arrays
__global__ void __launch_bounds__(128) wall_model_direct_kernel(const __grid_constant__ WmArgs a,
                                                                const __grid_constant__ WmDirect o) {
  const int count = min(a.cnt->wall_count, a.cap_list);
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
    const int64_t c = a.wall_idx[e];
    double y1v[3], vs[3], vw[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      y1v[q] = a.wall_y1n[3 * (int64_t)e + q];
      vs[q] = a.samp[6 * (int64_t)e + q];
      vw[q] = a.samp[6 * (int64_t)e + 3 + q];
    }
    wall_finish_cell<true>(a, c, y1v, vs, vw, &o, e);
  }
}

}  // namespace hhrr

extern "C" int hhrr_wall_model_noalloc(hhrr_lattice* L, int64_t capacity, const double* d_u_tau_start, double* d_u_tau,
                                       float* d_u_wm, float* d_s_wm) {
  using namespace hhrr;
  if (!L || !d_u_tau || !d_u_wm || !d_s_wm || capacity < 1)
    return set_error(HHRR_E_ARG, "hhrr_wall_model_noalloc: NULL output array or capacity < 1");
  if (capacity > HHRR_NOALLOC_MAX_WALL_CELLS)
    return set_error(HHRR_E_SIZE, "hhrr_wall_model_noalloc: capacity %lld exceeds the built-in scratch of %d wall cells "
                     "(HHRR_NOALLOC_MAX_WALL_CELLS); use hhrr_step, whose scratch lives in the caller's workspace",
                     (long long)capacity, (int)HHRR_NOALLOC_MAX_WALL_CELLS);
  int prev = -1;  // work on the lattice's device, leave the caller's current device as it was
  if (cudaGetDevice(&prev) != cudaSuccess) return set_error(HHRR_E_CUDA, "hhrr_wall_model_noalloc: no CUDA device");
  if (prev != L->device && cudaSetDevice(L->device) != cudaSuccess)
    return set_error(HHRR_E_CUDA, "hhrr_wall_model_noalloc: cannot select device %d", L->device);
  int rc = HHRR_OK;
  double* scratch = nullptr;
  cudaError_t e = scratch_address(L->device, &scratch);
  if (e != cudaSuccess) {
    rc = set_error(HHRR_E_CUDA, "hhrr_wall_model_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  } else {
    WmArgs w;
    fill_wm(L, w);
    w.samp = scratch;                                             // instead of the workspace's wall_samp
    w.cap_list = (int)std::min<int64_t>(w.cap_list, capacity);  // entries [0, min(wall count, capacity))
    WmDirect o{d_u_tau_start, d_u_tau, d_u_wm, d_s_wm};
    wall_sample_kernel<2, 8><<<4736, 128, 0, L->stream>>>(w);
    wall_model_direct_kernel<<<592, 128, 0, L->stream>>>(w, o);
    L->launches += 2;
    e = cudaGetLastError();
    if (e != cudaSuccess) rc = set_error(HHRR_E_CUDA, "hhrr_wall_model_noalloc: launch: %s", cudaGetErrorString(e));
  }
  if (prev != L->device) cudaSetDevice(prev);
  return rc;
}
