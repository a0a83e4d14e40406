// collide.cu -- K2: collide & stream (Listing 3 line 3; Eq. 6-14), plus
// initialisation and moment read-back.  Populations are stored post-stream (the state the
// paper's operators see) as deviations f_i - w_i in 27 SoA planes; a step reads buffer A at
// the own cell and pushes the post-collision values into buffer B.
//
// Variant 0 (two-pass): moments_kernel writes the time-n homogenised velocity field,
//   collide_kernel differentiates it (S^FD, Eq. 10 "non-local") and collides.
// Variant 1 (fused): see fused.cu.
#include "cell_model.cuh"

namespace hhrr {

struct CellCtx {
  const uint8_t* flags;
  const float* d;
  const float* wm_u;
  const float* wm_s;
};

__device__ __forceinline__ void load_cell(const float* __restrict__ f, int64_t n, int64_t c, float (&v)[Q]) {
#pragma unroll
  for (int i = 0; i < Q; ++i) v[i] = __ldg(f + (int64_t)i * n + c);
}

// porosity and u^B (+ wall-model slip, R8) of a cell
__device__ __forceinline__ void cell_solid_state(const PhysF& ph, const BodiesF& bo, uint8_t fl,
                                                 const float* __restrict__ dfield,
                                                 const float* __restrict__ wm_u, int64_t n, int64_t c, int x,
                                                 int y, int z, float& d, float uB[3]) {
  int type = fl & TYPE_MASK;
  d = 1.f;
  uB[0] = uB[1] = uB[2] = 0.f;
  if (type_has_solid_state(type)) {
    d = type_is_frontier(type) ? __ldg(dfield + c) : 0.f;
    solid_velocity(ph, bo, fl, x, y, z, uB);
    if (fl & WM_VALID) {
      uB[0] += __ldg(wm_u + c);
      uB[1] += __ldg(wm_u + n + c);
      uB[2] += __ldg(wm_u + 2 * n + c);
    }
  }
}

// ------------------------------------------------------------------ variant 0, pass 1
__global__ void __launch_bounds__(256) moments_kernel(Dom dm, PhysF ph, BodiesF bo,
                                                      const float* __restrict__ fin,
                                                      const uint8_t* __restrict__ flags,
                                                      const float* __restrict__ dfield,
                                                      const float* __restrict__ wm_u, float* __restrict__ uhat) {
  int x = blockIdx.x * blockDim.x + threadIdx.x;
  int y = blockIdx.y, z = blockIdx.z;
  if (x >= dm.nx) return;
  int64_t c = (int64_t)x + (int64_t)dm.nx * ((int64_t)y + (int64_t)dm.ny * z);
  float f[Q];
  load_cell(fin, dm.n, c, f);
  float drho, jx, jy, jz;
  moments_rho_j(f, drho, jx, jy, jz);
  uint8_t fl = flags[c];
  float d, uB[3], rho, uh[3];
  cell_solid_state(ph, bo, fl, dfield, wm_u, dm.n, c, x, y, z, d, uB);
  homogenised_velocity(ph, drho, jx, jy, jz, d, uB, rho, uh);
  uhat[c] = uh[0];
  uhat[dm.n + c] = uh[1];
  uhat[2 * dm.n + c] = uh[2];
}

// ------------------------------------------------------------------ variant 0, pass 2
__global__ void __launch_bounds__(256) collide_kernel(Dom dm, PhysF ph, BodiesF bo,
                                                      const float* __restrict__ fin, float* __restrict__ fout,
                                                      const uint8_t* __restrict__ flags,
                                                      const float* __restrict__ dfield,
                                                      const float* __restrict__ wm_u,
                                                      const float* __restrict__ wm_s,
                                                      const float* __restrict__ uhat) {
  int x = blockIdx.x * blockDim.x + threadIdx.x;
  int y = blockIdx.y, z = blockIdx.z;
  if (x >= dm.nx) return;
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  int64_t c = x + nx * y + nxy * z;
  float f[Q];
  load_cell(fin, n, c, f);
  Moments m = moments_all(f);
  uint8_t fl = flags[c];
  float d, uB[3], rho, uh[3];
  cell_solid_state(ph, bo, fl, dfield, wm_u, n, c, x, y, z, d, uB);
  homogenised_velocity(ph, m.drho, m.jx, m.jy, m.jz, d, uB, rho, uh);
  float S[6], sigma = cell_sigma(ph, fl);
  if (fl & WM_VALID) {  // sigma = 0, strain from the wall model
#pragma unroll
    for (int a = 0; a < 6; ++a) S[a] = __ldg(wm_s + (int64_t)a * n + c);
    sigma = 0.f;
  } else {  // S^FD: central differences of the time-n uhat field (R5)
    bool fm, fp;
    int xm = wrap_axis(x - 1, dm.nx, dm.mode[0], fm), xp = wrap_axis(x + 1, dm.nx, dm.mode[0], fp);
    int64_t cm = xm + nx * y + nxy * z, cp = xp + nx * y + nxy * z;
    float sm = fm ? -1.f : 1.f, sp = fp ? -1.f : 1.f;
    float dxu0 = sp * uhat[cp] - sm * uhat[cm];
    float dxu1 = uhat[n + cp] - uhat[n + cm];
    float dxu2 = uhat[2 * n + cp] - uhat[2 * n + cm];
    int ym = wrap_axis(y - 1, dm.ny, dm.mode[1], fm), yp = wrap_axis(y + 1, dm.ny, dm.mode[1], fp);
    cm = x + nx * ym + nxy * z, cp = x + nx * yp + nxy * z;
    sm = fm ? -1.f : 1.f, sp = fp ? -1.f : 1.f;
    float dyu0 = uhat[cp] - uhat[cm];
    float dyu1 = sp * uhat[n + cp] - sm * uhat[n + cm];
    float dyu2 = uhat[2 * n + cp] - uhat[2 * n + cm];
    int zm = wrap_axis(z - 1, dm.nz, dm.mode[2], fm), zp = wrap_axis(z + 1, dm.nz, dm.mode[2], fp);
    cm = x + nx * y + nxy * zm, cp = x + nx * y + nxy * zp;
    sm = fm ? -1.f : 1.f, sp = fp ? -1.f : 1.f;
    float dzu0 = uhat[cp] - uhat[cm];
    float dzu1 = uhat[n + cp] - uhat[n + cm];
    float dzu2 = sp * uhat[2 * n + cp] - sm * uhat[2 * n + cm];
    S[0] = 0.5f * dxu0;
    S[1] = 0.5f * dyu1;
    S[2] = 0.5f * dzu2;
    S[3] = 0.25f * (dyu0 + dxu1);
    S[4] = 0.25f * (dzu0 + dxu2);
    S[5] = 0.25f * (dzu1 + dyu2);
  }
  float o[Q];
  collide(ph, m, rho, uh, S, sigma, o);
  push_store(dm, fout, x, y, z, o);
}

// ------------------------------------------------------------------ initialisation
__global__ void fill_kernel(float* __restrict__ p, int64_t count, float v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (; i < count; i += stride) p[i] = v;
}

// f = f_eq(rho,u) [+ regularised f^(1) with a2 = -2 rho cs^2 tau0 S^FD(u)], evaluated in
// fp64 and stored as fp32 deviations (one-time, not on the hot path).
__global__ void init_kernel(Dom dm, double tau0, const float* __restrict__ rho_in,
                            const float* __restrict__ u_in, int with_neq, float* __restrict__ f) {
  int x = blockIdx.x * blockDim.x + threadIdx.x;
  int y = blockIdx.y, z = blockIdx.z;
  if (x >= dm.nx) return;
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  int64_t c = x + nx * y + nxy * z;
  double rho = rho_in[c], u[3] = {u_in[c], u_in[n + c], u_in[2 * n + c]};
  double a2[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
  if (with_neq) {
    int coord[3] = {x, y, z}, ext[3] = {dm.nx, dm.ny, dm.nz};
    double G[3][3];  // G[a][b] = d_b u_a
    for (int b = 0; b < 3; ++b) {
      bool fm, fp;
      int q[3] = {x, y, z};
      q[b] = wrap_axis(coord[b] - 1, ext[b], dm.mode[b], fm);
      int64_t cm = q[0] + nx * q[1] + nxy * q[2];
      q[b] = wrap_axis(coord[b] + 1, ext[b], dm.mode[b], fp);
      int64_t cp = q[0] + nx * q[1] + nxy * q[2];
      for (int a = 0; a < 3; ++a) {
        double up = u_in[(int64_t)a * n + cp], um = u_in[(int64_t)a * n + cm];
        if (a == b) {
          if (fp) up = -up;
          if (fm) um = -um;
        }
        G[a][b] = 0.5 * (up - um);
      }
    }
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) a2[a][b] = -2.0 * rho * (1.0 / 3.0) * tau0 * 0.5 * (G[a][b] + G[b][a]);
  }
  double A3[3][3][3];  // a0^(3) + a1^(3): rho u u u and the recursion of R3 on a2
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      for (int g = 0; g < 3; ++g)
        A3[a][b][g] = rho * u[a] * u[b] * u[g] + (u[a] * a2[b][g] + u[b] * a2[a][g] + u[g] * a2[a][b]);
  for (int i = 0; i < Q; ++i) {
    double cv[3] = {(double)dir_cx(i), (double)dir_cy(i), (double)dir_cz(i)};
    auto h3 = [&](int a, int b, int g) {
      return cv[a] * cv[b] * cv[g] - (1.0 / 3.0) * (cv[a] * (b == g) + cv[b] * (a == g) + cv[g] * (a == b));
    };
    double t1 = 0, t2 = 0, t3 = 0;
    for (int a = 0; a < 3; ++a) t1 += cv[a] * rho * u[a];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        double h2 = cv[a] * cv[b] - (a == b ? 1.0 / 3.0 : 0.0);
        t2 += h2 * (rho * u[a] * u[b] + a2[a][b]);
      }
    if (Q == 27) {  // full contraction / (3! cs^6) = 4.5 sum (R3)
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
          for (int g = 0; g < 3; ++g) t3 += 4.5 * h3(a, b, g) * A3[a][b][g];
    } else {  // D3Q19: basis of the paper's ref. [43] (R23): sums / (2 cs^6), differences / (6 cs^6)
      const int G1[3][3] = {{0, 0, 1}, {0, 2, 2}, {1, 1, 2}}, G2[3][3] = {{1, 2, 2}, {0, 1, 1}, {0, 0, 2}};
      for (int k = 0; k < 3; ++k) {
        double h1 = h3(G1[k][0], G1[k][1], G1[k][2]), h2 = h3(G2[k][0], G2[k][1], G2[k][2]);
        double a1 = A3[G1[k][0]][G1[k][1]][G1[k][2]], a2_ = A3[G2[k][0]][G2[k][1]][G2[k][2]];
        t3 += 13.5 * (h1 + h2) * (a1 + a2_) + 4.5 * (h1 - h2) * (a1 - a2_);
      }
    }
    double w = dir_wd(i);
    double dev = w * ((rho - 1.0) + 3.0 * t1 + 4.5 * t2 + t3);
    f[(int64_t)i * n + c] = (float)dev;
  }
}

// rho and v = (j + g/2)/rho of the stored populations (R11)
__global__ void __launch_bounds__(256) readback_kernel(Dom dm, PhysF ph, const float* __restrict__ fin,
                                                       float* __restrict__ rho_out, float* __restrict__ v_out) {
  int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= dm.n) return;
  const int x = (int)(c % dm.nx), y = (int)((c / dm.nx) % dm.ny), z = (int)(c / ((int64_t)dm.nx * dm.ny));
  float f[Q];
#pragma unroll
  for (int i = 0; i < Q; ++i) f[i] = __ldg(fin + pop_index(dm, i, x, y, z));
  double drho = 0, j[3] = {0, 0, 0};
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    drho += (double)f[i];
    j[0] += dir_cx(i) * (double)f[i];
    j[1] += dir_cy(i) * (double)f[i];
    j[2] += dir_cz(i) * (double)f[i];
  }
  double rho = 1.0 + drho;
  rho_out[c] = (float)rho;
  for (int a = 0; a < 3; ++a) v_out[(int64_t)a * dm.n + c] = (float)((j[a] + 0.5 * (double)ph.g[a]) / rho);
}

// re-store the populations with another x-shift: dst (storage xs_to) from src (storage dm.xs)
__global__ void __launch_bounds__(256) restore_kernel(Dom dm, int xs_to, const float* __restrict__ src,
                                                      float* __restrict__ dst) {
  int x = blockIdx.x * blockDim.x + threadIdx.x;
  int y = blockIdx.y, z = blockIdx.z;
  if (x >= dm.nx) return;
  Dom to = dm;
  to.xs = xs_to;
  // population i of the post-stream state of cell (x,y,z): read where dm keeps it, write where `to` keeps it
#pragma unroll
  for (int i = 0; i < Q; ++i) dst[pop_index(to, i, x, y, z)] = src[pop_index(dm, i, x, y, z)];
}

__global__ void finite_kernel(const float* __restrict__ f, int64_t count, Counters* cnt) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int bad = 0;
  for (; i < count; i += stride) bad |= !isfinite(f[i]);
  if (bad) cnt->nonfinite = 1;
}

// ------------------------------------------------------------------ launchers
PhysF make_phys(const hhrr_lattice* L) {
  PhysF ph;
  ph.tau0 = (float)L->p.tau0;
  ph.sigma = (float)L->p.sigma;
  ph.smag18 = (float)(18.0 * L->p.smagorinsky_cs * L->p.smagorinsky_cs);
  for (int a = 0; a < 3; ++a) {
    ph.g[a] = (float)L->p.body_force[a];
    ph.fr_u[a] = (float)L->fr_u[a];
  }
  return ph;
}
BodiesF make_bodies(const hhrr_lattice* L) {
  BodiesF b;
  for (int k = 0; k < MAX_TAGS; ++k)
    for (int a = 0; a < 3; ++a) {
      b.c[k][a] = (float)L->bodies.c[k][a];
      b.w[k][a] = (float)L->bodies.w[k][a];
      b.v[k][a] = (float)L->bodies.v[k][a];
    }
  return b;
}

static dim3 row_grid(const Dom& dm, int bx) { return dim3((dm.nx + bx - 1) / bx, dm.ny, dm.nz); }
static int row_block(const Dom& dm) { return dm.nx >= 256 ? 256 : (dm.nx >= 128 ? 128 : (dm.nx > 32 ? 64 : 32)); }

cudaError_t launch_fill_rest(hhrr_lattice* L) {
  fill_kernel<<<1184, 256, 0, L->stream>>>(L->fA, (int64_t)Q * L->dom.n, 0.f);
  L->launches++;
  return cudaGetLastError();
}

cudaError_t launch_init(hhrr_lattice* L, const float* d_rho, const float* d_u, int with_neq) {
  int bx = row_block(L->dom);
  init_kernel<<<row_grid(L->dom, bx), bx, 0, L->stream>>>(L->dom, L->p.tau0, d_rho, d_u, with_neq, L->fA);
  L->launches++;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess && L->dom.xs) {  // init_kernel writes the plain post-stream layout
    const int xs = L->dom.xs;
    L->dom.xs = 0;
    e = launch_restore(L, xs);
  }
  return e;
}

// buffer A: from storage dom.xs to storage xs (through buffer B, which is free between steps)
cudaError_t launch_restore(hhrr_lattice* L, int xs) {
  if (xs == L->dom.xs) return cudaSuccess;
  int bx = row_block(L->dom);
  restore_kernel<<<row_grid(L->dom, bx), bx, 0, L->stream>>>(L->dom, xs, L->fA, L->fB);
  L->launches++;
  float* t = L->fA;
  L->fA = L->fB;
  L->fB = t;
  L->dom.xs = xs;
  return cudaGetLastError();
}

cudaError_t launch_fused_ws(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo);  // fused_ws.cu
cudaError_t launch_fused_xpull(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo); // fused_xpull.cu

// Variant 5 (default) runs where its storage is in place (dom.xs, decided by hhrr_create /
// hhrr_set_kernel_variant from xpull_supported); a lattice it cannot tile keeps post-stream storage and runs
// variant 2 -- hhrr_set_kernel_variant reports that with HHRR_W_FALLBACK, hhrr_population_storage shows it.
cudaError_t launch_collide_stream(hhrr_lattice* L) {
  PhysF ph = make_phys(L);
  BodiesF bo = make_bodies(L);
  cudaError_t e;
  if (L->variant == 5 && L->dom.xs) {
    e = launch_fused_xpull(L, ph, bo);
  } else if (L->variant >= 2) {
    e = launch_fused_ws(L, ph, bo);
  } else {
    int bx = row_block(L->dom);
    dim3 g = row_grid(L->dom, bx);
    moments_kernel<<<g, bx, 0, L->stream>>>(L->dom, ph, bo, L->fA, L->flags, L->d, L->wm_u, L->uhat);
    collide_kernel<<<g, bx, 0, L->stream>>>(L->dom, ph, bo, L->fA, L->fB, L->flags, L->d, L->wm_u, L->wm_s,
                                            L->uhat);
    L->launches += 2;
    e = cudaGetLastError();
  }
  float* t = L->fA;
  L->fA = L->fB;
  L->fB = t;
  return e;
}

cudaError_t launch_moments(hhrr_lattice* L, float* d_rho, float* d_v) {
  PhysF ph = make_phys(L);
  int64_t blocks = (L->dom.n + 255) / 256;
  readback_kernel<<<(unsigned)blocks, 256, 0, L->stream>>>(L->dom, ph, L->fA, d_rho, d_v);
  L->launches++;
  return cudaGetLastError();
}

cudaError_t launch_check_finite(hhrr_lattice* L) {
  finite_kernel<<<1184, 256, 0, L->stream>>>(L->fA, (int64_t)Q * L->dom.n, L->counters);
  L->launches++;
  return cudaGetLastError();
}

}  // namespace hhrr
