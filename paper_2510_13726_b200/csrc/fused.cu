// fused.cu -- variant 1 of K2: ONE kernel for moments + HLBM shift + FD strain + Smagorinsky +
// hybrid recursive regularisation + collision + streaming (Listing 3 line 3, PAPER.md:313;
// Eq. 6-14).
//
// The only non-local input of the collision is S^FD, the central difference of the time-n
// homogenised velocity of the six face neighbours (Eq. 10, "non-local" PAPER.md:109).  A block
// owns a TX x TY column of cells and marches along z.  Per plane every thread loads the 27
// populations of its cell ONCE, reduces them to the ten moments the collision needs (kept in
// registers) and publishes uhat into a 4-deep shared-memory ring; a few threads do the same
// (rho, j only) for the one-cell xy halo, whose populations are L2 hits because neighbouring
// columns run concurrently.  Plane z is collided when plane z+1 has been published, so the
// populations cross HBM once in and once out: 216 B per cell update, no uhat field.
//
// Addressing: the 27 plane offsets i*n and the 27 interior push offsets are warp-uniform
// 64-bit constants in the kernel parameter block, so a load / store costs one 64-bit add.
#include "d3q27.cuh"

namespace hhrr {

template <int TX, int TY>
struct FusedCfg {
  static constexpr int THREADS = TX * TY;
  static constexpr int SX = TX + 2, SY = TY + 2;
  static constexpr int PLANE = SX * SY;
  static constexpr int HALO = 2 * TX + 2 * TY;
  static_assert(HALO <= THREADS, "halo duty must fit the block");
};

struct FusedArgs {
  Dom dm;
  PhysF ph;
  BodiesF bo;
  const float* fin;
  float* fout;
  const uint8_t* flags;
  const float* d;
  const float* wm_u;
  const float* wm_s;
  int zchunk;
  long long plane[Q];  // i * n                          (element offsets, warp-uniform)
  long long push[Q];   // i * n + cx + cy*nx + cz*nx*ny  (interior push target of direction i)
};

// porosity and u^B (+ wall-model slip) of a real cell
__device__ __forceinline__ void solid_state(const FusedArgs& a, uint8_t fl, int64_t c, int x, int y, int z,
                                            float& d, float uB[3]) {
  int type = fl & TYPE_MASK;
  d = 1.f;
  uB[0] = uB[1] = uB[2] = 0.f;
  if (type_has_solid_state(type)) {
    d = (type == HHRR_FRONTIER) ? __ldg(a.d + c) : 0.f;
    solid_velocity(a.ph, a.bo, fl, x, y, z, uB);
    if (fl & WM_VALID) {
      uB[0] += __ldg(a.wm_u + c);
      uB[1] += __ldg(a.wm_u + a.dm.n + c);
      uB[2] += __ldg(a.wm_u + 2 * a.dm.n + c);
    }
  }
}

// A virtual coordinate (may lie one cell outside the domain) -> real cell + reflection flag.
// ok = false if it is further out than the one-cell ring (ragged tiles).
__device__ __forceinline__ int virt(int v, int n, int mode, bool& flip, bool& ok) {
  flip = false;
  ok = (v >= -1 && v <= n);
  if (!ok) return 0;
  return wrap_axis(v, n, mode, flip);
}

template <int TX, int TY, int MINB>
__global__ void __launch_bounds__(TX* TY, MINB) fused_kernel(const __grid_constant__ FusedArgs a) {
  using C = FusedCfg<TX, TY>;
  __shared__ float ring[4][3][C::PLANE];
  const Dom& dm = a.dm;
  const int tid = threadIdx.x;
  const int tx = tid % TX, ty = tid / TX;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * a.zchunk, z1 = min(dm.nz, z0 + a.zchunk);
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;

  // own column
  const int xv = x0 + tx, yv = y0 + ty;
  bool fxo, fyo, okx, oky;
  const int xr = virt(xv, dm.nx, dm.mode[0], fxo, okx), yr = virt(yv, dm.ny, dm.mode[1], fyo, oky);
  const bool own_moment = okx && oky;                 // publishes uhat
  const bool own_collide = xv < dm.nx && yv < dm.ny;  // a real cell of this tile
  const bool xy_interior = xv > 0 && xv < dm.nx - 1 && yv > 0 && yv < dm.ny - 1;
  const int own_slot = (ty + 1) * C::SX + (tx + 1);
  const int64_t own_xy = xr + nx * yr;
  // halo duty
  bool halo = tid < C::HALO, fxh = false, fyh = false;
  int xh = 0, yh = 0, halo_slot = 0;
  if (halo) {
    int hx, hy;  // position in the extended tile
    if (tid < 2 * TX) {
      hx = tid % TX + 1;
      hy = (tid / TX) ? TY + 1 : 0;
    } else {
      int h = tid - 2 * TX;
      hx = (h / TY) ? TX + 1 : 0;
      hy = h % TY + 1;
    }
    bool ox, oy;
    xh = virt(x0 + hx - 1, dm.nx, dm.mode[0], fxh, ox);
    yh = virt(y0 + hy - 1, dm.ny, dm.mode[1], fyh, oy);
    halo = ox && oy;
    halo_slot = hy * C::SX + hx;
  }
  const int64_t halo_xy = xh + nx * yh;

  Moments mcur = {}, mnext = {};
  float rho_c = 1.f, rho_n = 1.f, uh_c[3] = {0, 0, 0}, uh_n[3] = {0, 0, 0};
  uint8_t fl_c = 0, fl_n = 0;

  // publishes uhat of virtual plane zq into ring slot (zq & 3); keeps the own cell's moments
  auto publish = [&](int zq, bool keep) {
    bool fz, okz;
    const int zr = virt(zq, dm.nz, dm.mode[2], fz, okz);
    float(*slot)[C::PLANE] = ring[zq & 3];
    const int64_t zoff = nxy * zr;
    if (own_moment) {
      const int64_t c = own_xy + zoff;
      const float* __restrict__ p = a.fin + c;
      float f[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) f[i] = __ldg(p + a.plane[i]);
      uint8_t fl = __ldg(a.flags + c);
      float d, uB[3], rho, uh[3];
      solid_state(a, fl, c, xr, yr, zr, d, uB);
      if (keep) {
        mnext = moments_all(f);
        homogenised_velocity(a.ph, mnext.drho, mnext.jx, mnext.jy, mnext.jz, d, uB, rho, uh);
        rho_n = rho;
        uh_n[0] = uh[0]; uh_n[1] = uh[1]; uh_n[2] = uh[2];
        fl_n = fl;
      } else {
        float drho, jx, jy, jz;
        moments_rho_j(f, drho, jx, jy, jz);
        homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
      }
      slot[0][own_slot] = fxo ? -uh[0] : uh[0];
      slot[1][own_slot] = fyo ? -uh[1] : uh[1];
      slot[2][own_slot] = fz ? -uh[2] : uh[2];
    }
    if (halo) {
      const int64_t c = halo_xy + zoff;
      const float* __restrict__ p = a.fin + c;
      float f[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) f[i] = __ldg(p + a.plane[i]);
      uint8_t fl = __ldg(a.flags + c);
      float d, uB[3], rho, uh[3], drho, jx, jy, jz;
      solid_state(a, fl, c, xh, yh, zr, d, uB);
      moments_rho_j(f, drho, jx, jy, jz);
      homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
      slot[0][halo_slot] = fxh ? -uh[0] : uh[0];
      slot[1][halo_slot] = fyh ? -uh[1] : uh[1];
      slot[2][halo_slot] = fz ? -uh[2] : uh[2];
    }
  };

  publish(z0 - 1, false);
  publish(z0, true);
  mcur = mnext; rho_c = rho_n; fl_c = fl_n;
  uh_c[0] = uh_n[0]; uh_c[1] = uh_n[1]; uh_c[2] = uh_n[2];

  for (int z = z0; z < z1; ++z) {
    publish(z + 1, z + 1 < z1);
    __syncthreads();
    if (own_collide) {
      float S[6], sigma = cell_sigma(a.ph, fl_c);
      const int64_t c = xv + nx * yv + nxy * z;
      if (fl_c & WM_VALID) {
#pragma unroll
        for (int q = 0; q < 6; ++q) S[q] = __ldg(a.wm_s + (int64_t)q * n + c);
        sigma = 0.f;
      } else {
        float(*sm)[C::PLANE] = ring[(z - 1) & 3];
        float(*s0)[C::PLANE] = ring[z & 3];
        float(*sp)[C::PLANE] = ring[(z + 1) & 3];
        const int o = own_slot;
        float dxu0 = s0[0][o + 1] - s0[0][o - 1], dxu1 = s0[1][o + 1] - s0[1][o - 1], dxu2 = s0[2][o + 1] - s0[2][o - 1];
        float dyu0 = s0[0][o + C::SX] - s0[0][o - C::SX], dyu1 = s0[1][o + C::SX] - s0[1][o - C::SX],
              dyu2 = s0[2][o + C::SX] - s0[2][o - C::SX];
        float dzu0 = sp[0][o] - sm[0][o], dzu1 = sp[1][o] - sm[1][o], dzu2 = sp[2][o] - sm[2][o];
        S[0] = 0.5f * dxu0;
        S[1] = 0.5f * dyu1;
        S[2] = 0.5f * dzu2;
        S[3] = 0.25f * (dyu0 + dxu1);
        S[4] = 0.25f * (dzu0 + dxu2);
        S[5] = 0.25f * (dzu1 + dyu2);
      }
      float o27[Q];
      collide(a.ph, mcur, rho_c, uh_c, S, sigma, o27);
      if (xy_interior && z > 0 && z < dm.nz - 1) {  // no wrap, no reflection: constant push offsets
        float* __restrict__ q = a.fout + c;
#pragma unroll
        for (int i = 0; i < Q; ++i) q[a.push[i]] = o27[i];
      } else {
        push_store(dm, a.fout, xv, yv, z, o27);
      }
    }
    mcur = mnext; rho_c = rho_n; fl_c = fl_n;
    uh_c[0] = uh_n[0]; uh_c[1] = uh_n[1]; uh_c[2] = uh_n[2];
  }
}

template <int TX, int TY, int MINB>
static cudaError_t launch_cfg(hhrr_lattice* L, const FusedArgs& a0) {
  FusedArgs a = a0;
  const Dom& dm = L->dom;
  int tiles = ((dm.nx + TX - 1) / TX) * ((dm.ny + TY - 1) / TY);
  int want = (8 * 148 * MINB + tiles - 1) / tiles;  // >= ~8 waves of resident blocks
  int maxchunks = (dm.nz + 15) / 16;                  // >= 16 planes per chunk
  int nch = want < 1 ? 1 : (want > maxchunks ? maxchunks : want);
  a.zchunk = (dm.nz + nch - 1) / nch;
  nch = (dm.nz + a.zchunk - 1) / a.zchunk;
  dim3 grid((dm.nx + TX - 1) / TX, (dm.ny + TY - 1) / TY, nch);
  fused_kernel<TX, TY, MINB><<<grid, TX * TY, 0, L->stream>>>(a);
  L->launches++;
  return cudaGetLastError();
}

cudaError_t launch_fused(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  FusedArgs a;
  a.dm = L->dom;
  a.ph = ph;
  a.bo = bo;
  a.fin = L->fA;
  a.fout = L->fB;
  a.flags = L->flags;
  a.d = L->d;
  a.wm_u = L->wm_u;
  a.wm_s = L->wm_s;
  a.zchunk = L->dom.nz;
  const long long n = L->dom.n, nx = L->dom.nx, nxy = (long long)L->dom.nx * L->dom.ny;
  for (int i = 0; i < Q; ++i) {
    a.plane[i] = i * n;
    a.push[i] = i * n + dir_cx(i) + dir_cy(i) * nx + dir_cz(i) * nxy;
  }
  switch (L->variant) {  // 1 = default; 11.. = tile shapes kept for tuning runs
    case 11: return launch_cfg<64, 8, 1>(L, a);
    case 12: return launch_cfg<64, 4, 4>(L, a);
    case 13: return launch_cfg<32, 8, 4>(L, a);
    case 14: return launch_cfg<128, 4, 2>(L, a);
    case 15: return launch_cfg<32, 16, 2>(L, a);
    case 16: return launch_cfg<64, 4, 2>(L, a);
    default: break;
  }
  if (L->dom.nx > 32) return launch_cfg<64, 8, 2>(L, a);
  return launch_cfg<32, 8, 2>(L, a);
}

}  // namespace hhrr
