// fused_ws2.cu -- variant 3 of K2: the warp-specialised fused collide-stream kernel of
// fused_ws.cu with TWO x-adjacent cells per lane in both roles (Listing 3 line 3, PAPER.md:313;
// Eq. 6-14).  Same ring, same barriers, same arithmetic; what changes is the instruction count
// of the memory side, which is what bounds the kernel (ncu: 872 instructions per cell, two
// 64-bit adds per global access):
//   producers : one LDG.64 per population for a cell pair (27 per pair instead of 54), one warp
//               per 64-cell row of the tile / halo, 54 loads in flight per lane;
//   consumers : LDS.64 for the pair's moments, one address per direction for the pair's two
//               stores (STG.64 where c_x = 0, else STG.32 at +0 / +4).
// Needs an even nx (pairs never straddle a row end and stay 8-byte aligned); launch_fused_ws2
// returns cudaErrorNotSupported otherwise and the caller falls back to fused_ws.cu.
#include <cstdlib>

#include "ws_common.cuh"

namespace hhrr {

template <int TX, int TY, int DEPTH>
struct Ws2Cfg {
  static constexpr int CELLS = TX * TY;
  static constexpr int CTHREADS = CELLS / 2;            // consumer threads: one cell pair each
  static constexpr int ROWW = TX / 64;                  // producer warps per row (64 cells per warp)
  static constexpr int NPW = ROWW * (TY + 2);           // row warps: TY interior rows + 2 halo rows
  static constexpr int PWARPS = NPW + 1;                // + one warp for the two x-halo columns
  static constexpr int THREADS = CTHREADS + PWARPS * 32;
  static constexpr int SX = TX + 2, SY = TY + 2;
  static constexpr int PLANE = SX * SY;
  static constexpr int SLOT_FLOATS = 3 * PLANE + 7 * CELLS;
  static constexpr size_t SLOT_BYTES = SLOT_FLOATS * 4 + CELLS;
  static constexpr size_t SLOT_STRIDE = (SLOT_BYTES + 15) / 16 * 16;
  static constexpr size_t SMEM = SLOT_STRIDE * DEPTH;
  static_assert(TX % 64 == 0 && 2 * TY <= 32, "tile shape");
  static_assert((3 * PLANE * 4) % 8 == 0, "moment arrays must stay 8-byte aligned");
  static_assert(2 * DEPTH + 1 <= 16, "named barriers");
};

// what a producer lane keeps about its (up to) two cells; fixed over the z march
struct PPair {
  int64_t cxy[2];  // xr + nx*yr, or -1 if the lane has no such cell
  int xr[2], yr;
  int o[2];        // index into the padded uhat plane
  int ci[2];       // interior cell index, or -1 for halo cells
  bool fx[2], fy;  // reflected in x / y (mirror axes)
  bool vec;        // both cells real, adjacent and 8-byte aligned: one LDG.64 per population
};

template <int TX, int TY>
__device__ __forceinline__ PPair make_pair(const Dom& dm, int x0, int y0, int hx0, int hy, bool a0, bool a1) {
  PPair t;
  bool oky;
  t.yr = virt_ws(y0 + hy - 1, dm.ny, dm.mode[1], t.fy, oky);
  const bool act[2] = {a0, a1};
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int hx = hx0 + k;
    bool okx;
    t.xr[k] = virt_ws(x0 + hx - 1, dm.nx, dm.mode[0], t.fx[k], okx);
    t.cxy[k] = (act[k] && okx && oky) ? (int64_t)t.xr[k] + (int64_t)dm.nx * t.yr : -1;
    t.o[k] = hy * (TX + 2) + hx;
    t.ci[k] = (hx >= 1 && hx <= TX && hy >= 1 && hy <= TY) ? (hy - 1) * TX + (hx - 1) : -1;
  }
  t.vec = t.cxy[0] >= 0 && t.cxy[1] == t.cxy[0] + 1 && !t.fx[0] && !t.fx[1] && (t.cxy[0] & 1) == 0;
  return t;
}

template <int TX, int TY, int DEPTH>
__global__ void __launch_bounds__(Ws2Cfg<TX, TY, DEPTH>::THREADS, 1)
    fused_ws2_kernel(const __grid_constant__ WsArgs a) {
  using C = Ws2Cfg<TX, TY, DEPTH>;
  extern __shared__ __align__(16) unsigned char smem[];
  const Dom& dm = a.dm;
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * a.zchunk, z1 = min(dm.nz, z0 + a.zchunk);
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  const int pfirst = z0 - 1;  // first plane produced; plane p lives in slot (p - pfirst) % DEPTH

  auto slot_uh = [&](int s) { return reinterpret_cast<float*>(smem + (size_t)s * C::SLOT_STRIDE); };
  auto slot_mom = [&](int s) { return slot_uh(s) + 3 * C::PLANE; };
  auto slot_fl = [&](int s) { return reinterpret_cast<uint8_t*>(slot_mom(s) + 7 * C::CELLS); };

  if (tid >= C::CTHREADS) {
    // ------------------------------------------------------------------ producers
    const int pw = (tid - C::CTHREADS) >> 5, lane = tid & 31;
    // warps 0..NPW-1: one 64-cell row segment each (two cells per lane); warp NPW: the x-halo columns
    const PPair t = pw < C::NPW
                        ? make_pair<TX, TY>(dm, x0, y0, (pw % C::ROWW) * 64 + 2 * lane + 1, pw / C::ROWW, true, true)
                        : make_pair<TX, TY>(dm, x0, y0, (lane / TY) ? TX + 1 : 0, lane % TY + 1, lane < 2 * TY, false);
    const char* fin_b = reinterpret_cast<const char*>(a.fin);
    int s = 0;
    for (int p = pfirst; p <= z1; ++p) {
      if (p - pfirst >= DEPTH) bar_sync(1 + DEPTH + s, C::THREADS);  // EMPTY[s]
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const int64_t zoff = nxy * zr;
      float* uhs = slot_uh(s);
      float* moms = slot_mom(s);
      uint8_t* fls = slot_fl(s);
      const bool need_moments = p >= z0 && p < z1;  // planes z0-1 and z1 only feed S^FD
      float f[2][Q];
      uint8_t fl[2] = {0, 0};
      if (t.vec) {
        const int64_t c = t.cxy[0] + zoff;
        const char* __restrict__ src = fin_b + 4 * c;
#pragma unroll
        for (int i = 0; i < Q; ++i) {
          const float2 v = __ldg(reinterpret_cast<const float2*>(src + a.plane_b[i]));
          f[0][i] = v.x;
          f[1][i] = v.y;
        }
        const uint16_t w = __ldg(reinterpret_cast<const uint16_t*>(a.flags + c));
        fl[0] = (uint8_t)(w & 0xff);
        fl[1] = (uint8_t)(w >> 8);
      } else {
#pragma unroll
        for (int k = 0; k < 2; ++k)
          if (t.cxy[k] >= 0) {
            const int64_t c = t.cxy[k] + zoff;
            const char* __restrict__ src = fin_b + 4 * c;
#pragma unroll
            for (int i = 0; i < Q; ++i) f[k][i] = __ldg(reinterpret_cast<const float*>(src + a.plane_b[i]));
            fl[k] = __ldg(a.flags + c);
          }
      }
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (t.cxy[k] < 0) continue;
        const int64_t c = t.cxy[k] + zoff;
        float d, uB[3], rho, uh[3];
        solid_state_ws(a, fl[k], c, t.xr[k], t.yr, zr, d, uB);
        if (t.ci[k] >= 0 && need_moments) {
          Moments m = moments_all(f[k]);
          homogenised_velocity(a.ph, m.drho, m.jx, m.jy, m.jz, d, uB, rho, uh);
          const int ci = t.ci[k];
          moms[ci] = m.drho;
          moms[C::CELLS + ci] = m.mxx;
          moms[2 * C::CELLS + ci] = m.myy;
          moms[3 * C::CELLS + ci] = m.mzz;
          moms[4 * C::CELLS + ci] = m.mxy;
          moms[5 * C::CELLS + ci] = m.mxz;
          moms[6 * C::CELLS + ci] = m.myz;
          fls[ci] = fl[k];
        } else {
          float drho, jx, jy, jz;
          moments_rho_j(f[k], drho, jx, jy, jz);
          homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
        }
        const int o = t.o[k];
        uhs[o] = t.fx[k] ? -uh[0] : uh[0];
        uhs[C::PLANE + o] = t.fy ? -uh[1] : uh[1];
        uhs[2 * C::PLANE + o] = fz ? -uh[2] : uh[2];
      }
      __syncwarp();
      bar_arrive(1 + s, C::THREADS);  // FULL[s]
      s = (s + 1 == DEPTH) ? 0 : s + 1;
    }
  } else {
    // ------------------------------------------------------------------ consumers
    constexpr int HX = TX / 2;
    const int tx2 = tid % HX, ty = tid / HX;
    const int xa = x0 + 2 * tx2, yv = y0 + ty;  // cells (xa, yv) and (xa + 1, yv)
    const bool row_ok = yv < dm.ny;
    const bool have[2] = {row_ok && xa < dm.nx, row_ok && xa + 1 < dm.nx};
    const bool pair_interior = xa > 0 && xa + 1 < dm.nx - 1 && yv > 0 && yv < dm.ny - 1;
    const int ci = ty * TX + 2 * tx2, o = (ty + 1) * C::SX + 2 * tx2 + 1;
    char* dst = reinterpret_cast<char*>(a.fout) + 4 * ((int64_t)xa + nx * yv + nxy * z0);
    const int64_t zstride_b = 4 * nxy;
    bar_sync(1 + 0, C::THREADS);            // plane z0-1
    bar_sync(1 + (1 % DEPTH), C::THREADS);  // plane z0
    int sm = 0, sc = 1 % DEPTH, sp = 2 % DEPTH;
    for (int z = z0; z < z1; ++z) {
      bar_sync(1 + sp, C::THREADS);  // FULL for plane z+1
      if (have[0]) {
        const float* u0 = slot_uh(sc);
        const float* up = slot_uh(sp);
        const float* um = slot_uh(sm);
        const float* mo = slot_mom(sc);
        const uint16_t flw = *reinterpret_cast<const uint16_t*>(slot_fl(sc) + ci);
        float2 mv[7];
#pragma unroll
        for (int q = 0; q < 7; ++q) mv[q] = *reinterpret_cast<const float2*>(mo + q * C::CELLS + ci);
        float out[2][Q];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          if (!have[k]) continue;
          const uint8_t fl = (uint8_t)(k ? (flw >> 8) : (flw & 0xff));
          Moments m;
          m.drho = k ? mv[0].y : mv[0].x;
          m.mxx = k ? mv[1].y : mv[1].x;
          m.myy = k ? mv[2].y : mv[2].x;
          m.mzz = k ? mv[3].y : mv[3].x;
          m.mxy = k ? mv[4].y : mv[4].x;
          m.mxz = k ? mv[5].y : mv[5].x;
          m.myz = k ? mv[6].y : mv[6].x;
          m.jx = m.jy = m.jz = 0.f;  // not used by collide()
          const float rho = 1.f + m.drho;
          const int ok = o + k;
          float uh[3] = {u0[ok], u0[C::PLANE + ok], u0[2 * C::PLANE + ok]};
          float S[6], sigma = cell_sigma(a.ph, fl);
          if (fl & WM_VALID) {
            const int64_t c = xa + k + nx * yv + nxy * z;
#pragma unroll
            for (int q = 0; q < 6; ++q) S[q] = __ldg(a.wm_s + (int64_t)q * n + c);
            sigma = 0.f;
          } else {
            float dxu0 = u0[ok + 1] - u0[ok - 1], dxu1 = u0[C::PLANE + ok + 1] - u0[C::PLANE + ok - 1],
                  dxu2 = u0[2 * C::PLANE + ok + 1] - u0[2 * C::PLANE + ok - 1];
            float dyu0 = u0[ok + C::SX] - u0[ok - C::SX],
                  dyu1 = u0[C::PLANE + ok + C::SX] - u0[C::PLANE + ok - C::SX],
                  dyu2 = u0[2 * C::PLANE + ok + C::SX] - u0[2 * C::PLANE + ok - C::SX];
            float dzu0 = up[ok] - um[ok], dzu1 = up[C::PLANE + ok] - um[C::PLANE + ok],
                  dzu2 = up[2 * C::PLANE + ok] - um[2 * C::PLANE + ok];
            S[0] = 0.5f * dxu0;
            S[1] = 0.5f * dyu1;
            S[2] = 0.5f * dzu2;
            S[3] = 0.25f * (dyu0 + dxu1);
            S[4] = 0.25f * (dzu0 + dxu2);
            S[5] = 0.25f * (dzu1 + dyu2);
          }
          collide(a.ph, m, rho, uh, S, sigma, out[k]);
        }
        if (pair_interior && z > 0 && z < dm.nz - 1) {  // no wrap, no reflection: constant push offsets
#pragma unroll
          for (int i = 0; i < Q; ++i) {
            char* q = dst + a.push_b[i];
            if (dir_cx(i) == 0) {  // the pair's targets are 8-byte aligned
              *reinterpret_cast<float2*>(q) = make_float2(out[0][i], out[1][i]);
            } else {
              *reinterpret_cast<float*>(q) = out[0][i];
              *reinterpret_cast<float*>(q + 4) = out[1][i];
            }
          }
        } else {
          push_store(dm, a.fout, xa, yv, z, out[0]);
          if (have[1]) push_store(dm, a.fout, xa + 1, yv, z, out[1]);
        }
      }
      dst += zstride_b;
      __syncwarp();
      if (z - 1 + DEPTH <= z1) bar_arrive(1 + DEPTH + sm, C::THREADS);  // EMPTY: plane z-1 is done with
      sm = sc;
      sc = sp;
      sp = (sp + 1 == DEPTH) ? 0 : sp + 1;
    }
  }
}

template <int TX, int TY, int DEPTH>
static cudaError_t launch_ws2_cfg(hhrr_lattice* L, const WsArgs& a0) {
  using C = Ws2Cfg<TX, TY, DEPTH>;
  WsArgs a = a0;
  const Dom& dm = L->dom;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(fused_ws2_kernel<TX, TY, DEPTH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)C::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int nch = ws_zchunks(dm.nz, 19);
  a.zchunk = (dm.nz + nch - 1) / nch;
  nch = (dm.nz + a.zchunk - 1) / a.zchunk;
  dim3 grid((dm.nx + TX - 1) / TX, (dm.ny + TY - 1) / TY, nch);
  fused_ws2_kernel<TX, TY, DEPTH><<<grid, C::THREADS, C::SMEM, L->stream>>>(a);
  L->launches++;
  return cudaGetLastError();
}

cudaError_t launch_fused_ws2(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  if (L->dom.nx % 2) return cudaErrorNotSupported;  // pairs need an even row length
  WsArgs a;
  fill_ws_args(L, ph, bo, a);
  switch (L->variant) {
    case 31: return launch_ws2_cfg<64, 8, 5>(L, a);
    case 32: return launch_ws2_cfg<64, 12, 4>(L, a);
    case 33: return launch_ws2_cfg<128, 8, 4>(L, a);
    case 34: return launch_ws2_cfg<64, 16, 4>(L, a);
    default: break;
  }
  return launch_ws2_cfg<64, 8, 4>(L, a);
}

}  // namespace hhrr
