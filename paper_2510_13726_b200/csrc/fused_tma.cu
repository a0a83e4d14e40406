// fused_tma.cu -- variant 4 of K2: the fused collide-stream kernel fed by TMA.
//
// Same step and the same sliding window along z as the other variants (Listing 3 line 3,
// PAPER.md:313; Eq. 6-14; S^FD of Eq. 10 from the time-n uhat of the six face neighbours).
// What changes is how the populations reach the SM: one elected lane of a producer warp issues
// cp.async.bulk.tensor (TMA) copies of the whole plane tile -- 27 populations x (64 x 8 cells +
// the two halo rows + two 4-cell-wide halo column strips) = 76 KB -- into a two-stage
// shared-memory pipeline guarded by mbarriers, one plane ahead of the arithmetic.  The 16 worker
// warps then read populations with LDS at immediate offsets (no address arithmetic, ~30-cycle
// latency instead of a DRAM round trip), reduce them to moments kept in registers, publish uhat
// into a 4-deep ring, and collide / push-store plane z once plane z+1 is published.
// Periodic wrap and mirror planes cost nothing extra: every halo region is its own TMA box with
// its own (wrapped or reflected) start coordinate.
//
// Needs nx % 64 == 0 and ny % 8 == 0 (whole tiles; TMA global strides multiples of 16 bytes);
// launch_fused_tma returns cudaErrorNotSupported otherwise and the caller falls back.
#include <cuda.h>

#include <cstdlib>

#include "ws_common.cuh"

namespace hhrr {

namespace tma {
constexpr int TX = 64, TY = 8, NS = 2;
constexpr int AUX = 96;                   // three warps for the xy halo
__host__ __device__ constexpr int workers(int cpt) { return TX * TY / cpt; }          // CPT cells per worker thread
__host__ __device__ constexpr int threads(int cpt) { return workers(cpt) + AUX + 32; }  // + one producer warp
constexpr int SX = TX + 2, SY = TY + 2, PLANE = SX * SY;
constexpr int HALO = 2 * TX + 2 * TY;
constexpr int MAIN_F = Q * TY * TX;       // floats per region of one stage
constexpr int YROW_F = Q * TX;
constexpr int XCOL_F = Q * TY * 4;
constexpr int STAGE_F = MAIN_F + 2 * YROW_F + 2 * XCOL_F;
constexpr uint32_t TMA_BYTES = STAGE_F * 4;     // what the five TMA boxes of one plane deliver
// the cells' flag bytes ride in the same stage (loaded by the idle lanes of the producer warp):
constexpr int FL_MAIN = 0, FL_YM = TY * TX, FL_YP = FL_YM + TX, FL_XM = FL_YP + TX, FL_XP = FL_XM + TY;
constexpr uint32_t STAGE_BYTES = TMA_BYTES + 768;
constexpr size_t RING_BYTES = 4 * 3 * PLANE * 4;
constexpr size_t SMEM = (size_t)NS * STAGE_BYTES + RING_BYTES + 64;
static_assert(FL_XP + TY <= 768 && STAGE_BYTES % 128 == 0, "flag region");
static_assert((MAIN_F * 4) % 128 == 0 && (YROW_F * 4) % 128 == 0 && (XCOL_F * 4) % 128 == 0, "TMA smem alignment");
}  // namespace tma

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
      : "memory");
}

// register reallocation between warpgroups (the kernel starts with 65536 / threads registers each;
// the producer/aux warpgroup hands most of its share to the two worker warpgroups)
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// uhat of plane `it` is published: one arrival per warp; waited for one iteration later (split phase:
// a warp may run up to one plane ahead of the slowest one instead of meeting it at a block barrier)
__device__ __forceinline__ void pub_arrive(uint32_t pub0, int it) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(pub0 + 8 * (it & 1));
}
__device__ __forceinline__ void pub_wait(uint32_t pub0, int it) { mbar_wait(pub0 + 8 * (it & 1), (it >> 1) & 1); }

template <int CPT>
__global__ void __launch_bounds__(tma::threads(CPT), 1)
    fused_tma_kernel(const __grid_constant__ WsArgs a, const __grid_constant__ CUtensorMap map_main,
                     const __grid_constant__ CUtensorMap map_row, const __grid_constant__ CUtensorMap map_col) {
  using namespace tma;
  constexpr int WORKERS = workers(CPT);
  extern __shared__ __align__(128) unsigned char smem[];
  float(*ring)[3][PLANE] = reinterpret_cast<float(*)[3][PLANE]>(smem + (size_t)NS * STAGE_BYTES);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)NS * STAGE_BYTES + RING_BYTES);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NS), pub0 = smem_u32(bars + 2 * NS);

  const Dom& dm = a.dm;
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int z0 = blockIdx.z * a.zchunk, z1 = min(dm.nz, z0 + a.zchunk);
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  const int pfirst = z0 - 1;

  // halo regions of this tile: real start coordinates (wrapped or reflected) and reflection flags
  bool fym, fyp, okh;
  const int ym = virt_ws(y0 - 1, dm.ny, dm.mode[1], fym, okh), yp = virt_ws(y0 + TY, dm.ny, dm.mode[1], fyp, okh);
  int xm_start, xm_idx, xp_start, xp_idx;
  bool fxm = false, fxp = false;
  if (x0 > 0) { xm_start = x0 - 4; xm_idx = 3; }
  else if (dm.mode[0] == HHRR_PERIODIC) { xm_start = dm.nx - 4; xm_idx = 3; }
  else { xm_start = 0; xm_idx = 0; fxm = true; }
  if (x0 + TX < dm.nx) { xp_start = x0 + TX; xp_idx = 0; }
  else if (dm.mode[0] == HHRR_PERIODIC) { xp_start = 0; xp_idx = 0; }
  else { xp_start = dm.nx - 4; xp_idx = 3; fxp = true; }

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(full0 + 8 * s, 2);  // TMA issue (+ its bytes) and the flag bytes
      mbar_init(empty0 + 8 * s, (WORKERS + AUX) / 32);
    }
    for (int s = 0; s < 2; ++s) mbar_init(pub0 + 8 * s, (WORKERS + AUX) / 32);  // uhat of a plane published
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if constexpr (CPT == 2) {  // 2 worker warpgroups + 1 warpgroup of aux/producer warps: 256*216 + 128*72 = 384*168
    if (tid >= WORKERS) reg_dec<72>(); else reg_inc<216>();
  }

  if (tid >= WORKERS + AUX) {
    // ------------------------------------------------------------------ producer: one lane issues TMA
    const int lane = tid & 31;
    for (int p = pfirst; p <= z1; ++p) {
      const int it = p - pfirst, s = it % NS, k = it / NS;
      if (k > 0) mbar_wait(empty0 + 8 * s, (k - 1) & 1);
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const uint32_t bar = full0 + 8 * s;
      unsigned char* stb = smem + (size_t)s * STAGE_BYTES;
      if (lane == 0) {
        const uint32_t st = smem_u32(stb);
        mbar_expect_tx(bar, TMA_BYTES);
        tma_load_4d(st, &map_main, x0, y0, zr, 0, bar);
        tma_load_4d(st + 4 * MAIN_F, &map_row, x0, ym, zr, 0, bar);
        tma_load_4d(st + 4 * (MAIN_F + YROW_F), &map_row, x0, yp, zr, 0, bar);
        tma_load_4d(st + 4 * (MAIN_F + 2 * YROW_F), &map_col, xm_start, y0, zr, 0, bar);
        tma_load_4d(st + 4 * (MAIN_F + 2 * YROW_F + XCOL_F), &map_col, xp_start, y0, zr, 0, bar);
      }
      // flag bytes of the same cells: 8 rows x 64 B + 2 halo rows as 16-byte loads, the columns bytewise
      const uint8_t* fz0 = a.flags + nxy * zr;
      unsigned char* flb = stb + TMA_BYTES;
      const uint4 vmain = __ldg(reinterpret_cast<const uint4*>(fz0 + (x0 + (lane & 3) * 16) + nx * (y0 + (lane >> 2))));
      uint4 vrow = make_uint4(0, 0, 0, 0);
      uint8_t vcol = 0;
      if (lane < 8) vrow = __ldg(reinterpret_cast<const uint4*>(fz0 + (x0 + (lane & 3) * 16) + nx * ((lane >> 2) ? yp : ym)));
      if (lane >= 8 && lane < 8 + 2 * TY) {
        const int h = lane - 8, right = h / TY, row = h % TY;
        vcol = __ldg(fz0 + (right ? xp_start + xp_idx : xm_start + xm_idx) + nx * (y0 + row));
      }
      *reinterpret_cast<uint4*>(flb + FL_MAIN + (lane >> 2) * TX + (lane & 3) * 16) = vmain;
      if (lane < 8) *reinterpret_cast<uint4*>(flb + FL_YM + (lane >> 2) * TX + (lane & 3) * 16) = vrow;
      if (lane >= 8 && lane < 8 + 2 * TY) flb[FL_XM + (lane - 8)] = vcol;
      __syncwarp();
      if (lane == 0) mbar_arrive(bar);
    }
    return;
  }

  if (tid >= WORKERS) {
    // ------------------------------------------------------------------ aux warps: uhat of the xy halo
    // lane a owns halo cells a and a + AUX (if < HALO): where the populations sit in a stage, where
    // uhat goes in the ring, which real cell it is
    const int a0 = tid - WORKERS;
    int h_off[2], h_stride[2], h_slot[2], h_x[2], h_y[2], h_fl[2];
    bool h_fx[2], h_fy[2], h_on[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int hc = a0 + k * AUX;
      h_on[k] = hc < HALO;
      h_fx[k] = h_fy[k] = false;
      if (hc < 2 * TX) {
        const int hx = hc % TX, top = hc / TX;
        h_off[k] = MAIN_F + top * YROW_F + hx;
        h_fl[k] = (top ? FL_YP : FL_YM) + hx;
        h_stride[k] = TX;
        h_slot[k] = (top ? TY + 1 : 0) * SX + hx + 1;
        h_x[k] = x0 + hx;
        h_y[k] = top ? yp : ym;
        h_fy[k] = top ? fyp : fym;
      } else {
        const int h = (hc - 2 * TX) % (2 * TY), right = h / TY, row = h % TY;
        h_off[k] = MAIN_F + 2 * YROW_F + right * XCOL_F + row * 4 + (right ? xp_idx : xm_idx);
        h_fl[k] = FL_XM + right * TY + row;
        h_stride[k] = TY * 4;
        h_slot[k] = (row + 1) * SX + (right ? TX + 1 : 0);
        h_x[k] = right ? xp_start + xp_idx : xm_start + xm_idx;
        h_y[k] = y0 + row;
        h_fx[k] = right ? fxp : fxm;
      }
    }
    for (int p = pfirst; p <= z1; ++p) {
      const int it = p - pfirst, s = it % NS, k2 = it / NS;
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const int64_t zoff = nxy * zr;
      const float* st = reinterpret_cast<const float*>(smem + (size_t)s * STAGE_BYTES);
      const uint8_t* flb = smem + (size_t)s * STAGE_BYTES + TMA_BYTES;
      float(*slot)[PLANE] = ring[it & 3];
      // every worker is past the collision that read this ring slot; waiting from it = 2 on (not only
      // once the slot is reused) also keeps any arrival for plane it behind the completed phase it - 2
      if (it >= 2) pub_wait(pub0, it - 2);
      mbar_wait(full0 + 8 * s, k2 & 1);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (!h_on[k]) continue;
        float f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = st[h_off[k] + i * h_stride[k]];
        const int64_t c = h_x[k] + nx * h_y[k] + zoff;
        float d, uB[3], rho, uh[3], drho, jx, jy, jz;
        solid_state_ws(a, flb[h_fl[k]], c, h_x[k], h_y[k], zr, d, uB);
        moments_rho_j(f, drho, jx, jy, jz);
        homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
        slot[0][h_slot[k]] = h_fx[k] ? -uh[0] : uh[0];
        slot[1][h_slot[k]] = h_fy[k] ? -uh[1] : uh[1];
        slot[2][h_slot[k]] = fz ? -uh[2] : uh[2];
      }
      __syncwarp();
      if ((tid & 31) == 0) {
        mbar_arrive(empty0 + 8 * s);
        mbar_arrive(pub0 + 8 * (it & 1));
      }
    }
    return;
  }

  if constexpr (CPT == 1) {
  // -------------------------------------------------------------------- workers, one cell each
  const int tx = tid % TX, ty = tid / TX;
  const int xv = x0 + tx, yv = y0 + ty;
  const bool xy_interior = xv > 0 && xv < dm.nx - 1 && yv > 0 && yv < dm.ny - 1;
  const int own_slot = (ty + 1) * SX + (tx + 1);
  const int own_off = ty * TX + tx;  // + i * TY * TX: population i of the own cell
  const int64_t own_xy = xv + nx * yv;

  Moments mcur = {}, mnext = {};
  float rho_c = 1.f, rho_n = 1.f, uh_c[3] = {0, 0, 0}, uh_n[3] = {0, 0, 0};
  uint8_t fl_c = 0, fl_n = 0;
  char* dst = reinterpret_cast<char*>(a.fout) + 4 * (own_xy + nxy * z0);
  const int64_t zstride_b = 4 * nxy;

  // one loop over the virtual planes z0-1 .. z1: publish plane p, then collide plane p-1
  for (int p = pfirst; p <= z1; ++p) {
    const int it = p - pfirst, s = it % NS, k2 = it / NS;
    {
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const int64_t c = own_xy + nxy * zr;
      const float* st = reinterpret_cast<const float*>(smem + (size_t)s * STAGE_BYTES);
      float(*slot)[PLANE] = ring[it & 3];
      mbar_wait(full0 + 8 * s, k2 & 1);
      const uint8_t fl = smem[(size_t)s * STAGE_BYTES + TMA_BYTES + FL_MAIN + own_off];
      float f[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) f[i] = st[i * (TY * TX) + own_off];
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * s);  // this warp has read its part of the stage
      float d, uB[3], rho, uh[3];
      solid_state_ws(a, fl, c, xv, yv, zr, d, uB);
      if (p >= z0 && p < z1) {
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
      slot[0][own_slot] = uh[0];
      slot[1][own_slot] = uh[1];
      slot[2][own_slot] = fz ? -uh[2] : uh[2];
    }
    pub_arrive(pub0, it);
    // the xy neighbours' uhat of plane p-1 (own cell of plane p: written above).  Waited for in EVERY
    // iteration, also the two that collide nothing: a warp must not arrive for plane it + 1 on the
    // barrier plane it - 1 still uses
    if (it >= 1) pub_wait(pub0, it - 1);
    const int z = p - 1;
    if (z >= z0) {
      float S[6], sigma = cell_sigma(a.ph, fl_c);
      if (fl_c & WM_VALID) {
        const int64_t c = own_xy + nxy * z;
#pragma unroll
        for (int q = 0; q < 6; ++q) S[q] = __ldg(a.wm_s + (int64_t)q * n + c);
        sigma = 0.f;
      } else {
        float(*sm)[PLANE] = ring[(it - 2) & 3];
        float(*s0)[PLANE] = ring[(it - 1) & 3];
        float(*sp)[PLANE] = ring[it & 3];
        const int o = own_slot;
        float dxu0 = s0[0][o + 1] - s0[0][o - 1], dxu1 = s0[1][o + 1] - s0[1][o - 1], dxu2 = s0[2][o + 1] - s0[2][o - 1];
        float dyu0 = s0[0][o + SX] - s0[0][o - SX], dyu1 = s0[1][o + SX] - s0[1][o - SX],
              dyu2 = s0[2][o + SX] - s0[2][o - SX];
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
#pragma unroll
        for (int i = 0; i < Q; ++i) *reinterpret_cast<float*>(dst + a.push_b[i]) = o27[i];
      } else {
        push_store(dm, a.fout, xv, yv, z, o27);
      }
      dst += zstride_b;
    }
    if (p >= z0) {
      mcur = mnext; rho_c = rho_n; fl_c = fl_n;
      uh_c[0] = uh_n[0]; uh_c[1] = uh_n[1]; uh_c[2] = uh_n[2];
    }
  }
  } else {
    // ------------------------------------------------------------------ workers, two x-adjacent cells each
    constexpr int HX = TX / 2;
    const int tx2 = tid % HX, ty = tid / HX;
    const int xa = x0 + 2 * tx2, yv = y0 + ty;  // cells (xa, yv) and (xa + 1, yv)
    const bool pair_interior = xa > 0 && xa + 1 < dm.nx - 1 && yv > 0 && yv < dm.ny - 1;
    const int own_slot = (ty + 1) * SX + 2 * tx2 + 1;
    const int own_off = ty * TX + 2 * tx2;  // + i * TY * TX: population i of the pair (8-byte aligned)
    const int64_t own_xy = xa + nx * yv;

    Moments mcur[2] = {}, mnext[2] = {};
    float rho_c[2] = {1.f, 1.f}, rho_n[2] = {1.f, 1.f}, uh_c[2][3] = {}, uh_n[2][3] = {};
    uint8_t fl_c[2] = {0, 0}, fl_n[2] = {0, 0};
    char* dst = reinterpret_cast<char*>(a.fout) + 4 * (own_xy + nxy * z0);
    const int64_t zstride_b = 4 * nxy;

    for (int p = pfirst; p <= z1; ++p) {
      const int it = p - pfirst, s = it % NS, k2 = it / NS;
      {
        bool fz, okz;
        const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
        const int64_t c = own_xy + nxy * zr;
        const float* st = reinterpret_cast<const float*>(smem + (size_t)s * STAGE_BYTES);
        float(*slot)[PLANE] = ring[it & 3];
        mbar_wait(full0 + 8 * s, k2 & 1);
        const uint16_t flw = *reinterpret_cast<const uint16_t*>(smem + (size_t)s * STAGE_BYTES + TMA_BYTES + FL_MAIN + own_off);
        float f[2][Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) {
          const float2 v = *reinterpret_cast<const float2*>(st + i * (TY * TX) + own_off);
          f[0][i] = v.x;
          f[1][i] = v.y;
        }
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * s);  // this warp has read its part of the stage
        const bool keep = p >= z0 && p < z1;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const uint8_t fl = (uint8_t)(k ? (flw >> 8) : (flw & 0xff));
          float d, uB[3], rho, uh[3];
          solid_state_ws(a, fl, c + k, xa + k, yv, zr, d, uB);
          if (keep) {
            mnext[k] = moments_all(f[k]);
            homogenised_velocity(a.ph, mnext[k].drho, mnext[k].jx, mnext[k].jy, mnext[k].jz, d, uB, rho, uh);
            rho_n[k] = rho;
            uh_n[k][0] = uh[0]; uh_n[k][1] = uh[1]; uh_n[k][2] = uh[2];
            fl_n[k] = fl;
          } else {
            float drho, jx, jy, jz;
            moments_rho_j(f[k], drho, jx, jy, jz);
            homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
          }
          slot[0][own_slot + k] = uh[0];
          slot[1][own_slot + k] = uh[1];
          slot[2][own_slot + k] = fz ? -uh[2] : uh[2];
        }
      }
      pub_arrive(pub0, it);
      // the xy neighbours' uhat of plane p-1 (own cell of plane p: written above).  Waited for in EVERY
      // iteration, also the two that collide nothing: a warp must not arrive for plane it + 1 on the
      // barrier plane it - 1 still uses
      if (it >= 1) pub_wait(pub0, it - 1);
      const int z = p - 1;
      if (z >= z0) {
        float(*sm)[PLANE] = ring[(it - 2) & 3];
        float(*s0)[PLANE] = ring[(it - 1) & 3];
        float(*sp)[PLANE] = ring[it & 3];
        float out[2][Q];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int o = own_slot + k;
          float S[6], sigma = cell_sigma(a.ph, fl_c[k]);
          float dxu0 = s0[0][o + 1] - s0[0][o - 1], dxu1 = s0[1][o + 1] - s0[1][o - 1], dxu2 = s0[2][o + 1] - s0[2][o - 1];
          float dyu0 = s0[0][o + SX] - s0[0][o - SX], dyu1 = s0[1][o + SX] - s0[1][o - SX],
                dyu2 = s0[2][o + SX] - s0[2][o - SX];
          float dzu0 = sp[0][o] - sm[0][o], dzu1 = sp[1][o] - sm[1][o], dzu2 = sp[2][o] - sm[2][o];
          S[0] = 0.5f * dxu0;
          S[1] = 0.5f * dyu1;
          S[2] = 0.5f * dzu2;
          S[3] = 0.25f * (dyu0 + dxu1);
          S[4] = 0.25f * (dzu0 + dxu2);
          S[5] = 0.25f * (dzu1 + dyu2);
          if (fl_c[k] & WM_VALID) {  // wall-model strain, sigma = 0 (rare)
            const int64_t c = own_xy + k + nxy * z;
#pragma unroll
            for (int q = 0; q < 6; ++q) S[q] = __ldg(a.wm_s + (int64_t)q * n + c);
            sigma = 0.f;
          }
          collide(a.ph, mcur[k], rho_c[k], uh_c[k], S, sigma, out[k]);
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
          push_store(dm, a.fout, xa + 1, yv, z, out[1]);
        }
        dst += zstride_b;
      }
      if (p >= z0) {
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          mcur[k] = mnext[k]; rho_c[k] = rho_n[k]; fl_c[k] = fl_n[k];
          uh_c[k][0] = uh_n[k][0]; uh_c[k][1] = uh_n[k][1]; uh_c[k][2] = uh_n[k][2];
        }
      }
    }
  }
}

// ---- host side: tensor maps (driver entry point through the runtime; libcuda is not linked) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// populations as a 4-D tensor (x, y, z, population) of fp32; box = bx x by x 1 x 27
static bool make_map(CUtensorMap* m, const float* base, const Dom& dm, uint32_t bx, uint32_t by) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t gdim[4] = {(cuuint64_t)dm.nx, (cuuint64_t)dm.ny, (cuuint64_t)dm.nz, (cuuint64_t)Q};
  cuuint64_t gstr[3] = {(cuuint64_t)dm.nx * 4, (cuuint64_t)dm.nx * dm.ny * 4, (cuuint64_t)dm.n * 4};
  cuuint32_t box[4] = {bx, by, 1, (cuuint32_t)Q};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float*>(base), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

cudaError_t launch_fused_tma(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  const Dom& dm = L->dom;
  if (dm.nx % tma::TX || dm.ny % tma::TY) return cudaErrorNotSupported;  // whole tiles only
  CUtensorMap m_main, m_row, m_col;
  if (!make_map(&m_main, L->fA, dm, tma::TX, tma::TY) || !make_map(&m_row, L->fA, dm, tma::TX, 1) ||
      !make_map(&m_col, L->fA, dm, 4, tma::TY))
    return cudaErrorNotSupported;
  WsArgs a;
  fill_ws_args(L, ph, bo, a);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(fused_tma_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma::SMEM);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(fused_tma_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int nch = ws_zchunks(dm.nz, 19);
  a.zchunk = (dm.nz + nch - 1) / nch;
  nch = (dm.nz + a.zchunk - 1) / a.zchunk;
  dim3 grid(dm.nx / tma::TX, dm.ny / tma::TY, nch);
  if (L->variant == 41)
    fused_tma_kernel<1><<<grid, tma::threads(1), tma::SMEM, L->stream>>>(a, m_main, m_row, m_col);
  else
    fused_tma_kernel<2><<<grid, tma::threads(2), tma::SMEM, L->stream>>>(a, m_main, m_row, m_col);
  L->launches++;
  return cudaGetLastError();
}

}  // namespace hhrr
