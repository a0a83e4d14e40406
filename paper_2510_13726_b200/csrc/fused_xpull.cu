// fused_xpull.cu -- variant 5 of K2 (default): the TMA-fed fused collide-stream kernel on
// "x-pull / yz-push" storage.
//
// Same step as every other variant (Listing 3 line 3; Eq. 6-14; S^FD of Eq. 10 from
// the time-n uhat of the six face neighbours, sliding window along z).  What changes is WHERE the
// streaming shift of Eq. 6 is paid:
//   * plane i of the buffer holds g_i(x,y,z) = f*_i(x, y - c_iy, z - c_iz): the post-collision value
//     already moved along y and z (whole, 128-byte aligned rows) but not yet along x;
//   * the x shift happens on the read side, in shared memory: the TMA box of a TX-wide tile is TX + 8 cells
//     wide (4 + TX + 4: box starts must be 16-byte aligned), population i of cell x is read at column x - c_ix.
// Every global store of the kernel is therefore an aligned, full-sector 8-byte store of two x-adjacent
// cells (27 per thread and plane instead of 45 partly half-filled ones), and the wide box carries the x
// halo of the tile.  Tiles at the periodic x boundary get three small extra boxes (the 4 wrapped columns)
// which only their edge lanes read.
//
// Region split (Listing 2; R20): a block with no cell in an FSI box takes the bulk
// path of the same code -- no halo rows, no flag bytes, no overlap planes, no uhat ring.
//
// Tile 64 x 8 (nx % 64 == 0, nx >= 128, ny % 8 == 0) or 128 x 4 (nx % 128 == 0, nx >= 256, ny % 4 == 0), periodic
// x axis (xpull_supported); other lattices keep post-stream storage and run variant 2.
#include <cuda.h>

#include <cstdlib>

#include "ws_common.cuh"

namespace hhrr {

// Tile shape TX x TY (512 cells).  128 x 4 is preferred: the box of a tile carries 4 cells of x halo on either
// side, which cost whole 32-byte sectors that the x neighbour's block reads again (and mostly finds evicted),
// 2 sectors per 16 with 128-cell rows, 2 per 8 with 64-cell rows.  64 x 8 serves lattices 128 x 4 cannot tile.
template <int TX_, int TY_>
struct XpCfg {
  // pipeline stages: two planes of 27 populations fill shared memory; the D3Q19 stages are 30 % smaller and a third one fits
  static constexpr int TX = TX_, TY = TY_, NS = (Q == 19 && TX_ == 64) ? 3 : 2, W = TX + 8;
  static constexpr int WORKERS = TX * TY / 2, AUX = 96, THREADS = WORKERS + AUX + 32;
  // uhat ring plane: SY rows of SX floats; tile cell lx sits at column lx + 2 (an EVEN slot: a worker's cell pair
  // is one aligned 8-byte word), the x halo at columns 1 and TX + 2, columns 0 and TX + 3 are padding
  static constexpr int SX = TX + 4, SY = TY + 2, PLANE = SX * SY;
  static constexpr int HALO = 2 * TX + 2 * TY, HSLOTS = (HALO + AUX - 1) / AUX;
  // one stage, in floats: [Q][TY][W] tile rows | [Q][W] row y0-1 | [Q][W] row y0+TY |
  //                       [Q][TY][4] wrapped columns of the tile rows | [Q][4] | [Q][4] of the halo rows
  static constexpr int pad32(int f) { return (f + 31) / 32 * 32; }  // 128-byte granules (TMA destination)
  static constexpr int MAIN_F = Q * TY * W, ROW_F = Q * W, ROW_PAD_F = pad32(ROW_F), PM_F = Q * TY * 4,
                       PM_PAD_F = pad32(PM_F), PR_F = Q * 4, PR_PAD_F = pad32(PR_F);
  static constexpr int O_RM = pad32(MAIN_F), O_RP = O_RM + ROW_PAD_F, O_PM = O_RP + ROW_PAD_F, O_PRM = O_PM + PM_PAD_F,
                       O_PRP = O_PRM + PR_PAD_F, END_F = O_PRP + PR_PAD_F;
  static constexpr uint32_t TMA_BYTES = (MAIN_F + 2 * ROW_F) * 4, TMA_EDGE_BYTES = (PM_F + 2 * PR_F) * 4;
  static constexpr int FL_MAIN = 0, FL_YM = TY * TX, FL_YP = FL_YM + TX, FL_XM = FL_YP + TX, FL_XP = FL_XM + TY;
  static constexpr uint32_t FLAG_OFF = END_F * 4, STAGE_BYTES = FLAG_OFF + 896;
  static constexpr size_t RING_BYTES = 4 * 3 * PLANE * 4;
  static constexpr size_t SMEM = (size_t)NS * STAGE_BYTES + RING_BYTES + 64;
  static_assert(WORKERS == 256 && TX % 64 == 0 && TY * TX == 512, "8 worker warps, 2 cells per thread, 32 x 16 B of flags");
  static_assert(FL_XP + TY <= 896 && STAGE_BYTES % 128 == 0, "flag region");
  static_assert(SMEM <= 227 * 1024, "shared memory");
};

namespace {

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
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];" ::"l"(map), "r"(c0), "r"(c1),
               "r"(c2), "r"(c3)
               : "memory");
}
#ifndef HHRR_PF
#define HHRR_PF 0
#endif
// register reallocation between warpgroups: 256 * 192 + 128 * 96 = 384 * 160 (the launch allocation)
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// uhat of plane `it` is published: one arrival per warp, waited for one iteration later (split phase)
__device__ __forceinline__ void pub_arrive(uint32_t pub0, int it) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(pub0 + 8 * (it & 1));
}
__device__ __forceinline__ void pub_wait(uint32_t pub0, int it) { mbar_wait(pub0 + 8 * (it & 1), (it >> 1) & 1); }

// store of the 27 post-collision values of cell (x,y,z), moved along y and z only, with rule R12
__device__ __forceinline__ void push_store_yz(const Dom& dm, float* __restrict__ fout, int x, int y, int z,
                                              const float (&o)[Q]) {
  bool fym, fyp, fzm, fzp;
  const int ym = wrap_axis(y - 1, dm.ny, dm.mode[1], fym), yp = wrap_axis(y + 1, dm.ny, dm.mode[1], fyp);
  const int zm = wrap_axis(z - 1, dm.nz, dm.mode[2], fzm), zp = wrap_axis(z + 1, dm.nz, dm.mode[2], fzp);
  const int64_t nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
#pragma unroll
  for (int i = 0; i < Q; ++i) {
    const int cy = dir_cy(i), cz = dir_cz(i);
    int ty = cy < 0 ? ym : (cy > 0 ? yp : y);
    int tz = cz < 0 ? zm : (cz > 0 ? zp : z);
    // a population leaving through a mirror plane returns to the same cell, component reversed
    const bool ry = (cy < 0 && fym) || (cy > 0 && fyp), rz = (cz < 0 && fzm) || (cz > 0 && fzp);
    if (ry) ty = y;
    if (rz) tz = z;
    const int io = ry ? (rz ? dir_flip(i, false, true, true) : dir_flip(i, false, true, false))
                      : (rz ? dir_flip(i, false, false, true) : i);
    fout[(int64_t)io * dm.n + tz * nxy + ty * nx + x] = o[i];
  }
}

}  // namespace

template <class C>
// 160 registers per thread at launch, re-divided into 192 per worker and 96 per aux / producer thread (the worker
// code needs about 190: 176 spills twelve registers and costs 3.5 %).  Registers are allocated per SM sub-partition:
// each holds three of the block's warps, 15 360 of its 16 384 registers, so the 4096 registers the block leaves free
// on an SM are 4 x 1024 -- nothing above 32 registers per thread is ever resident beside it.
__global__ void __maxnreg__(160)
    fused_xpull_kernel(const __grid_constant__ WsArgs a, const __grid_constant__ CUtensorMap map_main,
                       const __grid_constant__ CUtensorMap map_row, const __grid_constant__ CUtensorMap map_pm,
                       const __grid_constant__ CUtensorMap map_pr) {
  constexpr int TX = C::TX, TY = C::TY, NS = C::NS, W = C::W, WORKERS = C::WORKERS, AUX = C::AUX, SX = C::SX,
                PLANE = C::PLANE, HALO = C::HALO, HSLOTS = C::HSLOTS, MAIN_F = C::MAIN_F, PM_F = C::PM_F, O_RM = C::O_RM,
                O_RP = C::O_RP, O_PM = C::O_PM, O_PRM = C::O_PRM, O_PRP = C::O_PRP, FL_MAIN = C::FL_MAIN, FL_YM = C::FL_YM,
                FL_YP = C::FL_YP, FL_XM = C::FL_XM;
  constexpr uint32_t TMA_BYTES = C::TMA_BYTES, TMA_EDGE_BYTES = C::TMA_EDGE_BYTES, FLAG_OFF = C::FLAG_OFF,
                     STAGE_BYTES = C::STAGE_BYTES;
  constexpr size_t RING_BYTES = C::RING_BYTES;
  extern __shared__ __align__(128) unsigned char smem[];
  float(*ring)[3][PLANE] = reinterpret_cast<float(*)[3][PLANE]>(smem + (size_t)NS * STAGE_BYTES);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)NS * STAGE_BYTES + RING_BYTES);
  const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NS), pub0 = smem_u32(bars + 2 * NS);

  const Dom& dm = a.dm;
  const int tid = threadIdx.x;
  // Launch order: the tiles come in groups of a.group (one per SM); a group's blocks are ordered chunk by
  // chunk, so the block that takes chunk c+1 of a tile starts as the one that took chunk c ends -- the two
  // halo planes the chunks share are then still in L2 instead of being read from DRAM a second time.
  const int ntx = dm.nx / TX, ntiles = ntx * (dm.ny / TY);
  const int per_group = a.group * a.nch, grp = blockIdx.x / per_group, rem = blockIdx.x - grp * per_group;
  const int gsize = min(a.group, ntiles - grp * a.group);  // the last group may be short
  const int chunk = rem / gsize, tile = grp * a.group + (rem - chunk * gsize);
  const int x0 = (tile % ntx) * TX, y0 = (tile / ntx) * TY;
  const int z0 = chunk * a.zchunk, z1 = min(dm.nz, z0 + a.zchunk);
  const int64_t n = dm.n, nx = dm.nx, nxy = (int64_t)dm.nx * dm.ny;
  // Region split (Listing 2; R20): a block none of whose cells lies in an FSI box
  // holds BULK cells only -- sigma = 1, d = 1, no wall model -- so its collision is purely local: it loads
  // no halo rows, no flag bytes and no overlap planes, publishes no uhat, and its aux warps only keep the
  // barriers turning.  Everything else (pipeline, moments, collision, stores) is the code below.
  bool bulk = a.fsi.n > 0;
  for (int b = 0; b < a.fsi.n; ++b) {
    const Box& q = a.fsi.b[b];
    if (q.x0 < x0 + TX && q.x1 > x0 && q.y0 < y0 + TY && q.y1 > y0 && q.z0 < z1 && q.z1 > z0 && q.x1 > q.x0 &&
        q.y1 > q.y0 && q.z1 > q.z0)
      bulk = false;
  }
  const int pfirst = bulk ? z0 : z0 - 1;   // planes pfirst .. plast are loaded; the loops run to z1 (collide z1-1)
  const int plast = bulk ? z1 - 1 : z1;
  // tiles at the periodic x boundary: the 4 columns beyond it come from the other side (nx >= 128: one side only)
  const bool edge_l = x0 == 0, edge_r = x0 + TX == dm.nx, edge = edge_l || edge_r;
  const int px = edge_l ? dm.nx - 4 : 0;  // first wrapped column

  bool fym, fyp, okh;
  const int ym = virt_ws(y0 - 1, dm.ny, dm.mode[1], fym, okh), yp = virt_ws(y0 + TY, dm.ny, dm.mode[1], fyp, okh);

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(full0 + 8 * s, 2);  // TMA issue (+ its bytes) and the flag bytes
      mbar_init(empty0 + 8 * s, (WORKERS + AUX) / 32);
    }
    for (int s = 0; s < 2; ++s) mbar_init(pub0 + 8 * s, (WORKERS + AUX) / 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if (tid >= WORKERS) reg_dec<96>(); else reg_inc<192>();

  if (tid >= WORKERS + AUX) {
    // ------------------------------------------------------------------ producer: one lane issues TMA
    const int lane = tid & 31;
    const int xl = edge_l ? dm.nx - 1 : x0 - 1, xr = edge_r ? 0 : x0 + TX;  // real x of the halo columns
    for (int p = pfirst; p <= plast; ++p) {
      const int it = p - pfirst, s = it % NS, k = it / NS;
      if (HHRR_PF >= 0 && lane == 0 && p + HHRR_PF <= plast && (HHRR_PF > 0 || k > 0)) {
        bool f2_, ok2_;
        const int zq = virt_ws(p + HHRR_PF, dm.nz, dm.mode[2], f2_, ok2_);
        tma_prefetch_4d(&map_main, x0 - 4, y0, zq, 0);
        if (!bulk) {
          tma_prefetch_4d(&map_row, x0 - 4, ym, zq, 0);
          tma_prefetch_4d(&map_row, x0 - 4, yp, zq, 0);
        }
      }
      if (k > 0) mbar_wait(empty0 + 8 * s, (k - 1) & 1);
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const uint32_t bar = full0 + 8 * s;
      unsigned char* stb = smem + (size_t)s * STAGE_BYTES;
      if (bulk) {  // tile rows (and their wrapped columns) only
        if (lane == 0) {
          const uint32_t st = smem_u32(stb);
          mbar_expect_tx(bar, edge ? (MAIN_F + PM_F) * 4 : MAIN_F * 4);
          tma_load_4d(st, &map_main, x0 - 4, y0, zr, 0, bar);
          if (edge) tma_load_4d(st + 4 * O_PM, &map_pm, px, y0, zr, 0, bar);
          mbar_arrive(bar);
        }
        continue;
      }
      if (lane == 0) {
        const uint32_t st = smem_u32(stb);
        mbar_expect_tx(bar, edge ? TMA_BYTES + TMA_EDGE_BYTES : TMA_BYTES);
        tma_load_4d(st, &map_main, x0 - 4, y0, zr, 0, bar);  // columns outside the lattice arrive as zeros
        tma_load_4d(st + 4 * O_RM, &map_row, x0 - 4, ym, zr, 0, bar);
        tma_load_4d(st + 4 * O_RP, &map_row, x0 - 4, yp, zr, 0, bar);
        if (edge) {
          tma_load_4d(st + 4 * O_PM, &map_pm, px, y0, zr, 0, bar);
          tma_load_4d(st + 4 * O_PRM, &map_pr, px, ym, zr, 0, bar);
          tma_load_4d(st + 4 * O_PRP, &map_pr, px, yp, zr, 0, bar);
        }
      }
      // flag bytes of the same cells: 8 rows x 64 B + 2 halo rows as 16-byte loads, the columns bytewise
      const uint8_t* fz0 = a.flags + nxy * zr;
      unsigned char* flb = stb + FLAG_OFF;
      constexpr int L16 = TX / 16;  // 16-byte pieces per row; the two halo rows take 2 * L16 <= 16 lanes
      const uint4 vmain = __ldg(reinterpret_cast<const uint4*>(fz0 + (x0 + (lane % L16) * 16) + nx * (y0 + lane / L16)));
      uint4 vrow = make_uint4(0, 0, 0, 0);
      uint8_t vcol = 0;
      if (lane < 2 * L16) vrow = __ldg(reinterpret_cast<const uint4*>(fz0 + (x0 + (lane % L16) * 16) + nx * ((lane / L16) ? yp : ym)));
      if (lane >= 16 && lane < 16 + 2 * TY) {
        const int h = lane - 16, right = h / TY, row = h % TY;
        vcol = __ldg(fz0 + (right ? xr : xl) + nx * (y0 + row));
      }
      *reinterpret_cast<uint4*>(flb + FL_MAIN + (lane / L16) * TX + (lane % L16) * 16) = vmain;
      if (lane < 2 * L16) *reinterpret_cast<uint4*>(flb + FL_YM + (lane / L16) * TX + (lane % L16) * 16) = vrow;
      if (lane >= 16 && lane < 16 + 2 * TY) flb[FL_XM + (lane - 16)] = vcol;
      __syncwarp();
      if (lane == 0) mbar_arrive(bar);
    }
    return;
  }

  if (tid >= WORKERS) {
    // ------------------------------------------------------------------ aux warps: uhat of the xy halo
    // lane a owns halo cells a and a + AUX (if < HALO).  Per cell and per cx group: where population
    // (cx, k = 0) sits in a stage and the stride to k + 1 (column lx - cx of the 72-wide boxes, or the
    // wrapped columns at the periodic x boundary)
    if (bulk) {  // no halo: release the stages and keep the publication barrier in step
      for (int p = pfirst; p <= z1; ++p) {
        const int it = p - pfirst, s = it % NS, k2 = it / NS;
        if (it >= 2) pub_wait(pub0, it - 2);
        if (p <= plast) mbar_wait(full0 + 8 * s, k2 & 1);
        if ((tid & 31) == 0) {
          if (p <= plast) mbar_arrive(empty0 + 8 * s);
          mbar_arrive(pub0 + 8 * (it & 1));
        }
      }
      return;
    }
    // lane a owns halo cells a, a + AUX, ... (< HALO).  Per cell and per cx group: where population
    // (cx, k = 0) sits in a stage and the stride to k + 1 (column lx - cx of the wide boxes, or the wrapped
    // columns at the periodic x boundary)
    const int a0 = tid - WORKERS;
    int h_off[HSLOTS][3], h_str[HSLOTS][3], h_slot[HSLOTS], h_x[HSLOTS], h_y[HSLOTS], h_fl[HSLOTS];
    bool h_fy[HSLOTS], h_on[HSLOTS];
#pragma unroll
    for (int k = 0; k < HSLOTS; ++k) {
      const int hc = a0 + k * AUX;
      h_on[k] = hc < HALO;
      h_fy[k] = false;
      int lx, region, row = 0;  // region 0: tile rows, 1: row y0-1, 2: row y0+TY
      if (hc < 2 * TX) {
        const int top = hc / TX;
        lx = hc % TX;
        region = 1 + top;
        h_fl[k] = (top ? FL_YP : FL_YM) + lx;
        h_slot[k] = (top ? TY + 1 : 0) * SX + lx + 2;
        h_y[k] = top ? yp : ym;
        h_fy[k] = top ? fyp : fym;
      } else {
        const int h = (hc - 2 * TX) % (2 * TY), right = h / TY;
        row = h % TY;
        lx = right ? TX : -1;
        region = 0;
        h_fl[k] = FL_XM + right * TY + row;
        h_slot[k] = (row + 1) * SX + (right ? TX + 2 : 1);
        h_y[k] = y0 + row;
      }
      int xr = x0 + lx;
      h_x[k] = xr < 0 ? xr + dm.nx : (xr >= dm.nx ? xr - dm.nx : xr);
#pragma unroll
      for (int g = 0; g < 3; ++g) {  // cx = g - 1
        const int sx = x0 + lx - (g - 1);  // real (unwrapped) x of the source column
        if (sx >= 0 && sx < dm.nx) {
          const int col = 4 + lx - (g - 1);
          const int pstride = region == 0 ? TY * W : W;
          const int base = region == 0 ? row * W : (region == 1 ? O_RM : O_RP);
          h_off[k][g] = base + col;
          h_str[k][g] = pstride;
        } else {
          const int col = (sx < 0 ? sx + dm.nx : sx - dm.nx) - px;  // 0..3
          const int pstride = region == 0 ? TY * 4 : 4;
          const int base = region == 0 ? O_PM + row * 4 : (region == 1 ? O_PRM : O_PRP);
          h_off[k][g] = base + col;
          h_str[k][g] = pstride;
        }
      }
    }
    for (int p = pfirst; p <= z1; ++p) {
      const int it = p - pfirst, s = it % NS, k2 = it / NS;
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const int64_t zoff = nxy * zr;
      const float* st = reinterpret_cast<const float*>(smem + (size_t)s * STAGE_BYTES);
      const uint8_t* flb = smem + (size_t)s * STAGE_BYTES + FLAG_OFF;
      float(*slot)[PLANE] = ring[it & 3];
      // every worker is past the collision that read this ring slot; waiting from it = 2 on (not only
      // once the slot is reused) also keeps any arrival for plane it behind the completed phase it - 2
      if (it >= 2) pub_wait(pub0, it - 2);
      mbar_wait(full0 + 8 * s, k2 & 1);
#pragma unroll
      for (int k = 0; k < HSLOTS; ++k) {
        if (!h_on[k]) continue;
        float f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = st[h_off[k][dir_cx(i) + 1] + i * h_str[k][dir_cx(i) + 1]];
        const int64_t c = h_x[k] + nx * h_y[k] + zoff;
        float d, uB[3], rho, uh[3], drho, jx, jy, jz;
        solid_state_ws(a, flb[h_fl[k]], c, h_x[k], h_y[k], zr, d, uB);
        moments_rho_j(f, drho, jx, jy, jz);
        homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
        slot[0][h_slot[k]] = uh[0];
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

  // -------------------------------------------------------------------- workers, two x-adjacent cells each
  // The two cells of a thread run the same arithmetic: populations, moments, uhat, strain and the 27 results
  // live in register pairs (f2: .x = cell xa, .y = cell xa + 1) and go through FADD2 / FMUL2 / FFMA2.
  constexpr int HX = TX / 2;
  const int tx2 = tid % HX, ty = tid / HX;
  const int xa = x0 + 2 * tx2, yv = y0 + ty;  // cells (xa, yv) and (xa + 1, yv)
  const bool row_interior = yv > 0 && yv < dm.ny - 1;
  const int own_slot = (ty + 1) * SX + 2 * tx2 + 2;
  const int own_off = ty * W + 4 + 2 * tx2;   // + i * TY * W: population i of cell xa, unshifted column
  const int own_fl = ty * TX + 2 * tx2;
  const int64_t own_xy = xa + nx * yv;
  // the one lane of a boundary tile whose x neighbour column is a wrapped one
  const bool patch_l = edge_l && tx2 == 0, patch_r = edge_r && tx2 == HX - 1;
  const int patch_off = O_PM + ty * 4 + (patch_l ? 3 : 0);

  MomentsT<f2> mcur = {}, mnext = {};
  f2 rho_c = mk2(1.f, 1.f), rho_n = mk2(1.f, 1.f), uh_c[3] = {}, uh_n[3] = {};
  uint16_t fl_c = 0, fl_n = 0;  // flag bytes of the two cells
  char* dst = reinterpret_cast<char*>(a.fout) + 4 * (own_xy + nxy * z0);
  const int64_t zstride_b = 4 * nxy;

  for (int p = pfirst; p <= z1; ++p) {
    const int it = p - pfirst, s = it % NS, k2 = it / NS;
    if (p <= plast) {
      bool fz, okz;
      const int zr = virt_ws(p, dm.nz, dm.mode[2], fz, okz);
      const int64_t c = own_xy + nxy * zr;
      const float* st = reinterpret_cast<const float*>(smem + (size_t)s * STAGE_BYTES);
      float(*slot)[PLANE] = ring[it & 3];
      mbar_wait(full0 + 8 * s, k2 & 1);
      const uint16_t flw = bulk ? (uint16_t)(HHRR_BULK | (HHRR_BULK << 8))
                                : *reinterpret_cast<const uint16_t*>(smem + (size_t)s * STAGE_BYTES + FLAG_OFF + FL_MAIN + own_fl);
      f2 f[Q];
#pragma unroll
      for (int i = 0; i < Q; ++i) {  // population i of cell x sits at column x - cx (x-pull)
        const float* q = st + i * (TY * W) + own_off - dir_cx(i);
        if (dir_cx(i) == 0)
          f[i].v = *reinterpret_cast<const float2*>(q);
        else
          f[i] = mk2(q[0], q[1]);
      }
      if (edge) {
        if (patch_l) {
#pragma unroll
          for (int i = 0; i < Q; ++i)
            if (dir_cx(i) == 1) f[i].v.x = st[patch_off + i * (TY * 4)];   // cx = +1 from x = nx-1
        }
        if (patch_r) {
#pragma unroll
          for (int i = 0; i < Q; ++i)
            if (dir_cx(i) == -1) f[i].v.y = st[patch_off + i * (TY * 4)];  // cx = -1 from x = 0
        }
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * s);  // this warp has read its part of the stage
      const bool keep = p >= z0 && p < z1;
      // porosity and solid velocity of the two cells (plain fluid: d = 1, u^B = 0)
      f2 d = mk2(1.f, 1.f), uB[3] = {};
      if (type_has_solid_state(flw & TYPE_MASK) || type_has_solid_state((flw >> 8) & TYPE_MASK)) {
        float d0, d1, uB0[3], uB1[3];
        solid_state_ws(a, (uint8_t)(flw & 0xff), c, xa, yv, zr, d0, uB0);
        solid_state_ws(a, (uint8_t)(flw >> 8), c + 1, xa + 1, yv, zr, d1, uB1);
        d = mk2(d0, d1);
#pragma unroll
        for (int q = 0; q < 3; ++q) uB[q] = mk2(uB0[q], uB1[q]);
      }
      f2 rho, uh[3];
      if (keep) {
        mnext = moments_all(f);
        homogenised_velocity(a.ph, mnext.drho, mnext.jx, mnext.jy, mnext.jz, d, uB, rho, uh);
        rho_n = rho;
        uh_n[0] = uh[0]; uh_n[1] = uh[1]; uh_n[2] = uh[2];
        fl_n = flw;
      } else {
        f2 drho, jx, jy, jz;
        moments_rho_j(f, drho, jx, jy, jz);
        homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
      }
      if (!bulk) {
        *reinterpret_cast<float2*>(&slot[0][own_slot]) = uh[0].v;
        *reinterpret_cast<float2*>(&slot[1][own_slot]) = uh[1].v;
        *reinterpret_cast<float2*>(&slot[2][own_slot]) = fz ? (-uh[2]).v : uh[2].v;
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
      f2 S[6] = {}, sigma = mk2(cell_sigma(a.ph, (uint8_t)(fl_c & 0xff)), cell_sigma(a.ph, (uint8_t)(fl_c >> 8)));
      if (!bulk) {
        const int o = own_slot;
        f2 dxu[3], dyu[3], dzu[3];  // central differences (times 2) of uhat component q along x, y, z
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          // x: the pair's own values are in registers (a collided plane is never a reflected one)
          dxu[q] = mk2(uh_c[q].v.y, s0[q][o + 2]) - mk2(s0[q][o - 1], uh_c[q].v.x);
          dyu[q] = f2{*reinterpret_cast<const float2*>(&s0[q][o + SX])} - f2{*reinterpret_cast<const float2*>(&s0[q][o - SX])};
          dzu[q] = f2{*reinterpret_cast<const float2*>(&sp[q][o])} - f2{*reinterpret_cast<const float2*>(&sm[q][o])};
        }
        S[0] = 0.5f * dxu[0];
        S[1] = 0.5f * dyu[1];
        S[2] = 0.5f * dzu[2];
        S[3] = 0.25f * (dyu[0] + dxu[1]);
        S[4] = 0.25f * (dzu[0] + dxu[2]);
        S[5] = 0.25f * (dzu[1] + dyu[2]);
      }
      if (fl_c & (WM_VALID | (WM_VALID << 8))) {  // wall-model strain, sigma = 0 (rare)
        const int64_t c = own_xy + nxy * z;
        if (fl_c & WM_VALID) {
#pragma unroll
          for (int q = 0; q < 6; ++q) S[q].v.x = __ldg(a.wm_s + (int64_t)q * n + c);
          sigma.v.x = 0.f;
        }
        if (fl_c & (WM_VALID << 8)) {
#pragma unroll
          for (int q = 0; q < 6; ++q) S[q].v.y = __ldg(a.wm_s + (int64_t)q * n + c + 1);
          sigma.v.y = 0.f;
        }
      }
      f2 out[Q];
      collide(a.ph, mcur, rho_c, uh_c, S, sigma, out);
      if (row_interior && z > 0 && z < dm.nz - 1) {  // no wrap, no reflection: constant offsets, aligned pairs
#pragma unroll
        for (int i = 0; i < Q; ++i) *reinterpret_cast<float2*>(dst + a.push_b[i]) = out[i].v;
      } else {
        float o0[Q], o1[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) {
          o0[i] = out[i].v.x;
          o1[i] = out[i].v.y;
        }
        push_store_yz(dm, a.fout, xa, yv, z, o0);
        push_store_yz(dm, a.fout, xa + 1, yv, z, o1);
      }
      dst += zstride_b;
    }
    if (p >= z0) {
      mcur = mnext; rho_c = rho_n; fl_c = fl_n;
      uh_c[0] = uh_n[0]; uh_c[1] = uh_n[1]; uh_c[2] = uh_n[2];
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
  CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_256B;  // measured: 0.5-1 % faster than 128 B, 64 B slower
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float*>(base), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <class C>
static bool shape_tiles(const Dom& dm) {
  return dm.nx % C::TX == 0 && dm.nx >= 2 * C::TX && dm.ny % C::TY == 0;
}
using XpWide = XpCfg<128, 4>;
using XpTall = XpCfg<64, 8>;

bool xpull_supported(const Dom& dm) {
  return (shape_tiles<XpWide>(dm) || shape_tiles<XpTall>(dm)) && dm.mode[0] == HHRR_PERIODIC && encode_fn() != nullptr;
}

template <class C>
static cudaError_t launch_shape(hhrr_lattice* L, WsArgs& a) {
  const Dom& dm = L->dom;
  CUtensorMap m_main, m_row, m_pm, m_pr;
  if (!make_map(&m_main, L->fA, dm, C::W, C::TY) || !make_map(&m_row, L->fA, dm, C::W, 1) ||
      !make_map(&m_pm, L->fA, dm, 4, C::TY) || !make_map(&m_pr, L->fA, dm, 4, 1))
    return cudaErrorNotSupported;
  bool& attr_set = L->attr_xpull[C::TX == 128 ? 1 : 0];  // the attribute is per device: kept per lattice
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(fused_xpull_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  // with the grouped launch order the halo planes of a chunk are L2 hits: 22 planes without, 16 with the region split
  // z-chunk length: neighbouring tiles re-synchronise at every chunk start, and the halo rows / x-halo sectors they
  // share stay L2 hits only while they march within a few planes of each other.  Measured on config 5 with the
  // packed-fp32 workers (profiles/r02_k2_chunk_scan.md; bench.py --chunk-planes): 13-16 planes 4.01-4.03 ms, 18 planes
  // 4.06 ms, 22 planes 4.15 ms, 32 planes 4.51 ms (without clusters: 4.09 / 4.27 / 4.52 / 4.92 ms); with the region
  // split 12 planes 3.88 ms, 16 planes 3.92 ms; D3Q19 (19 populations per cell plane, three pipeline stages) 16 / 23 / 30 /
  // 40 / 52 / 73 planes 3.00 / 2.95 / 2.93 / 2.91 / 2.94 / 3.07 ms.  hhrr_set_launch_shape overrides.
  const int auto_planes = Q == 27 ? (a.fsi.n > 0 ? 12 : 16) : (a.fsi.n > 0 ? 22 : 40);
  if (!L->sm_count &&
      (cudaDeviceGetAttribute(&L->sm_count, cudaDevAttrMultiProcessorCount, L->device) != cudaSuccess || L->sm_count < 1))
    L->sm_count = 148;
  const int ntiles = (dm.nx / C::TX) * (dm.ny / C::TY);
  int nch = ws_zchunks(dm.nz, L->chunk_planes > 0 ? L->chunk_planes : auto_planes);
  if (L->chunk_planes <= 0 && (long long)ntiles * nch < 12LL * L->sm_count) {
    // A lattice of a few waves of blocks: the time is (waves of blocks) x (planes a block walks, its two overlap
    // planes included), and a last wave that is nearly empty costs as much as a full one.  Among chunk lengths
    // between 6 planes and twice the usual one take the cheapest, the one nearest the usual length among equals
    // (config 3, 256 x 128 x 128: 9 chunks, 576 blocks in 4 waves of 17 planes, instead of 8 x 64 = 512 in 4 of 18).
    long long best = -1;
    int best_n = nch;
    for (int c = 1; c <= dm.nz; ++c) {
      const int planes = (dm.nz + c - 1) / c;
      if (planes > 2 * auto_planes || planes < 6) continue;
      if ((dm.nz + planes - 1) / planes != c) continue;  // not a chunk count of its own
      const long long waves = ((long long)ntiles * c + L->sm_count - 1) / L->sm_count, cost = waves * (planes + 2);
      if (best < 0 || cost < best || (cost == best && abs(planes - auto_planes) < abs((dm.nz + best_n - 1) / best_n - auto_planes))) {
        best = cost;
        best_n = c;
      }
    }
    nch = best_n;
  }
  a.zchunk = (dm.nz + nch - 1) / nch;
  nch = (dm.nz + a.zchunk - 1) / a.zchunk;
  a.nch = nch;
  a.group = L->sm_count;  // one tile per SM and wave (one block per SM: shared memory)
  dim3 grid((unsigned)(ntiles * nch));
  // Two x-adjacent tiles form a thread-block cluster (no cluster barrier, no distributed shared memory): the pair
  // starts together on neighbouring SMs and asks L2 for the x-halo sectors it shares at the same time.  Measured
  // (profiles/r02_k2_chunk_scan.md): 4.09 -> 4.01 ms at 16-plane chunks, 3.99 -> 3.88 ms with the region split at 12,
  // and the cliff at longer chunks moves out (22 planes: 4.52 -> 4.15 ms); clusters of 4: 4.15 ms.
  const int cl = L->cluster > 0 ? L->cluster : 2;
  if (cl > 1 && grid.x % cl == 0 && a.group % cl == 0 && ntiles % cl == 0) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = C::SMEM;
    cfg.stream = L->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cl;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, fused_xpull_kernel<C>, a, m_main, m_row, m_pm, m_pr);
    L->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
  }
  fused_xpull_kernel<C><<<grid, C::THREADS, C::SMEM, L->stream>>>(a, m_main, m_row, m_pm, m_pr);
  L->launches++;
  return cudaGetLastError();
}

cudaError_t launch_fused_xpull(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  const Dom& dm = L->dom;
  if (!dm.xs || !xpull_supported(dm)) return cudaErrorNotSupported;
  WsArgs a;
  fill_ws_args(L, ph, bo, a);
  for (int i = 0; i < Q; ++i)  // y and z moves only: the x move is taken on the read side
    a.push_b[i] = 4LL * ((long long)i * dm.n + (long long)dir_cy(i) * dm.nx + (long long)dir_cz(i) * dm.nx * dm.ny);
  // Blocks that need the y halo rows (the FD strain) do better with 64 x 8 tiles (2 halo rows per 8), bulk
  // blocks (region split) with 128 x 4 (fewer x-halo sectors re-read): measured on config 5,
  // 4.06 / 4.39 ms without the split and 4.16 / 3.98 ms with it.
  bool wide = shape_tiles<XpWide>(dm) && (a.fsi.n > 0 || !shape_tiles<XpTall>(dm));
  return wide ? launch_shape<XpWide>(L, a) : launch_shape<XpTall>(L, a);
}

}  // namespace hhrr
