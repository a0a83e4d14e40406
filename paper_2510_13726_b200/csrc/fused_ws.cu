// fused_ws.cu -- variant 2 of K2: the fused collide-stream kernel, warp-specialised.
//
// Same arithmetic and the same sliding window along z as fused.cu (Listing 3 line 3,
// PAPER.md:313; Eq. 6-14; S^FD of Eq. 10 from the time-n uhat of the six face neighbours),
// but the two halves of a cell update run in different warps of the block and are decoupled by
// a DEPTH-deep shared-memory ring, so DRAM loads never wait for the collision arithmetic:
//
//   producer warps : load the 27 populations of a cell (tile + one-cell xy halo) of plane p,
//                    reduce them to rho-1, uhat and the six second moments, write them into
//                    ring slot p % DEPTH, signal FULL[slot]; run up to DEPTH-3 planes ahead.
//   consumer warps : wait FULL for plane z+1, read the moments of plane z and the uhat of the
//                    six neighbours from the ring, collide, push-store 27 populations,
//                    signal EMPTY for the slot of plane z-1.
//
// Synchronisation is by named barriers (bar.arrive / bar.sync), one FULL and one EMPTY per slot.
#include <cstdlib>

#include "ws_common.cuh"

namespace hhrr {

template <int TX, int TY, int NPW, int DEPTH, int CPT = 2>
struct WsCfg {
  static constexpr int CELLS = TX * TY;            // cells of one plane of the tile
  static constexpr int CTHREADS = CELLS / CPT;     // consumer threads, CPT cells each (rows ty, ty + TY/CPT, ..)
  static constexpr int PWARPS = NPW + 1;            // NPW row-task warps + one warp for the x-halo columns
  static constexpr int THREADS = CTHREADS + PWARPS * 32;
  static constexpr int SX = TX + 2, SY = TY + 2;
  static constexpr int PLANE = SX * SY;            // padded uhat plane
  static constexpr int ROW_TASKS = TX / 32;        // warp-tasks per row
  static constexpr int RTASKS = ROW_TASKS * (TY + 2);  // interior rows + two halo rows
  static constexpr int TPW = RTASKS / NPW;         // row tasks per producer warp (fixed assignment)
  static constexpr int SLOT_FLOATS = 3 * PLANE + 7 * CELLS;
  static constexpr size_t SLOT_BYTES = SLOT_FLOATS * 4 + CELLS;  // + flags
  static constexpr size_t SLOT_STRIDE = (SLOT_BYTES + 15) / 16 * 16;
  static constexpr size_t SMEM = SLOT_STRIDE * DEPTH;
  static_assert(TX % 32 == 0 && 2 * TY <= 32 && TY % CPT == 0, "tile shape");
  static_assert(RTASKS % NPW == 0, "row tasks must divide evenly over the producer warps");
  static_assert(2 * DEPTH + 1 <= 16, "named barriers");
};

// per-lane description of one producer task; fixed over the z march
struct PTask {
  int64_t cxy;  // xr + nx*yr, or -1 if this lane has no cell in this task
  int xr, yr;
  int o;        // index into the padded uhat plane
  int ci;       // interior cell index, or -1 for halo cells
  bool fx, fy;  // reflected in x / y (mirror axes)
};

template <int TX, int TY>
__device__ __forceinline__ PTask make_task(const Dom& dm, int x0, int y0, int hx, int hy, bool active) {
  PTask t;
  bool okx, oky;
  t.xr = virt_ws(x0 + hx - 1, dm.nx, dm.mode[0], t.fx, okx);
  t.yr = virt_ws(y0 + hy - 1, dm.ny, dm.mode[1], t.fy, oky);
  t.cxy = (active && okx && oky) ? (int64_t)t.xr + (int64_t)dm.nx * t.yr : -1;
  t.o = hy * (TX + 2) + hx;
  t.ci = (hx >= 1 && hx <= TX && hy >= 1 && hy <= TY) ? (hy - 1) * TX + (hx - 1) : -1;
  return t;
}

template <int TX, int TY, int NPW, int DEPTH, int CPT_>
__global__ void __launch_bounds__(WsCfg<TX, TY, NPW, DEPTH, CPT_>::THREADS, 1)
    fused_ws_kernel(const __grid_constant__ WsArgs a) {
  using C = WsCfg<TX, TY, NPW, DEPTH, CPT_>;
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
    // warps 0..NPW-1 own TPW fixed row tasks each; warp NPW owns the two x-halo columns, so every
    // producer warp has ONE load phase per plane (a second, serial one would halve the plane rate)
    PTask tk[C::TPW];
#pragma unroll
    for (int k = 0; k < C::TPW; ++k) {
      const int t = pw + k * NPW;
      if (pw < NPW)
        tk[k] = make_task<TX, TY>(dm, x0, y0, (t % C::ROW_TASKS) * 32 + lane + 1, t / C::ROW_TASKS, true);
      else
        tk[k] = make_task<TX, TY>(dm, x0, y0, (lane / TY) ? TX + 1 : 0, lane % TY + 1, k == 0 && lane < 2 * TY);
    }
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
      auto produce = [&](const PTask& t) {
        if (t.cxy < 0) return;
        const int64_t c = t.cxy + zoff;
        const char* __restrict__ src = fin_b + 4 * c;
        float f[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) f[i] = __ldg(reinterpret_cast<const float*>(src + a.plane_b[i]));
        const uint8_t fl = __ldg(a.flags + c);
        float d, uB[3], rho, uh[3];
        solid_state_ws(a, fl, c, t.xr, t.yr, zr, d, uB);
        if (t.ci >= 0 && need_moments) {
          Moments m = moments_all(f);
          homogenised_velocity(a.ph, m.drho, m.jx, m.jy, m.jz, d, uB, rho, uh);
          moms[t.ci] = m.drho;
          moms[C::CELLS + t.ci] = m.mxx;
          moms[2 * C::CELLS + t.ci] = m.myy;
          moms[3 * C::CELLS + t.ci] = m.mzz;
          moms[4 * C::CELLS + t.ci] = m.mxy;
          moms[5 * C::CELLS + t.ci] = m.mxz;
          moms[6 * C::CELLS + t.ci] = m.myz;
          fls[t.ci] = fl;
        } else {
          float drho, jx, jy, jz;
          moments_rho_j(f, drho, jx, jy, jz);
          homogenised_velocity(a.ph, drho, jx, jy, jz, d, uB, rho, uh);
        }
        uhs[t.o] = t.fx ? -uh[0] : uh[0];
        uhs[C::PLANE + t.o] = t.fy ? -uh[1] : uh[1];
        uhs[2 * C::PLANE + t.o] = fz ? -uh[2] : uh[2];
      };
#pragma unroll
      for (int k = 0; k < C::TPW; ++k) produce(tk[k]);
      __syncwarp();
      bar_arrive(1 + s, C::THREADS);  // FULL[s]
      s = (s + 1 == DEPTH) ? 0 : s + 1;
    }
  } else {
    // ------------------------------------------------------------------ consumers
    constexpr int CPT = C::CELLS / C::CTHREADS, YSTEP = TY / CPT;
    const int tx = tid % TX, ty = tid / TX;
    const int xv = x0 + tx;
    const bool x_interior = xv > 0 && xv < dm.nx - 1;
    char* dst = reinterpret_cast<char*>(a.fout) + 4 * ((int64_t)xv + nx * (y0 + ty) + nxy * z0);
    const int64_t zstride_b = 4 * nxy, ystep_b = 4 * nx * YSTEP;
    bar_sync(1 + 0, C::THREADS);            // plane z0-1
    bar_sync(1 + (1 % DEPTH), C::THREADS);  // plane z0
    int sm = 0, sc = 1 % DEPTH, sp = 2 % DEPTH;
    for (int z = z0; z < z1; ++z) {
      bar_sync(1 + sp, C::THREADS);  // FULL for plane z+1
      const float* u0 = slot_uh(sc);
      const float* up = slot_uh(sp);
      const float* um = slot_uh(sm);
      const float* mo = slot_mom(sc);
      const uint8_t* flp = slot_fl(sc);
      const bool z_interior = z > 0 && z < dm.nz - 1;
#pragma unroll
      for (int k = 0; k < CPT; ++k) {
        const int yl = ty + k * YSTEP, yv = y0 + yl;
        if (!(xv < dm.nx && yv < dm.ny)) continue;
        const int ci = yl * TX + tx, o = (yl + 1) * C::SX + (tx + 1);
        const uint8_t fl = flp[ci];
        Moments m;
        m.drho = mo[ci];
        m.mxx = mo[C::CELLS + ci];
        m.myy = mo[2 * C::CELLS + ci];
        m.mzz = mo[3 * C::CELLS + ci];
        m.mxy = mo[4 * C::CELLS + ci];
        m.mxz = mo[5 * C::CELLS + ci];
        m.myz = mo[6 * C::CELLS + ci];
        m.jx = m.jy = m.jz = 0.f;  // not used by collide()
        const float rho = 1.f + m.drho;
        float uh[3] = {u0[o], u0[C::PLANE + o], u0[2 * C::PLANE + o]};
        float S[6], sigma = cell_sigma(a.ph, fl);
        if (fl & WM_VALID) {
          const int64_t c = xv + nx * yv + nxy * z;
#pragma unroll
          for (int q = 0; q < 6; ++q) S[q] = __ldg(a.wm_s + (int64_t)q * n + c);
          sigma = 0.f;
        } else {
          float dxu0 = u0[o + 1] - u0[o - 1], dxu1 = u0[C::PLANE + o + 1] - u0[C::PLANE + o - 1],
                dxu2 = u0[2 * C::PLANE + o + 1] - u0[2 * C::PLANE + o - 1];
          float dyu0 = u0[o + C::SX] - u0[o - C::SX], dyu1 = u0[C::PLANE + o + C::SX] - u0[C::PLANE + o - C::SX],
                dyu2 = u0[2 * C::PLANE + o + C::SX] - u0[2 * C::PLANE + o - C::SX];
          float dzu0 = up[o] - um[o], dzu1 = up[C::PLANE + o] - um[C::PLANE + o],
                dzu2 = up[2 * C::PLANE + o] - um[2 * C::PLANE + o];
          S[0] = 0.5f * dxu0;
          S[1] = 0.5f * dyu1;
          S[2] = 0.5f * dzu2;
          S[3] = 0.25f * (dyu0 + dxu1);
          S[4] = 0.25f * (dzu0 + dxu2);
          S[5] = 0.25f * (dzu1 + dyu2);
        }
        float o27[Q];
        collide(a.ph, m, rho, uh, S, sigma, o27);
        if (x_interior && z_interior && yv > 0 && yv < dm.ny - 1) {  // constant push offsets
          char* q = dst + k * ystep_b;
#pragma unroll
          for (int i = 0; i < Q; ++i) *reinterpret_cast<float*>(q + a.push_b[i]) = o27[i];
        } else {
          push_store(dm, a.fout, xv, yv, z, o27);
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

template <int TX, int TY, int NPW, int DEPTH, int CPT = 2>
static cudaError_t launch_ws_cfg(hhrr_lattice* L, const WsArgs& a0) {
  using C = WsCfg<TX, TY, NPW, DEPTH, CPT>;
  WsArgs a = a0;
  const Dom& dm = L->dom;
  bool& attr_set = L->attr_ws;  // the attribute is per device: kept per lattice
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(fused_ws_kernel<TX, TY, NPW, DEPTH, CPT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  int nch = ws_zchunks(dm.nz, 19);
  a.zchunk = (dm.nz + nch - 1) / nch;
  nch = (dm.nz + a.zchunk - 1) / a.zchunk;
  dim3 grid((dm.nx + TX - 1) / TX, (dm.ny + TY - 1) / TY, nch);
  fused_ws_kernel<TX, TY, NPW, DEPTH, CPT><<<grid, C::THREADS, C::SMEM, L->stream>>>(a);
  L->launches++;
  return cudaGetLastError();
}

void fill_ws_args(const hhrr_lattice* L, const PhysF& ph, const BodiesF& bo, WsArgs& a) {
  a.dm = L->dom;
  a.ph = ph;
  a.bo = bo;
  a.fsi = L->fsi;
  a.fin = L->fA;
  a.fout = L->fB;
  a.flags = L->flags;
  a.d = L->d;
  a.wm_u = L->wm_u;
  a.wm_s = L->wm_s;
  a.zchunk = L->dom.nz;
  const long long n = L->dom.n, nx = L->dom.nx, nxy = (long long)L->dom.nx * L->dom.ny;
  for (int i = 0; i < Q; ++i) {
    a.plane_b[i] = 4 * (i * n);
    a.push_b[i] = 4 * (i * n + dir_cx(i) + dir_cy(i) * nx + dir_cz(i) * nxy);
  }
}

// number of z-chunks: short chunks (~24 planes).  Blocks are dispatched in (x, y, z-chunk) order, so
// all SMs work on one slab of the lattice at a time and a tile's halo rows are still in L2 when its
// neighbour tile loads them; long chunks let neighbouring blocks drift apart (measured: 6.3 ms at 2
// chunks vs 5.6 ms at 16 on 768x384x364).  Cost: two extra planes loaded per chunk.
int ws_zchunks(int nz, int planes) {  // ~planes planes per chunk: measured optima on config 5 (profiles/)
  int nch = (nz + planes / 2) / planes;
  if (nch < 1) nch = 1;
  return nch;
}

cudaError_t launch_fused_ws(hhrr_lattice* L, const PhysF& ph, const BodiesF& bo) {
  WsArgs a;
  fill_ws_args(L, ph, bo, a);
  return launch_ws_cfg<64, 8, 20, 4>(L, a);
}

}  // namespace hhrr
