// ws_common.cuh -- pieces shared by the fused collide-stream kernels
// (fused_xpull.cu: TMA-fed, x-pull / yz-push storage; fused_ws.cu: warp-specialised, LDG-fed, post-stream storage).
// CUDA path only; shares nothing with oracle/.
#pragma once
#include "cell_model.cuh"

namespace hhrr {

struct WsArgs {
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
  int nch, group;        // variant 5: z-chunks per tile column; tiles per launch-order group (see fused_xpull.cu)
  Boxes fsi;             // FSI region (n = 0: whole lattice); variant 5: blocks outside it take the bulk path
  long long plane_b[Q];  // 4 * i * n                            (byte offsets, warp-uniform)
  long long push_b[Q];   // 4 * (i * n + cx + cy*nx + cz*nx*ny)
};

__device__ __forceinline__ void bar_sync(int id, int count) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int count) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory");
}

__device__ __forceinline__ int virt_ws(int v, int n, int mode, bool& flip, bool& ok) {
  flip = false;
  ok = (v >= -1 && v <= n);
  if (!ok) return 0;
  return wrap_axis(v, n, mode, flip);
}

__device__ __forceinline__ void solid_state_ws(const WsArgs& a, uint8_t fl, int64_t c, int x, int y, int z,
                                               float& d, float uB[3]) {
  int type = fl & TYPE_MASK;
  d = 1.f;
  uB[0] = uB[1] = uB[2] = 0.f;
  if (type_has_solid_state(type)) {
    d = type_is_frontier(type) ? __ldg(a.d + c) : 0.f;
    solid_velocity(a.ph, a.bo, fl, x, y, z, uB);
    if (fl & WM_VALID) {
      uB[0] += __ldg(a.wm_u + c);
      uB[1] += __ldg(a.wm_u + a.dm.n + c);
      uB[2] += __ldg(a.wm_u + 2 * a.dm.n + c);
    }
  }
}

void fill_ws_args(const hhrr_lattice* L, const PhysF& ph, const BodiesF& bo, WsArgs& a);
int ws_zchunks(int nz, int planes);

}  // namespace hhrr
