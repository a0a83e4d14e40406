// lattice.h -- internal state of an hhrr_lattice and the parameter blocks handed to kernels.
// CUDA path only; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hhrr.h"

namespace hhrr {

constexpr int Q = HHRR_Q;
constexpr int MAX_TAGS = HHRR_MAX_TAGS;
constexpr int64_t FORCE_HISTORY = 4096;  // ring of per-step force records
constexpr double BIG_PHI = 1.0e30;       // "no geometry here"

// flags byte per cell: bits 0-2 hhrr_cell_type, bits 3-6 element tag, bit 7 wall-model state valid
constexpr uint8_t TYPE_MASK = 0x07;
constexpr int TAG_SHIFT = 3;
constexpr uint8_t TAG_MASK = 0x0f;
constexpr uint8_t WM_VALID = 0x80;
// Internal value of the type bits: a FRONTIER cell that belongs to the wall-model set W (reading R13).  The ABI
// reports it as HHRR_FRONTIER; the flag byte of the NEXT step's geometry (written ahead of time) thereby tells
// the wall-model kernel of THIS step which cells will consume the state it writes.
constexpr int T_FRONTIER_W = 6;
__host__ __device__ inline int public_type(int t) { return t == T_FRONTIER_W ? (int)HHRR_FRONTIER : t; }

struct Dom {
  int nx, ny, nz;
  int mode[3];
  int64_t n;
  // storage of the populations: xs = 0 "push" (post-stream: plane i holds f_i(x,y,z));
  // xs = 1 "x-pull / yz-push": plane i holds g_i(x,y,z) = f_i(x + c_ix, y, z), i.e. the post-collision
  // value already moved along y and z but not yet along x (periodic x axis only).  pop_index() hides it.
  int xs;
};

// rigid bodies, fp32 copy for the collide kernel, fp64 for wall model / force
struct BodiesF {
  float c[MAX_TAGS][3], w[MAX_TAGS][3], v[MAX_TAGS][3];
};
struct BodiesD {
  double c[MAX_TAGS][3], w[MAX_TAGS][3], v[MAX_TAGS][3];
};

struct PhysF {
  float tau0, sigma, smag18;  // smag18 = 18 C_S^2 (Eq. 14 closed form, R6)
  float g[3];
  float fr_u[3];
};

struct Box {  // half-open cell box
  int x0, x1, y0, y1, z0, z1;
};

struct Boxes {  // FSI region (hhrr_set_fsi_region); n = 0: the whole lattice
  int n;
  Box b[HHRR_MAX_FSI_BOXES];
};

struct RotorDev {
  const float* sdf;
  const uint8_t* tag;
  int gx, gy, gz;
  double spacing, origin[3], centre[3], axis[3];
};

// counters living in device memory
struct Counters {
  int wall_count, force_count;
  int wall_static, force_static;  // list prefix owned by cells outside the rotor box
  int overflow;
  int nonfinite;
  int region_violation;  // a cell that is not plain fluid lies outside the FSI region
  int pad[1];
};

}  // namespace hhrr

struct hhrr_lattice {
  hhrr_params p;
  hhrr::Dom dom;
  cudaStream_t stream;
  // Side stream (lowest priority, which is also the default's) and its ordering events.  Two things are queued there
  // behind the launch of the collide-stream kernel: the WHOLE porosity update of the next step (geometry.cu:
  // launch_geometry_ahead; a function of the step count only) into the alternate geometry set, and the
  // force / torque collection of the step just streamed (wallmodel.cu: launch_forces), which only reads.  They get SMs
  // from the collide-stream kernel's last wave of blocks on -- the block scheduler gives a grid of equal priority no SM
  // before the last block of the grid ahead of it is placed -- and then share the machine with the wall model.
  cudaStream_t side;
  cudaEvent_t ev_pre, ev_k1, ev_k2, ev_side, ev_f[2];  // ev_f[n & 1]: force kernel of step n has read its populations
  int64_t ahead_step;   // step whose geometry the alternate set holds (or is being written with); -1: none
  bool side_busy;       // something was queued on the side stream since the main stream last waited for it
  bool lookahead;       // hhrr_set_lookahead
  int device;
  // device arrays (inside the caller's workspace)
  float *fA, *fB;           // 27 planes each: post-stream populations minus weights
  uint8_t* flags;           // N
  float* d;                 // N porosity (read for FRONTIER cells only)
  // alternate geometry set (flags, porosity, lists, counters): written ahead for the next step, then swapped in
  uint8_t* alt_flags;
  float* alt_d;
  int32_t* alt_wall_idx;
  double* alt_wall_y1n;
  int32_t* alt_force_idx;
  hhrr::Counters* alt_counters;
  double* phi;              // N signed distance of the last geometry
  uint8_t* below;           // N: phi < eps/2
  uint8_t* tag_prov;        // N: provisional tag of geometry pass 1
  uint8_t *rowflag, *rowflag_static;  // ny*nz: row may hold a cell with phi < eps/2
  uint8_t* rowact[2];       // ny*nz each: row held a cell within ~3.9 cells of the rotor at the last even / odd step (geometry.cu)
  int32_t* rowlist;         // ny*nz: rows of the rotor box to evaluate this step
  int* n_rows;
  bool band_ok;             // the rotor moves less than a cell per step: the row band applies
  float* phi_static;        // N
  uint8_t* tag_static;      // N
  float* d_override;        // N
  float* uhat;              // 3N (two-pass variant, init, tests)
  double* wm_utau;          // N
  float* wm_u;              // 3N
  float* wm_s;              // 6N
  int32_t* wall_idx;        // cap_list
  double* wall_y1n;         // 3*cap_list (AoS)
  double* wall_samp;        // 6*cap_list: v_s and v(x_w) per wall cell, between the two phases of K3
  int32_t* force_idx;       // cap_list
  hhrr::Counters* counters; // 1
  double* force;            // FORCE_HISTORY * MAX_TAGS * 3
  double* torque;           // FORCE_HISTORY * MAX_TAGS * 3, about each element's body centre
  float* rot_sdf;
  uint8_t* rot_tag;
  int64_t rot_nodes_cap;
  int64_t cap_list;
  // host state
  bool has_static, has_tag_static, has_override, has_fringe, has_rotor, wm_enabled;
  int fr_x0, fr_x1;
  double fr_u[3];
  hhrr_rotor_desc rot;  // sdf/tag pointers nulled
  hhrr::Box rot_box;
  hhrr::Boxes fsi;
  int wall_function;  // 0 truncated Spalding (Eq. 18), 1 Musker
  int wm_slip, wm_shear;  // second readings of PAPER.md:314 / :324 (hhrr_set_wall_model_variant), default 0
  hhrr::BodiesD bodies;
  bool geometry_dirty;     // full-domain geometry pass needed
  bool geometry_current;   // geometry(step) evaluated
  int64_t step;
  int variant;       // requested kernel variant; dom.xs says how the populations are stored for it
  int64_t launches;
  int chunk_planes, cluster;  // hhrr_set_launch_shape: planes per z-chunk / tiles per cluster of the default kernel (0: automatic)
  int sm_count;          // of L->device (0: not yet asked)
  bool attr_xpull[2], attr_ws;  // dynamic shared-memory attribute set on L->device for the fused kernels
  // optional CUDA-event timing of the collide-stream kernel (hhrr_set_timing)
  bool timing;
  int ev_n;
  cudaEvent_t ev[2 * 1024];
};

// ---- kernel launchers (one per translation unit) ---------------------------------------
namespace hhrr {
// api.cu: records the thread-local message hhrr_last_error() returns and hands `code` back (for entry points that live
// in other translation units)
int set_error(int code, const char* fmt, ...);
// geometry.cu (compiled with -fmad=false: operation order is part of the definition)
cudaError_t launch_geometry(hhrr_lattice* L, bool full);
// collide.cu
cudaError_t launch_fill_rest(hhrr_lattice* L);
cudaError_t launch_init(hhrr_lattice* L, const float* d_rho, const float* d_u, int with_neq);
cudaError_t launch_collide_stream(hhrr_lattice* L);
cudaError_t launch_geometry_ahead(hhrr_lattice* L);     // geometry(step + 1) into the alternate set, side stream
void swap_geometry_sets(hhrr_lattice* L);
cudaError_t launch_moments(hhrr_lattice* L, float* d_rho, float* d_v);
cudaError_t launch_check_finite(hhrr_lattice* L);
bool xpull_supported(const Dom& dm);                    // fused_xpull.cu: variant 5 can run this lattice
cudaError_t launch_restore(hhrr_lattice* L, int xs);    // re-store the populations of buffer A with x-shift xs
// wallmodel.cu
cudaError_t launch_wall_model(hhrr_lattice* L);                 // K3 on the main stream
cudaError_t launch_merge_valid(hhrr_lattice* L);                // WM_VALID of the geometry written ahead
cudaError_t launch_forces(hhrr_lattice* L, cudaStream_t s);     // K4 (reads only) on stream s
}  // namespace hhrr
