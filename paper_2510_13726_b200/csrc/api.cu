// api.cu -- the C ABI of include/hhrr.h: argument checking, workspace carving, host<->device
// staging and the per-step launch sequence of Listing 3.
// CUDA path only; shares nothing with oracle/.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

#include "cell_model.cuh"

using namespace hhrr;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
int cuda_fail(cudaError_t e, const char* what) {
  return fail(HHRR_E_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define CU(call)                                   \
  do {                                             \
    cudaError_t e_ = (call);                       \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// Every entry point that takes a lattice works on the lattice's device, whatever device is current in the
// calling thread, and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(const hhrr_lattice* L) { enter(L ? L->device : -1); }
  explicit DeviceGuard(int device) { enter(device); }
  void enter(int device) {
    if (device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != device) cudaSetDevice(device);
    else prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

bool params_ok(const hhrr_params* p) {
  if (!p) return false;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1) return false;
  double n = (double)p->nx * p->ny * p->nz;
  if (n > 2.0e9) return false;  // int32 cell indices in the compact lists
  for (int a = 0; a < 3; ++a)
    if (p->mode[a] != HHRR_PERIODIC && p->mode[a] != HHRR_MIRROR) return false;
  if (!(p->tau0 > 0.5) || !(p->sigma >= 0.0 && p->sigma <= 1.0) || !(p->smagorinsky_cs >= 0.0)) return false;
  if (!(p->eps_cells > 0.0) || !(p->kappa > 0.0) || !(p->E > 0.0) || p->newton_max_iter < 0) return false;
  if (!(p->sampling_distance > 0.0)) return false;
  return true;
}

int64_t list_capacity(int64_t n) { return std::min<int64_t>(n, std::max<int64_t>(1 << 20, n / 4)); }

// Carves the workspace; with base == nullptr only sizes it.
struct Carver {
  char* base;
  size_t off = 0;
  template <class T>
  T* take(int64_t count) {
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += align_up(sizeof(T) * (size_t)count);
    return p;
  }
};

size_t carve(hhrr_lattice* L, const hhrr_params* p, int64_t rotor_nodes, char* base) {
  Carver c{base};
  int64_t n = (int64_t)p->nx * p->ny * p->nz;
  int64_t cap = list_capacity(n);
  float* fA = c.take<float>(Q * n);
  float* fB = c.take<float>(Q * n);
  uint8_t* flags = c.take<uint8_t>(n);
  float* d = c.take<float>(n);
  double* phi = c.take<double>(n);
  uint8_t* below = c.take<uint8_t>(n);
  uint8_t* tag_prov = c.take<uint8_t>(n);
  uint8_t* rowflag = c.take<uint8_t>((int64_t)p->ny * p->nz);
  uint8_t* rowflag_static = c.take<uint8_t>((int64_t)p->ny * p->nz);
  uint8_t* rowact0 = c.take<uint8_t>((int64_t)p->ny * p->nz);
  uint8_t* rowact1 = c.take<uint8_t>((int64_t)p->ny * p->nz);
  int32_t* rowlist = c.take<int32_t>((int64_t)p->ny * p->nz);
  int* n_rows = c.take<int>(1);
  float* phi_static = c.take<float>(n);
  uint8_t* tag_static = c.take<uint8_t>(n);
  float* d_override = c.take<float>(n);
  float* uhat = c.take<float>(3 * n);
  double* wm_utau = c.take<double>(n);
  float* wm_u = c.take<float>(3 * n);
  float* wm_s = c.take<float>(6 * n);
  int32_t* wall_idx = c.take<int32_t>(cap);
  double* wall_y1n = c.take<double>(3 * cap);
  double* wall_samp = c.take<double>(6 * cap);
  int32_t* force_idx = c.take<int32_t>(cap);
  Counters* counters = c.take<Counters>(1);
  uint8_t* alt_flags = c.take<uint8_t>(n);
  float* alt_d = c.take<float>(n);
  int32_t* alt_wall_idx = c.take<int32_t>(cap);
  double* alt_wall_y1n = c.take<double>(3 * cap);
  int32_t* alt_force_idx = c.take<int32_t>(cap);
  Counters* alt_counters = c.take<Counters>(1);
  double* force = c.take<double>(FORCE_HISTORY * MAX_TAGS * 3);
  double* torque = c.take<double>(FORCE_HISTORY * MAX_TAGS * 3);
  float* rot_sdf = c.take<float>(rotor_nodes);
  uint8_t* rot_tag = c.take<uint8_t>(rotor_nodes);
  if (L) {
    L->fA = fA; L->fB = fB; L->flags = flags; L->d = d; L->phi = phi; L->below = below; L->tag_prov = tag_prov; L->rowflag = rowflag; L->rowflag_static = rowflag_static; L->phi_static = phi_static;
    L->tag_static = tag_static; L->d_override = d_override; L->uhat = uhat; L->wm_utau = wm_utau;
    L->wm_u = wm_u; L->wm_s = wm_s; L->wall_idx = wall_idx; L->wall_y1n = wall_y1n; L->wall_samp = wall_samp;
    L->rowact[0] = rowact0; L->rowact[1] = rowact1; L->rowlist = rowlist; L->n_rows = n_rows;
    L->alt_flags = alt_flags; L->alt_d = alt_d; L->alt_wall_idx = alt_wall_idx; L->alt_wall_y1n = alt_wall_y1n;
    L->alt_force_idx = alt_force_idx; L->alt_counters = alt_counters;
    L->force_idx = force_idx; L->counters = counters; L->force = force; L->torque = torque; L->rot_sdf = rot_sdf;
    L->rot_tag = rot_tag; L->rot_nodes_cap = rotor_nodes; L->cap_list = cap;
  }
  return c.off;
}

__global__ void fill_bytes_kernel(uint8_t* p, int64_t count, uint8_t v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, s = (int64_t)gridDim.x * blockDim.x;
  for (; i < count; i += s) p[i] = v;
}
__global__ void fill_float_kernel(float* p, int64_t count, float v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, s = (int64_t)gridDim.x * blockDim.x;
  for (; i < count; i += s) p[i] = v;
}

// synchronous host <-> device copies on the lattice stream
int upload(hhrr_lattice* L, void* dst, const void* src, size_t bytes) {
  CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, L->stream));
  CU(cudaStreamSynchronize(L->stream));
  return HHRR_OK;
}
int download(hhrr_lattice* L, void* dst, const void* src, size_t bytes) {
  CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, L->stream));
  CU(cudaStreamSynchronize(L->stream));
  return HHRR_OK;
}

// Everything queued on the side stream (geometry look-ahead: reads the rotor grid and the static fields, writes the
// alternate geometry set; force collection: reads populations, writes the force ring) is ordered before whatever
// the caller's stream does next.
void join_side(hhrr_lattice* L) {
  if (L->side && L->side_busy) {
    cudaEventRecord(L->ev_side, L->side);
    cudaStreamWaitEvent(L->stream, L->ev_side, 0);
    L->side_busy = false;
  }
}

int read_counters(hhrr_lattice* L, Counters* h) { return download(L, h, L->counters, sizeof(Counters)); }

int ensure_geometry(hhrr_lattice* L) {
  if (L->geometry_current) return HHRR_OK;
  if (L->ahead_step == L->step && !L->geometry_dirty) {
    // geometry(step) was written ahead into the alternate set (and its WM_VALID bits by the wall-model kernel of
    // the step before): swap the sets
    cudaStreamWaitEvent(L->stream, L->ev_k1, 0);
    swap_geometry_sets(L);
    L->ahead_step = -1;
    L->geometry_current = true;
    return HHRR_OK;
  }
  join_side(L);  // a force kernel may still be reading the lists this pass rebuilds in place
  const bool full = L->geometry_dirty;
  cudaError_t e = launch_geometry(L, full);
  if (e != cudaSuccess) return cuda_fail(e, "geometry kernels");
  L->geometry_dirty = false;
  L->geometry_current = true;
  if (full && L->fsi.n > 0) {
    // The default kernel treats a block outside every FSI box as bulk fluid without looking at its cells: a region
    // that does not cover the structure must not get as far as a collision.  Full passes follow a setter and are
    // rare, so this one synchronises and looks.  (A rotor that leaves its boxes later is reported by
    // hhrr_check_finite.)
    Counters h;
    int rc = download(L, &h, L->counters, sizeof(Counters));
    if (rc) return rc;
    if (h.region_violation)
      return fail(HHRR_E_STATE, "a cell that is not plain fluid lies outside the FSI region (hhrr_set_fsi_region)");
  }
  return HHRR_OK;
}

}  // namespace

int hhrr::set_error(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

extern "C" {

const char* hhrr_last_error(void) { return g_err; }
const char* hhrr_version(void) { return Q == 27 ? "hhrr-b200 0.2 (D3Q27 fp32, sm_100a)" : "hhrr-b200 0.2 (D3Q19 fp32, sm_100a)"; }
int32_t hhrr_velocity_set(void) { return Q; }
int64_t hhrr_force_history(void) { return FORCE_HISTORY; }

size_t hhrr_workspace_bytes(const hhrr_params* p, const hhrr_rotor_desc* rotor) {
  if (!params_ok(p)) return 0;
  int64_t nodes = 0;
  if (rotor) {
    if (rotor->gx < 2 || rotor->gy < 2 || rotor->gz < 2) return 0;
    nodes = (int64_t)rotor->gx * rotor->gy * rotor->gz;
  }
  return carve(nullptr, p, nodes, nullptr) + 1024;
}

int hhrr_create(const hhrr_params* p, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                hhrr_lattice** out) {
  if (!out) return fail(HHRR_E_ARG, "hhrr_create: out is NULL");
  *out = nullptr;
  if (!params_ok(p)) return fail(HHRR_E_ARG, "hhrr_create: invalid parameters");
  if (!d_workspace) return fail(HHRR_E_ARG, "hhrr_create: workspace is NULL");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev < 1) return fail(HHRR_E_CUDA, "hhrr_create: no CUDA device (%s)", cudaGetErrorString(e));
  cudaPointerAttributes attr;
  e = cudaPointerGetAttributes(&attr, d_workspace);
  if (e != cudaSuccess || attr.type != cudaMemoryTypeDevice)
    return fail(HHRR_E_ARG, "hhrr_create: workspace is not device memory");
  DeviceGuard guard_(attr.device);  // streams, events and kernels of this lattice live on the workspace's device
  char* base = reinterpret_cast<char*>(align_up(reinterpret_cast<size_t>(d_workspace)));
  size_t lead = (size_t)(base - reinterpret_cast<char*>(d_workspace));
  size_t need_min = carve(nullptr, p, 0, nullptr);
  if (workspace_bytes < lead + need_min)
    return fail(HHRR_E_SIZE, "hhrr_create: workspace %zu bytes < %zu needed", workspace_bytes, lead + need_min);
  hhrr_lattice* L = new (std::nothrow) hhrr_lattice();
  if (!L) return fail(HHRR_E_SIZE, "hhrr_create: out of host memory");
  memset(L, 0, sizeof(*L));
  L->p = *p;
  L->dom.nx = p->nx; L->dom.ny = p->ny; L->dom.nz = p->nz;
  for (int a = 0; a < 3; ++a) L->dom.mode[a] = p->mode[a];
  L->dom.n = (int64_t)p->nx * p->ny * p->nz;
  L->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  L->device = attr.device;
  // rotor grid gets whatever the workspace has left
  int64_t rest = (int64_t)(workspace_bytes - lead - need_min);
  int64_t spare = std::max<int64_t>(0, (rest - 512) / 5);
  carve(L, p, spare, base);
  L->variant = 5;
  L->dom.xs = xpull_supported(L->dom) ? 1 : 0;  // buffers start as zeros: nothing to convert
  L->geometry_dirty = true;
  L->geometry_current = false;
  L->ahead_step = -1;
  L->side_busy = false;
  L->lookahead = true;
  {
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    if (cudaStreamCreateWithPriority(&L->side, cudaStreamNonBlocking, prio_lo) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_pre, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_k1, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_k2, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_side, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_f[0], cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&L->ev_f[1], cudaEventDisableTiming) != cudaSuccess) {
      delete L;
      return cuda_fail(cudaGetLastError(), "hhrr_create: side stream");
    }
  }
  const int64_t n = L->dom.n;
  cudaStream_t s = L->stream;
  fill_float_kernel<<<1184, 256, 0, s>>>(L->fA, Q * n, 0.f);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->fB, Q * n, 0.f);
  fill_bytes_kernel<<<1184, 256, 0, s>>>(L->flags, n, 0);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->d, n, 1.f);
  fill_bytes_kernel<<<1184, 256, 0, s>>>(L->alt_flags, n, 0);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->alt_d, n, 1.f);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->uhat, 3 * n, 0.f);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->wm_u, 3 * n, 0.f);
  fill_float_kernel<<<1184, 256, 0, s>>>(L->wm_s, 6 * n, 0.f);
  L->launches += 9;
  e = cudaMemsetAsync(L->wm_utau, 0, sizeof(double) * n, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(L->counters, 0, sizeof(Counters), s);
  if (e == cudaSuccess) e = cudaMemsetAsync(L->alt_counters, 0, sizeof(Counters), s);
  if (e == cudaSuccess) e = cudaMemsetAsync(L->force, 0, sizeof(double) * FORCE_HISTORY * MAX_TAGS * 3, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(L->torque, 0, sizeof(double) * FORCE_HISTORY * MAX_TAGS * 3, s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) {
    delete L;
    return cuda_fail(e, "hhrr_create: initialising the workspace");
  }
  *out = L;
  return HHRR_OK;
}

int hhrr_destroy(hhrr_lattice* L) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_destroy: NULL lattice");
  cudaStreamSynchronize(L->stream);
  if (L->side) {
    cudaStreamSynchronize(L->side);
    cudaEventDestroy(L->ev_pre);
    cudaEventDestroy(L->ev_k1);
    cudaEventDestroy(L->ev_k2);
    cudaEventDestroy(L->ev_side);
    cudaEventDestroy(L->ev_f[0]);
    cudaEventDestroy(L->ev_f[1]);
    cudaStreamDestroy(L->side);
  }
  if (L->ev[0])
    for (int k = 0; k < 2 * 1024; ++k) cudaEventDestroy(L->ev[k]);
  delete L;
  return HHRR_OK;
}

int hhrr_init_equilibrium(hhrr_lattice* L, const float* rho, const float* u, int with_neq) {
  DeviceGuard guard_(L);
  if (!L || !rho || !u) return fail(HHRR_E_ARG, "hhrr_init_equilibrium: NULL argument");
  const int64_t n = L->dom.n;
  // stage rho in buffer B (scratch between steps) and u in the uhat field
  int rc = upload(L, L->fB, rho, sizeof(float) * n);
  if (rc) return rc;
  rc = upload(L, L->uhat, u, sizeof(float) * 3 * n);
  if (rc) return rc;
  cudaError_t e = launch_init(L, L->fB, L->uhat, with_neq);
  if (e != cudaSuccess) return cuda_fail(e, "init kernel");
  CU(cudaStreamSynchronize(L->stream));
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_set_static_geometry(hhrr_lattice* L, const float* phi, const uint8_t* tag, const float* d_override) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_set_static_geometry: NULL lattice");
  const int64_t n = L->dom.n;
  join_side(L);
  L->has_static = L->has_tag_static = L->has_override = false;
  if (phi) {
    int rc = upload(L, L->phi_static, phi, sizeof(float) * n);
    if (rc) return rc;
    L->has_static = true;
    if (tag) {
      rc = upload(L, L->tag_static, tag, n);
      if (rc) return rc;
      L->has_tag_static = true;
    }
    if (d_override) {
      rc = upload(L, L->d_override, d_override, sizeof(float) * n);
      if (rc) return rc;
      L->has_override = true;
    }
  }
  L->geometry_dirty = true;
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_set_body(hhrr_lattice* L, int32_t tag, const double centre[3], const double omega[3],
                  const double vel[3]) {
  DeviceGuard guard_(L);
  if (!L || !centre || !omega || !vel) return fail(HHRR_E_ARG, "hhrr_set_body: NULL argument");
  if (tag < 0 || tag >= MAX_TAGS) return fail(HHRR_E_ARG, "hhrr_set_body: tag %d out of range", tag);
  for (int a = 0; a < 3; ++a) {
    L->bodies.c[tag][a] = centre[a];
    L->bodies.w[tag][a] = omega[a];
    L->bodies.v[tag][a] = vel[a];
  }
  return HHRR_OK;
}

int hhrr_set_fringe(hhrr_lattice* L, int32_t x_begin, int32_t x_end, const double u_in[3]) {
  DeviceGuard guard_(L);
  if (!L || !u_in) return fail(HHRR_E_ARG, "hhrr_set_fringe: NULL argument");
  L->has_fringe = x_end > x_begin;
  L->fr_x0 = x_begin;
  L->fr_x1 = x_end;
  for (int a = 0; a < 3; ++a) L->fr_u[a] = u_in[a];
  L->geometry_dirty = true;
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_set_wall_function(hhrr_lattice* L, int32_t kind) {
  DeviceGuard guard_(L);
  if (!L || (kind != 0 && kind != 1)) return fail(HHRR_E_ARG, "hhrr_set_wall_function: bad argument");
  L->wall_function = kind;
  return HHRR_OK;
}

int hhrr_set_wall_model_variant(hhrr_lattice* L, int32_t slip, int32_t shear) {
  DeviceGuard guard_(L);
  if (!L || (slip != 0 && slip != 1) || (shear != 0 && shear != 1))
    return fail(HHRR_E_ARG, "hhrr_set_wall_model_variant: bad argument");
  L->wm_slip = slip;
  L->wm_shear = shear;
  return HHRR_OK;
}

int hhrr_set_fsi_region(hhrr_lattice* L, int32_t n_boxes, const hhrr_box* boxes) {
  DeviceGuard guard_(L);
  if (!L || n_boxes < 0 || n_boxes > HHRR_MAX_FSI_BOXES || (n_boxes > 0 && !boxes))
    return fail(HHRR_E_ARG, "hhrr_set_fsi_region: bad argument");
  L->fsi.n = n_boxes;
  for (int b = 0; b < n_boxes; ++b)
    L->fsi.b[b] = Box{boxes[b].x0, boxes[b].x1, boxes[b].y0, boxes[b].y1, boxes[b].z0, boxes[b].z1};
  join_side(L);
  CU(cudaMemsetAsync(&L->counters->region_violation, 0, sizeof(int), L->stream));
  CU(cudaMemsetAsync(&L->alt_counters->region_violation, 0, sizeof(int), L->stream));
  L->geometry_dirty = true;
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_set_rotor(hhrr_lattice* L, const hhrr_rotor_desc* r) {
  DeviceGuard guard_(L);
  if (!L || !r || !r->sdf || !r->tag) return fail(HHRR_E_ARG, "hhrr_set_rotor: NULL argument");
  if (r->n_tags < 1 || r->n_tags >= MAX_TAGS) return fail(HHRR_E_ARG, "hhrr_set_rotor: n_tags out of range");
  if (r->gx < 2 || r->gy < 2 || r->gz < 2 || !(r->spacing > 0.0)) return fail(HHRR_E_ARG, "hhrr_set_rotor: bad grid");
  int64_t nodes = (int64_t)r->gx * r->gy * r->gz;
  if (nodes > L->rot_nodes_cap)
    return fail(HHRR_E_SIZE, "hhrr_set_rotor: reference grid of %lld nodes does not fit the workspace (%lld)",
                (long long)nodes, (long long)L->rot_nodes_cap);
  join_side(L);
  int rc = upload(L, L->rot_sdf, r->sdf, sizeof(float) * nodes);
  if (rc) return rc;
  rc = upload(L, L->rot_tag, r->tag, nodes);
  if (rc) return rc;
  L->rot = *r;
  L->rot.sdf = nullptr;
  L->rot.tag = nullptr;
  L->has_rotor = true;
  for (int k = 1; k <= r->n_tags; ++k)  // u^B = Omega x (x - x_c)
    for (int a = 0; a < 3; ++a) {
      L->bodies.c[k][a] = r->centre[a];
      L->bodies.w[k][a] = r->axis[a] * r->omega;
      L->bodies.v[k][a] = 0.0;
    }
  // Box swept under rotation about the axis by the part of the reference grid that can yield
  // phi < eps/2: a trilinear sample is below eps/2 only if one of its 8 nodes is, so bound the
  // axial coordinate and the radial distance (both invariant under the rotation) of the nodes
  // with sdf < eps/2, widened by one grid cell.  Cells outside keep phi >= eps/2 at every angle.
  const double hband = 0.5 * L->p.eps_cells;
  double amin = 1e300, amax = -1e300, rmax = 0.0;
  for (int iz = 0; iz < r->gz; ++iz)
    for (int iy = 0; iy < r->gy; ++iy) {
      const float* row = r->sdf + ((int64_t)iz * r->gy + iy) * r->gx;
      for (int ix = 0; ix < r->gx; ++ix) {
        if (!((double)row[ix] < hband)) continue;
        double q[3] = {r->origin[0] + ix * r->spacing, r->origin[1] + iy * r->spacing, r->origin[2] + iz * r->spacing};
        double ad = q[0] * r->axis[0] + q[1] * r->axis[1] + q[2] * r->axis[2];
        double rr = std::sqrt(std::max(0.0, q[0] * q[0] + q[1] * q[1] + q[2] * q[2] - ad * ad));
        amin = std::min(amin, ad);
        amax = std::max(amax, ad);
        rmax = std::max(rmax, rr);
      }
    }
  const bool any_node = amax >= amin;
  const double widen = 1.7320508075688772 * r->spacing;
  amin -= widen;
  amax += widen;
  rmax += widen;
  int lo[3], hi[3], ext[3] = {L->dom.nx, L->dom.ny, L->dom.nz};
  for (int a = 0; a < 3; ++a) {
    double ak = r->axis[a], perp = std::sqrt(std::max(0.0, 1.0 - ak * ak));
    double e0 = std::min(ak * amin, ak * amax) - perp * rmax, e1 = std::max(ak * amin, ak * amax) + perp * rmax;
    lo[a] = (int)std::floor(r->centre[a] + e0) - 3;
    hi[a] = (int)std::ceil(r->centre[a] + e1) + 4;
    lo[a] = std::max(0, std::min(ext[a], lo[a]));
    hi[a] = std::max(lo[a], std::min(ext[a], hi[a]));
    if (!any_node) lo[a] = hi[a] = 0;
  }
  L->rot_box = Box{lo[0], hi[0], lo[1], hi[1], lo[2], hi[2]};
  // the row band of geometry.cu rests on the paper's premise that the surface moves less than a cell per step
  L->band_ok = std::fabs(r->omega) * (rmax + 2.0) < 0.9;
  L->geometry_dirty = true;
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_enable_wall_model(hhrr_lattice* L, int enable) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_enable_wall_model: NULL lattice");
  L->wm_enabled = enable != 0;
  L->geometry_dirty = true;
  L->geometry_current = false;
  return HHRR_OK;
}

int hhrr_update_geometry(hhrr_lattice* L) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_update_geometry: NULL lattice");
  L->geometry_current = false;
  return ensure_geometry(L);
}

int hhrr_set_kernel_variant(hhrr_lattice* L, int32_t variant) {
  DeviceGuard guard_(L);
  if (!L || (variant != 0 && variant != 2 && variant != 5)) return fail(HHRR_E_ARG, "hhrr_set_kernel_variant: bad argument");
  L->variant = variant;
  // variant 5 keeps the populations x-pulled (where it can run); everything else stores them post-stream
  const bool tiles = xpull_supported(L->dom);
  cudaError_t e = launch_restore(L, (variant == 5 && tiles) ? 1 : 0);
  if (e != cudaSuccess) return cuda_fail(e, "restore kernel");
  if (variant == 5 && !tiles)
    return fail(HHRR_W_FALLBACK,
                "variant 5 cannot tile %d x %d x %d (needs a periodic x axis and nx %% 64 == 0, nx >= 128, ny %% 8 == 0, or "
                "nx %% 128 == 0, nx >= 256, ny %% 4 == 0): variant 2 runs on post-stream storage",
                L->dom.nx, L->dom.ny, L->dom.nz);
  return HHRR_OK;
}

int hhrr_set_launch_shape(hhrr_lattice* L, int32_t chunk_planes, int32_t cluster) {
  DeviceGuard guard_(L);
  if (!L || chunk_planes < 0 || chunk_planes > 4096 || cluster < 0 || cluster > 8 || (cluster & (cluster - 1)))
    return fail(HHRR_E_ARG, "hhrr_set_launch_shape: bad argument");
  L->chunk_planes = chunk_planes;
  L->cluster = cluster;
  return HHRR_OK;
}

int hhrr_set_lookahead(hhrr_lattice* L, int enable) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_set_lookahead: NULL lattice");
  const bool on = enable != 0;
  if (on && !L->lookahead) {
    // Steps taken without the look-ahead evaluate every geometry in place: the alternate set (and the row band's
    // view of it) is as old as the last step that used it.  The next geometry pass is a full one, which re-seeds it.
    L->geometry_dirty = true;
    L->geometry_current = false;
  }
  L->lookahead = on;
  return HHRR_OK;
}

int hhrr_population_storage(const hhrr_lattice* L) {
  DeviceGuard guard_(L); return L ? L->dom.xs : 0; }

int hhrr_set_timing(hhrr_lattice* L, int enable) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_set_timing: NULL lattice");
  if (enable && !L->ev[0])
    for (int k = 0; k < 2 * 1024; ++k) CU(cudaEventCreate(&L->ev[k]));
  L->timing = enable != 0;
  L->ev_n = 0;
  return HHRR_OK;
}

int hhrr_get_timing(hhrr_lattice* L, double* ms_collide_stream, int64_t* launches) {
  DeviceGuard guard_(L);
  if (!L || !ms_collide_stream || !launches) return fail(HHRR_E_ARG, "hhrr_get_timing: NULL argument");
  CU(cudaStreamSynchronize(L->stream));
  double total = 0.0;
  for (int k = 0; k < L->ev_n; ++k) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, L->ev[2 * k], L->ev[2 * k + 1]));
    total += ms;
  }
  *ms_collide_stream = total;
  *launches = L->ev_n;
  L->ev_n = 0;
  return HHRR_OK;
}

int64_t hhrr_launch_count(const hhrr_lattice* L) {
  DeviceGuard guard_(L); return L ? L->launches : 0; }
int64_t hhrr_step_count(const hhrr_lattice* L) {
  DeviceGuard guard_(L); return L ? L->step : 0; }

// One step = Listing 3.  On the caller's stream: [UpdatePorosityO(n): a pointer swap when it
// was written ahead] -> collide-stream(n) -> WallModelO(n).  On the side stream, beside collide-stream(n):
// UpdatePorosityO(n + 1) into the alternate geometry set; beside collide-stream(n + 1): the force collection
// of step n, which only reads.  The call returns with the side stream joined into the caller's stream.
int hhrr_step(hhrr_lattice* L, int32_t n_steps) {
  DeviceGuard guard_(L);
  if (!L || n_steps < 0) return fail(HHRR_E_ARG, "hhrr_step: bad argument");
  for (int32_t s = 0; s < n_steps; ++s) {
    int rc = ensure_geometry(L);  // Listing 3 line 2: UpdatePorosityO
    if (rc) return rc;
    if (L->side) {
      CU(cudaEventRecord(L->ev_pre, L->stream));
      // this launch overwrites the buffer the force kernel of two steps ago read (a no-op unless it is still running)
      if (L->step >= 2) CU(cudaStreamWaitEvent(L->stream, L->ev_f[L->step & 1], 0));
    }
    const bool timed = L->timing && L->ev_n < 1024;
    if (timed) CU(cudaEventRecord(L->ev[2 * L->ev_n], L->stream));
    cudaError_t e = launch_collide_stream(L);  // line 3
    if (e != cudaSuccess) return cuda_fail(e, "collide-stream kernel");
    if (timed) {
      CU(cudaEventRecord(L->ev[2 * L->ev_n + 1], L->stream));
      L->ev_n++;
    }
    if (L->side) CU(cudaEventRecord(L->ev_k2, L->stream));
    e = launch_geometry_ahead(L);  // line 2 of the NEXT step, on the side stream
    if (e != cudaSuccess) return cuda_fail(e, "geometry look-ahead");
    const bool ahead = L->ahead_step == L->step + 1;
    e = launch_wall_model(L);  // line 4: WallModelO -- beside the geometry look-ahead, which starts in the tail of K2
    if (e != cudaSuccess) return cuda_fail(e, "wall-model kernel");
    if (ahead && L->wm_enabled) {  // the two meet: the geometry written ahead learns which of its wall cells hold state
      CU(cudaStreamWaitEvent(L->stream, L->ev_k1, 0));
      e = launch_merge_valid(L);
      if (e != cudaSuccess) return cuda_fail(e, "wall-state merge kernel");
    }
    if (L->side) {  // lines 5-6: forces, beside the next collide-stream kernel
      CU(cudaStreamWaitEvent(L->side, L->ev_k2, 0));
      e = launch_forces(L, L->side);
      CU(cudaEventRecord(L->ev_f[L->step & 1], L->side));
      L->side_busy = true;
    } else {
      e = launch_forces(L, L->stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, "force kernel");
    L->step += 1;  // line 7: theta_{n+1} = theta_n + Omega
    L->geometry_current = !L->has_rotor;  // static geometry stays valid
  }
  join_side(L);
  return HHRR_OK;
}

int hhrr_get_moments_device(hhrr_lattice* L, float* d_rho, float* d_v) {
  DeviceGuard guard_(L);
  if (!L || !d_rho || !d_v) return fail(HHRR_E_ARG, "hhrr_get_moments_device: NULL argument");
  cudaError_t e = launch_moments(L, d_rho, d_v);
  if (e != cudaSuccess) return cuda_fail(e, "moments kernel");
  return HHRR_OK;
}

int hhrr_get_moments(hhrr_lattice* L, float* rho, float* v) {
  DeviceGuard guard_(L);
  if (!L || !rho || !v) return fail(HHRR_E_ARG, "hhrr_get_moments: NULL argument");
  const int64_t n = L->dom.n;
  float* scratch = L->fB;  // buffer B is free between steps
  cudaError_t e = launch_moments(L, scratch, scratch + n);
  if (e != cudaSuccess) return cuda_fail(e, "moments kernel");
  int rc = download(L, rho, scratch, sizeof(float) * n);
  if (rc) return rc;
  return download(L, v, scratch + n, sizeof(float) * 3 * n);
}

static int get_force_ring(hhrr_lattice* L, const double* ring, const char* who, int64_t first_step, int64_t n_steps,
                          double* F) {
  DeviceGuard guard_(L);
  if (!L || !F || n_steps < 0) return fail(HHRR_E_ARG, "%s: bad argument", who);
  if (first_step < 0 || first_step + n_steps > L->step || first_step < L->step - FORCE_HISTORY)
    return fail(HHRR_E_STATE, "%s: steps [%lld,%lld) not in the recorded history (step %lld)", who,
                (long long)first_step, (long long)(first_step + n_steps), (long long)L->step);
  const size_t rec = sizeof(double) * MAX_TAGS * 3;
  int64_t s = first_step;
  while (s < first_step + n_steps) {  // the ring may wrap once
    int64_t slot = s % FORCE_HISTORY;
    int64_t run = std::min<int64_t>(first_step + n_steps - s, FORCE_HISTORY - slot);
    CU(cudaMemcpyAsync(F + (s - first_step) * MAX_TAGS * 3, ring + slot * MAX_TAGS * 3, rec * run,
                       cudaMemcpyDeviceToHost, L->stream));
    s += run;
  }
  CU(cudaStreamSynchronize(L->stream));
  return HHRR_OK;
}

int hhrr_get_forces(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double* F) {
  DeviceGuard guard_(L);
  return get_force_ring(L, L ? L->force : nullptr, "hhrr_get_forces", first_step, n_steps, F);
}

int hhrr_get_torques(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double* M) {
  DeviceGuard guard_(L);
  return get_force_ring(L, L ? L->torque : nullptr, "hhrr_get_torques", first_step, n_steps, M);
}

int hhrr_get_rotor_coefficients(hhrr_lattice* L, int64_t first_step, int64_t n_steps, double rho, double u_inf,
                                double radius, double* c_t, double* c_p) {
  DeviceGuard guard_(L);
  if (!L || n_steps < 0 || (!c_t && !c_p)) return fail(HHRR_E_ARG, "hhrr_get_rotor_coefficients: bad argument");
  if (!(rho > 0.0) || !(u_inf > 0.0) || !(radius > 0.0))
    return fail(HHRR_E_ARG, "hhrr_get_rotor_coefficients: rho, u_inf and radius must be positive");
  if (!L->has_rotor) return fail(HHRR_E_STATE, "hhrr_get_rotor_coefficients: no rotor set");
  std::vector<double> F((size_t)n_steps * MAX_TAGS * 3), M((size_t)n_steps * MAX_TAGS * 3);
  int rc = get_force_ring(L, L->force, "hhrr_get_rotor_coefficients", first_step, n_steps, F.data());
  if (rc) return rc;
  rc = get_force_ring(L, L->torque, "hhrr_get_rotor_coefficients", first_step, n_steps, M.data());
  if (rc) return rc;
  const double* ax = L->rot.axis;  // unit vector (include/hhrr.h: hhrr_rotor_desc)
  const double q = 0.5 * rho * M_PI * radius * radius * u_inf * u_inf;  // denominator of Eq. 26
  for (int64_t s = 0; s < n_steps; ++s) {
    double thrust = 0.0, torque = 0.0;  // axial force on / axial torque on the rotor: all its elements
    for (int k = 1; k <= L->rot.n_tags; ++k) {
      const double* f = F.data() + ((size_t)s * MAX_TAGS + k) * 3;
      const double* m = M.data() + ((size_t)s * MAX_TAGS + k) * 3;
      thrust += f[0] * ax[0] + f[1] * ax[1] + f[2] * ax[2];
      torque += m[0] * ax[0] + m[1] * ax[1] + m[2] * ax[2];
    }
    if (c_t) c_t[s] = thrust / q;
    if (c_p) c_p[s] = torque * L->rot.omega / (q * u_inf);
  }
  return HHRR_OK;
}

int hhrr_get_cell_types(hhrr_lattice* L, uint8_t* type, uint8_t* tag, float* d) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_get_cell_types: NULL lattice");
  const int64_t n = L->dom.n;
  if (type || tag) {
    std::vector<uint8_t> fl((size_t)n);
    int rc = download(L, fl.data(), L->flags, (size_t)n);
    if (rc) return rc;
    for (int64_t c = 0; c < n; ++c) {
      if (type) type[c] = (uint8_t)public_type(fl[c] & TYPE_MASK);
      if (tag) tag[c] = (fl[c] >> TAG_SHIFT) & TAG_MASK;
    }
  }
  if (d) return download(L, d, L->d, sizeof(float) * n);
  return HHRR_OK;
}

namespace {
__global__ void gather_wall_kernel(const int32_t* idx, int count, const double* wm_utau, const uint8_t* flags,
                                   double* out_utau, uint8_t* out_valid) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  int64_t c = idx[e];
  out_utau[e] = wm_utau[c];
  out_valid[e] = (flags[c] & WM_VALID) ? 1 : 0;
}
__global__ void gather_cells_kernel(const float* f, const uint8_t* flags, Dom dm, const int64_t* cells,
                                    int64_t count, float* out, uint8_t* out_flags) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= count) return;
  int64_t c = cells[k];
  const int x = (int)(c % dm.nx), y = (int)((c / dm.nx) % dm.ny), z = (int)(c / ((int64_t)dm.nx * dm.ny));
  for (int i = 0; i < Q; ++i) out[k * Q + i] = f[pop_index(dm, i, x, y, z)];
  out_flags[k] = (uint8_t)((flags[c] & ~TYPE_MASK) | public_type(flags[c] & TYPE_MASK));
}
}  // namespace

int hhrr_get_wall_list(hhrr_lattice* L, int64_t capacity, int32_t* idx, double* y1n, double* u_tau,
                       uint8_t* valid, int64_t* count) {
  DeviceGuard guard_(L);
  if (!L || !count) return fail(HHRR_E_ARG, "hhrr_get_wall_list: NULL argument");
  Counters h;
  int rc = read_counters(L, &h);
  if (rc) return rc;
  if (h.overflow) return fail(HHRR_E_SIZE, "compact cell list overflowed its capacity of %lld", (long long)L->cap_list);
  int64_t k = h.wall_count;
  *count = k;
  if (k == 0 || capacity <= 0 || !idx) return HHRR_OK;
  std::vector<int32_t> hidx((size_t)k);
  std::vector<double> hy((size_t)3 * k), hu((size_t)k);
  std::vector<uint8_t> hv((size_t)k);
  rc = download(L, hidx.data(), L->wall_idx, sizeof(int32_t) * k);
  if (rc) return rc;
  rc = download(L, hy.data(), L->wall_y1n, sizeof(double) * 3 * k);
  if (rc) return rc;
  double* s_utau = reinterpret_cast<double*>(L->fB);  // scratch
  uint8_t* s_valid = reinterpret_cast<uint8_t*>(s_utau + k);
  gather_wall_kernel<<<(unsigned)((k + 255) / 256), 256, 0, L->stream>>>(L->wall_idx, (int)k, L->wm_utau, L->flags,
                                                                         s_utau, s_valid);
  L->launches++;
  CU(cudaGetLastError());
  rc = download(L, hu.data(), s_utau, sizeof(double) * k);
  if (rc) return rc;
  rc = download(L, hv.data(), s_valid, (size_t)k);
  if (rc) return rc;
  std::vector<int64_t> order((size_t)k);
  for (int64_t e = 0; e < k; ++e) order[e] = e;
  std::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return hidx[a] < hidx[b]; });
  int64_t m = std::min(k, capacity);
  for (int64_t e = 0; e < m; ++e) {
    int64_t o = order[e];
    idx[e] = hidx[o];
    if (y1n)
      for (int a = 0; a < 3; ++a) y1n[3 * e + a] = hy[3 * o + a];
    if (u_tau) u_tau[e] = hu[o];
    if (valid) valid[e] = hv[o];
  }
  return HHRR_OK;
}

int hhrr_get_wall_state(hhrr_lattice* L, int64_t cell, double* u_tau, double u_wm[3], double s_wm[6],
                        int32_t* valid) {
  DeviceGuard guard_(L);
  if (!L || cell < 0 || cell >= L->dom.n) return fail(HHRR_E_ARG, "hhrr_get_wall_state: bad argument");
  const int64_t n = L->dom.n;
  double ut;
  float u[3], s[6];
  uint8_t fl;
  CU(cudaMemcpyAsync(&ut, L->wm_utau + cell, sizeof(double), cudaMemcpyDeviceToHost, L->stream));
  for (int a = 0; a < 3; ++a)
    CU(cudaMemcpyAsync(&u[a], L->wm_u + a * n + cell, sizeof(float), cudaMemcpyDeviceToHost, L->stream));
  for (int a = 0; a < 6; ++a)
    CU(cudaMemcpyAsync(&s[a], L->wm_s + a * n + cell, sizeof(float), cudaMemcpyDeviceToHost, L->stream));
  CU(cudaMemcpyAsync(&fl, L->flags + cell, 1, cudaMemcpyDeviceToHost, L->stream));
  CU(cudaStreamSynchronize(L->stream));
  if (u_tau) *u_tau = ut;
  if (u_wm) for (int a = 0; a < 3; ++a) u_wm[a] = u[a];
  if (s_wm) for (int a = 0; a < 6; ++a) s_wm[a] = s[a];
  if (valid) *valid = (fl & WM_VALID) ? 1 : 0;
  return HHRR_OK;
}

int hhrr_get_cell_populations(hhrr_lattice* L, int64_t n_cells, const int64_t* cells, float* out,
                              uint8_t* flags) {
  DeviceGuard guard_(L);
  if (!L || !cells || !out || n_cells < 0) return fail(HHRR_E_ARG, "hhrr_get_cell_populations: bad argument");
  if (n_cells == 0) return HHRR_OK;
  for (int64_t k = 0; k < n_cells; ++k)
    if (cells[k] < 0 || cells[k] >= L->dom.n) return fail(HHRR_E_ARG, "hhrr_get_cell_populations: cell out of range");
  // scratch in buffer B, [cells 8 B | out 108 B | flags 1 B] per cell: as many cells per pass as fit
  char* sb = reinterpret_cast<char*>(L->fB);
  const int64_t per_pass = std::max<int64_t>(1, (int64_t)(sizeof(float) * Q * (size_t)L->dom.n / (8 + 4 * Q + 1)));
  for (int64_t k0 = 0; k0 < n_cells; k0 += per_pass) {
    const int64_t m = std::min(per_pass, n_cells - k0);
    int64_t* d_cells = reinterpret_cast<int64_t*>(sb);
    float* d_out = reinterpret_cast<float*>(sb + 8 * m);
    uint8_t* d_fl = reinterpret_cast<uint8_t*>(sb + 8 * m + 4 * Q * m);
    int rc = upload(L, d_cells, cells + k0, 8 * (size_t)m);
    if (rc) return rc;
    gather_cells_kernel<<<(unsigned)((m + 127) / 128), 128, 0, L->stream>>>(L->fA, L->flags, L->dom, d_cells, m, d_out,
                                                                         d_fl);
    L->launches++;
    CU(cudaGetLastError());
    rc = download(L, out + (size_t)Q * k0, d_out, 4 * (size_t)Q * m);
    if (rc) return rc;
    if (flags) {
      rc = download(L, flags + k0, d_fl, (size_t)m);
      if (rc) return rc;
    }
  }
  return HHRR_OK;
}

int hhrr_get_populations(hhrr_lattice* L, float* f_minus_w) {
  DeviceGuard guard_(L);
  if (!L || !f_minus_w) return fail(HHRR_E_ARG, "hhrr_get_populations: NULL argument");
  if (!L->dom.xs) return download(L, f_minus_w, L->fA, sizeof(float) * Q * L->dom.n);
  // the ABI speaks the plain post-stream layout: convert into buffer B (free between steps), read that
  const int xs = L->dom.xs;
  cudaError_t e = launch_restore(L, 0);  // A <-> B swapped, A now plain
  if (e != cudaSuccess) return cuda_fail(e, "restore kernel");
  int rc = download(L, f_minus_w, L->fA, sizeof(float) * Q * L->dom.n);
  float* t = L->fA;  // swap back: the stored state is untouched
  L->fA = L->fB;
  L->fB = t;
  L->dom.xs = xs;
  return rc;
}
int hhrr_set_populations(hhrr_lattice* L, const float* f_minus_w) {
  DeviceGuard guard_(L);
  if (!L || !f_minus_w) return fail(HHRR_E_ARG, "hhrr_set_populations: NULL argument");
  int rc = upload(L, L->fA, f_minus_w, sizeof(float) * Q * L->dom.n);
  if (rc || !L->dom.xs) return rc;
  const int xs = L->dom.xs;
  L->dom.xs = 0;  // what was uploaded is the plain post-stream layout
  cudaError_t e = launch_restore(L, xs);
  if (e != cudaSuccess) return cuda_fail(e, "restore kernel");
  return HHRR_OK;
}
int hhrr_get_uhat(hhrr_lattice* L, float* uhat) {
  DeviceGuard guard_(L);
  if (!L || !uhat) return fail(HHRR_E_ARG, "hhrr_get_uhat: NULL argument");
  if (L->variant != 0 || L->step == 0)
    return fail(HHRR_E_STATE, "hhrr_get_uhat: only the two-pass kernel (variant 0) stores the field, and only after a step");
  return download(L, uhat, L->uhat, sizeof(float) * 3 * L->dom.n);
}


namespace {
__global__ void gather_wall_state_kernel(const int32_t* idx, int count, int64_t n, const double* wm_utau, const float* wm_u,
                                         const float* wm_s, const uint8_t* flags, double* o_utau, float* o_u, float* o_s,
                                         uint8_t* o_valid) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  const int64_t c = idx[e];
  o_utau[e] = wm_utau[c];
  for (int q = 0; q < 3; ++q) o_u[3 * (int64_t)e + q] = wm_u[q * n + c];
  for (int q = 0; q < 6; ++q) o_s[6 * (int64_t)e + q] = wm_s[q * n + c];
  o_valid[e] = (flags[c] & WM_VALID) ? 1 : 0;
}
__global__ void scatter_wall_state_kernel(const int32_t* idx, int count, int64_t n, const double* i_utau, const float* i_u,
                                          const float* i_s, const uint8_t* i_valid, double* wm_utau, float* wm_u,
                                          float* wm_s, uint8_t* flags) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  const int64_t c = idx[e];
  const uint8_t fl = flags[c];
  if ((fl & TYPE_MASK) != T_FRONTIER_W) return;  // not in the wall-model set of the current geometry: no state to hold
  wm_utau[c] = i_utau[e];
  for (int q = 0; q < 3; ++q) wm_u[q * n + c] = i_u[3 * (int64_t)e + q];
  for (int q = 0; q < 6; ++q) wm_s[q * n + c] = i_s[6 * (int64_t)e + q];
  flags[c] = i_valid[e] ? (fl | WM_VALID) : (fl & ~WM_VALID);
}
}  // namespace

int hhrr_get_wall_model_state(hhrr_lattice* L, int64_t capacity, int32_t* idx, double* u_tau, float* u_wm, float* s_wm,
                              uint8_t* valid, int64_t* count) {
  DeviceGuard guard_(L);
  if (!L || !count) return fail(HHRR_E_ARG, "hhrr_get_wall_model_state: NULL argument");
  Counters h;
  int rc = read_counters(L, &h);
  if (rc) return rc;
  if (h.overflow) return fail(HHRR_E_SIZE, "compact cell list overflowed its capacity of %lld", (long long)L->cap_list);
  const int64_t k = h.wall_count;
  *count = k;
  if (k == 0 || capacity <= 0) return HHRR_OK;
  if (capacity < k || !idx || !u_tau || !u_wm || !s_wm || !valid)
    return fail(HHRR_E_ARG, "hhrr_get_wall_model_state: capacity %lld < %lld cells, or a NULL array", (long long)capacity,
                (long long)k);
  char* sb = reinterpret_cast<char*>(L->fB);  // scratch: buffer B is free between steps
  double* s_utau = reinterpret_cast<double*>(sb);
  float* s_u = reinterpret_cast<float*>(s_utau + k);
  float* s_s = s_u + 3 * k;
  uint8_t* s_v = reinterpret_cast<uint8_t*>(s_s + 6 * k);
  gather_wall_state_kernel<<<(unsigned)((k + 255) / 256), 256, 0, L->stream>>>(L->wall_idx, (int)k, L->dom.n, L->wm_utau,
                                                                              L->wm_u, L->wm_s, L->flags, s_utau, s_u, s_s, s_v);
  L->launches++;
  CU(cudaGetLastError());
  if ((rc = download(L, idx, L->wall_idx, sizeof(int32_t) * k))) return rc;
  if ((rc = download(L, u_tau, s_utau, sizeof(double) * k))) return rc;
  if ((rc = download(L, u_wm, s_u, sizeof(float) * 3 * k))) return rc;
  if ((rc = download(L, s_wm, s_s, sizeof(float) * 6 * k))) return rc;
  return download(L, valid, s_v, (size_t)k);
}

int hhrr_set_wall_model_state(hhrr_lattice* L, int64_t count, const int32_t* idx, const double* u_tau, const float* u_wm,
                              const float* s_wm, const uint8_t* valid) {
  DeviceGuard guard_(L);
  if (!L || count < 0 || (count > 0 && (!idx || !u_tau || !u_wm || !s_wm || !valid)))
    return fail(HHRR_E_ARG, "hhrr_set_wall_model_state: bad argument");
  if (count > L->cap_list) return fail(HHRR_E_SIZE, "hhrr_set_wall_model_state: more cells than the wall list can hold");
  for (int64_t e = 0; e < count; ++e)
    if (idx[e] < 0 || idx[e] >= L->dom.n) return fail(HHRR_E_ARG, "hhrr_set_wall_model_state: cell out of range");
  int rc = ensure_geometry(L);  // the state belongs to cells of W of the current step's geometry
  if (rc || count == 0) return rc;
  const int64_t k = count;
  char* sb = reinterpret_cast<char*>(L->fB);
  double* s_utau = reinterpret_cast<double*>(sb);
  float* s_u = reinterpret_cast<float*>(s_utau + k);
  float* s_s = s_u + 3 * k;
  uint8_t* s_v = reinterpret_cast<uint8_t*>(s_s + 6 * k);
  int32_t* s_idx = reinterpret_cast<int32_t*>(sb + align_up((size_t)k * (8 + 12 + 24 + 1)));
  if ((rc = upload(L, s_utau, u_tau, sizeof(double) * k))) return rc;
  if ((rc = upload(L, s_u, u_wm, sizeof(float) * 3 * k))) return rc;
  if ((rc = upload(L, s_s, s_wm, sizeof(float) * 6 * k))) return rc;
  if ((rc = upload(L, s_v, valid, (size_t)k))) return rc;
  if ((rc = upload(L, s_idx, idx, sizeof(int32_t) * k))) return rc;
  scatter_wall_state_kernel<<<(unsigned)((k + 255) / 256), 256, 0, L->stream>>>(s_idx, (int)k, L->dom.n, s_utau, s_u, s_s, s_v,
                                                                               L->wm_utau, L->wm_u, L->wm_s, L->flags);
  L->launches++;
  CU(cudaGetLastError());
  CU(cudaStreamSynchronize(L->stream));
  return HHRR_OK;
}

int hhrr_set_step_count(hhrr_lattice* L, int64_t step) {
  DeviceGuard guard_(L);
  if (!L || step < 0) return fail(HHRR_E_ARG, "hhrr_set_step_count: bad argument");
  join_side(L);
  if (L->ahead_step >= 0) {  // a geometry written ahead belongs to the run that was going on: dropped
    cudaStreamWaitEvent(L->stream, L->ev_k1, 0);
    L->ahead_step = -1;
  }
  L->step = step;
  if (L->has_rotor) {  // the rotor angle follows the step count; the row band of the last steps is void
    L->geometry_current = false;
    L->geometry_dirty = true;
  }
  return HHRR_OK;
}

int hhrr_check_finite(hhrr_lattice* L) {
  DeviceGuard guard_(L);
  if (!L) return fail(HHRR_E_ARG, "hhrr_check_finite: NULL lattice");
  cudaError_t e = launch_check_finite(L);
  if (e != cudaSuccess) return cuda_fail(e, "finite-check kernel");
  Counters h;
  int rc = read_counters(L, &h);
  if (rc) return rc;
  if (h.overflow) return fail(HHRR_E_SIZE, "compact cell list overflowed its capacity of %lld", (long long)L->cap_list);
  if (h.region_violation)
    return fail(HHRR_E_STATE, "a cell that is not plain fluid lies outside the FSI region (hhrr_set_fsi_region)");
  if (h.nonfinite) return fail(HHRR_E_NAN, "non-finite population at step %lld", (long long)L->step);
  return HHRR_OK;
}

}  // extern "C"

// ---- slab decomposition along z (the paper's weak-scaling layout) -------
// A rank holds nz - 2 planes of the global lattice plus one halo plane at either end (z = 0 and z = nz - 1) on a
// z-periodic local lattice.  After a collide-stream step the halo exchange makes the local state exact again:
//   * what this rank's collision pushed INTO a halo plane (the 9 populations moving outward) belongs to the
//     neighbour's first real plane;
//   * the other populations of the neighbour's halo plane (those not moving towards the neighbour) are copied from
//     this rank's last real plane, so that the neighbour can form the time-n homogenised velocity of the plane next
//     to its slab (S^FD, Eq. 10) and the momentum-exchange links that reach into it (Eq. 23 :211).
// Per face and direction: Q planes of nx * ny floats (9 + 18 on D3Q27; 5 + 14 on D3Q19), packed into one contiguous
// device buffer so that the transport (NCCL send / recv, a peer copy, or -- d_buf being a peer-mapped pointer -- the
// pack kernel's own stores over NVLink) is one transfer per face.  Planes are copied as stored: both ranks keep the
// same population storage.
namespace {
// face 0 = low z, 1 = high z; c = the c_z of the populations that cross the face (pack: leaving, c = +-1 outward;
// unpack: arriving, the same c seen from the receiver).  Slot i of the buffer carries
//   c_z(i) ==  c : population i of the HALO plane of the sender   -> population i of the first REAL plane of the receiver
//   c_z(i) ==  0 : population i of the last REAL plane of the sender -> population i of the HALO plane of the receiver
//   c_z(i) == -c : population j = i with c_z reversed (c_z(j) = c) of the last REAL plane of the sender
//                                                                   -> population j of the HALO plane of the receiver
// (the receiver's halo plane already holds its populations with c_z = -c: its own collision pushed them there).
// grid (blocks per plane, Q): blockIdx.y is the buffer slot, so all Q planes move at once; 16-byte accesses when VEC
template <bool VEC>
__global__ void __launch_bounds__(256) halo_copy_kernel(float* __restrict__ f, float* __restrict__ buf, int64_t n,
                                                        int64_t plane, int nz, int face, int unpack) {
  const int i = blockIdx.y;
  const int c = unpack ? (face ? -1 : 1) : (face ? 1 : -1);
  const int z_halo = face ? nz - 1 : 0, z_real = face ? nz - 2 : 1;
  const int cz = dir_cz(i);
  const int pop = cz == -c ? dir_flip(i, false, false, true) : i;
  // sender: crossing populations sit in its halo plane; receiver: they land in its first real plane
  const int z = (cz == c) ? (unpack ? z_real : z_halo) : (unpack ? z_halo : z_real);
  float* p = f + (int64_t)pop * n + plane * z;
  float* b = buf + (int64_t)i * plane;
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, T = (int64_t)gridDim.x * blockDim.x;
  if (VEC) {
    float4* p4 = reinterpret_cast<float4*>(p);
    float4* b4 = reinterpret_cast<float4*>(b);
    if (!unpack)
      for (int64_t k = t; k < plane / 4; k += T) b4[k] = p4[k];
    else
      for (int64_t k = t; k < plane / 4; k += T) p4[k] = b4[k];
  } else {
    if (!unpack)
      for (int64_t k = t; k < plane; k += T) b[k] = p[k];
    else
      for (int64_t k = t; k < plane; k += T) p[k] = b[k];
  }
}

cudaError_t launch_halo_copy(hhrr_lattice* L, float* buf, int face, int unpack) {
  const int64_t plane = (int64_t)L->dom.nx * L->dom.ny;
  const bool vec = plane % 4 == 0 && (reinterpret_cast<uintptr_t>(buf) & 15) == 0;
  const int64_t items = vec ? plane / 4 : plane;
  dim3 grid((unsigned)std::min<int64_t>(148, (items + 255) / 256), Q);
  if (vec)
    halo_copy_kernel<true><<<grid, 256, 0, L->stream>>>(L->fA, buf, L->dom.n, plane, L->dom.nz, face, unpack);
  else
    halo_copy_kernel<false><<<grid, 256, 0, L->stream>>>(L->fA, buf, L->dom.n, plane, L->dom.nz, face, unpack);
  L->launches++;
  return cudaGetLastError();
}
}  // namespace

extern "C" {
int64_t hhrr_halo_floats(const hhrr_lattice* L) { return L ? (int64_t)Q * L->dom.nx * L->dom.ny : 0; }

int hhrr_halo_pack(hhrr_lattice* L, int32_t face, float* d_buf) {
  DeviceGuard guard_(L);
  if (!L || !d_buf || (face != 0 && face != 1)) return fail(HHRR_E_ARG, "hhrr_halo_pack: bad argument");
  if (L->dom.nz < 4 || L->dom.mode[2] != HHRR_PERIODIC)
    return fail(HHRR_E_STATE, "hhrr_halo_pack: a slab needs a periodic z axis of at least 4 planes (2 halo + 2 real)");
  CU(launch_halo_copy(L, d_buf, face, 0));
  return HHRR_OK;
}

int hhrr_halo_unpack(hhrr_lattice* L, int32_t face, const float* d_buf) {
  DeviceGuard guard_(L);
  if (!L || !d_buf || (face != 0 && face != 1)) return fail(HHRR_E_ARG, "hhrr_halo_unpack: bad argument");
  if (L->dom.nz < 4 || L->dom.mode[2] != HHRR_PERIODIC)
    return fail(HHRR_E_STATE, "hhrr_halo_unpack: a slab needs a periodic z axis of at least 4 planes (2 halo + 2 real)");
  CU(launch_halo_copy(L, const_cast<float*>(d_buf), face, 1));
  return HHRR_OK;
}
}  // extern "C"
