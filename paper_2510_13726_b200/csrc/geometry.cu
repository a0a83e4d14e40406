// geometry.cu -- K1: UpdatePorosityO (Listing 3 line 2).
//
// Signed distance -> porosity (Def. 1, Eq. 21-22), cell types of Fig. 4
// (:254-263), integer element tag (:267), wall-model set with the y1 vector (:324) and the
// compact lists the wall-model and force kernels run over.  The rotor is re-embedded every
// step by rotating cell centres into the rotor frame and sampling the reference grid
// (:219, :265).  Instead of the paper's incremental growth-layer walk (:269) the kernels
// re-evaluate the fixed box swept by the rotor -- a few percent of the cells -- which gives
// the brute-force classification by construction.
//
// Integer results (types, tags, lists) are defined by the fp64 operation order below; this
// file is compiled with -fmad=false so no contraction changes it.
#include <utility>

#include "lattice.h"

namespace hhrr {

struct GeoArgs {
  Dom dm;
  Boxes fsi;        // FSI region: fluid cells outside every box are BULK (R20)
  Box box;          // cells processed (inside == true) or skipped (inside == false)
  int inside;
  double h;         // eps/2
  double eps;
  int has_static, has_tag_static, has_override, has_fringe, has_rotor, wm_enabled;
  int fr_x0, fr_x1;
  double cth, sth;  // cos / sin of the rotor angle, evaluated once on the host
  RotorDev rot;
  const float* phi_static;
  const uint8_t* tag_static;
  const float* d_override;
  double* phi;
  uint8_t* below;   // phi < eps/2 per cell: what the growth-layer test reads (1 B instead of 8)
  uint8_t* rowflag; // per (y,z) row: some cell of the row may have phi < eps/2 (superset)
  // Row band of the rotor (see "K1 on the band" below): rowact_w = the parity written by this evaluation,
  // rowact0 / rowact1 = both parities (read by the row selection), rowlist / n_rows = the rows to evaluate
  uint8_t* rowact_w;
  uint8_t *rowact0, *rowact1;
  const uint8_t* rowflag_static;
  int32_t* rowlist;
  int* n_rows;
  int all_rows;     // 1: every row of the box (the rotor may move more than a cell per step: no band argument)
  uint8_t* tag_prov;  // provisional tag of pass 1 (its own array: pass 1 may run ahead of the step that reads flags)
  const uint8_t* flags_prev;  // flag bytes the wall-model state bit is carried over from; NULL: written as 0 (look-ahead:
                              // the wall-model kernel of the step in between sets it, wallmodel.cu)
  uint8_t* flags;
  float* d;
  int32_t* wall_idx;
  double* wall_y1n;
  int32_t* force_idx;
  Counters* cnt;
  int cap_list;
};

__device__ __forceinline__ int wrap_any(int v, int n, int mode) {
  if (v >= 0 && v < n) return v;
  if (mode == HHRR_PERIODIC) return ((v % n) + n) % n;
  return v < 0 ? -1 - v : 2 * n - 1 - v;
}

// rotate (p - centre) by -theta about the axis, trilinear-sample the reference grid
__device__ double rotor_phi(const RotorDev& R, double cth, double sth, double px, double py, double pz,
                            int* tag_out) {
  double rx = px - R.centre[0], ry = py - R.centre[1], rz = pz - R.centre[2];
  double ax = R.axis[0], ay = R.axis[1], az = R.axis[2];
  double kx = ay * rz - az * ry, ky = az * rx - ax * rz, kz = ax * ry - ay * rx;
  double ad = ax * rx + ay * ry + az * rz;
  double omc = 1.0 - cth;
  double qx = rx * cth - kx * sth + ax * ad * omc;
  double qy = ry * cth - ky * sth + ay * ad * omc;
  double qz = rz * cth - kz * sth + az * ad * omc;
  double gx = (qx - R.origin[0]) / R.spacing;
  double gy = (qy - R.origin[1]) / R.spacing;
  double gz = (qz - R.origin[2]) / R.spacing;
  double fx = floor(gx), fy = floor(gy), fz = floor(gz);
  *tag_out = 0;
  if (!(fx >= 0.0 && fy >= 0.0 && fz >= 0.0 && fx < (double)(R.gx - 1) && fy < (double)(R.gy - 1) &&
        fz < (double)(R.gz - 1)))
    return BIG_PHI;
  int ix = (int)fx, iy = (int)fy, iz = (int)fz;
  double tx = gx - fx, ty = gy - fy, tz = gz - fz;
  const float* s = R.sdf;
  int64_t sx = 1, sy = R.gx, sz = (int64_t)R.gx * R.gy;
  int64_t b = ix * sx + iy * sy + iz * sz;
  double v000 = s[b], v100 = s[b + sx], v010 = s[b + sy], v110 = s[b + sx + sy];
  double v001 = s[b + sz], v101 = s[b + sx + sz], v011 = s[b + sy + sz], v111 = s[b + sx + sy + sz];
  double c00 = v000 + tx * (v100 - v000);
  double c10 = v010 + tx * (v110 - v010);
  double c01 = v001 + tx * (v101 - v001);
  double c11 = v011 + tx * (v111 - v011);
  double c0 = c00 + ty * (c10 - c00);
  double c1 = c01 + ty * (c11 - c01);
  double phi = c0 + tz * (c1 - c0);
  int nx_ = (int)floor(gx + 0.5), ny_ = (int)floor(gy + 0.5), nz_ = (int)floor(gz + 0.5);
  if (nx_ > R.gx - 1) nx_ = R.gx - 1;
  if (ny_ > R.gy - 1) ny_ = R.gy - 1;
  if (nz_ > R.gz - 1) nz_ = R.gz - 1;
  *tag_out = R.tag[nx_ * sx + ny_ * sy + nz_ * sz];
  return phi;
}

// iteration space: the box itself, or the whole domain minus the box
__device__ __forceinline__ bool geo_cell(const GeoArgs& a, int& x, int& y, int& z) {
  if (a.inside) {
    int bx = a.box.x1 - a.box.x0, by = a.box.y1 - a.box.y0;
    x = a.box.x0 + blockIdx.y * blockDim.x + threadIdx.x;
    int yz = blockIdx.x;
    y = a.box.y0 + yz % by;
    z = a.box.z0 + yz / by;
    return x < a.box.x1 && bx > 0;
  }
  x = blockIdx.y * blockDim.x + threadIdx.x;
  int yz = blockIdx.x;
  y = yz % a.dm.ny;
  z = yz / a.dm.ny;
  if (x >= a.dm.nx) return false;
  bool in_box = x >= a.box.x0 && x < a.box.x1 && y >= a.box.y0 && y < a.box.y1 && z >= a.box.z0 && z < a.box.z1;
  return !in_box;
}

constexpr double ROW_ACT = 3.9;   // see "K1 on the band" below
constexpr int ROW_DILATE = 3;

// pass 1: phi and provisional tag
__global__ void __launch_bounds__(128) geometry_phi_kernel(GeoArgs a) {
  int x, y, z;
  if (!geo_cell(a, x, y, z)) return;
  int64_t c = (int64_t)x + (int64_t)a.dm.nx * ((int64_t)y + (int64_t)a.dm.ny * z);
  double phi = BIG_PHI;
  int tg = 0;
  if (a.has_static) {
    phi = (double)a.phi_static[c];
    tg = a.has_tag_static ? a.tag_static[c] : 1;
  }
  if (a.has_rotor) {
    int rt;
    double pr = rotor_phi(a.rot, a.cth, a.sth, (double)x, (double)y, (double)z, &rt);
    if (pr < phi) {
      phi = pr;
      tg = rt;
    }
  }
  a.phi[c] = phi;
  const bool below = phi < a.h;
  a.below[c] = below ? 1 : 0;
  if (below) a.rowflag[y + a.dm.ny * z] = 1;
  if (phi < ROW_ACT) a.rowact0[y + a.dm.ny * z] = a.rowact1[y + a.dm.ny * z] = 1;
  a.tag_prov[c] = (uint8_t)(tg & TAG_MASK);
}

// ---------------------------------------------------------------------------------------------- K1 on the band
// The paper re-embeds the tagged porosities only in the growth layer around the structure, because the surface
// moves less than a cell per step (Fig. 4 :254-263).  Here the unit is a ROW of the rotor box (fixed y, z;
// the rows run along the rotor axis for the paper's layout): a row is ACTIVE at step m if one of its cells has
// phi_m < ROW_ACT (the reference grid is clipped at 4 cells: an inactive row is at least ~3.9 cells from the
// surface).  Step m evaluates the rows within ROW_DILATE rows (in y and z) of a row that was active at step m-1 or
// m-2 -- two steps, because the two geometry sets alternate and each must see a row turn plain fluid once.  Every
// other row keeps what it has: plain fluid in both sets, no cell below eps/2, no list entry.  A cell can only get
// phi < eps/2 + 1 (anything but plain fluid) at step m if a cell within a few cells of it was active before.
// The rows to evaluate are compacted into a list; both passes then run as a few hundred blocks that walk the list
// (a block per row of a 5-million-cell box is bound by the block dispatch rate, ncu round 1).

__global__ void rows_select_kernel(GeoArgs a) {
  const int by = a.box.y1 - a.box.y0, bz = a.box.z1 - a.box.z0;
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  bool take = false;
  int y = 0, z = 0;
  if (r < by * bz) {
    y = a.box.y0 + r % by;
    z = a.box.z0 + r / by;
    take = a.all_rows != 0;
    for (int dz = -ROW_DILATE; dz <= ROW_DILATE && !take; ++dz) {
      const int zz = wrap_any(z + dz, a.dm.nz, a.dm.mode[2]);
      for (int dy = -ROW_DILATE; dy <= ROW_DILATE; ++dy) {
        const int row = wrap_any(y + dy, a.dm.ny, a.dm.mode[1]) + a.dm.ny * zz;
        take |= (a.rowact0[row] | a.rowact1[row]) != 0;
      }
    }
  }
  const unsigned m = __ballot_sync(0xffffffffu, take);
  if (m) {
    const unsigned lane = threadIdx.x & 31;
    int base = 0;
    if (lane == 0) base = atomicAdd(a.n_rows, __popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (take) a.rowlist[base + __popc(m & ((1u << lane) - 1))] = y + a.dm.ny * z;
  }
}

// pass 1 over the listed rows: phi, below, provisional tag; per row the two flags
__global__ void __launch_bounds__(128) geometry_phi_rows_kernel(GeoArgs a) {
  const int n_rows = *a.n_rows;
  for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
    const int row = a.rowlist[r], y = row % a.dm.ny, z = row / a.dm.ny;
    int any_below = 0, any_act = 0;
    for (int x = a.box.x0 + threadIdx.x; x < a.box.x1; x += blockDim.x) {
      const int64_t c = (int64_t)x + (int64_t)a.dm.nx * row;
      double phi = BIG_PHI;
      int tg = 0;
      if (a.has_static) {
        phi = (double)a.phi_static[c];
        tg = a.has_tag_static ? a.tag_static[c] : 1;
      }
      int rt;
      const double pr = rotor_phi(a.rot, a.cth, a.sth, (double)x, (double)y, (double)z, &rt);
      if (pr < phi) {
        phi = pr;
        tg = rt;
      }
      a.phi[c] = phi;
      const bool below = phi < a.h;
      a.below[c] = below ? 1 : 0;
      a.tag_prov[c] = (uint8_t)(tg & TAG_MASK);
      any_below |= below;
      any_act |= phi < ROW_ACT;
    }
    any_below = __syncthreads_or(any_below);
    any_act = __syncthreads_or(any_act);
    if (threadIdx.x == 0) {
      a.rowflag[row] = (uint8_t)(a.rowflag_static[row] | (any_below ? 1 : 0));
      a.rowact_w[row] = any_act ? 1 : 0;
    }
  }
}

// pass 2: type, porosity, wall-model set (R13) and the compact lists
// pass 2 for the cells (x .. x + blockDim.x) of row (y, z), one cell per thread; `active`: this thread has a cell.
// All threads of the block call it together (shared memory, barrier, ballots).
__device__ __forceinline__ void type_cells(const GeoArgs& a, int x, int y, int z, bool active) {
  int inw = 0, inf = 0;
  int64_t c = 0;
  double y1v[3] = {0, 0, 0};
  // growth-layer test (Fig. 4): some cell of the 3x3x3 neighbourhood has phi < eps/2.
  // The block owns a run of cells of one (y,z) row: every thread ORs the nine rows around it at its own
  // x into one byte (the columns just outside the run by the first and last thread), the 3-wide OR along
  // x then comes from shared memory -- 9 byte loads per cell instead of 26.
  __shared__ uint8_t col[128 + 2];
  bool near_row = false;  // rows with no cell below eps/2 in any of the nine neighbouring rows need no cell test
  {
    const int nx = a.dm.nx, ny = a.dm.ny, nz = a.dm.nz;
    int rows[9];
#pragma unroll
    for (int r = 0; r < 9; ++r) {
      rows[r] = wrap_any(y + r % 3 - 1, ny, a.dm.mode[1]) + ny * wrap_any(z + r / 3 - 1, nz, a.dm.mode[2]);
      near_row |= a.rowflag[rows[r]] != 0;
    }
    if (!near_row) {
      // Most rows of the box (the blades cover a small part of the disc): every cell has phi >= eps/2 and no cell
      // below eps/2 next to it -- plain fluid / fringe / bulk, no tag, not in W, in no list.  The whole block
      // leaves here (y, z are block-uniform), before the barrier and the ballots.
      if (active) {
        int type = HHRR_FLUID;
        float d = 1.f;
        if (a.has_fringe && x >= a.fr_x0 && x < a.fr_x1) {
          type = HHRR_FRINGE;
          d = 0.f;
        }
        if (a.fsi.n > 0) {
          bool inside = false;
          for (int b = 0; b < a.fsi.n; ++b)
            inside |= x >= a.fsi.b[b].x0 && x < a.fsi.b[b].x1 && y >= a.fsi.b[b].y0 && y < a.fsi.b[b].y1 &&
                      z >= a.fsi.b[b].z0 && z < a.fsi.b[b].z1;
          if (!inside) {
            if (type == HHRR_FLUID) type = HHRR_BULK;
            else a.cnt->region_violation = 1;
          }
        }
        const int64_t cc = x + (int64_t)nx * (y + (int64_t)ny * z);
        a.flags[cc] = (uint8_t)type;
        a.d[cc] = d;
      }
      return;
    }
    const int t = threadIdx.x, T = blockDim.x;
    if (near_row) {
      for (int s = t; s < T + 2; s += T) {  // s = t, and t + T for the first two threads
        const int xv = x - t + s - 1;  // columns beyond one past the lattice belong to idle lanes only
        uint8_t v = 0;
        if (xv >= -1 && xv <= nx) {
          const int xs = wrap_any(xv, nx, a.dm.mode[0]);
#pragma unroll
          for (int r = 0; r < 9; ++r) v |= a.below[xs + (int64_t)nx * rows[r]];
        }
        col[s] = v;
      }
    } else {
      for (int s = t; s < T + 2; s += T) col[s] = 0;
    }
    __syncthreads();
  }
  const bool near_below = (col[threadIdx.x] | col[threadIdx.x + 1] | col[threadIdx.x + 2]) != 0;
  if (active) {
    const int nx = a.dm.nx, ny = a.dm.ny, nz = a.dm.nz;
    const int64_t snx = nx, snxy = (int64_t)nx * ny;
    c = x + snx * y + snxy * z;
    // a row with no cell below eps/2 in it or around it (most rows of the box: the blades cover a small part of the
    // disc) holds plain fluid / fringe cells only: phi >= eps/2, no tag, not in W -- nothing to read
    double phi = near_row ? a.phi[c] : BIG_PHI;
    uint8_t fl = (near_row && a.flags_prev) ? a.flags_prev[c] : (uint8_t)0;
    int tg = near_row ? a.tag_prov[c] : 0;
    int type;
    float d;
    if (a.has_fringe && x >= a.fr_x0 && x < a.fr_x1) {
      type = HHRR_FRINGE;
      d = 0.f;
    } else if (phi <= -a.h) {
      type = HHRR_SOLID;
      d = 0.f;
    } else if (phi < a.h) {
      type = HHRR_FRONTIER;
      double dd = phi / a.eps + 0.5;  // Eq. 22
      if (a.has_override && a.has_static && (double)a.phi_static[c] == phi) dd = (double)a.d_override[c];
      d = (float)dd;
    } else {
      type = HHRR_FLUID;
      d = 1.f;
      if (near_below) type = HHRR_GROWTH;
    }
    if (a.fsi.n > 0) {
      bool inside = false;
      for (int b = 0; b < a.fsi.n; ++b)
        inside |= x >= a.fsi.b[b].x0 && x < a.fsi.b[b].x1 && y >= a.fsi.b[b].y0 && y < a.fsi.b[b].y1 &&
                  z >= a.fsi.b[b].z0 && z < a.fsi.b[b].z1;
      if (!inside) {
        if (type == HHRR_FLUID) type = HHRR_BULK;
        else a.cnt->region_violation = 1;  // the boxes do not cover the structure: reported, type kept
      }
    }
    if (type == HHRR_FLUID || type == HHRR_FRINGE || type == HHRR_BULK) tg = 0;
    if (a.wm_enabled && type == HHRR_FRONTIER && phi > 0.0) {
      int xm = wrap_any(x - 1, nx, a.dm.mode[0]), xp = wrap_any(x + 1, nx, a.dm.mode[0]);
      int ym = wrap_any(y - 1, ny, a.dm.mode[1]), yp = wrap_any(y + 1, ny, a.dm.mode[1]);
      int zm = wrap_any(z - 1, nz, a.dm.mode[2]), zp = wrap_any(z + 1, nz, a.dm.mode[2]);
      double gr0 = 0.5 * (a.phi[xp + snx * y + snxy * z] - a.phi[xm + snx * y + snxy * z]);
      double gr1 = 0.5 * (a.phi[x + snx * yp + snxy * z] - a.phi[x + snx * ym + snxy * z]);
      double gr2 = 0.5 * (a.phi[x + snx * y + snxy * zp] - a.phi[x + snx * y + snxy * zm]);
      double nn = sqrt(gr0 * gr0 + gr1 * gr1 + gr2 * gr2);
      if (nn > 1e-12 && nn < 1e20) {
        inw = 1;
        y1v[0] = phi * (gr0 / nn);
        y1v[1] = phi * (gr1 / nn);
        y1v[2] = phi * (gr2 / nn);
      }
    }
    inf = (type == HHRR_SOLID || type == HHRR_FRONTIER) && tg > 0;
    uint8_t valid = inw ? (fl & WM_VALID) : 0;  // arrays of cells not in W_n are invalidated
    const int stored = (type == HHRR_FRONTIER && inw) ? T_FRONTIER_W : type;  // membership of W rides in the type bits
    a.flags[c] = (uint8_t)(stored | (tg << TAG_SHIFT) | valid);
    a.d[c] = d;
  }
  // warp-aggregated appends keep the lists nearly in cell order
  unsigned lane = threadIdx.x & 31;
  unsigned mw = __ballot_sync(0xffffffffu, inw);
  if (mw) {
    int base = 0;
    if (lane == 0) base = atomicAdd(&a.cnt->wall_count, __popc(mw));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (inw) {
      int slot = base + __popc(mw & ((1u << lane) - 1));
      if (slot < a.cap_list) {
        a.wall_idx[slot] = (int32_t)c;
        a.wall_y1n[3 * (int64_t)slot] = y1v[0];
        a.wall_y1n[3 * (int64_t)slot + 1] = y1v[1];
        a.wall_y1n[3 * (int64_t)slot + 2] = y1v[2];
      } else {
        a.cnt->overflow = 1;
      }
    }
  }
  unsigned mf = __ballot_sync(0xffffffffu, inf);
  if (mf) {
    int base = 0;
    if (lane == 0) base = atomicAdd(&a.cnt->force_count, __popc(mf));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (inf) {
      int slot = base + __popc(mf & ((1u << lane) - 1));
      if (slot < a.cap_list)
        a.force_idx[slot] = (int32_t)c;
      else
        a.cnt->overflow = 1;
    }
  }
}

__global__ void __launch_bounds__(128) geometry_type_kernel(GeoArgs a) {
  int x, y, z;
  const bool active = geo_cell(a, x, y, z);
  type_cells(a, x, y, z, active);
}

// pass 2 over the listed rows
__global__ void __launch_bounds__(128) geometry_type_rows_kernel(GeoArgs a) {
  const int n_rows = *a.n_rows;
  for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
    const int row = a.rowlist[r], y = row % a.dm.ny, z = row / a.dm.ny;
    for (int xb = a.box.x0; xb < a.box.x1; xb += blockDim.x) {
      const int x = xb + threadIdx.x;
      type_cells(a, x, y, z, x < a.box.x1);
      __syncthreads();  // the shared column bytes are reused by the next segment / row
    }
  }
}

__global__ void counters_kernel(Counters* cnt, int op) {
  if (op == 0) {  // start a full rebuild
    cnt->wall_count = cnt->force_count = 0;
    cnt->wall_static = cnt->force_static = 0;
  } else if (op == 1) {  // static prefix complete
    cnt->wall_count = min(cnt->wall_count, 0x7fffffff);
    cnt->wall_static = cnt->wall_count;
    cnt->force_static = cnt->force_count;
  } else {  // start a box update
    cnt->wall_count = cnt->wall_static;
    cnt->force_count = cnt->force_static;
  }
}

static void geo_grid(const GeoArgs& a, dim3& g, dim3& b) {
  const int max_threads = 128;
  if (a.inside) {
    int bx = a.box.x1 - a.box.x0, by = a.box.y1 - a.box.y0, bz = a.box.z1 - a.box.z0;
    int t = bx >= max_threads ? max_threads : ((bx + 31) / 32) * 32;  // a rotor box is thin along its axis: do not idle warps
    b = dim3(t);
    g = dim3(by * bz, (bx + t - 1) / t);
  } else {
    b = dim3(128);
    g = dim3(a.dm.ny * a.dm.nz, (a.dm.nx + 127) / 128);
  }
}

static void fill_geo(hhrr_lattice* L, GeoArgs& a, int64_t step) {
  a.dm = L->dom;
  a.h = 0.5 * L->p.eps_cells;
  a.eps = L->p.eps_cells;
  a.has_static = L->has_static;
  a.has_tag_static = L->has_tag_static;
  a.has_override = L->has_override;
  a.has_fringe = L->has_fringe;
  a.has_rotor = L->has_rotor;
  a.wm_enabled = L->wm_enabled;
  a.fsi = L->fsi;
  a.fr_x0 = L->fr_x0;
  a.fr_x1 = L->fr_x1;
  a.cth = 1.0;
  a.sth = 0.0;
  if (L->has_rotor) {
    double th = L->rot.theta0 + (double)step * L->rot.omega;  // rigid rotation only
    a.cth = cos(th);
    a.sth = sin(th);
    a.rot.sdf = L->rot_sdf;
    a.rot.tag = L->rot_tag;
    a.rot.gx = L->rot.gx;
    a.rot.gy = L->rot.gy;
    a.rot.gz = L->rot.gz;
    a.rot.spacing = L->rot.spacing;
    for (int k = 0; k < 3; ++k) {
      a.rot.origin[k] = L->rot.origin[k];
      a.rot.centre[k] = L->rot.centre[k];
      a.rot.axis[k] = L->rot.axis[k];
    }
  } else {
    a.rot = RotorDev{};
  }
  a.phi_static = L->phi_static;
  a.tag_static = L->tag_static;
  a.d_override = L->d_override;
  a.phi = L->phi;
  a.below = L->below;
  a.rowflag = L->rowflag;
  a.rowflag_static = L->rowflag_static;
  a.rowact0 = L->rowact[0];
  a.rowact1 = L->rowact[1];
  a.rowact_w = L->rowact[step & 1];
  a.rowlist = L->rowlist;
  a.n_rows = L->n_rows;
  a.all_rows = L->band_ok ? 0 : 1;
  a.tag_prov = L->tag_prov;
  a.flags_prev = L->flags;
  a.flags = L->flags;
  a.d = L->d;
  a.wall_idx = L->wall_idx;
  a.wall_y1n = L->wall_y1n;
  a.force_idx = L->force_idx;
  a.cnt = L->counters;
  a.cap_list = (int)L->cap_list;
}

static bool rotor_box_empty(const hhrr_lattice* L) {
  const Box& rb = L->rot_box;
  return !L->has_rotor || rb.x1 <= rb.x0 || rb.y1 <= rb.y0 || rb.z1 <= rb.z0;
}

// geometry(step) over the rotor box on stream s, into the geometry set `a` points at: row selection, pass 1
// (phi / below / row flags / provisional tag -- nothing a collide-stream, wall-model or force kernel touches),
// list reset, pass 2.  Both passes walk the row list with a fixed number of blocks.
static void launch_box_rows(hhrr_lattice* L, GeoArgs& a, cudaStream_t s) {
  a.box = L->rot_box;
  a.inside = 1;
  const int rows = (a.box.y1 - a.box.y0) * (a.box.z1 - a.box.z0);
  const int bx = a.box.x1 - a.box.x0;
  const int t = bx >= 128 ? 128 : ((bx + 31) / 32) * 32;  // a rotor box is thin along its axis: do not idle warps
  cudaMemsetAsync(L->n_rows, 0, sizeof(int), s);
  rows_select_kernel<<<(rows + 127) / 128, 128, 0, s>>>(a);
  geometry_phi_rows_kernel<<<4736, t, 0, s>>>(a);  // latency-bound rows: many short blocks in flight, still 14 x fewer than one per row
  counters_kernel<<<1, 1, 0, s>>>(a.cnt, 2);
  geometry_type_rows_kernel<<<4736, t, 0, s>>>(a);
  L->launches += 4;
}

void swap_geometry_sets(hhrr_lattice* L) {
  std::swap(L->flags, L->alt_flags);
  std::swap(L->d, L->alt_d);
  std::swap(L->wall_idx, L->alt_wall_idx);
  std::swap(L->wall_y1n, L->alt_wall_y1n);
  std::swap(L->force_idx, L->alt_force_idx);
  std::swap(L->counters, L->alt_counters);
}

// Look-ahead: geometry(step + 1) depends on the step count only (rigid rotation).  Both passes are
// queued on the side stream behind the launch of the collide-stream kernel of `step` (they get SMs from its last
// wave of blocks on, and then share the machine with the wall model), and write the
// ALTERNATE geometry set (flags, porosity, lists, counters), which nothing of `step` reads; hhrr_step swaps the
// sets when it reaches step + 1.  The one thing that depends on the step in between -- whether a cell of
// W_{n+1} holds wall-model state -- is the WM_VALID bit, left 0 here and set by that step's wall-model kernel
// (it knows the cell is in W_{n+1} from the type bits written here).
// Ordering: ev_pre (main stream, recorded before the collide-stream launch) covers every earlier reader of the
// alternate set and of phi / below / rowflag / tag_prov; the side stream itself orders the force kernel of the
// previous step (which reads the alternate set's flags and force list) before this.
cudaError_t launch_geometry_ahead(hhrr_lattice* L) {
  if (!L->side || !L->lookahead || rotor_box_empty(L) || L->geometry_dirty) return cudaSuccess;
  cudaStreamWaitEvent(L->side, L->ev_pre, 0);
  GeoArgs a;
  fill_geo(L, a, L->step + 1);
  a.flags_prev = nullptr;
  a.flags = L->alt_flags;
  a.d = L->alt_d;
  a.wall_idx = L->alt_wall_idx;
  a.wall_y1n = L->alt_wall_y1n;
  a.force_idx = L->alt_force_idx;
  a.cnt = L->alt_counters;
  launch_box_rows(L, a, L->side);
  cudaEventRecord(L->ev_k1, L->side);
  L->ahead_step = L->step + 1;
  L->side_busy = true;
  return cudaGetLastError();
}

// after a full pass: the alternate set starts as a copy of the current one (cells outside the rotor box and the
// static prefix of the lists never change afterwards)
__global__ void copy_static_lists_kernel(const Counters* cnt, Counters* alt_cnt, const int32_t* wall_idx,
                                         const double* wall_y1n, const int32_t* force_idx, int32_t* alt_wall_idx,
                                         double* alt_wall_y1n, int32_t* alt_force_idx, int cap) {
  const int nw = min(cnt->wall_static, cap), nf = min(cnt->force_static, cap);
  const int t = blockIdx.x * blockDim.x + threadIdx.x, T = gridDim.x * blockDim.x;
  for (int e = t; e < nw; e += T) {
    alt_wall_idx[e] = wall_idx[e];
    for (int q = 0; q < 3; ++q) alt_wall_y1n[3 * (int64_t)e + q] = wall_y1n[3 * (int64_t)e + q];
  }
  for (int e = t; e < nf; e += T) alt_force_idx[e] = force_idx[e];
  if (t == 0) *alt_cnt = *cnt;
}

cudaError_t launch_geometry(hhrr_lattice* L, bool full) {
  GeoArgs a;
  fill_geo(L, a, L->step);
  Box none = {0, 0, 0, 0, 0, 0};
  Box rb = L->has_rotor ? L->rot_box : none;
  dim3 g, b;
  bool box_empty = rb.x1 <= rb.x0 || rb.y1 <= rb.y0 || rb.z1 <= rb.z0;
  const size_t rows = (size_t)L->dom.ny * L->dom.nz;
  if (L->ahead_step >= 0) {  // a look-ahead result nobody will use: let the side stream finish writing first
    cudaStreamWaitEvent(L->stream, L->ev_k1, 0);
    L->ahead_step = -1;
  }
  if (full) {
    // phi everywhere, then types: outside the rotor box first (static list prefix), box last
    a.box = none;
    a.inside = 0;
    geo_grid(a, g, b);
    cudaMemsetAsync(L->rowflag, 0, rows, L->stream);
    cudaMemsetAsync(L->rowact[0], 0, rows, L->stream);
    cudaMemsetAsync(L->rowact[1], 0, rows, L->stream);
    geometry_phi_kernel<<<g, b, 0, L->stream>>>(a);
    // what the full pass marks (static geometry and the rotor at this angle) stays marked: a superset
    cudaMemcpyAsync(L->rowflag_static, L->rowflag, rows, cudaMemcpyDeviceToDevice, L->stream);
    counters_kernel<<<1, 1, 0, L->stream>>>(L->counters, 0);
    a.box = rb;
    geometry_type_kernel<<<g, b, 0, L->stream>>>(a);
    counters_kernel<<<1, 1, 0, L->stream>>>(L->counters, 1);
    L->launches += 4;
    // alternate set := current set outside the rotor box (the box part is rewritten by every look-ahead pass)
    cudaMemcpyAsync(L->alt_flags, L->flags, (size_t)L->dom.n, cudaMemcpyDeviceToDevice, L->stream);
    cudaMemcpyAsync(L->alt_d, L->d, sizeof(float) * (size_t)L->dom.n, cudaMemcpyDeviceToDevice, L->stream);
    copy_static_lists_kernel<<<592, 256, 0, L->stream>>>(L->counters, L->alt_counters, L->wall_idx, L->wall_y1n,
                                                         L->force_idx, L->alt_wall_idx, L->alt_wall_y1n,
                                                         L->alt_force_idx, (int)L->cap_list);
    L->launches++;
    if (!box_empty) {
      a.inside = 1;
      geo_grid(a, g, b);
      geometry_type_kernel<<<g, b, 0, L->stream>>>(a);
      L->launches++;
    }
  } else if (!box_empty) {
    launch_box_rows(L, a, L->stream);
  }
  return cudaGetLastError();
}

}  // namespace hhrr
