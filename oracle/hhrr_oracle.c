/*
 * hhrr_oracle.c -- plain fp64 CPU oracle of the HHRRLBM + wall-model time step.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.  It
 * shares no code, header, table or constant generator with the CUDA path
 * (paper_2510_13726_b200/csrc); neither includes or links the other.
 *
 * Written from /root/reference/PAPER.md (arxiv 2510.13726); every function cites
 * the PAPER.md line / equation it follows.  Where the paper is silent or garbled
 * the reading taken is the one listed in DESIGN.md ("Readings", R1..R19) and is
 * named in the comment.  Everything is the algorithm step by step in the order of
 * Listing 3: two full population buffers, every cell treated
 * identically, geometry recomputed brute force for all cells each step.  No
 * blocking, fusion or reordering.  OpenMP over cells is wall-clock only.
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): lattice isotropy,
 * equilibrium moments, collision invariants, HLBM d=1 / d=0 limits, Taylor-Green
 * decay rate (viscosity + sign of Eq. 7/10), Smagorinsky closed form, Poiseuille
 * second difference (body force + porosity-0 wall), momentum-exchange force =
 * total body force, Spalding relation to 1e-12 + asymptotes, level set d=1/2,
 * sphere volume, rigid rotation => S^FD = 0, bulk region = the sigma = 1 scheme.
 * PARITY UNPINNED: rotor thrust / wake against the paper's Fig. 7-10 (needs the
 * geometry and data of its ref. [19], not available) -- see DESIGN.md.
 *
 * Conventions: cell (x,y,z), linear index
 * x + nx*(y + ny*z); direction i = (cx+1) + 3(cy+1) + 9(cz+1); rest i=13;
 * opposite 26-i; w(0)=2/3, w(+-1)=1/6; cs^2 = 1/3; dx = dt = 1.  (D3Q19: the 19 of these
 * directions with |c|^2 <= 2 renumbered in the same order, rest 9, opposite 18-i, weights
 * 1/3, 1/18, 1/36.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* Velocity set: D3Q27 (BASELINE.json's configs; default) or D3Q19 (the paper's own lattice, Fig. 2
 * :107) when compiled through oracle/hhrr_oracle_q19.c, which defines OHRR_Q 19 and includes this file.  The
 * directions of D3Q19 are those of D3Q27 with |c|^2 <= 2, in the same order.                                 */
#ifndef OHRR_Q
#define OHRR_Q 27
#endif
#define Q OHRR_Q
#define MAX_TAGS 16
#define BIG_PHI 1.0e30

enum { T_FLUID = 0, T_GROWTH = 1, T_FRONTIER = 2, T_SOLID = 3, T_FRINGE = 4, T_BULK = 5 };
#define MAX_FSI_BOXES 8
enum { AX_PERIODIC = 0, AX_MIRROR = 1 };

typedef struct {
  int32_t nx, ny, nz;
  int32_t mode[3];
  double tau0, sigma, smagorinsky_cs;
  double body_force[3];
  double eps_cells;
  double kappa, E;
  int32_t newton_max_iter;
  double newton_tol;
  double sampling_distance;
} ohrr_params;

typedef struct {
  const float *sdf;
  const uint8_t *tag;
  int32_t gx, gy, gz;
  double spacing;
  double origin[3];
  double centre[3], axis[3], omega, theta0;
  int32_t n_tags;
} ohrr_rotor_desc;

typedef struct {
  double centre[3], omega[3], vel[3];
} body_t;

typedef struct ohrr_lattice {
  ohrr_params p;
  int64_t n;
  double *f, *f2;      /* Q planes of n doubles each: f[i*n + cell]                      */
  double *uhat, *rho;  /* time-n homogenised velocity (3 planes) and density, step 2 of O2 */
  /* geometry inputs */
  double *phi_static;  /* n or NULL */
  uint8_t *tag_static; /* n or NULL */
  double *d_override;  /* n or NULL */
  int has_fringe, fr_x0, fr_x1;
  double fr_u[3];
  int has_rotor;
  ohrr_rotor_desc rot;
  float *rot_sdf;
  uint8_t *rot_tag;
  body_t body[MAX_TAGS];
  int wm_enabled;
  /* geometry state, recomputed brute force every step (O1) */
  double *phi, *d;
  uint8_t *type, *tag, *in_w;
  double *y1n; /* 3 per cell (AoS)  */
  /* wall-model state keyed by cell */
  uint8_t *wm_valid;
  double *wm_utau, *wm_u /*3 AoS*/, *wm_s /*6 AoS: xx yy zz xy xz yz*/;
  /* forces */
  double *force; /* [cap][MAX_TAGS][3] */
  double *torque; /* [cap][MAX_TAGS][3]: moment of the same per-cell forces about the body's centre */
  int64_t force_cap;
  int64_t step;
  int geometry_current; /* geometry(step) already evaluated */
  /* region split (Listing 2 :271-302): union of half-open cell boxes x0 x1 y0 y1 z0 z1 that
   * holds the wall-modelled / FSI part of the domain; fluid cells outside run the bulk RRLBM-LES model */
  int n_fsi;
  int32_t fsi[MAX_FSI_BOXES][6];
  int region_violation; /* a cell that is not plain fluid was found outside every box */
  int wm_slip;          /* 0: u_wm = u_tau e_t (R8); 1: u_wm = u_tau u+(y1+) e_t (R22, SURVEY C8 alt.) */
  int wm_shear;         /* 0: one-sided difference (R10); 1: analytic slope of the wall function (R22, C10 alt.) */
  int wall_function;    /* 0: truncated Spalding (the paper's, Eq. 18); 1: Musker's profile (BASELINE.json config 3) */
} ohrr_lattice;

/* ---------------------------------------------------------------- lattice tables */
static int CX[Q], CY[Q], CZ[Q];
static double W[Q];
static int DIR_OF[27]; /* index of direction (cx,cy,cz) at slot (cx+1) + 3(cy+1) + 9(cz+1); -1: not in the set */
static int REST;       /* index of the rest direction */
static int tables_ready = 0;
static const double CS2 = 1.0 / 3.0;

static void init_tables(void) {
  if (tables_ready) return;
  int i = 0;
  for (int k = 0; k < 27; ++k) {
    int cx = k % 3 - 1, cy = (k / 3) % 3 - 1, cz = k / 9 - 1;
    int nn = abs(cx) + abs(cy) + abs(cz);
    DIR_OF[k] = -1;
    if (Q == 19 && nn == 3) continue; /* D3Q19 has no corner directions (Fig. 2) */
    CX[i] = cx;
    CY[i] = cy;
    CZ[i] = cz;
    if (Q == 27) {
      double w = 1.0;
      w *= (cx == 0) ? 2.0 / 3.0 : 1.0 / 6.0;
      w *= (cy == 0) ? 2.0 / 3.0 : 1.0 / 6.0;
      w *= (cz == 0) ? 2.0 / 3.0 : 1.0 / 6.0;
      W[i] = w;
    } else {
      W[i] = nn == 0 ? 1.0 / 3.0 : (nn == 1 ? 1.0 / 18.0 : 1.0 / 36.0);
    }
    if (nn == 0) REST = i;
    DIR_OF[k] = i;
    ++i;
  }
  tables_ready = 1;
}
static inline int dir_of(int cx, int cy, int cz) { return DIR_OF[(cx + 1) + 3 * (cy + 1) + 9 * (cz + 1)]; }
static inline int opposite(int i) { return dir_of(-CX[i], -CY[i], -CZ[i]); }
int32_t ohrr_q(void) { return Q; }

static inline void cvec(int i, double c[3]) {
  c[0] = CX[i];
  c[1] = CY[i];
  c[2] = CZ[i];
}
static inline double delta(int a, int b) { return a == b ? 1.0 : 0.0; }
/* Hermite polynomials of the discrete velocity (Eq. 8). */
static inline double H2(const double c[3], int a, int b) { return c[a] * c[b] - (1.0 / 3.0) * delta(a, b); }
static inline double H3(const double c[3], int a, int b, int g) {
  return c[a] * c[b] * c[g] - (1.0 / 3.0) * (c[a] * delta(b, g) + c[b] * delta(a, g) + c[g] * delta(a, b));
}

/* Third-order part of the Hermite expansion, sum over the supported third-order polynomials of
 * H^(3)_i : a^(3) with the normalisation of Eq. 8.
 * D3Q27: every H^(3)_abg is supported (H_aaa = 0 identically): the full contraction / (3! c_s^6)  (reading R3).
 * D3Q19: the six H_aab are no longer independent; the supported third-order basis is the one of the paper's
 * ref. [43] (Jacob, Malaspinas, Sagaut 2018; named at PAPER.md:94): the sums H_xxy + H_yzz, H_xzz + H_xyy,
 * H_yyz + H_xxz (squared norm 2 c_s^6 -- the "2 c_s^6" printed in Eq. 11) and the differences
 * H_xxy - H_yzz, H_xzz - H_xyy, H_yyz - H_xxz (squared norm 6 c_s^6); H_xyz is not supported  (reading R23). */
static double third_order(const double c[3], double a3[3][3][3]) {
  const double cs6 = CS2 * CS2 * CS2;
  if (Q == 27) {
    double t3 = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        for (int g = 0; g < 3; ++g) t3 += H3(c, a, b, g) * a3[a][b][g];
    return t3 / (6.0 * cs6);
  }
  static const int G1[3][3] = {{0, 0, 1}, {0, 2, 2}, {1, 1, 2}}; /* xxy, xzz, yyz */
  static const int G2[3][3] = {{1, 2, 2}, {0, 1, 1}, {0, 0, 2}}; /* yzz, xyy, xxz */
  double t3 = 0.0;
  for (int k = 0; k < 3; ++k) {
    double h1 = H3(c, G1[k][0], G1[k][1], G1[k][2]), h2 = H3(c, G2[k][0], G2[k][1], G2[k][2]);
    double a1 = a3[G1[k][0]][G1[k][1]][G1[k][2]], a2 = a3[G2[k][0]][G2[k][1]][G2[k][2]];
    t3 += (h1 + h2) * (a1 + a2) / (2.0 * cs6) + (h1 - h2) * (a1 - a2) / (6.0 * cs6);
  }
  return t3;
}

/* exported for the pins */
void ohrr_lattice_tables(int32_t *cx, int32_t *cy, int32_t *cz, double *w) {
  init_tables();
  for (int i = 0; i < Q; ++i) {
    cx[i] = CX[i];
    cy[i] = CY[i];
    cz[i] = CZ[i];
    w[i] = W[i];
  }
}

/* ---------------------------------------------------------------- cell-model pieces */

/* Third-order Hermite equilibrium, PAPER.md:126-129 (Eq. 11) with a0^(n) = a0^(n-1) u.
 * Reading R3: the third-order term is the full tensor contraction with 1/(c_s^6 3!)
 * of Eq. 8; Eq. 11's "2 c_s^6" counts the distinct components.     */
void ohrr_equilibrium(double rho, const double u[3], double feq[Q]) {
  init_tables();
  for (int i = 0; i < Q; ++i) {
    double c[3];
    cvec(i, c);
    double t1 = 0.0, t2 = 0.0;
    for (int a = 0; a < 3; ++a) t1 += c[a] * rho * u[a];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += H2(c, a, b) * rho * u[a] * u[b];
    double a3[3][3][3]; /* a0^(3) = a0^(2) u = rho u u u */
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        for (int g = 0; g < 3; ++g) a3[a][b][g] = rho * u[a] * u[b] * u[g];
    feq[i] = W[i] * (rho + t1 / CS2 + t2 / (2.0 * CS2 * CS2) + third_order(c, a3));
  }
}

/* Regularised non-equilibrium from a1^(2) (symmetric 3x3) and the recursion
 * a1^(3)_abg = u_a a2_bg + u_b a2_ag + u_g a2_ab (reading R3; refs [42,43] of the
 * paper).  n = 0, 1 terms of Eq. 8 are zero (mass, momentum).         */
static void regularised_f1(const double a2[3][3], const double u[3], double f1[Q]) {
  double a3[3][3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      for (int g = 0; g < 3; ++g) a3[a][b][g] = u[a] * a2[b][g] + u[b] * a2[a][g] + u[g] * a2[a][b];
  for (int i = 0; i < Q; ++i) {
    double c[3];
    cvec(i, c);
    double t2 = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += H2(c, a, b) * a2[a][b];
    f1[i] = W[i] * (t2 / (2.0 * CS2 * CS2) + third_order(c, a3));
  }
}

/* Smagorinsky effective relaxation time, PAPER.md:84-90 (Eq. 3-5) and :144 (Eq. 14).
 * Reading R6: |S| from the local Pi^neq via S = -Pi^neq/(2 rho cs^2 tau_eff);
 * solving Eq. 4 + Eq. 14 for tau_eff gives the closed form below, with
 * Q = sqrt(2 Pi:Pi).                                                                */
double ohrr_tau_eff(double tau0, double cs_smago, double rho, const double pi[3][3]) {
  double pp = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) pp += pi[a][b] * pi[a][b];
  double Qn = sqrt(2.0 * pp);
  return 0.5 * (tau0 + sqrt(tau0 * tau0 + 18.0 * cs_smago * cs_smago * Qn / rho));
}

/* One HHRRLBM collision (O2 steps 1-7), PAPER.md:98 (Eq. 6), :102 (Eq. 7),
 * :122 (Eq. 10), :133 (Eq. 12, orientation per reading R1: d=1 fluid).
 *   fin[Q]      pre-collision populations of the cell
 *   g[3]        body force (reading R11)
 *   d, uB[3]    porosity and solid (+ wall-model slip) velocity
 *   S[3][3]     strain rate handed to the hybrid term (FD or wall-model)
 *   sigma       hybridisation factor used for THIS cell (0 on wall-model cells)
 * outputs: fout[Q]; diag[0]=rho, diag[1..3]=uhat, diag[4]=tau_eff                   */
void ohrr_collide_cell(const double fin[Q], const double g[3], double d, const double uB[3],
                       const double S[3][3], double sigma, double tau0, double cs_smago,
                       double fout[Q], double diag[5]) {
  init_tables();
  /* 1. rho, j, u   (Listing 1 lines 4-5) */
  double rho = 0.0, j[3] = {0, 0, 0};
  for (int i = 0; i < Q; ++i) {
    rho += fin[i];
    j[0] += CX[i] * fin[i];
    j[1] += CY[i] * fin[i];
    j[2] += CZ[i] * fin[i];
  }
  double u[3], uh[3];
  for (int a = 0; a < 3; ++a) u[a] = (j[a] + g[a]) / rho;
  /* 2. homogenised velocity, Eq. 12 (R1) */
  for (int a = 0; a < 3; ++a) uh[a] = d * u[a] + (1.0 - d) * uB[a];
  /* 3. Pi^neq = sum H2 f - rho uh uh   (BulkStress; reading R4) */
  double pi[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      double s = 0.0;
      for (int i = 0; i < Q; ++i) {
        double c[3];
        cvec(i, c);
        s += H2(c, a, b) * fin[i];
      }
      pi[a][b] = s - rho * uh[a] * uh[b];
    }
  /* 4. tau_eff */
  double tau = ohrr_tau_eff(tau0, cs_smago, rho, pi);
  /* 6. hybrid a1^(2) = sigma Pi^neq - (1-sigma) 2 rho cs^2 tau_eff S   (Eq. 7 + Eq. 10, R2) */
  double a2[3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      a2[a][b] = sigma * pi[a][b] - (1.0 - sigma) * 2.0 * rho * CS2 * tau * S[a][b];
  double f1[Q], feq[Q];
  regularised_f1(a2, uh, f1);
  ohrr_equilibrium(rho, uh, feq);
  /* 7. Eq. 6 */
  for (int i = 0; i < Q; ++i) fout[i] = feq[i] + (1.0 - 1.0 / tau) * f1[i];
  if (diag) {
    diag[0] = rho;
    diag[1] = uh[0];
    diag[2] = uh[1];
    diag[3] = uh[2];
    diag[4] = tau;
  }
}

/* Truncated Spalding wall function residual, PAPER.md:172 (Eq. 18), and its
 * derivative with respect to u_tau (derived; R9).                         */
double ohrr_spalding_f(double utau, double U, double y, double nu, double kappa, double E) {
  double up = U / utau, k = kappa * up;
  return up + (exp(k) - 1.0 - k - 0.5 * k * k - k * k * k / 6.0) / E - y * utau / nu;
}
static double spalding_df(double utau, double U, double y, double nu, double kappa, double E) {
  double up = U / utau, k = kappa * up;
  return -(U / (utau * utau)) * (1.0 + (kappa / E) * (exp(k) - 1.0 - k - 0.5 * k * k)) - y / nu;
}
/* Musker's explicit law of the wall (A. J. Musker, AIAA J. 17 (1979) 655): the closed-form integral of
 * du+/dy+ = (kappa + C y+^2) / (kappa + C y+^2 + C kappa y+^3), kappa = 0.41, C = 0.001093,
 *   u+(y+) = 5.424 atan((2 y+ - 8.15)/16.7) + log10((y+ + 10.6)^9.6 / (y+^2 - 8.15 y+ + 86)^2) - 3.52.
 * Alternative wall function named by BASELINE.json ("Spalding/Musker", config 3); the paper
 * itself uses Spalding only.  Residual in the same form as Eq. 18: f(u_tau) = U/u_tau - u+(y u_tau/nu).  */
double ohrr_musker_uplus(double yp) {
  return 5.424 * atan((2.0 * yp - 8.15) / 16.7) +
         log10(pow(yp + 10.6, 9.6) / ((yp * yp - 8.15 * yp + 86.0) * (yp * yp - 8.15 * yp + 86.0))) - 3.52;
}
static double musker_duplus(double yp) {
  double a = (2.0 * yp - 8.15) / 16.7;
  return 5.424 * (2.0 / 16.7) / (1.0 + a * a) +
         (9.6 / (yp + 10.6) - 2.0 * (2.0 * yp - 8.15) / (yp * yp - 8.15 * yp + 86.0)) / log(10.0);
}
double ohrr_musker_f(double utau, double U, double y, double nu) { return U / utau - ohrr_musker_uplus(y * utau / nu); }
static double musker_df(double utau, double U, double y, double nu) {
  return -U / (utau * utau) - musker_duplus(y * utau / nu) * y / nu;
}
/* the same Newton iteration and stop rule as ohrr_newton_utau (Eq. 19) on Musker's residual */
double ohrr_newton_utau_musker(double u0, double U, double y, double nu, int max_iter, double tol, int32_t *iters) {
  double ua = u0, fa = ohrr_musker_f(ua, U, y, nu);
  int it = 0;
  double ub = ua;
  for (it = 0; it < max_iter; ++it) {
    ub = ua - fa / musker_df(ua, U, y, nu);
    if (!(ub > 0.0)) ub = 0.5 * ua;
    double fb = ohrr_musker_f(ub, U, y, nu);
    double df = fabs(fb - fa);
    ua = ub;
    fa = fb;
    if (df < tol) {
      ++it;
      break;
    }
  }
  if (iters) *iters = it;
  return ub;
}

/* Second readings of the two ambiguous wall-model passages (R22; SURVEY 8(c) C8 / C10 alt., 8(f)-4).
 *
 * u+(y+) of the truncated Spalding law: Eq. 17 gives y+(u+); its inverse by Newton on
 *   h(u+) = u+ + (exp(k) - 1 - k - k^2/2 - k^3/6)/E - y+,  k = kappa u+,  h' = 1 + (kappa/E)(exp(k) - 1 - k - k^2/2),
 * h increasing and convex for u+ >= 0, start at min(y+, 60/kappa) (y+ >= root: the bracket is >= 0), run until
 * the step no longer changes u+ in double precision (at most 200 steps).                                      */
double ohrr_spalding_uplus(double yp, double kappa, double E) {
  if (!(yp > 0.0)) return 0.0;
  double u = yp < 60.0 / kappa ? yp : 60.0 / kappa;
  for (int it = 0; it < 200; ++it) {
    double k = kappa * u, ek = exp(k);
    double h = u + (ek - 1.0 - k - 0.5 * k * k - k * k * k / 6.0) / E - yp;
    double dh = 1.0 + (kappa / E) * (ek - 1.0 - k - 0.5 * k * k);
    double un = u - h / dh;
    int done = !(fabs(un - u) > 1e-15 * fabs(un));
    u = un;
    if (done) break;
  }
  return u;
}
/* "wall modelled velocities ... at Y1": the wall-function velocity at the cell's own wall
 * distance y1, u(y1) = u_tau u+(y1 u_tau/nu), in units of u_tau (Eq. 15-16).                            */
double ohrr_wall_uplus(int kind, double yp, double kappa, double E) {
  return kind == 1 ? ohrr_musker_uplus(yp) : ohrr_spalding_uplus(yp, kappa, E);
}
/* Wall-normal slope du/dy of the wall-function profile at the sampling point (y, U), given u_tau:
 * du/dy = (u_tau^2/nu) du+/dy+ (Eq. 15-16); Spalding: du+/dy+ = 1/(dy+/du+) from Eq. 17 at u+ = U/u_tau,
 * Musker: his defining slope at y+ = y u_tau/nu.                                                          */
double ohrr_wall_shear(int kind, double utau, double U, double y, double nu, double kappa, double E) {
  double slope;
  if (kind == 1) {
    slope = musker_duplus(y * utau / nu);
  } else {
    double k = kappa * (U / utau);
    slope = 1.0 / (1.0 + (kappa / E) * (exp(k) - 1.0 - k - 0.5 * k * k));
  }
  return utau * utau / nu * slope;
}

/* Newton-Raphson, PAPER.md:177 (Eq. 19), stop rule PAPER.md:184: until
 * |f(u^{j+1}) - f(u^j)| < tol or max_iter iterations.  Safeguard (R9): a step to a
 * non-positive value is replaced by halving.  Returns u_tau; *iters = iterations run. */
double ohrr_newton_utau(double u0, double U, double y, double nu, double kappa, double E,
                        int max_iter, double tol, int32_t *iters) {
  double ua = u0, fa = ohrr_spalding_f(ua, U, y, nu, kappa, E);
  int it = 0;
  double ub = ua;
  for (it = 0; it < max_iter; ++it) {
    ub = ua - fa / spalding_df(ua, U, y, nu, kappa, E);
    if (!(ub > 0.0)) ub = 0.5 * ua;
    double fb = ohrr_spalding_f(ub, U, y, nu, kappa, E);
    double df = fabs(fb - fa);
    ua = ub;
    fa = fb;
    if (df < tol) {
      ++it;
      break;
    }
  }
  if (iters) *iters = it;
  return ub;
}

/* ---------------------------------------------------------------- lattice helpers */
static inline int64_t lidx(const ohrr_lattice *L, int x, int y, int z) {
  return (int64_t)x + (int64_t)L->p.nx * ((int64_t)y + (int64_t)L->p.ny * (int64_t)z);
}
/* Neighbour lookup with the outer-boundary rule of reading R12: PERIODIC wraps;
 * on a MIRROR axis the image of an outside cell is the cell reflected in the plane
 * half a cell outside the last cell, and flip[a]=1 says component a changes sign.  */
static inline int wrap1(int v, int n, int mode, int *flip) {
  *flip = 0;
  if (v >= 0 && v < n) return v;
  if (mode == AX_PERIODIC) return ((v % n) + n) % n;
  *flip = 1;
  if (v < 0) return -1 - v;
  return 2 * n - 1 - v;
}

static void body_velocity(const ohrr_lattice *L, int tag, int x, int y, int z, double us[3]) {
  const body_t *b = &L->body[tag];
  double r[3] = {x - b->centre[0], y - b->centre[1], z - b->centre[2]};
  us[0] = b->vel[0] + (b->omega[1] * r[2] - b->omega[2] * r[1]);
  us[1] = b->vel[1] + (b->omega[2] * r[0] - b->omega[0] * r[2]);
  us[2] = b->vel[2] + (b->omega[0] * r[1] - b->omega[1] * r[0]);
}

/* ---------------------------------------------------------------- O1 geometry
 * Rotor signed distance at a lattice point: rotate (x - x_c) by -theta about the
 * axis (Rodrigues), trilinear-sample the rotor-frame reference grid
 * (PAPER.md:219, :265).  Operation order is part of the definition (bit-exact
 * cell types on the GPU side): compiled with -ffp-contract=off.                   */
static double rotor_phi(const ohrr_lattice *L, double cth, double sth, double px, double py,
                        double pz, int *tag_out) {
  const ohrr_rotor_desc *R = &L->rot;
  double rx = px - R->centre[0], ry = py - R->centre[1], rz = pz - R->centre[2];
  double ax = R->axis[0], ay = R->axis[1], az = R->axis[2];
  double kx = ay * rz - az * ry, ky = az * rx - ax * rz, kz = ax * ry - ay * rx;
  double ad = ax * rx + ay * ry + az * rz;
  double omc = 1.0 - cth;
  /* rotation by -theta: r c - (a x r) s + a (a.r)(1-c) */
  double qx = rx * cth - kx * sth + ax * ad * omc;
  double qy = ry * cth - ky * sth + ay * ad * omc;
  double qz = rz * cth - kz * sth + az * ad * omc;
  double gx = (qx - R->origin[0]) / R->spacing;
  double gy = (qy - R->origin[1]) / R->spacing;
  double gz = (qz - R->origin[2]) / R->spacing;
  double fx = floor(gx), fy = floor(gy), fz = floor(gz);
  *tag_out = 0;
  if (!(fx >= 0.0 && fy >= 0.0 && fz >= 0.0 && fx < (double)(R->gx - 1) &&
        fy < (double)(R->gy - 1) && fz < (double)(R->gz - 1)))
    return BIG_PHI;
  int ix = (int)fx, iy = (int)fy, iz = (int)fz;
  double tx = gx - fx, ty = gy - fy, tz = gz - fz;
  const float *s = L->rot_sdf;
  int64_t sx = 1, sy = R->gx, sz = (int64_t)R->gx * R->gy;
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
  if (nx_ > R->gx - 1) nx_ = R->gx - 1;
  if (ny_ > R->gy - 1) ny_ = R->gy - 1;
  if (nz_ > R->gz - 1) nz_ = R->gz - 1;
  *tag_out = L->rot_tag[nx_ * sx + ny_ * sy + nz_ * sz];
  return phi;
}

static double rotor_angle(const ohrr_lattice *L, int64_t step) {
  return L->rot.theta0 + (double)step * L->rot.omega; /* O6: rigid rotation only */
}

/* Def. 1 (Eq. 21) with the linear transition Eq. 22 (:203), the
 * cell types of Fig. 4 (:254-263), the integer tag (:267) and the y1 vector (:324).
 * Brute force over all cells.                                                       */
static void geometry(ohrr_lattice *L) {
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
  const double h = 0.5 * L->p.eps_cells;
  double cth = 1.0, sth = 0.0;
  if (L->has_rotor) {
    double th = rotor_angle(L, L->step);
    cth = cos(th);
    sth = sin(th);
  }
  /* pass 1: phi and provisional tag */
#pragma omp parallel for schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        double phi = BIG_PHI;
        int tg = 0;
        if (L->phi_static) {
          phi = L->phi_static[c];
          tg = L->tag_static ? L->tag_static[c] : 1;
        }
        if (L->has_rotor) {
          int rt;
          double pr = rotor_phi(L, cth, sth, (double)x, (double)y, (double)z, &rt);
          if (pr < phi) {
            phi = pr;
            tg = rt;
          }
        }
        L->phi[c] = phi;
        L->tag[c] = (uint8_t)tg;
      }
  /* pass 2: type, porosity, wall-model set */
#pragma omp parallel for schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        double phi = L->phi[c];
        int type;
        double d;
        if (L->has_fringe && x >= L->fr_x0 && x < L->fr_x1) {
          type = T_FRINGE;
          d = 0.0;
        } else if (phi <= -h) {
          type = T_SOLID;
          d = 0.0;
        } else if (phi < h) {
          type = T_FRONTIER;
          d = phi / L->p.eps_cells + 0.5; /* Eq. 22 */
          if (L->d_override && L->phi_static && L->phi_static[c] == phi) d = L->d_override[c];
        } else {
          type = T_FLUID;
          d = 1.0;
          for (int dz = -1; dz <= 1 && type == T_FLUID; ++dz)
            for (int dy = -1; dy <= 1 && type == T_FLUID; ++dy)
              for (int dx = -1; dx <= 1; ++dx) {
                if (!dx && !dy && !dz) continue;
                int fl;
                int xx = wrap1(x + dx, nx, L->p.mode[0], &fl);
                int yy = wrap1(y + dy, ny, L->p.mode[1], &fl);
                int zz = wrap1(z + dz, nz, L->p.mode[2], &fl);
                if (L->phi[lidx(L, xx, yy, zz)] < h) {
                  type = T_GROWTH;
                  break;
                }
              }
        }
        if (L->n_fsi > 0) { /* bulk model where no moving wall-modelled structure can be */
          int inside = 0;
          for (int b = 0; b < L->n_fsi; ++b)
            inside |= x >= L->fsi[b][0] && x < L->fsi[b][1] && y >= L->fsi[b][2] && y < L->fsi[b][3] &&
                      z >= L->fsi[b][4] && z < L->fsi[b][5];
          if (!inside) {
            if (type == T_FLUID) type = T_BULK;
            else L->region_violation = 1; /* the caller's boxes do not cover the structure: reported */
          }
        }
        L->type[c] = (uint8_t)type;
        L->d[c] = d;
        if (type == T_FLUID || type == T_FRINGE || type == T_BULK) L->tag[c] = 0;
        /* wall-model set W = {FRONTIER, phi > 0} (reading R13), y1 = phi, n = grad phi/|grad phi| */
        int inw = 0;
        if (L->wm_enabled && type == T_FRONTIER && phi > 0.0) {
          double gr[3];
          int fl;
          int xm = wrap1(x - 1, nx, L->p.mode[0], &fl), xp = wrap1(x + 1, nx, L->p.mode[0], &fl);
          int ym = wrap1(y - 1, ny, L->p.mode[1], &fl), yp = wrap1(y + 1, ny, L->p.mode[1], &fl);
          int zm = wrap1(z - 1, nz, L->p.mode[2], &fl), zp = wrap1(z + 1, nz, L->p.mode[2], &fl);
          gr[0] = 0.5 * (L->phi[lidx(L, xp, y, z)] - L->phi[lidx(L, xm, y, z)]);
          gr[1] = 0.5 * (L->phi[lidx(L, x, yp, z)] - L->phi[lidx(L, x, ym, z)]);
          gr[2] = 0.5 * (L->phi[lidx(L, x, y, zp)] - L->phi[lidx(L, x, y, zm)]);
          double nn = sqrt(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2]);
          if (nn > 1e-12 && nn < 1e20) {
            inw = 1;
            for (int a = 0; a < 3; ++a) L->y1n[3 * c + a] = phi * (gr[a] / nn);
          }
        }
        L->in_w[c] = (uint8_t)inw;
        if (!inw) L->wm_valid[c] = 0; /* arrays of cells not in W_n are invalidated */
      }
  L->geometry_current = 1;
}

/* ---------------------------------------------------------------- O2 + O3 */
static void homogenised_velocity_field(ohrr_lattice *L) {
  const int64_t n = L->n;
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
#pragma omp parallel for schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        double rho = 0.0, j[3] = {0, 0, 0};
        for (int i = 0; i < Q; ++i) {
          double fi = L->f[(int64_t)i * n + c];
          rho += fi;
          j[0] += CX[i] * fi;
          j[1] += CY[i] * fi;
          j[2] += CZ[i] * fi;
        }
        double uB[3] = {0, 0, 0};
        int t = L->type[c];
        if (t == T_FRINGE) {
          for (int a = 0; a < 3; ++a) uB[a] = L->fr_u[a];
        } else if (t == T_SOLID || t == T_FRONTIER) {
          body_velocity(L, L->tag[c], x, y, z, uB);
          if (L->wm_valid[c])
            for (int a = 0; a < 3; ++a) uB[a] += L->wm_u[3 * c + a];
        }
        double d = L->d[c];
        L->rho[c] = rho;
        for (int a = 0; a < 3; ++a) {
          double u = (j[a] + L->p.body_force[a]) / rho;
          L->uhat[(int64_t)a * n + c] = d * u + (1.0 - d) * uB[a];
        }
      }
}

/* uhat of a face neighbour with the boundary rule R12 (mirror flips the normal component) */
static inline void uhat_at(const ohrr_lattice *L, int x, int y, int z, double u[3]) {
  int fx, fy, fz;
  int xx = wrap1(x, L->p.nx, L->p.mode[0], &fx);
  int yy = wrap1(y, L->p.ny, L->p.mode[1], &fy);
  int zz = wrap1(z, L->p.nz, L->p.mode[2], &fz);
  int64_t c = lidx(L, xx, yy, zz);
  u[0] = L->uhat[c] * (fx ? -1.0 : 1.0);
  u[1] = L->uhat[L->n + c] * (fy ? -1.0 : 1.0);
  u[2] = L->uhat[2 * L->n + c] * (fz ? -1.0 : 1.0);
}

/* S^FD: second-order central differences of the time-n uhat field over the six
 * face neighbours ("non-local finite difference", Eq. 5 :90; R5).    */
static void fd_strain(const ohrr_lattice *L, int x, int y, int z, double S[3][3]) {
  double up[3][3], um[3][3]; /* [direction b][component a] */
  uhat_at(L, x + 1, y, z, up[0]);
  uhat_at(L, x - 1, y, z, um[0]);
  uhat_at(L, x, y + 1, z, up[1]);
  uhat_at(L, x, y - 1, z, um[1]);
  uhat_at(L, x, y, z + 1, up[2]);
  uhat_at(L, x, y, z - 1, um[2]);
  double G[3][3]; /* G[a][b] = d_b u_a */
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) G[a][b] = 0.5 * (up[b][a] - um[b][a]);
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) S[a][b] = 0.5 * (G[a][b] + G[b][a]);
}

static void collide_and_stream(ohrr_lattice *L) {
  const int64_t n = L->n;
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
  homogenised_velocity_field(L); /* the time-n field the FD strain differentiates */
#pragma omp parallel for schedule(static)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        double fin[Q], fout[Q];
        for (int i = 0; i < Q; ++i) fin[i] = L->f[(int64_t)i * n + c];
        double uB[3] = {0, 0, 0};
        int t = L->type[c];
        double S[3][3];
        double sigma = L->p.sigma;
        if (t == T_FRINGE) {
          for (int a = 0; a < 3; ++a) uB[a] = L->fr_u[a];
        } else if (t == T_SOLID || t == T_FRONTIER) {
          body_velocity(L, L->tag[c], x, y, z, uB);
          if (L->wm_valid[c])
            for (int a = 0; a < 3; ++a) uB[a] += L->wm_u[3 * c + a];
        }
        if (L->wm_valid[c]) { /* sigma = 0 on wall-modelled cells, strain from the wall model (:314) */
          const double *s = &L->wm_s[6 * c];
          S[0][0] = s[0]; S[1][1] = s[1]; S[2][2] = s[2];
          S[0][1] = S[1][0] = s[3];
          S[0][2] = S[2][0] = s[4];
          S[1][2] = S[2][1] = s[5];
          sigma = 0.0;
        } else if (t == T_BULK) {
          /* Listing 2: bulk cells run RRLBM-LES -- plain momentum (d = 1 here),
           * third-order recursive-regularised collision with the Smagorinsky effective relaxation and NO
           * hybrid finite-difference part, i.e. Eq. 7 at sigma = 1 */
          memset(S, 0, sizeof(S));
          sigma = 1.0;
        } else {
          fd_strain(L, x, y, z, S);
        }
        ohrr_collide_cell(fin, L->p.body_force, L->d[c], uB, S, sigma, L->p.tau0,
                          L->p.smagorinsky_cs, fout, NULL);
        /* O3 stream (Eq. 6 lhs): f_i(x + c_i, n+1) = f*_i(x, n); R12 at the outer faces */
        for (int i = 0; i < Q; ++i) {
          int tx = x + CX[i], ty = y + CY[i], tz = z + CZ[i];
          int ci[3] = {CX[i], CY[i], CZ[i]};
          if (tx < 0 || tx >= nx) {
            if (L->p.mode[0] == AX_PERIODIC) tx = (tx + nx) % nx;
            else { tx = x; ci[0] = -ci[0]; }
          }
          if (ty < 0 || ty >= ny) {
            if (L->p.mode[1] == AX_PERIODIC) ty = (ty + ny) % ny;
            else { ty = y; ci[1] = -ci[1]; }
          }
          if (tz < 0 || tz >= nz) {
            if (L->p.mode[2] == AX_PERIODIC) tz = (tz + nz) % nz;
            else { tz = z; ci[2] = -ci[2]; }
          }
          int io = dir_of(ci[0], ci[1], ci[2]);
          L->f2[(int64_t)io * n + lidx(L, tx, ty, tz)] = fout[i];
        }
      }
  double *t = L->f;
  L->f = L->f2;
  L->f2 = t;
}

/* reported velocity moment v = (j + g/2)/rho (reading R11) of the current populations */
static void cell_velocity(const ohrr_lattice *L, int64_t c, double *rho_out, double v[3]) {
  double rho = 0.0, j[3] = {0, 0, 0};
  for (int i = 0; i < Q; ++i) {
    double fi = L->f[(int64_t)i * L->n + c];
    rho += fi;
    j[0] += CX[i] * fi;
    j[1] += CY[i] * fi;
    j[2] += CZ[i] * fi;
  }
  for (int a = 0; a < 3; ++a) v[a] = (j[a] + 0.5 * L->p.body_force[a]) / rho;
  if (rho_out) *rho_out = rho;
}
static void velocity_at(const ohrr_lattice *L, int x, int y, int z, double v[3]) {
  int fx, fy, fz;
  int xx = wrap1(x, L->p.nx, L->p.mode[0], &fx);
  int yy = wrap1(y, L->p.ny, L->p.mode[1], &fy);
  int zz = wrap1(z, L->p.nz, L->p.mode[2], &fz);
  cell_velocity(L, lidx(L, xx, yy, zz), NULL, v);
  if (fx) v[0] = -v[0];
  if (fy) v[1] = -v[1];
  if (fz) v[2] = -v[2];
}

/* ---------------------------------------------------------------- O4 wall model
 * PAPER.md:157-188 (Eq. 15-20), :314, :324; readings R8, R9, R10, R13, R15.       */
static void wall_model(ohrr_lattice *L) {
  if (!L->wm_enabled) return;
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
  const double hs = L->p.sampling_distance;
  const double nu = CS2 * (L->p.tau0 - 0.5);
#pragma omp parallel for schedule(dynamic, 4)
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        if (!L->in_w[c]) continue;
        double y1v[3] = {L->y1n[3 * c], L->y1n[3 * c + 1], L->y1n[3 * c + 2]};
        double y1 = sqrt(y1v[0] * y1v[0] + y1v[1] * y1v[1] + y1v[2] * y1v[2]);
        double nrm[3] = {y1v[0] / y1, y1v[1] / y1, y1v[2] / y1};
        /* interpolated velocity at x_w + h_s n  (R15: trilinear) */
        double px = x + hs * nrm[0], py = y + hs * nrm[1], pz = z + hs * nrm[2];
        double fx = floor(px), fy = floor(py), fz = floor(pz);
        double tx = px - fx, ty = py - fy, tz = pz - fz;
        int ix = (int)fx, iy = (int)fy, iz = (int)fz;
        double vs[3] = {0, 0, 0};
        for (int k = 0; k < 8; ++k) {
          int ox = k & 1, oy = (k >> 1) & 1, oz = (k >> 2) & 1;
          double w = (ox ? tx : 1.0 - tx) * (oy ? ty : 1.0 - ty) * (oz ? tz : 1.0 - tz);
          double v[3];
          velocity_at(L, ix + ox, iy + oy, iz + oz, v);
          for (int a = 0; a < 3; ++a) vs[a] += w * v[a];
        }
        double vw[3], us[3];
        cell_velocity(L, c, NULL, vw);
        body_velocity(L, L->tag[c], x, y, z, us);
        double r[3], rn = 0.0;
        for (int a = 0; a < 3; ++a) {
          r[a] = vs[a] - us[a];
          rn += r[a] * nrm[a];
        }
        double ut[3], U = 0.0;
        for (int a = 0; a < 3; ++a) {
          ut[a] = r[a] - rn * nrm[a];
          U += ut[a] * ut[a];
        }
        U = sqrt(U);
        double utau = 0.0;
        if (U < 1e-14) {
          for (int a = 0; a < 3; ++a) L->wm_u[3 * c + a] = 0.0;
          for (int a = 0; a < 6; ++a) L->wm_s[6 * c + a] = 0.0;
        } else {
          double yy = y1 + hs;
          double u0 = (L->wm_valid[c] && L->wm_utau[c] > 0.0) ? L->wm_utau[c] : sqrt(nu * U / yy); /* Eq. 20 */
          utau = L->wall_function == 1
                     ? ohrr_newton_utau_musker(u0, U, yy, nu, L->p.newton_max_iter, L->p.newton_tol, NULL)
                     : ohrr_newton_utau(u0, U, yy, nu, L->p.kappa, L->p.E, L->p.newton_max_iter,
                                        L->p.newton_tol, NULL);
          double upl = 1.0; /* R8: the friction velocity itself; R22: the wall-function velocity at y1 */
          if (L->wm_slip == 1) upl = ohrr_wall_uplus(L->wall_function, y1 * utau / nu, L->p.kappa, L->p.E);
          for (int a = 0; a < 3; ++a) L->wm_u[3 * c + a] = utau * upl * ut[a] / U;
          double G[3][3];
          if (L->wm_shear == 1) { /* R22: analytic slope of the wall function, tangential velocity along n */
            double dudy = ohrr_wall_shear(L->wall_function, utau, U, yy, nu, L->p.kappa, L->p.E);
            for (int a = 0; a < 3; ++a)
              for (int b = 0; b < 3; ++b) G[a][b] = dudy * (ut[a] / U) * nrm[b];
          } else {
            for (int a = 0; a < 3; ++a)
              for (int b = 0; b < 3; ++b) G[a][b] = (vs[a] - vw[a]) * nrm[b] / hs; /* R10 */
          }
          double *s = &L->wm_s[6 * c];
          s[0] = G[0][0]; s[1] = G[1][1]; s[2] = G[2][2];
          s[3] = 0.5 * (G[0][1] + G[1][0]);
          s[4] = 0.5 * (G[0][2] + G[2][0]);
          s[5] = 0.5 * (G[1][2] + G[2][1]);
        }
        L->wm_utau[c] = utau;
        L->wm_valid[c] = 1;
      }
}

/* ---------------------------------------------------------------- O5 force
 * Momentum exchange, PAPER.md:211 (Eq. 23) with reading R7 (second population is
 * the opposite one; reported with a leading minus = force ON the solid), summed
 * literally over all cells with d < 1 and all 26 links, per tag (:267, :315-317).
 * Kahan summation in cell order.
 * Torque (SURVEY 8(f)-4; the paper integrates forces only, :209-211, so this is the
 * textbook moment of the SAME per-cell momentum-exchange forces F(x) of Eq. 23 about the
 * centre x_c of the element's rigid body (:140): M_k = sum_x (x - x_c) x F(x).      */
static void forces(ohrr_lattice *L) {
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
  const int64_t n = L->n;
  if (L->step >= L->force_cap) {
    int64_t ncap = L->force_cap * 2;
    L->force = (double *)realloc(L->force, sizeof(double) * ncap * MAX_TAGS * 3);
    memset(L->force + L->force_cap * MAX_TAGS * 3, 0, sizeof(double) * (ncap - L->force_cap) * MAX_TAGS * 3);
    L->torque = (double *)realloc(L->torque, sizeof(double) * ncap * MAX_TAGS * 3);
    memset(L->torque + L->force_cap * MAX_TAGS * 3, 0, sizeof(double) * (ncap - L->force_cap) * MAX_TAGS * 3);
    L->force_cap = ncap;
  }
  double sum[MAX_TAGS][3], comp[MAX_TAGS][3];
  double tsum[MAX_TAGS][3], tcomp[MAX_TAGS][3];
  memset(sum, 0, sizeof(sum));
  memset(comp, 0, sizeof(comp));
  memset(tsum, 0, sizeof(tsum));
  memset(tcomp, 0, sizeof(tcomp));
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        int t = L->type[c];
        if (!(t == T_SOLID || t == T_FRONTIER)) continue; /* d < 1; fringe excluded (R12) */
        int k = L->tag[c];
        if (k <= 0 || k >= MAX_TAGS) continue;
        double us[3];
        body_velocity(L, k, x, y, z, us);
        double acc[3] = {0, 0, 0};
        for (int i = 0; i < Q; ++i) {
          if (i == REST) continue;
          /* R12: the cell behind a MIRROR plane is the reflected image of the lattice, so f_i there is the
           * population of the reflected cell whose normal velocity component is reversed (the same rule the
           * streaming step O3 applies to a population leaving through the plane)                          */
          int flx, fly, flz;
          int xx = wrap1(x + CX[i], nx, L->p.mode[0], &flx);
          int yy = wrap1(y + CY[i], ny, L->p.mode[1], &fly);
          int zz = wrap1(z + CZ[i], nz, L->p.mode[2], &flz);
          int ir = dir_of(flx ? -CX[i] : CX[i], fly ? -CY[i] : CY[i], flz ? -CZ[i] : CZ[i]);
          double fa = L->f[(int64_t)ir * n + lidx(L, xx, yy, zz)];
          double fb = L->f[(int64_t)opposite(i) * n + c];
          double ci[3] = {CX[i], CY[i], CZ[i]};
          for (int a = 0; a < 3; ++a) acc[a] += (ci[a] - us[a]) * fa + (ci[a] + us[a]) * fb;
        }
        for (int a = 0; a < 3; ++a) {
          double v = -acc[a] - comp[k][a];
          double tt = sum[k][a] + v;
          comp[k][a] = (tt - sum[k][a]) - v;
          sum[k][a] = tt;
        }
        const body_t *b = &L->body[k];
        double r[3] = {x - b->centre[0], y - b->centre[1], z - b->centre[2]};
        double F[3] = {-acc[0], -acc[1], -acc[2]};
        double m[3] = {r[1] * F[2] - r[2] * F[1], r[2] * F[0] - r[0] * F[2], r[0] * F[1] - r[1] * F[0]};
        for (int a = 0; a < 3; ++a) {
          double v = m[a] - tcomp[k][a];
          double tt = tsum[k][a] + v;
          tcomp[k][a] = (tt - tsum[k][a]) - v;
          tsum[k][a] = tt;
        }
      }
  memcpy(L->force + L->step * MAX_TAGS * 3, sum, sizeof(sum));
  memcpy(L->torque + L->step * MAX_TAGS * 3, tsum, sizeof(tsum));
}

/* ---------------------------------------------------------------- public API */
ohrr_lattice *ohrr_create(const ohrr_params *p) {
  init_tables();
  if (!p || p->nx < 1 || p->ny < 1 || p->nz < 1) return NULL;
  ohrr_lattice *L = (ohrr_lattice *)calloc(1, sizeof(*L));
  L->p = *p;
  L->n = (int64_t)p->nx * p->ny * p->nz;
  int64_t n = L->n;
  L->f = (double *)calloc(Q * n, sizeof(double));
  L->f2 = (double *)calloc(Q * n, sizeof(double));
  L->uhat = (double *)calloc(3 * n, sizeof(double));
  L->rho = (double *)calloc(n, sizeof(double));
  L->phi = (double *)calloc(n, sizeof(double));
  L->d = (double *)calloc(n, sizeof(double));
  L->type = (uint8_t *)calloc(n, 1);
  L->tag = (uint8_t *)calloc(n, 1);
  L->in_w = (uint8_t *)calloc(n, 1);
  L->y1n = (double *)calloc(3 * n, sizeof(double));
  L->wm_valid = (uint8_t *)calloc(n, 1);
  L->wm_utau = (double *)calloc(n, sizeof(double));
  L->wm_u = (double *)calloc(3 * n, sizeof(double));
  L->wm_s = (double *)calloc(6 * n, sizeof(double));
  L->force_cap = 1024;
  L->force = (double *)calloc(L->force_cap * MAX_TAGS * 3, sizeof(double));
  L->torque = (double *)calloc(L->force_cap * MAX_TAGS * 3, sizeof(double));
  for (int64_t c = 0; c < n; ++c) L->d[c] = 1.0;
  for (int i = 0; i < Q; ++i)
    for (int64_t c = 0; c < n; ++c) L->f[(int64_t)i * n + c] = W[i];
  return L;
}

void ohrr_destroy(ohrr_lattice *L) {
  if (!L) return;
  free(L->f); free(L->f2); free(L->uhat); free(L->rho); free(L->phi_static); free(L->tag_static);
  free(L->d_override); free(L->rot_sdf); free(L->rot_tag); free(L->phi); free(L->d); free(L->type);
  free(L->tag); free(L->in_w); free(L->y1n); free(L->wm_valid); free(L->wm_utau); free(L->wm_u);
  free(L->wm_s); free(L->force); free(L->torque);
  free(L);
}

/* f = f_eq(rho,u) [+ f^(1) with a1^(2) = -2 rho cs^2 tau0 S^FD(u) if with_neq]; u: 3 SoA planes */
int ohrr_init_equilibrium(ohrr_lattice *L, const double *rho, const double *u, int with_neq) {
  const int64_t n = L->n;
  const int nx = L->p.nx, ny = L->p.ny, nz = L->p.nz;
  for (int64_t c = 0; c < n; ++c) {
    L->rho[c] = rho[c];
    for (int a = 0; a < 3; ++a) L->uhat[(int64_t)a * n + c] = u[(int64_t)a * n + c];
  }
  for (int z = 0; z < nz; ++z)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        int64_t c = lidx(L, x, y, z);
        double uu[3] = {u[c], u[n + c], u[2 * n + c]};
        double feq[Q], f1[Q];
        ohrr_equilibrium(rho[c], uu, feq);
        for (int i = 0; i < Q; ++i) f1[i] = 0.0;
        if (with_neq) {
          double S[3][3], a2[3][3];
          fd_strain(L, x, y, z, S);
          for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) a2[a][b] = -2.0 * rho[c] * CS2 * L->p.tau0 * S[a][b];
          regularised_f1(a2, uu, f1);
        }
        for (int i = 0; i < Q; ++i) L->f[(int64_t)i * n + c] = feq[i] + f1[i];
      }
  L->geometry_current = 0;
  return 0;
}

int ohrr_set_static_geometry(ohrr_lattice *L, const double *phi, const uint8_t *tag,
                             const double *d_override) {
  const int64_t n = L->n;
  free(L->phi_static); free(L->tag_static); free(L->d_override);
  L->phi_static = NULL; L->tag_static = NULL; L->d_override = NULL;
  if (phi) {
    L->phi_static = (double *)malloc(sizeof(double) * n);
    memcpy(L->phi_static, phi, sizeof(double) * n);
  }
  if (tag) {
    L->tag_static = (uint8_t *)malloc(n);
    memcpy(L->tag_static, tag, n);
  }
  if (d_override) {
    L->d_override = (double *)malloc(sizeof(double) * n);
    memcpy(L->d_override, d_override, sizeof(double) * n);
  }
  L->geometry_current = 0;
  return 0;
}

int ohrr_set_body(ohrr_lattice *L, int tag, const double centre[3], const double omega[3],
                  const double vel[3]) {
  if (tag < 0 || tag >= MAX_TAGS) return -1;
  for (int a = 0; a < 3; ++a) {
    L->body[tag].centre[a] = centre[a];
    L->body[tag].omega[a] = omega[a];
    L->body[tag].vel[a] = vel[a];
  }
  return 0;
}

int ohrr_set_fringe(ohrr_lattice *L, int x0, int x1, const double u_in[3]) {
  L->has_fringe = x1 > x0;
  L->fr_x0 = x0;
  L->fr_x1 = x1;
  for (int a = 0; a < 3; ++a) L->fr_u[a] = u_in[a];
  L->geometry_current = 0;
  return 0;
}

/* Region split of PAPER.md:215: boxes = n_boxes x {x0,x1,y0,y1,z0,z1}, half-open; n_boxes = 0: HHRRLBM everywhere */
int ohrr_set_fsi_region(ohrr_lattice *L, int32_t n_boxes, const int32_t *boxes) {
  if (n_boxes < 0 || n_boxes > MAX_FSI_BOXES || (n_boxes > 0 && !boxes)) return -1;
  L->n_fsi = n_boxes;
  for (int b = 0; b < n_boxes; ++b)
    for (int k = 0; k < 6; ++k) L->fsi[b][k] = boxes[6 * b + k];
  L->region_violation = 0;
  L->geometry_current = 0;
  return 0;
}
int ohrr_region_violation(const ohrr_lattice *L) { return L->region_violation; }
/* 0: truncated Spalding (Eq. 18, the paper's); 1: Musker's profile */
int ohrr_set_wall_function(ohrr_lattice *L, int kind) {
  if (kind != 0 && kind != 1) return -1;
  L->wall_function = kind;
  return 0;
}

/* slip: 0 = R8, 1 = wall-function velocity at y1; shear: 0 = R10, 1 = analytic slope (R22) */
int ohrr_set_wall_model_variant(ohrr_lattice *L, int slip, int shear) {
  if ((slip != 0 && slip != 1) || (shear != 0 && shear != 1)) return -1;
  L->wm_slip = slip;
  L->wm_shear = shear;
  return 0;
}

int ohrr_set_rotor(ohrr_lattice *L, const ohrr_rotor_desc *r) {
  if (!r || r->n_tags < 1 || r->n_tags >= MAX_TAGS) return -1;
  L->rot = *r;
  int64_t g = (int64_t)r->gx * r->gy * r->gz;
  free(L->rot_sdf); free(L->rot_tag);
  L->rot_sdf = (float *)malloc(sizeof(float) * g);
  L->rot_tag = (uint8_t *)malloc(g);
  memcpy(L->rot_sdf, r->sdf, sizeof(float) * g);
  memcpy(L->rot_tag, r->tag, g);
  L->rot.sdf = NULL;
  L->rot.tag = NULL;
  L->has_rotor = 1;
  /* solid velocity u^B = Omega x (x - x_c) for every rotor tag */
  for (int k = 1; k <= r->n_tags; ++k) {
    double om[3] = {r->axis[0] * r->omega, r->axis[1] * r->omega, r->axis[2] * r->omega};
    double zero[3] = {0, 0, 0};
    ohrr_set_body(L, k, r->centre, om, zero);
  }
  L->geometry_current = 0;
  return 0;
}

int ohrr_enable_wall_model(ohrr_lattice *L, int enable) {
  L->wm_enabled = enable != 0;
  L->geometry_current = 0;
  return 0;
}

/* evaluates geometry(step) without stepping (InitializePorosityO) */
int ohrr_update_geometry(ohrr_lattice *L) {
  geometry(L);
  return 0;
}

/* pins only: geometry + WallModelO on the current populations, nothing else */
int ohrr_wall_model_only(ohrr_lattice *L) {
  geometry(L);
  wall_model(L);
  return 0;
}
/* pins only: geometry + force sum on the current populations -> F[MAX_TAGS][3] */
int ohrr_force_only(ohrr_lattice *L, double *F) {
  geometry(L);
  forces(L);
  memcpy(F, L->force + L->step * MAX_TAGS * 3, sizeof(double) * MAX_TAGS * 3);
  return 0;
}

/* pins only: same, the torque sums M[MAX_TAGS][3] */
int ohrr_torque_only(ohrr_lattice *L, double *M) {
  geometry(L);
  forces(L);
  memcpy(M, L->torque + L->step * MAX_TAGS * 3, sizeof(double) * MAX_TAGS * 3);
  return 0;
}

/* Listing 3 */
int ohrr_step(ohrr_lattice *L, int32_t n_steps) {
  for (int s = 0; s < n_steps; ++s) {
    geometry(L);            /* line 2  UpdatePorosityO   */
    collide_and_stream(L);  /* line 3                    */
    wall_model(L);          /* line 4  WallModelO        */
    forces(L);              /* lines 5-6                 */
    L->step += 1;           /* line 7: theta_{n+1} = theta_n + Omega */
    L->geometry_current = 0;
  }
  return 0;
}

int ohrr_get_moments(const ohrr_lattice *L, double *rho, double *v) {
  for (int64_t c = 0; c < L->n; ++c) {
    double vv[3];
    cell_velocity(L, c, &rho[c], vv);
    for (int a = 0; a < 3; ++a) v[(int64_t)a * L->n + c] = vv[a];
  }
  return 0;
}
int ohrr_get_forces(const ohrr_lattice *L, int64_t first, int64_t count, double *F) {
  if (first < 0 || first + count > L->step) return -1;
  memcpy(F, L->force + first * MAX_TAGS * 3, sizeof(double) * count * MAX_TAGS * 3);
  return 0;
}
int ohrr_get_torques(const ohrr_lattice *L, int64_t first, int64_t count, double *M) {
  if (first < 0 || first + count > L->step) return -1;
  memcpy(M, L->torque + first * MAX_TAGS * 3, sizeof(double) * count * MAX_TAGS * 3);
  return 0;
}
/* Definition 3 / Eq. 26: C_T = T / (0.5 rho pi r^2 U^2), T = "the integral of all axial forces
 * acting on the rotor" = sum over the rotor's elements (tags 1..n_tags) of F_k . a, a = the (unit) rotor axis.  With the
 * torques of the same elements, the power coefficient C_P = (sum_k M_k . a) Omega / (0.5 rho pi r^2 U^3) (torque /
 * power output of SURVEY 8(f)-4; the paper reports C_T only).  One value per step. */
int ohrr_rotor_coefficients(const ohrr_lattice *L, int64_t first, int64_t count, double rho, double u_inf,
                            double radius, double *c_t, double *c_p) {
  if (!L->has_rotor || first < 0 || first + count > L->step || !(rho > 0) || !(u_inf > 0) || !(radius > 0)) return -1;
  const double *ax = L->rot.axis; /* a unit vector by the rotor description's contract */
  const double area = 3.14159265358979323846 * radius * radius;
  for (int64_t s = 0; s < count; ++s) {
    double T = 0, Mz = 0;
    for (int k = 1; k <= L->rot.n_tags; ++k)
      for (int a = 0; a < 3; ++a) {
        T += L->force[((first + s) * MAX_TAGS + k) * 3 + a] * ax[a];
        Mz += L->torque[((first + s) * MAX_TAGS + k) * 3 + a] * ax[a];
      }
    if (c_t) c_t[s] = T / (0.5 * rho * area * u_inf * u_inf);
    if (c_p) c_p[s] = Mz * L->rot.omega / (0.5 * rho * area * u_inf * u_inf * u_inf);
  }
  return 0;
}
/* geometry of the LAST evaluated step (call ohrr_update_geometry first for the current one) */
int ohrr_get_cell_types(const ohrr_lattice *L, uint8_t *type, uint8_t *tag, double *d) {
  memcpy(type, L->type, L->n);
  memcpy(tag, L->tag, L->n);
  if (d) memcpy(d, L->d, sizeof(double) * L->n);
  return 0;
}
/* wall list in ascending cell index */
int64_t ohrr_get_wall_list(const ohrr_lattice *L, int32_t *idx, double *y1n, double *utau,
                           uint8_t *valid, int64_t cap) {
  int64_t k = 0;
  for (int64_t c = 0; c < L->n; ++c) {
    if (!L->in_w[c]) continue;
    if (k < cap && idx) {
      idx[k] = (int32_t)c;
      if (y1n) for (int a = 0; a < 3; ++a) y1n[3 * k + a] = L->y1n[3 * c + a];
      if (utau) utau[k] = L->wm_utau[c];
      if (valid) valid[k] = L->wm_valid[c];
    }
    ++k;
  }
  return k;
}
int ohrr_get_wall_state(const ohrr_lattice *L, int64_t cell, double *utau, double uwm[3], double swm[6]) {
  *utau = L->wm_utau[cell];
  for (int a = 0; a < 3; ++a) uwm[a] = L->wm_u[3 * cell + a];
  for (int a = 0; a < 6; ++a) swm[a] = L->wm_s[6 * cell + a];
  return L->wm_valid[cell];
}
int ohrr_get_populations(const ohrr_lattice *L, double *f) {
  memcpy(f, L->f, sizeof(double) * Q * L->n);
  return 0;
}
int ohrr_set_populations(ohrr_lattice *L, const double *f) {
  memcpy(L->f, f, sizeof(double) * Q * L->n);
  return 0;
}
int ohrr_get_uhat(const ohrr_lattice *L, double *uhat) { /* time-n field of the last collide */
  memcpy(uhat, L->uhat, sizeof(double) * 3 * L->n);
  return 0;
}
int64_t ohrr_step_count(const ohrr_lattice *L) { return L->step; }
