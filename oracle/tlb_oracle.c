/*
 * tlb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU statement of one time step of the 2D thermal
 * two-component D2Q9 lattice-Boltzmann model of the TLBfind paper (arXiv 2109.12565,
 * /root/reference/PAPER.md, cited below as "PAPER L<line>").  It exists only so that
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs can
 * check and time against it.  It shares no code, header, table or helper with the CUDA
 * path under paper_2109_12565_b200/ and neither side includes the other.
 *
 * The method is an explicit iteration, so the oracle follows it step by step in the
 * paper's order and notation (PAPER Eqs. (1)-(22)); readings of silent / garbled passages
 * are the ones listed in DESIGN.md ("Readings R1..R32").  No blocking, fusion or reordering:
 * every sub-step is a full sweep over the lattice writing a full array.
 *
 * Parity pins (tests/test_oracle_pins.py, all run with -m "not gpu"):
 *   weights            rational invariants of Fig. 1(b)
 *   bulk update        the paper's printed Table B.8(b) (tests/golden/)
 *   bounce-back        exact mass conservation, Poiseuille profile            PAPER L151, Eq. (14)
 *   thermal wall rule  exact linear conduction profile, Nu = 1                PAPER L314, Eq. (24)
 *   transport coeffs   decay of a shear wave (nu) and of a T mode (kappa)     Eqs. (14), (20)
 *   forces + pressure  Laplace law on one droplet, flat-interface coexistence Eq. (9)
 *   buoyancy           barometric density gradient at rest                    Eq. (22)
 *   moving flat walls  exact linear Couette profile between the wall velocities, exact mass
 *                      conservation (reading R20 of L147-151, Eq. (15))
 *   observables        mass, E and the convective term of Nu against closed forms on states with
 *                      known moments (random masks, posts, buoyancy so that u^(H) != u);
 *                      u_av on rows through posts                            L248, Eq. (24)
 *   stress P_xy        exact -rho nu (U_t - U_b)/ny in single-phase Couette for three tau; Pxy_av constant across
 *                      the interface of a sheared two-layer state; exact row-by-row momentum balance of one step
 *                      on a random two-component state (interaction part, NN couplings) and its first moment
 *                      (all couplings)                                       L248-250, L294-296, Eq. (14) (R21)
 *   droplets           hand-made masks with known clusters, a droplet across the x seam, exact centroids of
 *                      discs, invariance under x shifts                      section 2.4 L198 (R22)
 *   Voronoi / Delaunay half planes, rectangular cells and ties by hand; the defining minimum property checked in numpy;
 *   / T1 / Nu_drop     links equal to the continuum Delaunay triangulation (scipy.spatial, periodic images and
 *                      wall mirror images) of jittered triangular arrangements; a hand-made diagonal flip and
 *                      flips of a triangulated grid; Nu_drop = 1 + U T(y_i) ny / (kappa dT) in a uniform stream
 *                      (tests/test_oracle_analysis.py)               section 2.4, Eq. (25) (R23-R26)
 *   rough walls        alpha = 0 is the rectangular post mask; site counts of the trapezoid; vertical side of the
 *                      asymmetric one; mirror images                          section 4, Table A.6 (R27)
 *   perturbation       densities unchanged, momentum rho du, u^(H) = du on a rest state         L322 (R29)
 *   posts / corners    second, independently written streaming formulation
 *                      (orc_step_push_ghost) must agree bit for bit with the link-wise
 *                      pull of orc_step, and the rule commutes with the symmetries of the lattice
 *                      (transpose, mirrors); beyond that and mass conservation the post-corner
 *                      rule is a reading (R7/R19): "parity unpinned" for it.
 *
 * Build: gcc -O2 -ffp-contract=off -shared -fPIC -o liborc.so tlb_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- D2Q9 lattice, PAPER L74 and Fig. 1(b) L95-102; direction order = reading R1 ---- */
static const int CX[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
static const int CY[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
static const int OPP[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};
static const double W[9] = {4.0 / 9.0,  1.0 / 9.0,  1.0 / 9.0,  1.0 / 9.0, 1.0 / 9.0,
                            1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};

/* weight p(c) of Fig. 1(b) as a function of |c|^2 (the column printed as "|c_i|") */
static double p_of_c2(int c2) {
  switch (c2) {
    case 0: return 247.0 / 420.0;
    case 1: return 4.0 / 63.0;
    case 2: return 4.0 / 135.0;
    case 4: return 1.0 / 180.0;
    case 5: return 2.0 / 945.0;
    case 8: return 1.0 / 15120.0;
  }
  return 0.0;
}
/* weight w(c) of Fig. 1(b): zero outside the NN zone */
static double w_of_c2(int c2) {
  switch (c2) {
    case 0: return 4.0 / 9.0;
    case 1: return 1.0 / 9.0;
    case 2: return 1.0 / 36.0;
  }
  return 0.0;
}

typedef struct orc_params {
  double tau, tau_g;                  /* Eqs. (2), (16)                       */
  double rho0;                        /* Eqs. (8), (12)                       */
  double G12, G11a, G11r, G22a, G22r; /* Eqs. (7), (10), (11)                 */
  double rho_wall_A, rho_wall_B;      /* rhoWallMax / rhoWallMin, L155        */
  double T_bottom, T_top, T_ref;      /* Tdown / Tup L314; footnote 3 L182    */
  double alpha_g;                     /* Eq. (22)                             */
  double body_ax;                     /* extension: uniform acceleration in x */
  double u_wall_bottom, u_wall_top;   /* x-velocity of the flat walls, L147-151 (R20) */
  int32_t periodic_y;                 /* L147, L284-302                       */
  int32_t thermal;                    /* THERMAL, L314                        */
} orc_params;

typedef struct orc_state {
  int nx, ny;
  orc_params p;
  double *fA, *fB, *g;       /* [9][ny][nx], time-t populations; 0 on solid sites */
  double *fAs, *fBs, *gs;    /* post-collision scratch                             */
  double *rhoA, *rhoB, *T;   /* step 1                                              */
  double *jx, *jy;           /* step 1                                              */
  double *psxA, *psxB;       /* psi of Eq. (8)                                      */
  double *pssA, *pssB;       /* psi of Eq. (12)                                     */
  double *FAx, *FAy, *FBx, *FBy; /* step 3                                          */
  double *uHx, *uHy;         /* L139                                                */
  uint8_t *solid;            /* [ny][nx]                                            */
} orc_state;

#define IDX(s, x, y) ((size_t)(y) * (size_t)(s)->nx + (size_t)(x))
#define PIDX(s, i, x, y) ((size_t)(i) * (size_t)(s)->nx * (size_t)(s)->ny + IDX(s, x, y))

static int wrap(int a, int n) {
  a %= n;
  return a < 0 ? a + n : a;
}

/* Is lattice node (x, y) solid?  x is periodic always (L147); y is periodic or bounded by
 * walls whose first solid rows are y = -1 and y = ny (half-way planes at y = -1/2 and
 * ny - 1/2); every node beyond a wall is solid (R9). */
static int is_solid(const orc_state *s, int x, int y) {
  x = wrap(x, s->nx);
  if (s->p.periodic_y) y = wrap(y, s->ny);
  else if (y < 0 || y >= s->ny) return 1;
  return s->solid[IDX(s, x, y)] != 0;
}

/* Wall temperature carried by a solid node (R8): bottom half -> T_bottom, top half -> T_top. */
static double T_wall(const orc_state *s, int y) { return (2 * y < s->ny) ? s->p.T_bottom : s->p.T_top; }

orc_state *orc_create(int nx, int ny, const orc_params *p) {
  if (nx < 1 || ny < 1 || !p) return NULL;
  orc_state *s = (orc_state *)calloc(1, sizeof(orc_state));
  size_t n = (size_t)nx * (size_t)ny;
  s->nx = nx; s->ny = ny; s->p = *p;
  double **nine[] = {&s->fA, &s->fB, &s->g, &s->fAs, &s->fBs, &s->gs};
  for (int k = 0; k < 6; k++) *nine[k] = (double *)calloc(9 * n, sizeof(double));
  double **one[] = {&s->rhoA, &s->rhoB, &s->T, &s->jx, &s->jy, &s->psxA, &s->psxB, &s->pssA,
                    &s->pssB, &s->FAx, &s->FAy, &s->FBx, &s->FBy, &s->uHx, &s->uHy};
  for (int k = 0; k < 15; k++) *one[k] = (double *)calloc(n, sizeof(double));
  s->solid = (uint8_t *)calloc(n, 1);
  return s;
}

void orc_destroy(orc_state *s) {
  if (!s) return;
  double *all[] = {s->fA, s->fB, s->g, s->fAs, s->fBs, s->gs, s->rhoA, s->rhoB, s->T, s->jx, s->jy,
                   s->psxA, s->psxB, s->pssA, s->pssB, s->FAx, s->FAy, s->FBx, s->FBy, s->uHx, s->uHy};
  for (int k = 0; k < 21; k++) free(all[k]);
  free(s->solid);
  free(s);
}

void orc_set_solid(orc_state *s, const uint8_t *solid) {
  size_t n = (size_t)s->nx * s->ny;
  memcpy(s->solid, solid, n);
  for (int i = 0; i < 9; i++)
    for (size_t k = 0; k < n; k++)
      if (s->solid[k]) s->fA[i * n + k] = s->fB[i * n + k] = s->g[i * n + k] = 0.0;
}

/* Initial populations (R14): equilibrium at rest, f = w rho, g = w T. */
void orc_set_fields(orc_state *s, const double *rhoA, const double *rhoB, const double *T) {
  size_t n = (size_t)s->nx * s->ny;
  for (int i = 0; i < 9; i++)
    for (size_t k = 0; k < n; k++) {
      int sol = s->solid[k];
      s->fA[i * n + k] = sol ? 0.0 : W[i] * rhoA[k];
      s->fB[i * n + k] = sol ? 0.0 : W[i] * rhoB[k];
      s->g[i * n + k] = sol ? 0.0 : W[i] * T[k];
    }
}

void orc_set_populations(orc_state *s, const double *fA, const double *fB, const double *g) {
  size_t n9 = 9 * (size_t)s->nx * s->ny;
  memcpy(s->fA, fA, n9 * sizeof(double));
  memcpy(s->fB, fB, n9 * sizeof(double));
  memcpy(s->g, g, n9 * sizeof(double));
}

void orc_get_populations(const orc_state *s, double *fA, double *fB, double *g) {
  size_t n9 = 9 * (size_t)s->nx * s->ny;
  memcpy(fA, s->fA, n9 * sizeof(double));
  memcpy(fB, s->fB, n9 * sizeof(double));
  memcpy(g, s->g, n9 * sizeof(double));
}

/* densities / pseudopotentials seen by the force stencil at ANY node, incl. walls (L155, R9) */
static double rho_at(const orc_state *s, const double *rho, double rho_wall, int x, int y) {
  if (is_solid(s, x, y)) return rho_wall;
  x = wrap(x, s->nx);
  if (s->p.periodic_y) y = wrap(y, s->ny);
  return rho[IDX(s, x, y)];
}
static double psi_x_of(const orc_state *s, double rho) { return rho / s->p.rho0; }                      /* Eq. (8)  */
static double psi_s_of(const orc_state *s, double rho) { return s->p.rho0 * (1.0 - exp(-rho / s->p.rho0)); } /* Eq. (12) */

/* Steps 1-4 of the update: moments, pseudopotentials, forces, hydrodynamic velocity.
 * Everything is a time-t quantity (R13). */
static void moments_and_forces(orc_state *s) {
  const int nx = s->nx, ny = s->ny;
  const orc_params *p = &s->p;
  /* step 1: Eqs. (4), (5), (17) */
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      size_t k = IDX(s, x, y);
      if (s->solid[k]) {
        s->rhoA[k] = p->rho_wall_A; s->rhoB[k] = p->rho_wall_B;
        s->T[k] = T_wall(s, y); s->jx[k] = s->jy[k] = 0.0;
        continue;
      }
      double ra = 0, rb = 0, t = 0, jx = 0, jy = 0;
      for (int i = 0; i < 9; i++) {
        double a = s->fA[PIDX(s, i, x, y)], b = s->fB[PIDX(s, i, x, y)];
        ra += a; rb += b;
        jx += CX[i] * a + CX[i] * b;
        jy += CY[i] * a + CY[i] * b;
        t += s->g[PIDX(s, i, x, y)];
      }
      s->rhoA[k] = ra; s->rhoB[k] = rb; s->T[k] = t; s->jx[k] = jx; s->jy[k] = jy;
    }
  /* step 2: Eqs. (8), (12) on every in-domain node (solid nodes hold the wall densities) */
  for (size_t k = 0; k < (size_t)nx * ny; k++) {
    s->psxA[k] = psi_x_of(s, s->rhoA[k]); s->psxB[k] = psi_x_of(s, s->rhoB[k]);
    s->pssA[k] = psi_s_of(s, s->rhoA[k]); s->pssB[k] = psi_s_of(s, s->rhoB[k]);
  }
  const double psx_wA = psi_x_of(s, p->rho_wall_A), psx_wB = psi_x_of(s, p->rho_wall_B);
  const double pss_wA = psi_s_of(s, p->rho_wall_A), pss_wB = psi_s_of(s, p->rho_wall_B);
  /* step 3: Eqs. (7), (10), (11) then (22) */
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      size_t k = IDX(s, x, y);
      if (s->solid[k]) { s->FAx[k] = s->FAy[k] = s->FBx[k] = s->FBy[k] = 0; s->uHx[k] = s->uHy[k] = 0; continue; }
      double xA[2] = {0, 0}, xB[2] = {0, 0}; /* sum_NN w psi^x_{l'}(x+c) c          */
      double aA[2] = {0, 0}, aB[2] = {0, 0}; /* sum_NN w psi^s_l(x+c) c              */
      double rA[2] = {0, 0}, rB[2] = {0, 0}; /* sum_{NN+NNN} p psi^s_l(x+c) c        */
      for (int dy = -2; dy <= 2; dy++)
        for (int dx = -2; dx <= 2; dx++) {
          int c2 = dx * dx + dy * dy;
          if (c2 == 0) continue;
          int xx = x + dx, yy = y + dy;
          double nxA, nxB, nsA, nsB;
          if (is_solid(s, xx, yy)) { nxA = psx_wA; nxB = psx_wB; nsA = pss_wA; nsB = pss_wB; }
          else {
            size_t kk = IDX(s, wrap(xx, nx), p->periodic_y ? wrap(yy, ny) : yy);
            nxA = s->psxA[kk]; nxB = s->psxB[kk]; nsA = s->pssA[kk]; nsB = s->pssB[kk];
          }
          double w = w_of_c2(c2), pp = p_of_c2(c2);
          if (w != 0.0) {
            xA[0] += w * nxB * dx; xA[1] += w * nxB * dy; /* A feels psi^x of B */
            xB[0] += w * nxA * dx; xB[1] += w * nxA * dy;
            aA[0] += w * nsA * dx; aA[1] += w * nsA * dy;
            aB[0] += w * nsB * dx; aB[1] += w * nsB * dy;
          }
          rA[0] += pp * nsA * dx; rA[1] += pp * nsA * dy;
          rB[0] += pp * nsB * dx; rB[1] += pp * nsB * dy;
        }
      double Tk = p->thermal ? s->T[k] : p->T_ref;
      double FAx = -p->G12 * s->psxA[k] * xA[0] - p->G11a * s->pssA[k] * aA[0] - p->G11r * s->pssA[k] * rA[0];
      double FAy = -p->G12 * s->psxA[k] * xA[1] - p->G11a * s->pssA[k] * aA[1] - p->G11r * s->pssA[k] * rA[1];
      double FBx = -p->G12 * s->psxB[k] * xB[0] - p->G22a * s->pssB[k] * aB[0] - p->G22r * s->pssB[k] * rB[0];
      double FBy = -p->G12 * s->psxB[k] * xB[1] - p->G22a * s->pssB[k] * aB[1] - p->G22r * s->pssB[k] * rB[1];
      FAy += s->rhoA[k] * p->alpha_g * (Tk - p->T_ref); /* Eq. (22), R12 */
      FBy += s->rhoB[k] * p->alpha_g * (Tk - p->T_ref);
      FAx += s->rhoA[k] * p->body_ax;                    /* extension     */
      FBx += s->rhoB[k] * p->body_ax;
      s->FAx[k] = FAx; s->FAy[k] = FAy; s->FBx[k] = FBx; s->FBy[k] = FBy;
      /* L139: rho u^(H) = rho u + F/2 */
      double rho = s->rhoA[k] + s->rhoB[k];
      s->uHx[k] = (s->jx[k] + 0.5 * (FAx + FBx)) / rho;
      s->uHy[k] = (s->jy[k] + 0.5 * (FAy + FBy)) / rho;
    }
}

/* Eq. (3) / Eq. (18) with c_s^2 = 1/3 */
static double equilibrium(int i, double dens, double ux, double uy) {
  double cu = CX[i] * ux + CY[i] * uy;
  return W[i] * dens * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * (ux * ux + uy * uy));
}

/* step 5: BGK collision, Eqs. (2), (6), (16) */
static void collide(orc_state *s) {
  const orc_params *p = &s->p;
  for (int y = 0; y < s->ny; y++)
    for (int x = 0; x < s->nx; x++) {
      size_t k = IDX(s, x, y);
      if (s->solid[k]) continue;
      double rho = s->rhoA[k] + s->rhoB[k];
      double ux = s->jx[k] / rho, uy = s->jy[k] / rho;            /* Eq. (5) */
      double uAx = ux + p->tau * s->FAx[k] / s->rhoA[k];          /* Eq. (6) */
      double uAy = uy + p->tau * s->FAy[k] / s->rhoA[k];
      double uBx = ux + p->tau * s->FBx[k] / s->rhoB[k];
      double uBy = uy + p->tau * s->FBy[k] / s->rhoB[k];
      for (int i = 0; i < 9; i++) {
        size_t q = PIDX(s, i, x, y);
        s->fAs[q] = s->fA[q] - (s->fA[q] - equilibrium(i, s->rhoA[k], uAx, uAy)) / p->tau;
        s->fBs[q] = s->fB[q] - (s->fB[q] - equilibrium(i, s->rhoB[k], uBx, uBy)) / p->tau;
        if (p->thermal)
          s->gs[q] = s->g[q] - (s->g[q] - equilibrium(i, s->T[k], s->uHx[k], s->uHy[k])) / p->tau_g;
        else
          s->gs[q] = s->g[q];
      }
    }
}

/* step 6, link-wise pull: f_i(x,t+1) = f*_i(x - c_i) if that node is fluid, else half-way
 * bounce-back f*_opp(i)(x) (L151, R7) and anti-bounce-back for g (R8). */
static void stream_pull(orc_state *s) {
  const int nx = s->nx, ny = s->ny;
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      if (s->solid[IDX(s, x, y)]) continue;
      for (int i = 0; i < 9; i++) {
        int sx = x - CX[i], sy = y - CY[i];
        size_t q = PIDX(s, i, x, y);
        if (!is_solid(s, sx, sy)) {
          size_t src = PIDX(s, i, wrap(sx, nx), s->p.periodic_y ? wrap(sy, ny) : sy);
          s->fA[q] = s->fAs[src]; s->fB[q] = s->fBs[src];
          if (s->p.thermal) s->g[q] = s->gs[src];
        } else {
          size_t loc = PIDX(s, OPP[i], x, y);
          s->fA[q] = s->fAs[loc]; s->fB[q] = s->fBs[loc];
          /* R20: a flat wall (ghost row beyond y = -1/2 or ny - 1/2, not a post) moving along x with
           * velocity u_w hands the population back with the momentum of the wall,
           * f_i = f*_opp(i) + 2 w_i rho_l (c_i . u_w) / c_s^2, c_s^2 = 1/3 (L147-151, Eq. (15)). */
          if (!s->p.periodic_y && (sy < 0 || sy >= ny)) {
            double uw = sy < 0 ? s->p.u_wall_bottom : s->p.u_wall_top;
            s->fA[q] += 6.0 * W[i] * s->rhoA[IDX(s, x, y)] * (CX[i] * uw);
            s->fB[q] += 6.0 * W[i] * s->rhoB[IDX(s, x, y)] * (CX[i] * uw);
          }
          if (s->p.thermal) {
            int wy = s->p.periodic_y ? wrap(sy, ny) : sy;
            s->g[q] = -s->gs[loc] + 2.0 * W[i] * T_wall(s, wy);
          }
        }
      }
    }
}

void orc_step(orc_state *s, long n) {
  for (long t = 0; t < n; t++) {
    moments_and_forces(s);
    collide(s);
    stream_pull(s);
  }
}

/* Second, independently written streaming formulation used only to pin the post-corner /
 * ghost-node logic: push every post-collision population into a lattice padded by one ghost
 * layer (PAPER footnote 2, L180), fold periodic ghosts back, then let every solid or ghost
 * node hand each population it received back to the fluid node it came from, reversed. */
void orc_step_push_ghost(orc_state *s, long n) {
  const int nx = s->nx, ny = s->ny, px = nx + 2, py = ny + 2;
  const size_t pn = (size_t)px * py;
  double *PA = (double *)malloc(9 * pn * sizeof(double));
  double *PB = (double *)malloc(9 * pn * sizeof(double));
  double *PG = (double *)malloc(9 * pn * sizeof(double));
  uint8_t *got = (uint8_t *)malloc(9 * pn);
  for (long t = 0; t < n; t++) {
    moments_and_forces(s);
    collide(s);
    memset(got, 0, 9 * pn);
    /* push */
    for (int y = 0; y < ny; y++)
      for (int x = 0; x < nx; x++) {
        if (s->solid[IDX(s, x, y)]) continue;
        for (int i = 0; i < 9; i++) {
          size_t d = (size_t)i * pn + (size_t)(y + CY[i] + 1) * px + (size_t)(x + CX[i] + 1);
          PA[d] = s->fAs[PIDX(s, i, x, y)]; PB[d] = s->fBs[PIDX(s, i, x, y)]; PG[d] = s->gs[PIDX(s, i, x, y)];
          got[d] = 1;
        }
      }
    /* every padded node, ghost or not, passes on what it received */
    for (int gy = -1; gy <= ny; gy++)
      for (int gx = -1; gx <= nx; gx++)
        for (int i = 0; i < 9; i++) {
          size_t d = (size_t)i * pn + (size_t)(gy + 1) * px + (size_t)(gx + 1);
          if (!got[d]) continue;
          int tx = wrap(gx, nx), ty = gy;
          if (s->p.periodic_y) ty = wrap(gy, ny);
          int solid_here = (ty < 0 || ty >= ny) ? 1 : (s->solid[IDX(s, tx, ty)] != 0);
          if (!solid_here) { /* fluid target (possibly reached through a periodic ghost) */
            s->fA[PIDX(s, i, tx, ty)] = PA[d]; s->fB[PIDX(s, i, tx, ty)] = PB[d];
            if (s->p.thermal) s->g[PIDX(s, i, tx, ty)] = PG[d];
          } else {           /* wall / post: hand back reversed to the sender */
            int ox = wrap(gx - CX[i], nx), oy = gy - CY[i];
            if (s->p.periodic_y) oy = wrap(oy, ny);
            s->fA[PIDX(s, OPP[i], ox, oy)] = PA[d]; s->fB[PIDX(s, OPP[i], ox, oy)] = PB[d];
            if (ty < 0 || ty >= ny) { /* moving flat wall, R20: the returned direction is opp(i) */
              double uw = ty < 0 ? s->p.u_wall_bottom : s->p.u_wall_top;
              s->fA[PIDX(s, OPP[i], ox, oy)] += 6.0 * W[OPP[i]] * s->rhoA[IDX(s, ox, oy)] * (CX[OPP[i]] * uw);
              s->fB[PIDX(s, OPP[i], ox, oy)] += 6.0 * W[OPP[i]] * s->rhoB[IDX(s, ox, oy)] * (CX[OPP[i]] * uw);
            }
            if (s->p.thermal) s->g[PIDX(s, OPP[i], ox, oy)] = -PG[d] + 2.0 * W[i] * T_wall(s, ty);
          }
        }
  }
  free(PA); free(PB); free(PG); free(got);
}

/* Hydrodynamic fields at the current time: rho_A, rho_B, u^(H) (2 planes), T.
 * Solid sites report rho = rho_wall, u = 0, T = that wall's temperature. */
void orc_fields(orc_state *s, double *rhoA, double *rhoB, double *u, double *T) {
  size_t n = (size_t)s->nx * s->ny;
  moments_and_forces(s);
  memcpy(rhoA, s->rhoA, n * sizeof(double));
  memcpy(rhoB, s->rhoB, n * sizeof(double));
  memcpy(u, s->uHx, n * sizeof(double));
  memcpy(u + n, s->uHy, n * sizeof(double));
  memcpy(T, s->T, n * sizeof(double));
}

/* Interaction + external force on each component (for the tests of Eq. (9) / Eq. (22)). */
void orc_forces(orc_state *s, double *FA, double *FB) {
  size_t n = (size_t)s->nx * s->ny;
  moments_and_forces(s);
  memcpy(FA, s->FAx, n * sizeof(double)); memcpy(FA + n, s->FAy, n * sizeof(double));
  memcpy(FB, s->FBx, n * sizeof(double)); memcpy(FB + n, s->FBy, n * sizeof(double));
}

/* Observables: out = {mass_A, mass_B, E, Nu}.
 *   mass_l = sum over fluid sites of rho_l                                   (north_star)
 *   E      = (1/N_fluid) sum |u^(H)|^2                                       (L248, R11)
 *   Nu     = [<u_y^(H) T> - kappa <d_y T>] / (kappa dT / ny)                 (Eq. (24), R10)
 * with kappa = (tau_g - 1/2)/3 (Eq. (20)), averages over fluid sites, and
 * d_y T(x,y) = Tface(x,y+1/2) - Tface(x,y-1/2), Tface = mean of the two adjacent rows when the
 * neighbour is fluid, the wall temperature when it is solid.  long double accumulators. */
void orc_observables(orc_state *s, double out[4]) {
  const int nx = s->nx, ny = s->ny;
  moments_and_forces(s);
  long double mA = 0, mB = 0, e = 0, uT = 0, dT = 0;
  long nf = 0;
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      size_t k = IDX(s, x, y);
      if (s->solid[k]) continue;
      nf++;
      mA += s->rhoA[k]; mB += s->rhoB[k];
      e += s->uHx[k] * s->uHx[k] + s->uHy[k] * s->uHy[k];
      uT += s->uHy[k] * s->T[k];
      double up, dn;
      if (is_solid(s, x, y + 1)) up = T_wall(s, s->p.periodic_y ? wrap(y + 1, ny) : y + 1);
      else up = 0.5 * (s->T[k] + s->T[IDX(s, x, s->p.periodic_y ? wrap(y + 1, ny) : y + 1)]);
      if (is_solid(s, x, y - 1)) dn = T_wall(s, s->p.periodic_y ? wrap(y - 1, ny) : y - 1);
      else dn = 0.5 * (s->T[k] + s->T[IDX(s, x, s->p.periodic_y ? wrap(y - 1, ny) : y - 1)]);
      dT += up - dn;
    }
  double kappa = (s->p.tau_g - 0.5) / 3.0;
  double DT = s->p.T_bottom - s->p.T_top;
  out[0] = (double)mA; out[1] = (double)mB;
  out[2] = nf ? (double)(e / nf) : 0.0;
  out[3] = (nf && DT != 0.0) ? (double)((uT / nf - kappa * (dT / nf)) / (kappa * DT / ny)) : 0.0;
}

/* x-averaged velocity profile of the Couette output u_av: u_av[y] = mean over the fluid
 * sites of row y of u_x^(H); 0 for a row without fluid sites. */
void orc_x_average(orc_state *s, double *u_av) {
  moments_and_forces(s);
  for (int y = 0; y < s->ny; y++) {
    long double a = 0;
    long n = 0;
    for (int x = 0; x < s->nx; x++)
      if (!s->solid[IDX(s, x, y)]) { a += s->uHx[IDX(s, x, y)]; n++; }
    u_av[y] = n ? (double)(a / n) : 0.0;
  }
}

/* Stress field P_xy (the paper's Ptot_xy.dat, L248-250; "the sum of all components contributions", L296).
 * The paper prints no formula; reading R21:
 *   kinetic part      sum_l (1/2) sum_i c_ix c_iy (f_l,i + f*_l,i): the momentum flux carried by the populations
 *                     that arrive at the site (f, time t) and by those that leave it (f*, post-collision, Eq. (2))
 *   interaction part  for every pairwise force F(x) = -G psi(x) sum_c k(c) psi'(x+c) c of Eqs. (7), (10), (11)
 *                     the tensor (G/2) psi(x) sum_c k(c) psi'(x+c) c_x c_y, wall values at solid nodes (L155)
 * 0 on solid sites.  Sign: pressure tensor, P_xy = -eta d_y u_x in a simple shear (L143). */
void orc_stress_xy(orc_state *s, double *Pxy) {
  const int nx = s->nx, ny = s->ny;
  const orc_params *p = &s->p;
  moments_and_forces(s);
  collide(s);
  const double psx_wA = psi_x_of(s, p->rho_wall_A), psx_wB = psi_x_of(s, p->rho_wall_B);
  const double pss_wA = psi_s_of(s, p->rho_wall_A), pss_wB = psi_s_of(s, p->rho_wall_B);
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      size_t k = IDX(s, x, y);
      if (s->solid[k]) { Pxy[k] = 0.0; continue; }
      double kin = 0.0;
      for (int i = 0; i < 9; i++) {
        size_t q = PIDX(s, i, x, y);
        kin += 0.5 * (CX[i] * CY[i]) * ((s->fA[q] + s->fAs[q]) + (s->fB[q] + s->fBs[q]));
      }
      double cross = 0.0, selfA = 0.0, selfB = 0.0;
      for (int dy = -2; dy <= 2; dy++)
        for (int dx = -2; dx <= 2; dx++) {
          int c2 = dx * dx + dy * dy;
          if (c2 == 0) continue;
          int xx = x + dx, yy = y + dy;
          double nxA, nxB, nsA, nsB;
          if (is_solid(s, xx, yy)) { nxA = psx_wA; nxB = psx_wB; nsA = pss_wA; nsB = pss_wB; }
          else {
            size_t kk = IDX(s, wrap(xx, nx), p->periodic_y ? wrap(yy, ny) : yy);
            nxA = s->psxA[kk]; nxB = s->psxB[kk]; nsA = s->pssA[kk]; nsB = s->pssB[kk];
          }
          double w = w_of_c2(c2), pp = p_of_c2(c2);
          cross += w * (s->psxA[k] * nxB + s->psxB[k] * nxA) * (dx * dy);
          selfA += (p->G11a * w + p->G11r * pp) * s->pssA[k] * nsA * (dx * dy);
          selfB += (p->G22a * w + p->G22r * pp) * s->pssB[k] * nsB * (dx * dy);
        }
      Pxy[k] = kin + 0.5 * (p->G12 * cross + selfA + selfB);
    }
}

/* x-average over the fluid sites of every row of a field plane (Pxy_av.dat, L250); 0 for a row without fluid. */
void orc_row_average(const orc_state *s, const double *plane, double *av) {
  for (int y = 0; y < s->ny; y++) {
    long double a = 0;
    long n = 0;
    for (int x = 0; x < s->nx; x++)
      if (!s->solid[IDX(s, x, y)]) { a += plane[IDX(s, x, y)]; n++; }
    av[y] = n ? (double)(a / n) : 0.0;
  }
}

/* x-momentum of every row, sum over x, both species and all directions of c_ix f_l,i (the conserved quantity
 * the stress pins balance). */
void orc_row_momentum_x(const orc_state *s, double *mx) {
  for (int y = 0; y < s->ny; y++) {
    long double a = 0;
    for (int x = 0; x < s->nx; x++)
      for (int i = 0; i < 9; i++) a += CX[i] * (s->fA[PIDX(s, i, x, y)] + s->fB[PIDX(s, i, x, y)]);
    mx[y] = (double)a;
  }
}

/* Droplet analysis, first stage (section 2.4; reading R22): bulk sites are the fluid sites with
 * rho_A > B_th; a droplet is a cluster of bulk sites connected through nearest-neighbour bonds (the bonds of the
 * Ising cluster algorithms the paper adapts, L198), x periodic, y periodic iff periodic_y.  Plain flood fill in
 * site-index order, so a cluster's label is its smallest site index y nx + x; -1 off the bulk.
 * stats[k] = {label, sites, centre x, centre y} in ascending label order, the centre being the mean position of
 * the cluster's sites: integer sums of minimum-image offsets from the label site (signed, in [-n/2, n/2)),
 * one division, wrapped to [0, nx) (and [0, ny) when y is periodic).  Returns the number of droplets; only the
 * first max_droplets rows of stats are written. */
static int min_image(int a, int b, int n) {
  int d = a - b;
  if (2 * d >= n) d -= n;
  else if (2 * d < -n) d += n;
  return d;
}
int orc_droplets(orc_state *s, double B_th, int32_t *labels, int max_droplets, double *stats) {
  const int nx = s->nx, ny = s->ny;
  const size_t n = (size_t)nx * ny;
  moments_and_forces(s);
  int32_t *lab = labels ? labels : (int32_t *)malloc(n * sizeof(int32_t));
  int *stack = (int *)malloc(n * sizeof(int));
  for (size_t k = 0; k < n; k++) lab[k] = (!s->solid[k] && s->rhoA[k] > B_th) ? -2 : -1; /* -2: bulk, unvisited */
  int found = 0;
  for (size_t k = 0; k < n; k++) {
    if (lab[k] != -2) continue;
    const int xr = (int)(k % nx), yr = (int)(k / nx);
    long long cnt = 0, sdx = 0, sdy = 0;
    int top = 0;
    stack[top++] = (int)k;
    lab[k] = (int32_t)k;
    while (top) {
      const int q = stack[--top], x = q % nx, y = q / nx;
      cnt++;
      sdx += min_image(x, xr, nx);
      sdy += s->p.periodic_y ? min_image(y, yr, ny) : y - yr;
      const int nbx[4] = {wrap(x + 1, nx), wrap(x - 1, nx), x, x};
      int nby[4] = {y, y, y + 1, y - 1};
      for (int b = 0; b < 4; b++) {
        if (s->p.periodic_y) nby[b] = wrap(nby[b], ny);
        else if (nby[b] < 0 || nby[b] >= ny) continue;
        const size_t m = IDX(s, nbx[b], nby[b]);
        if (lab[m] == -2) { lab[m] = (int32_t)k; stack[top++] = (int)m; }
      }
    }
    if (found < max_droplets) {
      double cx = (double)xr + (double)sdx / (double)cnt, cy = (double)yr + (double)sdy / (double)cnt;
      if (cx < 0.0) cx += nx;
      if (cx >= nx) cx -= nx;
      if (s->p.periodic_y) { if (cy < 0.0) cy += ny; if (cy >= ny) cy -= ny; }
      stats[4 * found + 0] = (double)k; stats[4 * found + 1] = (double)cnt;
      stats[4 * found + 2] = cx; stats[4 * found + 3] = cy;
    }
    found++;
  }
  free(stack);
  if (!labels) free(lab);
  return found;
}

/* ---- Droplet analysis, second stage (section 2.4; readings R23-R26 of DESIGN.md).  The paper gives the
 * ingredients in prose and defers the details to its ref. [58], which is not available; every choice below is a
 * reading.  These functions are geometric: they take the centres / colours / link lists as arguments. ---- */

/* signed offset a - c for a lattice coordinate a and a real centre coordinate c, minimum image when periodic */
static double offset_to(int a, double c, int n, int periodic) {
  double d = (double)a - c;
  if (periodic) {
    const double half = 0.5 * (double)n;
    if (d > half) d -= (double)n;
    else if (d < -half) d += (double)n;
  }
  return d;
}

/* R23, digital Voronoi tessellation (L198: "each point of the lattice is coloured by the label of the nearest centre
 * of mass"): colour[y][x] = index k of the centre with the smallest squared distance dx*dx + dy*dy (fp64, x minimum
 * image, y minimum image iff periodic_y); ties go to the smallest index; -1 when there are no centres.  Brute force. */
void orc_voronoi(int nx, int ny, int periodic_y, const double *centres, int n, int32_t *colour) {
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      int best = -1;
      double bd = 0.0;
      for (int k = 0; k < n; k++) {
        const double dx = offset_to(x, centres[2 * k], nx, 1), dy = offset_to(y, centres[2 * k + 1], ny, periodic_y);
        const double d2 = dx * dx + dy * dy;
        if (best < 0 || d2 < bd) { best = k; bd = d2; }
      }
      colour[(size_t)y * nx + x] = best;
    }
}

/* the same for a list of m sites (site = y nx + x): lets a test check a large colouring on sampled sites */
void orc_voronoi_at(int nx, int ny, int periodic_y, const double *centres, int n, const int64_t *sites, int m, int32_t *colour) {
  for (int q = 0; q < m; q++) {
    const int x = (int)(sites[q] % nx), y = (int)(sites[q] / nx);
    int best = -1;
    double bd = 0.0;
    for (int k = 0; k < n; k++) {
      const double dx = offset_to(x, centres[2 * k], nx, 1), dy = offset_to(y, centres[2 * k + 1], ny, periodic_y);
      const double d2 = dx * dx + dy * dy;
      if (best < 0 || d2 < bd) { best = k; bd = d2; }
    }
    colour[q] = best;
  }
}

static int cmp_pair(const void *a, const void *b) {
  const int32_t *p = (const int32_t *)a, *q = (const int32_t *)b;
  if (p[0] != q[0]) return p[0] < q[0] ? -1 : 1;
  if (p[1] != q[1]) return p[1] < q[1] ? -1 : 1;
  return 0;
}
static int sort_unique_pairs(int32_t *v, int n) {
  qsort(v, (size_t)n, 2 * sizeof(int32_t), cmp_pair);
  int m = 0;
  for (int k = 0; k < n; k++)
    if (m == 0 || v[2 * k] != v[2 * m - 2] || v[2 * k + 1] != v[2 * m - 1]) { v[2 * m] = v[2 * k]; v[2 * m + 1] = v[2 * k + 1]; m++; }
  return m;
}

/* R24, Delaunay links (L198: "The vertices at which adjacent digital Voronoi cells converge are used to identify the
 * Delaunay triangulation").  A vertex is a 2 x 2 block of lattice sites {(x, y), (x+1, y), (x, y+1), (x+1, y+1)}
 * (x periodic; y periodic iff periodic_y, else the rows y = -1 and y = ny beyond the flat walls carry the wall
 * colour -1, so that a Voronoi edge that ends on a wall still ends in a vertex) that holds at least 3 distinct
 * colours.  Three colours: every pair of droplet colours in the block is a link.  Four colours (the degenerate
 * quadrilateral): the four side-adjacent pairs and the pair on the main diagonal (x, y)-(x+1, y+1).
 * Output: the distinct links (a < b) in lexicographic order; returns their number, writes at most max_links. */
int orc_delaunay(int nx, int ny, int periodic_y, const int32_t *colour, int max_links, int32_t *links) {
  int cap = 1024, n = 0;
  int32_t *v = (int32_t *)malloc((size_t)cap * 2 * sizeof(int32_t));
  for (int y = periodic_y ? 0 : -1; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      const int x1 = x + 1 == nx ? 0 : x + 1;
      int y1 = y + 1;
      if (periodic_y && y1 == ny) y1 = 0;
      const int32_t c00 = y < 0 ? -1 : colour[(size_t)y * nx + x], c10 = y < 0 ? -1 : colour[(size_t)y * nx + x1];
      const int32_t c01 = y1 >= ny ? -1 : colour[(size_t)y1 * nx + x], c11 = y1 >= ny ? -1 : colour[(size_t)y1 * nx + x1];
      const int32_t c[4] = {c00, c10, c01, c11};
      int distinct = 0;
      for (int i = 0; i < 4; i++) {
        int seen = 0;
        for (int j = 0; j < i; j++) seen |= c[j] == c[i];
        distinct += !seen;
      }
      if (distinct < 3) continue;
      /* pairs of block positions: sides 0-1, 2-3, 0-2, 1-3, diagonals 0-3 (main), 1-2 */
      static const int PA[6] = {0, 2, 0, 1, 0, 1}, PB[6] = {1, 3, 2, 3, 3, 2};
      for (int e = 0; e < 6; e++) {
        if (distinct == 4 && e == 5) continue;
        int32_t a = c[PA[e]], b = c[PB[e]];
        if (a < 0 || b < 0 || a == b) continue;
        if (a > b) { const int32_t t = a; a = b; b = t; }
        if (n == cap) { cap *= 2; v = (int32_t *)realloc(v, (size_t)cap * 2 * sizeof(int32_t)); }
        v[2 * n] = a; v[2 * n + 1] = b; n++;
      }
    }
  n = sort_unique_pairs(v, n);
  for (int k = 0; k < n && k < max_links; k++) { links[2 * k] = v[2 * k]; links[2 * k + 1] = v[2 * k + 1]; }
  free(v);
  return n;
}

/* R25 (first half), droplet identity between two frames: droplet i of the present frame is the droplet of the past
 * frame in whose digital Voronoi cell its centre lies, map[i] = colour_past at the lattice site nearest to the
 * centre (floor(c + 1/2), x wrapped, y wrapped or clamped). */
static int nearest_site(double c, int n, int periodic) {
  int r = (int)floor(c + 0.5);
  if (periodic) { r %= n; if (r < 0) r += n; }
  else { if (r < 0) r = 0; if (r >= n) r = n - 1; }
  return r;
}
void orc_match(int nx, int ny, int periodic_y, const int32_t *colour_past, const double *centres_now, int n_now, int32_t *map) {
  for (int i = 0; i < n_now; i++)
    map[i] = colour_past[(size_t)nearest_site(centres_now[2 * i + 1], ny, periodic_y) * nx + nearest_site(centres_now[2 * i], nx, 1)];
}

/* Droplet displacement field (L326, L340: "Lagrangian droplet displacement vector fields d(X_i(t), t) ... computed for all
 * droplet centre-of-mass"; the deltaAnalysis output): d_i = X_i(now) - X_map[i](past), minimum image in x (and in y when
 * periodic); a droplet without a past partner (map < 0) gets (0, 0). */
void orc_displacements(int nx, int ny, int periodic_y, const double *centres_past, const double *centres_now, const int32_t *map,
                       int n_now, double *disp) {
  for (int i = 0; i < n_now; i++) {
    double dx = 0.0, dy = 0.0;
    if (map[i] >= 0) {
      dx = centres_now[2 * i] - centres_past[2 * map[i]];
      dy = centres_now[2 * i + 1] - centres_past[2 * map[i] + 1];
      const double hx = 0.5 * (double)nx, hy = 0.5 * (double)ny;
      if (dx > hx) dx -= (double)nx; else if (dx < -hx) dx += (double)nx;
      if (periodic_y) { if (dy > hy) dy -= (double)ny; else if (dy < -hy) dy += (double)ny; }
    }
    disp[2 * i] = dx; disp[2 * i + 1] = dy;
  }
}

static int has_pair(const int32_t *v, int n, int32_t a, int32_t b) {
  if (a > b) { const int32_t t = a; a = b; b = t; }
  for (int k = 0; k < n; k++)
    if (v[2 * k] == a && v[2 * k + 1] == b) return 1;
  return 0;
}

/* R25 (second half), T1 events (L198-200: "Subsequent Delaunay triangulations are compared in order to detect T1
 * plastic rearrangements ... These topological events only involve 4 droplets ... at the four vertices of a
 * quadrilateral labelled a, b, c and d, and they are associated with a 'flip' of the diagonal link": "the diagonal
 * link between a and b is replaced by the link between c and d").  The links of the present frame are first written
 * in the indices of the past frame through `map` (links with an unmatched end, map < 0, or with both ends on the same
 * past droplet are dropped).  An event (a, b, c, d), a < b, c < d, is: link a-b in the past and not now; link c-d now
 * and not in the past; the four sides a-c, a-d, b-c, b-d present in both frames.  Plain search over all quadruples
 * of links; output in lexicographic order; returns the number of events, writes at most max_events. */
int orc_t1_events(const int32_t *past, int n_past, const int32_t *now, int n_now, const int32_t *map, int max_events,
                  int32_t *events) {
  int32_t *cur = (int32_t *)malloc((size_t)(n_now > 0 ? n_now : 1) * 2 * sizeof(int32_t));
  int m = 0;
  for (int k = 0; k < n_now; k++) {
    int32_t a = map ? map[now[2 * k]] : now[2 * k], b = map ? map[now[2 * k + 1]] : now[2 * k + 1];
    if (a < 0 || b < 0 || a == b) continue;
    if (a > b) { const int32_t t = a; a = b; b = t; }
    cur[2 * m] = a; cur[2 * m + 1] = b; m++;
  }
  m = sort_unique_pairs(cur, m);
  int found = 0;
  for (int k = 0; k < n_past; k++) {          /* past links in lexicographic order -> events come out sorted by (a, b) */
    const int32_t a = past[2 * k], b = past[2 * k + 1];
    if (has_pair(cur, m, a, b)) continue;
    for (int j = 0; j < m; j++) {             /* present links in lexicographic order -> then by (c, d) */
      const int32_t c = cur[2 * j], d = cur[2 * j + 1];
      if (has_pair(past, n_past, c, d)) continue;
      if (c == a || c == b || d == a || d == b) continue;
      const int sides = has_pair(past, n_past, a, c) && has_pair(past, n_past, a, d) && has_pair(past, n_past, b, c) &&
                        has_pair(past, n_past, b, d) && has_pair(cur, m, a, c) && has_pair(cur, m, a, d) &&
                        has_pair(cur, m, b, c) && has_pair(cur, m, b, d);
      if (!sides) continue;
      if (found < max_events) { events[4 * found] = a; events[4 * found + 1] = b; events[4 * found + 2] = c; events[4 * found + 3] = d; }
      found++;
    }
  }
  free(cur);
  return found;
}

/* R26, droplet Nusselt number, Eq. (25): Nu_i = [u_y T - kappa d_y T](X_i) / (kappa dT / ny) with the fields
 * "evaluated for the i-th droplet" read at the lattice site nearest to its centre X_i: u_y = u_y^(H), kappa and d_y T as
 * in Eq. (24) / R10; 0 if that site is solid or dT = 0. */
void orc_droplet_nusselt(orc_state *s, const double *centres, int n, double *nu) {
  const int nx = s->nx, ny = s->ny;
  moments_and_forces(s);
  const double kappa = (s->p.tau_g - 0.5) / 3.0, DT = s->p.T_bottom - s->p.T_top;
  for (int i = 0; i < n; i++) {
    const int x = nearest_site(centres[2 * i], nx, 1), y = nearest_site(centres[2 * i + 1], ny, s->p.periodic_y);
    const size_t k = IDX(s, x, y);
    if (s->solid[k] || DT == 0.0) { nu[i] = 0.0; continue; }
    double up, dn;
    if (is_solid(s, x, y + 1)) up = T_wall(s, s->p.periodic_y ? wrap(y + 1, ny) : y + 1);
    else up = 0.5 * (s->T[k] + s->T[IDX(s, x, s->p.periodic_y ? wrap(y + 1, ny) : y + 1)]);
    if (is_solid(s, x, y - 1)) dn = T_wall(s, s->p.periodic_y ? wrap(y - 1, ny) : y - 1);
    else dn = 0.5 * (s->T[k] + s->T[IDX(s, x, s->p.periodic_y ? wrap(y - 1, ny) : y - 1)]);
    nu[i] = (s->uHy[k] * s->T[k] - kappa * (up - dn)) / (kappa * DT / ny);
  }
}

/* ---- Workflow pieces of the paper (readings R27, R29 of DESIGN.md) ---- */

/* R27, rough walls with trapezoidal obstacles (section 4, Fig. 7(a) -- the figure is missing --, Table A.6:
 * roughWallUp, roughWallDown, width, height, lambda, alpha, asymmetric): "The height, the width, the periodicity
 * (via lambda), and the angle (via alpha) can be varied"; alpha = 0 gives "a simple rectangular-shape roughness".
 * Reading: an obstacle stands on the wall every `lambda` nodes; in the row j = 0 .. height - 1 counted from the wall
 * it covers the nodes l(j) <= (x mod lambda) < width - r(j), r(j) = floor(j tan(alpha)) (alpha in radians), l(j) =
 * r(j) for a symmetric trapezoid and 0 (a vertical side) for the asymmetric one.  The top wall carries the mirror
 * image in y.  solid[ny][nx] is overwritten. */
void orc_rough_walls(int nx, int ny, int up, int down, int width, int height, int lambda, double alpha, int asymmetric,
                     uint8_t *solid) {
  const double t = tan(alpha);
  memset(solid, 0, (size_t)nx * ny);
  for (int j = 0; j < height && j < ny; j++) {
    const int r = (int)floor((double)j * t), l = asymmetric ? 0 : r;
    for (int x = 0; x < nx; x++) {
      const int m = x % lambda;
      if (m < l || m >= width - r) continue;
      if (down) solid[(size_t)j * nx + x] = 1;
      if (up) solid[(size_t)(ny - 1 - j) * nx + x] = 1;
    }
  }
}

/* R29, initial velocity perturbation (L322: "a finite perturbation is necessary to destabilise the conductive
 * state"; "initial velocity perturbation" 1e-4 in Table A.5; its shape is not given).  Reading: one convection
 * roll pair, du = (0, A sin(2 pi x / nx) sin(pi (y + 1/2) / ny)), given to both fluids by shifting every population of
 * a fluid site by the first-order equilibrium term, f_l,i += 3 w_i rho_l (c_i . du) with rho_l = sum_i f_l,i: each
 * component's density is unchanged (sum_i w_i c_i = 0) and its momentum grows by rho_l du (sum_i w_i c_i c_i = 1/3). */
void orc_perturb_velocity(orc_state *s, double amplitude) {
  const int nx = s->nx, ny = s->ny;
  const double pi = 3.14159265358979323846;
  for (int y = 0; y < ny; y++)
    for (int x = 0; x < nx; x++) {
      if (s->solid[IDX(s, x, y)]) continue;
      const double duy = amplitude * sin(2.0 * pi * (double)x / (double)nx) * sin(pi * ((double)y + 0.5) / (double)ny);
      double ra = 0.0, rb = 0.0;
      for (int i = 0; i < 9; i++) { ra += s->fA[PIDX(s, i, x, y)]; rb += s->fB[PIDX(s, i, x, y)]; }
      for (int i = 0; i < 9; i++) {
        const double cu = (double)CY[i] * duy;
        s->fA[PIDX(s, i, x, y)] += 3.0 * W[i] * ra * cu;
        s->fB[PIDX(s, i, x, y)] += 3.0 * W[i] * rb * cu;
      }
    }
}

/* lattice constants exported for the weight-invariant pins */
double orc_w(int dx, int dy) { return w_of_c2(dx * dx + dy * dy); }
double orc_p(int dx, int dy) { return p_of_c2(dx * dx + dy * dy); }
void orc_direction(int i, int *cx, int *cy, int *opp) { *cx = CX[i]; *cy = CY[i]; *opp = OPP[i]; }
