/*
 * clip_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded fp64 CPU implementation of one time step of the conservative phase-field
 * lattice Boltzmann method of arxiv 2505.12205 ("CLIP"), D3Q19, written from PAPER.md equation by equation.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.  It
 * shares no code, header, table or constant generator with the CUDA path (paper_2505_12205_b200/csrc).
 *
 * Build:  gcc -O3 -ffp-contract=off -shared -fPIC -o libclip_oracle.so clip_oracle.c -lm
 *         gcc ... -DCLIPO_D2Q9 -o libclip_oracle_d2q9.so clip_oracle.c -lm     (the 2-D lattice of the paper's 2-D benchmarks,
 *         same equations, D2Q9 velocities and weights, nz = 1, faces PERIODIC / WALL / FREESLIP in x and y)
 *
 * Storage follows the paper as written: populations f[index][a], g[index][a] (Alg. 1-3),
 * index = x + nx*(y + ny*z) (Fig. 4b), two full population buffers (the in-place Alg. 2 is a data
 * race, reading G15), dense 19x19 M^-1 S M (Eq. 27).  No fusion, blocking or reordering.
 *
 * Readings of garbled / silent passages are marked [Gn]/[Rn] below.
 * Parity pins: see tests/test_oracle_pins.py, test_oracle_invariants.py (free-slip = mirror plane), test_oracle_physics.py.
 * "parity unpinned" items: R9 at OPEN faces (phi ghost; both readings available: open_ghost), R12's time level of U (the
 * paper's two sentences disagree, PAPER.md:1107 vs :1117; both readings available: outlet_u_time), R13 (lagged u inside the
 * macro update's F_mu).  The algebra of B.25 itself (constant lambda: first-order upwind response, growth factor 1/(1+lambda)
 * per step, hence unstable for lambda < 0 without the clamp) is pinned in tests/test_oracle_outlet.py.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef CLIPO_D2Q9
#define Q 9
#else
#define Q 19
#endif
enum { BC_PERIODIC = 0, BC_WALL = 1, BC_INLET = 2, BC_OUTLET = 3, BC_FREESLIP = 4 };

#ifdef CLIPO_D2Q9
/* D2Q9 (Fig. B.24 :969): rest, 4 axis and 4 diagonal velocities, weights 4/9, 1/9, 1/36; opposite pairs adjacent.
 * The ordering is immaterial [G1] (the 2-D inlet of :1044 is not built). */
static const int EX[Q] = {0, 1, -1, 0, 0, 1, -1, 1, -1};
static const int EY[Q] = {0, 0, 0, 1, -1, 1, -1, -1, 1};
static const int EZ[Q] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
static double weight_of(int a) { return a == 0 ? 4.0 / 9.0 : (a < 5 ? 1.0 / 9.0 : 1.0 / 36.0); }
#define SHEAR_LO 3 /* rows of the traceless second-order moments in the basis below: e_x e_y, e_x^2 - e_y^2 */
#define SHEAR_HI 4
#else
/* D3Q19 velocities, Eq. 14, in the ordering consistent with the inlet set {1,7,9,11,13} being
 * the +x-pointing directions [G1]; opposite pairs adjacent. */
static const int EX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
static const int EY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
static const int EZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
static double weight_of(int a) { return a == 0 ? 1.0 / 3.0 : (a < 7 ? 1.0 / 18.0 : 1.0 / 36.0); } /* Eq. 15 */
#define SHEAR_LO 4 /* rows of the 5 traceless second-order moments in the basis below */
#define SHEAR_HI 8
#endif
static int opp(int a) { return a == 0 ? 0 : ((a & 1) ? a + 1 : a - 1); }

typedef struct clipo_params {
  double rho_h, rho_l;     /* Eq. 39 */
  double tau_h, tau_l;     /* Eq. 23-24 (paper tau: nu = tau/3) */
  double sigma, W, M;      /* Eq. 12, 34, 37 */
  double g[3], rho_ref;    /* F_b = (rho - rho_ref) g [G16] */
  int bc[6];               /* -x,+x,-y,+y,-z,+z */
  double inlet_u[3], inlet_phi, inlet_c[2], inlet_r;
  int outlet_u_mode;       /* B.22: 0 = U_local, 1 = U_ave, 2 = U_max of u_z over layer N-1 */
  int visc_interp;         /* 0: Eq. 24 linear tau; 1: harmonic (1/tau linear; non-paper);
                              2: Eq. 25 linear dynamic viscosity mu = rho tau c_s^2, tau = 3 mu(phi) / rho(phi) */
  int collision;           /* 0: WMRT, Eq. 27-28, 30; 1: BGK, Eq. 26, 29 */
  int phase_only;          /* 1: only the phase-field LBE (Eq. 33) is advanced; u is prescribed (clipo_set_u), f stays 0:
                              the set-up of the interface-in-shear-flow test, PAPER.md:675-713 (Sec. 5.4) */
  int outlet_clamp;        /* 0: lambda = U dt/dy exactly as B.25 prints it; 1: lambda = max(0, U) -- B.21 is an
                              OUTFLOW condition; for U < 0 the implicit upwind form B.23-B.25 amplifies chi(N) - chi(N-1) by
                              1/(1 + lambda) > 1 per step (pinned), the clamp replaces that by chi(N,t+dt) = chi(N,t) [R12] */
  int outlet_u_time;       /* which U enters lambda [R12]: 0: the stored macroscopic u_z(x,y,N-1,t) ("computed based on the
                              distribution function from the previous time step"); 1: the first moment
                              sum_a e_az f_a(x,y,N-1,t+dt) of the post-stream populations ("lambda = U(t+dt) dt/dy, determined after
                              the streaming step in the (N-1)th layer"), without the half-force term (F needs
                              grad phi(t+dt), which involves the outlet layer itself) */
  int macro_u_refine;      /* ORACLE ONLY, sensitivity of reading R13 (Alg. 3 evaluates F_mu with the velocity of the PREVIOUS step,
                              PAPER.md:501, before u is updated): 0: as printed (lagged u, one evaluation); 1: one fixed-point refinement,
                              F is evaluated again with the u just obtained and u = sum f e + F / 2 rho is redone */
  int open_ghost;          /* ORACLE ONLY, sensitivity of reading R9 at the OPEN parts of the z faces (inlet disc, outlet): 0: clamp
                              (zero gradient, the reading the product takes); 1: linear extrapolation phi(-1) = 2 phi(0) - phi(1);
                              the plate around the nozzle is a wall and keeps the mirror value */
} clipo_params;

typedef struct clipo {
  int nx, ny, nz;
  size_t n;
  clipo_params p;
  double w[Q];
  double Mm[Q][Q], Minv[Q][Q]; /* weighted-orthogonal moment basis [G2, G2b] */
  double *f, *g, *f2, *g2;     /* [n][Q]; f,g hold the pre-collision populations at the current time */
  double *fp, *gp;             /* post-collision scratch */
  double *phi, *ux, *uy, *uz, *pstar;
  long t;
} clipo;

/* ---------------------------------------------------------------- basis: weighted Gram-Schmidt [G2b] ------ */
static void build_basis(clipo *h) {
  double poly[Q][Q];
  for (int a = 0; a < Q; ++a) {
    double x = EX[a], y = EY[a], z = EZ[a], e2 = x * x + y * y + z * z;
#ifdef CLIPO_D2Q9
    (void)z; /* 9 polynomials of rank 9 on D2Q9; rows 3, 4 = the traceless second-order moments [G2 in two dimensions] */
    poly[0][a] = 1.0; poly[1][a] = x; poly[2][a] = y;
    poly[3][a] = x * y; poly[4][a] = x * x - y * y;
    poly[5][a] = e2; poly[6][a] = x * e2; poly[7][a] = y * e2; poly[8][a] = e2 * e2;
#else
    poly[0][a] = 1.0;
    poly[1][a] = x; poly[2][a] = y; poly[3][a] = z;
    poly[4][a] = x * y; poly[5][a] = y * z; poly[6][a] = x * z;          /* the 5 traceless 2nd-order moments */
    poly[7][a] = x * x - y * y; poly[8][a] = x * x + y * y - 2.0 * z * z;
    poly[9][a] = e2;
    poly[10][a] = e2 * e2;
    poly[11][a] = x * e2; poly[12][a] = y * e2; poly[13][a] = z * e2;
    poly[14][a] = (x * x - y * y) * e2; poly[15][a] = (x * x + y * y - 2.0 * z * z) * e2;
    poly[16][a] = x * (y * y - z * z); poly[17][a] = y * (z * z - x * x); poly[18][a] = z * (x * x - y * y);
#endif
  }
  for (int k = 0; k < Q; ++k) {
    double v[Q];
    for (int a = 0; a < Q; ++a) v[a] = poly[k][a];
    for (int pass = 0; pass < 2; ++pass) /* re-orthogonalise once for round-off */
      for (int j = 0; j < k; ++j) {
        double num = 0.0, den = 0.0;
        for (int a = 0; a < Q; ++a) { num += h->w[a] * v[a] * h->Mm[j][a]; den += h->w[a] * h->Mm[j][a] * h->Mm[j][a]; }
        for (int a = 0; a < Q; ++a) v[a] -= num / den * h->Mm[j][a];
      }
    for (int a = 0; a < Q; ++a) h->Mm[k][a] = v[a];
  }
  /* M W M^T is diagonal => M^-1 = W M^T (M W M^T)^-1 */
  for (int k = 0; k < Q; ++k) {
    double d = 0.0;
    for (int a = 0; a < Q; ++a) d += h->w[a] * h->Mm[k][a] * h->Mm[k][a];
    for (int a = 0; a < Q; ++a) h->Minv[a][k] = h->w[a] * h->Mm[k][a] / d;
  }
}

/* S-hat of Eq. 28 read as: rate s_nu on the 5 traceless second-order moments (rows 4..8), rate 1
 * on the others [G2] (D2Q9: the 2 traceless second-order moments, the other 7 at rate 1). */
static double S_of(int k, double s_nu) { return (k >= SHEAR_LO && k <= SHEAR_HI) ? s_nu : 1.0; }

/* Collision operator applied to r = f - feq_bar (or f - feq in the viscous force):
 * WMRT: M^-1 S M r (Eq. 27);  BGK: r / (tau + 1/2) (Eq. 26; the same factor multiplies the stress in Eq. 29). */
static void apply_MSM(const clipo *h, double s_nu, const double *r, double *out);
static void apply_collision(const clipo *h, double s_nu, const double *r, double *out) {
  if (h->p.collision == 1) { for (int a = 0; a < Q; ++a) out[a] = s_nu * r[a]; }
  else apply_MSM(h, s_nu, r, out);
}

/* out = M^-1 S M r  (Eq. 27) */
static void apply_MSM(const clipo *h, double s_nu, const double *r, double *out) {
  double m[Q];
  for (int k = 0; k < Q; ++k) {
    double s = 0.0;
    for (int a = 0; a < Q; ++a) s += h->Mm[k][a] * r[a];
    m[k] = S_of(k, s_nu) * s;
  }
  for (int a = 0; a < Q; ++a) {
    double s = 0.0;
    for (int k = 0; k < Q; ++k) s += h->Minv[a][k] * m[k];
    out[a] = s;
  }
}

/* ---------------------------------------------------------------- geometry helpers ----------------------- */
static size_t IDX(const clipo *h, int x, int y, int z) { return (size_t)x + (size_t)h->nx * ((size_t)y + (size_t)h->ny * (size_t)z); }

/* phi ghost rule: PERIODIC -> wrap (B.7); other faces -> clamp [R9] */
static int ghost(int i, int n, int bc_lo, int bc_hi) {
  if (i < 0) return bc_lo == BC_PERIODIC ? i + n : 0;
  if (i >= n) return bc_hi == BC_PERIODIC ? i - n : n - 1;
  return i;
}
static int in_disc(const clipo *h, int x, int y);
static int is_open(int bc) { return bc == BC_INLET || bc == BC_OUTLET; }
static double phi_at(const clipo *h, const double *phi, int x, int y, int z) {
  x = ghost(x, h->nx, h->p.bc[0], h->p.bc[1]);
  y = ghost(y, h->ny, h->p.bc[2], h->p.bc[3]);
  if (h->p.open_ghost == 1 && h->nz >= 2) { /* sensitivity variant of [R9]: linear extrapolation through open z faces */
    if (z < 0 && is_open(h->p.bc[4]) && (h->p.bc[4] != BC_INLET || in_disc(h, x, y))) return 2.0 * phi[IDX(h, x, y, 0)] - phi[IDX(h, x, y, 1)];
    if (z >= h->nz && is_open(h->p.bc[5])) return 2.0 * phi[IDX(h, x, y, h->nz - 1)] - phi[IDX(h, x, y, h->nz - 2)];
  }
  z = ghost(z, h->nz, h->p.bc[4], h->p.bc[5]);
  return phi[IDX(h, x, y, z)];
}
static int in_disc(const clipo *h, int x, int y) {
  double dx = x - h->p.inlet_c[0], dy = y - h->p.inlet_c[1];
  return dx * dx + dy * dy <= h->p.inlet_r * h->p.inlet_r;
}
static int is_inlet_node(const clipo *h, int x, int y, int z) {
  return h->p.bc[4] == BC_INLET && z == 0 && in_disc(h, x, y);
}

/* ---------------------------------------------------------------- per-node pieces ------------------------ */
/* Eq. 40a/b: isotropic gradient (pairwise differences, identical to Eq. 40a because
 * sum_a w_a e_a = 0) and Laplacian as printed. */
static void stencils(const clipo *h, const double *phi, int x, int y, int z, double G[3], double *L) {
  double gx = 0, gy = 0, gz = 0, lap = 0;
  double pc = phi[IDX(h, x, y, z)];
  for (int a = 1; a < Q; a += 2) { /* pairs (a, a+1) are opposite */
    double pp = phi_at(h, phi, x + EX[a], y + EY[a], z + EZ[a]);
    double pm = phi_at(h, phi, x - EX[a], y - EY[a], z - EZ[a]);
    double d = h->w[a] * (pp - pm);
    gx += EX[a] * d; gy += EY[a] * d; gz += EZ[a] * d;
  }
  for (int a = 1; a < Q; ++a) lap += h->w[a] * (phi_at(h, phi, x + EX[a], y + EY[a], z + EZ[a]) - pc);
  G[0] = 3.0 * gx; G[1] = 3.0 * gy; G[2] = 3.0 * gz; /* c/(c_s^2 dx) = 3 */
  *L = 6.0 * lap;                                     /* 2c^2/(c_s^2 dx^2) = 6 */
}

static double tau_of(const clipo *h, double phi) {
  if (h->p.visc_interp == 1) return 1.0 / (1.0 / h->p.tau_l + phi * (1.0 / h->p.tau_h - 1.0 / h->p.tau_l));
  if (h->p.visc_interp == 2) { /* Eq. 25 with mu_X = rho_X tau_X c_s^2 (Eq. 23), phi_L = 0; then tau = mu / (rho c_s^2) */
    const double mu_l = h->p.rho_l * h->p.tau_l / 3.0, mu_h = h->p.rho_h * h->p.tau_h / 3.0;
    const double mu = mu_l + phi * (mu_h - mu_l);
    return 3.0 * mu / (h->p.rho_l + phi * (h->p.rho_h - h->p.rho_l));
  }
  return h->p.tau_l + phi * (h->p.tau_h - h->p.tau_l); /* Eq. 24, phi_L = 0 */
}
static double rho_of(const clipo *h, double phi) { return h->p.rho_l + phi * (h->p.rho_h - h->p.rho_l); } /* Eq. 39 */

/* Eq. 11 with the corrected sign [G4]; beta, kappa from Eq. 12 */
static double mu_phi_of(const clipo *h, double phi, double L) {
  double beta = 12.0 * h->p.sigma / h->p.W, kappa = 1.5 * h->p.sigma * h->p.W;
  return 4.0 * beta * phi * (phi - 1.0) * (phi - 0.5) - kappa * L;
}

/* Eq. 18 */
static double Gamma(const clipo *h, int a, double ux, double uy, double uz) {
  double eu = EX[a] * ux + EY[a] * uy + EZ[a] * uz;
  return h->w[a] * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * (ux * ux + uy * uy + uz * uz));
}

/* Total force, Eq. 20, from f (pre-collision), p*, u, and the phi stencils at the node.
 * F_mu: Eq. 30 with nu/(c_s^2 dt) = tau (Eq. 23) and grad rho = (rho_h - rho_l) grad phi (Eq. 32);
 * F_p: Eq. 21;  F_s: Eq. 10;  F_b = (rho - rho_ref) g [G16]. */
static void total_force(const clipo *h, const double *f, double pstar, double ux, double uy, double uz,
                        double phi, const double G[3], double L, double F[3]) {
  double rho = rho_of(h, phi), tau = tau_of(h, phi), s_nu = 1.0 / (tau + 0.5); /* [G3] */
  double drho = h->p.rho_h - h->p.rho_l;
  double r[Q], t[Q];
  for (int a = 0; a < Q; ++a) r[a] = f[a] - (pstar * h->w[a] + (Gamma(h, a, ux, uy, uz) - h->w[a])); /* f - feq, Eq. 17 */
  apply_collision(h, s_nu, r, t);
  double Pi[3][3] = {{0}};
  for (int b = 0; b < Q; ++b) {
    double e[3] = {(double)EX[b], (double)EY[b], (double)EZ[b]};
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Pi[i][j] += e[i] * e[j] * t[b];
  }
  double mu = mu_phi_of(h, phi, L);
  for (int i = 0; i < 3; ++i) {
    double Fmu = 0.0;
    for (int j = 0; j < 3; ++j) Fmu += Pi[i][j] * drho * G[j];
    Fmu *= -tau;
    double Fp = -pstar * (1.0 / 3.0) * drho * G[i];
    double Fs = mu * G[i];
    double Fb = (rho - h->p.rho_ref) * h->p.g[i];
    F[i] = Fs + Fb + Fp + Fmu;
  }
}

/* Barred equilibria and forcing terms of one node state -- the lines the collision executes (also exported for pin P12):
 * F_a Eq. 19, feq Eq. 17, feq_bar Eq. 16; F^phi_a Eq. 34, geq = phi Gamma_a Eq. 36, geq_bar Eq. 35. */
static void node_terms(const clipo *h, double pstar, const double *u, double phi, const double *F, const double *nvec,
                       double *feqbar, double *Fa, double *geqbar, double *Fphi) {
  double rho = rho_of(h, phi);
  double pref = (1.0 - 4.0 * (phi - 0.5) * (phi - 0.5)) / h->p.W;
  for (int a = 0; a < Q; ++a) {
    double Gam = Gamma(h, a, u[0], u[1], u[2]);
    Fa[a] = h->w[a] * (EX[a] * F[0] + EY[a] * F[1] + EZ[a] * F[2]) / (rho * (1.0 / 3.0));   /* Eq. 19 */
    feqbar[a] = pstar * h->w[a] + (Gam - h->w[a]) - 0.5 * Fa[a];                           /* Eq. 16-17 */
    Fphi[a] = pref * h->w[a] * (EX[a] * nvec[0] + EY[a] * nvec[1] + EZ[a] * nvec[2]);       /* Eq. 34 */
    geqbar[a] = phi * Gam - 0.5 * Fphi[a];                                                 /* Eq. 35-36 */
  }
}

/* Steps 1-6 of SURVEY 8(c) for one node: Alg. 1.  fin/gin pre-collision, fout/gout post. */
static void collide_node(const clipo *h, const double *phi_field, int x, int y, int z, const double *fin,
                         const double *gin, double ux, double uy, double uz, double *fout, double *gout) {
  double phi = phi_field[IDX(h, x, y, z)];
  double G[3], L, F[3] = {0.0, 0.0, 0.0};
  stencils(h, phi_field, x, y, z, G, &L);
  double pstar = 0.0;
  for (int a = 0; a < Q; ++a) pstar += fin[a]; /* Eq. 31a */
  if (!h->p.phase_only) total_force(h, fin, pstar, ux, uy, uz, phi, G, L, F);
  double nrm = sqrt(G[0] * G[0] + G[1] * G[1] + G[2] * G[2]) + 1e-32; /* [R10] */
  double u[3] = {ux, uy, uz}, nvec[3] = {G[0] / nrm, G[1] / nrm, G[2] / nrm};
  double feqbar[Q], Fa[Q], geqbar[Q], Fphi[Q];
  node_terms(h, pstar, u, phi, F, nvec, feqbar, Fa, geqbar, Fphi);
  if (h->p.phase_only) { /* prescribed u: the hydrodynamic populations are not advanced */
    for (int a = 0; a < Q; ++a) fout[a] = fin[a];
  } else { /* hydrodynamic collision: Eq. 13 with Eq. 27 (or Eq. 26) */
    double tau = tau_of(h, phi), s_nu = 1.0 / (tau + 0.5);
    double r[Q], t[Q];
    for (int a = 0; a < Q; ++a) r[a] = fin[a] - feqbar[a];
    apply_collision(h, s_nu, r, t);
    for (int a = 0; a < Q; ++a) fout[a] = fin[a] - t[a] + Fa[a];
  }
  /* phase-field collision: Eq. 33, tau_phi = M / c_s^2 (Eq. 37) */
  double tau_phi = 3.0 * h->p.M, om = 1.0 / (tau_phi + 0.5);
  for (int a = 0; a < Q; ++a) gout[a] = gin[a] - om * (gin[a] - geqbar[a]) + Fphi[a];
}

/* Velocity inlet on one node, App. B.4 as read in [G6]: inward normal +z, unknown set =
 * the 5 directions with e_z = +1; f' = f (F = 0 at the inlet). */
static void inlet_node(const clipo *h, double *f, double *g) {
  const double *u = h->p.inlet_u;
  double phin = h->p.inlet_phi;
  /* B.14 with sum_{a in Lambda} e_a feq_a = (2/3) u_t in closed form */
  double Mt[3] = {0, 0, 0};
  for (int a = 0; a < Q; ++a) if (EZ[a] == 0) { Mt[0] += EX[a] * f[a]; Mt[1] += EY[a] * f[a]; }
  Mt[0] -= (2.0 / 3.0) * u[0]; Mt[1] -= (2.0 / 3.0) * u[1];
  double theta = 0.0; /* B.18 */
  for (int a = 0; a < Q; ++a) if (EZ[a] == 0) theta += g[a] - phin * Gamma(h, a, u[0], u[1], u[2]);
  for (int a = 0; a < Q; ++a) if (EZ[a] == 1) {
    int b = opp(a);
    double eu = EX[a] * u[0] + EY[a] * u[1] + EZ[a] * u[2];
    f[a] = f[b] + 6.0 * h->w[a] * eu - 0.5 * (EX[a] * Mt[0] + EY[a] * Mt[1]);           /* B.15, N -> 2 per axis */
    double geq_a = phin * Gamma(h, a, u[0], u[1], u[2]);
    double gneq_b = g[b] - phin * Gamma(h, b, u[0], u[1], u[2]);
    g[a] = geq_a - gneq_b - ((EX[a] != 0 || EY[a] != 0) ? theta / 4.0 : 0.0);            /* B.19-B.20 */
  }
}

/* Step 10 of SURVEY 8(c): Alg. 3 on the whole lattice; f,g are the new pre-collision sets. */
static void macros(clipo *h) {
  for (int z = 0; z < h->nz; ++z) for (int y = 0; y < h->ny; ++y) for (int x = 0; x < h->nx; ++x) {
    size_t i = IDX(h, x, y, z);
    double s = 0.0;
    for (int a = 0; a < Q; ++a) s += h->g[i * Q + a]; /* Eq. 38 */
    h->phi[i] = is_inlet_node(h, x, y, z) ? h->p.inlet_phi : s;
  }
  if (h->p.phase_only) return; /* u stays as prescribed, p* = 0 */
  for (int z = 0; z < h->nz; ++z) for (int y = 0; y < h->ny; ++y) for (int x = 0; x < h->nx; ++x) {
    size_t i = IDX(h, x, y, z);
    const double *f = h->f + i * Q;
    double pstar = 0.0;
    for (int a = 0; a < Q; ++a) pstar += f[a]; /* Eq. 31a, before u */
    h->pstar[i] = pstar;
    double G[3], L, F[3];
    stencils(h, h->phi, x, y, z, G, &L);
    total_force(h, f, pstar, h->ux[i], h->uy[i], h->uz[i], h->phi[i], G, L, F); /* lagged u [R13] */
    double rho = rho_of(h, h->phi[i]);
    double mx = 0, my = 0, mz = 0;
    for (int a = 0; a < Q; ++a) { mx += f[a] * EX[a]; my += f[a] * EY[a]; mz += f[a] * EZ[a]; }
    if (is_inlet_node(h, x, y, z)) {
      h->ux[i] = h->p.inlet_u[0]; h->uy[i] = h->p.inlet_u[1]; h->uz[i] = h->p.inlet_u[2];
    } else { /* Eq. 31b */
      h->ux[i] = mx + 0.5 * F[0] / rho; h->uy[i] = my + 0.5 * F[1] / rho; h->uz[i] = mz + 0.5 * F[2] / rho;
      if (h->p.macro_u_refine == 1) { /* sensitivity variant of [R13] */
        total_force(h, f, pstar, h->ux[i], h->uy[i], h->uz[i], h->phi[i], G, L, F);
        h->ux[i] = mx + 0.5 * F[0] / rho; h->uy[i] = my + 0.5 * F[1] / rho; h->uz[i] = mz + 0.5 * F[2] / rho;
      }
    }
  }
}

/* ---------------------------------------------------------------- C ABI ---------------------------------- */
clipo *clipo_create(int nx, int ny, int nz, const clipo_params *p) {
  if (nx < 1 || ny < 1 || nz < 1 || !p) return NULL;
#ifdef CLIPO_D2Q9
  if (nz != 1 || p->bc[4] != BC_PERIODIC || p->bc[5] != BC_PERIODIC) return NULL; /* 2-D: one plane, nothing happens in z */
  for (int k = 0; k < 4; ++k) if (p->bc[k] == BC_INLET || p->bc[k] == BC_OUTLET) return NULL;
#endif
  clipo *h = (clipo *)calloc(1, sizeof(clipo));
  h->nx = nx; h->ny = ny; h->nz = nz; h->n = (size_t)nx * ny * nz; h->p = *p;
  for (int a = 0; a < Q; ++a) h->w[a] = weight_of(a);
  build_basis(h);
  size_t nq = h->n * Q;
  h->f = calloc(nq, 8); h->g = calloc(nq, 8); h->f2 = calloc(nq, 8); h->g2 = calloc(nq, 8);
  h->fp = calloc(nq, 8); h->gp = calloc(nq, 8);
  h->phi = calloc(h->n, 8); h->ux = calloc(h->n, 8); h->uy = calloc(h->n, 8); h->uz = calloc(h->n, 8);
  h->pstar = calloc(h->n, 8);
  return h;
}

void clipo_destroy(clipo *h) {
  if (!h) return;
  free(h->f); free(h->g); free(h->f2); free(h->g2); free(h->fp); free(h->gp);
  free(h->phi); free(h->ux); free(h->uy); free(h->uz); free(h->pstar); free(h);
}

/* Init I1-I4 [R8]: phi = phi0, u = u0, p* = 0; F = F_s + F_b; g = phi Gamma - F^phi/2, f = (Gamma - w) - F_a/2 */
int clipo_init(clipo *h, const double *phi0, const double *u0) {
  size_t n = h->n;
  memcpy(h->phi, phi0, n * 8);
  memcpy(h->ux, u0, n * 8); memcpy(h->uy, u0 + n, n * 8); memcpy(h->uz, u0 + 2 * n, n * 8);
  for (int z = 0; z < h->nz; ++z) for (int y = 0; y < h->ny; ++y) for (int x = 0; x < h->nx; ++x) {
    size_t i = IDX(h, x, y, z);
    double phi = h->phi[i], G[3], L;
    stencils(h, h->phi, x, y, z, G, &L);
    double rho = rho_of(h, phi), mu = mu_phi_of(h, phi, L);
    double F[3];
    for (int k = 0; k < 3; ++k) F[k] = mu * G[k] + (rho - h->p.rho_ref) * h->p.g[k];
    double nrm = sqrt(G[0] * G[0] + G[1] * G[1] + G[2] * G[2]) + 1e-32;
    double pref = (1.0 - 4.0 * (phi - 0.5) * (phi - 0.5)) / h->p.W;
    for (int a = 0; a < Q; ++a) {
      double Gam = Gamma(h, a, h->ux[i], h->uy[i], h->uz[i]);
      double Fphi = pref * h->w[a] * (EX[a] * G[0] / nrm + EY[a] * G[1] / nrm + EZ[a] * G[2] / nrm);
      double Fa = h->w[a] * (EX[a] * F[0] + EY[a] * F[1] + EZ[a] * F[2]) / (rho * (1.0 / 3.0));
      h->g[i * Q + a] = phi * Gam - 0.5 * Fphi;
      h->f[i * Q + a] = h->p.phase_only ? 0.0 : (Gam - h->w[a]) - 0.5 * Fa;
    }
    h->pstar[i] = 0.0;
  }
  h->t = 0;
  return 0;
}

static void step_once(clipo *h) {
  const int nx = h->nx, ny = h->ny, nz = h->nz;
  const int *bc = h->p.bc;
  /* steps 1-6: collision on every node */
  for (int z = 0; z < nz; ++z) for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
    size_t i = IDX(h, x, y, z);
    collide_node(h, h->phi, x, y, z, h->f + i * Q, h->g + i * Q, h->ux[i], h->uy[i], h->uz[i], h->fp + i * Q, h->gp + i * Q);
  }
  /* step 7: streaming (B.3-B.6) with halfway bounce-back (B.10-B.11) and free-slip (B.8-B.9) into the second buffer.
   * Free-slip: a population that leaves node x_b through a free-slip face comes back with its wall-normal
   * velocity component reversed and the tangential ones kept, and lands on x_b + e_tangential.  Pull form: the population
   * a arriving at x whose upstream node x - e_a lies behind a free-slip face in dimension d was sent, as direction a' = a
   * with component d reversed, by the node that has x's coordinate in d and the upstream coordinates in the other dimensions. */
  for (int z = 0; z < nz; ++z) for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
    size_t i = IDX(h, x, y, z);
    for (int a = 0; a < Q; ++a) {
      int sx = x - EX[a], sy = y - EY[a], sz = z - EZ[a];
      int bounce = 0, open = 0;
      int s[3] = {sx, sy, sz}, nn[3] = {nx, ny, nz}, here[3] = {x, y, z}, e[3] = {EX[a], EY[a], EZ[a]};
      for (int d = 0; d < 3; ++d) {
        int face = -1;
        if (s[d] < 0) face = 2 * d; else if (s[d] >= nn[d]) face = 2 * d + 1;
        if (face < 0) continue;
        int type = bc[face];
        if (type == BC_PERIODIC) s[d] += (s[d] < 0) ? nn[d] : -nn[d];
        else if (type == BC_WALL) bounce = 1;
        else if (type == BC_FREESLIP) { s[d] = here[d]; e[d] = -e[d]; }
        else if (type == BC_INLET) { if (in_disc(h, x, y)) open = 1; else bounce = 1; }
        else open = 1; /* OUTLET: the destination layer is overwritten in step 9 */
      }
      if (bounce) { /* a no-slip wall crossing wins at edges / corners [R11] */
        h->f2[i * Q + a] = h->fp[i * Q + opp(a)];
        h->g2[i * Q + a] = h->gp[i * Q + opp(a)];
      } else if (open) { /* unknown: filled by step 8 or 9; keep a defined value */
        h->f2[i * Q + a] = 0.0; h->g2[i * Q + a] = 0.0;
      } else {
        int as = a;
        if (e[0] != EX[a] || e[1] != EY[a] || e[2] != EZ[a]) {
          as = -1;
          for (int b = 0; b < Q; ++b) if (EX[b] == e[0] && EY[b] == e[1] && EZ[b] == e[2]) as = b;
        }
        size_t j = IDX(h, s[0], s[1], s[2]);
        h->f2[i * Q + a] = h->fp[j * Q + as];
        h->g2[i * Q + a] = h->gp[j * Q + as];
      }
    }
  }
  /* step 8: velocity inlet on the disc of the -z face */
  if (bc[4] == BC_INLET)
    for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) if (in_disc(h, x, y)) {
      size_t i = IDX(h, x, y, 0);
      inlet_node(h, h->f2 + i * Q, h->g2 + i * Q);
    }
  /* step 9: convective outlet on layer N = nz-1 (B.26-B.27); lambda = U dt/dy with U one of
   * the three schemes of B.22 built on the normal velocity of layer N-1 [R12: outlet_u_time, outlet_clamp] */
  if (bc[5] == BC_OUTLET) {
    double *Ucol = (double *)malloc((size_t)nx * ny * sizeof(double));
    double usum = 0.0, umax = 0.0;
    for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
      size_t iM = IDX(h, x, y, nz - 2);
      double v;
      if (h->p.outlet_u_time == 1 && !h->p.phase_only) { /* first moment of the post-stream f of layer N-1 at t+dt */
        v = 0.0;
        for (int a = 0; a < Q; ++a) v += EZ[a] * h->f2[iM * Q + a];
      } else v = h->uz[iM];                               /* stored macroscopic velocity of the previous time step */
      Ucol[(size_t)y * nx + x] = v;
      usum += v;
      if ((x == 0 && y == 0) || v > umax) umax = v;
    }
    double uplane = h->p.outlet_u_mode == 1 ? usum / ((double)nx * ny) : umax;
    for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
      size_t iN = IDX(h, x, y, nz - 1), iM = IDX(h, x, y, nz - 2);
      double U = h->p.outlet_u_mode == 0 ? Ucol[(size_t)y * nx + x] : uplane;
      double lam = (h->p.outlet_clamp && U < 0.0) ? 0.0 : U;
      for (int a = 0; a < Q; ++a) {
        h->f2[iN * Q + a] = (h->f[iN * Q + a] + lam * h->f2[iM * Q + a]) / (1.0 + lam);
        h->g2[iN * Q + a] = (h->g[iN * Q + a] + lam * h->g2[iM * Q + a]) / (1.0 + lam);
      }
    }
    free(Ucol);
  }
  double *tf = h->f; h->f = h->f2; h->f2 = tf;
  double *tg = h->g; h->g = h->g2; h->g2 = tg;
  /* step 10 */
  macros(h);
  h->t += 1;
}

int clipo_step(clipo *h, int n) {
  if (h->p.bc[5] == BC_OUTLET && h->nz < 2) return -1;
  for (int k = 0; k < n; ++k) step_once(h);
  return 0;
}

/* Prescribe the velocity field used by the following collisions (phase_only mode; u = [3][n]). */
int clipo_set_u(clipo *h, const double *u) {
  size_t n = h->n;
  memcpy(h->ux, u, n * 8); memcpy(h->uy, u + n, n * 8); memcpy(h->uz, u + 2 * n, n * 8);
  return 0;
}

/* phi, p = p* rho c_s^2, u = [3][n]; any may be NULL */
int clipo_get(const clipo *h, double *phi, double *p, double *u) {
  size_t n = h->n;
  if (phi) memcpy(phi, h->phi, n * 8);
  if (p) for (size_t i = 0; i < n; ++i) p[i] = h->pstar[i] * rho_of(h, h->phi[i]) * (1.0 / 3.0);
  if (u) { memcpy(u, h->ux, n * 8); memcpy(u + n, h->uy, n * 8); memcpy(u + 2 * n, h->uz, n * 8); }
  return 0;
}

/* ------------------------------------------------------------- introspection hooks used only by the pins -- */
int clipo_get_populations(const clipo *h, double *f, double *g) { /* [n][19] */
  if (f) memcpy(f, h->f, h->n * Q * 8);
  if (g) memcpy(g, h->g, h->n * Q * 8);
  return 0;
}
int clipo_set_populations(clipo *h, const double *f, const double *g) {
  if (f) memcpy(h->f, f, h->n * Q * 8);
  if (g) memcpy(h->g, g, h->n * Q * 8);
  return 0;
}
void clipo_lattice(const clipo *h, int *ex, int *ey, int *ez, double *w) {
  for (int a = 0; a < Q; ++a) { ex[a] = EX[a]; ey[a] = EY[a]; ez[a] = EZ[a]; w[a] = h->w[a]; }
}
void clipo_basis(const clipo *h, double *M, double *Minv) { /* row-major 19x19 */
  for (int i = 0; i < Q; ++i) for (int j = 0; j < Q; ++j) { M[i * Q + j] = h->Mm[i][j]; Minv[i * Q + j] = h->Minv[i][j]; }
}
void clipo_collision_matrix(const clipo *h, double s_nu, double *A) { /* dense M^-1 S M, row-major */
  for (int b = 0; b < Q; ++b) {
    double e[Q] = {0}, col[Q];
    e[b] = 1.0;
    apply_MSM(h, s_nu, e, col);
    for (int a = 0; a < Q; ++a) A[a * Q + b] = col[a];
  }
}
/* stencils + chemical potential of an arbitrary field (P4, P11) */
void clipo_stencil_field(const clipo *h, const double *phi, double *G, double *L, double *mu) {
  size_t n = h->n;
  for (int z = 0; z < h->nz; ++z) for (int y = 0; y < h->ny; ++y) for (int x = 0; x < h->nx; ++x) {
    size_t i = IDX(h, x, y, z);
    double g3[3], l;
    stencils(h, phi, x, y, z, g3, &l);
    G[i] = g3[0]; G[n + i] = g3[1]; G[2 * n + i] = g3[2]; L[i] = l;
    mu[i] = mu_phi_of(h, phi[i], l);
  }
}
/* barred equilibria and forcing terms of one node state (P12): the very function collide_node calls */
void clipo_node_terms(const clipo *h, double pstar, const double *u, double phi, const double *F, const double *nvec,
                      double *feqbar, double *Fa, double *geqbar, double *Fphi) {
  node_terms(h, pstar, u, phi, F, nvec, feqbar, Fa, geqbar, Fphi);
}
/* inlet rule on a caller-provided node (P13) */
void clipo_inlet_node(const clipo *h, double *f, double *g) { inlet_node(h, f, g); }
/* total force of one node from caller-provided state (F_mu pin) */
void clipo_total_force(const clipo *h, const double *f, double pstar, const double *u, double phi, const double *G,
                       double L, double *F) {
  total_force(h, f, pstar, u[0], u[1], u[2], phi, G, L, F);
}
long clipo_time(const clipo *h) { return h->t; }
int clipo_q(void) { return Q; }
