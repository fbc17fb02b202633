/*
 * pasta_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, FP64 CPU statement of what the nuclear-pasta MD hot path computes
 * (arXiv:1412.8502, "Pasta Nucleosynthesis"; citations are PAPER.md line numbers).
 * It shares no code, header, table or constant generator with the CUDA library under
 * paper_1412_8502_b200/csrc/.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It is never tuned for speed: the
 * OpenMP pragma over targets exists only so that the timed baseline can use the host cores.
 *
 * Units: lengths fm, times fm/c, energies and T in MeV, velocities in c, forces MeV/fm.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form two-particle table P1, finite
 * differences P2, np extremum P3, two-body oscillation period P4, Newton's third law P5,
 * translation/permutation invariance P6, all-pairs vs cell-list P7, dt^2 energy error P8,
 * thermostat P9, scaling P10, ideal-gas <PE> P11, neighbour count P12, cells P13, FoF P14; the paper's own variants:
 * r_nuc (range split), coul_nocut (Coulomb at the nearest image without a cut-off), linear box-only expansion,
 * two-radius MST clusters, composition summary -- each by hand-built cases and invariants.
 * Parity unpinned: the paper's physics outputs (Table II, Figs. 3-9) -- unreachable run lengths.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct orc_params {
  double a, b, c, Lambda; /* Table I: 110, -26, 24 MeV, 1.25 fm^2 */
  double alpha;           /* alpha*hbar*c = 1.44 MeV fm (Eq. 1c) */
  double lambda;          /* screening length, fixed to 10 fm */
  double r_c;             /* single cut-off of the BASELINE configs (reading D1) */
  double mass;            /* M = 939 MeV */
  double r_nuc;           /* the paper's own range split: the nuclear (Gaussian) terms are "assumed
                             to be zero and not computed" beyond r_nuc = 11.5 fm, independently of the Coulomb
                             term.  <= 0 (default): no separate nuclear cut-off, every term lives inside r_c (D1) */
  double coul_nocut;      /* != 0: the paper's own Coulomb sum ("we do not use a cutoff radius for the
                             Coulomb potential ... each proton interacts with the nearest periodic image of every
                             other proton"): every proton pair interacts through its nearest image whatever the
                             distance (a cube of side L around the target, not a sphere); needs r_nuc > 0, which then
                             is the only cut-off of the nuclear terms.  0 (default): Coulomb lives inside r_c (D1) */
} orc_params;

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* Nearest periodic image of a separation component. */
static inline double nearest_image(double d, double L) { return d - L * round(d / L); }

/*
 * Pair potential V(r) and g(r) = -(1/r) dV/dr for one pair (Eq. 1a-c).
 *   u = exp(-r^2 / 2 Lambda);  V = a u^2 + B u,  B = b+c (nn, pp) or b-c (np)
 *   -(1/r) dV/dr = (2 a u^2 + B u) / Lambda
 *   pp adds E_c = alpha exp(-r/lambda)/r to V and E_c (1/r + 1/lambda)/r to g.
 * Reading D2: at r^2 == 0 between distinct particles the Gaussian terms are evaluated as
 * written (finite V, zero force because d = 0); the divergent Coulomb term is skipped.
 */
static inline void pair_terms(const orc_params* p, double r2, int pi, int pj, double* V, double* g) {
  double u = exp(-r2 / (2.0 * p->Lambda));
  double B = (pi == pj) ? (p->b + p->c) : (p->b - p->c);
  *V = p->a * u * u + B * u;
  *g = (2.0 * p->a * u * u + B * u) / p->Lambda;
  if (p->r_nuc > 0.0 && !(r2 < p->r_nuc * p->r_nuc)) { /* strict r < r_nuc, plain truncation */
    *V = 0.0;
    *g = 0.0;
  }
  if (pi && pj && r2 > 0.0) {
    double r = sqrt(r2);
    double Ec = p->alpha * exp(-r / p->lambda) / r;
    *V += Ec;
    *g += Ec * (1.0 / r + 1.0 / p->lambda) / r;
  }
}

/* V(r) and F(r) = -dV/dr of an isolated pair; used by the closed-form pins only. */
void orc_pair(const orc_params* p, double r, int pi, int pj, double* V, double* F) {
  double g;
  pair_terms(p, r * r, pi, pj, V, &g);
  *F = g * r;
}

/*
 * O1. Force and energy by definition: every ordered pair i != j, nearest image, strict
 * r^2 < r_c^2, no cell list, no Newton's-third-law shortcut.
 *   F[i] = sum_j g(r_ij) (x_i - x_j);  e[i] = 1/2 sum_j V(r_ij);  PE = sum_i e[i].
 * n_targets/targets: optional subset of targets (NULL = all), for bounded timing samples.
 * diag[0] = ordered in-range pairs, diag[1] = ordered pairs with |r2/rc2 - 1| < 1e-5,
 * diag[2] = sum |V| over those boundary pairs (D2 diagnosis of cut-off classification).
 */
void orc_forces(int64_t N, const double* x, const uint8_t* is_p, double L, const orc_params* p,
                int64_t n_targets, const int64_t* targets, double* F, double* e, double* PE,
                double* diag) {
  const double rc2 = p->r_c * p->r_c;
  const int64_t nt = targets ? n_targets : N;
  double pe = 0.0, npairs = 0.0, nbnd = 0.0, vbnd = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : pe, npairs, nbnd, vbnd)
  for (int64_t t = 0; t < nt; ++t) {
    const int64_t i = targets ? targets[t] : t;
    double fx = 0.0, fy = 0.0, fz = 0.0, ei = 0.0;
    for (int64_t j = 0; j < N; ++j) {
      if (j == i) continue;
      double dx = nearest_image(x[3 * i + 0] - x[3 * j + 0], L);
      double dy = nearest_image(x[3 * i + 1] - x[3 * j + 1], L);
      double dz = nearest_image(x[3 * i + 2] - x[3 * j + 2], L);
      double r2 = dx * dx + dy * dy + dz * dz;
      if (r2 < rc2 || (p->coul_nocut != 0.0 && is_p[i] && is_p[j])) {
        double V, g;
        pair_terms(p, r2, is_p[i], is_p[j], &V, &g); /* beyond r_c >= r_nuc only the Coulomb term is left */
        fx += g * dx;
        fy += g * dy;
        fz += g * dz;
        ei += 0.5 * V;
        npairs += 1.0;
        if (fabs(r2 / rc2 - 1.0) < 1e-5) {
          nbnd += 1.0;
          vbnd += fabs(V);
        }
      }
    }
    F[3 * t + 0] = fx;
    F[3 * t + 1] = fy;
    F[3 * t + 2] = fz;
    if (e) e[t] = ei;
    pe += ei;
  }
  if (PE) *PE = pe;
  if (diag) {
    diag[0] = npairs;
    diag[1] = nbnd;
    diag[2] = vbnd;
  }
}

/* Position wrap of O2 step 2: x <- x - L floor(x/L); a result equal to L becomes 0. */
static inline double wrap_coord(double x, double L) {
  double w = x - L * floor(x / L);
  if (w >= L) w = 0.0;
  if (w < 0.0) w = 0.0;
  return w;
}
void orc_wrap(int64_t N, double* x, double L) {
  for (int64_t k = 0; k < 3 * N; ++k) x[k] = wrap_coord(x[k], L);
}

/*
 * O3. Cell grid (cubical cells, here of width >= r_c/k):
 *   ncell = max(1, floor(L k / r_c)); inv_w = ncell / L;
 *   c = min(ncell-1, (int)floor(x inv_w)) per axis (x already in [0,L));
 *   id = (cz ncell + cy) ncell + cx; cell_start = exclusive prefix sum of the histogram.
 */
int32_t orc_ncell(double L, double r_c, int32_t k) {
  double q = floor(L * (double)k / r_c);
  if (q < 1.0) q = 1.0;
  if (q > 2000.0) q = 2000.0;
  return (int32_t)q;
}
void orc_cells(int64_t N, const double* x, double L, int32_t ncell, int32_t* cell_id,
               int32_t* cell_start /* ncell^3 + 1 */) {
  const double inv_w = (double)ncell / L;
  const int64_t nc3 = (int64_t)ncell * ncell * ncell;
  memset(cell_start, 0, (size_t)(nc3 + 1) * sizeof(int32_t));
  for (int64_t i = 0; i < N; ++i) {
    int32_t c[3];
    for (int a = 0; a < 3; ++a) {
      int32_t q = (int32_t)floor(x[3 * i + a] * inv_w);
      if (q > ncell - 1) q = ncell - 1;
      if (q < 0) q = 0;
      c[a] = q;
    }
    cell_id[i] = (c[2] * ncell + c[1]) * ncell + c[0];
    cell_start[cell_id[i] + 1] += 1;
  }
  for (int64_t q = 0; q < nc3; ++q) cell_start[q + 1] += cell_start[q];
}

/*
 * O3 per axis: c = min(n-1, (int)floor(x (n / L))) for every coordinate of x (3N of them), the
 * statement inside orc_cells above written out on its own, so that a grid with different cell
 * counts per axis (the force path's thin cells along x: n = ncx for x, n = ncell for y, z) can be
 * checked without allocating an n^3 table (reading D14).
 */
void orc_cell_coords(int64_t N3, const double* x, double L, int32_t n, int32_t* c) {
  const double inv_w = (double)n / L;
  for (int64_t k = 0; k < N3; ++k) {
    int32_t q = (int32_t)floor(x[k] * inv_w);
    if (q > n - 1) q = n - 1;
    if (q < 0) q = 0;
    c[k] = q;
  }
}

/*
 * P7 helper: the same force definition evaluated through the O3 cell grid (own + 26
 * neighbour cells) -- an independent pair enumeration used to pin orc_forces
 * against itself on tiny N and as the labelled "list-based" second CPU baseline.
 * Needs ncell >= 3 and cell width >= r_c (k = 1); returns -1 otherwise.
 */
int orc_forces_cells(int64_t N, const double* x, const uint8_t* is_p, double L, const orc_params* p,
                     double* F, double* e, double* PE, double* npairs_out) {
  const int32_t nc = orc_ncell(L, p->r_c, 1);
  if (nc < 3) return -1;
  const int64_t nc3 = (int64_t)nc * nc * nc;
  int32_t* cid = (int32_t*)malloc((size_t)N * sizeof(int32_t));
  int32_t* start = (int32_t*)malloc((size_t)(nc3 + 1) * sizeof(int32_t));
  int32_t* fill = (int32_t*)malloc((size_t)nc3 * sizeof(int32_t));
  int32_t* order = (int32_t*)malloc((size_t)N * sizeof(int32_t));
  orc_cells(N, x, L, nc, cid, start);
  memcpy(fill, start, (size_t)nc3 * sizeof(int32_t));
  for (int64_t i = 0; i < N; ++i) order[fill[cid[i]]++] = (int32_t)i;
  const double rc2 = p->r_c * p->r_c;
  double pe = 0.0, npairs = 0.0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : pe, npairs)
  for (int64_t i = 0; i < N; ++i) {
    const int32_t cx = cid[i] % nc, cy = (cid[i] / nc) % nc, cz = cid[i] / (nc * nc);
    double fx = 0.0, fy = 0.0, fz = 0.0, ei = 0.0;
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          const int32_t q = (((cz + dz + nc) % nc) * nc + (cy + dy + nc) % nc) * nc + (cx + dx + nc) % nc;
          for (int32_t s = start[q]; s < start[q + 1]; ++s) {
            const int64_t j = order[s];
            if (j == i) continue;
            double ddx = nearest_image(x[3 * i + 0] - x[3 * j + 0], L);
            double ddy = nearest_image(x[3 * i + 1] - x[3 * j + 1], L);
            double ddz = nearest_image(x[3 * i + 2] - x[3 * j + 2], L);
            double r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            if (r2 < rc2) {
              double V, g;
              pair_terms(p, r2, is_p[i], is_p[j], &V, &g);
              fx += g * ddx;
              fy += g * ddy;
              fz += g * ddz;
              ei += 0.5 * V;
              npairs += 1.0;
            }
          }
        }
    F[3 * i + 0] = fx;
    F[3 * i + 1] = fy;
    F[3 * i + 2] = fz;
    if (e) e[i] = ei;
    pe += ei;
  }
  if (PE) *PE = pe;
  if (npairs_out) *npairs_out = npairs;
  free(cid);
  free(start);
  free(fill);
  free(order);
  return 0;
}

/* Kinetic energy sum 1/2 M |v|^2. */
double orc_kinetic(int64_t N, const double* v, double mass) {
  double ke = 0.0;
  for (int64_t k = 0; k < 3 * N; ++k) ke += 0.5 * mass * v[k] * v[k];
  return ke;
}

/*
 * O2. Velocity Verlet (ref. [31]) with the BASELINE variant of the box growth
 * (box AND positions scaled by s in the drift, reading D9/D10) and the isokinetic rescale
 * every `interval` steps (reading D7/D8).  F holds F(x) on entry and on exit.
 *   (1) v += (dt/2M) F   (2) x = s (x + dt v); L = s L; wrap   (3) F = O1(x, L)
 *   (4) v += (dt/2M) F   (5) count += 1; if interval > 0 and count % interval == 0 and KE > 0:
 *                            v *= sqrt(1.5 N T / KE)
 */
void orc_step(int64_t N, double* x, double* v, const uint8_t* is_p, double* L, const orc_params* p,
              double T, int32_t interval, double scale_per_step, double dt, int64_t nsteps,
              int64_t* step_count, double* F, double* PE) {
  const double h = dt / (2.0 * p->mass);
  for (int64_t s = 0; s < nsteps; ++s) {
    for (int64_t k = 0; k < 3 * N; ++k) v[k] += h * F[k];
    *L = scale_per_step * (*L);
    for (int64_t k = 0; k < 3 * N; ++k) x[k] = wrap_coord(scale_per_step * (x[k] + dt * v[k]), *L);
    orc_forces(N, x, is_p, *L, p, 0, NULL, F, NULL, PE, NULL);
    for (int64_t k = 0; k < 3 * N; ++k) v[k] += h * F[k];
    *step_count += 1;
    if (interval > 0 && (*step_count % interval) == 0) {
      double ke = orc_kinetic(N, v, p->mass);
      if (ke > 0.0) {
        double f = sqrt(1.5 * (double)N * T / ke);
        for (int64_t k = 0; k < 3 * N; ++k) v[k] *= f;
      }
    }
  }
}

/*
 * O2'. The paper's own expansion (Eq. 3a): the side of the box grows linearly in time,
 * l(t) = l(0) (1 + xi_dot t), and "particle positions and velocities are not incremented with the change in box
 * volume"; the thermostat is the same.  Reading D25: the box is enlarged right after the drift, before the force
 * evaluation (PAPER.md:100 says "after the timestep is completed"; like D10, one force evaluation then serves
 * the closing kick of this step and the opening kick of the next).  n_exp = steps since the expansion began
 * (in/out); L0 = the side at that moment; t = n_exp * dt with a constant dt.
 *   (1) v += (dt/2M) F   (2) x = wrap(x + dt v) in the CURRENT box   (3) n_exp += 1; L = L0 (1 + xi_dot dt n_exp)
 *   (4) F = O1(x, L)     (5) v += (dt/2M) F   (6) thermostat as in O2
 */
void orc_step_linear(int64_t N, double* x, double* v, const uint8_t* is_p, double L0, double xi_dot,
                     int64_t* n_exp, double* L, const orc_params* p, double T, int32_t interval, double dt,
                     int64_t nsteps, int64_t* step_count, double* F, double* PE) {
  const double h = dt / (2.0 * p->mass);
  for (int64_t s = 0; s < nsteps; ++s) {
    for (int64_t k = 0; k < 3 * N; ++k) v[k] += h * F[k];
    for (int64_t k = 0; k < 3 * N; ++k) x[k] = wrap_coord(x[k] + dt * v[k], *L);
    *n_exp += 1;
    *L = L0 * (1.0 + xi_dot * (dt * (double)(*n_exp)));
    orc_forces(N, x, is_p, *L, p, 0, NULL, F, NULL, PE, NULL);
    for (int64_t k = 0; k < 3 * N; ++k) v[k] += h * F[k];
    *step_count += 1;
    if (interval > 0 && (*step_count % interval) == 0) {
      double ke = orc_kinetic(N, v, p->mass);
      if (ke > 0.0) {
        double f = sqrt(1.5 * (double)N * T / ke);
        for (int64_t k = 0; k < 3 * N; ++k) v[k] *= f;
      }
    }
  }
}

/* One-shot uniform scaling (pasta_expand): L *= s, x *= s, v untouched (reading D9). */
void orc_expand(int64_t N, double* x, double* L, double s) {
  *L = (*L) * s;
  for (int64_t k = 0; k < 3 * N; ++k) x[k] = wrap_coord(x[k] * s, *L);
}

/*
 * O4 link predicate, pinned (reading D13): FP64, every operation a separately rounded IEEE
 * operation in this order (compile with -ffp-contract=off):
 *   d = x_i - x_j;  d = d - L * rint(d * (1/L));  r2 = (dx dx + dy dy) + dz dz;  r2 <= r_cl^2
 */
static inline int linked(const double* xi, const double* xj, double L, double invL, double rcl2) {
  double dx = xi[0] - xj[0], dy = xi[1] - xj[1], dz = xi[2] - xj[2];
  dx = dx - L * rint(dx * invL);
  dy = dy - L * rint(dy * invL);
  dz = dz - L * rint(dz * invL);
  double r2 = (dx * dx + dy * dy) + dz * dz;
  return r2 <= rcl2;
}
static int64_t uf_find(int64_t* parent, int64_t i) {
  while (parent[i] != i) {
    parent[i] = parent[parent[i]];
    i = parent[i];
  }
  return i;
}
static void uf_union(int64_t* parent, int64_t a, int64_t b) {
  a = uf_find(parent, a);
  b = uf_find(parent, b);
  if (a == b) return;
  if (a < b) parent[b] = a; else parent[a] = b; /* root = smallest index of the component */
}
static void finish_labels(int64_t N, int64_t* parent, const uint8_t* is_p, int32_t* label,
                          int32_t* A, int32_t* Z, int64_t* n_clusters) {
  int64_t nc = 0;
  for (int64_t i = 0; i < N; ++i) { A[i] = 0; Z[i] = 0; }
  for (int64_t i = 0; i < N; ++i) {
    int64_t r = uf_find(parent, i);
    label[i] = (int32_t)r;
    A[r] += 1;
    Z[r] += is_p[i] ? 1 : 0;
    if (r == i) nc += 1;
  }
  if (n_clusters) *n_clusters = nc;
}

/*
 * O4. Friends-of-friends clusters (BASELINE variant of PAPER.md:154-158, reading D13): the
 * connected components of {(i,j): r_ij <= r_cl} over ALL nucleons, by brute force over i < j.
 * label[i] = smallest member index; A[r], Z[r] = mass and charge number of the cluster whose
 * label is r (0 elsewhere).
 */
void orc_clusters(int64_t N, const double* x, const uint8_t* is_p, double L, double r_cl,
                  int32_t* label, int32_t* A, int32_t* Z, int64_t* n_clusters) {
  int64_t* parent = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  const double invL = 1.0 / L, rcl2 = r_cl * r_cl;
  for (int64_t i = 0; i < N; ++i) parent[i] = i;
  for (int64_t i = 0; i < N; ++i)
    for (int64_t j = i + 1; j < N; ++j)
      if (linked(x + 3 * i, x + 3 * j, L, invL, rcl2)) uf_union(parent, i, j);
  finish_labels(N, parent, is_p, label, A, Z, n_clusters);
  free(parent);
}

/*
 * O4'. The paper's own "MST" cluster algorithm, brute force:
 *   (1) protons i, j belong to the same cluster if r_ij <= r_pp (4.5 fm), transitively; a proton with no
 *       proton in range is its own cluster;
 *   (2) a neutron is counted as a member of cluster C "if it is within a distance r_np [3 fm] of at least one
 *       proton j that also belongs to C"; neutrons in no cluster are free (a cluster of their own, A = 1, Z = 0).
 * Reading D24 (the paper is silent on a neutron within r_np of protons of two clusters): it joins the cluster of
 * its NEAREST proton (smallest pinned r2; equal r2: the smaller proton index).  Nearest periodic images
 * throughout, same pinned distance arithmetic as `linked`.  label[i] = smallest PROTON index of
 * i's cluster (own index for a free neutron); A, Z as in orc_clusters.
 */
static inline double pinned_r2(const double* xi, const double* xj, double L, double invL) {
  double dx = xi[0] - xj[0], dy = xi[1] - xj[1], dz = xi[2] - xj[2];
  dx = dx - L * rint(dx * invL);
  dy = dy - L * rint(dy * invL);
  dz = dz - L * rint(dz * invL);
  return (dx * dx + dy * dy) + dz * dz;
}
void orc_clusters_mst(int64_t N, const double* x, const uint8_t* is_p, double L, double r_pp, double r_np,
                      int32_t* label, int32_t* A, int32_t* Z, int64_t* n_clusters) {
  int64_t* parent = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  const double invL = 1.0 / L, rpp2 = r_pp * r_pp, rnp2 = r_np * r_np;
  for (int64_t i = 0; i < N; ++i) parent[i] = i;
  for (int64_t i = 0; i < N; ++i) {
    if (!is_p[i]) continue;
    for (int64_t j = i + 1; j < N; ++j)
      if (is_p[j] && pinned_r2(x + 3 * i, x + 3 * j, L, invL) <= rpp2) uf_union(parent, i, j);
  }
  for (int64_t n = 0; n < N; ++n) {
    if (is_p[n]) continue;
    int64_t best = -1;
    double best_r2 = 0.0;
    for (int64_t j = 0; j < N; ++j) {
      if (!is_p[j]) continue;
      const double r2 = pinned_r2(x + 3 * n, x + 3 * j, L, invL);
      if (r2 <= rnp2 && (best < 0 || r2 < best_r2)) { best = j; best_r2 = r2; }
    }
    if (best >= 0) parent[n] = uf_find(parent, best); /* a leaf: nothing is ever hooked under a neutron */
  }
  finish_labels(N, parent, is_p, label, A, Z, n_clusters);
  free(parent);
}

/*
 * P14 helper: the same components through a cell grid of width >= r_cl (independent pair
 * enumeration; validated against orc_clusters at N <= 4096, then used where N^2 is too slow).
 * Needs floor(L / r_cl) >= 3; returns -1 otherwise.
 */
int orc_clusters_cells(int64_t N, const double* x, const uint8_t* is_p, double L, double r_cl,
                       int32_t* label, int32_t* A, int32_t* Z, int64_t* n_clusters) {
  const int32_t nc = orc_ncell(L, r_cl * (1.0 + 1e-9), 1);
  if (nc < 3) return -1;
  const int64_t nc3 = (int64_t)nc * nc * nc;
  int32_t* cid = (int32_t*)malloc((size_t)N * sizeof(int32_t));
  int32_t* start = (int32_t*)malloc((size_t)(nc3 + 1) * sizeof(int32_t));
  int32_t* fill = (int32_t*)malloc((size_t)nc3 * sizeof(int32_t));
  int32_t* order = (int32_t*)malloc((size_t)N * sizeof(int32_t));
  int64_t* parent = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  orc_cells(N, x, L, nc, cid, start);
  memcpy(fill, start, (size_t)nc3 * sizeof(int32_t));
  for (int64_t i = 0; i < N; ++i) order[fill[cid[i]]++] = (int32_t)i;
  for (int64_t i = 0; i < N; ++i) parent[i] = i;
  const double invL = 1.0 / L, rcl2 = r_cl * r_cl;
  for (int64_t i = 0; i < N; ++i) {
    const int32_t cx = cid[i] % nc, cy = (cid[i] / nc) % nc, cz = cid[i] / (nc * nc);
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          const int32_t q = (((cz + dz + nc) % nc) * nc + (cy + dy + nc) % nc) * nc + (cx + dx + nc) % nc;
          for (int32_t s = start[q]; s < start[q + 1]; ++s) {
            const int64_t j = order[s];
            if (j > i && linked(x + 3 * i, x + 3 * j, L, invL, rcl2)) uf_union(parent, i, j);
          }
        }
  }
  finish_labels(N, parent, is_p, label, A, Z, n_clusters);
  free(cid); free(start); free(fill); free(order); free(parent);
  return 0;
}

/*
 * Composition summary: free-neutron mass fraction = #(A=1,Z=0)/N;
 * mean and population sigma of A and Z over clusters with A >= a_min (12 in the paper).
 * out = {free_n_fraction, n_heavy, mean_A, sigma_A, mean_Z, sigma_Z}
 */
void orc_composition(int64_t N, const int32_t* A, const int32_t* Z, int32_t a_min, double* out) {
  double nfree = 0, nh = 0, sA = 0, sAA = 0, sZ = 0, sZZ = 0;
  for (int64_t r = 0; r < N; ++r) {
    if (A[r] == 1 && Z[r] == 0) nfree += 1;
    if (A[r] >= a_min) {
      nh += 1;
      sA += A[r]; sAA += (double)A[r] * A[r];
      sZ += Z[r]; sZZ += (double)Z[r] * Z[r];
    }
  }
  out[0] = nfree / (double)N;
  out[1] = nh;
  if (nh > 0) {
    double mA = sA / nh, mZ = sZ / nh;
    double vA = sAA / nh - mA * mA, vZ = sZZ / nh - mZ * mZ;
    out[2] = mA; out[3] = sqrt(vA > 0 ? vA : 0);
    out[4] = mZ; out[5] = sqrt(vZ > 0 ? vZ : 0);
  } else {
    out[2] = out[3] = out[4] = out[5] = 0.0;
  }
}
