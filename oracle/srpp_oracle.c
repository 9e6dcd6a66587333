/*
 * srpp_oracle.c -- fp64 CPU ORACLE for the short-range particle-particle path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, header, table or constant with the CUDA path (paper_1411_3396_b200/csrc);
 * neither side includes or imports the other.
 *
 * What it computes, and the passages it follows (PAPER.md = /root/reference/PAPER.md,
 * Heitmann et al., "The Q Continuum Simulation", arXiv:1411.3396):
 *
 *   PAPER.md:63  (Sec. 2)  the force is split into a long-range PM part and a short-range
 *                part; on accelerated systems the short-range solver is a direct
 *                particle-particle ("N^2") sum.
 *   PAPER.md:65  (Sec. 2)  spectral filtering sets a "hand-over" between the two solvers at a
 *                small length scale, so the short-range pair force is the Newtonian force minus
 *                the (filtered) grid force and vanishes beyond the hand-over radius.
 *   PAPER.md:71,73 (Sec. 2.1) the GPU kernel itself is "described elsewhere"; a "short-range
 *                force timestep" updates the active particles (the kick).
 *
 * PAPER.md does not print the force law; BASELINE.json `north_star` fixes its form and
 * SURVEY.md 8(c) lists the readings R1..R18 taken here (DESIGN.md repeats them):
 *
 *   a_i = sum_{j != i, s_ij < rc^2}  m_j * d_ij * [ (s_ij + eps^2)^(-3/2) - P(s_ij) ]      (R1, R2)
 *   d_ij = minimum image of (x_j - x_i) per axis, s_ij = d_ij . d_ij                     (R8)
 *   P(s) = sum_{k=0..5} c_k s^k, c_k = the six fp32 inputs widened to fp64                 (R4)
 *   strict cutoff on the UNSOFTENED s; G = 1; output is an acceleration                   (R5, R2)
 *
 * Because the chaining mesh only accelerates the neighbour search, the oracle is this plain
 * definition: orc_accel_bruteforce() is the O(N^2) double loop, written out.  orc_accel() is
 * the same sum restricted to candidate pairs from the oracle's OWN cell list (cell edge >= rc,
 * fp64 cell assignment), which tests/ check against the brute force (pin P6).
 *
 * Binning (R10-R12): per axis, in fp32, inv = (float)ncell / box; c = (int)floorf(x * inv);
 * c = min(c, ncell-1); cid = cx + ncx*(cy + ncy*cz); stable counting sort on cid.  This is the
 * only place the oracle deliberately computes in fp32 (compile with -ffp-contract=off).
 *
 * Pins: see tests/test_oracle_pins.py (P1..P11 of SURVEY.md 8(c)).  The one unpinned item is
 * the fidelity of the DEFAULT polynomial to the real HACC grid force: "parity unpinned"
 * (PAPER.md gives nothing to compare with); it does not affect GPU-vs-oracle parity because
 * both sides take poly[6] as data.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  float box[3];
  float rcut;
  float eps;
  float poly[6];
  int32_t periodic[3]; /* 1: periodic axis, minimum image (R8); 0: open axis, plain differences and no neighbours
                          across the faces -- the overloaded (non-periodic) node volume of PAPER.md:65 */
} orc_params;

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  return (int32_t)omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---------------------------------------------------------------- binning (R10-R12) -- */

/* fp32 cell coordinate of one position component (R10). Returns -1 outside [0, L) or non-finite (R13). */
static int32_t cell_coord_f32(float x, float box, int32_t ncell) {
  if (!(x >= 0.0f) || !(x < box)) return -1;
  volatile float inv = (float)ncell / box; /* one IEEE fp32 division */
  volatile float prod = x * inv;           /* one IEEE fp32 multiply, never fused */
  int32_t c = (int32_t)floorf(prod);
  if (c > ncell - 1) c = ncell - 1;
  return c;
}

/* cid[i] = cx + ncx*(cy + ncy*cz) (R11). Returns 0, or -3 if any position violates R13. */
int32_t orc_cell_ids(const float *pos_mass, int64_t n, const float *box, const int32_t *ncell,
                     uint32_t *cid) {
  int32_t bad = 0;
  for (int64_t i = 0; i < n; ++i) {
    int32_t cx = cell_coord_f32(pos_mass[4 * i + 0], box[0], ncell[0]);
    int32_t cy = cell_coord_f32(pos_mass[4 * i + 1], box[1], ncell[1]);
    int32_t cz = cell_coord_f32(pos_mass[4 * i + 2], box[2], ncell[2]);
    if (cx < 0 || cy < 0 || cz < 0) { bad = 1; cid[i] = 0; continue; }
    cid[i] = (uint32_t)cx + (uint32_t)ncell[0] * ((uint32_t)cy + (uint32_t)ncell[1] * (uint32_t)cz);
  }
  return bad ? -3 : 0;
}

/* Stable counting sort by cell id (R12): cell_start[ncells+1], perm[n], sorted[4n]. */
int32_t orc_build_mesh(const float *pos_mass, int64_t n, const float *box, const int32_t *ncell,
                       uint32_t *cell_start, uint32_t *perm, float *sorted) {
  int64_t ncells = (int64_t)ncell[0] * ncell[1] * ncell[2];
  uint32_t *cid = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
  if (!cid) return -6;
  int32_t rc = orc_cell_ids(pos_mass, n, box, ncell, cid);
  if (rc != 0) { free(cid); return rc; }
  /* histogram */
  for (int64_t c = 0; c <= ncells; ++c) cell_start[c] = 0;
  for (int64_t i = 0; i < n; ++i) cell_start[cid[i] + 1] += 1;
  /* exclusive scan: cell_start[c] = number of particles in cells < c */
  for (int64_t c = 0; c < ncells; ++c) cell_start[c + 1] += cell_start[c];
  /* stable scatter: ascending original index inside a cell */
  uint32_t *cursor = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(ncells > 0 ? ncells : 1));
  if (!cursor) { free(cid); return -6; }
  memcpy(cursor, cell_start, sizeof(uint32_t) * (size_t)ncells);
  for (int64_t i = 0; i < n; ++i) {
    uint32_t k = cursor[cid[i]]++;
    perm[k] = (uint32_t)i;
    if (sorted) memcpy(sorted + 4 * (size_t)k, pos_mass + 4 * (size_t)i, 4 * sizeof(float));
  }
  free(cursor);
  free(cid);
  return 0;
}

/* ---------------------------------------------------------------- pair force (R1-R9) -- */

/* P(s), exact real polynomial with the fp32 coefficients, evaluated in fp64 (R4). */
static double poly_eval(const double c[6], double s) {
  return c[0] + s * (c[1] + s * (c[2] + s * (c[3] + s * (c[4] + s * c[5]))));
}

/* f(s) = (s + eps^2)^(-3/2) - P(s) for s < rc^2, else 0 (R1, R3, R5). */
double orc_pair_factor(const orc_params *p, double s) {
  double c[6];
  for (int k = 0; k < 6; ++k) c[k] = (double)p->poly[k];
  double rc2 = (double)p->rcut * (double)p->rcut;
  double e2 = (double)p->eps * (double)p->eps;
  if (!(s < rc2)) return 0.0;
  double u = s + e2;
  return 1.0 / (u * sqrt(u)) - poly_eval(c, s);
}

double orc_poly(const orc_params *p, double s) {
  double c[6];
  for (int k = 0; k < 6; ++k) c[k] = (double)p->poly[k];
  return poly_eval(c, s);
}

/* minimum image of a coordinate difference in a periodic box of length L (R8) */
static inline double min_image(double d, double L) {
  if (d > 0.5 * L) d -= L;
  else if (d < -0.5 * L) d += L;
  return d;
}

/* coordinate difference on one axis: minimum image if the axis is periodic, the plain difference if it is open */
static inline double axis_diff(double d, double L, int32_t periodic) { return periodic ? min_image(d, L) : d; }

/*
 * The plain definition, O(N^2): for every target i the sum over ALL j != i.
 * acc[3n] fp64.  Optional outputs (may be NULL): n_in[n] = number of in-cutoff neighbours,
 * sum_abs[n] = sum_j |m_j f d| (scale of the terms, for fp32 error budgets).
 */
void orc_accel_bruteforce(const float *pos_mass, int64_t n, const orc_params *p, double *acc,
                          int64_t *n_in, double *sum_abs) {
  const double L[3] = {(double)p->box[0], (double)p->box[1], (double)p->box[2]};
  const double rc2 = (double)p->rcut * (double)p->rcut;
  const double e2 = (double)p->eps * (double)p->eps;
  double c[6];
  for (int k = 0; k < 6; ++k) c[k] = (double)p->poly[k];
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < n; ++i) {
    double xi = pos_mass[4 * i], yi = pos_mass[4 * i + 1], zi = pos_mass[4 * i + 2];
    double ax = 0, ay = 0, az = 0, sa = 0;
    int64_t cnt = 0;
    for (int64_t j = 0; j < n; ++j) {
      if (j == i) continue; /* R7 */
      double dx = axis_diff((double)pos_mass[4 * j] - xi, L[0], p->periodic[0]);
      double dy = axis_diff((double)pos_mass[4 * j + 1] - yi, L[1], p->periodic[1]);
      double dz = axis_diff((double)pos_mass[4 * j + 2] - zi, L[2], p->periodic[2]);
      double s = dx * dx + dy * dy + dz * dz;
      if (s < rc2) { /* strict cutoff on the unsoftened s (R5) */
        double u = s + e2;
        double f = 1.0 / (u * sqrt(u)) - poly_eval(c, s);
        double mf = (double)pos_mass[4 * j + 3] * f;
        ax += mf * dx; ay += mf * dy; az += mf * dz;
        sa += fabs(mf) * sqrt(s);
        ++cnt;
      }
    }
    acc[3 * i] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az;
    if (n_in) n_in[i] = cnt;
    if (sum_abs) sum_abs[i] = sa;
  }
}

/* ---- the oracle's own neighbour search: fp64 cell list with edge >= rc (checked by pin P6) ---- */

typedef struct {
  int32_t nc[3];
  int64_t ncells;
  uint32_t *start; /* ncells+1 */
  uint32_t *order; /* particle indices grouped by cell */
} orc_grid;

static int32_t grid_coord(double x, double L, int32_t nc) {
  int32_t c = (int32_t)floor(x / L * (double)nc);
  if (c < 0) c = 0;
  if (c > nc - 1) c = nc - 1;
  return c;
}

static int grid_build(orc_grid *g, const float *pos_mass, int64_t n, const orc_params *p) {
  for (int a = 0; a < 3; ++a) {
    int32_t k = (int32_t)floor((double)p->box[a] / (double)p->rcut);
    /* fewer than 3 cells of edge >= rc on an axis: one cell spans the axis (no neighbour wrap there) */
    g->nc[a] = (k >= 3) ? k : 1;
  }
  g->ncells = (int64_t)g->nc[0] * g->nc[1] * g->nc[2];
  g->start = (uint32_t *)calloc((size_t)g->ncells + 1, sizeof(uint32_t));
  g->order = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
  uint32_t *cell = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
  if (!g->start || !g->order || !cell) return -1;
  for (int64_t i = 0; i < n; ++i) {
    int32_t cx = grid_coord(pos_mass[4 * i], p->box[0], g->nc[0]);
    int32_t cy = grid_coord(pos_mass[4 * i + 1], p->box[1], g->nc[1]);
    int32_t cz = grid_coord(pos_mass[4 * i + 2], p->box[2], g->nc[2]);
    cell[i] = (uint32_t)(cx + g->nc[0] * (cy + (int64_t)g->nc[1] * cz));
    g->start[cell[i] + 1]++;
  }
  for (int64_t c = 0; c < g->ncells; ++c) g->start[c + 1] += g->start[c];
  uint32_t *cur = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)g->ncells);
  if (!cur) return -1;
  memcpy(cur, g->start, sizeof(uint32_t) * (size_t)g->ncells);
  for (int64_t i = 0; i < n; ++i) g->order[cur[cell[i]]++] = (uint32_t)i;
  free(cur);
  free(cell);
  return 0;
}

/*
 * Same sum as orc_accel_bruteforce, for the listed targets only (targets == NULL: all n, nt = n),
 * candidates taken from the oracle's own cell list.
 *   acc[3*nt]        fp64 accelerations
 *   n_in[nt]         in-cutoff neighbour count                       (may be NULL)
 *   sum_abs[nt]      sum_j |m_j f d|                                 (may be NULL)
 *   allowance[nt]    sum |m_j f d| over pairs with |s - rc^2| <= 2^-18 rc^2, f taken as if inside:
 *                    the R9 allowance for fp32 cutoff classification   (may be NULL)
 *   n_cand[nt]       candidate pairs examined by THIS cell list        (may be NULL)
 */
int32_t orc_accel(const float *pos_mass, int64_t n, const orc_params *p, const int64_t *targets,
                  int64_t nt, double *acc, int64_t *n_in, double *sum_abs, double *allowance,
                  int64_t *n_cand) {
  orc_grid g;
  if (grid_build(&g, pos_mass, n, p) != 0) return -6;
  const double L[3] = {(double)p->box[0], (double)p->box[1], (double)p->box[2]};
  const double rc2 = (double)p->rcut * (double)p->rcut;
  const double e2 = (double)p->eps * (double)p->eps;
  const double band = ldexp(rc2, -18);
  double c[6];
  for (int k = 0; k < 6; ++k) c[k] = (double)p->poly[k];
  if (!targets) nt = n;
#pragma omp parallel for schedule(dynamic, 8)
  for (int64_t t = 0; t < nt; ++t) {
    int64_t i = targets ? targets[t] : t;
    double xi = pos_mass[4 * i], yi = pos_mass[4 * i + 1], zi = pos_mass[4 * i + 2];
    int32_t ci[3] = {grid_coord(xi, L[0], g.nc[0]), grid_coord(yi, L[1], g.nc[1]),
                     grid_coord(zi, L[2], g.nc[2])};
    double ax = 0, ay = 0, az = 0, sa = 0, al = 0;
    int64_t cnt = 0, cand = 0;
    int lo[3], hi[3];
    for (int a = 0; a < 3; ++a) { lo[a] = (g.nc[a] >= 3) ? -1 : 0; hi[a] = (g.nc[a] >= 3) ? 1 : 0; }
    for (int oz = lo[2]; oz <= hi[2]; ++oz)
      for (int oy = lo[1]; oy <= hi[1]; ++oy)
        for (int ox = lo[0]; ox <= hi[0]; ++ox) {
          int32_t cx = ci[0] + ox, cy = ci[1] + oy, cz = ci[2] + oz;
          /* open axis: no neighbour cell beyond the faces; periodic axis: wrap */
          if ((!p->periodic[0] && (cx < 0 || cx >= g.nc[0])) || (!p->periodic[1] && (cy < 0 || cy >= g.nc[1])) ||
              (!p->periodic[2] && (cz < 0 || cz >= g.nc[2])))
            continue;
          cx = (cx + g.nc[0]) % g.nc[0];
          cy = (cy + g.nc[1]) % g.nc[1];
          cz = (cz + g.nc[2]) % g.nc[2];
          int64_t cc = cx + g.nc[0] * (cy + (int64_t)g.nc[1] * cz);
          for (uint32_t q = g.start[cc]; q < g.start[cc + 1]; ++q) {
            int64_t j = g.order[q];
            if (j == i) continue; /* R7 */
            ++cand;
            double dx = axis_diff((double)pos_mass[4 * j] - xi, L[0], p->periodic[0]);
            double dy = axis_diff((double)pos_mass[4 * j + 1] - yi, L[1], p->periodic[1]);
            double dz = axis_diff((double)pos_mass[4 * j + 2] - zi, L[2], p->periodic[2]);
            double s = dx * dx + dy * dy + dz * dz;
            double m = (double)pos_mass[4 * j + 3];
            if (s < rc2) {
              double u = s + e2;
              double f = 1.0 / (u * sqrt(u)) - poly_eval(c, s);
              ax += m * f * dx; ay += m * f * dy; az += m * f * dz;
              sa += fabs(m * f) * sqrt(s);
              ++cnt;
            }
            if (fabs(s - rc2) <= band) {
              double u = s + e2;
              double f = 1.0 / (u * sqrt(u)) - poly_eval(c, s);
              al += fabs(m * f) * sqrt(s);
            }
          }
        }
    acc[3 * t] = ax; acc[3 * t + 1] = ay; acc[3 * t + 2] = az;
    if (n_in) n_in[t] = cnt;
    if (sum_abs) sum_abs[t] = sa;
    if (allowance) allowance[t] = al;
    if (n_cand) n_cand[t] = cand;
  }
  free(g.start);
  free(g.order);
  return 0;
}

/* ---------------------------------------------------------------- kick / stream (R16, R17, R13) -- */

/* v <- fmaf(a, kdt, v) per component in fp32 (R16); .w lanes untouched. */
void orc_kick(float *vel, const float *acc, float kdt, int64_t n) {
  for (int64_t i = 0; i < n; ++i)
    for (int a = 0; a < 3; ++a) vel[4 * i + a] = fmaf(acc[4 * i + a], kdt, vel[4 * i + a]);
}

/* x <- wrap(fmaf(v, dt, x)) per component in fp32; a value that rounds to L becomes 0 (R13, R17).
 * Precondition |v*dt| < L (one wrap suffices). */
void orc_stream(float *pos_mass, const float *vel, float dt, const float *box, int64_t n) {
  for (int64_t i = 0; i < n; ++i)
    for (int a = 0; a < 3; ++a) {
      float L = box[a];
      float y = fmaf(vel[4 * i + a], dt, pos_mass[4 * i + a]);
      if (y >= L) y -= L;
      else if (y < 0.0f) y += L;
      if (!(y < L)) y = 0.0f;
      pos_mass[4 * i + a] = y;
    }
}

/* ---------------------------------------------------------------- most bound particle (MBP) -- */
/*
 * Halo centre as the potential minimum, "most bound particle" (Sec. 2.2).
 * The paper names the operation (its version is built from Thrust scan/transform/reduce) and prints no formula;
 * the reading taken here (R19): for every member i of halo h = [halo_start[h], halo_start[h+1])
 *
 *     phi_i = - sum_{j in h, j != i}  m_j / sqrt(|x_j - x_i|^2 + eps^2)          (G = 1)
 *
 * with PLAIN coordinate differences (a halo finder hands over unwrapped members) and the Plummer softening of the
 * force law (R3: -d/dr of -1/sqrt(r^2+eps^2) is the (s+eps^2)^(-3/2) term), and the centre is the member with the
 * smallest phi, the lowest index winning ties.  An empty halo has index -1; a one-particle halo has phi = 0.
 * phi[n] (fp64) and mbp[nhalo] (index into pos_mass) are outputs.  The plain definition, written out.
 */
void orc_mbp(const float *pos_mass, int64_t n, const int64_t *halo_start, int64_t nhalo, float eps, double *phi,
             int64_t *mbp) {
  (void)n;
  const double e2 = (double)eps * (double)eps;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t h = 0; h < nhalo; ++h) {
    const int64_t b = halo_start[h], e = halo_start[h + 1];
    int64_t best = -1;
    for (int64_t i = b; i < e; ++i) {
      const double xi = pos_mass[4 * i], yi = pos_mass[4 * i + 1], zi = pos_mass[4 * i + 2];
      double s = 0.0;
      for (int64_t j = b; j < e; ++j) {
        if (j == i) continue;
        const double dx = (double)pos_mass[4 * j] - xi, dy = (double)pos_mass[4 * j + 1] - yi,
                     dz = (double)pos_mass[4 * j + 2] - zi;
        s += (double)pos_mass[4 * j + 3] / sqrt(dx * dx + dy * dy + dz * dz + e2);
      }
      phi[i] = -s;
    }
    for (int64_t i = b; i < e; ++i)
      if (best < 0 || phi[i] < phi[best]) best = i;
    mbp[h] = best;
  }
}

/* ---------------------------------------------------------------- short-range sub-cycle -- */
/*
 * The "short-range force timestep" of PAPER.md:73 (Sec. 2.1: every block is evolved, its active particles updated,
 * the passive ones only streamed) as one call.  PAPER.md does not print the integrator; the reading taken here
 * (R20; SURVEY.md 8(f) item 1 "stream-kick-stream", R16, R17) is the symmetric split
 *
 *     repeat nsub times:   x <- stream(x, v, dt/2);   a = accel(x);   v <- kick(v, a, kdt);   x <- stream(x, v, dt/2)
 *
 * written out with the pieces above and nothing else: orc_stream (fp32 fma + wrap, R13/R17), the fp64 cell-list sum
 * orc_accel rounded ONCE to fp32 (the kick is an fp32 operation on fp32 accelerations, R16), orc_kick.  dt/2 is the
 * fp32 product 0.5f*dt (exact).  pos_mass[4n], vel[4n] are updated in place; acc[4n] (may be NULL) receives the fp32
 * accelerations of the LAST sub-step, .w = 0.  Returns 0, or -6 if out of memory.
 */
int32_t orc_subcycle(float *pos_mass, float *vel, int64_t n, const orc_params *p, float dt, float kdt, int32_t nsub,
                     float *acc) {
  double *a64 = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
  float *a32 = (float *)calloc(4 * (size_t)(n > 0 ? n : 1), sizeof(float));
  if (!a64 || !a32) { free(a64); free(a32); return -6; }
  const float half = 0.5f * dt;
  for (int32_t s = 0; s < nsub; ++s) {
    orc_stream(pos_mass, vel, half, p->box, n);
    int32_t rc = orc_accel(pos_mass, n, p, NULL, n, a64, NULL, NULL, NULL, NULL);
    if (rc != 0) { free(a64); free(a32); return rc; }
    for (int64_t i = 0; i < n; ++i)
      for (int a = 0; a < 3; ++a) a32[4 * i + a] = (float)a64[3 * i + a];
    orc_kick(vel, a32, kdt, n);
    orc_stream(pos_mass, vel, half, p->box, n);
  }
  if (acc) memcpy(acc, a32, sizeof(float) * 4 * (size_t)n);
  free(a64);
  free(a32);
  return 0;
}
