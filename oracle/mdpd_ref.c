/*
 * mdpd_ref.c -- fp64 CPU ORACLE for one mDPD velocity-Verlet timestep.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_1903_10134_b200/csrc/ and is written from the paper's text
 * (/root/reference/PAPER.md, cited as P:L<line>) plus the readings listed in
 * DESIGN.md ("Readings of the paper", R1..R18).  Plain serial C, double precision, no
 * blocking / fusion / reordering beyond what the paper's Algorithm 1 states.
 *
 * What it computes (section 2.1, Eq. (1); Algorithm 1):
 *   rho_i = sum_{j != i, r_ij < rd} 15/(2 pi rd^3) (1 - r_ij/rd)^2                       [P:L81]
 *   F_ij  = [ A wC + B (rho_i + rho_j) wd  - gamma wR^2 (e_ij . v_ij) + sigma wR xi_ij / sqrt(dt) ] e_ij
 *           wC = 1 - r/rc, wR = wC^s, wd = max(0, 1 - r/rd), e_ij = r_ij/|r_ij|, r_ij = r_i - r_j   [P:L75-81]
 *   xi_ij = sqrt(3) 2^-23 ( (int)(h >> 8) - 2^23 ),  h = HASH(min tag, max tag, step, seed)  [DESIGN.md R5]
 *   velocity Verlet: half kick, drift (+ periodic wrap, voxel-mask bounce-back), forces at the new
 *   time level with the half-step velocities, half kick                                   [P:L75, Alg. 1; R6, R7]
 *   frozen wall particles (type 1) never move, have v = 0, get rho, interact with fluid   [P:L162; R8]
 *
 * Pins (tests/test_oracle_*.py): closed-form 2-/3-particle rho and F, lattice sums, the
 * normalisation integral of w_rho, O(N^2) brute force (numpy, written in the test) for pair
 * sets / rho / F, zero beyond cut-offs, momentum conservation, Poisson statistics of a random
 * state, thermostat kT = sigma^2 / 2 gamma, the paper's EOS closed form, the analytic
 * Poiseuille parabola.  Whole trajectories beyond a few steps: PARITY UNPINNED (chaotic) --
 * only statistics are comparable.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define REF_OK 0
#define REF_EINVAL (-1)
#define REF_ENOMEM (-2)
#define REF_ESTATE (-5)
#define REF_EINSOLID (-7)

#define MDPD_REF_MAXTYPES 8

typedef struct {
  double box[3];
  double rc, rd;
  double A, B;
  double gamma, sigma;
  double kT;
  double s;
  double mass, dt;
  double g[3];
  uint32_t seed;
  uint32_t pad;
} mdpd_ref_params;

typedef struct mdpd_ref_ctx {
  mdpd_ref_params p;
  int have_params;
  uint64_t n;
  double *x, *v, *f, *fpair, *rho; /* [n][3], [n] ; index == tag == load order */
  uint8_t *type;    /* 1: frozen (never integrated), 0: mobile */
  uint8_t *species; /* material type of the particle: row / column of the pair-parameter matrices below */
  uint32_t *tag;    /* NULL: tag == index (load order, R5).  mdpd_ref_set_tags: the particles are a SUBSET of a larger
                     * system and keep the tags they have there, so that the hashed random force of a pair is the one the
                     * whole system evaluates (the hash is a function of the two tags, the step and the seed). */
  /* Per-type-pair conservative parameters ("A_SL, B_SL"; Tables 1-2): ntypes == 0 means
   * one material, A and B of mdpd_ref_params for every pair, type byte != 0 <=> frozen.  Otherwise the type byte of a
   * particle is its species s in [0, ntypes), the pair (i, j) uses Am[s_i][s_j], Bm[s_i][s_j] (symmetric), and species s
   * is frozen iff bit s of frozen_mask is set. */
  int ntypes;
  double Am[MDPD_REF_MAXTYPES * MDPD_REF_MAXTYPES], Bm[MDPD_REF_MAXTYPES * MDPD_REF_MAXTYPES];
  uint32_t frozen_mask;
  /* Per-type-pair dissipative / random amplitudes (every pair carries F^D = -gamma wD (e.v) e and
   * F^R = sigma wR xi / sqrt(dt) e with sigma^2 = 2 gamma kT; the paper runs water at gamma = 12.4, and its
   * other fluids at 4.5, so a two-fluid system needs gamma_ij, sigma_ij).  have_gs == 0: gamma and sigma
   * of mdpd_ref_params for every pair. */
  int have_gs;
  double Gm[MDPD_REF_MAXTYPES * MDPD_REF_MAXTYPES], Sm[MDPD_REF_MAXTYPES * MDPD_REF_MAXTYPES];
  uint8_t *mask; /* [nz][ny][nx], 1 = solid */
  uint32_t mdim[3];
  double voxel;
  uint64_t step;      /* index k of the time level at which f was evaluated */
  int brute;          /* 1: O(N^2) pair enumeration */
  uint64_t bounces;   /* cumulative bounce-back events */
  uint64_t npairs_rc; /* pairs with r < rc at the last force evaluation */
  double virial_c;    /* sum over pairs of r_ij . F^C_ij at the last force evaluation */
  double vir_t[6];    /* its tensor: sum over pairs of r_ij,a F^C_ij,b for ab = xx, yy, zz, xy, xz, yz (symmetric) */
  /* scratch for the cell list */
  int64_t *cell_head, *next;
  uint64_t cell_cap;
} mdpd_ref_ctx;

/* ---------------------------------------------------------------------------------------------
 * HASH (frozen; this function is written from that text).
 *   x = a, y = b                      (a = min tag, b = max tag)
 *   for r = 0..5:  key = (r even) ? step + (r/2)*0x9E3779B9 : seed + (r/2)*0xBB67AE85   (mod 2^32)
 *                  p = 0xD256D193 * x  (64-bit) ; (x, y) <- (hi32(p) ^ y ^ key, lo32(p))
 *   h = x
 * ------------------------------------------------------------------------------------------- */
uint32_t mdpd_ref_hash(uint32_t a, uint32_t b, uint32_t step, uint32_t seed) {
  uint32_t x = a, y = b;
  for (uint32_t r = 0; r < 6; ++r) {
    uint32_t key = (r % 2 == 0) ? (uint32_t)(step + (r / 2) * 0x9E3779B9u) : (uint32_t)(seed + (r / 2) * 0xBB67AE85u);
    uint64_t p = (uint64_t)0xD256D193u * (uint64_t)x;
    uint32_t hi = (uint32_t)(p >> 32), lo = (uint32_t)p;
    x = hi ^ y ^ key;
    y = lo;
  }
  return x;
}

/* xi in [-sqrt 3, sqrt 3): zero mean, unit variance (uniform).  DESIGN.md R5. */
double mdpd_ref_xi(uint32_t h) {
  int32_t u = (int32_t)(h >> 8) - (1 << 23);
  return sqrt(3.0) * ldexp((double)u, -23);
}

int mdpd_ref_rng_fill(uint32_t seed, uint64_t npairs, const uint32_t *pairs, uint32_t step, uint32_t *out) {
  for (uint64_t q = 0; q < npairs; ++q) {
    uint32_t a = pairs[2 * q], b = pairs[2 * q + 1];
    uint32_t lo = a < b ? a : b, hi = a < b ? b : a;
    out[q] = mdpd_ref_hash(lo, hi, step, seed);
  }
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------- */
int mdpd_ref_create(mdpd_ref_ctx **out) {
  if (!out) return REF_EINVAL;
  mdpd_ref_ctx *h = (mdpd_ref_ctx *)calloc(1, sizeof(mdpd_ref_ctx));
  if (!h) return REF_ENOMEM;
  *out = h;
  return REF_OK;
}

static void free_particles(mdpd_ref_ctx *h) {
  free(h->x); free(h->v); free(h->f); free(h->fpair); free(h->rho); free(h->type); free(h->species); free(h->next); free(h->tag);
  h->x = h->v = h->f = h->fpair = h->rho = NULL;
  h->type = NULL; h->species = NULL; h->next = NULL; h->tag = NULL; h->n = 0;
}

int mdpd_ref_destroy(mdpd_ref_ctx *h) {
  if (!h) return REF_EINVAL;
  free_particles(h);
  free(h->mask);
  free(h->cell_head);
  free(h);
  return REF_OK;
}

int mdpd_ref_set_params(mdpd_ref_ctx *h, const mdpd_ref_params *p) {
  if (!h || !p) return REF_EINVAL;
  if (!(p->rc > 0) || !(p->rd > 0) || !(p->rd <= p->rc) || !(p->dt > 0) || !(p->mass > 0)) return REF_EINVAL;
  for (int d = 0; d < 3; ++d)
    if (!(p->box[d] >= 2.0 * p->rc)) return REF_EINVAL; /* minimum image needs L >= 2 rc */
  h->p = *p;
  h->have_params = 1;
  return REF_OK;
}

/* Pair-parameter matrices ([ntypes][ntypes], symmetric) and the set of frozen species; before load_particles.
 * ntypes == 0 returns to one material. */
int mdpd_ref_set_pair_params(mdpd_ref_ctx *h, int ntypes, const double *A, const double *B, uint32_t frozen_mask) {
  if (!h || ntypes < 0 || ntypes > MDPD_REF_MAXTYPES) return REF_EINVAL;
  if (h->n) return REF_ESTATE;
  if (ntypes && (!A || !B)) return REF_EINVAL;
  for (int a = 0; a < ntypes; ++a)
    for (int b = 0; b < ntypes; ++b) {
      if (A[a * ntypes + b] != A[b * ntypes + a] || B[a * ntypes + b] != B[b * ntypes + a]) return REF_EINVAL;
      h->Am[a * ntypes + b] = A[a * ntypes + b];
      h->Bm[a * ntypes + b] = B[a * ntypes + b];
    }
  h->ntypes = ntypes;
  h->frozen_mask = frozen_mask;
  h->have_gs = 0; /* the amplitude matrices belong to a species set: a new set starts without them */
  return REF_OK;
}

/* gamma_ij, sigma_ij ([ntypes][ntypes], symmetric, ntypes = that of the last mdpd_ref_set_pair_params).  G == NULL or
 * S == NULL: back to gamma, sigma of mdpd_ref_params for every pair.  The values may change at any time (they enter the
 * next force evaluation); nothing is checked against kT: sigma_ij^2 = 2 gamma_ij kT is the caller's business. */
int mdpd_ref_set_pair_gamma_sigma(mdpd_ref_ctx *h, int ntypes, const double *G, const double *S) {
  if (!h) return REF_EINVAL;
  if (!G || !S) {
    h->have_gs = 0;
    return REF_OK;
  }
  if (ntypes <= 0 || ntypes != h->ntypes) return REF_EINVAL;
  for (int a = 0; a < ntypes; ++a)
    for (int b = 0; b < ntypes; ++b) {
      if (G[a * ntypes + b] != G[b * ntypes + a] || S[a * ntypes + b] != S[b * ntypes + a]) return REF_EINVAL;
      if (!(G[a * ntypes + b] >= 0.0) || !(S[a * ntypes + b] >= 0.0)) return REF_EINVAL;
      h->Gm[a * ntypes + b] = G[a * ntypes + b];
      h->Sm[a * ntypes + b] = S[a * ntypes + b];
    }
  h->have_gs = 1;
  return REF_OK;
}

int mdpd_ref_set_brute_force(mdpd_ref_ctx *h, int on) {
  if (!h) return REF_EINVAL;
  h->brute = on ? 1 : 0;
  return REF_OK;
}

/* periodic wrap into [0, L): x <- x - L floor(x/L); a result equal to L becomes 0  (R12) */
static double wrap(double x, double L) {
  double y = x - L * floor(x / L);
  if (y >= L) y = 0.0;
  if (y < 0.0) y = 0.0;
  return y;
}

/* minimum-image component of r_i - r_j for coordinates in [0, L) */
static double minimg(double d, double L) {
  if (d > 0.5 * L) d -= L;
  else if (d < -0.5 * L) d += L;
  return d;
}

/* ------------------------------------------------------------------------------------------- *
 * Pair enumeration: every unordered pair (i < j by index == tag) with |minimg(x_i - x_j)| < rcut,
 * strict "<" on r^2 < rcut^2 (R3).  Brute force, or a cell list with edge L/floor(L/rcut) >= rcut
 * (falls back to brute force when a dimension has fewer than 3 cells).
 * ------------------------------------------------------------------------------------------- */
typedef void (*pair_fn)(mdpd_ref_ctx *h, uint64_t i, uint64_t j, const double d[3], double r2, void *arg);

static inline __attribute__((always_inline)) void try_pair(mdpd_ref_ctx *h, uint64_t i, uint64_t j, double rc2, pair_fn fn, void *arg) {
  double d[3];
  for (int k = 0; k < 3; ++k) d[k] = minimg(h->x[3 * i + k] - h->x[3 * j + k], h->p.box[k]);
  double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
  if (r2 < rc2) {
    if (i < j) fn(h, i, j, d, r2, arg);
    else {
      double e[3] = {-d[0], -d[1], -d[2]};
      fn(h, j, i, e, r2, arg);
    }
  }
}

static inline __attribute__((always_inline)) int for_each_pair(mdpd_ref_ctx *h, double rcut, pair_fn fn, void *arg) {
  const uint64_t n = h->n;
  const double rc2 = rcut * rcut;
  int nc[3];
  int use_cells = !h->brute;
  for (int k = 0; k < 3; ++k) {
    nc[k] = (int)floor(h->p.box[k] / rcut);
    if (nc[k] < 3) use_cells = 0;
  }
  if (!use_cells) {
    for (uint64_t i = 0; i < n; ++i)
      for (uint64_t j = i + 1; j < n; ++j) try_pair(h, i, j, rc2, fn, arg);
    return REF_OK;
  }
  uint64_t ncell = (uint64_t)nc[0] * nc[1] * nc[2];
  if (ncell > h->cell_cap) {
    free(h->cell_head);
    h->cell_head = (int64_t *)malloc(ncell * sizeof(int64_t));
    if (!h->cell_head) { h->cell_cap = 0; return REF_ENOMEM; }
    h->cell_cap = ncell;
  }
  for (uint64_t c = 0; c < ncell; ++c) h->cell_head[c] = -1;
  /* linked cells; insert in decreasing i so that each chain is in increasing i */
  for (uint64_t ii = n; ii-- > 0;) {
    int c[3];
    for (int k = 0; k < 3; ++k) {
      c[k] = (int)floor(h->x[3 * ii + k] / h->p.box[k] * nc[k]);
      if (c[k] >= nc[k]) c[k] = nc[k] - 1;
      if (c[k] < 0) c[k] = 0;
    }
    uint64_t lin = ((uint64_t)c[2] * nc[1] + c[1]) * nc[0] + c[0];
    h->next[ii] = h->cell_head[lin];
    h->cell_head[lin] = (int64_t)ii;
  }
  for (int cz = 0; cz < nc[2]; ++cz)
    for (int cy = 0; cy < nc[1]; ++cy)
      for (int cx = 0; cx < nc[0]; ++cx) {
        uint64_t lin = ((uint64_t)cz * nc[1] + cy) * nc[0] + cx;
        /* pairs inside the cell */
        for (int64_t i = h->cell_head[lin]; i >= 0; i = h->next[i])
          for (int64_t j = h->next[i]; j >= 0; j = h->next[j]) try_pair(h, (uint64_t)i, (uint64_t)j, rc2, fn, arg);
        /* 13 forward neighbour cells (half stencil), periodic; nc >= 3 so images are distinct */
        for (int dz = -1; dz <= 1; ++dz)
          for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
              int code = (dz + 1) * 9 + (dy + 1) * 3 + (dx + 1);
              if (code <= 13) continue; /* 13 == self; lower codes are the mirrored half */
              int ox = (cx + dx + nc[0]) % nc[0], oy = (cy + dy + nc[1]) % nc[1], oz = (cz + dz + nc[2]) % nc[2];
              uint64_t lin2 = ((uint64_t)oz * nc[1] + oy) * nc[0] + ox;
              for (int64_t i = h->cell_head[lin]; i >= 0; i = h->next[i])
                for (int64_t j = h->cell_head[lin2]; j >= 0; j = h->next[j])
                  try_pair(h, (uint64_t)i, (uint64_t)j, rc2, fn, arg);
            }
      }
  return REF_OK;
}

/* ------------------------------------------------------------------------------------------- */
static void density_pair(mdpd_ref_ctx *h, uint64_t i, uint64_t j, const double d[3], double r2, void *arg) {
  (void)d; (void)arg;
  const double rd = h->p.rd;
  const double K = 15.0 / (2.0 * M_PI * rd * rd * rd);
  double r = sqrt(r2);
  double w = 1.0 - r / rd;
  double wr = K * w * w;
  h->rho[i] += wr;
  h->rho[j] += wr;
}

static void force_pair(mdpd_ref_ctx *h, uint64_t i, uint64_t j, const double d[3], double r2, void *arg) {
  (void)arg;
  const mdpd_ref_params *p = &h->p;
  h->npairs_rc++;
  if (h->type[i] && h->type[j]) return; /* wall-wall forces are skipped (R8) */
  if (r2 < 1e-20) return;               /* R10 */
  double r = sqrt(r2);
  double e[3] = {d[0] / r, d[1] / r, d[2] / r};
  double w = 1.0 - r / p->rc;
  double wd = 1.0 - r / p->rd;
  if (wd < 0.0) wd = 0.0;
  double wR = (p->s == 1.0) ? w : pow(w, p->s);
  double ev = 0.0;
  for (int k = 0; k < 3; ++k) ev += e[k] * (h->v[3 * i + k] - h->v[3 * j + k]);
  uint32_t ta = (uint32_t)i, tb = (uint32_t)j; /* i < j here */
  if (h->tag) { /* caller-supplied tags: a = min tag, b = max tag */
    ta = h->tag[i] < h->tag[j] ? h->tag[i] : h->tag[j];
    tb = h->tag[i] < h->tag[j] ? h->tag[j] : h->tag[i];
  }
  uint32_t hh = mdpd_ref_hash(ta, tb, (uint32_t)h->step, p->seed);
  double xi = mdpd_ref_xi(hh);
  double Aij = p->A, Bij = p->B;
  if (h->ntypes) { /* per-type-pair parameters */
    Aij = h->Am[h->species[i] * h->ntypes + h->species[j]];
    Bij = h->Bm[h->species[i] * h->ntypes + h->species[j]];
  }
  double gij = p->gamma, sij = p->sigma;
  if (h->ntypes && h->have_gs) { /* per-type-pair amplitudes, P:L75 with P:L89 / P:L141 */
    gij = h->Gm[h->species[i] * h->ntypes + h->species[j]];
    sij = h->Sm[h->species[i] * h->ntypes + h->species[j]];
  }
  double FC = Aij * w + Bij * (h->rho[i] + h->rho[j]) * wd;            /* Eq. (1) */
  double FD = -gij * wR * wR * ev;                                     /* P:L75, wD = wR^2 */
  double FR = sij * wR * xi / sqrt(p->dt);                             /* P:L75; R2 */
  double F = FC + FD + FR;
  for (int k = 0; k < 3; ++k) {
    h->fpair[3 * i + k] += F * e[k];
    h->fpair[3 * j + k] -= F * e[k];
  }
  h->virial_c += FC * r;
  /* configurational part of the stress (conservative forces): r_a F_b = FC d_a d_b / r; the interfacial tension of
   * section 4.1 is L_x < s_xx - (s_yy + s_zz) / 2 > */
  h->vir_t[0] += FC * d[0] * d[0] / r;
  h->vir_t[1] += FC * d[1] * d[1] / r;
  h->vir_t[2] += FC * d[2] * d[2] / r;
  h->vir_t[3] += FC * d[0] * d[1] / r;
  h->vir_t[4] += FC * d[0] * d[2] / r;
  h->vir_t[5] += FC * d[1] * d[2] / r;
}

int mdpd_ref_compute_forces(mdpd_ref_ctx *h) {
  if (!h || !h->have_params || !h->x) return REF_ESTATE;
  const uint64_t n = h->n;
  int rcode;
  for (uint64_t i = 0; i < n; ++i) h->rho[i] = 0.0;
  if ((rcode = for_each_pair(h, h->p.rd, density_pair, NULL)) != REF_OK) return rcode;
  for (uint64_t i = 0; i < 3 * n; ++i) h->fpair[i] = 0.0;
  h->npairs_rc = 0;
  h->virial_c = 0.0;
  for (int k = 0; k < 6; ++k) h->vir_t[k] = 0.0;
  if ((rcode = for_each_pair(h, h->p.rc, force_pair, NULL)) != REF_OK) return rcode;
  for (uint64_t i = 0; i < n; ++i)
    for (int k = 0; k < 3; ++k)
      h->f[3 * i + k] = h->fpair[3 * i + k] + (h->type[i] ? 0.0 : h->p.mass * h->p.g[k]);
  return REF_OK;
}

static int in_solid(const mdpd_ref_ctx *h, const double x[3]) {
  if (!h->mask) return 0;
  uint32_t iv[3];
  for (int k = 0; k < 3; ++k) {
    double q = floor(x[k] / h->voxel);
    if (q < 0) q = 0;
    uint32_t u = (uint32_t)q;
    if (u >= h->mdim[k]) u = h->mdim[k] - 1;
    iv[k] = u;
  }
  return h->mask[((uint64_t)iv[2] * h->mdim[1] + iv[1]) * h->mdim[0] + iv[0]] != 0;
}

int mdpd_ref_load_particles(mdpd_ref_ctx *h, uint64_t n, const double *pos, const double *vel, const uint8_t *type) {
  if (!h || !h->have_params) return REF_ESTATE;
  if (n && (!pos || !vel)) return REF_EINVAL;
  free_particles(h);
  h->n = n;
  uint64_t m = n ? n : 1;
  h->x = (double *)calloc(3 * m, sizeof(double));
  h->v = (double *)calloc(3 * m, sizeof(double));
  h->f = (double *)calloc(3 * m, sizeof(double));
  h->fpair = (double *)calloc(3 * m, sizeof(double));
  h->rho = (double *)calloc(m, sizeof(double));
  h->type = (uint8_t *)calloc(m, 1);
  h->species = (uint8_t *)calloc(m, 1);
  h->next = (int64_t *)calloc(m, sizeof(int64_t));
  if (!h->x || !h->v || !h->f || !h->fpair || !h->rho || !h->type || !h->species || !h->next) return REF_ENOMEM;
  for (uint64_t i = 0; i < n; ++i) {
    if (h->ntypes) {
      const uint8_t sp = type ? type[i] : 0;
      if (sp >= h->ntypes) return REF_EINVAL;
      h->species[i] = sp;
      h->type[i] = (uint8_t)((h->frozen_mask >> sp) & 1u);
    } else {
      h->type[i] = type ? (type[i] != 0) : 0;
      h->species[i] = h->type[i];
    }
    for (int k = 0; k < 3; ++k) {
      h->x[3 * i + k] = wrap(pos[3 * i + k], h->p.box[k]);
      h->v[3 * i + k] = h->type[i] ? 0.0 : vel[3 * i + k]; /* frozen: v == 0 (R8) */
    }
  }
  h->step = 0;
  h->bounces = 0;
  return mdpd_ref_compute_forces(h);
}

int mdpd_ref_load_wall_mask(mdpd_ref_ctx *h, const uint8_t *mask, const uint32_t dims[3], double voxel) {
  if (!h || !h->have_params) return REF_ESTATE;
  free(h->mask);
  h->mask = NULL;
  if (!mask) return REF_OK;
  if (!dims || !(voxel > 0)) return REF_EINVAL;
  for (int k = 0; k < 3; ++k)
    if (fabs(dims[k] * voxel - h->p.box[k]) > 1e-6 * h->p.box[k]) return REF_EINVAL;
  uint64_t nv = (uint64_t)dims[0] * dims[1] * dims[2];
  h->mask = (uint8_t *)malloc(nv);
  if (!h->mask) return REF_ENOMEM;
  memcpy(h->mask, mask, nv);
  for (int k = 0; k < 3; ++k) h->mdim[k] = dims[k];
  h->voxel = voxel;
  uint64_t bad = 0;
  for (uint64_t i = 0; i < h->n; ++i)
    if (!h->type[i] && in_solid(h, &h->x[3 * i])) bad++;
  return bad ? REF_EINSOLID : REF_OK;
}

/* Tags of a subset of a larger system (see mdpd_ref_ctx.tag): [n] distinct uint32, or NULL to return to tag == index.
 * Forces are re-evaluated.  Pair lists (mdpd_ref_get_pairs) keep reporting indices. */
int mdpd_ref_set_tags(mdpd_ref_ctx *h, const uint32_t *tags) {
  if (!h || !h->x) return REF_ESTATE;
  free(h->tag);
  h->tag = NULL;
  if (tags) {
    uint64_t m = h->n ? h->n : 1;
    h->tag = (uint32_t *)malloc(m * sizeof(uint32_t));
    if (!h->tag) return REF_ENOMEM;
    memcpy(h->tag, tags, h->n * sizeof(uint32_t));
  }
  return mdpd_ref_compute_forces(h);
}

int mdpd_ref_set_step(mdpd_ref_ctx *h, uint64_t step) {
  if (!h) return REF_EINVAL;
  h->step = step;
  return REF_OK;
}

int mdpd_ref_set_velocities(mdpd_ref_ctx *h, const double *vel) {
  if (!h || !h->x || !vel) return REF_EINVAL;
  for (uint64_t i = 0; i < h->n; ++i)
    for (int k = 0; k < 3; ++k) h->v[3 * i + k] = h->type[i] ? 0.0 : vel[3 * i + k];
  return REF_OK;
}

/* One velocity-Verlet step, Algorithm 1 order without the inter-rank steps; R6, R7. */
int mdpd_ref_step(mdpd_ref_ctx *h, uint32_t nsteps) {
  if (!h || !h->have_params || !h->x) return REF_ESTATE;
  const mdpd_ref_params *p = &h->p;
  const double hdt = 0.5 * p->dt;
  for (uint32_t it = 0; it < nsteps; ++it) {
    for (uint64_t i = 0; i < h->n; ++i) {
      if (h->type[i]) continue;
      double xs[3];
      for (int k = 0; k < 3; ++k) {
        h->v[3 * i + k] += hdt * h->f[3 * i + k] / p->mass;              /* half kick */
        xs[k] = wrap(h->x[3 * i + k] + p->dt * h->v[3 * i + k], p->box[k]); /* Alg. 1 line 1 */
      }
      if (in_solid(h, xs)) { /* bounce-back: position kept, velocity reversed (R7) */
        for (int k = 0; k < 3; ++k) h->v[3 * i + k] = -h->v[3 * i + k];
        h->bounces++;
      } else {
        for (int k = 0; k < 3; ++k) h->x[3 * i + k] = xs[k];
      }
    }
    h->step += 1;
    int rcode = mdpd_ref_compute_forces(h); /* Alg. 1 lines 4 and 6, half-step velocities in F^D */
    if (rcode != REF_OK) return rcode;
    for (uint64_t i = 0; i < h->n; ++i) {
      if (h->type[i]) continue;
      for (int k = 0; k < 3; ++k) h->v[3 * i + k] += hdt * h->f[3 * i + k] / p->mass; /* Alg. 1 line 7 */
    }
  }
  return REF_OK;
}

int mdpd_ref_get_state(mdpd_ref_ctx *h, double *pos, double *vel, double *force, double *rho, uint64_t *step) {
  if (!h || !h->x) return REF_ESTATE;
  if (pos) memcpy(pos, h->x, 3 * h->n * sizeof(double));
  if (vel) memcpy(vel, h->v, 3 * h->n * sizeof(double));
  if (force) memcpy(force, h->f, 3 * h->n * sizeof(double));
  if (rho) memcpy(rho, h->rho, h->n * sizeof(double));
  if (step) *step = h->step;
  return REF_OK;
}

/* pairwise part of the force (without m g), for the momentum-conservation pin */
int mdpd_ref_get_pair_force(mdpd_ref_ctx *h, double *fpair) {
  if (!h || !h->x || !fpair) return REF_ESTATE;
  memcpy(fpair, h->fpair, 3 * h->n * sizeof(double));
  return REF_OK;
}

/* out[0] steps, [1] bounces, [2] pairs r<rc at last evaluation; out_f[0] = sum r_ij F^C_ij */
/* sum over interacting pairs of r_ij,a F^C_ij,b at the last force evaluation: xx, yy, zz, xy, xz, yz */
int mdpd_ref_get_virial(mdpd_ref_ctx *h, double out[6]) {
  if (!h || !out) return REF_EINVAL;
  for (int k = 0; k < 6; ++k) out[k] = h->vir_t[k];
  return REF_OK;
}

int mdpd_ref_get_counters(mdpd_ref_ctx *h, uint64_t out[4], double out_f[2]) {
  if (!h) return REF_EINVAL;
  if (out) { out[0] = h->step; out[1] = h->bounces; out[2] = h->npairs_rc; out[3] = h->n; }
  if (out_f) { out_f[0] = h->virial_c; out_f[1] = 0.0; }
  return REF_OK;
}

typedef struct { uint32_t *pairs; uint64_t cap, count; } pair_sink;

static void collect_pair(mdpd_ref_ctx *h, uint64_t i, uint64_t j, const double d[3], double r2, void *arg) {
  (void)h; (void)d; (void)r2;
  pair_sink *s = (pair_sink *)arg;
  if (s->pairs && s->count < s->cap) {
    s->pairs[2 * s->count] = (uint32_t)i;
    s->pairs[2 * s->count + 1] = (uint32_t)j;
  }
  s->count++;
}

static int cmp_pair(const void *a, const void *b) {
  const uint32_t *p = (const uint32_t *)a, *q = (const uint32_t *)b;
  if (p[0] != q[0]) return p[0] < q[0] ? -1 : 1;
  if (p[1] != q[1]) return p[1] < q[1] ? -1 : 1;
  return 0;
}

/* all tag pairs a < b with r < rcut, sorted; *count is the true count even if it exceeds cap */
int mdpd_ref_get_pairs(mdpd_ref_ctx *h, double rcut, uint64_t *count, uint32_t *pairs, uint64_t cap) {
  if (!h || !h->x || !count) return REF_ESTATE;
  pair_sink s = {pairs, cap, 0};
  int rcode = for_each_pair(h, rcut, collect_pair, &s);
  if (rcode != REF_OK) return rcode;
  *count = s.count;
  if (pairs) qsort(pairs, (size_t)(s.count < cap ? s.count : cap), 2 * sizeof(uint32_t), cmp_pair);
  return REF_OK;
}
