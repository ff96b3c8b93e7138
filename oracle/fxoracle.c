/*
 * fxoracle.c -- plain, slow CPU oracle of the batched block Euler update.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load this library.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2208_11630_b200/csrc/ (it re-declares its own enums; the values are
 * compared numerically by the tests, not through a common header).
 *
 * What it computes: the hot path BASELINE.json's north_star names -- guard-cell
 * fill, primitive recovery with the gamma-law EOS, PLM-minmod or WENO5-JS
 * reconstruction, HLLE or HLLC fluxes, flux divergence, SSP-RK2/3 and the CFL
 * time step -- block by block [PAPER.md L69, section 2: "Bulk of their code is
 * written for block-by-block update"], explicit shock capturing [PAPER.md L71],
 * SSP-RK of order 2 or 3 [PAPER.md L103, section 2.2], perfect gas [PAPER.md
 * L105].  PAPER.md prints no formula; every formula below is the textbook one
 * in the reading SURVEY.md section 8(c) fixes (tags O1..O7, A1..A27) and
 * DESIGN.md lists.  The method is an explicit iteration, so the oracle is the
 * algorithm itself, step by step, in fp64, with no blocking, fusion or
 * reordering.  Built with -O2 -ffp-contract=off (no FMA contraction).
 *
 * Passive mass scalars (nvars = 5 + ns, reading B11 of DESIGN.md; "multispecies variant"): carried as
 * rho X_s, reconstructed as X_s, and given by each Riemann solver the flux it gives a transverse velocity.  Pinned in
 * tests/test_oracle_scalars.py.
 *
 * Communication-avoiding step (fxo_hydro_advance_ca, reading B17): one guard fill per step, stages on a
 * shrinking extension of the interior.  Pinned in tests/test_oracle_ca.py: bit for bit the result of fxo_hydro_advance.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md "Oracle pins".
 * Parity unpinned: none of the routines; the Kelvin-Helmholtz field after 100
 * steps and the config-5 field after 10 steps have no exact solution and are
 * pinned only through conservation, symmetry and the per-routine pins.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define FXO_OK 0
#define FXO_ERR_INVALID_ARG (-1)
#define FXO_ERR_STATE (-2)
#define FXO_ERR_UNSUPPORTED (-3)
#define FXO_ERR_NOMEM (-4)

#define FXO_RECON_PLM_MINMOD 0
#define FXO_RECON_WENO5 1
#define FXO_RIEMANN_HLLE 0
#define FXO_RIEMANN_HLLC 1
#define FXO_BC_OUTFLOW (-1)
#define FXO_BC_NONE (-2)
#define FXO_BC_REFLECT (-3) /* reflecting wall [B9]: mirror image of the interior, normal momentum negated */
#define FXO_NEIGH_COARSER (-4) /* the block behind this face is one level coarser (dx twice as large) [B12] */
#define FXO_NEIGH_FINER (-5)   /* 2^(ndim-1) blocks one level finer lie behind this face [B12] */
#define FXO_OPT_RHO_FLOOR 0
#define FXO_OPT_P_FLOOR 1
#define FXO_OPT_WENO_EPS 2
#define FXO_OPT_WAVESPEED 3
#define FXO_OPT_GRAVITY_X 6 /* constant acceleration g_d [B10]; 4 and 5 are options of the CUDA library only */
#define FXO_OPT_GRAVITY_Y 7
#define FXO_OPT_GRAVITY_Z 8
#define FXO_MAXV 32 /* 5 hydro variables + up to 27 passive mass scalars [B11] */
#define FXO_STATUS_NONFINITE 1u
#define FXO_STATUS_RHO_FLOOR 2u
#define FXO_STATUS_P_FLOOR 4u
#define FXO_STATUS_WENO_FALLBACK 8u

typedef struct fxo_plan {
  int n[3];       /* interior zones per block, x y z */
  int g;          /* guard depth in active dimensions */
  int gd[3];      /* guard depth per dimension (0 if inactive) [A26] */
  int np[3];      /* padded extent per dimension */
  int active[3];
  int nvars;
  int64_t nblocks;
  double gamma;
  int recon, riemann, rk;
  int64_t S_j, S_k, S_b, S_v;
  double rho_floor, p_floor, weno_eps;
  double grav[3];
  int wavespeed; /* 0 Einfeldt, 1 Davis [A8] */
  const int32_t *neigh;
  const int32_t *jump; /* refinement jumps [B12]: [nblocks][6][4], see fxo_plan_set_refinement */
  double *Fb;          /* scratch: boundary-face fluxes of the blocks with a coarser neighbour [B14] */
  unsigned long long n_nonfinite, n_rho_floor, n_p_floor, n_weno_fb;
} fxo_plan;

typedef struct fxo_layout {
  int32_t np[3];
  int32_t gd[3];
  int64_t S_j, S_k, S_b, S_v;
  int64_t bytes_per_state;
} fxo_layout;

double fxo_minmod(double a, double b);
static void fill_jump_faces(const fxo_plan *p, double *U);

/* ------------------------------------------------------------------ plan */

int fxo_plan_create(fxo_plan **out, const int dims[3], int nguard, int nvars, int64_t nblocks,
                    double gamma, int recon, int riemann, int rk_order) {
  if (!out || !dims) return FXO_ERR_INVALID_ARG;
  *out = NULL;
  if (nvars < 5 || nvars > FXO_MAXV || nblocks < 0 || !(gamma > 1.0)) return FXO_ERR_INVALID_ARG;
  if (recon != FXO_RECON_PLM_MINMOD && recon != FXO_RECON_WENO5) return FXO_ERR_INVALID_ARG;
  if (riemann != FXO_RIEMANN_HLLE && riemann != FXO_RIEMANN_HLLC) return FXO_ERR_INVALID_ARG;
  if (rk_order != 2 && rk_order != 3) return FXO_ERR_INVALID_ARG;
  if (nguard < (recon == FXO_RECON_WENO5 ? 3 : 2)) return FXO_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d)
    if (dims[d] < 1) return FXO_ERR_INVALID_ARG;
  fxo_plan *p = (fxo_plan *)calloc(1, sizeof(fxo_plan));
  if (!p) return FXO_ERR_NOMEM;
  int nactive = 0;
  for (int d = 0; d < 3; ++d) {
    p->n[d] = dims[d];
    p->active[d] = dims[d] > 1;
    if (p->active[d]) {
      ++nactive;
      if (nguard > dims[d]) {
        free(p);
        return FXO_ERR_INVALID_ARG;
      }
    }
    p->gd[d] = p->active[d] ? nguard : 0;
    p->np[d] = dims[d] + 2 * p->gd[d];
  }
  if (nactive == 0) {
    free(p);
    return FXO_ERR_INVALID_ARG;
  }
  p->g = nguard;
  p->nvars = nvars;
  p->nblocks = nblocks;
  p->gamma = gamma;
  p->recon = recon;
  p->riemann = riemann;
  p->rk = rk_order;
  p->S_j = p->np[0];
  p->S_k = (int64_t)p->np[0] * p->np[1];
  p->S_b = p->S_k * p->np[2];
  p->S_v = p->S_b * nblocks;
  p->rho_floor = 1e-12;
  p->p_floor = 1e-12;
  p->weno_eps = 1e-6;
  p->wavespeed = 0;
  *out = p;
  return FXO_OK;
}

void fxo_plan_destroy(fxo_plan *p) {
  if (p) free(p->Fb);
  free(p);
}

int fxo_plan_layout(const fxo_plan *p, fxo_layout *L) {
  if (!p || !L) return FXO_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d) {
    L->np[d] = p->np[d];
    L->gd[d] = p->gd[d];
  }
  L->S_j = p->S_j;
  L->S_k = p->S_k;
  L->S_b = p->S_b;
  L->S_v = p->S_v;
  L->bytes_per_state = p->S_v * p->nvars * (int64_t)sizeof(double);
  return FXO_OK;
}

int fxo_plan_set_option(fxo_plan *p, int key, double value) {
  if (!p) return FXO_ERR_INVALID_ARG;
  switch (key) {
  case FXO_OPT_RHO_FLOOR: p->rho_floor = value; return FXO_OK;
  case FXO_OPT_P_FLOOR: p->p_floor = value; return FXO_OK;
  case FXO_OPT_WENO_EPS: p->weno_eps = value; return FXO_OK;
  case FXO_OPT_GRAVITY_X: p->grav[0] = value; return FXO_OK;
  case FXO_OPT_GRAVITY_Y: p->grav[1] = value; return FXO_OK;
  case FXO_OPT_GRAVITY_Z: p->grav[2] = value; return FXO_OK;
  case FXO_OPT_WAVESPEED:
    if (value != 0.0 && value != 1.0) return FXO_ERR_INVALID_ARG;
    p->wavespeed = (int)value;
    return FXO_OK;
  default: return FXO_ERR_INVALID_ARG;
  }
}

int fxo_plan_set_topology(fxo_plan *p, const int32_t *neigh) {
  if (!p || (!neigh && p->nblocks > 0)) return FXO_ERR_INVALID_ARG;
  for (int64_t b = 0; b < p->nblocks; ++b)
    for (int f = 0; f < 6; ++f) {
      int32_t v = neigh[b * 6 + f];
      int d = f / 2;
      if (!p->active[d]) continue; /* entries of inactive dims are ignored [A26] */
      if (v >= 0) {
        if (v >= p->nblocks) return FXO_ERR_INVALID_ARG;
      } else if (v == FXO_NEIGH_COARSER || v == FXO_NEIGH_FINER) {
        if (!p->jump) return FXO_ERR_UNSUPPORTED; /* a jump needs the refinement table [B12] */
        int nq = v == FXO_NEIGH_COARSER ? 1 : (1 << (p->active[0] + p->active[1] + p->active[2] - 1));
        for (int q = 0; q < nq; ++q) {
          int32_t id = p->jump[(b * 6 + f) * 4 + q];
          if (id < 0 || id >= p->nblocks) return FXO_ERR_INVALID_ARG;
        }
      } else if (v != FXO_BC_OUTFLOW && v != FXO_BC_REFLECT) {
        return FXO_ERR_UNSUPPORTED;
      }
    }
  p->neigh = neigh;
  return FXO_OK;
}

/* Refinement jumps [B12] ("fine-coarse boundary resolution related API functions of the Grid unit").
 * Blocks of all levels have the same zone counts; a block one level finer has half the zone width (the caller's dx says
 * so); neighbours differ by at most one level.  neigh[b][f] = FXO_NEIGH_COARSER: jump[b][f][0] is the coarser block and
 * jump[b][f][1] says which part of its face this block abuts: bit 0 = upper half along the first transverse dimension,
 * bit 1 = along the second (transverse dimensions in ascending order; 0 for an inactive one).  neigh[b][f] =
 * FXO_NEIGH_FINER: jump[b][f][q], q = bit pattern as above, are the finer blocks.  Call before fxo_plan_set_topology.
 * Needs even block extents and nguard <= n_d / 2 in every active dimension. */
int fxo_plan_set_refinement(fxo_plan *p, const int32_t *jump) {
  if (!p) return FXO_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d)
    if (p->active[d] && (p->n[d] % 2 != 0 || 2 * p->g > p->n[d])) return FXO_ERR_INVALID_ARG;
  p->jump = jump;
  return FXO_OK;
}

int fxo_status(fxo_plan *p, uint32_t *flags, unsigned long long counts[4]) {
  if (!p || !flags) return FXO_ERR_INVALID_ARG;
  uint32_t f = 0;
  if (p->n_nonfinite) f |= FXO_STATUS_NONFINITE;
  if (p->n_rho_floor) f |= FXO_STATUS_RHO_FLOOR;
  if (p->n_p_floor) f |= FXO_STATUS_P_FLOOR;
  if (p->n_weno_fb) f |= FXO_STATUS_WENO_FALLBACK;
  *flags = f;
  if (counts) {
    counts[0] = p->n_nonfinite;
    counts[1] = p->n_rho_floor;
    counts[2] = p->n_p_floor;
    counts[3] = p->n_weno_fb;
  }
  return FXO_OK;
}

void fxo_status_reset(fxo_plan *p) {
  if (p) p->n_nonfinite = p->n_rho_floor = p->n_p_floor = p->n_weno_fb = 0;
}

/* ------------------------------------------------- regular-tiling topology */

static uint64_t morton3(uint32_t x, uint32_t y, uint32_t z) {
  uint64_t m = 0;
  for (int b = 0; b < 21; ++b) {
    m |= (uint64_t)((x >> b) & 1u) << (3 * b);
    m |= (uint64_t)((y >> b) & 1u) << (3 * b + 1);
    m |= (uint64_t)((z >> b) & 1u) << (3 * b + 2);
  }
  return m;
}

typedef struct {
  uint64_t key;
  int32_t lex;
} fxo_sortrec;

static int cmp_sortrec(const void *a, const void *b) {
  const fxo_sortrec *x = (const fxo_sortrec *)a, *y = (const fxo_sortrec *)b;
  return (x->key > y->key) - (x->key < y->key);
}

/* bc codes: 0 periodic, 1 outflow, 2 none (inactive dimension), 3 reflecting.  order: 0 lexicographic
 * (x fastest), 1 Morton.  neigh_out [nb][6], coords_out [nb][3] (block coordinates). */
int fxo_topology_cartesian(const int nb[3], const int bc_lo[3], const int bc_hi[3], int order,
                           int32_t *neigh_out, int32_t *coords_out) {
  if (!nb || !bc_lo || !bc_hi || !neigh_out) return FXO_ERR_INVALID_ARG;
  int64_t N = (int64_t)nb[0] * nb[1] * nb[2];
  if (nb[0] < 1 || nb[1] < 1 || nb[2] < 1 || N > 2147483647LL) return FXO_ERR_INVALID_ARG;
  int32_t *id_of_lex = (int32_t *)malloc((size_t)N * sizeof(int32_t));
  fxo_sortrec *rec = (fxo_sortrec *)malloc((size_t)N * sizeof(fxo_sortrec));
  if (!id_of_lex || !rec) {
    free(id_of_lex);
    free(rec);
    return FXO_ERR_NOMEM;
  }
  for (int64_t l = 0; l < N; ++l) {
    int bx = (int)(l % nb[0]), by = (int)((l / nb[0]) % nb[1]), bz = (int)(l / ((int64_t)nb[0] * nb[1]));
    rec[l].lex = (int32_t)l;
    rec[l].key = order == 1 ? morton3((uint32_t)bx, (uint32_t)by, (uint32_t)bz) : (uint64_t)l;
  }
  if (order == 1) qsort(rec, (size_t)N, sizeof(fxo_sortrec), cmp_sortrec);
  for (int64_t id = 0; id < N; ++id) id_of_lex[rec[id].lex] = (int32_t)id;
  for (int64_t id = 0; id < N; ++id) {
    int64_t l = rec[id].lex;
    int c[3] = {(int)(l % nb[0]), (int)((l / nb[0]) % nb[1]), (int)(l / ((int64_t)nb[0] * nb[1]))};
    if (coords_out)
      for (int d = 0; d < 3; ++d) coords_out[id * 3 + d] = c[d];
    for (int d = 0; d < 3; ++d)
      for (int s = 0; s < 2; ++s) {
        int bc = s ? bc_hi[d] : bc_lo[d];
        int32_t v;
        if (bc == 2) {
          v = FXO_BC_NONE;
        } else {
          int cc[3] = {c[0], c[1], c[2]};
          cc[d] += s ? 1 : -1;
          if (cc[d] < 0 || cc[d] >= nb[d]) {
            if (bc == 0) {
              cc[d] = (cc[d] + nb[d]) % nb[d];
              v = id_of_lex[((int64_t)cc[2] * nb[1] + cc[1]) * nb[0] + cc[0]];
            } else {
              v = bc == 3 ? FXO_BC_REFLECT : FXO_BC_OUTFLOW;
            }
          } else {
            v = id_of_lex[((int64_t)cc[2] * nb[1] + cc[1]) * nb[0] + cc[0]];
          }
        }
        neigh_out[id * 6 + 2 * d + s] = v;
      }
  }
  free(id_of_lex);
  free(rec);
  return FXO_OK;
}

/* --------------------------------------------------------- O1 guard fill */

/* Source of padded zone (i,j,k) of block b: hops in the order z, y, x [O1, A14].
 * Returns the flat variable-0 element index of the interior zone it images.  At a reflecting wall [B9] guard
 * zone -1-m images interior zone m (16+m images 15-m) and bit d of *flip is set: the momentum component
 * normal to that wall changes sign in the image. */
static int64_t guard_source(const fxo_plan *p, int64_t b, int i, int j, int k, unsigned *flip) {
  *flip = 0;
  int c[3] = {i, j, k};
  int64_t bs = b;
  for (int d = 2; d >= 0; --d) {
    if (!p->active[d]) continue;
    int lo = p->gd[d], hi = p->gd[d] + p->n[d];
    if (c[d] < lo) {
      int32_t nb = p->neigh[bs * 6 + 2 * d];
      if (nb >= 0) {
        bs = nb;
        c[d] += p->n[d];
      } else if (nb == FXO_BC_REFLECT) {
        c[d] = 2 * lo - 1 - c[d];
        *flip |= 1u << d;
      } else {
        c[d] = lo; /* outflow: zero-gradient clamp */
      }
    } else if (c[d] >= hi) {
      int32_t nb = p->neigh[bs * 6 + 2 * d + 1];
      if (nb >= 0) {
        bs = nb;
        c[d] -= p->n[d];
      } else if (nb == FXO_BC_REFLECT) {
        c[d] = 2 * hi - 1 - c[d];
        *flip |= 1u << d;
      } else {
        c[d] = hi - 1;
      }
    }
  }
  return bs * p->S_b + c[2] * p->S_k + c[1] * p->S_j + c[0];
}

int fxo_guardcell_index_map(fxo_plan *p, int64_t block_begin, int64_t block_count, int64_t *src) {
  if (!p || !src || block_begin < 0 || block_count < 0 || block_begin + block_count > p->nblocks)
    return FXO_ERR_INVALID_ARG;
  if (!p->neigh && p->nblocks > 0) return FXO_ERR_STATE;
  for (int64_t bb = 0; bb < block_count; ++bb)
    for (int k = 0; k < p->np[2]; ++k)
      for (int j = 0; j < p->np[1]; ++j)
        for (int i = 0; i < p->np[0]; ++i)
        {
          unsigned flip;
          src[bb * p->S_b + k * p->S_k + j * p->S_j + i] = guard_source(p, block_begin + bb, i, j, k, &flip);
        }
  return FXO_OK;
}

int fxo_fill_guardcells(fxo_plan *p, double *U) {
  if (!p || (!U && p->nblocks > 0)) return FXO_ERR_INVALID_ARG;
  if (!p->neigh && p->nblocks > 0) return FXO_ERR_STATE;
  /* Sources are always interior zones, which a fill never writes: in-place is safe. */
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < p->nblocks; ++b)
    for (int k = 0; k < p->np[2]; ++k)
      for (int j = 0; j < p->np[1]; ++j)
        for (int i = 0; i < p->np[0]; ++i) {
          int interior = i >= p->gd[0] && i < p->gd[0] + p->n[0] && j >= p->gd[1] &&
                         j < p->gd[1] + p->n[1] && k >= p->gd[2] && k < p->gd[2] + p->n[2];
          if (interior) continue;
          unsigned flip;
          int64_t s = guard_source(p, b, i, j, k, &flip);
          int64_t t = b * p->S_b + k * p->S_k + j * p->S_j + i;
          for (int v = 0; v < p->nvars; ++v) {
            double x = U[v * p->S_v + s];
            U[v * p->S_v + t] = (v >= 1 && v <= 3 && ((flip >> (v - 1)) & 1u)) ? -x : x;
          }
        }
  if (p->jump) fill_jump_faces(p, U); /* second pass: restriction / prolongation behind refinement jumps [B12, B13] */
  return FXO_OK;
}

/* ------------------------------------------- O9 fine-coarse boundaries [B12, B13] */

/* Variable v of the zone at INTERIOR coordinates c (0-based) of block cb, where at most one coordinate may lie outside
 * [0, n): then the zone is resolved by ONE hop through that face -- the same-level neighbour's interior zone, the clamp
 * (outflow), the mirror zone (wall; normal momentum negated), or, behind a face with finer neighbours, the RESTRICTION
 * of their interior zones: the plain mean of the 2^ndim children, summed in the order i fastest, then j, then k [B13].
 * Behind a face with a coarser neighbour nothing is defined here: returns 0 (and 1 otherwise).  A pure function of
 * interior data, so fills can run in any order. */
static int amr_zone(const fxo_plan *p, const double *X, int64_t cb, const int cin[3], int v, double *val) {
  int c[3] = {cin[0], cin[1], cin[2]};
  double sign = 1.0;
  for (int d = 0; d < 3; ++d) {
    if (c[d] >= 0 && c[d] < p->n[d]) continue;
    int side = c[d] >= p->n[d];
    int f = 2 * d + side;
    int32_t nb = p->neigh[cb * 6 + f];
    if (nb >= 0) {
      cb = nb;
      c[d] += side ? -p->n[d] : p->n[d];
    } else if (nb == FXO_BC_REFLECT) {
      c[d] = side ? 2 * p->n[d] - 1 - c[d] : -1 - c[d];
      if (v == 1 + d) sign = -1.0;
    } else if (nb == FXO_NEIGH_FINER) {
      int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2; /* transverse dimensions, ascending */
      int q = 0, fc[3], cnt[3];
      int tr[2] = {d1, d2};
      for (int t = 0; t < 2; ++t) {
        int e = tr[t];
        if (!p->active[e]) { fc[e] = 0; cnt[e] = 1; continue; }
        int half = c[e] >= p->n[e] / 2;
        q |= half << t;
        fc[e] = 2 * (c[e] - half * (p->n[e] / 2));
        cnt[e] = 2;
      }
      int m = side ? c[d] - p->n[d] : -1 - c[d]; /* distance behind the face, 0 = adjacent */
      fc[d] = side ? 2 * m : p->n[d] - 2 - 2 * m;
      cnt[d] = 2;
      int64_t fb = p->jump[(cb * 6 + f) * 4 + q];
      double sum = 0.0;
      for (int kk = 0; kk < cnt[2]; ++kk)
        for (int jj = 0; jj < cnt[1]; ++jj)
          for (int ii = 0; ii < cnt[0]; ++ii)
            sum += X[v * p->S_v + fb * p->S_b + (int64_t)(fc[2] + kk + p->gd[2]) * p->S_k +
                     (int64_t)(fc[1] + jj + p->gd[1]) * p->S_j + (fc[0] + ii + p->gd[0])];
      *val = sum * (1.0 / (double)(cnt[0] * cnt[1] * cnt[2]));
      return 1;
    } else if (nb == FXO_NEIGH_COARSER) {
      return 0;
    } else {
      c[d] = side ? p->n[d] - 1 : 0; /* outflow */
    }
    break; /* one hop */
  }
  *val = sign * X[v * p->S_v + cb * p->S_b + (int64_t)(c[2] + p->gd[2]) * p->S_k + (int64_t)(c[1] + p->gd[1]) * p->S_j +
                  (c[0] + p->gd[0])];
  return 1;
}

/* Face guard zones behind refinement jumps [B12, B13], after the same-level fill: for every block face with finer
 * neighbours the guard zones are the restriction of the fine interiors; for every face with a coarser neighbour they are
 * PROLONGED from the parent coarse zone C: q = q_C + sum over active d of sigma_d (1/4) minmod(q_C - q_{C-e_d},
 * q_{C+e_d} - q_C), sigma_d = +-1 the child's side of C along d, the neighbours of C resolved by amr_zone (a neighbour that
 * lies behind a coarser jump is not defined: that slope is 0).  Conserved variables, all of them; the children of a zone
 * average to the zone.  Only zones outside the block in exactly ONE dimension are written (the stage reads no others
 * [A11]); edge and corner zones next to a jump keep the clamp of the first pass. */
static void fill_jump_faces(const fxo_plan *p, double *U) {
#pragma omp parallel for schedule(static)
  for (int64_t b = 0; b < p->nblocks; ++b)
    for (int f = 0; f < 6; ++f) {
      int d = f / 2, side = f & 1;
      if (!p->active[d]) continue;
      int32_t code = p->neigh[b * 6 + f];
      if (code != FXO_NEIGH_COARSER && code != FXO_NEIGH_FINER) continue;
      int d1 = d == 0 ? 1 : 0, d2 = d == 2 ? 1 : 2;
      for (int m = 0; m < p->gd[d]; ++m)
        for (int t2 = 0; t2 < p->n[d2]; ++t2)
          for (int t1 = 0; t1 < p->n[d1]; ++t1) {
            int c[3];
            c[d] = side ? p->n[d] + m : -1 - m;
            c[d1] = t1;
            c[d2] = t2;
            int64_t t = b * p->S_b + (int64_t)(c[2] + p->gd[2]) * p->S_k + (int64_t)(c[1] + p->gd[1]) * p->S_j + (c[0] + p->gd[0]);
            for (int v = 0; v < p->nvars; ++v) {
              double val = 0.0;
              if (code == FXO_NEIGH_FINER) {
                amr_zone(p, U, b, c, v, &val);
              } else {
                int64_t cb = p->jump[(b * 6 + f) * 4 + 0];
                int qd = p->jump[(b * 6 + f) * 4 + 1];
                int C[3] = {0, 0, 0};
                double sg[3] = {0.0, 0.0, 0.0};
                C[d] = side ? m / 2 : p->n[d] - 1 - m / 2;
                sg[d] = ((m % 2 == 0) == (side == 0)) ? 1.0 : -1.0; /* the child next to the face is the one on the face's side */
                int tr[2] = {d1, d2}, tc[2] = {t1, t2};
                for (int t_ = 0; t_ < 2; ++t_) {
                  int e = tr[t_];
                  if (!p->active[e]) continue;
                  C[e] = ((qd >> t_) & 1) * (p->n[e] / 2) + tc[t_] / 2;
                  sg[e] = (tc[t_] % 2) ? 1.0 : -1.0;
                }
                double qC;
                amr_zone(p, U, cb, C, v, &qC);
                val = qC;
                for (int e = 0; e < 3; ++e) {
                  if (!p->active[e]) continue;
                  int Cm[3] = {C[0], C[1], C[2]}, Cp[3] = {C[0], C[1], C[2]};
                  Cm[e] -= 1;
                  Cp[e] += 1;
                  double qm, qp;
                  if (amr_zone(p, U, cb, Cm, v, &qm) && amr_zone(p, U, cb, Cp, v, &qp))
                    val += (sg[e] * 0.25) * fxo_minmod(qC - qm, qp - qC);
                }
              }
              U[v * p->S_v + t] = val;
            }
          }
    }
}

/* ---------------------------------------------------- O2 cons -> prim */

/* U = (rho, mx, my, mz, E, rho X_1 ..) -> W = (rho, u, v, w, p, X_1 ..).  Floors touch primitives only [A7].
 * Passive mass scalars [B11]: X_s = (rho X_s) / rho with the same (floored) density the velocities use; nv = 5 + ns. */
static void cons2prim(const fxo_plan *p, int nv, const double *U, double *W, unsigned *hit) {
  double rho = U[0];
  if (rho < p->rho_floor) { /* NaN compares false and stays NaN */
    rho = p->rho_floor;
    *hit |= FXO_STATUS_RHO_FLOOR;
  }
  double r = 1.0 / rho;
  double u = U[1] * r, v = U[2] * r, w = U[3] * r;
  double pr = (p->gamma - 1.0) * (U[4] - 0.5 * (U[1] * u + U[2] * v + U[3] * w));
  if (pr < p->p_floor) {
    pr = p->p_floor;
    *hit |= FXO_STATUS_P_FLOOR;
  }
  W[0] = rho;
  W[1] = u;
  W[2] = v;
  W[3] = w;
  W[4] = pr;
  if (!isfinite(rho) || !isfinite(u) || !isfinite(v) || !isfinite(w) || !isfinite(pr))
    *hit |= FXO_STATUS_NONFINITE;
  for (int s = 5; s < nv; ++s) {
    W[s] = U[s] * r;
    if (!isfinite(W[s])) *hit |= FXO_STATUS_NONFINITE;
  }
}

void fxo_cons2prim(const fxo_plan *p, const double U[5], double W[5]) {
  unsigned hit = 0;
  cons2prim(p, 5, U, W, &hit);
}

/* The same with the plan's passive scalars: U and W hold p->nvars entries [B11]. */
void fxo_cons2prim_nv(const fxo_plan *p, const double *U, double *W) {
  unsigned hit = 0;
  cons2prim(p, p->nvars, U, W, &hit);
}

/* ------------------------------------------------- O3 reconstruction */

/* minmod in comparison form [A4]: no products, NaN -> 0. */
double fxo_minmod(double a, double b) {
  if (a > 0.0 && b > 0.0) return a < b ? a : b;
  if (a < 0.0 && b < 0.0) return a > b ? a : b;
  return 0.0;
}

/* WENO5-JS value at the +1/2 face of the cell holding c, from cell values a..e (textbook,
 * Jiang & Shu 1996) [O3, A5].  eps absolute, exponent 2. */
double fxo_weno5(double a, double b, double c, double d, double e, double eps) {
  const double sixth = 1.0 / 6.0;
  double p0 = (2.0 * a - 7.0 * b + 11.0 * c) * sixth;
  double p1 = (-b + 5.0 * c + 2.0 * d) * sixth;
  double p2 = (2.0 * c + 5.0 * d - e) * sixth;
  double t0 = a - 2.0 * b + c, u0 = a - 4.0 * b + 3.0 * c;
  double t1 = b - 2.0 * c + d, u1 = b - d;
  double t2 = c - 2.0 * d + e, u2 = 3.0 * c - 4.0 * d + e;
  double b0 = (13.0 / 12.0) * (t0 * t0) + 0.25 * (u0 * u0);
  double b1 = (13.0 / 12.0) * (t1 * t1) + 0.25 * (u1 * u1);
  double b2 = (13.0 / 12.0) * (t2 * t2) + 0.25 * (u2 * u2);
  double a0 = 0.1 / ((eps + b0) * (eps + b0));
  double a1 = 0.6 / ((eps + b1) * (eps + b1));
  double a2 = 0.3 / ((eps + b2) * (eps + b2));
  return (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
}

/* Left and right primitive states at the face between padded cells iL and iR = iL + 1 along a
 * line of stride s in the primitive array W (nv slabs of size slab; every component, passive scalars
 * included [B11], is reconstructed the same way and the positivity fallback replaces all of them). */
static void reconstruct_face(const fxo_plan *p, int nv, const double *W, int64_t slab, int64_t cL, int64_t s,
                             double *WL, double *WR, unsigned *hit) {
  int64_t cR = cL + s;
  if (p->recon == FXO_RECON_PLM_MINMOD) {
    for (int v = 0; v < nv; ++v) {
      const double *q = W + v * slab;
      double dL = fxo_minmod(q[cL] - q[cL - s], q[cL + s] - q[cL]);
      double dR = fxo_minmod(q[cR] - q[cR - s], q[cR + s] - q[cR]);
      WL[v] = q[cL] + 0.5 * dL;
      WR[v] = q[cR] - 0.5 * dR;
    }
  } else {
    for (int v = 0; v < nv; ++v) {
      const double *q = W + v * slab;
      WL[v] = fxo_weno5(q[cL - 2 * s], q[cL - s], q[cL], q[cL + s], q[cL + 2 * s], p->weno_eps);
      WR[v] = fxo_weno5(q[cR + 2 * s], q[cR + s], q[cR], q[cR - s], q[cR - 2 * s], p->weno_eps);
    }
    /* positivity fallback, per side [A6] */
    if (!(WL[0] > 0.0) || !(WL[4] > 0.0)) {
      for (int v = 0; v < nv; ++v) WL[v] = W[v * slab + cL];
      *hit |= FXO_STATUS_WENO_FALLBACK;
    }
    if (!(WR[0] > 0.0) || !(WR[4] > 0.0)) {
      for (int v = 0; v < nv; ++v) WR[v] = W[v * slab + cR];
      *hit |= FXO_STATUS_WENO_FALLBACK;
    }
  }
}

/* Test hook: the face states [O3, A6] at the face between cells cL and cL + s of a line of primitives
 * W[v * slab + cell] (a call of reconstruct_face, nothing else); *hit receives the status bits it raises. */
void fxo_face_states(const fxo_plan *p, const double *W, int64_t slab, int64_t cL, int64_t s, double *WL, double *WR,
                     unsigned *hit) {
  *hit = 0;
  reconstruct_face(p, p->nvars, W, slab, cL, s, WL, WR, hit);
}

/* ---------------------------------------------------- O4 Riemann flux */

/* States in the face frame: W = (rho, un, ut1, ut2, p); flux F = (mass, normal momentum,
 * t1 momentum, t2 momentum, energy).  Einfeldt (Roe-average) or Davis wave-speed bounds [A8];
 * HLLE in branching form [A10]; Toro's HLLC with the test order of O4 [A9]. */
/* Passive scalars [B11]: W[5 + s] = X_s, U = rho X_s, F = (rho un) X_s -- each solver treats X_s exactly as it
 * treats a transverse velocity (an advected quantity): upwind flux when supersonic, the HLL average for HLLE,
 * rho* X_K in the star state of HLLC (which makes the flux X_K times the mass flux). */
static void riemann_flux(const fxo_plan *p, int nv, const double *WL, const double *WR, double *F) {
  const double gam = p->gamma, gm1 = p->gamma - 1.0, igm1 = 1.0 / (p->gamma - 1.0);
  double rL = WL[0], unL = WL[1], t1L = WL[2], t2L = WL[3], pL = WL[4];
  double rR = WR[0], unR = WR[1], t1R = WR[2], t2R = WR[3], pR = WR[4];
  double irL = 1.0 / rL, irR = 1.0 / rR;
  double cL = sqrt(gam * pL * irL), cR = sqrt(gam * pR * irR);
  double EL = pL * igm1 + 0.5 * rL * (unL * unL + t1L * t1L + t2L * t2L);
  double ER = pR * igm1 + 0.5 * rR * (unR * unR + t1R * t1R + t2R * t2R);
  double UL[FXO_MAXV]; /* entries 5.. are the scalars, set below */
  UL[0] = rL;
  UL[1] = rL * unL;
  UL[2] = rL * t1L;
  UL[3] = rL * t2L;
  UL[4] = EL;
  double UR[FXO_MAXV]; /* entries 5.. are the scalars, set below */
  UR[0] = rR;
  UR[1] = rR * unR;
  UR[2] = rR * t1R;
  UR[3] = rR * t2R;
  UR[4] = ER;
  double FL[FXO_MAXV]; /* entries 5.. are the scalars, set below */
  FL[0] = UL[1];
  FL[1] = UL[1] * unL + pL;
  FL[2] = UL[1] * t1L;
  FL[3] = UL[1] * t2L;
  FL[4] = unL * (EL + pL);
  double FR[FXO_MAXV]; /* entries 5.. are the scalars, set below */
  FR[0] = UR[1];
  FR[1] = UR[1] * unR + pR;
  FR[2] = UR[1] * t1R;
  FR[3] = UR[1] * t2R;
  FR[4] = unR * (ER + pR);
  for (int s = 5; s < nv; ++s) {
    UL[s] = rL * WL[s];
    UR[s] = rR * WR[s];
    FL[s] = UL[1] * WL[s];
    FR[s] = UR[1] * WR[s];
  }
  double SL, SR;
  if (p->wavespeed == 0) {
    double HL = (EL + pL) * irL, HR = (ER + pR) * irR;
    double sl = sqrt(rL), sr = sqrt(rR);
    double wi = 1.0 / (sl + sr);
    double un = (sl * unL + sr * unR) * wi;
    double t1 = (sl * t1L + sr * t1R) * wi;
    double t2 = (sl * t2L + sr * t2R) * wi;
    double H = (sl * HL + sr * HR) * wi;
    double c = sqrt(gm1 * (H - 0.5 * (un * un + t1 * t1 + t2 * t2)));
    double a = unL - cL, b = un - c;
    SL = a < b ? a : b;
    a = unR + cR;
    b = un + c;
    SR = a > b ? a : b;
  } else {
    double a = unL - cL, b = unR - cR;
    SL = a < b ? a : b;
    a = unL + cL;
    b = unR + cR;
    SR = a > b ? a : b;
  }
  if (SL >= 0.0) {
    for (int v = 0; v < nv; ++v) F[v] = FL[v];
    return;
  }
  if (SR <= 0.0) {
    for (int v = 0; v < nv; ++v) F[v] = FR[v];
    return;
  }
  if (p->riemann == FXO_RIEMANN_HLLE) {
    double den = SR - SL, ss = SL * SR;
    for (int v = 0; v < nv; ++v) F[v] = (SR * FL[v] - SL * FR[v] + ss * (UR[v] - UL[v])) / den;
    return;
  }
  /* HLLC */
  double aL = rL * (SL - unL), aR = rR * (SR - unR);
  double Ss = ((pR - pL) + (aL * unL - aR * unR)) / (aL - aR);
  if (Ss >= 0.0) {
    double f = aL / (SL - Ss);
    double Us[FXO_MAXV]; /* entries 5.. are the scalars, set below */
    Us[0] = f;
    Us[1] = f * Ss;
    Us[2] = f * t1L;
    Us[3] = f * t2L;
    Us[4] = f * (EL * irL + (Ss - unL) * (Ss + pL / aL));
    for (int s = 5; s < nv; ++s) Us[s] = f * WL[s];
    for (int v = 0; v < nv; ++v) F[v] = FL[v] + SL * (Us[v] - UL[v]);
  } else {
    double f = aR / (SR - Ss);
    double Us[FXO_MAXV]; /* entries 5.. are the scalars, set below */
    Us[0] = f;
    Us[1] = f * Ss;
    Us[2] = f * t1R;
    Us[3] = f * t2R;
    Us[4] = f * (ER * irR + (Ss - unR) * (Ss + pR / aR));
    for (int s = 5; s < nv; ++s) Us[s] = f * WR[s];
    for (int v = 0; v < nv; ++v) F[v] = FR[v] + SR * (Us[v] - UR[v]);
  }
}

/* Public, for the per-routine pins: states and flux in the face frame (rho, un, ut1, ut2, p). */
void fxo_riemann_flux(const fxo_plan *p, const double WL[5], const double WR[5], double F[5]) {
  riemann_flux(p, 5, WL, WR, F);
}

/* The same with the plan's passive scalars: WL, WR, F hold p->nvars entries [B11]. */
void fxo_riemann_flux_nv(const fxo_plan *p, const double *WL, const double *WR, double *F) {
  riemann_flux(p, p->nvars, WL, WR, F);
}

/* ------------------------------------------------ O5 spatial operator */

/* Face flux in direction d at the face whose left cell has flat in-block index cL, returned in
 * the un-rotated variable order (rho, mx, my, mz, E, scalars). */
static void face_flux(const fxo_plan *p, const double *W, int64_t slab, int64_t cL, int d, double *F,
                      unsigned *hit) {
  const int nv = p->nvars;
  const int64_t stride[3] = {1, p->S_j, p->S_k};
  /* frame of direction d: normal = d, t1 = (d+1)%3, t2 = (d+2)%3 */
  int in = 1 + d, it1 = 1 + (d + 1) % 3, it2 = 1 + (d + 2) % 3;
  double WLu[FXO_MAXV], WRu[FXO_MAXV], WLf[FXO_MAXV], WRf[FXO_MAXV], Ff[FXO_MAXV];
  reconstruct_face(p, nv, W, slab, cL, stride[d], WLu, WRu, hit);
  WLf[0] = WLu[0]; WLf[1] = WLu[in]; WLf[2] = WLu[it1]; WLf[3] = WLu[it2]; WLf[4] = WLu[4];
  WRf[0] = WRu[0]; WRf[1] = WRu[in]; WRf[2] = WRu[it1]; WRf[3] = WRu[it2]; WRf[4] = WRu[4];
  for (int s = 5; s < nv; ++s) {
    WLf[s] = WLu[s];
    WRf[s] = WRu[s];
  }
  riemann_flux(p, nv, WLf, WRf, Ff);
  for (int s = 5; s < nv; ++s) F[s] = Ff[s];
  F[0] = Ff[0];
  F[in] = Ff[1];
  F[it1] = Ff[2];
  F[it2] = Ff[3];
  F[4] = Ff[4];
  for (int v = 0; v < nv; ++v)
    if (!isfinite(F[v])) *hit |= FXO_STATUS_NONFINITE;
}

static void count_hits(fxo_plan *p, unsigned hit, unsigned long long n) {
  if (!hit) return;
  if (hit & FXO_STATUS_NONFINITE) {
#pragma omp atomic
    p->n_nonfinite += n;
  }
  if (hit & FXO_STATUS_RHO_FLOOR) {
#pragma omp atomic
    p->n_rho_floor += n;
  }
  if (hit & FXO_STATUS_P_FLOOR) {
#pragma omp atomic
    p->n_p_floor += n;
  }
  if (hit & FXO_STATUS_WENO_FALLBACK) {
#pragma omp atomic
    p->n_weno_fb += n;
  }
}

/* Primitives of every padded zone of block b of X into W[nvars][S_b] (guards must be filled). */
static void block_prims(fxo_plan *p, const double *X, int64_t b, double *W) {
  for (int k = 0; k < p->np[2]; ++k)
    for (int j = 0; j < p->np[1]; ++j)
      for (int i = 0; i < p->np[0]; ++i) {
        int64_t c = k * p->S_k + j * p->S_j + i;
        double U[FXO_MAXV], Wz[FXO_MAXV];
        for (int v = 0; v < p->nvars; ++v) U[v] = X[v * p->S_v + b * p->S_b + c];
        unsigned hit = 0;
        cons2prim(p, p->nvars, U, Wz, &hit);
        for (int v = 0; v < p->nvars; ++v) W[v * p->S_b + c] = Wz[v];
        int interior = i >= p->gd[0] && i < p->gd[0] + p->n[0] && j >= p->gd[1] &&
                       j < p->gd[1] + p->n[1] && k >= p->gd[2] && k < p->gd[2] + p->n[2];
        if (interior) count_hits(p, hit, 1); /* count each zone once, where it is owned */
      }
}

/* One RK stage on block b: out = U0 + beta*((X - U0) - S(X)), S = sum_d (dt/dx_d)(F+ - F-)
 * summed in the order x, y, z [O5, O6], minus dt times the constant-gravity source of the stage input [B10]:
 * (0, rho g_x, rho g_y, rho g_z, g . m) from the zone's conserved values (none for the scalars [B11]).  W and Fline
 * are per-thread scratch. */
static void block_stage(fxo_plan *p, const double *X, const double *U0, double *out, int64_t b,
                        const double *dx, double dt, double beta, int first, double *W, double *S,
                        double *Fline) {
  const int nv = p->nvars;
  block_prims(p, X, b, W);
  const int64_t stride[3] = {1, p->S_j, p->S_k};
  memset(S, 0, sizeof(double) * (size_t)nv * (size_t)p->S_b);
  for (int d = 0; d < 3; ++d) {
    if (!p->active[d]) continue;
    double r = dt / dx[b * 3 + d];
    int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    for (int a2 = p->gd[d2]; a2 < p->gd[d2] + p->n[d2]; ++a2)
      for (int a1 = p->gd[d1]; a1 < p->gd[d1] + p->n[d1]; ++a1) {
        int64_t base = a1 * stride[d1] + a2 * stride[d2];
        unsigned hit = 0;
        for (int f = 0; f <= p->n[d]; ++f) {
          int64_t cL = base + (int64_t)(p->gd[d] + f - 1) * stride[d];
          face_flux(p, W, p->S_b, cL, d, Fline + nv * f, &hit);
        }
        count_hits(p, hit & (FXO_STATUS_NONFINITE | FXO_STATUS_WENO_FALLBACK), 1);
        /* flux correction [B14]: at a face with finer neighbours the flux of a coarse face is the mean of the fluxes
         * of the 2^(ndim-1) fine faces that cover it (computed by the fine blocks from their prolonged guard zones),
         * so that what leaves the fine blocks enters the coarse one */
        for (int side = 0; side < 2; ++side)
          if (p->jump && p->neigh[b * 6 + 2 * d + side] == FXO_NEIGH_FINER) {
            int lo1 = d == 0 ? 1 : 0, lo2 = d == 2 ? 1 : 2; /* transverse dimensions, ascending */
            int tc[3];
            tc[d1] = a1 - p->gd[d1];
            tc[d2] = a2 - p->gd[d2];
            int tr[2] = {lo1, lo2}, q = 0, ft[2] = {0, 0}, cnt[2] = {1, 1};
            for (int t = 0; t < 2; ++t) {
              int e = tr[t];
              if (!p->active[e]) continue;
              int half = tc[e] >= p->n[e] / 2;
              q |= half << t;
              ft[t] = 2 * (tc[e] - half * (p->n[e] / 2));
              cnt[t] = 2;
            }
            int64_t fb = p->jump[(b * 6 + 2 * d + side) * 4 + q];
            int ff = 2 * d + (1 - side); /* the fine block's face that touches ours */
            int64_t A = (int64_t)p->n[lo1] * p->n[lo2];
            for (int v = 0; v < nv; ++v) {
              double sum = 0.0;
              for (int j2 = 0; j2 < cnt[1]; ++j2)
                for (int j1 = 0; j1 < cnt[0]; ++j1)
                  sum += p->Fb[((fb * 6 + ff) * nv + v) * A + (int64_t)(ft[1] + j2) * p->n[lo1] + (ft[0] + j1)];
              Fline[nv * (side ? p->n[d] : 0) + v] = sum * (1.0 / (double)(cnt[0] * cnt[1]));
            }
          }
        for (int f = 0; f < p->n[d]; ++f) {
          int64_t c = base + (int64_t)(p->gd[d] + f) * stride[d];
          for (int v = 0; v < nv; ++v) S[v * p->S_b + c] += r * (Fline[nv * (f + 1) + v] - Fline[nv * f + v]);
        }
      }
  }
  for (int k = p->gd[2]; k < p->gd[2] + p->n[2]; ++k)
    for (int j = p->gd[1]; j < p->gd[1] + p->n[1]; ++j)
      for (int i = p->gd[0]; i < p->gd[0] + p->n[0]; ++i) {
        int64_t c = k * p->S_k + j * p->S_j + i;
        if (p->grav[0] != 0.0 || p->grav[1] != 0.0 || p->grav[2] != 0.0) {
          int64_t z = b * p->S_b + c;
          double rho = X[z], gm = 0.0;
          for (int d = 0; d < 3; ++d) {
            S[(1 + d) * p->S_b + c] -= dt * (rho * p->grav[d]);
            gm += p->grav[d] * X[(1 + d) * p->S_v + z];
          }
          S[4 * p->S_b + c] -= dt * gm;
        }
        for (int v = 0; v < nv; ++v) {
          int64_t g = v * p->S_v + b * p->S_b + c;
          if (first)
            out[g] = U0[g] - S[v * p->S_b + c];
          else
            out[g] = U0[g] + beta * ((X[g] - U0[g]) - S[v * p->S_b + c]);
        }
      }
}

static int run_stage(fxo_plan *p, double *X, const double *U0, double *out, const double *dx, double dt,
                     double beta, int first) {
  int rc = fxo_fill_guardcells(p, X); /* O1 on the stage input before every S(.) [A15] */
  if (rc) return rc;
  int fail = 0;
  if (p->jump) { /* [B14] first the boundary-face fluxes of every block face that has a coarser neighbour */
    int nmx = p->n[0] > p->n[1] ? p->n[0] : p->n[1];
    if (p->n[2] > nmx) nmx = p->n[2];
    if (!p->Fb) p->Fb = (double *)malloc(sizeof(double) * (size_t)p->nblocks * 6 * (size_t)p->nvars * (size_t)nmx * (size_t)nmx);
    if (!p->Fb) return FXO_ERR_NOMEM;
#pragma omp parallel
    {
      double *W = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
#pragma omp for schedule(dynamic, 4)
      for (int64_t b = 0; b < p->nblocks; ++b) {
        int any = 0;
        for (int f = 0; f < 6; ++f) any |= p->active[f / 2] && p->neigh[b * 6 + f] == FXO_NEIGH_COARSER;
        if (!any || !W) continue;
        block_prims(p, X, b, W);
        const int64_t stride[3] = {1, p->S_j, p->S_k};
        for (int f = 0; f < 6; ++f) {
          int d = f / 2, side = f & 1;
          if (!p->active[d] || p->neigh[b * 6 + f] != FXO_NEIGH_COARSER) continue;
          int lo1 = d == 0 ? 1 : 0, lo2 = d == 2 ? 1 : 2;
          int64_t A = (int64_t)p->n[lo1] * p->n[lo2];
          for (int t2 = 0; t2 < p->n[lo2]; ++t2)
            for (int t1 = 0; t1 < p->n[lo1]; ++t1) {
              int c[3];
              c[d] = p->gd[d] + (side ? p->n[d] : 0) - 1; /* left cell of the face */
              c[lo1] = t1 + p->gd[lo1];
              c[lo2] = t2 + p->gd[lo2];
              double Ff[FXO_MAXV];
              unsigned hit = 0;
              face_flux(p, W, p->S_b, c[2] * stride[2] + c[1] * stride[1] + c[0], d, Ff, &hit);
              for (int v = 0; v < p->nvars; ++v) p->Fb[((b * 6 + f) * p->nvars + v) * A + (int64_t)t2 * p->n[lo1] + t1] = Ff[v];
            }
        }
      }
      free(W);
    }
  }
#pragma omp parallel
  {
    double *W = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
    double *S = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
    int nmax = p->n[0] > p->n[1] ? p->n[0] : p->n[1];
    if (p->n[2] > nmax) nmax = p->n[2];
    double *Fl = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)(nmax + 1));
    if (!W || !S || !Fl) {
#pragma omp atomic write
      fail = 1;
    } else {
#pragma omp for schedule(dynamic, 4)
      for (int64_t b = 0; b < p->nblocks; ++b) block_stage(p, X, U0, out, b, dx, dt, beta, first, W, S, Fl);
    }
    free(W);
    free(S);
    free(Fl);
  }
  return fail ? FXO_ERR_NOMEM : FXO_OK;
}

/* Forward-Euler stage U <- U - S(U) (used by tests to compose the SSP-RK schemes). */
int fxo_euler_step(fxo_plan *p, double *U, const double *dx, double dt) {
  if (!p || (!U && p->nblocks) || (!dx && p->nblocks)) return FXO_ERR_INVALID_ARG;
  if (!p->neigh && p->nblocks > 0) return FXO_ERR_STATE;
  size_t n = (size_t)p->S_v * (size_t)p->nvars;
  double *U1 = (double *)malloc(sizeof(double) * (n ? n : 1));
  if (!U1) return FXO_ERR_NOMEM;
  int rc = run_stage(p, U, U, U1, dx, dt, 1.0, 1);
  if (!rc) {
    /* copy interiors back (guards of U keep the fill) */
    for (int64_t b = 0; b < p->nblocks; ++b)
      for (int k = p->gd[2]; k < p->gd[2] + p->n[2]; ++k)
        for (int j = p->gd[1]; j < p->gd[1] + p->n[1]; ++j)
          for (int i = p->gd[0]; i < p->gd[0] + p->n[0]; ++i)
            for (int v = 0; v < p->nvars; ++v) {
              int64_t g = v * p->S_v + b * p->S_b + k * p->S_k + j * p->S_j + i;
              U[g] = U1[g];
            }
  }
  free(U1);
  return rc;
}

/* O6: one SSP-RK step (Shu-Osher in increment form [A12]), in place on the interior of U. */
int fxo_hydro_advance(fxo_plan *p, double *U, const double *dx, double dt) {
  if (!p || (!U && p->nblocks) || (!dx && p->nblocks)) return FXO_ERR_INVALID_ARG;
  if (!(dt > 0.0) || !isfinite(dt)) return FXO_ERR_INVALID_ARG;
  if (!p->neigh && p->nblocks > 0) return FXO_ERR_STATE;
  if (p->nblocks == 0) return FXO_OK;
  size_t n = (size_t)p->S_v * (size_t)p->nvars;
  double *U1 = (double *)malloc(sizeof(double) * n);
  double *U2 = p->rk == 3 ? (double *)malloc(sizeof(double) * n) : NULL;
  if (!U1 || (p->rk == 3 && !U2)) {
    free(U1);
    free(U2);
    return FXO_ERR_NOMEM;
  }
  /* guards of U1/U2 are filled by run_stage before they are read; interiors are fully written */
  memset(U1, 0, sizeof(double) * n);
  if (U2) memset(U2, 0, sizeof(double) * n);
  int rc = run_stage(p, U, U, U1, dx, dt, 1.0, 1); /* U1 = U0 - S(U0) */
  if (!rc && p->rk == 2) {
    rc = run_stage(p, U1, U, U, dx, dt, 0.5, 0); /* U = U0 + 1/2((U1-U0) - S(U1)) */
  } else if (!rc) {
    rc = run_stage(p, U1, U, U2, dx, dt, 0.25, 0); /* U2 = U0 + 1/4((U1-U0) - S(U1)) */
    if (!rc) rc = run_stage(p, U2, U, U, dx, dt, 2.0 / 3.0, 0); /* U = U0 + 2/3((U2-U0) - S(U2)) */
  }
  free(U1);
  free(U2);
  return rc;
}

/* ------------------------------------------- O10 communication-avoiding step [B17; SURVEY 8(f) NEXT-4]
 *
 * The same SSP-RK step with ONE guard fill: O1 fills every guard zone of U0 (edges and corners too) once; stage s of n
 * then updates the interior EXTENDED by E_s = (n - s) R zones in every active dimension (the whole box, edge and corner
 * zones of the extension included), R = 2 (PLM) or 3 (WENO5) being the reach of one S(.), reading its stencils in place
 * from the padded array: the stage input is known on the box extended by E_s + R = E_(s-1) -- the filled U0 for s = 1
 * (n R <= nguard needed), the previous stage's result after that.  Behind a face with a same-level neighbour the extended
 * zones are the neighbour's interior zones, updated with the same formula from the same numbers (the blocks must share
 * dx): they carry what a fill of the stage result would copy there.  Behind a physical boundary that is not so: O1 of the
 * stage result puts the boundary's IMAGE of the result there (clamp, or mirror with the normal momentum negated), so after
 * each stage but the last those zones are re-imaged from the block's own zones -- local work, no neighbour is read. */

/* Stage on block b over the interior extended by E zones in every active dimension; stencils in place from X. */
static void block_stage_ext(fxo_plan *p, const double *X, const double *U0, double *out, int64_t b, const double *dx,
                            double dt, double beta, int first, int E, double *W, double *S, double *Fline) {
  const int nv = p->nvars;
  block_prims(p, X, b, W);
  const int64_t stride[3] = {1, p->S_j, p->S_k};
  int lo[3], hi[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = p->gd[d] - (p->active[d] ? E : 0);
    hi[d] = p->gd[d] + p->n[d] + (p->active[d] ? E : 0);
  }
  memset(S, 0, sizeof(double) * (size_t)nv * (size_t)p->S_b);
  for (int d = 0; d < 3; ++d) {
    if (!p->active[d]) continue;
    double r = dt / dx[b * 3 + d];
    int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    int nf = hi[d] - lo[d]; /* zones along d; faces 0 .. nf */
    for (int a2 = lo[d2]; a2 < hi[d2]; ++a2)
      for (int a1 = lo[d1]; a1 < hi[d1]; ++a1) {
        int64_t base = a1 * stride[d1] + a2 * stride[d2];
        unsigned hit = 0;
        for (int f = 0; f <= nf; ++f) face_flux(p, W, p->S_b, base + (int64_t)(lo[d] + f - 1) * stride[d], d, Fline + nv * f, &hit);
        count_hits(p, hit & (FXO_STATUS_NONFINITE | FXO_STATUS_WENO_FALLBACK), 1);
        for (int f = 0; f < nf; ++f) {
          int64_t c = base + (int64_t)(lo[d] + f) * stride[d];
          for (int v = 0; v < nv; ++v) S[v * p->S_b + c] += r * (Fline[nv * (f + 1) + v] - Fline[nv * f + v]);
        }
      }
  }
  for (int k = lo[2]; k < hi[2]; ++k)
    for (int j = lo[1]; j < hi[1]; ++j)
      for (int i = lo[0]; i < hi[0]; ++i) {
        int64_t c = k * p->S_k + j * p->S_j + i;
        if (p->grav[0] != 0.0 || p->grav[1] != 0.0 || p->grav[2] != 0.0) {
          int64_t z = b * p->S_b + c;
          double rho = X[z], gm = 0.0;
          for (int d = 0; d < 3; ++d) {
            S[(1 + d) * p->S_b + c] -= dt * (rho * p->grav[d]);
            gm += p->grav[d] * X[(1 + d) * p->S_v + z];
          }
          S[4 * p->S_b + c] -= dt * gm;
        }
        for (int v = 0; v < nv; ++v) {
          int64_t g = v * p->S_v + b * p->S_b + c;
          if (first)
            out[g] = U0[g] - S[v * p->S_b + c];
          else
            out[g] = U0[g] + beta * ((X[g] - U0[g]) - S[v * p->S_b + c]);
        }
      }
}

/* Zones of the box (interior + E) that lie behind a PHYSICAL boundary take the boundary's image of the block's own zone:
 * every coordinate that is out of range on a side without a neighbour is clamped (outflow) or mirrored (wall, that
 * momentum component negated); coordinates out of range behind a neighbour stay.  Sources are never destinations. */
static void physical_refill(const fxo_plan *p, double *U, int64_t b, int E) {
  int lo[3], hi[3];
  for (int d = 0; d < 3; ++d) {
    lo[d] = p->gd[d] - (p->active[d] ? E : 0);
    hi[d] = p->gd[d] + p->n[d] + (p->active[d] ? E : 0);
  }
  for (int k = lo[2]; k < hi[2]; ++k)
    for (int j = lo[1]; j < hi[1]; ++j)
      for (int i = lo[0]; i < hi[0]; ++i) {
        int c[3] = {i, j, k};
        unsigned flip = 0;
        int moved = 0;
        for (int d = 0; d < 3; ++d) {
          if (!p->active[d]) continue;
          int l = p->gd[d], h = p->gd[d] + p->n[d];
          int side = c[d] < l ? 0 : (c[d] >= h ? 1 : -1);
          if (side < 0) continue;
          int32_t nb = p->neigh[b * 6 + 2 * d + side];
          if (nb >= 0) continue;
          if (nb == FXO_BC_REFLECT) {
            c[d] = side ? 2 * h - 1 - c[d] : 2 * l - 1 - c[d];
            flip |= 1u << d;
          } else {
            c[d] = side ? h - 1 : l;
          }
          moved = 1;
        }
        if (!moved) continue;
        int64_t t = b * p->S_b + k * p->S_k + j * p->S_j + i;
        int64_t s = b * p->S_b + c[2] * p->S_k + c[1] * p->S_j + c[0];
        for (int v = 0; v < p->nvars; ++v) {
          double x = U[v * p->S_v + s];
          U[v * p->S_v + t] = (v >= 1 && v <= 3 && ((flip >> (v - 1)) & 1u)) ? -x : x;
        }
      }
}

static int run_stage_ext(fxo_plan *p, const double *X, const double *U0, double *out, const double *dx, double dt,
                         double beta, int first, int E) {
  int fail = 0;
#pragma omp parallel
  {
    double *W = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
    double *S = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
    int nmax = p->np[0] > p->np[1] ? p->np[0] : p->np[1];
    if (p->np[2] > nmax) nmax = p->np[2];
    double *Fl = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)(nmax + 1));
    if (!W || !S || !Fl) {
#pragma omp atomic write
      fail = 1;
    } else {
#pragma omp for schedule(dynamic, 4)
      for (int64_t b = 0; b < p->nblocks; ++b) {
        block_stage_ext(p, X, U0, out, b, dx, dt, beta, first, E, W, S, Fl);
        if (E > 0) physical_refill(p, out, b, E);
      }
    }
    free(W);
    free(S);
    free(Fl);
  }
  return fail ? FXO_ERR_NOMEM : FXO_OK;
}

/* One SSP-RK step with a single guard fill [B17].  FXO_ERR_UNSUPPORTED: rk_order R > nguard in an active dimension, or
 * refinement jumps.  The blocks must share dx with their same-level neighbours (not checked). */
int fxo_hydro_advance_ca(fxo_plan *p, double *U, const double *dx, double dt) {
  if (!p || (!U && p->nblocks) || (!dx && p->nblocks)) return FXO_ERR_INVALID_ARG;
  if (!(dt > 0.0) || !isfinite(dt)) return FXO_ERR_INVALID_ARG;
  if (!p->neigh && p->nblocks > 0) return FXO_ERR_STATE;
  const int R = p->recon == FXO_RECON_WENO5 ? 3 : 2;
  if (p->jump) return FXO_ERR_UNSUPPORTED;
  for (int d = 0; d < 3; ++d)
    if (p->active[d] && p->rk * R > p->gd[d]) return FXO_ERR_UNSUPPORTED;
  if (p->nblocks == 0) return FXO_OK;
  size_t n = (size_t)p->S_v * (size_t)p->nvars;
  double *U1 = (double *)malloc(sizeof(double) * n);
  double *U2 = p->rk == 3 ? (double *)malloc(sizeof(double) * n) : NULL;
  if (!U1 || (p->rk == 3 && !U2)) {
    free(U1);
    free(U2);
    return FXO_ERR_NOMEM;
  }
  /* zones outside a stage's box are never read by the next one: poison them so that a wrong reach shows */
  for (size_t q = 0; q < n; ++q) U1[q] = NAN;
  if (U2)
    for (size_t q = 0; q < n; ++q) U2[q] = NAN;
  int rc = fxo_fill_guardcells(p, U); /* the step's only O1 */
  if (!rc) rc = run_stage_ext(p, U, U, U1, dx, dt, 1.0, 1, (p->rk - 1) * R);
  if (!rc && p->rk == 2) {
    rc = run_stage_ext(p, U1, U, U, dx, dt, 0.5, 0, 0);
  } else if (!rc) {
    rc = run_stage_ext(p, U1, U, U2, dx, dt, 0.25, 0, R);
    if (!rc) rc = run_stage_ext(p, U2, U, U, dx, dt, 2.0 / 3.0, 0, 0);
  }
  free(U1);
  free(U2);
  return rc;
}

/* Face fluxes of direction dir from U (guards must already be filled) [A17]:
 * F[v][b][k][j][i] with extents (nz, ny, nx) and n_dir + 1 along dir, i fastest. */
int fxo_debug_compute_fluxes(fxo_plan *p, const double *U, int dir, double *F) {
  if (!p || !U || !F || dir < 0 || dir > 2 || !p->active[dir]) return FXO_ERR_INVALID_ARG;
  int e[3] = {p->n[0], p->n[1], p->n[2]};
  e[dir] += 1;
  int64_t FS_j = e[0], FS_k = (int64_t)e[0] * e[1], FS_b = FS_k * e[2], FS_v = FS_b * p->nblocks;
  const int64_t stride[3] = {1, p->S_j, p->S_k};
  int fail = 0;
#pragma omp parallel
  {
    double *W = (double *)malloc(sizeof(double) * (size_t)p->nvars * (size_t)p->S_b);
    if (!W) {
#pragma omp atomic write
      fail = 1;
    } else {
#pragma omp for schedule(dynamic, 4)
      for (int64_t b = 0; b < p->nblocks; ++b) {
        block_prims(p, U, b, W);
        for (int k = 0; k < e[2]; ++k)
          for (int j = 0; j < e[1]; ++j)
            for (int i = 0; i < e[0]; ++i) {
              int c[3] = {i + p->gd[0], j + p->gd[1], k + p->gd[2]};
              c[dir] -= 1; /* left cell of face f is padded cell g + f - 1 */
              int64_t cL = c[2] * p->S_k + c[1] * p->S_j + c[0];
              (void)stride;
              double Ff[FXO_MAXV];
              unsigned hit = 0;
              face_flux(p, W, p->S_b, cL, dir, Ff, &hit);
              for (int v = 0; v < p->nvars; ++v) F[v * FS_v + b * FS_b + k * FS_k + j * FS_j + i] = Ff[v];
            }
      }
    }
    free(W);
  }
  return fail ? FXO_ERR_NOMEM : FXO_OK;
}

/* ---------------------------------------------------------------- O7 dt */

int fxo_hydro_compute_dt(fxo_plan *p, const double *U, const double *dx, double cfl, double *dt_out) {
  if (!p || !dt_out || (!U && p->nblocks) || (!dx && p->nblocks)) return FXO_ERR_INVALID_ARG;
  double best = INFINITY;
#pragma omp parallel for schedule(static) reduction(min : best)
  for (int64_t b = 0; b < p->nblocks; ++b)
    for (int k = p->gd[2]; k < p->gd[2] + p->n[2]; ++k)
      for (int j = p->gd[1]; j < p->gd[1] + p->n[1]; ++j)
        for (int i = p->gd[0]; i < p->gd[0] + p->n[0]; ++i) {
          int64_t c = b * p->S_b + k * p->S_k + j * p->S_j + i;
          double Uz[5], W[5];
          for (int v = 0; v < 5; ++v) Uz[v] = U[v * p->S_v + c];
          unsigned hit = 0;
          cons2prim(p, 5, Uz, W, &hit); /* the scalars do not enter the time step [B11] */
          double cs = sqrt(p->gamma * W[4] / W[0]);
          for (int d = 0; d < 3; ++d) {
            if (!p->active[d]) continue;
            double s = fabs(W[1 + d]) + cs;
            double t = dx[b * 3 + d] / s;
            if (!(s > 0.0) || !isfinite(s)) hit |= FXO_STATUS_NONFINITE;
            if (t < best) best = t;
          }
          count_hits(p, hit & FXO_STATUS_NONFINITE, 1);
        }
  *dt_out = cfl * best;
  return FXO_OK;
}
