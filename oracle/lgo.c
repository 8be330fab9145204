/* lgo.c — ORACLE (test infrastructure, not product code).  See lgo.h.
 *
 * Plain C, FP64, one thread, operation order exactly as written (compile with
 * -O2 -ffp-contract=off, no -ffast-math).  Section tags S0..S8 are DESIGN.md's
 * "What a candidate is and what it costs"; every step cites PAPER.md.
 * Nothing here is shared with, generated from, or imported by the CUDA path.
 */
#include "lgo.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

struct lgo_instance {
  int n_f, n_b, n_hu, n_su, n_t, n_v;
  double *x, *y;                 /* vertex coordinates: 0 HQ, 1..n_b BPs, then fields */
  int64_t *s_q, *h_q, *d_q, *r_q, *c_q;
  double v_hu, v_su, kappa, w_path, w_time;
  uint32_t thresh, flags;
};

/* ------------------------------------------------------------------ S0 */

static int finite_nonneg(double v) { return isfinite(v) && v >= 0.0; }

/* Quantise with Q = 1024, round-half-even (R18). */
static int64_t quantise(double v) { return (int64_t)llrint(v * (double)LGO_Q); }

int lgo_instance_create(const lgo_instance_desc *d, lgo_instance **out)
{
  if (!d || !out) return LGO_EINVAL;
  *out = NULL;
  if (d->n_fields < 1 || d->n_bps < 1 || d->n_hu_total < 1 || d->n_su_total < 1) return LGO_EINVAL;
  if (d->n_tours < 1 || d->n_tours > d->n_bps || d->n_tours > d->n_hu_total ||
      d->n_tours > d->n_su_total) return LGO_EINVAL;   /* N_T <= N_HU^total; R22 */
  if (d->n_fields > 65535 || d->n_bps > 255 || d->n_tours > 255 ||
      d->n_hu_total > 255 || d->n_su_total > 255) return LGO_EINVAL;
  if (!d->field_x || !d->field_y || !d->field_supply_t || !d->field_area_ha || !d->bp_x ||
      !d->bp_y || !d->bp_demand_t || !d->hu_rate_ha_per_h || !d->su_capacity_t) return LGO_EINVAL;
  if (!isfinite(d->hq_x) || !isfinite(d->hq_y)) return LGO_EINVAL;
  if (!(isfinite(d->v_hu_road_kmh) && d->v_hu_road_kmh > 0.0)) return LGO_EINVAL;
  if (!(isfinite(d->v_su_road_kmh) && d->v_su_road_kmh > 0.0)) return LGO_EINVAL;
  if (!finite_nonneg(d->su_fill_h_per_t) || !finite_nonneg(d->w_path) ||
      !finite_nonneg(d->w_time)) return LGO_EINVAL;

  lgo_instance *I = (lgo_instance *)calloc(1, sizeof *I);
  if (!I) return LGO_ENOMEM;
  I->n_f = d->n_fields; I->n_b = d->n_bps; I->n_hu = d->n_hu_total; I->n_su = d->n_su_total;
  I->n_t = d->n_tours;  I->n_v = 1 + I->n_b + I->n_f;
  I->x = (double *)malloc(sizeof(double) * I->n_v);
  I->y = (double *)malloc(sizeof(double) * I->n_v);
  I->s_q = (int64_t *)malloc(sizeof(int64_t) * I->n_f);
  I->h_q = (int64_t *)malloc(sizeof(int64_t) * I->n_f);
  I->d_q = (int64_t *)malloc(sizeof(int64_t) * I->n_b);
  I->r_q = (int64_t *)malloc(sizeof(int64_t) * I->n_hu);
  I->c_q = (int64_t *)malloc(sizeof(int64_t) * I->n_su);
  if (!I->x || !I->y || !I->s_q || !I->h_q || !I->d_q || !I->r_q || !I->c_q) {
    lgo_instance_destroy(I); return LGO_ENOMEM;
  }
  int rc = LGO_OK;
  /* Vertex numbering: 0 = HQ, 1..N_B = BPs, N_B+1.. = fields. */
  I->x[0] = d->hq_x; I->y[0] = d->hq_y;
  for (int b = 0; b < I->n_b; b++) {
    if (!isfinite(d->bp_x[b]) || !isfinite(d->bp_y[b]) || !finite_nonneg(d->bp_demand_t[b])) rc = LGO_EINVAL;
    I->x[1 + b] = d->bp_x[b]; I->y[1 + b] = d->bp_y[b];
    I->d_q[b] = quantise(d->bp_demand_t[b]);                     /* d_b^min, eq. (2) */
  }
  int64_t s_max = 0, s_sum = 0, h_sum = 0;
  for (int f = 0; f < I->n_f; f++) {
    if (!isfinite(d->field_x[f]) || !isfinite(d->field_y[f]) ||
        !finite_nonneg(d->field_supply_t[f]) || !finite_nonneg(d->field_area_ha[f])) rc = LGO_EINVAL;
    I->x[1 + I->n_b + f] = d->field_x[f]; I->y[1 + I->n_b + f] = d->field_y[f];
    I->s_q[f] = quantise(d->field_supply_t[f]);                  /* s_f, eq. (2)/(3) L79-85 */
    I->h_q[f] = quantise(d->field_area_ha[f]);                   /* h_f, L83 */
    if (I->s_q[f] > s_max) s_max = I->s_q[f];
    s_sum += I->s_q[f]; h_sum += I->h_q[f];
  }
  int64_t c_sum = 0, r_sum = 0;
  for (int u = 0; u < I->n_hu; u++) {
    if (!finite_nonneg(d->hu_rate_ha_per_h[u])) rc = LGO_EINVAL;
    I->r_q[u] = quantise(d->hu_rate_ha_per_h[u]);                /* v_HU^area, L96 (ii) */
    if (I->r_q[u] <= 0) rc = LGO_EINVAL;
    r_sum += I->r_q[u];
  }
  for (int u = 0; u < I->n_su; u++) {
    if (!finite_nonneg(d->su_capacity_t[u])) rc = LGO_EINVAL;
    I->c_q[u] = quantise(d->su_capacity_t[u]);                   /* l_SU^load, L87 */
    if (I->c_q[u] <= 0) rc = LGO_EINVAL;
    c_sum += I->c_q[u];
  }
  /* Documented integer ranges (keep eq. (4)'s ceil-division and all sums in 32 bits). */
  if (rc == LGO_OK) {
    const int64_t lim = (int64_t)1 << 32;
    if (s_max * (int64_t)I->n_su + c_sum >= lim || s_sum >= lim || h_sum >= lim ||
        r_sum >= lim) rc = LGO_ETOOBIG;
    for (int b = 0; b < I->n_b; b++) if (I->d_q[b] >= lim) rc = LGO_ETOOBIG;
  }
  if (rc != LGO_OK) { lgo_instance_destroy(I); return rc; }
  I->v_hu = d->v_hu_road_kmh; I->v_su = d->v_su_road_kmh;
  I->kappa = d->su_fill_h_per_t;                                  /* t_load = kappa*cap, L96 (iii); R8 */
  I->w_path = d->w_path; I->w_time = d->w_time;
  I->thresh = d->extra_field_thresh; I->flags = d->flags;
  *out = I;
  return LGO_OK;
}

int lgo_instance_destroy(lgo_instance *I)
{
  if (!I) return LGO_EINVAL;
  free(I->x); free(I->y); free(I->s_q); free(I->h_q); free(I->d_q); free(I->r_q); free(I->c_q);
  free(I);
  return LGO_OK;
}

/* Straight-line edge cost ("path length of straight line segments"; R23).
 * Each *, + and sqrt is one IEEE-rounded operation. */
static double D(const lgo_instance *I, int u, int v)
{
  if (u == v) return 0.0;
  double dx = I->x[u] - I->x[v];
  double dy = I->y[u] - I->y[v];
  double xx = dx * dx;
  double yy = dy * dy;
  double ss = xx + yy;
  return sqrt(ss);
}
double lgo_distance(const lgo_instance *I, int32_t u, int32_t v) { return D(I, u, v); }

int64_t lgo_quantum(const lgo_instance *I, int what, int32_t i)
{
  switch (what) {
    case 0: return I->s_q[i]; case 1: return I->h_q[i]; case 2: return I->d_q[i];
    case 3: return I->r_q[i]; case 4: return I->c_q[i]; default: return -1;
  }
}

/* ------------------------------------------------------------------ S1 */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds; the "identical random
 * process control" of PAPER.md:L233 is realised as a counter-based stream (R21). */
void lgo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; round++) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* A (seed,id,stream) draw source with a one-block cache (pure speed; same values). */
typedef struct { uint32_t key[2], ctr[4], blk[4]; int have; } stream_t;

static void stream_init(stream_t *s, uint64_t seed, uint64_t id, uint32_t stream)
{
  s->key[0] = (uint32_t)seed; s->key[1] = (uint32_t)(seed >> 32);
  s->ctr[0] = (uint32_t)id;   s->ctr[1] = (uint32_t)(id >> 32);
  s->ctr[2] = stream;         s->ctr[3] = 0;
  s->have = 0;
}
static uint32_t stream_draw(stream_t *s, uint32_t d)
{
  uint32_t block = d / 4u;
  if (!s->have || s->ctr[3] != block) {
    s->ctr[3] = block;
    lgo_philox4x32_10(s->ctr, s->key, s->blk);
    s->have = 1;
  }
  return s->blk[d % 4u];
}
uint32_t lgo_draw(uint64_t seed, uint64_t id, uint32_t stream, uint32_t d)
{
  stream_t s; stream_init(&s, seed, id, stream);
  return stream_draw(&s, d);
}
/* Bounded draw without rejection: floor(x*m / 2^32). */
static uint32_t below(uint32_t x, uint32_t m) { return (uint32_t)(((uint64_t)x * (uint64_t)m) >> 32); }

/* ------------------------------------------------------------------ S2 */

/* Descending Fisher-Yates over n items with draws 0..n-2 of the stream.  After the
 * loop, consumption position p holds item order[p] = a[n-1-p]. */
static void fisher_yates(stream_t *s, int n, int *order)
{
  int *a = (int *)malloc(sizeof(int) * (size_t)n);
  for (int i = 0; i < n; i++) a[i] = i;
  for (int i = n - 1; i >= 1; i--) {
    int j = (int)below(stream_draw(s, (uint32_t)(n - 1 - i)), (uint32_t)(i + 1));
    int t = a[i]; a[i] = a[j]; a[j] = t;
  }
  for (int p = 0; p < n; p++) order[p] = a[n - 1 - p];
  free(a);
}

/* ordered_partition: item at consumption position p goes to bin p if p < k (every bin
 * gets one: R22), else to bin below(draw((n-1)+(p-k)), k); order in a bin = consumption
 * order.  Tasks (i),(ii),(v),(vi) of PAPER.md:L116-118; eq. (1) L73 holds by construction. */
static void ordered_partition(uint64_t seed, uint64_t id, uint32_t stream, int n, int k,
                              int *bin_of, int *pos_of)
{
  stream_t s; stream_init(&s, seed, id, stream);
  int *order = (int *)malloc(sizeof(int) * (size_t)n);
  int *count = (int *)calloc((size_t)k, sizeof(int));
  fisher_yates(&s, n, order);
  for (int p = 0; p < n; p++) {
    int bin = (p < k) ? p : (int)below(stream_draw(&s, (uint32_t)((n - 1) + (p - k))), (uint32_t)k);
    bin_of[order[p]] = bin;
    pos_of[order[p]] = count[bin]++;
  }
  free(order); free(count);
}

/* ------------------------------------------------------------------ S2 + S3 */

int lgo_decode(const lgo_instance *I, uint64_t seed, uint64_t id,
               uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
               uint8_t *hu_tour, uint8_t *su_tour)
{
  if (!I) return LGO_EINVAL;
  int nmax = I->n_b; if (I->n_hu > nmax) nmax = I->n_hu; if (I->n_su > nmax) nmax = I->n_su;
  int *bin = (int *)malloc(sizeof(int) * (size_t)nmax);
  int *pos = (int *)malloc(sizeof(int) * (size_t)nmax);

  /* BPs -> tours, stream 0 (tasks (i),(ii)). */
  ordered_partition(seed, id, 0, I->n_b, I->n_t, bin, pos);
  int *bpt = (int *)malloc(sizeof(int) * (size_t)I->n_b), *bpp = (int *)malloc(sizeof(int) * (size_t)I->n_b);
  for (int b = 0; b < I->n_b; b++) { bpt[b] = bin[b]; bpp[b] = pos[b]; }
  /* HU units -> tours, stream 1 (task (v)); SU units -> tours, stream 2 (task (vi)); R30. */
  ordered_partition(seed, id, 1, I->n_hu, I->n_t, bin, pos);
  for (int u = 0; u < I->n_hu; u++) if (hu_tour) hu_tour[u] = (uint8_t)bin[u];
  ordered_partition(seed, id, 2, I->n_su, I->n_t, bin, pos);
  for (int u = 0; u < I->n_su; u++) if (su_tour) su_tour[u] = (uint8_t)bin[u];
  for (int b = 0; b < I->n_b; b++) {
    if (bp_tour) bp_tour[b] = (uint8_t)bpt[b];
    if (bp_pos)  bp_pos[b]  = (uint8_t)bpp[b];
  }

  /* "Plan order" of BPs: tour 0's list, then tour 1's, ... */
  int *plan = (int *)malloc(sizeof(int) * (size_t)I->n_b);
  int np = 0;
  for (int g = 0; g < I->n_t; g++) {
    int cnt = 0;
    for (int b = 0; b < I->n_b; b++) if (bpt[b] == g) cnt++;
    for (int q = 0; q < cnt; q++)
      for (int b = 0; b < I->n_b; b++) if (bpt[b] == g && bpp[b] == q) plan[np++] = b;
  }

  /* Fields -> BPs (tasks (iii),(iv)); stream 3 = permutation, stream 4 = extras (R21).
   * Non-last BP: minimal prefix of the stream meeting its demand (the idea of Alg. 1
   * step 2), then geometric extras; last BP: all remaining fields. */
  stream_t s3, s4; stream_init(&s3, seed, id, 3); stream_init(&s4, seed, id, 4);
  int *perm = (int *)malloc(sizeof(int) * (size_t)I->n_f);
  fisher_yates(&s3, I->n_f, perm);
  int p = 0; uint32_t e = 0;
  for (int q = 0; q < I->n_b; q++) {
    int b = plan[q];
    int k = 0;
    if (q == I->n_b - 1) {
      while (p < I->n_f) { field_bp[perm[p]] = (uint16_t)b; field_pos[perm[p]] = (uint16_t)k; k++; p++; }
    } else {
      int64_t Sq = 0;
      while (Sq < I->d_q[b] && p < I->n_f) {
        Sq += I->s_q[perm[p]];
        field_bp[perm[p]] = (uint16_t)b; field_pos[perm[p]] = (uint16_t)k; k++; p++;
      }
      while (p < I->n_f && stream_draw(&s4, e++) < I->thresh) {
        field_bp[perm[p]] = (uint16_t)b; field_pos[perm[p]] = (uint16_t)k; k++; p++;
      }
    }
  }
  free(bin); free(pos); free(bpt); free(bpp); free(plan); free(perm);
  return LGO_OK;
}

/* ------------------------------------------------------------------ S6 */

/* T_wait(g) = E(g) - kappa*((S_g - M_g)/Q) / n_HU(g): eq. (6) PAPER.md:L196 for the
 * critical case l^case = l^largest (L200-201): every SU on the tour except one of the
 * largest class contributes its fill time kappa*cap, divided by the HU count (R7). */
static double wait_time(double E, int64_t S, int64_t M, int n_hu, double kappa)
{
  double tonnes = (double)(S - M) * (1.0 / 1024.0);
  double fill   = kappa * tonnes;
  double per_hu = fill / (double)n_hu;
  return E - per_hu;
}

static void tour_sums(int g, int n_su, const int64_t *c_q, const uint8_t *su_tour,
                      int *n, int64_t *S, int64_t *M)
{
  *n = 0; *S = 0; *M = 0;
  for (int u = 0; u < n_su; u++) if (su_tour[u] == g) {
    (*n)++; *S += c_q[u]; if (c_q[u] > *M) *M = c_q[u];
  }
}

static double tour_wait(int g, double E, int n_hu, int n_su, const int64_t *c_q,
                        const uint8_t *su_tour, double kappa)
{
  int n; int64_t S, M;
  tour_sums(g, n_su, c_q, su_tour, &n, &S, &M);
  return wait_time(E, S, M, n_hu, kappa);
}

/* Algorithm 2 with readings R11-R16. */
static int su_local_min(int n_t, const double *E, const int *n_hu, int n_su,
                        const int64_t *c_q, uint8_t *su_tour, double kappa, double *W)
{
  int moves = 0;
  for (int g = 0; g < n_t; g++) W[g] = tour_wait(g, E[g], n_hu[g], n_su, c_q, su_tour, kappa);
  for (int iter = 0; iter < n_su; iter++) {                         /* R14: cap */
    if (n_t < 2) break;                                             /* R12 */
    /* Step 1-2 (L211-219): waits and the three indices; ties -> lowest index (R16). */
    for (int g = 0; g < n_t; g++) W[g] = tour_wait(g, E[g], n_hu[g], n_su, c_q, su_tour, kappa);
    int g_max = 0;
    for (int g = 1; g < n_t; g++) if (W[g] > W[g_max]) g_max = g;
    double old_max = W[g_max];
    int g_2nd = -1;                                                 /* R11: arg max */
    for (int g = 0; g < n_t; g++) if (g != g_max && (g_2nd < 0 || W[g] > W[g_2nd])) g_2nd = g;
    int g_min = -1;
    for (int g = 0; g < n_t; g++)
      if (g != g_max && g != g_2nd && (g_min < 0 || W[g] < W[g_min])) g_min = g;
    if (g_min < 0) g_min = g_2nd;                                   /* R12: N_T = 2 */
    int n_min = 0;
    for (int u = 0; u < n_su; u++) if (su_tour[u] == g_min) n_min++;
    if (n_min <= 1) break;                                          /* R15 */
    /* Step 3-10 (L221-226): donor's units by rising fill time = rising (c_q,u). */
    int moved = -1;
    uint8_t *tried = (uint8_t *)calloc((size_t)n_su, 1);
    for (int t = 0; t < n_min; t++) {
      int u = -1;
      for (int w = 0; w < n_su; w++)
        if (su_tour[w] == g_min && !tried[w] && (u < 0 || c_q[w] < c_q[u])) u = w;
      tried[u] = 1;
      su_tour[u] = (uint8_t)g_max;                                  /* remove + add */
      double w_new = tour_wait(g_max, E[g_max], n_hu[g_max], n_su, c_q, su_tour, kappa);
      int is_last = (t == n_min - 1);
      if (w_new < W[g_2nd] || is_last) { moved = u; break; }        /* L225; R13 */
      su_tour[u] = (uint8_t)g_min;                                  /* undo */
    }
    free(tried);
    /* Step 11 (L227): keep while the global maximum wait strictly decreases (R14). */
    double new_max = 0.0;
    for (int g = 0; g < n_t; g++) {
      double w = tour_wait(g, E[g], n_hu[g], n_su, c_q, su_tour, kappa);
      if (g == 0 || w > new_max) new_max = w;
    }
    if (new_max < old_max) { moves++; }
    else { su_tour[moved] = (uint8_t)g_min; break; }
  }
  for (int g = 0; g < n_t; g++) W[g] = tour_wait(g, E[g], n_hu[g], n_su, c_q, su_tour, kappa);
  return moves;
}

int lgo_su_local_min(int32_t n_tours, const double *E_h, const int32_t *n_hu,
                     int32_t n_su, const int64_t *cap_q, uint8_t *su_tour,
                     double kappa_h_per_t, double *wait_h)
{
  int *nh = (int *)malloc(sizeof(int) * (size_t)n_tours);
  for (int g = 0; g < n_tours; g++) nh[g] = n_hu[g];
  int m = su_local_min(n_tours, E_h, nh, n_su, cap_q, su_tour, kappa_h_per_t, wait_h);
  free(nh);
  return m;
}

/* ------------------------------------------------------------------ embedded HU assignment (NEXT row N2) */

/* "tours with minimum and maximum completion times, g_min and g_max, are identified, before
 * their assigned number of HUs ... is decreased and increased by one HU, respectively.  This is repeated until
 * the maximum completion time over all tours cannot be further reduced."  L203: for non-uniform HUs "an
 * equivalent method is employed ... where the set of available HUs classes is now sorted according to rising
 * in-field working rates".  Reading R39: the procedure is Algorithm 2 with the completion time
 * T(g) = road_h(g) + H_q(g)/R_g in place of T_wait and the rates in place of the fill times: donor = the tour
 * with the smallest T among the others, its units tried by rising (rate, index), the first that brings
 * T(g_max) below T(g_2nd) or else the fastest is moved, the move is kept while the maximum T strictly
 * decreases; a tour keeps >= 1 HU; at most N_HU moves.  Returns the accepted moves; T receives the final times. */
static double tour_time(int g, double road_h, int64_t Hq, int n_hu, const int64_t *r_q, const uint8_t *hu_tour)
{
  int64_t R = 0;
  for (int u = 0; u < n_hu; u++) if (hu_tour[u] == g) R += r_q[u];
  return road_h + (double)Hq / (double)R;
}

static int hu_balance(int n_t, const double *road_h, const int64_t *Hq, int n_hu, const int64_t *r_q,
                      uint8_t *hu_tour, double *T)
{
  int moves = 0;
  for (int g = 0; g < n_t; g++) T[g] = tour_time(g, road_h[g], Hq[g], n_hu, r_q, hu_tour);
  for (int iter = 0; iter < n_hu; iter++) {
    if (n_t < 2) break;
    for (int g = 0; g < n_t; g++) T[g] = tour_time(g, road_h[g], Hq[g], n_hu, r_q, hu_tour);
    int g_max = 0;
    for (int g = 1; g < n_t; g++) if (T[g] > T[g_max]) g_max = g;
    double old_max = T[g_max];
    int g_2nd = -1;
    for (int g = 0; g < n_t; g++) if (g != g_max && (g_2nd < 0 || T[g] > T[g_2nd])) g_2nd = g;
    int g_min = -1;
    for (int g = 0; g < n_t; g++)
      if (g != g_max && g != g_2nd && (g_min < 0 || T[g] < T[g_min])) g_min = g;
    if (g_min < 0) g_min = g_2nd;
    int n_min = 0;
    for (int u = 0; u < n_hu; u++) if (hu_tour[u] == g_min) n_min++;
    if (n_min <= 1) break;
    int moved = -1;
    uint8_t *tried = (uint8_t *)calloc((size_t)n_hu, 1);
    for (int t = 0; t < n_min; t++) {
      int u = -1;
      for (int w = 0; w < n_hu; w++)
        if (hu_tour[w] == g_min && !tried[w] && (u < 0 || r_q[w] < r_q[u])) u = w;
      tried[u] = 1;
      hu_tour[u] = (uint8_t)g_max;
      double t_new = tour_time(g_max, road_h[g_max], Hq[g_max], n_hu, r_q, hu_tour);
      if (t_new < T[g_2nd] || t == n_min - 1) { moved = u; break; }
      hu_tour[u] = (uint8_t)g_min;
    }
    free(tried);
    double new_max = 0.0;
    for (int g = 0; g < n_t; g++) {
      double t = tour_time(g, road_h[g], Hq[g], n_hu, r_q, hu_tour);
      if (g == 0 || t > new_max) new_max = t;
    }
    if (new_max < old_max) moves++;
    else { hu_tour[moved] = (uint8_t)g_min; break; }
  }
  for (int g = 0; g < n_t; g++) T[g] = tour_time(g, road_h[g], Hq[g], n_hu, r_q, hu_tour);
  return moves;
}

int lgo_hu_balance(int32_t n_tours, const double *road_h, const int64_t *area_q, int32_t n_hu, const int64_t *rate_q,
                   uint8_t *hu_tour, double *time_h)
{
  return hu_balance(n_tours, road_h, area_q, n_hu, rate_q, hu_tour, time_h);
}

/* ------------------------------------------------------------------ S4, S5, S7 */

int lgo_score(const lgo_instance *I,
              const uint8_t *bp_tour, const uint8_t *bp_pos,
              const uint16_t *field_bp, const uint16_t *field_pos,
              const uint8_t *hu_tour, const uint8_t *su_tour_init,
              double *scalars, double *tour_route_km, double *tour_time_h, double *tour_E_h,
              double *tour_wait_h, double *tour_len_km, int64_t *bp_supply_q,
              int64_t *field_shuttles, uint8_t *su_tour_final)
{
  return lgo_score_ex(I, bp_tour, bp_pos, field_bp, field_pos, hu_tour, su_tour_init, 0, scalars, tour_route_km,
                      tour_time_h, tour_E_h, tour_wait_h, tour_len_km, bp_supply_q, field_shuttles, su_tour_final, NULL);
}

/* lgo_score with the embedded HU assignment (hu_balance != 0: PAPER.md:L190, L203; R39) run between pass 1 and
 * Algorithm 2 (the paper's order: "First, the assignment of HUs ... Second ... SUs", L190-192).
 * hu_tour_final (may be NULL) receives the HU sets the cost was computed with. */
int lgo_score_ex(const lgo_instance *I,
              const uint8_t *bp_tour, const uint8_t *bp_pos,
              const uint16_t *field_bp, const uint16_t *field_pos,
              const uint8_t *hu_tour_in, const uint8_t *su_tour_init, int hu_balance_on,
              double *scalars, double *tour_route_km, double *tour_time_h, double *tour_E_h,
              double *tour_wait_h, double *tour_len_km, int64_t *bp_supply_q,
              int64_t *field_shuttles, uint8_t *su_tour_final, uint8_t *hu_tour_final)
{
  const uint8_t *hu_tour = hu_tour_in;
  uint8_t *hu_work = NULL;
  if (!I || !bp_tour || !bp_pos || !field_bp || !field_pos || !hu_tour || !su_tour_init || !scalars)
    return LGO_EINVAL;
  const int nt = I->n_t, nb = I->n_b, nf = I->n_f;
  int rc = LGO_OK;
  /* Build the ordered lists and validate the plan (each field exactly once on exactly one
   * BP, each BP on exactly one tour: PAPER.md:L21, L116-118). */
  int *tour_nbp = (int *)calloc((size_t)nt, sizeof(int));
  int *tour_bp  = (int *)malloc(sizeof(int) * (size_t)nt * (size_t)nb);
  int *bp_nf    = (int *)calloc((size_t)nb, sizeof(int));
  int *bp_field = (int *)malloc(sizeof(int) * (size_t)nb * (size_t)nf);
  int *n_hu = (int *)calloc((size_t)nt, sizeof(int));
  int *n_su = (int *)calloc((size_t)nt, sizeof(int));
  double *Lt = (double *)calloc((size_t)nt, sizeof(double));
  double *E  = (double *)calloc((size_t)nt, sizeof(double));
  double *W  = (double *)calloc((size_t)nt, sizeof(double));
  int64_t *Hq = (int64_t *)calloc((size_t)nt, sizeof(int64_t));
  int64_t *Sq = (int64_t *)calloc((size_t)nb, sizeof(int64_t));
  uint8_t *su = (uint8_t *)malloc((size_t)I->n_su);
  for (int i = 0; i < nt * nb; i++) tour_bp[i] = -1;
  for (int i = 0; i < nb * nf; i++) bp_field[i] = -1;
  for (int b = 0; b < nb; b++) {
    if (bp_tour[b] >= nt || bp_pos[b] >= nb || tour_bp[bp_tour[b] * nb + bp_pos[b]] >= 0) { rc = LGO_EINVAL; break; }
    tour_bp[bp_tour[b] * nb + bp_pos[b]] = b; tour_nbp[bp_tour[b]]++;
  }
  for (int f = 0; f < nf && rc == LGO_OK; f++) {
    if (field_bp[f] >= nb || field_pos[f] >= nf || bp_field[field_bp[f] * nf + field_pos[f]] >= 0) { rc = LGO_EINVAL; break; }
    bp_field[field_bp[f] * nf + field_pos[f]] = f; bp_nf[field_bp[f]]++;
  }
  for (int g = 0; g < nt && rc == LGO_OK; g++)
    for (int q = 0; q < tour_nbp[g]; q++) if (tour_bp[g * nb + q] < 0) rc = LGO_EINVAL;
  for (int b = 0; b < nb && rc == LGO_OK; b++)
    for (int q = 0; q < bp_nf[b]; q++) if (bp_field[b * nf + q] < 0) rc = LGO_EINVAL;
  for (int u = 0; u < I->n_hu && rc == LGO_OK; u++) { if (hu_tour[u] >= nt) rc = LGO_EINVAL; else n_hu[hu_tour[u]]++; }
  for (int u = 0; u < I->n_su && rc == LGO_OK; u++) { if (su_tour_init[u] >= nt) rc = LGO_EINVAL; else { n_su[su_tour_init[u]]++; su[u] = su_tour_init[u]; } }
  for (int g = 0; g < nt && rc == LGO_OK; g++) if (n_hu[g] < 1 || n_su[g] < 1) rc = LGO_EINVAL;
  if (rc != LGO_OK) goto done;

  /* S4 — pass 1: HU route, areas, supplies, E(g).  "The cost function is evaluated
   * tracing traveled distances according to Fig. 1". */
  const int HQ = 0;
  for (int g = 0; g < nt; g++) {
    int prev = HQ; double lt = 0.0; int64_t hq = 0; double sumE = 0.0; int m = 0; int visited = 0;
    for (int q = 0; q < tour_nbp[g]; q++) {
      int b = tour_bp[g * nb + q];
      double sd = 0.0; int k = 0; int64_t sq = 0;
      for (int r = 0; r < bp_nf[b]; r++) {
        int f = bp_field[b * nf + r];
        int vf = 1 + nb + f, vb = 1 + b;
        lt = lt + D(I, prev, vf);              /* HUs travel field to field, never to BPs (L69) */
        prev = vf; visited = 1;
        hq += I->h_q[f];
        sq += I->s_q[f];
        sd = sd + D(I, vf, vb);                /* one-way field -> BP leg */
        k++;
      }
      Sq[b] = sq;
      if (k > 0) { sumE = sumE + sd / (double)k; m++; }            /* R10 */
    }
    if (visited) lt = lt + D(I, prev, HQ);     /* tours start and end at HQ (L21); R2 */
    Lt[g] = lt; Hq[g] = hq;
    /* Alg. 2 step 1 (L213): average over BPs of average over fields of t_edge, the
     * round trip field -> BP -> field at v_SU (L199); R9. */
    E[g] = (m > 0) ? (2.0 * (sumE / (double)m)) / I->v_su : 0.0;
  }

  /* S5 — eq. (2) (L79), on quanta, ">=" (R18); infeasible => discarded (L186; R19). */
  int feasible = 1;
  for (int b = 0; b < nb; b++) if (Sq[b] < I->d_q[b]) feasible = 0;
  if (bp_supply_q) for (int b = 0; b < nb; b++) bp_supply_q[b] = Sq[b];
  if (tour_route_km) for (int g = 0; g < nt; g++) tour_route_km[g] = Lt[g];
  if (tour_E_h) for (int g = 0; g < nt; g++) tour_E_h[g] = E[g];
  if (!feasible) {
    scalars[0] = 0.0;
    for (int i = 1; i <= 6; i++) scalars[i] = INFINITY;
    scalars[7] = 0.0;
    if (su_tour_final) memcpy(su_tour_final, su, (size_t)I->n_su);
    if (hu_tour_final) memcpy(hu_tour_final, hu_tour_in, (size_t)I->n_hu);
    if (tour_time_h) for (int g = 0; g < nt; g++) tour_time_h[g] = INFINITY;
    if (tour_wait_h) for (int g = 0; g < nt; g++) tour_wait_h[g] = INFINITY;
    if (tour_len_km) for (int g = 0; g < nt; g++) tour_len_km[g] = INFINITY;
    if (field_shuttles) for (int f = 0; f < nf; f++) field_shuttles[f] = 0;
    goto done;
  }

  /* Embedded HU assignment (NEXT row N2; L190, L203; R39): before the SUs, as the paper lists them. */
  if (hu_balance_on) {
    hu_work = (uint8_t *)malloc((size_t)I->n_hu);
    double *road = (double *)malloc(sizeof(double) * (size_t)nt), *Tt = (double *)malloc(sizeof(double) * (size_t)nt);
    memcpy(hu_work, hu_tour_in, (size_t)I->n_hu);
    for (int g = 0; g < nt; g++) road[g] = Lt[g] / I->v_hu;
    hu_balance(nt, road, Hq, I->n_hu, I->r_q, hu_work, Tt);
    free(road); free(Tt);
    hu_tour = hu_work;
    for (int g = 0; g < nt; g++) n_hu[g] = 0;
    for (int u = 0; u < I->n_hu; u++) n_hu[hu_tour[u]]++;
  }
  if (hu_tour_final) memcpy(hu_tour_final, hu_tour, (size_t)I->n_hu);

  /* S6 — embedded local minimisation of the SU assignment (Algorithm 2). */
  int moves = su_local_min(nt, E, n_hu, I->n_su, I->c_q, su, I->kappa, W);

  /* S7 — pass 2: shuttles (eq. (4) L89 with the tour's mean capacity, R4), lengths
   * (N_HU(g), N_SU(g) multiply the tour distance; shuttles x2, L106), times (L190). */
  double L_HU = 0.0, L_eSU = 0.0, L_lSU = 0.0, path = 0.0, makespan = 0.0;
  for (int g = 0; g < nt; g++) {
    int n_g; int64_t C_g, M_g;
    tour_sums(g, I->n_su, I->c_q, su, &n_g, &C_g, &M_g);
    double sh = 0.0;
    for (int q = 0; q < tour_nbp[g]; q++) {
      int b = tour_bp[g * nb + q];
      for (int r = 0; r < bp_nf[b]; r++) {
        int f = bp_field[b * nf + r];
        int64_t N = (I->s_q[f] * (int64_t)n_g + C_g - 1) / C_g;    /* ceil(s / (C/n)) */
        if (field_shuttles) field_shuttles[f] = N;
        sh = sh + (double)N * D(I, 1 + nb + f, 1 + b);
      }
    }
    double l_hu  = (double)n_hu[g] * Lt[g];
    double l_esu = (double)n_g * Lt[g] + sh;   /* SUs follow the route empty + empty return legs */
    double l_lsu = sh;                         /* loaded legs field -> BP */
    double l_g   = (l_hu + l_esu) + l_lsu;
    int64_t R_g = 0;
    for (int u = 0; u < I->n_hu; u++) if (hu_tour[u] == g) R_g += I->r_q[u];   /* L69; R7 */
    double t_g = Lt[g] / I->v_hu + (double)Hq[g] / (double)R_g;    /* L190; R6 */
    L_HU = L_HU + l_hu; L_eSU = L_eSU + l_esu; L_lSU = L_lSU + l_lsu;
    path = path + l_g;
    if (g == 0 || t_g > makespan) makespan = t_g;
    if (tour_time_h) tour_time_h[g] = t_g;
    if (tour_len_km) tour_len_km[g] = l_g;
  }
  double cost = I->w_path * path + I->w_time * makespan;           /* R1; abstract L7 */
  scalars[0] = 1.0; scalars[1] = L_HU; scalars[2] = L_eSU; scalars[3] = L_lSU;
  scalars[4] = path; scalars[5] = makespan; scalars[6] = cost; scalars[7] = (double)moves;
  if (tour_wait_h) for (int g = 0; g < nt; g++) tour_wait_h[g] = W[g];
  if (su_tour_final) memcpy(su_tour_final, su, (size_t)I->n_su);

done:
  free(tour_nbp); free(tour_bp); free(bp_nf); free(bp_field); free(n_hu); free(n_su);
  free(Lt); free(E); free(W); free(Hq); free(Sq); free(su); free(hu_work);
  return rc;
}

/* ------------------------------------------------------------------ batch + S8 */

typedef struct {
  uint8_t *bp_tour, *bp_pos, *hu_tour, *hu_final, *su_init, *su_final; uint16_t *field_bp, *field_pos;
} plan_buf;

static int plan_alloc(const lgo_instance *I, plan_buf *P)
{
  P->bp_tour = (uint8_t *)malloc((size_t)I->n_b); P->bp_pos = (uint8_t *)malloc((size_t)I->n_b);
  P->hu_tour = (uint8_t *)malloc((size_t)I->n_hu); P->hu_final = (uint8_t *)malloc((size_t)I->n_hu);
  P->su_init = (uint8_t *)malloc((size_t)I->n_su);
  P->su_final = (uint8_t *)malloc((size_t)I->n_su);
  P->field_bp = (uint16_t *)malloc(sizeof(uint16_t) * (size_t)I->n_f);
  P->field_pos = (uint16_t *)malloc(sizeof(uint16_t) * (size_t)I->n_f);
  return (P->bp_tour && P->bp_pos && P->hu_tour && P->hu_final && P->su_init && P->su_final && P->field_bp && P->field_pos)
         ? LGO_OK : LGO_ENOMEM;
}
static void plan_free(plan_buf *P)
{
  free(P->bp_tour); free(P->bp_pos); free(P->hu_tour); free(P->hu_final); free(P->su_init); free(P->su_final);
  free(P->field_bp); free(P->field_pos);
}

int lgo_eval_batch(const lgo_instance *I, uint64_t seed, const uint64_t *ids,
                   uint64_t first_id, uint64_t n,
                   double *cost, double *path_km, double *makespan_h, uint8_t *feasible)
{
  if (!I) return LGO_EINVAL;
  plan_buf P; if (plan_alloc(I, &P) != LGO_OK) { plan_free(&P); return LGO_ENOMEM; }
  for (uint64_t i = 0; i < n; i++) {
    uint64_t id = ids ? ids[i] : first_id + i;
    double sc[8];
    lgo_decode(I, seed, id, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init);
    lgo_score(I, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init, sc,
              NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL);
    if (cost) cost[i] = sc[6];
    if (path_km) path_km[i] = sc[4];
    if (makespan_h) makespan_h[i] = sc[5];
    if (feasible) feasible[i] = (uint8_t)(sc[0] != 0.0);
  }
  plan_free(&P);
  return LGO_OK;
}

int lgo_decode_batch(const lgo_instance *I, uint64_t seed, const uint64_t *ids,
                     uint64_t first_id, uint64_t n,
                     uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                     uint8_t *hu_tour, uint8_t *su_tour_init, uint8_t *su_tour_final)
{
  if (!I) return LGO_EINVAL;
  plan_buf P; if (plan_alloc(I, &P) != LGO_OK) { plan_free(&P); return LGO_ENOMEM; }
  for (uint64_t i = 0; i < n; i++) {
    uint64_t id = ids ? ids[i] : first_id + i;
    double sc[8];
    lgo_decode(I, seed, id, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init);
    lgo_score(I, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init, sc,
              NULL, NULL, NULL, NULL, NULL, NULL, NULL, P.su_final);
    if (bp_tour) memcpy(bp_tour + i * (size_t)I->n_b, P.bp_tour, (size_t)I->n_b);
    if (bp_pos)  memcpy(bp_pos + i * (size_t)I->n_b, P.bp_pos, (size_t)I->n_b);
    if (field_bp)  memcpy(field_bp + i * (size_t)I->n_f, P.field_bp, sizeof(uint16_t) * (size_t)I->n_f);
    if (field_pos) memcpy(field_pos + i * (size_t)I->n_f, P.field_pos, sizeof(uint16_t) * (size_t)I->n_f);
    if (hu_tour) memcpy(hu_tour + i * (size_t)I->n_hu, P.hu_tour, (size_t)I->n_hu);
    if (su_tour_init)  memcpy(su_tour_init + i * (size_t)I->n_su, P.su_init, (size_t)I->n_su);
    if (su_tour_final) memcpy(su_tour_final + i * (size_t)I->n_su, P.su_final, (size_t)I->n_su);
  }
  plan_free(&P);
  return LGO_OK;
}

/* S8: i* = argmin_i C_i, ordered on (bit pattern of cost, id) so the
 * lowest id wins a tie (R29).  Costs are >= 0 or +inf, so their IEEE bit patterns order
 * like the values. */
int lgo_search(const lgo_instance *I, uint64_t seed, uint64_t first_id, uint64_t budget,
               double *best_cost, uint64_t *best_id)
{
  if (!I || !best_cost || !best_id || budget == 0) return LGO_EINVAL;
  plan_buf P; if (plan_alloc(I, &P) != LGO_OK) { plan_free(&P); return LGO_ENOMEM; }
  uint64_t bbits = 0, bid = 0; int have = 0;
  for (uint64_t i = 0; i < budget; i++) {
    uint64_t id = first_id + i;
    double sc[8];
    lgo_decode(I, seed, id, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init);
    lgo_score(I, P.bp_tour, P.bp_pos, P.field_bp, P.field_pos, P.hu_tour, P.su_init, sc,
              NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL);
    uint64_t bits; double c = sc[6]; memcpy(&bits, &c, 8);
    if (!have || bits < bbits || (bits == bbits && id < bid)) { bbits = bits; bid = id; have = 1; }
  }
  memcpy(best_cost, &bbits, 8);
  *best_id = bid;
  plan_free(&P);
  return LGO_OK;
}

/* ================================================================== NEXT rows: Algorithm 1 */

/* Explicit plan as ordered lists (built from / written back to the array form). */
typedef struct {
  int n_t, n_b, n_f;
  int *tour_len, *tour_bp;      /* tour_bp[g*n_b + pos] */
  int *bp_len, *bp_field;       /* bp_field[b*n_f + pos] */
} plan_lists;

static int lists_from_arrays(const lgo_instance *I, plan_lists *L, const uint8_t *bp_tour, const uint8_t *bp_pos,
                             const uint16_t *field_bp, const uint16_t *field_pos)
{
  L->n_t = I->n_t; L->n_b = I->n_b; L->n_f = I->n_f;
  L->tour_len = (int *)calloc((size_t)I->n_t, sizeof(int));
  L->tour_bp = (int *)malloc(sizeof(int) * (size_t)I->n_t * (size_t)I->n_b);
  L->bp_len = (int *)calloc((size_t)I->n_b, sizeof(int));
  L->bp_field = (int *)malloc(sizeof(int) * (size_t)I->n_b * (size_t)I->n_f);
  for (int b = 0; b < I->n_b; b++) {
    if (bp_tour[b] >= I->n_t || bp_pos[b] >= I->n_b) return LGO_EINVAL;
    L->tour_bp[bp_tour[b] * I->n_b + bp_pos[b]] = b; L->tour_len[bp_tour[b]]++;
  }
  for (int f = 0; f < I->n_f; f++) {
    if (field_bp[f] >= I->n_b || field_pos[f] >= I->n_f) return LGO_EINVAL;
    L->bp_field[field_bp[f] * I->n_f + field_pos[f]] = f; L->bp_len[field_bp[f]]++;
  }
  return LGO_OK;
}
static void lists_to_arrays(const plan_lists *L, uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos)
{
  for (int g = 0; g < L->n_t; g++)
    for (int q = 0; q < L->tour_len[g]; q++) { int b = L->tour_bp[g * L->n_b + q]; bp_tour[b] = (uint8_t)g; bp_pos[b] = (uint8_t)q; }
  for (int b = 0; b < L->n_b; b++)
    for (int q = 0; q < L->bp_len[b]; q++) { int f = L->bp_field[b * L->n_f + q]; field_bp[f] = (uint16_t)b; field_pos[f] = (uint16_t)q; }
}
static void lists_free(plan_lists *L) { free(L->tour_len); free(L->tour_bp); free(L->bp_len); free(L->bp_field); }

static void list_remove(int *list, int *len, int value)
{
  int k = 0;
  while (list[k] != value) k++;
  for (; k + 1 < *len; k++) list[k] = list[k + 1];
  (*len)--;
}
static void list_insert(int *list, int *len, int pos, int value)
{
  for (int k = *len; k > pos; k--) list[k] = list[k - 1];
  list[pos] = value; (*len)++;
}

/* Algorithm 1, steps 1-3. */
int lgo_init_plan(const lgo_instance *I, uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                  uint8_t *hu_tour, uint8_t *su_tour)
{
  if (!I || !bp_tour || !bp_pos || !field_bp || !field_pos || !hu_tour || !su_tour) return LGO_EINVAL;
  const int nt = I->n_t, nb = I->n_b, nf = I->n_f;
  /* Step 1 (i) (L122): "approximately equal number of HUs to each tour ... N_HU(N_T) capturing
   * the integer residual" (the printed N_B/N_T is read as N_HU^total/N_T, R25): units in index
   * order, floor(N_HU/N_T) per tour, the rest on the last tour. */
  { int per = I->n_hu / nt;
    for (int u = 0; u < I->n_hu; u++) { int g = u / per; hu_tour[u] = (uint8_t)(g < nt ? g : nt - 1); } }
  /* SUs: Case 1 gives every tour the same number of each class (L273: 2 small + 4 large):
   * units sorted by (capacity, index) are dealt round-robin (R31). */
  { int *ord = (int *)malloc(sizeof(int) * (size_t)I->n_su); char *used = (char *)calloc((size_t)I->n_su, 1);
    for (int r = 0; r < I->n_su; r++) {
      int u = -1;
      for (int w = 0; w < I->n_su; w++) if (!used[w] && (u < 0 || I->c_q[w] < I->c_q[u])) u = w;
      used[u] = 1; ord[r] = u;
    }
    for (int r = 0; r < I->n_su; r++) su_tour[ord[r]] = (uint8_t)(r % nt);
    free(ord); free(used); }
  /* Step 1 (ii) (L122): nearest-neighbour chain over the BPs starting at HQ; the chain is cut
   * into N_T consecutive runs, tour g taking chain[floor(g N_B/N_T) .. floor((g+1) N_B/N_T)) (R32). */
  { char *used = (char *)calloc((size_t)nb, 1); int *chain = (int *)malloc(sizeof(int) * (size_t)nb);
    int cur = 0 /* HQ */;
    for (int k = 0; k < nb; k++) {
      int best = -1; double bd = 0.0;
      for (int b = 0; b < nb; b++) if (!used[b]) { double d = D(I, cur, 1 + b); if (best < 0 || d < bd) { best = b; bd = d; } }
      used[best] = 1; chain[k] = best; cur = 1 + best;
    }
    for (int g = 0; g < nt; g++) {
      int lo = (int)(((long)g * nb) / nt), hi = (int)(((long)(g + 1) * nb) / nt);
      for (int k = lo; k < hi; k++) { bp_tour[chain[k]] = (uint8_t)g; bp_pos[chain[k]] = (uint8_t)(k - lo); }
    }
    free(used); free(chain); }
  /* Step 2 (L124): fields, in identification order (L173), go to their closest BP not yet
   * supplied up to its minimum demand; once every BP is supplied, to their closest BP. */
  int64_t *Sq = (int64_t *)calloc((size_t)nb, sizeof(int64_t));
  int *fb = (int *)malloc(sizeof(int) * (size_t)nf);
  for (int f = 0; f < nf; f++) {
    int best = -1; double bd = 0.0;
    for (int b = 0; b < nb; b++) if (Sq[b] < I->d_q[b]) { double d = D(I, 1 + nb + f, 1 + b); if (best < 0 || d < bd) { best = b; bd = d; } }
    if (best < 0)
      for (int b = 0; b < nb; b++) { double d = D(I, 1 + nb + f, 1 + b); if (best < 0 || d < bd) { best = b; bd = d; } }
    fb[f] = best; Sq[best] += I->s_q[f];
  }
  /* Step 3 (L126, L171): per BP, nearest-neighbour order "from the HQ to the first field of its
   * assigned BP, from that field to a closest second field assigned to the same BP, and so forth". */
  { char *used = (char *)calloc((size_t)nf, 1);
    for (int b = 0; b < nb; b++) {
      int cur = 0 /* HQ */, k = 0;
      for (;;) {
        int best = -1; double bd = 0.0;
        for (int f = 0; f < nf; f++) if (fb[f] == b && !used[f]) { double d = D(I, cur, 1 + nb + f); if (best < 0 || d < bd) { best = f; bd = d; } }
        if (best < 0) break;
        used[best] = 1; field_bp[best] = (uint16_t)b; field_pos[best] = (uint16_t)k++; cur = 1 + nb + best;
      }
    }
    free(used); }
  free(Sq); free(fb);
  return LGO_OK;
}

/* Step 8: "a simple remove- and reinsert-operation for vertices, which can
 * represent either a field or a BP".  A field may go to any BP at any position; a BP may go to
 * any tour or to another index of its tour, and takes all its fields with it (L184).  The vertex
 * is drawn uniformly over fields and BPs ("since N_F >> N_B, it is more likely to draw fields").
 * R35: v = below(w0, N_F+N_B); target = below(w1, N_B or N_T); position = below(w2, len+1) with
 * len the target list's length after the removal. */
int lgo_apply_move(const lgo_instance *I, uint32_t w0, uint32_t w1, uint32_t w2,
                   uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos)
{
  if (!I) return LGO_EINVAL;
  plan_lists L;
  int rc = lists_from_arrays(I, &L, bp_tour, bp_pos, field_bp, field_pos);
  if (rc == LGO_OK) {
    const int nf = I->n_f, nb = I->n_b, nt = I->n_t;
    uint32_t v = below(w0, (uint32_t)(nf + nb));
    if ((int)v < nf) {
      int f = (int)v, a = field_bp[f];
      list_remove(L.bp_field + (size_t)a * nf, &L.bp_len[a], f);
      int t = (int)below(w1, (uint32_t)nb);
      /* §2.6 (L249): with the field->BP assignment fixed, a removed field "must be reinserted into the same group of
       * fields assigned to that given BP.  This is the only change."  (flag bit 3; the draw w1 is then unused) */
      if (I->flags & LGO_FLAG_FIX_FIELD_BP) t = a;
      int q = (int)below(w2, (uint32_t)(L.bp_len[t] + 1));
      list_insert(L.bp_field + (size_t)t * nf, &L.bp_len[t], q, f);
    } else {
      int b = (int)v - nf, g = bp_tour[b];
      list_remove(L.tour_bp + (size_t)g * nb, &L.tour_len[g], b);
      int t = (int)below(w1, (uint32_t)nt);
      int q = (int)below(w2, (uint32_t)(L.tour_len[t] + 1));
      list_insert(L.tour_bp + (size_t)t * nb, &L.tour_len[t], q, b);
    }
    lists_to_arrays(&L, bp_tour, bp_pos, field_bp, field_pos);
  }
  lists_free(&L);
  return rc;
}

/* One worker (L163-165): x_i = move(x), then constraint check and cost as in lgo_score. */
/* t_best: the best-so-far maximum completion time; with LGO_FLAG_MAKESPAN_FILTER a feasible x_i whose makespan
 * exceeds it is discarded by C_i = inf (reading R38). */
static void worker_eval(const lgo_instance *I, const plan_buf *X, plan_buf *Y, uint64_t seed, uint64_t id, double t_best, double *sc)
{
  uint32_t ctr[4] = { (uint32_t)id, (uint32_t)(id >> 32), 5u, 0u }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, w[4];
  lgo_philox4x32_10(ctr, key, w);
  memcpy(Y->bp_tour, X->bp_tour, (size_t)I->n_b); memcpy(Y->bp_pos, X->bp_pos, (size_t)I->n_b);
  memcpy(Y->field_bp, X->field_bp, sizeof(uint16_t) * (size_t)I->n_f);
  memcpy(Y->field_pos, X->field_pos, sizeof(uint16_t) * (size_t)I->n_f);
  memcpy(Y->hu_tour, X->hu_tour, (size_t)I->n_hu); memcpy(Y->su_init, X->su_init, (size_t)I->n_su);
  lgo_apply_move(I, w[0], w[1], w[2], Y->bp_tour, Y->bp_pos, Y->field_bp, Y->field_pos);
  lgo_score_ex(I, Y->bp_tour, Y->bp_pos, Y->field_bp, Y->field_pos, Y->hu_tour, Y->su_init, (I->flags & LGO_FLAG_HU_BALANCE) != 0, sc,
               NULL, NULL, NULL, NULL, NULL, NULL, NULL, Y->su_final, Y->hu_final);
  if ((I->flags & LGO_FLAG_MAKESPAN_FILTER) && sc[0] != 0.0 && sc[5] > t_best) sc[6] = INFINITY;
}

int lgo_move_eval_batch(const lgo_instance *I,
                        const uint8_t *bp_tour, const uint8_t *bp_pos, const uint16_t *field_bp, const uint16_t *field_pos,
                        const uint8_t *hu_tour, const uint8_t *su_tour,
                        uint64_t seed, uint64_t first_id, uint64_t n,
                        double *cost, double *path_km, double *makespan_h, uint8_t *feasible)
{
  if (!I) return LGO_EINVAL;
  plan_buf X, Y;
  if (plan_alloc(I, &X) != LGO_OK || plan_alloc(I, &Y) != LGO_OK) return LGO_ENOMEM;
  memcpy(X.bp_tour, bp_tour, (size_t)I->n_b); memcpy(X.bp_pos, bp_pos, (size_t)I->n_b);
  memcpy(X.field_bp, field_bp, sizeof(uint16_t) * (size_t)I->n_f); memcpy(X.field_pos, field_pos, sizeof(uint16_t) * (size_t)I->n_f);
  memcpy(X.hu_tour, hu_tour, (size_t)I->n_hu); memcpy(X.su_init, su_tour, (size_t)I->n_su);
  /* best-so-far makespan = that of x itself (scored like a worker's plan) */
  double t_best = INFINITY;
  { double s0[8];
    lgo_score_ex(I, X.bp_tour, X.bp_pos, X.field_bp, X.field_pos, X.hu_tour, X.su_init, (I->flags & LGO_FLAG_HU_BALANCE) != 0, s0,
                 NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL, NULL);
    if (s0[0] != 0.0) t_best = s0[5]; }
  for (uint64_t i = 0; i < n; i++) {
    double sc[8];
    worker_eval(I, &X, &Y, seed, first_id + i, t_best, sc);
    if (cost) cost[i] = sc[6];
    if (path_km) path_km[i] = sc[4];
    if (makespan_h) makespan_h[i] = sc[5];
    if (feasible) feasible[i] = (uint8_t)(sc[0] != 0.0);
  }
  plan_free(&X); plan_free(&Y);
  return LGO_OK;
}

/* Algorithm 1, steps 4-16.  R36: worker ids of iteration k are
 * k*n_workers .. (k+1)*n_workers-1; the exploration draw u of iteration k is word 0 of the Philox
 * block (seed; k, stream 6, block 0), u < eps  <=>  draw < eps_thresh (eq. (5)).
 * R37: an adopted x_i carries the SU assignment Alg. 2 left it with; if every worker of an
 * iteration is infeasible (C_i* = inf), x_old is kept. */
int lgo_local_search(const lgo_instance *I,
                     uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                     uint8_t *hu_tour, uint8_t *su_tour,
                     uint64_t seed, uint32_t n_iters, uint32_t n_workers, uint32_t eps_thresh,
                     double *best_cost, double *hist_cost, uint64_t *hist_id)
{
  if (!I || !best_cost || n_workers == 0) return LGO_EINVAL;
  plan_buf best, old, cur, Y, win;
  if (plan_alloc(I, &best) || plan_alloc(I, &old) || plan_alloc(I, &cur) || plan_alloc(I, &Y) || plan_alloc(I, &win)) return LGO_ENOMEM;
  const size_t nb = (size_t)I->n_b, nf2 = sizeof(uint16_t) * (size_t)I->n_f;
#define PLAN_COPY(dst, src) do { memcpy((dst).bp_tour, (src).bp_tour, nb); memcpy((dst).bp_pos, (src).bp_pos, nb); \
    memcpy((dst).field_bp, (src).field_bp, nf2); memcpy((dst).field_pos, (src).field_pos, nf2); \
    memcpy((dst).hu_tour, (src).hu_tour, (size_t)I->n_hu); memcpy((dst).su_init, (src).su_init, (size_t)I->n_su); } while (0)
  /* Step 4 (L133): x* = x_0 with cost C*, x_old = x*. */
  memcpy(best.bp_tour, bp_tour, nb); memcpy(best.bp_pos, bp_pos, nb);
  memcpy(best.field_bp, field_bp, nf2); memcpy(best.field_pos, field_pos, nf2);
  memcpy(best.hu_tour, hu_tour, (size_t)I->n_hu); memcpy(best.su_init, su_tour, (size_t)I->n_su);
  double sc[8];
  int rc = lgo_score_ex(I, best.bp_tour, best.bp_pos, best.field_bp, best.field_pos, best.hu_tour, best.su_init,
                        (I->flags & LGO_FLAG_HU_BALANCE) != 0, sc,
                        NULL, NULL, NULL, NULL, NULL, NULL, NULL, best.su_final, best.hu_final);
  if (rc != LGO_OK) goto out;
  memcpy(best.su_init, best.su_final, (size_t)I->n_su);
  memcpy(best.hu_tour, best.hu_final, (size_t)I->n_hu);
  double c_star = sc[6];
  double t_star = (sc[0] != 0.0) ? sc[5] : INFINITY;       /* best-so-far maximum completion time (L205; R38) */
  PLAN_COPY(old, best);
  for (uint32_t k = 0; k < n_iters; k++) {
    /* Step 6, eq. (5): x = x* if u < eps else x_old (on the host, L231). */
    uint32_t u = lgo_draw(seed, (uint64_t)k, 6u, 0u);
    if (u < eps_thresh) PLAN_COPY(cur, best); else PLAN_COPY(cur, old);
    /* Steps 9-13: every worker moves x once and evaluates; i* = arg min C_i (lowest id on ties). */
    uint64_t bbits = 0, bid = 0; int have = 0; double t_win = INFINITY;
    for (uint32_t i = 0; i < n_workers; i++) {
      uint64_t id = (uint64_t)k * n_workers + i;
      worker_eval(I, &cur, &Y, seed, id, t_star, sc);
      uint64_t bits; memcpy(&bits, &sc[6], 8);
      if (!have || bits < bbits) {
        bbits = bits; bid = id; have = 1; t_win = sc[5]; PLAN_COPY(win, Y);
        memcpy(win.su_init, Y.su_final, (size_t)I->n_su); memcpy(win.hu_tour, Y.hu_final, (size_t)I->n_hu);
      }
    }
    double c_win; memcpy(&c_win, &bbits, 8);
    if (hist_cost) hist_cost[k] = c_win;
    if (hist_id) hist_id[k] = bid;
    /* Steps 14-15 (L169): update x*, C* if improving; x_old <- x_i*. */
    if (isfinite(c_win)) {
      if (c_win < c_star) { c_star = c_win; t_star = t_win; PLAN_COPY(best, win); }
      PLAN_COPY(old, win);
    }
  }
  memcpy(bp_tour, best.bp_tour, nb); memcpy(bp_pos, best.bp_pos, nb);
  memcpy(field_bp, best.field_bp, nf2); memcpy(field_pos, best.field_pos, nf2);
  memcpy(hu_tour, best.hu_tour, (size_t)I->n_hu); memcpy(su_tour, best.su_init, (size_t)I->n_su);
  *best_cost = c_star;
out:
  plan_free(&best); plan_free(&old); plan_free(&cur); plan_free(&Y); plan_free(&win);
  return rc;
#undef PLAN_COPY
}
