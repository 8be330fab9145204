/* lgo.h — ORACLE (test infrastructure, not product code).
 *
 * Plain, slow, single-threaded CPU implementation of the paper's plan evaluation
 * (arxiv 1909.10286, /root/reference/PAPER.md) with the readings listed in DESIGN.md.
 * It shares no code with the CUDA path under paper_1909_10286_b200/csrc/: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Every function below cites the passage of PAPER.md it follows.
 * Pins (tests/test_oracle_*.py): Philox known answers + cuRAND header; hand toy A (P1);
 * Alg. 2 traces B and C (P2, P3); decoder / score invariants (P4, P5); brute force (P8);
 * Algorithm 1 (initialisation, moves, loop): hand instance and hand moves (tests/test_oracle_alg1.py);
 * embedded HU assignment: two hand traces, degenerate cases, invariants (tests/test_oracle_hu.py).
 * No function is "parity unpinned".
 */
#ifndef LGO_H
#define LGO_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LGO_OK       0
#define LGO_EINVAL  (-1)
#define LGO_ETOOBIG (-2)
#define LGO_ENOMEM  (-4)

#define LGO_Q 1024   /* quanta per unit (t, ha, ha/h); R18 */
#define LGO_FLAG_HU_BALANCE 2u   /* desc.flags bit 1: Algorithm 1's workers embed the HU assignment (N2; R39) */
#define LGO_FLAG_FIX_FIELD_BP 8u   /* desc.flags bit 3: a moved field stays with its BP (§2.6; Cases 2-3 L273) */
#define LGO_FLAG_MAKESPAN_FILTER 4u /* desc.flags bit 2: workers whose makespan exceeds the best-so-far one get C_i = inf (L205; R38) */

/* Same field order as the product's lgx_instance_desc (restated, not shared). */
typedef struct {
  double   hq_x, hq_y;
  int32_t  n_fields;   const double *field_x, *field_y, *field_supply_t, *field_area_ha;
  int32_t  n_bps;      const double *bp_x, *bp_y, *bp_demand_t;
  int32_t  n_hu_total; const double *hu_rate_ha_per_h;
  int32_t  n_su_total; const double *su_capacity_t;
  int32_t  n_tours;
  double   v_hu_road_kmh, v_su_road_kmh, v_infield_kmh;
  double   su_fill_h_per_t;
  double   w_path, w_time;
  uint32_t extra_field_thresh;
  uint32_t flags;
} lgo_instance_desc;

typedef struct lgo_instance lgo_instance;

int  lgo_instance_create (const lgo_instance_desc *desc, lgo_instance **out);
int  lgo_instance_destroy(lgo_instance *inst);

/* S1: one Philox4x32-10 block. key=(seed_lo,seed_hi), counter=(id_lo,id_hi,stream,block). */
void lgo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* S1: draw d of stream s for (seed,id) = word d%4 of block d/4. */
uint32_t lgo_draw(uint64_t seed, uint64_t id, uint32_t stream, uint32_t d);

/* S0: distance between vertices (0=HQ, 1..N_B=BPs, then fields), quantised inputs. */
double  lgo_distance(const lgo_instance *inst, int32_t u, int32_t v);
int64_t lgo_quantum(const lgo_instance *inst, int what, int32_t i); /* 0 s_q,1 h_q,2 d_q,3 r_q,4 c_q */

/* S2+S3: decode (seed,id) into an explicit plan.  Arrays are caller-allocated:
 * bp_tour[N_B], bp_pos[N_B]  : tour of each BP and its position on that tour
 * field_bp[N_F], field_pos[N_F]: BP of each field and its position in that BP's list
 * hu_tour[N_HU], su_tour[N_SU]: tour of each unit (S2)                                */
int lgo_decode(const lgo_instance *inst, uint64_t seed, uint64_t id,
               uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
               uint8_t *hu_tour, uint8_t *su_tour);

/* S4-S7: score an explicit plan.  Any of the array outputs may be NULL.
 * scalars[8] = {feasible(0/1), L_HU, L_eSU, L_lSU, path_km, makespan_h, cost, n_alg2_moves}
 * infeasible: scalars[1..6] = +inf.                                                     */
int lgo_score(const lgo_instance *inst,
              const uint8_t *bp_tour, const uint8_t *bp_pos,
              const uint16_t *field_bp, const uint16_t *field_pos,
              const uint8_t *hu_tour, const uint8_t *su_tour_init,
              double *scalars,
              double *tour_route_km,      /* [N_T] L_tour(g)                 */
              double *tour_time_h,        /* [N_T] T(g)                      */
              double *tour_E_h,           /* [N_T] E(g)                      */
              double *tour_wait_h,        /* [N_T] T_wait(g) after Alg. 2    */
              double *tour_len_km,        /* [N_T] L(g)                      */
              int64_t *bp_supply_q,       /* [N_B] S_q(b)                    */
              int64_t *field_shuttles,    /* [N_F] eq. (4) count             */
              uint8_t *su_tour_final);    /* [N_SU]                          */

/* lgo_score with the embedded HU assignment of PAPER.md:L190, L203 (R39) when hu_balance != 0; hu_tour_final
 * (may be NULL) receives the HU sets the cost was computed with (= the input for an infeasible plan). */
int lgo_score_ex(const lgo_instance *inst,
                 const uint8_t *bp_tour, const uint8_t *bp_pos,
                 const uint16_t *field_bp, const uint16_t *field_pos,
                 const uint8_t *hu_tour, const uint8_t *su_tour_init, int hu_balance,
                 double *scalars, double *tour_route_km, double *tour_time_h, double *tour_E_h,
                 double *tour_wait_h, double *tour_len_km, int64_t *bp_supply_q,
                 int64_t *field_shuttles, uint8_t *su_tour_final, uint8_t *hu_tour_final);

/* The HU assignment alone on explicit numbers (for hand traces): road_h[g] = L_tour(g)/v_HU, area_q[g] = H_q(g),
 * rate_q per unit; hu_tour in/out; time_h out = T(g); returns the accepted moves. */
int lgo_hu_balance(int32_t n_tours, const double *road_h, const int64_t *area_q, int32_t n_hu, const int64_t *rate_q,
                   uint8_t *hu_tour, double *time_h);

/* S6 alone (Algorithm 2) on explicit numbers, for traces B and C.
 * cap_q: capacities in quanta; su_tour in/out; wait_h out; returns accepted moves.    */
int lgo_su_local_min(int32_t n_tours, const double *E_h, const int32_t *n_hu,
                     int32_t n_su, const int64_t *cap_q, uint8_t *su_tour,
                     double kappa_h_per_t, double *wait_h);

/* eval = score o decode on host arrays; ids==NULL => ids = first_id + i. */
int lgo_eval_batch(const lgo_instance *inst, uint64_t seed, const uint64_t *ids,
                   uint64_t first_id, uint64_t n,
                   double *cost, double *path_km, double *makespan_h, uint8_t *feasible);
int lgo_decode_batch(const lgo_instance *inst, uint64_t seed, const uint64_t *ids,
                     uint64_t first_id, uint64_t n,
                     uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                     uint8_t *hu_tour, uint8_t *su_tour_init, uint8_t *su_tour_final);
/* S8: ordered min over ids [first_id, first_id+budget) of (cost bits, id). */
int lgo_search(const lgo_instance *inst, uint64_t seed, uint64_t first_id, uint64_t budget,
               double *best_cost, uint64_t *best_id);

/* ---- NEXT rows of the scope table: the paper's own search loop --------- */

/* Algorithm 1 steps 1-3: the nearest-neighbour initialisation
 * "a human scheduler may implicitly conduct".  Writes an explicit plan (same arrays as
 * lgo_decode).  Readings R31-R34 in DESIGN.md.                                           */
int lgo_init_plan(const lgo_instance *inst,
                  uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                  uint8_t *hu_tour, uint8_t *su_tour);

/* Step 8 (L158, L184): remove one vertex (field or BP) and reinsert it.  The three draws
 * w0,w1,w2 choose the vertex, the target BP / tour and the position (R35).  In place.    */
int lgo_apply_move(const lgo_instance *inst, uint32_t w0, uint32_t w1, uint32_t w2,
                   uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos);

/* Workers i = first_id .. first_id+n-1 of one iteration: x_i = move_i(x), C_i = cost(x_i)
 * (L163-165).  Draws = Philox block (seed; id, stream 5, block 0).                        */
int lgo_move_eval_batch(const lgo_instance *inst,
                        const uint8_t *bp_tour, const uint8_t *bp_pos,
                        const uint16_t *field_bp, const uint16_t *field_pos,
                        const uint8_t *hu_tour, const uint8_t *su_tour,
                        uint64_t seed, uint64_t first_id, uint64_t n,
                        double *cost, double *path_km, double *makespan_h, uint8_t *feasible);

/* Algorithm 1 steps 5-16 (L136-169) with the exploration rule eq. (5) (L177): n_iters
 * iterations of n_workers workers.  The plan arrays hold x_0 on entry (its SU assignment
 * is replaced by Alg. 2's result) and x* on return; hist_cost/hist_id (may be NULL) receive
 * (C_i*, i*) of every iteration.  eps_thresh = eps * 2^32 (u < eps <=> draw < eps_thresh). */
int lgo_local_search(const lgo_instance *inst,
                     uint8_t *bp_tour, uint8_t *bp_pos, uint16_t *field_bp, uint16_t *field_pos,
                     uint8_t *hu_tour, uint8_t *su_tour,
                     uint64_t seed, uint32_t n_iters, uint32_t n_workers, uint32_t eps_thresh,
                     double *best_cost, double *hist_cost, uint64_t *hist_id);

#ifdef __cplusplus
}
#endif
#endif
