/* lgx.h — C ABI of lgx: B200-native mass evaluation of biomass-logistics plans.
 *
 * Hot path of arxiv 1909.10286 (M. Graf Plessen, "GPU-accelerated Logistics Optimisation
 * for Biomass Production with Multiple Simultaneous Harvesters Tours, Fields and Plants";
 * citations are lines of /root/reference/PAPER.md): every candidate plan is decoded from
 * (seed, id), checked against the BP demand constraints (eq. (2)), scored by the
 * path-length criterion of §2.2 (L100-106) plus the maximum completion time (L190, L205)
 * after the embedded SU assignment of Algorithm 2 (L209-227), and reduced to a global
 * argmin (L167).  DESIGN.md states every reading (R1..R30) the paper leaves open.
 *
 * Conventions
 *  - extern "C", no exceptions.  Return 0 (LGX_OK) or a negative code.  The library reads no environment
 *    variables; every tuning knob is a flag of the descriptor or an lgx_instance_set_option key.  Process-wide
 *    state, all of it result-neutral: the opt-in shared-memory size of a kernel (set once, to the device maximum,
 *    when an instance that uses the kernel is created) and ONE cached workspace pool per device (the queue of
 *    feasible candidates is allocated stream-ordered from it and stays mapped between calls and instances;
 *    lgx_workspace_trim releases it).
 *  - Every compute call must run with the CUDA device the instance was created on as the current device
 *    (its images live there): otherwise LGX_EINVAL.
 *  - "d_" pointers are DEVICE pointers (caller-allocated, e.g. torch tensors' data_ptr());
 *    "h_" pointers and everything inside lgx_instance_desc are HOST pointers.
 *  - cuda_stream is a cudaStream_t passed as void* (NULL = default stream).
 *  - No CPU fallback: without a CUDA device every compute call returns LGX_ECUDA.
 */
#ifndef LGX_H
#define LGX_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LGX_OK        0
#define LGX_EINVAL   (-1)   /* bad argument / instance violates the documented ranges        */
#define LGX_ETOOBIG  (-2)   /* instance image or per-candidate state does not fit on an SM,
                               or a kernel limit below is exceeded                           */
#define LGX_ECUDA    (-3)   /* CUDA runtime error; text via lgx_strerror(LGX_ECUDA)          */
#define LGX_ENOMEM   (-4)
#define LGX_ESTATIC  (-5)   /* lgx_eval_batch_static: n above lgx_eval_batch_static_max()     */

/* Kernel limits of this build (beyond them lgx_instance_create returns LGX_ETOOBIG; the move kernels'
 * limits make lgx_move_eval_batch / lgx_local_search return LGX_ETOOBIG, the instance itself is still created). */
#define LGX_MAX_BPS         127   /* N_B: 7-bit BP ids in the plan-order entries                                */
#define LGX_MAX_SUS         128   /* N_SU: SU sets are 2 x 64-bit masks over capacity ranks                     */
#define LGX_MAX_MOVE_TOURS   64   /* N_T of the Algorithm-1 entry points: 64-bit sets of tours                  */
#define LGX_MAX_MOVE_HUS     64   /* N_HU of the Algorithm-1 entry points: 64-bit sets of HUs                   */

/* lgx_instance_desc.flags */
#define LGX_FLAG_HU_BALANCE 2u   /* lgx_move_eval_batch / lgx_local_search embed the HU assignment of PAPER.md:L190, L203 */
#define LGX_FLAG_FIX_FIELD_BP 8u /* a moved field is reinserted into its own BP (the assignment of fields to BPs is fixed:
                                    PAPER.md §2.6, Cases 2-3 L273); the target draw w1 is then unused for fields */
#define LGX_FLAG_MAKESPAN_FILTER 4u /* ... and discard (C_i = +inf, feasible stays 1) every worker whose makespan exceeds the
                                       best-so-far one = that of x* (of x in lgx_move_eval_batch): PAPER.md:L205, R38 */

/* Tuning flags: how the walk/finish kernel gets its distances.  Default: packed tables in shared memory while
 * they fit next to >= 256 candidates per SM, else the field x BP table + coordinates while that table is <= 32 KB,
 * else coordinates only.  D(u,v) is the same bit pattern in every mode (one rounding per operation, S0),
 * so results do not depend on these flags.  Both set => LGX_EINVAL.                                             */
#define LGX_FLAG_DIST_COORDS 16u /* vertex coordinates only, sqrt on the fly                                    */
#define LGX_FLAG_DIST_MIXED  32u /* field x BP table + coordinates for the field-to-field legs (if it fits)     */

/* lgx_instance_set_option keys: launch configuration only, never results.  Not to be called while a compute
 * call on the same instance is in flight.  Values outside the stated range => LGX_EINVAL.                      */
#define LGX_OPT_THREADS_A   1    /* threads per block of the decode/cut kernel: multiple of 32, 32 .. what fits */
#define LGX_OPT_THREADS_B   2    /* threads per block of the walk/finish kernel: multiple of 32, 32 .. what fits */
#define LGX_OPT_THREADS_MV  3    /* threads per block of the move kernels: multiple of 32, 64 .. what fits      */
#define LGX_OPT_CHUNK_LOG2  4    /* log2 of the candidates per kernel pair, 10 .. 26 (queue memory = chunk * record bytes) */
/* (key 6 was LGX_OPT_CUT_WARP, a one-candidate-per-warp decode/cut kernel that measured slower on every config and was
 * removed in round 3; profiles/r02_alt_cut_per_warp_paper_scale.md keeps the measurement.  The key is LGX_EINVAL now.) */
#define LGX_OPT_WALK_LOCKSTEP 7  /* 1: the warps of a walk/finish block draw their queue records together (one barrier per batch; they
                                    then share instruction-cache lines), 0: every warp on its own.  Only with coordinates (distance modes 1, 2;
                                    ignored with the tables, where it measured slower).  Default: 1 with coordinates and N_F < 1024 */
#define LGX_OPT_SQ_SHIFT    5    /* log2 of the replication of the s_q table in the decode/cut kernel's shared memory, 0 .. 5;
                                    synchronises the device, uploads a new image and then resets LGX_OPT_THREADS_A to its
                                    default for the new image size (set this key first).  On
                                    failure (LGX_ETOOBIG, LGX_ECUDA) the instance keeps its previous image and settings */

typedef struct lgx_instance lgx_instance;   /* opaque; owns host + device copies */

/* Problem statement (Table 1 L51-65 and the list under it, L65; §2.1).
 * All arrays are copied by lgx_instance_create; the caller may free them afterwards.   */
typedef struct {
  double   hq_x, hq_y;                       /* km; HQ, "at the origin" in §3.1 (L267)          */
  int32_t  n_fields;                         /* N_F, 1..65535                                    */
  const double *field_x, *field_y;           /* km, field centroids (Fig. 1, L21)                */
  const double *field_supply_t;              /* s_f, expected supply (t), eq. (2)/(3) L79-85     */
  const double *field_area_ha;               /* h_f (ha), L83                                    */
  int32_t  n_bps;                            /* N_B, 1..LGX_MAX_BPS (128..255: LGX_ETOOBIG)      */
  const double *bp_x, *bp_y;                 /* km                                               */
  const double *bp_demand_t;                 /* d_b^min (t), eq. (2)                         */
  int32_t  n_hu_total;                       /* N_HU^total, eq. (1); 1..255                  */
  const double *hu_rate_ha_per_h;            /* v_HU^area per unit (ha/h), L96 (ii), classes L75 */
  int32_t  n_su_total;                       /* N_SU^total, eq. (1); 1..LGX_MAX_SUS (129..255: LGX_ETOOBIG) */
  const double *su_capacity_t;               /* l_SU^load per unit (t), L87                      */
  int32_t  n_tours;                          /* N_T <= min(N_B, N_HU^total, N_SU^total) (L69)    */
  double   v_hu_road_kmh, v_su_road_kmh;     /* v_HU^edge, v_SU^edge (Table 1: 40, 40)           */
  double   v_infield_kmh;                    /* configs only; stored, not used by the cost (R24) */
  double   su_fill_h_per_t;                  /* kappa: t_SU^load = kappa * capacity (L96 (iii))  */
  double   w_path, w_time;                   /* cost = w_path*path_km + w_time*makespan_h (R1)   */
  uint32_t extra_field_thresh;               /* decoder knob: P(extra field) = thresh / 2^32     */
  uint32_t flags;                            /* OR of LGX_FLAG_* (other bits: LGX_EINVAL)         */
} lgx_instance_desc;

/* Instance encoder.  Quantises supply/area/demand/rate/capacity to Q=1024
 * quanta, builds the two shared-memory images (supply/demand quanta for the integer decode/cut kernel;
 * distance tables or coordinates and the unit tables for the walk/finish kernel) and uploads them.
 * Errors: LGX_EINVAL (null pointer, n_tours out of range, non-finite or negative input, zero
 * rate/capacity/velocity, counts above 65535 fields / 255 BPs, tours, HUs, SUs, unknown flag bits),
 * LGX_ETOOBIG (integer ranges: max s_q*N_SU + sum c_q, sum h_q, sum r_q, d_q must stay below 2^32
 * and sum s_q below 2^32 - 1; N_B > LGX_MAX_BPS or N_SU > LGX_MAX_SUS; or the per-candidate state does not fit in
 * 227 KB of shared memory), LGX_ECUDA, LGX_ENOMEM.                                          */
int lgx_instance_create (const lgx_instance_desc *desc, lgx_instance **out);
int lgx_instance_destroy(lgx_instance *inst);

/* Hands the workspace memory the library caches per device (see Conventions) back to the driver.  Safe at any
 * time no compute call is in flight; the next compute call maps what it needs again.  LGX_OK or LGX_ECUDA.    */
int lgx_workspace_trim(void);

/* Candidate decoder + tour simulator + demand check + Algorithm 2 + cost (a2..a6), one
 * candidate per thread.  ids: d_ids[i] if d_ids != NULL, else first_id + i.  Row i of every
 * output belongs to candidate i; any output pointer may be NULL.  Infeasible candidates
 * (eq. (2) violated) get feasible=0 and +inf in the three doubles.
 * Asynchronous on cuda_stream.                                                              */
int lgx_eval_batch(const lgx_instance *inst, uint64_t seed,
                   const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                   double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible,
                   void *cuda_stream);

/* Same, with HOST buffers: copies ids in (if given) and results out inside the call, which returns when every
 * output is in place.  Chunks of 2^21 candidates alternate between two internal streams: with page-locked host
 * buffers (cudaHostAlloc / cudaHostRegister, torch pin_memory) the copies of one chunk overlap the kernels of the
 * next; pageable buffers work too, chunk after chunk.  Any output pointer may be NULL.  Used for the
 * end-to-end number of lgx_eval_batch in bench.py.                                          */
int lgx_eval_batch_host(const lgx_instance *inst, uint64_t seed,
                        const uint64_t *h_ids, uint64_t first_id, uint64_t n,
                        double *h_cost, double *h_path_km, double *h_makespan_h, uint8_t *h_feasible);

/* lgx_eval_batch for callers that must not allocate device memory at call time.
 *
 * Who needs it: lgx_eval_batch takes the queue between its two kernels from the library's memory pool, and a pool
 * that has to grow goes to the driver for memory.  Some hosts cannot afford or are not allowed that: a service whose
 * start-up phase hands every free byte of HBM to another owner (a tensor framework's caching allocator, a
 * pre-sized cache), so that a later request to the driver simply fails; a control or serving loop with a latency
 * bound, because driver allocation and release may stall the whole device for an unbounded time; a plug-in running
 * under a host application that forbids allocator calls after initialisation.  For them the queue and the
 * kernels' counters live in ONE fixed array of LGX_STATIC_SCRATCH_BYTES (16 MiB) that is part of the library's
 * device image: a GPU carries those 16 MiB from the moment the CUDA runtime loads that image on it (with eager
 * module loading when the library is first used there, otherwise at the latest at the first call below) until
 * the process exits, whether the call is used again or not; nothing releases them earlier.  The call itself
 * issues one 64-byte memset and the two kernels on cuda_stream: no cudaMalloc / cudaFree, no pool, no stream or
 * event creation, no library routine that allocates.  Inputs and outputs are the caller's, exactly as in
 * lgx_eval_batch (same arguments, same results bit for bit, asynchronous on cuda_stream).
 *
 * Limit: the whole call is one kernel pair, so n queue records must fit in the array:
 * n <= lgx_eval_batch_static_max(inst) = (16 MiB - a header of 64 B + 16 B per SM) / record bytes, rounded down
 * to a multiple of 32 (record bytes = lgx_instance_query what 11: about 135 000 candidates on the 100-field
 * config, about 6 700 with 1200 fields).  A larger n returns LGX_ESTATIC before anything is launched; split the
 * ids over several calls on the same stream instead.
 *
 * First call on a device: the library looks up the array's device address (cudaGetSymbolAddress, with the
 * instance's device current) and remembers it per device; that call loads the module if it is not loaded yet.
 * Make this first call during set-up, outside any stream capture; a small n is enough.  Later calls only read
 * the remembered address.
 *
 * Sharing: there is one array per device, not per instance, stream or call, and it keeps the previous call's
 * contents; each call zeroes the counters it needs before its kernels start.  Two calls may therefore follow each
 * other on ONE stream (stream order keeps them apart), but calls that can overlap on the GPU (different streams
 * without an event between them, different host threads on different streams, two instances at once) race on the
 * queue and give wrong results.  Callers that need concurrency use lgx_eval_batch.                             */
#define LGX_STATIC_SCRATCH_BYTES (16u << 20)
int lgx_eval_batch_static(const lgx_instance *inst, uint64_t seed,
                          const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                          double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible,
                          void *cuda_stream);
/* Largest n lgx_eval_batch_static accepts for this instance (host-only arithmetic, no CUDA call). */
int lgx_eval_batch_static_max(const lgx_instance *inst, uint64_t *max_n);

/* a2..a7: evaluate ids [first_id, first_id + n) and return the ordered minimum of
 * (cost bit pattern, id): lowest cost, lowest id on ties (R29).  No feasible
 * candidate => *h_best_cost = +inf and *h_best_id = first_id.  n == 0 => LGX_EINVAL.
 * Synchronises cuda_stream before returning; results go to host pointers.                  */
int lgx_search_range(const lgx_instance *inst, uint64_t seed, uint64_t first_id, uint64_t n,
                     double *h_best_cost, uint64_t *h_best_id, void *cuda_stream);
/* lgx_search(budget) == lgx_search_range(0, budget). */
int lgx_search(const lgx_instance *inst, uint64_t seed, uint64_t budget,
               double *h_best_cost, uint64_t *h_best_id, void *cuda_stream);

/* Diagnostic export of decoded plans (needed for the "plans bit-exact" parity clause; SURVEY §8(b) lists it
 * without first_id — added so that implicit id ranges work as in lgx_eval_batch).
 * Layouts: d_bp_tour/d_bp_pos [n][N_B] (tour of BP b, its position on that tour);
 * d_field_bp/d_field_pos [n][N_F] (BP of field f, its position in that BP's list);
 * d_hu_tour [n][N_HU]; d_su_tour_init / d_su_tour_final [n][N_SU] (before / after Alg. 2;
 * equal for infeasible candidates).  Any pointer may be NULL.  Asynchronous.               */
int lgx_decode_batch(const lgx_instance *inst, uint64_t seed,
                     const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                     uint8_t *d_bp_tour, uint8_t *d_bp_pos,
                     uint16_t *d_field_bp, uint16_t *d_field_pos,
                     uint8_t *d_hu_tour, uint8_t *d_su_tour_init, uint8_t *d_su_tour_final,
                     void *cuda_stream);

/* Introspection for bench.py / tests: what = 0 image bytes (both images), 1 threads per block
 * of the decode/cut kernel, 2 blocks in the persistent grid, 3 its dynamic shared memory
 * bytes per block, 4 distance mode (0 = packed tables in smem, 1 = coordinates, 2 = field x BP table + coordinates),
 * 5 per-candidate state bytes of the decode/cut kernel, 6 SM count, 7 kernel launches issued
 * so far through this instance, 8 / 9 threads per block / shared memory bytes of the walk/finish
 * kernel, 10 candidates per kernel pair (chunk), 11 bytes per queue record, 15 / 16 threads per
 * block / shared memory bytes of the move kernels (Algorithm 1 entry points below; 0 threads: they do not fit),
 * 17 log2 of the s_q replication, 18 threads per block of the decode/cut kernel in lgx_decode_batch,
 * 19 per-candidate state bytes of the walk/finish kernel, 20 the instance's CUDA device, 24 LGX_OPT_WALK_LOCKSTEP
 * (21-23 belonged to the removed per-warp decode/cut kernel: LGX_EINVAL).                                      */
int lgx_instance_query(const lgx_instance *inst, int what, int64_t *out);

/* Launch-configuration knobs (LGX_OPT_* above).  Results never depend on them.              */
int lgx_instance_set_option(lgx_instance *inst, int key, int64_t value);

/* Per-kernel timing for bench.py's roofline: when enabled, every lgx_search(_range) call
 * brackets each kernel launch with CUDA events on the caller's stream and accumulates the
 * device time; lgx_instance_query what = 12 / 13 return the nanoseconds spent in the
 * decode/cut / walk/finish kernels, 14 the number of kernel pairs timed.  Enabling or disabling
 * resets the counters.                                                                     */
int lgx_instance_set_timing(lgx_instance *inst, int enable);

/* ---- The paper's own search loop, Algorithm 1 -----------
 * A plan x is six HOST arrays (the layouts of lgx_decode_batch, one row): h_bp_tour/h_bp_pos [N_B],
 * h_field_bp/h_field_pos [N_F], h_hu_tour [N_HU], h_su_tour [N_SU].  A plan passed IN must be valid
 * (every BP on one tour at a unique position 0..len-1, every field on one BP likewise, every tour with
 * >= 1 HU and >= 1 SU; tours without BPs and BPs without fields are allowed, L184), else LGX_EINVAL.
 * LGX_ETOOBIG when the move kernels do not fit this instance (what = 15 reports 0): their tables (about 64 B per
 * field + 16 B per tour and SU) and three plans live in shared memory next to >= 64 workers' rows, and the workers
 * keep 64-bit sets of tours and of HUs (N_T <= 64, N_HU <= 64).
 * With desc.flags & LGX_FLAG_HU_BALANCE the workers (and the scoring of x_0) first rebalance the HUs over the tours
 * (R39): Algorithm 2's procedure on the completion times T(g), donor units by
 * rising rate; x_{i*} and x* then carry the HU sets they were scored with (h_hu_tour is in/out).
 * Readings R31-R39 cover what the paper leaves open.                                 */

/* Steps 1-3 (L122-126, L171-173): the nearest-neighbour initialisation "a human scheduler may tacitly
 * conduct" (Case 1, L273).  HUs: floor(N_HU/N_T) per tour in index order, the residual on the last tour;
 * SUs dealt round-robin over the (capacity, unit) order; BPs: nearest-neighbour chain from HQ cut into
 * N_T consecutive runs; fields, in index order, to their closest BP still short of its demand, else to
 * their closest BP; per BP a nearest-neighbour order from HQ.  Runs on the device (one block); writes
 * the six host arrays; synchronises cuda_stream.                                                    */
int lgx_init_plan(const lgx_instance *inst,
                  uint8_t *h_bp_tour, uint8_t *h_bp_pos, uint16_t *h_field_bp, uint16_t *h_field_pos,
                  uint8_t *h_hu_tour, uint8_t *h_su_tour, void *cuda_stream);

/* Steps 8-12 for workers i = first_id .. first_id+n-1 (L158-165, L184): x_i = x with ONE vertex removed
 * and reinserted, scored like lgx_eval_batch (eq. (2), Algorithm 2 starting from x's SU sets, cost).
 * Worker i draws Philox block (seed; counter = (i, stream 5, block 0)) = (w0, w1, w2, -):
 * v = floor(w0 (N_F+N_B) / 2^32) is a field (v < N_F) or BP v-N_F; a field goes to BP floor(w1 N_B / 2^32),
 * a BP (with all its fields) to tour floor(w1 N_T / 2^32); position floor(w2 (len+1) / 2^32), len = the
 * target list's length after the removal.  Outputs are DEVICE pointers (any may be NULL), row i-first_id.
 * The plan arrays are copied into a buffer of the library's before the call returns (the caller may change them
 * at once, page-locked or not); the upload from that buffer and the kernel are asynchronous on cuda_stream.  */
int lgx_move_eval_batch(const lgx_instance *inst,
                        const uint8_t *h_bp_tour, const uint8_t *h_bp_pos,
                        const uint16_t *h_field_bp, const uint16_t *h_field_pos,
                        const uint8_t *h_hu_tour, const uint8_t *h_su_tour,
                        uint64_t seed, uint64_t first_id, uint64_t n,
                        double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible,
                        void *cuda_stream);

/* Steps 4-16 (L133-169) with the exploration rule eq. (5) (L177), all n_iters iterations inside ONE
 * persistent cooperative kernel.  x_0 comes in through the plan arrays (its SU sets are replaced by what
 * Algorithm 2 leaves them with) and x* goes out through them; *h_best_cost = C*.  Iteration k starts from
 * x* if word 0 of Philox block (seed; (k, stream 6, block 0)) < eps_thresh (= eps 2^32), else from the
 * winner of iteration k-1; its workers are ids k n_workers .. (k+1) n_workers - 1 of lgx_move_eval_batch;
 * i* = the ordered minimum of (cost bits, id).  If C_i* is finite x_old <- x_i* (with the SU sets
 * Algorithm 2 gave it) and x* <- x_i* when C_i* < C*.  h_hist_cost / h_hist_id [n_iters] (may be NULL)
 * receive (C_i*, i*) of every iteration.  HU sets stay as given (R20).  Synchronises cuda_stream.
 * n_workers == 0 => LGX_EINVAL; n_iters == 0 scores x_0 only.                                        */
int lgx_local_search(const lgx_instance *inst,
                     uint8_t *h_bp_tour, uint8_t *h_bp_pos, uint16_t *h_field_bp, uint16_t *h_field_pos,
                     uint8_t *h_hu_tour, uint8_t *h_su_tour,
                     uint64_t seed, uint32_t n_iters, uint32_t n_workers, uint32_t eps_thresh,
                     double *h_best_cost, double *h_hist_cost, uint64_t *h_hist_id, void *cuda_stream);

/* Diagnostic self-test of a device routine against its library counterpart, on the current device's default stream
 * (synchronous).  what = 0: the in-line correctly rounded square root of the walk/finish kernel against __dsqrt_rn
 * on n pseudo-random arguments drawn from `seed` (squared coordinate differences, random mantissas over 120 binades,
 * exact squares and their neighbours); h_out[0] = arguments checked, h_out[1] = mismatches (must be 0).
 * what = 1..5: issue-rate microbenchmark of one execution pipe, n = loop iterations (2^14 takes about a millisecond):
 * 1 IMAD.WIDE.U32 (Philox's 32x32->64 products), 2 LOP3 (the ALU pipe), 3 LDS.U8 + STS.U8 on per-thread shared-memory
 * columns, 4 DFMA (the FP64 pipe), 5 MUFU.RSQ64H (the square root's seed); eight independent chains per thread, two
 * blocks of 1024 threads per SM.  h_out[0] = warp-instructions of that kind issued by the whole grid, h_out[1] = clock
 * cycles of the slowest block: h_out[0] / h_out[1] / SMs = the pipe's sustained warp-instructions per clock per SM
 * (bench.py: roofline.pipe_peaks).  `seed` is unused there.
 * Other `what`, n == 0 or a null pointer => LGX_EINVAL.                                                         */
int lgx_selftest(int what, uint64_t n, uint64_t seed, uint64_t *h_out);

const char *lgx_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
