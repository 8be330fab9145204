// lgx_moves.cuh — the paper's own search loop as CUDA for sm_100a:
//   lgx_init_plan_k      Algorithm 1 steps 1-3: nearest-neighbour initialisation
//   lgx_move_eval_k      step 8 + cost for a batch of workers (L158-165, L184): every worker applies ONE
//                        remove/reinsert move to the broadcast incumbent x and scores the result
//   lgx_local_search_k   steps 4-16 (L133-169) with the exploration rule eq. (5) (L177): ONE persistent
//                        cooperative kernel runs all N_iters iterations; nothing returns to the host in between
// Product code (CUDA path); shares nothing with oracle/.
//
// Design (B200-first, not the paper's host loop).  The paper broadcasts x, collects every C_i on the host,
// takes the argmin there and rebuilds x_{i*} by replaying the random stream (L163-169, L233).  Here the
// incumbent lives in the shared memory of every SM as a FLAT SEQUENCE: the fields in plan order (tour 0's
// first BP's fields, ...), each entry carrying its BP.  A move (one field, or one BP with all its fields,
// L184) is a rotation of one block of that sequence, so a worker never materialises x_i: three breakpoints
// (worker position -> incumbent index) describe it.  After the block/grid reduction of (cost bits, id) every
// block rebuilds x_{i*} ITSELF from the winning id ("identical random process control", L233, taken one step
// further): the only inter-SM traffic per iteration is one slot of (cost, id, SU / HU sets, makespan) per block
// and one grid barrier.
//
// Evaluation is incremental and exact (mv_eval): per iteration and SM the encoder tabulates, for every position of
// the incumbent, its two legs, its shuttle count and the tour's running sums before it, and per tour / per BP the
// finished sums; a worker re-adds only what its move changes — the tail of the <= 2 touched tours from the first
// changed position, the mean leg of the two BPs of a field move, the shuttle sums of tours whose SU set its
// Algorithm 2 changed (tabulated too when the set is one unit away) — and reads the rest: same operands in the same
// order, hence the same bits.  The workers of up to kSuper block rounds are sorted by (touched tours, first changed
// position) so that a warp's lanes do the same work, and the warps draw sorted chunks from a shared counter.
//
// FP64 arithmetic follows DESIGN.md S4-S7 operation by operation (compiled with -fmad=false), in the
// oracle's summation order, so costs are bit-equal.
#pragma once
#include <cooperative_groups.h>
#include "lgx_kernels.cuh"

namespace lgx {
namespace cg = cooperative_groups;

constexpr int      kMvThreads = 512;            // __launch_bounds__ of the move kernels
constexpr uint32_t kNone      = 0xFFFFFFFFu;
constexpr uint32_t kSortKeys  = 1024;           // (tour pair, position bucket | BP move) keys of the worker sort

// Shared-memory layout of the move kernels (byte offsets from the start of dynamic shared memory):
//   vertex coordinates | demand quanta | tail of image C (from offc_cs) | incumbent tables | plan store | per-thread state rows
struct MvHdr {
  uint32_t off_xy;      // f64x2 [1 + n_b + n_f]  vertex coordinates: HQ, BPs, fields
  uint32_t off_dq;      // u32 [n_b]      demand quanta
  uint32_t off_c;       // tail of image C: byte x of image C (x >= offc_cs) sits at off_c + x - offc_cs
  // the incumbent's positions in plan order, one array per quantity (the walks read 4 or 8 bytes per position and lane)
  uint32_t off_pfb;     // u32 [n_f]      f | b << 16
  uint32_t off_psq;     // u32 [n_f]      s_q[f]
  uint32_t off_phq;     // u32 [n_f]      h_q[f]
  uint32_t off_term;    // f64 [n_f]      N * D(f, b): the position's shuttle term under the incumbent's SU sets (N = eq. (4) count)
  uint32_t off_legx;    // f64 [n_f]      D(predecessor on the tour or HQ, f)
  uint32_t off_legy;    // f64 [n_f]      D(f, b)
  uint32_t off_prex;    // f64 [n_f]      the tour's running route sum BEFORE this position
  uint32_t off_prey;    // f64 [n_f]      the tour's running shuttle sum BEFORE this position
  uint32_t off_posf;    // u16 [n_f]      position of field f in plan order
  uint32_t off_bp;      // u32x2 [n_b]    x = start | len << 16;  y = plan index | tour << 8 | pos << 16
  uint32_t off_bsh;     // u32x2 [n_b]    S_q(b), area quanta of b's fields
  uint32_t off_bpq;     // f64 [n_b]      mean field->BP leg of b (0 without fields)
  uint32_t off_pre;     // u16 [n_b + 1]  start of the BP at plan index j; pre[n_b] = n_f
  uint32_t off_bpat;    // u8 [n_b]       BP at plan index j
  uint32_t off_cnt;     // u32 [n_b]      scratch: fields per BP
  uint32_t off_tpl;     // u32 [n_t]      first plan index | BPs on the tour << 8
  uint32_t off_thu;     // u32x2 [n_t]    n_HU(g), R_g of the incumbent (fixed during a search unless the HU assignment is embedded: R20, R39)
  uint32_t off_thm;     // u64 [n_t]      HU membership by rate rank
  uint32_t off_tsn;     // u32x2 [n_t]    S_g = capacity quanta of the tour's SUs, n_g = their number
  uint32_t off_tmask;   // u64 [n_t*MW]   SU membership by capacity rank
  uint32_t off_trng;    // u32x2 [n_t]    the tour's positions [begin, end) in plan order
  uint32_t off_tst;     // f64 [7][n_t]   the incumbent's L_tour(g), E(g), T(g), T_wait(g), shuttle sum(g), route sum before the leg back to HQ, L_tour(g)/v_HU
  uint32_t off_thq;     // u32 [n_t]      H_q(g)
  uint32_t off_sv;      // f64 [n_t][2][n_su]  the tour's shuttle sum with one SU of capacity class r removed (0) / added (1)
  uint32_t off_misc;    // u32 [16]       [0] BPs that miss their demand (eq. (2)); [4..9] the move being applied
  uint32_t off_sort;    // u32 [kSortKeys + 2]  counting sort of the workers by the tours they touch; the warps' draw counter
  uint32_t off_order;   // u16 [kSuper * kMvThreads]  sorted workers: round << 10 | thread
  uint32_t off_plans;   // 3 plans (x*, x_old, scratch); the batch kernel uses the first
  uint32_t plan_bytes;  // one plan: bp_tour u8[n_b] | bp_pos u8[n_b] | field_bp u16[n_f] | field_pos u16[n_f] | SU masks u64[n_t*MW] | HU masks u64[n_t]
  uint32_t pl_bpos, pl_fbp, pl_fpos, pl_mask, pl_hmask;
  uint32_t off_state;   // per-thread rows (64-bit region, then 32-bit region)
  uint32_t m64_w, m64_mask, m64_bmask, m64_rows;
  uint32_t m32_s, m32_rows;
  uint32_t m64_t, m64_hmask, m64_bhmask, m32_r;   // rows of the embedded HU assignment (only with LGX_FLAG_HU_BALANCE)
  uint32_t slot_words;  // 64-bit words per block slot: cost bits, id, SU masks, HU masks
  uint32_t pad_[2];
};

struct MvParams {
  ImgHdr          H;
  MvHdr           M;
  const uint8_t  *image, *image_c;      // device copies of the instance images (global memory)
  const double2  *xy;                   // vertex coordinates (global memory)
  uint32_t        rk[20];               // Philox round keys of the seed
  // the plan x (device arrays; in for the batch kernel, in/out for the search)
  uint8_t *bp_tour, *bp_pos; uint16_t *field_bp, *field_pos; uint8_t *hu_tour, *su_tour;
  // batch: workers first_id .. first_id + n - 1
  uint64_t first_id, n;
  double *cost, *path_km, *makespan_h; uint8_t *feasible;
  // search
  uint32_t n_iters, n_workers, eps_thresh;
  unsigned long long *slots;            // [2][gridDim.x][slot_words]
  double *hist_cost; unsigned long long *hist_id;   // [n_iters] or nullptr
  double *best_cost;
};

#define MV_TAB(type, off) (reinterpret_cast<type *>(sm + (off)))
#define MV_CTAB(type, offc) (reinterpret_cast<const type *>(sm + (P.M.off_c + ((offc) - P.H.offc_cs))))

// ------------------------------------------------------------------ plan -> shared memory

// Copy the plan arrays from global memory into a plan slot; SU sets become masks over capacity ranks.
// HU sets likewise, over rate ranks (at most 64 HUs).
template <int MASKW>
__device__ void mv_load_plan(const MvParams &P, uint8_t *sm, uint8_t *plan, uint32_t tid, uint32_t T)
{
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  const uint32_t n_f = H.n_f, n_b = H.n_b, n_t = H.n_t;
  for (uint32_t b = tid; b < n_b; b += T) { plan[b] = P.bp_tour[b]; plan[M.pl_bpos + b] = P.bp_pos[b]; }
  uint16_t *fb = reinterpret_cast<uint16_t *>(plan + M.pl_fbp), *fp = reinterpret_cast<uint16_t *>(plan + M.pl_fpos);
  for (uint32_t f = tid; f < n_f; f += T) { fb[f] = P.field_bp[f]; fp[f] = P.field_pos[f]; }
  if (tid == 0) {
    uint64_t *mk = reinterpret_cast<uint64_t *>(plan + M.pl_mask), *hm = reinterpret_cast<uint64_t *>(plan + M.pl_hmask);
    const uint8_t *rank_of = MV_CTAB(uint8_t, H.offc_rank), *hrank_of = MV_CTAB(uint8_t, H.offc_hrank);
    for (uint32_t i = 0; i < n_t * MASKW; ++i) mk[i] = 0ull;
    for (uint32_t g = 0; g < n_t; ++g) hm[g] = 0ull;
    for (uint32_t u = 0; u < (uint32_t)H.n_su; ++u) { const uint32_t r = rank_of[u]; mk[P.su_tour[u] * MASKW + (r >> 6)] |= 1ull << (r & 63u); }
    for (uint32_t u = 0; u < (uint32_t)H.n_hu; ++u) hm[P.hu_tour[u]] |= 1ull << hrank_of[u];
  }
  __syncthreads();
}

// Incumbent tables from a plan slot (block-wide; ends with a barrier): the flat sequence with its legs and
// shuttle counts, and per tour everything a worker needs of the tours its move does not touch.
template <int MASKW>
__device__ void mv_encode(const MvParams &P, uint8_t *sm, const uint8_t *plan, uint32_t tid, uint32_t T)
{
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  const uint32_t n_f = H.n_f, n_b = H.n_b, n_t = H.n_t;
  const uint8_t *p_bt = plan, *p_bp = plan + M.pl_bpos;
  const uint16_t *p_fb = reinterpret_cast<const uint16_t *>(plan + M.pl_fbp), *p_fp = reinterpret_cast<const uint16_t *>(plan + M.pl_fpos);
  const uint64_t *p_mk = reinterpret_cast<const uint64_t *>(plan + M.pl_mask);
  const uint32_t *dq = MV_TAB(const uint32_t, M.off_dq);
  const uint32_t *cs = MV_CTAB(uint32_t, H.offc_cs);
  const double   *rcp = MV_CTAB(double, H.offc_rcp);
  uint32_t *cnt = MV_TAB(uint32_t, M.off_cnt);
  uint2 *bp = MV_TAB(uint2, M.off_bp);
  uint2 *trng = MV_TAB(uint2, M.off_trng);
  uint2 *tsn = MV_TAB(uint2, M.off_tsn);
  uint64_t *tmask = MV_TAB(uint64_t, M.off_tmask);
  uint32_t *misc = MV_TAB(uint32_t, M.off_misc);
  for (uint32_t b = tid; b < n_b; b += T) cnt[b] = 0u;
  __syncthreads();
  for (uint32_t f = tid; f < n_f; f += T) atomicAdd(&cnt[p_fb[f]], 1u);
  __syncthreads();
  if (tid == 0) {
    uint32_t *tpl = MV_TAB(uint32_t, M.off_tpl);
    uint16_t *pre = MV_TAB(uint16_t, M.off_pre);
    uint8_t *bpat = MV_TAB(uint8_t, M.off_bpat);
    for (uint32_t g = 0; g < n_t; ++g) tpl[g] = 0u;
    for (uint32_t b = 0; b < n_b; ++b) tpl[p_bt[b]] += 0x100u;
    uint32_t acc = 0;
    for (uint32_t g = 0; g < n_t; ++g) { const uint32_t len = tpl[g] >> 8; tpl[g] = acc | (len << 8); acc += len; }
    for (uint32_t b = 0; b < n_b; ++b) bpat[(tpl[p_bt[b]] & 0xFFu) + p_bp[b]] = (uint8_t)b;
    acc = 0;
    for (uint32_t j = 0; j < n_b; ++j) {
      const uint32_t b = bpat[j], len = cnt[b];
      pre[j] = (uint16_t)acc;
      bp[b] = make_uint2(acc | (len << 16), j | ((uint32_t)p_bt[b] << 8) | ((uint32_t)p_bp[b] << 16));
      acc += len;
    }
    pre[n_b] = (uint16_t)acc;
    for (uint32_t g = 0; g < n_t; ++g) { const uint32_t j0 = tpl[g] & 0xFFu, j1 = j0 + (tpl[g] >> 8); trng[g] = make_uint2(pre[j0], pre[j1]); }
  }
  if (tid >= 32u) {
    for (uint32_t g = tid - 32u; g < n_t; g += T - 32u) {
      uint32_t S = 0, n = 0;
#pragma unroll
      for (int i = 0; i < MASKW; ++i) {
        uint64_t w = p_mk[g * MASKW + i];
        tmask[g * MASKW + i] = w;
        n += (uint32_t)__popcll(w);
        while (w) { const int r = __ffsll((long long)w) - 1; w &= w - 1; S += cs[64 * i + r]; }
      }
      tsn[g] = make_uint2(S, n);
      // n_HU(g), R_g = sum of the tour's rate quanta (L69; R7)
      const uint32_t *hrs = MV_CTAB(uint32_t, H.offc_hrs);
      uint64_t hw = reinterpret_cast<const uint64_t *>(plan + M.pl_hmask)[g];
      MV_TAB(uint64_t, M.off_thm)[g] = hw;
      uint32_t R = 0;
      const uint32_t nh = (uint32_t)__popcll(hw);
      while (hw) { const int r = __ffsll((long long)hw) - 1; hw &= hw - 1; R += hrs[r]; }
      MV_TAB(uint2, M.off_thu)[g] = make_uint2(nh, R);
    }
  }
  __syncthreads();
  uint32_t *pfb = MV_TAB(uint32_t, M.off_pfb), *psq = MV_TAB(uint32_t, M.off_psq), *phq = MV_TAB(uint32_t, M.off_phq);
  uint16_t *posf = MV_TAB(uint16_t, M.off_posf);
  const uint2 *sh = reinterpret_cast<const uint2 *>(P.image_c + H.offc_sh);  // {s_q, h_q} per field (global, L2-resident)
  for (uint32_t f = tid; f < n_f; f += T) {
    const uint32_t b = p_fb[f];
    const uint32_t pos = (bp[b].x & 0xFFFFu) + p_fp[f];
    const uint2 q = sh[f];
    pfb[pos] = f | (b << 16); psq[pos] = q.x; phq[pos] = q.y;
    posf[f] = (uint16_t)pos;
  }
  __syncthreads();
  // the two legs of every position of the incumbent (S0: one rounding per operation) and its shuttle term
  // N * D(f, b) under the tour's SU set (eq. (4); R4)
  const double2 *xy = MV_TAB(const double2, M.off_xy);
  double *legx = MV_TAB(double, M.off_legx), *legy = MV_TAB(double, M.off_legy), *term = MV_TAB(double, M.off_term);
  for (uint32_t p = tid; p < n_f; p += T) {
    const uint32_t e = pfb[p];
    const uint32_t f = e & 0xFFFFu, b = e >> 16;
    uint32_t pred = 0u;                                                        // HQ: first field of its tour (L21)
    if (p > 0u) { const uint32_t ep = pfb[p - 1u]; if (((bp[ep >> 16].y ^ bp[b].y) & 0xFF00u) == 0u) pred = 1u + n_b + (ep & 0xFFFFu); }
    const double ly = edge_from_xy(xy, 1u + n_b + f, 1u + b);
    const uint2 sn = tsn[(bp[b].y >> 8) & 0xFFu];
    legx[p] = edge_from_xy(xy, pred, 1u + n_b + f); legy[p] = ly;
    term[p] = __dmul_rn((double)shuttle_count(psq[p], sn.y, sn.x, 0xFFFFFFFFu / sn.x), ly);
  }
  __syncthreads();
  // per tour, one lane each: the walk of DESIGN.md S4 / S7 over the tour's positions, in order; it also leaves the
  // running sums before every position (prex, prey) and the per-BP supplies, areas and mean legs
  uint2 *bsh = MV_TAB(uint2, M.off_bsh);
  double *bpq = MV_TAB(double, M.off_bpq);
  for (uint32_t b = tid; b < n_b; b += T) { bsh[b] = make_uint2(0u, 0u); bpq[b] = 0.0; }
  __syncthreads();
  {
    const uint2 *thu = MV_TAB(const uint2, M.off_thu);
    double *tst = MV_TAB(double, M.off_tst);
    double *prex = MV_TAB(double, M.off_prex), *prey = MV_TAB(double, M.off_prey);
    uint32_t *thq = MV_TAB(uint32_t, M.off_thq);
    const uint32_t n_warps = T >> 5;
    if ((tid & 31u) == 0u)
      for (uint32_t g = tid >> 5; g < n_t; g += n_warps) {
        const uint2 r = trng[g];
        double Lt = 0.0, sd = 0.0, sumE = 0.0, shut = 0.0;
        uint32_t Hq = 0, Sq = 0, Hb = 0, k = 0, m = 0, b_cur = kNone, f_last = 0;
        for (uint32_t p = r.x; p < r.y; ++p) {
          const uint32_t e = pfb[p], sq_p = psq[p], hq_p = phq[p];
          const double lgx = legx[p], lgy = legy[p];
          const uint32_t b = e >> 16;
          if (b != b_cur) {
            if (b_cur != kNone) {
              const double q = div_small(sd, k, rcp);
              bsh[b_cur] = make_uint2(Sq, Hb); bpq[b_cur] = q;
              sumE = __dadd_rn(sumE, q); ++m;
            }
            b_cur = b; sd = 0.0; Sq = 0u; Hb = 0u; k = 0u;
          }
          prex[p] = Lt; prey[p] = shut;
          Lt = __dadd_rn(Lt, lgx); sd = __dadd_rn(sd, lgy); Hq += hq_p; Hb += hq_p; Sq += sq_p; ++k;
          shut = __dadd_rn(shut, term[p]);
          f_last = e & 0xFFFFu;
        }
        double E = 0.0;
        const double lt_open = Lt;
        if (b_cur != kNone) {
          const double q = div_small(sd, k, rcp);
          bsh[b_cur] = make_uint2(Sq, Hb); bpq[b_cur] = q;
          sumE = __dadd_rn(sumE, q); ++m;
          Lt = __dadd_rn(Lt, edge_from_xy(xy, 1u + n_b + f_last, 0u));
          E = __ddiv_rn(__dmul_rn(2.0, div_small(sumE, m, rcp)), H.v_su);
        }
        const uint2 hu = thu[g]; const uint2 sn = tsn[g];
        Mask<MASKW> mk;
#pragma unroll
        for (int i = 0; i < MASKW; ++i) mk.w[i] = tmask[g * MASKW + i];
        tst[g] = Lt; tst[n_t + g] = E;
        const double road = __ddiv_rn(Lt, H.v_hu);
        tst[2u * n_t + g] = __dadd_rn(road, __ddiv_rn((double)Hq, (double)hu.y));
        tst[6u * n_t + g] = road;
        tst[3u * n_t + g] = wait_time(E, sn.x, cs[mask_top(mk)], hu.x, H.kappa, rcp);
        tst[4u * n_t + g] = shut;
        tst[5u * n_t + g] = lt_open;
        thq[g] = Hq;
      }
  }
  __syncthreads();
  if (tid == 0) {                                   // eq. (2) (L79) over all BPs: a BP without fields has S_q = 0
    uint32_t bad = 0;
    for (uint32_t b = 0; b < n_b; ++b) bad += (bsh[b].x < dq[b]) ? 1u : 0u;
    misc[0] = bad;
  }
  // Shuttle sums of every tour under the SU sets one Algorithm-2 move away (one unit of capacity class r removed or
  // added): a worker whose Algorithm 2 changed an untouched tour that way looks the sum up instead of walking it.
  // One thread per (tour, direction, class); a class is named by the first rank holding its capacity.
  {
    const uint32_t n_su = H.n_su;
    double *sv = MV_TAB(double, M.off_sv);
    for (uint32_t task = tid; task < n_t * 2u * n_su; task += T) {
      const uint32_t r0 = task % n_su, dir = (task / n_su) & 1u, g = task / (2u * n_su);
      if (r0 > 0u && cs[r0] == cs[r0 - 1u]) continue;
      const uint2 sn = tsn[g];
      if (dir == 0u && (sn.y < 2u || sn.x <= cs[r0])) continue;
      const uint32_t n2 = dir ? sn.y + 1u : sn.y - 1u, C2 = dir ? sn.x + cs[r0] : sn.x - cs[r0];
      const uint32_t magic = 0xFFFFFFFFu / C2;
      const uint2 r = trng[g];
      double shut = 0.0;
      for (uint32_t p = r.x; p < r.y; ++p) shut = __dadd_rn(shut, __dmul_rn((double)shuttle_count(psq[p], n2, C2, magic), legy[p]));
      sv[task] = shut;
    }
  }
  __syncthreads();
}

// ------------------------------------------------------------------ step 8: one remove/reinsert move

// The moved block [a, a+len) of the incumbent's sequence reappears at position c of the worker's sequence.
struct Move {
  uint32_t a, len, c;
  uint32_t fld_b;     // field move: the BP the moved field now belongs to; else kNone
  uint32_t g1, g2;    // the tours the move touches: source and target (kNone, kNone: no move)
  uint32_t src;       // field move: the BP the field leaves; BP move: the moved BP
  uint32_t jo, jq;    // BP move: its plan index before / after the move (0, 0 for a field move)
};

// PAPER.md:L158, L184; R35: v = below(w0, N_F+N_B) picks a field or a BP ("since N_F >> N_B it is
// more likely to draw fields"), target = below(w1, N_B | N_T), position = below(w2, len+1), len = length of the
// target list after the removal.  raw (optional) receives {kind, vertex, source list, source position, target, position}.
__device__ __forceinline__ Move mv_derive(const MvParams &P, const uint8_t *sm, uint32_t w0, uint32_t w1, uint32_t w2, uint32_t *raw)
{
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  const uint32_t n_f = H.n_f, n_b = H.n_b, n_t = H.n_t;
  const uint2 *bp = MV_TAB(const uint2, M.off_bp);
  const uint32_t v = __umulhi(w0, n_f + n_b);
  Move m;
  if (v < n_f) {
    const uint32_t a = MV_TAB(const uint16_t, M.off_posf)[v];
    const uint32_t A = MV_TAB(const uint32_t, M.off_pfb)[a] >> 16;
    // §2.6 (L249): with the field->BP assignment fixed (flag bit 3) the field is reinserted into its own BP
    const uint32_t t = (H.flags & 8u) ? A : __umulhi(w1, n_b);
    const uint2 bt = bp[t], bA = bp[A];
    const uint32_t len_t = bt.x >> 16, start_t = bt.x & 0xFFFFu;
    const uint32_t q = __umulhi(w2, len_t - (A == t ? 1u : 0u) + 1u);
    m.a = a; m.len = 1u; m.c = start_t - (a < start_t ? 1u : 0u) + q;
    m.fld_b = t; m.g1 = (bA.y >> 8) & 0xFFu; m.g2 = (bt.y >> 8) & 0xFFu;
    m.src = A; m.jo = 0u; m.jq = 0u;
    if (raw) { raw[0] = 0u; raw[1] = v; raw[2] = A; raw[3] = a - (bA.x & 0xFFFFu); raw[4] = t; raw[5] = q; }
  } else {
    const uint32_t b = v - n_f;
    const uint2 bb = bp[b];
    const uint32_t j = bb.y & 0xFFu, g = (bb.y >> 8) & 0xFFu, len = bb.x >> 16;
    const uint32_t t = __umulhi(w1, n_t);
    const uint32_t tp = MV_TAB(const uint32_t, M.off_tpl)[t];
    const uint32_t t_start = tp & 0xFFu, t_len = tp >> 8;
    const uint32_t q = __umulhi(w2, t_len - (g == t ? 1u : 0u) + 1u);
    const uint32_t jq = t_start - (j < t_start ? 1u : 0u) + q;       // plan index of b after the move
    const uint16_t *pre = MV_TAB(const uint16_t, M.off_pre);
    m.a = bb.x & 0xFFFFu; m.len = len;
    m.c = (jq <= j) ? (uint32_t)pre[jq] : (uint32_t)pre[jq + 1u] - len;
    m.fld_b = kNone; m.g1 = g; m.g2 = t;
    m.src = b; m.jo = j; m.jq = jq;
    if (raw) { raw[0] = 1u; raw[1] = b; raw[2] = g; raw[3] = (bb.y >> 16) & 0xFFu; raw[4] = t; raw[5] = q; }
  }
  return m;
}

__device__ __forceinline__ Move mv_identity()
{
  Move m; m.a = m.len = m.c = 0u; m.fld_b = m.g1 = m.g2 = kNone; m.src = 0u; m.jo = m.jq = 0u;
  return m;
}

// ------------------------------------------------------------------ cost of move(x) (S4-S7)

struct EvalOut { bool feasible; double cost, path, makespan; };

// Incremental evaluation, exact.  Everything a move leaves alone keeps the incumbent's value — same operands in the
// same order, hence the same bits: integer sums (supplies, areas: eq. (2) is decided in O(1)), the mean leg of every
// BP whose field list is unchanged, L_tour / E / T / T_wait / shuttle sum of the tours the move does not touch.  In a
// touched tour the FP64 running sums restart from the incumbent's prefix value at the first position the move
// changes (prex, prey) and only the rest of the tour is re-added in order; the mean legs of the two BPs a field move
// changes are re-summed over those BPs alone; E(g) re-sums the tour's per-BP means.
template <int MASKW, bool HB>
__device__ __forceinline__ EvalOut mv_eval(const MvParams &P, const uint8_t *sm, const St &s, const Move &mv)
{
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  const uint32_t n_b = H.n_b, n_t = H.n_t, n_su = H.n_su;
  const uint32_t *pfb  = MV_TAB(const uint32_t, M.off_pfb);
  const uint32_t *psq  = MV_TAB(const uint32_t, M.off_psq);
  const double   *term = MV_TAB(const double, M.off_term);
  const double   *legx = MV_TAB(const double, M.off_legx);
  const double   *legy = MV_TAB(const double, M.off_legy);
  const double   *prex = MV_TAB(const double, M.off_prex);
  const double   *prey = MV_TAB(const double, M.off_prey);
  const uint2    *bp   = MV_TAB(const uint2, M.off_bp);
  const uint2    *bsh  = MV_TAB(const uint2, M.off_bsh);
  const double   *bpq  = MV_TAB(const double, M.off_bpq);
  const uint8_t  *bpat = MV_TAB(const uint8_t, M.off_bpat);
  const uint32_t *tpl  = MV_TAB(const uint32_t, M.off_tpl);
  const uint2    *thu  = MV_TAB(const uint2, M.off_thu);
  const uint2    *tsn  = MV_TAB(const uint2, M.off_tsn);
  const uint2    *trng = MV_TAB(const uint2, M.off_trng);
  const double   *tst  = MV_TAB(const double, M.off_tst);
  const uint32_t *thq  = MV_TAB(const uint32_t, M.off_thq);
  const uint64_t *tmask = MV_TAB(const uint64_t, M.off_tmask);
  const uint32_t *dq   = MV_TAB(const uint32_t, M.off_dq);
  const double2  *xy   = MV_TAB(const double2, M.off_xy);
  const uint32_t *cs   = MV_CTAB(uint32_t, H.offc_cs);
  const double   *rcp  = MV_CTAB(double, H.offc_rcp);
  const double inf = __longlong_as_double(0x7FF0000000000000ll);
  EvalOut out; out.feasible = false; out.cost = out.path = out.makespan = inf;

  const uint32_t L = mv.len;
  const uint32_t ga = min(mv.g1, mv.g2), gb = max(mv.g1, mv.g2);
  const uint32_t nr = (mv.g1 == kNone) ? 0u : (ga == gb ? 1u : 2u);
  const bool fld = (mv.fld_b != kNone);
  const uint32_t A = mv.src, t = mv.fld_b;

  // ---- S5: eq. (2) (L79) — only the two BPs of a field move change their supply
  uint32_t h_blk = 0;                                                         // area quanta that change tours
  {
    uint32_t bad = MV_TAB(const uint32_t, M.off_misc)[0];
    if (fld) {
      const uint32_t sq_f = psq[mv.a];
      h_blk = MV_TAB(const uint32_t, M.off_phq)[mv.a];
      if (A != t) {
        const uint32_t SA = bsh[A].x, ST = bsh[t].x, dA = dq[A], dT = dq[t];
        bad = bad - (SA < dA ? 1u : 0u) - (ST < dT ? 1u : 0u) + (SA - sq_f < dA ? 1u : 0u) + (ST + sq_f < dT ? 1u : 0u);
      }
    } else if (nr > 0u) h_blk = bsh[A].y;
    if (bad != 0u) return out;                                                 // discarded (L186; R19)
  }

  // worker position -> incumbent index: p -> p outside [lo, lo+span); three breakpoints (Q, K) inside, ascending
  const uint32_t lo = min(mv.a, mv.c), span = max(mv.a, mv.c) + L - lo;
  const uint32_t shift = (mv.c <= mv.a) ? (0u - L) : L;
  uint32_t Q1, K1, Q2, K2, Q3, K3;
  if (mv.c <= mv.a) { Q1 = mv.c; K1 = mv.a; Q2 = mv.c + L; K2 = mv.c; Q3 = mv.a + L; K3 = mv.a + L; }
  else              { Q1 = mv.a; K1 = mv.a + L; Q2 = mv.c; K2 = mv.a; Q3 = mv.c + L; K3 = mv.c + L; }
  auto map_idx = [&](uint32_t p) -> uint32_t {
    if (p - lo < span) { const uint32_t o = p - mv.c; return (o < L) ? mv.a + o : p + shift; }
    return p;
  };
  // the worker's positions [wb, we) of tour g
  auto wrange = [&](uint32_t g, uint32_t &wb, uint32_t &we) {
    const uint2 r = trng[g];
    wb = r.x - ((mv.g1 < g) ? L : 0u) + ((mv.g2 < g) ? L : 0u);
    we = wb + (r.y - r.x) - ((g == mv.g1) ? L : 0u) + ((g == mv.g2) ? L : 0u);
  };
  // first position of [wb, we) the move changes (a breakpoint), else we
  auto first_change = [&](uint32_t wb, uint32_t we) -> uint32_t {
    const uint32_t q = (Q1 >= wb) ? Q1 : ((Q2 >= wb) ? Q2 : ((Q3 >= wb) ? Q3 : we));
    return min(q, we);
  };

  // The legs a worker cannot read from the tables — into each breakpoint from the worker's own predecessor, and
  // the moved field's leg to its new BP — are computed here, by all lanes together, not inside the divergent walks.
  uint32_t wb_a = 0, we_a = 0, wb_b = 0, we_b = 0;
  if (nr > 0u) wrange(ga, wb_a, we_a);
  if (nr > 1u) wrange(gb, wb_b, we_b);
  double X1 = 0.0, X2 = 0.0, X3 = 0.0, xlb = 0.0;
  if (nr > 0u) {
    auto into = [&](uint32_t q) -> double {
      if (q >= (uint32_t)H.n_f) return 0.0;                                    // past the last position: never reached
      const uint32_t vf = 1u + n_b + (pfb[map_idx(q)] & 0xFFFFu);
      const bool first = (q == wb_a) || (nr > 1u && q == wb_b);                // first field of its tour: from HQ (L21)
      const uint32_t vp = first ? 0u : 1u + n_b + (pfb[map_idx(q - 1u)] & 0xFFFFu);
      return edge_from_xy(xy, vp, vf);
    };
    X1 = into(Q1); X2 = into(Q2); X3 = into(Q3);
    if (fld) xlb = edge_from_xy(xy, 1u + n_b + (pfb[mv.a] & 0xFFFFu), 1u + t);
  }

  // ---- untouched tours: the incumbent's values
  double makespan = 0.0;                                                       // every T(g) >= 0
  for (uint32_t g = 0; g < n_t; ++g) {
    s.d(M.m64_w + g) = tst[3u * n_t + g];
    s.w(M.m32_s + g) = tsn[g].x;
#pragma unroll
    for (int i = 0; i < MASKW; ++i) s.q(M.m64_mask + MASKW * g + i) = tmask[g * MASKW + i];
    if (g != ga && g != gb) { const double t_g = tst[2u * n_t + g]; if (t_g > makespan) makespan = t_g; }
    if (HB) { s.d(M.m64_t + g) = tst[2u * n_t + g]; s.q(M.m64_hmask + g) = MV_TAB(const uint64_t, M.off_thm)[g]; s.w(M.m32_r + g) = thu[g].y; }
  }

  // ---- the two BPs of a field move: their mean field->BP leg, re-summed in the worker's order (L213)
  double qA = 0.0, qT = 0.0;
  uint32_t kA = 0, kT = 0;
  if (fld) {
    const uint2 bA = bp[A], bT = bp[t];
    const uint32_t jA = bA.y & 0xFFu, jT = bT.y & 0xFFu;
    // the BP's k fields in the worker's order, straight from the incumbent's segment [start, ...): element `ra` of it is
    // skipped when the moved field left this BP, and the moved field sits at offset q when it joined it
    auto mean_leg = [&](uint32_t start, uint32_t k, bool has_rem, uint32_t ra, bool has_ins, uint32_t q) -> double {
      // Offset i of the worker's list reads incumbent offset i - (i > q, once the field is in) + (>= ra, once it is out).
      // ONE loop for the whole list (the lanes of a warp stay together): four table legs at a time where neither the
      // inserted field nor the removal's shift falls among them, else one.
      const uint32_t bq = has_ins ? q : kNone;
      const uint32_t br = has_rem ? ra + ((has_ins && ra >= q) ? 1u : 0u) : kNone;   // first offset shifted by the removal
      const double *lg = legy + start;
      double sd = 0.0;
      uint32_t i = 0;
      while (i < k) {
        const uint32_t off = (i >= br ? 1u : 0u) - ((has_ins && i > q) ? 1u : 0u);    // (mod 2^32)
        if (i + 4u <= k && (bq - i) >= 4u && (br - i - 1u) >= 3u) {             // bq not in [i, i+4), br not in (i, i+4)
          const double *lp = lg + (i + off);
          const double a0 = lp[0], a1 = lp[1], a2 = lp[2], a3 = lp[3];
          sd = __dadd_rn(sd, a0); sd = __dadd_rn(sd, a1); sd = __dadd_rn(sd, a2); sd = __dadd_rn(sd, a3);
          i += 4u;
        } else {
          sd = __dadd_rn(sd, (i == bq) ? xlb : lg[i + off]);
          ++i;
        }
      }
      return div_small(sd, k, rcp);
    };
    const uint32_t sA = bA.x & 0xFFFFu, sT = bT.x & 0xFFFFu;
    if (A == t) { kA = bA.x >> 16; qA = mean_leg(sA, kA, true, mv.a - sA, true, mv.c - sA); }
    else {
      kA = (bA.x >> 16) - 1u; kT = (bT.x >> 16) + 1u;
      if (kA > 0u) qA = mean_leg(sA, kA, true, mv.a - sA, false, 0u);
      qT = mean_leg(sT, kT, false, 0u, true, mv.c - (sT - (jA < jT ? 1u : 0u)));
    }
  }
  // worker plan index -> incumbent plan index (a BP move relocates one BP in the plan order)
  auto jmap = [&](uint32_t jj) -> uint32_t {
    if (fld) return jj;
    if (jj == mv.jq) return mv.jo;
    if (mv.jq <= mv.jo) return (jj > mv.jq && jj <= mv.jo) ? jj - 1u : jj;
    return (jj >= mv.jo && jj < mv.jq) ? jj + 1u : jj;
  };

  // ---- S4 for the touched tours (L69, L106, L213)
  double lt_a = 0.0, lt_b = 0.0, E_a = 0.0, E_b = 0.0, road_a = 0.0, road_b = 0.0;
  uint32_t hq_a = 0, hq_b = 0;
  double sh_a = 0.0, sh_b = 0.0;          // the touched tours' shuttle sums IF Algorithm 2 leaves their SU sets alone
  for (uint32_t r = 0; r < nr; ++r) {
    const uint32_t g = r ? gb : ga;
    const uint32_t wb = r ? wb_b : wb_a, we = r ? we_b : we_a;
    // E(g): the tour's BPs in the worker's plan order, each with its mean leg (R10: only BPs with fields)
    double E = 0.0;
    {
      const uint32_t tp = tpl[g];
      uint32_t js = tp & 0xFFu, jl = tp >> 8;
      if (!fld) { js = js - ((mv.g1 < g) ? 1u : 0u) + ((mv.g2 < g) ? 1u : 0u); jl = jl - ((g == mv.g1) ? 1u : 0u) + ((g == mv.g2) ? 1u : 0u); }
      double sumE = 0.0; uint32_t m = 0;
      for (uint32_t jj = js; jj < js + jl; ++jj) {
        const uint32_t b = bpat[jmap(jj)];
        uint32_t k = bp[b].x >> 16; double q = bpq[b];
        if (fld) { if (b == A) { k = kA; q = qA; } else if (b == t) { k = kT; q = qT; } }
        if (k > 0u) { sumE = __dadd_rn(sumE, q); ++m; }
      }
      if (m > 0u) E = __ddiv_rn(__dmul_rn(2.0, div_small(sumE, m, rcp)), H.v_su);    // L199, L213; R9
    }
    // L_tour(g): the incumbent's running sum before the first changed position, the rest re-added in order
    const uint2 rg = trng[g];
    const uint32_t p0 = first_change(wb, we);
    const bool at_end = (p0 - wb == rg.y - rg.x);
    double Lt = at_end ? tst[5u * n_t + g] : prex[rg.x + (p0 - wb)];
    // ... and, in the same walk, the tour's shuttle sum under the incumbent's SU set (a second, independent chain of
    // additions): table terms N * D(f,b); inside the moved block — tabulated under another tour's SU set, and a moved
    // field has a new BP — the count is re-derived.  Pass 2 below takes it if Algorithm 2 left this tour's set alone.
    double sh = at_end ? tst[4u * n_t + g] : prey[rg.x + (p0 - wb)];
    {
      const uint2 sn_g = tsn[g];
      const uint32_t magic_g = 0xFFFFFFFFu / sn_g.x;
      uint32_t P1 = Q1, J1 = K1, P2 = Q2, J2 = K2, P3 = Q3, J3 = K3;
      double Y1 = X1, Y2 = X2, Y3 = X3;
      while (P1 < p0) { P1 = P2; J1 = J2; Y1 = Y2; P2 = P3; J2 = J3; Y2 = Y3; P3 = kNone; }
      // ONE loop (the lanes of a warp stay together): eight or four positions at a time while no breakpoint lies among
      // them, else one — a breakpoint's route leg was computed up front.  cur = incumbent index of position p.
      uint32_t cur = 0, p = p0;
      bool inblk = false;
      while (p < we) {
        const uint32_t room = min(we, P1) - p;                                 // positions before the next breakpoint / the end
        if (room >= 8u && !inblk) {
          const double *lp = legx + cur, *tp = term + cur;
          const double l0 = lp[0], l1 = lp[1], l2 = lp[2], l3 = lp[3], l4 = lp[4], l5 = lp[5], l6 = lp[6], l7 = lp[7];
          const double t0 = tp[0], t1 = tp[1], t2 = tp[2], t3 = tp[3], t4 = tp[4], t5 = tp[5], t6 = tp[6], t7 = tp[7];
          Lt = __dadd_rn(Lt, l0); sh = __dadd_rn(sh, t0); Lt = __dadd_rn(Lt, l1); sh = __dadd_rn(sh, t1);
          Lt = __dadd_rn(Lt, l2); sh = __dadd_rn(sh, t2); Lt = __dadd_rn(Lt, l3); sh = __dadd_rn(sh, t3);
          Lt = __dadd_rn(Lt, l4); sh = __dadd_rn(sh, t4); Lt = __dadd_rn(Lt, l5); sh = __dadd_rn(sh, t5);
          Lt = __dadd_rn(Lt, l6); sh = __dadd_rn(sh, t6); Lt = __dadd_rn(Lt, l7); sh = __dadd_rn(sh, t7);
          cur += 8u; p += 8u;
        } else if (room >= 4u && !(inblk && fld)) {
          const double *lp = legx + cur;
          const double l0 = lp[0], l1 = lp[1], l2 = lp[2], l3 = lp[3];
          double t0, t1, t2, t3;
          if (inblk) {
            const uint32_t *sp = psq + cur; const double *yp = legy + cur;
            t0 = __dmul_rn((double)shuttle_count(sp[0], sn_g.y, sn_g.x, magic_g), yp[0]); t1 = __dmul_rn((double)shuttle_count(sp[1], sn_g.y, sn_g.x, magic_g), yp[1]);
            t2 = __dmul_rn((double)shuttle_count(sp[2], sn_g.y, sn_g.x, magic_g), yp[2]); t3 = __dmul_rn((double)shuttle_count(sp[3], sn_g.y, sn_g.x, magic_g), yp[3]);
          } else { const double *tp = term + cur; t0 = tp[0]; t1 = tp[1]; t2 = tp[2]; t3 = tp[3]; }
          Lt = __dadd_rn(Lt, l0); sh = __dadd_rn(sh, t0); Lt = __dadd_rn(Lt, l1); sh = __dadd_rn(sh, t1);
          Lt = __dadd_rn(Lt, l2); sh = __dadd_rn(sh, t2); Lt = __dadd_rn(Lt, l3); sh = __dadd_rn(sh, t3);
          cur += 4u; p += 4u;
        } else {
          double lh;
          if (room == 0u) {
            do { cur = J1; lh = Y1; P1 = P2; J1 = J2; Y1 = Y2; P2 = P3; J2 = J3; Y2 = Y3; P3 = kNone; } while (p == P1);
            inblk = (p - mv.c) < L;
          } else lh = legx[cur];                                               // field to field (L69)
          double tm = term[cur];
          if (inblk) tm = __dmul_rn((double)shuttle_count(psq[cur], sn_g.y, sn_g.x, magic_g), fld ? xlb : legy[cur]);
          Lt = __dadd_rn(Lt, lh); sh = __dadd_rn(sh, tm);
          ++cur; ++p;
        }
      }
    }
    if (we > wb) Lt = __dadd_rn(Lt, edge_from_xy(xy, 1u + n_b + (pfb[map_idx(we - 1u)] & 0xFFFFu), 0u));   // back to HQ (L21; R2)
    const uint32_t Hq = thq[g] - ((g == mv.g1) ? h_blk : 0u) + ((g == mv.g2) ? h_blk : 0u);
    const uint2 hu = thu[g];
    const double road = __ddiv_rn(Lt, H.v_hu);
    const double t_g = __dadd_rn(road, __ddiv_rn((double)Hq, (double)hu.y));   // L190; R6
    if (t_g > makespan) makespan = t_g;
    if (HB) s.d(M.m64_t + g) = t_g;
    const Mask<MASKW> mk = mask_load<MASKW>(s, M.m64_mask + MASKW * g);
    s.d(M.m64_w + g) = wait_time(E, tsn[g].x, cs[mask_top(mk)], hu.x, H.kappa, rcp);
    if (r == 0u) { lt_a = Lt; E_a = E; sh_a = sh; road_a = road; hq_a = Hq; } else { lt_b = Lt; E_b = E; sh_b = sh; road_b = road; hq_b = Hq; }
  }
  auto E_of  = [&](uint32_t g) -> double { return g == ga ? E_a : (g == gb ? E_b : tst[n_t + g]); };
  auto lt_of = [&](uint32_t g) -> double { return g == ga ? lt_a : (g == gb ? lt_b : tst[g]); };
  auto nhu_of = [&](uint32_t g) -> uint32_t { return HB ? (uint32_t)__popcll(s.q(M.m64_hmask + g)) : thu[g].x; };

  // ---- the embedded HU assignment (N2; L190, L203; R39): Algorithm 2's procedure on T(g) = L_tour/v_HU + H_q/R_g,
  // the donor's units tried by rising rate; before the SUs, as the paper lists them
  if (HB) {
    if (n_t >= 2u) {
      const uint32_t *hrs = MV_CTAB(uint32_t, H.offc_hrs);
      auto road_of = [&](uint32_t g) -> double { return g == ga ? road_a : (g == gb ? road_b : tst[6u * n_t + g]); };
      auto hq_of   = [&](uint32_t g) -> double { return (double)(g == ga ? hq_a : (g == gb ? hq_b : thq[g])); };
      bool changed = false;
      for (uint32_t iter = 0; iter < (uint32_t)H.n_hu; ++iter) {
        uint32_t g_max = 0, g_2nd = kNone; double t_max = s.d(M.m64_t), t_2nd = 0.0;
        for (uint32_t g = 1; g < n_t; ++g) {
          const double w = s.d(M.m64_t + g);
          if (w > t_max) { t_2nd = t_max; g_2nd = g_max; t_max = w; g_max = g; }
          else if (g_2nd == kNone || w > t_2nd) { t_2nd = w; g_2nd = g; }
        }
        uint32_t g_min = kNone; double t_min = 0.0;
        for (uint32_t g = 0; g < n_t; ++g) {
          const double w = s.d(M.m64_t + g);
          if (g != g_max && g != g_2nd && (g_min == kNone || w < t_min)) { t_min = w; g_min = g; }
        }
        const bool two = (g_min == kNone);
        if (two) g_min = g_2nd;
        const uint64_t hm_min = s.q(M.m64_hmask + g_min);
        if (__popcll(hm_min) <= 1) break;
        const uint32_t R_max = s.w(M.m32_r + g_max);
        const double road_max = road_of(g_max), hq_max = hq_of(g_max);
        uint64_t rest = hm_min; int r; uint32_t rr; double t_new;
        for (;;) {
          r = __ffsll((long long)rest) - 1; rest &= rest - 1ull; rr = hrs[r];
          t_new = __dadd_rn(road_max, __ddiv_rn(hq_max, (double)(R_max + rr)));
          if (t_new < t_2nd || rest == 0ull) break;
        }
        const uint32_t R_min = s.w(M.m32_r + g_min) - rr;
        const double t_don = __dadd_rn(road_of(g_min), __ddiv_rn(hq_of(g_min), (double)R_min));
        double new_max = t_new > t_don ? t_new : t_don;
        if (!two && t_2nd > new_max) new_max = t_2nd;
        if (!(new_max < t_max)) break;
        s.q(M.m64_hmask + g_min) = hm_min ^ (1ull << r); s.w(M.m32_r + g_min) = R_min; s.d(M.m64_t + g_min) = t_don;
        s.q(M.m64_hmask + g_max) ^= (1ull << r);         s.w(M.m32_r + g_max) = R_max + rr; s.d(M.m64_t + g_max) = t_new;
        changed = true;
      }
      if (changed)                                       // eq. (6) divides by the HU count (R7)
        for (uint32_t g = 0; g < n_t; ++g) {
          const Mask<MASKW> mk = mask_load<MASKW>(s, M.m64_mask + MASKW * g);
          s.d(M.m64_w + g) = wait_time(E_of(g), tsn[g].x, cs[mask_top(mk)], nhu_of(g), H.kappa, rcp);
        }
    }
    makespan = 0.0;
    for (uint32_t g = 0; g < n_t; ++g) { const double t_g = s.d(M.m64_t + g); if (t_g > makespan) makespan = t_g; }
  }

  // ---- S6: Algorithm 2 (L209-227), readings R11-R16 (same procedure as in lgx_walk_finish)
  if (n_t >= 2u) {
    for (uint32_t iter = 0; iter < n_su; ++iter) {
      uint32_t g_max = 0, g_2nd = kNone; double w_max = s.d(M.m64_w), w_2nd = 0.0;
      for (uint32_t g = 1; g < n_t; ++g) {
        const double w = s.d(M.m64_w + g);
        if (w > w_max) { w_2nd = w_max; g_2nd = g_max; w_max = w; g_max = g; }
        else if (g_2nd == kNone || w > w_2nd) { w_2nd = w; g_2nd = g; }
      }
      uint32_t g_min = kNone; double w_min = 0.0;
      for (uint32_t g = 0; g < n_t; ++g) {
        const double w = s.d(M.m64_w + g);
        if (g != g_max && g != g_2nd && (g_min == kNone || w < w_min)) { w_min = w; g_min = g; }
      }
      const bool two = (g_min == kNone);
      if (two) g_min = g_2nd;                                                // R12
      Mask<MASKW> mk_min = mask_load<MASKW>(s, M.m64_mask + MASKW * g_min);
      if (mask_count(mk_min) <= 1) break;                                    // R15
      Mask<MASKW> mk_max = mask_load<MASKW>(s, M.m64_mask + MASKW * g_max);
      const uint32_t S_max = s.w(M.m32_s + g_max), M_max = cs[mask_top(mk_max)];
      const uint32_t hu_max = nhu_of(g_max);
      const double   E_max = E_of(g_max);
      // donor's units by rising fill time (L221): the first that brings T_wait(g_max) below T_wait(g_2nd),
      // else the largest (L225; R13).  The test is monotone in the capacity: bisect over the ranks.
      int r = mask_top(mk_min);
      uint32_t cr = cs[r];
      double w_new = wait_time(E_max, S_max + cr, max(M_max, cr), hu_max, H.kappa, rcp);
      if (w_new < w_2nd) {
        uint32_t lo2 = 0, hi2 = (uint32_t)r;
        while (lo2 < hi2) {
          const uint32_t mid = (lo2 + hi2) >> 1;
          const uint32_t cm = cs[mid];
          const double wm = wait_time(E_max, S_max + cm, max(M_max, cm), hu_max, H.kappa, rcp);
          if (wm < w_2nd) hi2 = mid; else lo2 = mid + 1u;
        }
        Mask<MASKW> ge = mk_min;
#pragma unroll
        for (int i = 0; i < MASKW; ++i) {
          const int sft = (int)lo2 - 64 * i;
          if (sft >= 64) ge.w[i] = 0ull; else if (sft > 0) ge.w[i] &= ~0ull << sft;
        }
        r = mask_pop_lowest(ge);
        cr = cs[r];
        w_new = wait_time(E_max, S_max + cr, max(M_max, cr), hu_max, H.kappa, rcp);
      }
      mask_flip(mk_min, r);
      const uint32_t S_min = s.w(M.m32_s + g_min) - cr;
      const double w_don = wait_time(E_of(g_min), S_min, cs[mask_top(mk_min)], nhu_of(g_min), H.kappa, rcp);
      double new_max = w_new > w_don ? w_new : w_don;                        // step 11 (L227; R14)
      if (!two && w_2nd > new_max) new_max = w_2nd;
      if (!(new_max < w_max)) break;
      mask_flip(mk_max, r);
      mask_store<MASKW>(s, M.m64_mask + MASKW * g_min, mk_min); s.w(M.m32_s + g_min) = S_min; s.d(M.m64_w + g_min) = w_don;
      mask_store<MASKW>(s, M.m64_mask + MASKW * g_max, mk_max); s.w(M.m32_s + g_max) = S_max + cr; s.d(M.m64_w + g_max) = w_new;
    }
  }

  // ---- S7 pass 2: shuttles (eq. (4); R4).  T_wait is dead: its row now holds the tour's shuttle sum.
  uint64_t need = 0ull;
  for (uint32_t g = 0; g < n_t; ++g) {
    const uint2 sn = tsn[g];
    const bool same = (s.w(M.m32_s + g) == sn.x) && ((uint32_t)mask_count(mask_load<MASKW>(s, M.m64_mask + MASKW * g)) == sn.y);
    if (g == ga || g == gb) {                  // a touched tour: its sum under the old SU set came with the route walk
      if (same) s.d(M.m64_w + g) = (g == ga) ? sh_a : sh_b; else need |= 1ull << g;
      continue;
    }
    if (same) { s.d(M.m64_w + g) = tst[4u * n_t + g]; continue; }
    // an untouched tour one SU away from the incumbent's set: tabulated (mv_encode)
    const uint32_t C2 = s.w(M.m32_s + g), n2 = (uint32_t)mask_count(mask_load<MASKW>(s, M.m64_mask + MASKW * g));
    uint32_t dir = 2u, delta = 0u;
    if (n2 == sn.y + 1u && C2 > sn.x) { dir = 1u; delta = C2 - sn.x; }
    else if (n2 + 1u == sn.y && C2 < sn.x) { dir = 0u; delta = sn.x - C2; }
    if (dir < 2u) {
      uint32_t lo2 = 0, hi2 = n_su;                                            // first rank with capacity >= delta
      while (lo2 < hi2) { const uint32_t mid = (lo2 + hi2) >> 1; if (cs[mid] < delta) lo2 = mid + 1u; else hi2 = mid; }
      if (lo2 < n_su && cs[lo2] == delta) { s.d(M.m64_w + g) = MV_TAB(const double, M.off_sv)[(g * 2u + dir) * n_su + lo2]; continue; }
    }
    need |= 1ull << g;
  }
  while (need) {
    const uint32_t g = (uint32_t)__ffsll((long long)need) - 1u;
    need &= need - 1ull;
    const uint32_t C_g = s.w(M.m32_s + g), n_g = (uint32_t)mask_count(mask_load<MASKW>(s, M.m64_mask + MASKW * g));
    const uint32_t magic = 0xFFFFFFFFu / C_g;
    // every tour that gets here has a changed SU set: all its counts are re-derived, from the tour's first position
    uint32_t p, pe;
    wrange(g, p, pe);
    double shut = 0.0;
    uint32_t P0 = p, J0 = map_idx(p), P1 = Q1, J1 = K1, P2 = Q2, J2 = K2, P3 = Q3, J3 = K3;
    while (P1 < p) { P1 = P2; J1 = J2; P2 = P3; J2 = J3; P3 = kNone; }
    // ONE loop (the lanes of a warp stay together), four positions at a time while no breakpoint lies among them
    uint32_t idx = 0;
    bool inblk = false;
    while (p < pe) {
      const uint32_t room = min(pe, P0) - p;
      if (room == 0u) {                          // a breakpoint: position p reads incumbent index J0
        do { idx = J0; P0 = P1; J0 = J1; P1 = P2; J1 = J2; P2 = P3; J2 = J3; P3 = kNone; } while (p == P0);
        inblk = (p - mv.c) < L;
        continue;
      }
      if (room >= 4u && !(inblk && fld)) {
        const uint32_t *sp = psq + idx; const double *lp = legy + idx;
        const double t0 = __dmul_rn((double)shuttle_count(sp[0], n_g, C_g, magic), lp[0]), t1 = __dmul_rn((double)shuttle_count(sp[1], n_g, C_g, magic), lp[1]);
        const double t2 = __dmul_rn((double)shuttle_count(sp[2], n_g, C_g, magic), lp[2]), t3 = __dmul_rn((double)shuttle_count(sp[3], n_g, C_g, magic), lp[3]);
        shut = __dadd_rn(shut, t0); shut = __dadd_rn(shut, t1); shut = __dadd_rn(shut, t2); shut = __dadd_rn(shut, t3);
        idx += 4u; p += 4u;
      } else {
        shut = __dadd_rn(shut, __dmul_rn((double)shuttle_count(psq[idx], n_g, C_g, magic), (inblk && fld) ? xlb : legy[idx]));
        ++idx; ++p;
      }
    }
    s.d(M.m64_w + g) = shut;
  }
  // ---- lengths (L106): N_HU(g), N_SU(g) multiply the tour distance, shuttles x2; cost (R1)
  double path = 0.0;
  for (uint32_t g = 0; g < n_t; ++g) {
    const double lt = lt_of(g), shut = s.d(M.m64_w + g);
    const uint32_t n_g = (uint32_t)mask_count(mask_load<MASKW>(s, M.m64_mask + MASKW * g));
    const double l_hu  = __dmul_rn((double)nhu_of(g), lt);
    const double l_esu = __dadd_rn(__dmul_rn((double)n_g, lt), shut);
    path = __dadd_rn(path, __dadd_rn(__dadd_rn(l_hu, l_esu), shut));
  }
  out.feasible = true; out.path = path; out.makespan = makespan;
  out.cost = __dadd_rn(__dmul_rn(H.w_path, path), __dmul_rn(H.w_time, makespan));
  return out;
}

// ------------------------------------------------------------------ common prologue

template <int MASKW>
__device__ __forceinline__ void mv_prologue(const MvParams &P, uint8_t *sm, St &s, uint32_t tid, uint32_t T)
{
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  {
    const uint4 *src = reinterpret_cast<const uint4 *>(P.xy);
    uint4 *dst = reinterpret_cast<uint4 *>(sm + M.off_xy);
    for (uint32_t i = tid; i < 1u + (uint32_t)H.n_b + (uint32_t)H.n_f; i += T) dst[i] = src[i];
    const uint32_t *dqg = reinterpret_cast<const uint32_t *>(P.image + H.off_dq);
    uint32_t *dqs = reinterpret_cast<uint32_t *>(sm + M.off_dq);
    for (uint32_t i = tid; i < (uint32_t)H.n_b; i += T) dqs[i] = dqg[i];
    src = reinterpret_cast<const uint4 *>(P.image_c + H.offc_cs);
    dst = reinterpret_cast<uint4 *>(sm + M.off_c);
    for (uint32_t i = tid; i < (H.imagec_bytes - H.offc_cs) / 16u; i += T) dst[i] = src[i];
  }
  s.T4 = 4u * T; s.T8 = 8u * T;
  s.b64 = sm + M.off_state + 8u * tid;
  s.b32 = sm + M.off_state + M.m64_rows * s.T8 + 4u * tid;
  __syncthreads();
}

// A block's share of n_total workers = rounds of blockDim.x consecutive indices, gridDim.x * blockDim.x apart.
// Which lane scores which worker is free, so up to kSuper rounds at a time are counting-sorted by the tours their
// moves touch — the lanes of a warp then walk the same tours (equal trip counts, the same shared-memory words,
// similar Algorithm-2 paths) — and the warps DRAW chunks of 32 sorted workers from a shared counter, so a warp
// stuck with expensive workers does not hold the others at a barrier.  eval(i) scores worker index i.
constexpr uint32_t kSuper = 8;                  // rounds sorted and scheduled together (order: u16 [kSuper * 1024])

template <class F>
__device__ __forceinline__ void mv_for_workers(const MvParams &P, uint8_t *sm, uint64_t id0, uint64_t n_total,
                                               uint32_t tid, uint32_t T, F &&eval)
{
  const uint32_t n_t = P.H.n_t;
  // key = (unordered pair of touched tours, bucket of the first changed position inside the lower tour): lanes of a
  // warp then share the tours AND roughly the point from which their running sums must be re-added
  const uint32_t n_pairs = n_t * (n_t + 1u) / 2u;
  // A BP move re-derives the shuttle counts of the whole moved block (its terms were tabulated under another tour's SU
  // set): such workers get keys of their own so that they share warps — the lowest keys: the warps draw the sorted
  // chunks in order, so the longest jobs start first.
  uint32_t nbk = 1u;
  while (nbk < 16u && n_pairs * (nbk * 2u + 1u) <= kSortKeys) nbk *= 2u;
  const bool by_pair = n_pairs * 2u <= kSortKeys;
  const uint32_t nk = by_pair ? n_pairs * (nbk + 1u) : 2u * n_t;
  const uint2 *trng = MV_TAB(const uint2, P.M.off_trng);
  uint32_t *hist = MV_TAB(uint32_t, P.M.off_sort);       // [nk + 2]: offsets per key, total, the warps' draw counter
  uint16_t *order = MV_TAB(uint16_t, P.M.off_order);
  const uint64_t stride = (uint64_t)gridDim.x * T;
  const uint32_t lane = tid & 31u;
  for (uint64_t base = (uint64_t)blockIdx.x * T; base < n_total; base += (uint64_t)kSuper * stride) {
    for (uint32_t k = tid; k <= nk + 1u; k += T) hist[k] = 0u;
    __syncthreads();
    uint32_t key[kSuper], rank[kSuper];
#pragma unroll
    for (uint32_t r = 0; r < kSuper; ++r) {
      const uint64_t i = base + (uint64_t)r * stride + tid;
      key[r] = kNone; rank[r] = 0u;
      if (i < n_total) {
        const uint64_t id = id0 + i;
        uint32_t w[4];
        philox_block(P, (uint32_t)id, (uint32_t)(id >> 32), 5u, 0u, w);
        const Move mv = mv_derive(P, sm, w[0], w[1], w[2], nullptr);
        const uint32_t ga = min(mv.g1, mv.g2), gb = max(mv.g1, mv.g2);
        if (by_pair) {
          const uint2 rg = trng[ga];
          const uint32_t pos = (mv.g1 == mv.g2) ? min(mv.a, mv.c) : ((mv.g1 == ga) ? mv.a : mv.c);
          const uint32_t rel = pos > rg.x ? pos - rg.x : 0u;
          const uint32_t bk = min(nbk - 1u, rel * nbk / (rg.y - rg.x + 1u));
          const uint32_t pair = ga * (2u * n_t - ga + 1u) / 2u + (gb - ga);
          key[r] = (mv.fld_b == kNone) ? pair : n_pairs + pair * nbk + bk;
        } else key[r] = ga + ((mv.fld_b == kNone) ? 0u : n_t);
        rank[r] = atomicAdd(&hist[key[r]], 1u);
      }
    }
    __syncthreads();
    if (tid < 32u) {                                   // exclusive scan of the histogram; hist[nk] = number of workers
      const uint32_t per = (nk + 1u + 31u) / 32u, k0 = tid * per;
      uint32_t sum = 0;
      for (uint32_t k = k0; k < k0 + per && k <= nk; ++k) sum += hist[k];
      uint32_t incl = sum;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) { const uint32_t o = __shfl_up_sync(0xFFFFFFFFu, incl, off); if ((int)tid >= off) incl += o; }
      uint32_t run = incl - sum;
      for (uint32_t k = k0; k < k0 + per && k <= nk; ++k) { const uint32_t h = hist[k]; hist[k] = run; run += h; }
    }
    __syncthreads();
#pragma unroll
    for (uint32_t r = 0; r < kSuper; ++r)
      if (key[r] != kNone) order[hist[key[r]] + rank[r]] = (uint16_t)((r << 10) | tid);
    __syncthreads();
    const uint32_t n_local = hist[nk];
    for (;;) {
      uint32_t c = 0;
      if (lane == 0u) c = atomicAdd(&hist[nk + 1u], 32u);
      c = __shfl_sync(0xFFFFFFFFu, c, 0);
      if (c >= n_local) break;
      if (c + lane < n_local) {
        const uint32_t L = order[c + lane];
        eval(base + (uint64_t)(L >> 10) * stride + (L & 1023u));
      }
      __syncwarp();
    }
    __syncthreads();
  }
}

// ================================================================== batch kernel (L163-165)

template <int MASKW, bool HB>
__global__ void __launch_bounds__(kMvThreads, 1) lgx_move_eval_k(const __grid_constant__ MvParams P)
{
  LGX_DYN_SMEM(smem);
  uint8_t *sm = smem;
  const uint32_t tid = threadIdx.x, T = blockDim.x;
  St s;
  mv_prologue<MASKW>(P, sm, s, tid, T);
  uint8_t *plan = sm + P.M.off_plans;
  mv_load_plan<MASKW>(P, sm, plan, tid, T);
  mv_encode<MASKW>(P, sm, plan, tid, T);
  // the paper's selection rule (L205; R38), optional: the best-so-far maximum completion time is x's own
  __shared__ double s_tbest;
  const bool filter = (P.H.flags & 4u) != 0u;
  if (filter) {
    if (tid == 0) { const EvalOut r0 = mv_eval<MASKW, HB>(P, sm, s, mv_identity()); s_tbest = r0.makespan; }   // +inf if x is infeasible
    __syncthreads();
  }
  const double t_best = filter ? s_tbest : 0.0;
  mv_for_workers(P, sm, P.first_id, P.n, tid, T, [&](uint64_t i) {
    const uint64_t id = P.first_id + i;
    uint32_t w[4];
    philox_block(P, (uint32_t)id, (uint32_t)(id >> 32), 5u, 0u, w);
    const Move mv = mv_derive(P, sm, w[0], w[1], w[2], nullptr);
    EvalOut r = mv_eval<MASKW, HB>(P, sm, s, mv);
    if (filter && r.feasible && r.makespan > t_best) r.cost = __longlong_as_double(0x7FF0000000000000ll);
    if (P.cost)       P.cost[i] = r.cost;
    if (P.path_km)    P.path_km[i] = r.path;
    if (P.makespan_h) P.makespan_h[i] = r.makespan;
    if (P.feasible)   P.feasible[i] = r.feasible ? 1 : 0;
  });
}

// ================================================================== Algorithm 1 steps 4-16, persistent

template <int MASKW, bool HB>
__global__ void __launch_bounds__(kMvThreads, 1) lgx_local_search_k(const __grid_constant__ MvParams P)
{
  LGX_DYN_SMEM(smem);
  uint8_t *sm = smem;
  cg::grid_group grid = cg::this_grid();
  const ImgHdr &H = P.H; const MvHdr &M = P.M;
  const uint32_t tid = threadIdx.x, T = blockDim.x;
  const uint32_t n_f = H.n_f, n_b = H.n_b, n_t = H.n_t;
  __shared__ unsigned long long s_bits[kMvThreads / 32], s_id[kMvThreads / 32];
  __shared__ unsigned long long s_win[3];      // global winner of the iteration: cost bits, id, block
  __shared__ unsigned long long s_cstar;       // cost bits of x*
  __shared__ double s_tstar;                   // makespan of x*: the best-so-far maximum completion time (L205; R38)
  const bool filter = (H.flags & 4u) != 0u;
  St s;
  mv_prologue<MASKW>(P, sm, s, tid, T);
  uint8_t *x_best = sm + M.off_plans, *x_old = x_best + M.plan_bytes, *x_tmp = x_old + M.plan_bytes;
  uint32_t *misc = MV_TAB(uint32_t, M.off_misc);
  auto copy_plan = [&](uint8_t *dst, const uint8_t *src) {
    for (uint32_t i = tid; i < M.plan_bytes / 8u; i += T) reinterpret_cast<uint64_t *>(dst)[i] = reinterpret_cast<const uint64_t *>(src)[i];
  };

  // ---- step 4 (L133): x* = x_0 with its cost; x_0 takes the SU sets Algorithm 2 leaves it with (R37)
  mv_load_plan<MASKW>(P, sm, x_best, tid, T);
  mv_encode<MASKW>(P, sm, x_best, tid, T);
  if (tid == 0) {
    const EvalOut r = mv_eval<MASKW, HB>(P, sm, s, mv_identity());
    s_cstar = (unsigned long long)__double_as_longlong(r.cost);
    s_tstar = r.makespan;                                                      // +inf if x_0 is infeasible
    if (r.feasible) {
      uint64_t *mk = reinterpret_cast<uint64_t *>(x_best + M.pl_mask);
      for (uint32_t i = 0; i < n_t * MASKW; ++i) mk[i] = s.q(M.m64_mask + i);
      if (HB) { uint64_t *hm = reinterpret_cast<uint64_t *>(x_best + M.pl_hmask); for (uint32_t g = 0; g < n_t; ++g) hm[g] = s.q(M.m64_hmask + g); }
    }
  }
  __syncthreads();
  copy_plan(x_old, x_best);
  __syncthreads();

  const uint32_t SW = M.slot_words;
  for (uint32_t k = 0; k < P.n_iters; ++k) {
    // ---- step 6, eq. (5) (L177): x = x* with probability eps, else the previous iteration's winner
    uint32_t uw[4];
    philox_block(P, k, 0u, 6u, 0u, uw);
    const uint8_t *x_cur = (uw[0] < P.eps_thresh) ? x_best : x_old;
    mv_encode<MASKW>(P, sm, x_cur, tid, T);

    // ---- steps 7-12: every worker moves x once and scores it; running (cost, id) minimum per thread
    unsigned long long best_bits = ~0ull, best_id = ~0ull;
    double best_mk = 0.0;
    const double t_star = s_tstar;
    const uint64_t id0 = (uint64_t)k * P.n_workers;
    mv_for_workers(P, sm, id0, (uint64_t)P.n_workers, tid, T, [&](uint64_t i) {
      const uint64_t id = id0 + i;
      uint32_t w[4];
      philox_block(P, (uint32_t)id, (uint32_t)(id >> 32), 5u, 0u, w);
      const Move mv = mv_derive(P, sm, w[0], w[1], w[2], nullptr);
      const EvalOut r = mv_eval<MASKW, HB>(P, sm, s, mv);
      unsigned long long bits = (unsigned long long)__double_as_longlong(r.cost);
      if (filter && r.feasible && r.makespan > t_star) bits = 0x7FF0000000000000ull;   // discarded (L205; R38)
      if (bits < best_bits || (bits == best_bits && id < best_id)) {
        best_bits = bits; best_id = id; best_mk = r.makespan;
        if (r.feasible) {
          for (uint32_t q = 0; q < n_t * MASKW; ++q) s.q(M.m64_bmask + q) = s.q(M.m64_mask + q);
          if (HB) for (uint32_t g = 0; g < n_t; ++g) s.q(M.m64_bhmask + g) = s.q(M.m64_hmask + g);
        }
      }
    });
    // ---- step 13 (L167): i* = arg min C_i.  warp -> block -> one slot per block -> grid barrier -> every block folds
    unsigned long long bb = best_bits, bi = best_id;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
      const unsigned long long ob = __shfl_down_sync(0xFFFFFFFFu, bb, off), oi = __shfl_down_sync(0xFFFFFFFFu, bi, off);
      take_min(bb, bi, ob, oi);
    }
    if ((tid & 31u) == 0u) { s_bits[tid >> 5] = bb; s_id[tid >> 5] = bi; }
    __syncthreads();
    if (tid < 32u) {
      const uint32_t nw = (T + 31u) >> 5;
      bb = tid < nw ? s_bits[tid] : ~0ull; bi = tid < nw ? s_id[tid] : ~0ull;
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) {
        const unsigned long long ob = __shfl_down_sync(0xFFFFFFFFu, bb, off), oi = __shfl_down_sync(0xFFFFFFFFu, bi, off);
        take_min(bb, bi, ob, oi);
      }
      if (tid == 0u) { s_win[0] = bb; s_win[1] = bi; }
    }
    __syncthreads();
    unsigned long long *slot = P.slots + ((size_t)(k & 1u) * gridDim.x + blockIdx.x) * SW;
    if (tid == 0u) { slot[0] = s_win[0]; slot[1] = s_win[1]; }
    if (best_id == s_win[1] && best_id != ~0ull)                             // the block's winner publishes its SU sets
    {
      for (uint32_t q = 0; q < n_t * MASKW; ++q) slot[2 + q] = s.q(M.m64_bmask + q);
      if (HB) for (uint32_t g = 0; g < n_t; ++g) slot[2 + n_t * MASKW + g] = s.q(M.m64_bhmask + g);
      slot[2 + n_t * MASKW + n_t] = (unsigned long long)__double_as_longlong(best_mk);
    }
    grid.sync();
    if (tid < 32u) {
      const unsigned long long *all = P.slots + (size_t)(k & 1u) * gridDim.x * SW;
      bb = ~0ull; bi = ~0ull; unsigned long long bw = 0;
      for (uint32_t blk = tid; blk < gridDim.x; blk += 32u) {
        const unsigned long long ob = __ldcg(all + (size_t)blk * SW), oi = __ldcg(all + (size_t)blk * SW + 1);
        if (ob < bb || (ob == bb && oi < bi)) { bb = ob; bi = oi; bw = blk; }
      }
#pragma unroll
      for (int off = 16; off >= 1; off >>= 1) {
        const unsigned long long ob = __shfl_down_sync(0xFFFFFFFFu, bb, off), oi = __shfl_down_sync(0xFFFFFFFFu, bi, off);
        const unsigned long long ow = __shfl_down_sync(0xFFFFFFFFu, bw, off);
        if (ob < bb || (ob == bb && oi < bi)) { bb = ob; bi = oi; bw = ow; }
      }
      if (tid == 0u) {
        s_win[0] = bb; s_win[1] = bi; s_win[2] = bw;
        if (blockIdx.x == 0u) {
          if (P.hist_cost) P.hist_cost[k] = __longlong_as_double((long long)bb);
          if (P.hist_id)   P.hist_id[k] = bi;
        }
        // the winning move, replayed from its id (L233), for the block-wide update below
        uint32_t w[4];
        philox_block(P, (uint32_t)bi, (uint32_t)(bi >> 32), 5u, 0u, w);
        (void)mv_derive(P, sm, w[0], w[1], w[2], misc + 4);
      }
    }
    __syncthreads();
    // ---- steps 14-15 (L169): x_old <- x_{i*}; x* <- x_{i*} if it improves C*.  All workers infeasible: keep x_old (R37)
    const unsigned long long win_bits = s_win[0];
    if (win_bits < 0x7FF0000000000000ull) {
      if (x_cur != x_tmp) copy_plan(x_tmp, x_cur);
      __syncthreads();
      const uint32_t kind = misc[4], vx = misc[5], src = misc[6], sp = misc[7], dst = misc[8], dp = misc[9];
      if (kind == 0u) {
        uint16_t *fb = reinterpret_cast<uint16_t *>(x_tmp + M.pl_fbp), *fp = reinterpret_cast<uint16_t *>(x_tmp + M.pl_fpos);
        for (uint32_t f = tid; f < n_f; f += T) {
          if (f == vx) { fb[f] = (uint16_t)dst; fp[f] = (uint16_t)dp; continue; }
          const uint32_t b = fb[f]; uint32_t q = fp[f];
          if (b == src && q > sp) --q;
          if (b == dst && q >= dp) ++q;
          fp[f] = (uint16_t)q;
        }
      } else {
        uint8_t *bt = x_tmp, *bq = x_tmp + M.pl_bpos;
        for (uint32_t b = tid; b < n_b; b += T) {
          if (b == vx) { bt[b] = (uint8_t)dst; bq[b] = (uint8_t)dp; continue; }
          const uint32_t g = bt[b]; uint32_t q = bq[b];
          if (g == src && q > sp) --q;
          if (g == dst && q >= dp) ++q;
          bq[b] = (uint8_t)q;
        }
      }
      {
        const unsigned long long *wm = P.slots + ((size_t)(k & 1u) * gridDim.x + (size_t)s_win[2]) * SW + 2;
        uint64_t *mk = reinterpret_cast<uint64_t *>(x_tmp + M.pl_mask);
        for (uint32_t q = tid; q < n_t * MASKW; q += T) mk[q] = __ldcg(wm + q);
        if (HB) { uint64_t *hm = reinterpret_cast<uint64_t *>(x_tmp + M.pl_hmask); for (uint32_t g = tid; g < n_t; g += T) hm[g] = __ldcg(wm + n_t * MASKW + g); }
      }
      __syncthreads();
      const bool improves = win_bits < s_cstar;
      __syncthreads();
      if (improves) {
        copy_plan(x_best, x_tmp);
        if (tid == 0u) {
          s_cstar = win_bits;
          s_tstar = __longlong_as_double((long long)__ldcg(P.slots + ((size_t)(k & 1u) * gridDim.x + (size_t)s_win[2]) * SW + 2 + n_t * MASKW + n_t));
        }
      }
      copy_plan(x_old, x_tmp);
      __syncthreads();
    }
  }

  // ---- x* and C* back to the caller's arrays
  if (blockIdx.x == 0u) {
    for (uint32_t b = tid; b < n_b; b += T) { P.bp_tour[b] = x_best[b]; P.bp_pos[b] = x_best[M.pl_bpos + b]; }
    const uint16_t *fb = reinterpret_cast<const uint16_t *>(x_best + M.pl_fbp), *fp = reinterpret_cast<const uint16_t *>(x_best + M.pl_fpos);
    for (uint32_t f = tid; f < n_f; f += T) { P.field_bp[f] = fb[f]; P.field_pos[f] = fp[f]; }
    if (tid == 0u) {
      const uint64_t *mk = reinterpret_cast<const uint64_t *>(x_best + M.pl_mask);
      const uint8_t *unit_of = MV_CTAB(uint8_t, H.offc_unit);
      for (uint32_t g = 0; g < n_t; ++g)
        for (int i = 0; i < MASKW; ++i) {
          uint64_t w = mk[g * MASKW + i];
          while (w) { const int r = __ffsll((long long)w) - 1; w &= w - 1; P.su_tour[unit_of[64 * i + r]] = (uint8_t)g; }
        }
      const uint64_t *hm = reinterpret_cast<const uint64_t *>(x_best + M.pl_hmask);
      const uint8_t *hunit_of = MV_CTAB(uint8_t, H.offc_hunit);
      for (uint32_t g = 0; g < n_t; ++g) { uint64_t w = hm[g]; while (w) { const int r = __ffsll((long long)w) - 1; w &= w - 1; P.hu_tour[hunit_of[r]] = (uint8_t)g; } }
      *P.best_cost = __longlong_as_double((long long)s_cstar);
    }
  }
}

// ================================================================== Algorithm 1 steps 1-3

struct InitParams {
  int32_t n_f, n_b, n_t, n_hu, n_su;
  const double2  *xy;        // [1 + n_b + n_f] vertex coordinates: HQ, BPs, fields
  const uint2    *sh;        // {s_q, h_q} per field
  const uint32_t *dq;        // demand quanta
  const uint8_t  *unit_of;   // SU of capacity rank r (ascending (capacity, unit))
  uint8_t *bp_tour, *bp_pos; uint16_t *field_bp, *field_pos; uint8_t *hu_tour, *su_tour;
  uint32_t *scratch;         // [n_b] supplies | [n_b + 1] list offsets | [n_b] cursors | u16 [n_f] lists | u8 [n_b] chain, flags
};

// lexicographic (distance, index) minimum over a warp: "closest", lowest index on ties
__device__ __forceinline__ void warp_argmin(double &d, uint32_t &i)
{
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    const double od = __shfl_xor_sync(0xFFFFFFFFu, d, off);
    const uint32_t oi = __shfl_xor_sync(0xFFFFFFFFu, i, off);
    if (oi != kNone && (i == kNone || od < d || (od == d && oi < i))) { d = od; i = oi; }
  }
}

// One block.  Step 1 (L122): HUs in index order, floor(N_HU/N_T) per tour, the residual on the last tour (R25);
// SUs dealt round-robin over the capacity order (Case 1: the same number of each class per tour, L273; R31);
// nearest-neighbour chain over the BPs from HQ, cut into N_T consecutive runs (R32).  Step 2 (L124): fields in
// identification order (L173) to their closest BP not yet supplied, else to their closest BP.  Step 3 (L126,
// L171): per BP a nearest-neighbour order starting from HQ.
#ifdef LGX_INSTANTIATE_INIT_PLAN      // non-template kernel: compiled by one translation unit (lgx_inst_moves.cu)
__global__ void __launch_bounds__(256, 1) lgx_init_plan_k(const InitParams P)
{
  const uint32_t tid = threadIdx.x, T = blockDim.x, lane = tid & 31u, warp = tid >> 5, n_warps = T >> 5;
  const uint32_t n_f = P.n_f, n_b = P.n_b, n_t = P.n_t;
  uint32_t *Sq = P.scratch, *off = Sq + n_b, *cur_w = off + n_b + 1u;
  uint16_t *lst = reinterpret_cast<uint16_t *>(cur_w + n_b);
  uint8_t *chain = reinterpret_cast<uint8_t *>(lst + n_f + (n_f & 1u)), *used = chain + n_b;
  for (uint32_t b = tid; b < n_b; b += T) { Sq[b] = 0u; used[b] = 0; }
  { const uint32_t per = (uint32_t)P.n_hu / n_t;
    for (uint32_t u = tid; u < (uint32_t)P.n_hu; u += T) { const uint32_t g = u / per; P.hu_tour[u] = (uint8_t)(g < n_t ? g : n_t - 1u); } }
  for (uint32_t r = tid; r < (uint32_t)P.n_su; r += T) P.su_tour[P.unit_of[r]] = (uint8_t)(r % n_t);
  __syncthreads();
  if (warp == 0u) {
    // step 1 (ii): BP chain
    uint32_t cur = 0;
    for (uint32_t k = 0; k < n_b; ++k) {
      double bd = 0.0; uint32_t best = kNone;
      for (uint32_t b = lane; b < n_b; b += 32u) if (!used[b]) { const double d = edge_from_xy(P.xy, cur, 1u + b); if (best == kNone || d < bd) { best = b; bd = d; } }
      warp_argmin(bd, best);
      if (lane == 0u) { used[best] = 1; chain[k] = (uint8_t)best; }
      __syncwarp();
      cur = 1u + best;
    }
    for (uint32_t g = 0; g < n_t; ++g) {
      const uint32_t lo = (g * n_b) / n_t, hi = ((g + 1u) * n_b) / n_t;
      for (uint32_t k = lo + lane; k < hi; k += 32u) { P.bp_tour[chain[k]] = (uint8_t)g; P.bp_pos[chain[k]] = (uint8_t)(k - lo); }
    }
    // step 2: fields -> BPs, serial over the fields (the supplies change), the BP scan across the lanes
    for (uint32_t f = 0; f < n_f; ++f) {
      double bd = 0.0, ad = 0.0; uint32_t best = kNone, any = kNone;
      for (uint32_t b = lane; b < n_b; b += 32u) {
        const double d = edge_from_xy(P.xy, 1u + n_b + f, 1u + b);
        if (any == kNone || d < ad) { any = b; ad = d; }
        if (Sq[b] < P.dq[b] && (best == kNone || d < bd)) { best = b; bd = d; }
      }
      warp_argmin(bd, best);
      if (best == kNone) { warp_argmin(ad, any); best = any; }
      if (lane == 0u) { P.field_bp[f] = (uint16_t)best; Sq[best] += P.sh[f].x; }
      __syncwarp();
    }
  }
  __syncthreads();
  // per-BP field lists
  for (uint32_t b = tid; b <= n_b; b += T) off[b] = 0u;
  __syncthreads();
  for (uint32_t f = tid; f < n_f; f += T) atomicAdd(&off[P.field_bp[f] + 1u], 1u);
  __syncthreads();
  if (tid == 0u) for (uint32_t b = 0; b < n_b; ++b) { off[b + 1u] += off[b]; cur_w[b] = off[b]; }
  __syncthreads();
  for (uint32_t f = tid; f < n_f; f += T) lst[atomicAdd(&cur_w[P.field_bp[f]], 1u)] = (uint16_t)f;
  __syncthreads();
  // step 3: one warp per BP, nearest neighbour from HQ; a visited list entry becomes 0xFFFF
  for (uint32_t b = warp; b < n_b; b += n_warps) {
    uint32_t cur = 0;
    const uint32_t lo = off[b], hi = off[b + 1u];
    for (uint32_t k = 0; k < hi - lo; ++k) {
      double bd = 0.0; uint32_t best = kNone, slot = 0;
      for (uint32_t e = lo + lane; e < hi; e += 32u) {
        const uint32_t f = lst[e];
        if (f != 0xFFFFu) { const double d = edge_from_xy(P.xy, cur, 1u + n_b + f); if (best == kNone || d < bd || (d == bd && f < best)) { best = f; bd = d; slot = e; } }
      }
      // the warp minimum over (distance, field); its owner clears the entry
      double wd = bd; uint32_t wf = best;
      warp_argmin(wd, wf);
      if (best == wf && best != kNone) { lst[slot] = 0xFFFFu; P.field_pos[wf] = (uint16_t)k; }
      __syncwarp();
      cur = 1u + n_b + wf;
    }
  }
}

#undef MV_TAB
#undef MV_CTAB
#endif

}  // namespace lgx
