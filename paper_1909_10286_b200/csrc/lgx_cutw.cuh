// lgx_cutw.cuh — lgx_decode_cut_w: the decode/cut kernel with ONE CANDIDATE PER WARP, for
// instances whose Fisher-Yates array is so large that the thread-per-candidate mapping of lgx_decode_cut leaves
// only two or three warps on an SM (N_F of the order of 1000: the paper's own size).  See "Status".
// Product code (CUDA path); shares nothing with oracle/.
//
// Same definition as lgx_decode_cut (S1-S3, S5), same queue records, bit for bit; what differs is who does
// the work.  The permutation of a candidate lives ONCE in shared memory (2 N_F bytes per warp instead of per thread),
// so an SM holds up to 32 resident warps, each on its own candidate, and the 32 lanes of a warp split
//   * Philox: lane L draws block 32 K + L of stream 3, i.e. 128 draws per round;
//   * Fisher-Yates: 32 consecutive steps at once.  Step t of the block reads slot j_t and slot i_t = i_0 - t as the
//     earlier steps of the block left them.  Only a store "a[j_m] <- y_m" (m < t) can have touched them (j_t <= i_t <
//     i_m), so lane t needs the LATEST lane m < t with j_m = j_t (match.any) resp. j_m = i_t (a 32-entry scatter with
//     atomicMax), takes that lane's y (chains of such references are followed until nothing changes: y_m may itself
//     come from an earlier lane), and the stores go out in the step-by-step order: a[j] by the last lane of every
//     group of equal j, then a[i_0..i_31];
//   * the cuts: supplies are prefix-summed over the lanes; the first position whose running supply meets the demand
//     is a ballot, the "one more field" draws (stream 4, taken up front as a shift register of bits) are a count of
//     trailing ones; one warp-uniform iteration per BP that closes inside the block.
// The BP -> tour partition (N_B items) is done by lane 0 with the draws computed by all lanes.
//
// Status: an ALTERNATIVE mapping, opt-in through LGX_OPT_CUT_WARP, parity-tested like the default one (tests/
// test_gpu_parity.py), never chosen by default.  Measured on B200 (profiles/r02_alt_cut_per_warp_paper_scale.md): 32
// resident warps instead of 2 and 47 % instead of 14 % of the SM's issue slots busy, but 8.5 k instead of 2.3 k
// warp-instructions per candidate (the conflict resolution, the scans and the lane-0 BP partition), most of them
// shuffles, votes and shared-memory accesses that queue in the MIO pipe: paper_scale 13.2 ms vs 9.8 ms per 860 k
// candidates, Sweep 14.2 ms vs 4.4 ms per 1.97 M.  It cannot be used when a BP has zero demand or in the decode mode.
#pragma once
#include "lgx_kernels.cuh"

#ifndef LGX_EMU      // tests/emu emulates one lane per block: a kernel whose lanes cooperate is not emulated there
namespace lgx {

constexpr int kMaxThreadsW = 1024;        // 32 warps = 32 candidates in flight per SM (<= 64 registers)

// Per-warp shared-memory region (byte offsets from the warp's base; all 4-byte aligned):
//   perm  u16 [n_f + perm_pad]    the Fisher-Yates array in the queue record's own layout (record word w = perm32[w])
//   ds    u32 [n_b]               demands in plan order; cut j overwrites demand j once consumed (as in lgx_decode_cut)
//   bpseq u8  [4 ceil(n_b/4)]     plan order of the BPs | 0x80 = first BP of its tour
//   fa, bin u8 [n_b] each, cnt u8 [n_t]   scratch of the BP partition
//   tgt   i32 [32]                scatter of the "who stored to my position" look-up
struct CutWLayout { uint32_t o_ds, o_bpseq, o_fa, o_bin, o_cnt, o_tgt, bytes; };
__host__ __device__ inline CutWLayout cutw_layout(const ImgHdr &H)
{
  CutWLayout L; uint32_t o = 4u * H.n_perm_words;
  const uint32_t nb4 = ((uint32_t)H.n_b + 3u) & ~3u, nt4 = ((uint32_t)H.n_t + 3u) & ~3u;
  L.o_ds = o; o += 4u * (uint32_t)H.n_b;
  L.o_bpseq = o; o += nb4;
  L.o_fa = o; o += nb4;
  L.o_bin = o; o += nb4;
  L.o_cnt = o; o += nt4;
  L.o_tgt = o; o += 128u;
  L.bytes = (o + 15u) & ~15u;
  return L;
}

template <bool XB64, int MODE>
__global__ void __launch_bounds__(kMaxThreadsW, 1) lgx_decode_cut_w(const __grid_constant__ KParams P)
{
  typedef typename XBits<XB64>::type xb_t;
  extern __shared__ __align__(16) uint8_t smem[];
  const ImgHdr &H = P.H;
  const uint32_t tid = threadIdx.x, T = blockDim.x, lane = tid & 31u, warp = tid >> 5;
  {
    const uint4 *src = reinterpret_cast<const uint4 *>(P.image);
    uint4 *dst = reinterpret_cast<uint4 *>(smem);
    for (uint32_t i = tid; i < H.image_bytes / 16u; i += T) dst[i] = src[i];
  }
  __syncthreads();
  const uint8_t *img = smem;
  const CutWLayout L = cutw_layout(H);
  uint8_t *const wb = smem + H.image_bytes + warp * L.bytes;
  uint16_t *const perm = reinterpret_cast<uint16_t *>(wb);
  uint32_t *const perm32 = reinterpret_cast<uint32_t *>(wb);
  uint32_t *const ds = reinterpret_cast<uint32_t *>(wb + L.o_ds);
  uint8_t *const bpseq = wb + L.o_bpseq, *const fa = wb + L.o_fa, *const binp = wb + L.o_bin, *const cnt = wb + L.o_cnt;
  int *const tgt = reinterpret_cast<int *>(wb + L.o_tgt);
  uint32_t *const draws = perm32;                          // the BP partition's draws, before the permutation is set up

  const uint32_t n_f = H.n_f, n_b = H.n_b, n_t = H.n_t;
  const uint32_t *dq = reinterpret_cast<const uint32_t *>(img + H.off_dq);
  const uint32_t sqs2 = H.sq_shift + 2u;
  const uint8_t *sqb = img + H.off_sq + 4u * (lane & ((1u << H.sq_shift) - 1u));   // this lane's replica of the s_q table
  const uint32_t pad = H.perm_pad;
  const uint32_t n_pre = 4u * H.n_extra_blocks;
  const uint32_t lt_mask = (1u << lane) - 1u;
  constexpr unsigned FULL = 0xFFFFFFFFu;

  for (;;) {
    uint32_t li32 = 0;
    if (lane == 0u) li32 = atomicAdd(P.ctr_a, 1u);        // this warp's next candidate
    li32 = __shfl_sync(FULL, li32, 0);
    if ((uint64_t)li32 >= P.n) break;
    const uint64_t gi = P.base_i + (uint64_t)li32;
    const uint64_t id = P.ids ? P.ids[gi] : P.first_id + gi;
    const uint32_t id_lo = (uint32_t)id, id_hi = (uint32_t)(id >> 32);

    // ---- S2: BPs -> tours (stream 0).  Draw d of the stream = word d mod 4 of block d div 4: FY step p uses d = p, the
    // bin of position p >= n_t uses d = (n_b - 1 - n_t) + p.  All lanes draw, lane 0 places (N_B is small).
    {
      const uint32_t n_draws = 2u * n_b - 1u - n_t;       // draws 0 .. 2 n_b - 2 - n_t
      for (uint32_t blk = lane; 4u * blk < n_draws; blk += 32u) {
        uint32_t w[4];
        philox_block(P, id_lo, id_hi, 0u, blk, w);
        *reinterpret_cast<uint4 *>(draws + 4u * blk) = make_uint4(w[0], w[1], w[2], w[3]);
      }
      __syncwarp();
      if (lane == 0u) {
        for (uint32_t i = 0; i < n_b; ++i) fa[i] = (uint8_t)i;
        for (uint32_t g = 0; g < n_t; ++g) cnt[g] = 1u;   // every tour holds the item of position g ...
        const uint32_t dbin0 = n_b - 1u - n_t;
        for (uint32_t p = 0; p < n_b; ++p) {              // descending Fisher-Yates; position p reads a[n_b-1-p]
          const uint32_t i = n_b - 1u - p;
          const uint32_t j = __umulhi(draws[p], i + 1u);
          const uint8_t x = fa[j], y = fa[i]; fa[j] = y; fa[i] = x;
          uint32_t bin = p;
          if (p >= n_t) { bin = __umulhi(draws[dbin0 + p], n_t); cnt[bin] = (uint8_t)(cnt[bin] + 1u); }   // ... and its share of the rest
          binp[p] = (uint8_t)bin;
        }
        uint32_t acc = 0;
        for (uint32_t g = 0; g < n_t; ++g) { const uint32_t v = cnt[g]; cnt[g] = (uint8_t)acc; acc += v; }
        for (uint32_t p = 0; p < n_b; ++p) {              // plan order = tour 0's list, tour 1's list, ...; inside a tour = consumption order
          const uint32_t g = binp[p];
          const uint32_t pos = cnt[g]; cnt[g] = (uint8_t)(pos + 1u);
          const uint32_t b = fa[n_b - 1u - p];
          bpseq[pos] = (uint8_t)(b | (p < n_t ? 0x80u : 0u));
          ds[pos] = (pos == n_b - 1u) ? 0xFFFFFFFFu : dq[b];          // the last BP never closes (lgx_decode_cut)
        }
      }
      __syncwarp();
    }
    const uint32_t d_last = dq[bpseq[n_b - 1u] & 0x7Fu];   // demand of the last BP in plan order

    // ---- stream 4 up front: bit e = (draw e < thresh) for the first 4*n_extra_blocks draws, a sentinel 1 above
    xb_t xb;
    {
      uint32_t nib = 0;
      if (lane < H.n_extra_blocks) {
        uint32_t w[4];
        philox_block(P, id_lo, id_hi, 4u, lane, w);
        nib = (w[0] < H.thresh ? 1u : 0u) | (w[1] < H.thresh ? 2u : 0u) | (w[2] < H.thresh ? 4u : 0u) | (w[3] < H.thresh ? 8u : 0u);
      }
      const uint32_t lo = __reduce_or_sync(FULL, lane < 8u ? nib << (4u * lane) : 0u);
      const uint32_t hi = __reduce_or_sync(FULL, (lane >= 8u && lane < 16u) ? nib << (4u * (lane - 8u)) : 0u);
      xb = XB64 ? (xb_t)(((unsigned long long)hi << 32) | lo) : (xb_t)lo;
      xb |= (xb_t)1 << n_pre;
    }
    uint32_t e_over = n_pre;                              // index of the next draw beyond the shift register

    // ---- the identity permutation, in the record's layout (element e holds slot e - pad)
    for (uint32_t w = lane; w < H.n_perm_words; w += 32u)
      perm32[w] = (w == 0u) ? H.perm_w0 : ((2u * w - pad) | ((2u * w + 1u - pad) << 16));
    __syncwarp();

    // ---- S3 + S5: fields -> BPs (stream 3), 32 positions per iteration
    uint32_t cur = 0;                                      // plan index of the BP being filled
    uint32_t d_cur = ds[0];
    uint32_t Sq = 0;                                       // its supply so far
    uint32_t fw[4] = {0u, 0u, 0u, 0u};                     // this lane's Philox block of the current round of 128 draws
    for (uint32_t p0 = 0; p0 < n_f; p0 += 32u) {
      if ((p0 & 127u) == 0u) philox_block(P, id_lo, id_hi, 3u, (p0 >> 2) + lane, fw);
      // draw of position p0 + lane = word (lane & 3) of block (p0 >> 2) + (lane >> 2), held by lane 8 b + (lane >> 2), b = sub-block
      const uint32_t src = ((p0 & 127u) >> 2) + (lane >> 2);
      const uint32_t g0 = __shfl_sync(FULL, fw[0], src), g1 = __shfl_sync(FULL, fw[1], src);
      const uint32_t g2 = __shfl_sync(FULL, fw[2], src), g3 = __shfl_sync(FULL, fw[3], src);
      const uint32_t draw = (lane & 2u) ? ((lane & 1u) ? g3 : g2) : ((lane & 1u) ? g1 : g0);
      const uint32_t p = p0 + lane;
      const bool active = p < n_f;
      const uint32_t left = n_f - p;                       // (active lanes) fields still to place = i + 1 of the Fisher-Yates step
      const uint32_t i0 = n_f - 1u - p0;                   // slot of lane 0's step; lane t's is i0 - t
      const uint32_t j = active ? __umulhi(draw, left) : (0xFFFF0000u | lane);   // inactive lanes: a key nobody shares
      uint32_t X = 0, Y = 0;
      if (active) { X = perm[j + pad]; Y = perm[i0 - lane + pad]; }
      // latest earlier lane that stored to slot j (same j) / to this lane's own slot i0 - lane (its j equals it)
      const unsigned same_j = __match_any_sync(FULL, j);
      const uint32_t lower = same_j & lt_mask;
      const int src_x = lower ? (31 - __clz((int)lower)) : -1;
      const bool last_of_j = (same_j >> lane) == 1u;       // no later lane stores to slot j again
      tgt[lane] = -1;
      __syncwarp();
      const uint32_t tpos = i0 - j;                        // lane whose own slot is j (if below 32 and later than this lane)
      if (active && tpos < 32u && tpos > lane) atomicMax(&tgt[tpos], (int)lane);
      __syncwarp();
      const int src_y = tgt[lane];
      // y of every lane as the earlier steps left it: follow the references until nothing changes
      for (;;) {
        const uint32_t Ys = __shfl_sync(FULL, Y, src_y >= 0 ? src_y : (int)lane);
        const bool ch = (src_y >= 0) && (Ys != Y);
        if (ch) Y = Ys;
        if (!__any_sync(FULL, ch)) break;
      }
      {
        const uint32_t Yx = __shfl_sync(FULL, Y, src_x >= 0 ? src_x : (int)lane);
        if (src_x >= 0) X = Yx;
      }
      if (active && last_of_j) perm[j + pad] = (uint16_t)Y;
      __syncwarp();
      if (active) perm[i0 - lane + pad] = (uint16_t)X;    // position p holds field X
      __syncwarp();
      const uint32_t sv = active ? *reinterpret_cast<const uint32_t *>(sqb + (X << sqs2)) : 0u;
      // exclusive prefix sums of the supplies over the lanes
      uint32_t inc = sv;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t u = __shfl_up_sync(FULL, inc, o); if ((int)lane >= o) inc += u; }
      const uint32_t exc = inc - sv;
      const uint32_t n_act = min(32u, n_f - p0);           // active lanes of this block
      const uint32_t tot = __shfl_sync(FULL, inc, 31);
      // the cuts (R21): a BP takes fields until its supply meets its demand, then one more per stream-4 draw below thresh
      uint32_t start = 0, exc_start = 0;                   // first lane of the block that belongs to the current BP, its prefix
      for (;;) {
        const bool cond = active && lane >= start && (Sq + (exc - exc_start)) >= d_cur;
        const unsigned cb = __ballot_sync(FULL, cond);
        if (cb == 0u) { Sq += tot - exc_start; break; }
        const uint32_t c = (uint32_t)__ffs((int)cb) - 1u; // from lane c on every position draws; the BP closes at the first 0 bit
        uint32_t z = c;                                    // lane at which it closes (n_act: not inside this block)
        for (;;) {
          if (z >= n_act) break;
          bool take;
          if (xb > (xb_t)1) { take = ((uint32_t)xb & 1u) != 0u; xb >>= 1; }
          else take = extra_draw(P, id_lo, id_hi, e_over++) != 0u;
          if (!take) break;
          ++z;
        }
        if (z >= n_act) { Sq += tot - exc_start; break; }
        // plan BP `cur` is complete before position p0 + z: its cut is the number of fields still to place there
        if (lane == 0u) ds[cur] = n_f - (p0 + z);
        ++cur;
        __syncwarp();
        d_cur = ds[cur];
        Sq = 0u; start = z; exc_start = __shfl_sync(FULL, exc, (int)z);
      }
    }

    // ---- S5: eq. (2) (L79).  Closed BPs met their demand by construction; the BP that holds the stream's tail and any
    // BP after it (no fields) are the only ones that can fail.
    bool feasible = Sq >= (cur == n_b - 1u ? d_last : d_cur);
    if (lane == 0u) {
      ds[cur] = 0u;                                        // cut at n_f
      uint32_t k = cur;
      while (feasible && k != n_b - 1u) {                  // BPs the stream never reached
        ++k;
        const uint32_t dem = (k == n_b - 1u) ? d_last : ds[k];
        feasible = (dem == 0u);
        ds[k] = 0u;
      }
    }
    feasible = __shfl_sync(FULL, (int)feasible, 0) != 0;
    __syncwarp();
    if (!feasible) {
      if (MODE == MODE_EVAL && lane == 0u) {               // discarded (L186; R19)
        const double inf = __longlong_as_double(0x7FF0000000000000ll);
        if (P.cost)       P.cost[gi] = inf;
        if (P.path_km)    P.path_km[gi] = inf;
        if (P.makespan_h) P.makespan_h[gi] = inf;
        if (P.feasible)   P.feasible[gi] = 0;
      }
      continue;
    }
    // ---- the candidate's record (same layout as lgx_decode_cut writes)
    uint32_t slot = 0;
    if (lane == 0u) slot = atomicAdd(P.q_count, 1u);
    slot = __shfl_sync(FULL, slot, 0);
    const size_t cap = P.cap;
    uint32_t *rec = P.queue + slot;
    if (lane == 0u) { rec[0] = (uint32_t)gi; rec[cap] = (uint32_t)(gi >> 32); }
    for (uint32_t w = lane; w < H.n_bpseq_words; w += 32u) rec[(size_t)(H.rec_bpseq + w) * cap] = *reinterpret_cast<const uint32_t *>(bpseq + 4u * w);
    for (uint32_t w = lane; w < H.n_segend_words; w += 32u) {    // two 16-bit end positions per word
      uint32_t v = n_f - ds[2u * w];
      if (2u * w + 1u < n_b) v |= (n_f - ds[2u * w + 1u]) << 16;
      rec[(size_t)(H.rec_segend + w) * cap] = v;
    }
    for (uint32_t w = lane; w < H.n_perm_words; w += 32u) rec[(size_t)(H.rec_perm + w) * cap] = perm32[w];
    __syncwarp();                                          // the region is reused by the next candidate's draws
  }
}

}  // namespace lgx
#endif  // LGX_EMU
