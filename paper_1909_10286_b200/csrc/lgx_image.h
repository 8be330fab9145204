// lgx_image.h — layout of the instance image that lives in shared memory.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// The image is one contiguous, 16-byte aligned blob built on the host by
// lgx_instance_create and copied global -> shared once per (persistent) block:
//
//   ImgHdr | distance tables or coordinates | per-field quanta | per-BP demand quanta |
//   HU rate quanta | SU capacities sorted by (capacity, unit) | unit<->rank maps
//
// It is followed in shared memory by the per-candidate state: `words_per_thread` rows of
// blockDim.x 32-bit words, row-major, so that word r of thread t sits at
// state[r * blockDim.x + t] — every dynamically indexed per-thread access (Fisher-Yates
// swaps, per-tour accumulators) then hits bank t % 32 whatever the index: conflict-free
// by construction.
#pragma once
#include <stdint.h>

namespace lgx {

constexpr int      kQ           = 1024;          // quanta per t / ha / (ha/h)   (R18)
constexpr uint32_t kPhiloxM0    = 0xD2511F53u;   // Philox4x32 multipliers (Salmon et al., SC'11)
constexpr uint32_t kPhiloxM1    = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0    = 0x9E3779B9u;   // key increments
constexpr uint32_t kPhiloxW1    = 0xBB67AE85u;
constexpr int      kMaxSmem     = 227 * 1024;    // opt-in dynamic shared memory per block, sm_100a
constexpr int      kMaxThreads  = 512;           // __launch_bounds__ of the candidate kernels

// Per-tour rows of the per-candidate state (32-bit words).
enum TourRow : uint32_t {
  TR_LT   = 0,   // f64  closed HU route length L_tour(g)             (pass 1)
  TR_E    = 2,   // f64  sumE during pass 1, then E(g)                (Alg. 2 step 1)
  TR_W    = 4,   // f64  T_wait(g) cache                              (Alg. 2)
  TR_SH   = 6,   // f64  shuttle distance sum of the tour             (pass 2)
  TR_HQ   = 8,   // u32  harvested area quanta H_q(g)
  TR_R    = 9,   // u32  sum of HU rate quanta R_g
  TR_S    = 10,  // u32  sum of SU capacity quanta S_g = C_g
  TR_CNT  = 11,  // u32  n_HU(g) | m(g) << 16
  TR_MASK = 12,  // u64 x MASKW  SU membership by capacity rank
};

struct ImgHdr {
  int32_t  n_f, n_b, n_hu, n_su, n_t;
  uint32_t thresh;
  int32_t  coords;          // 0: packed HQ+field triangle + field x BP table; 1: coordinates
  int32_t  perm16;          // field ids / segment ends stored as u16 instead of u8
  double   v_hu, v_su, kappa, w_path, w_time;
  uint32_t off_dtri;        // f64 [(n_f+1) n_f / 2]  strict lower triangle over {HQ, fields}
  uint32_t off_dfb;         // f64 [n_f][n_b]         field -> BP legs
  uint32_t off_xy;          // f64x2 [1 + n_b + n_f]  vertex coordinates (coords mode)
  uint32_t off_sh;          // u32x2 [n_f]            {s_q, h_q}
  uint32_t off_dq;          // u32 [n_b]              demand quanta
  uint32_t off_rq;          // u32 [n_hu]             HU rate quanta
  uint32_t off_cs;          // u32 [n_su]             SU capacity quanta, ascending (c_q, unit)
  uint32_t off_rank;        // u8  [n_su]             unit -> rank
  uint32_t off_unit;        // u8  [n_su]             rank -> unit
  uint32_t off_rcp;         // f64 [max(n_f,n_b,n_hu)+1]  RN(1/k), for the exact small-divisor division
  uint32_t row_perm, row_bpseq, row_segend, row_scra, row_scrb, row_tour;
  uint32_t tour_words, words_per_thread;
  uint32_t image_bytes;
  uint32_t mask_words;      // 64-bit words per SU mask (1 or 2)
  uint32_t n_extra_blocks;  // Philox blocks of stream 4 drawn up front (<= 16)
};
static_assert(sizeof(ImgHdr) % 16 == 0, "image header must keep 16-byte alignment");

}  // namespace lgx
