// lgx_image.h — layout of the instance images that live in shared memory,
// of the per-candidate state rows, and of the queue record that carries a feasible
// candidate from the decode/cut kernel to the walk/finish kernel.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Image A (lgx_decode_cut: decode + eq. (2), integers only):
//     s_q per field (replicated 2^sq_shift times so that lanes read different banks) | demand quanta
// Image C (lgx_walk_finish: geometry, Algorithm 2, shuttles, cost):
//     distance tables and/or coordinates | {s_q, h_q} per field | SU capacities by rank | RN(1/k) table |
//     unit <-> rank maps | HU rate quanta
// Both are contiguous, 16-byte aligned blobs built on the host by lgx_instance_create and
// copied global -> shared once per (persistent) block.
//
// Per-candidate state follows the image in shared memory as ROWS of blockDim.x cells:
// cell (row r, thread t) of the 64-bit region at  state64 + (r*blockDim.x + t)*8,
// cell (row r, thread t) of the 32-bit region at  state32 + (r*blockDim.x + t)*4,
// so every dynamically indexed per-thread access (Fisher-Yates swaps, per-BP / per-tour
// accumulators) hits bank(s) fixed by t alone: conflict-free whatever the index
// (SURVEY §7 H2).
#pragma once
#include <stdint.h>

// Dynamic shared memory of a kernel.  (tests/emu compiles the kernels for the host, single lane, to check their
// indexing under AddressSanitizer; it predefines the three macros below.  The CUDA build always takes these defaults.)
#ifndef LGX_DYN_SMEM
#define LGX_DYN_SMEM(name) extern __shared__ __align__(16) uint8_t name[]
#endif
#ifndef LGX_LANES
#define LGX_LANES 32u            // lanes that draw work together (a warp)
#endif
#ifndef LGX_BLOCK_THREADS
#define LGX_BLOCK_THREADS(t) (t) // threads a launch of the sampling kernels uses (the host-side check of tests/emu runs one)
#endif

namespace lgx {

constexpr int      kQ           = 1024;          // quanta per t / ha / (ha/h)   (R18)
constexpr uint32_t kPhiloxM0    = 0xD2511F53u;   // Philox4x32 multipliers (Salmon et al., SC'11)
constexpr uint32_t kPhiloxM1    = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0    = 0x9E3779B9u;   // key increments
constexpr uint32_t kPhiloxW1    = 0xBB67AE85u;
constexpr int      kMaxSmem     = 227 * 1024;    // opt-in dynamic shared memory per block, sm_100a
constexpr int      kMaxThreadsA = 1024;          // __launch_bounds__ of the decode/cut kernel (<= 64 registers)
constexpr int      kMaxThreadsA16 = 384;         // ... with 16-bit field ids (N_F > 255: the permutation caps the residency anyway; <= 168 registers)
constexpr int      kMaxThreadsB = 640;           // __launch_bounds__ of the walk/finish kernel with distance tables (<= 96 registers)
constexpr int      kMaxThreadsBC = 448;          // ... with coordinates (<= 144 registers: several square-root chains in flight)
constexpr uint32_t kLanes       = LGX_LANES;

struct ImgHdr {
  int32_t  n_f, n_b, n_hu, n_su, n_t;
  uint32_t thresh;
  int32_t  coords;          // distance mode 0: HQ+field triangle + field x BP table; 1: coordinates; 2: field x BP table + coordinates
  int32_t  perm16;          // field ids / segment ends stored as u16 instead of u8
  double   v_hu, v_su, kappa, w_path, w_time;
  uint32_t mask_words;      // 64-bit words per SU mask (1 or 2)
  uint32_t n_extra_blocks;  // Philox blocks of stream 4 drawn up front (<= 16)
  uint32_t perm_pad;        // right-alignment of the permutation array inside its words
  uint32_t perm_w0;         // initial value of permutation word 0 (bytes below perm_pad unused)
  uint32_t sq_shift;        // log2 of the replication factor of image A's s_q table
  uint32_t zero_demand;     // some BP has zero demand: one field step may close several BPs (R21)

  // ---- image A (byte offsets)
  uint32_t off_sq;          // u32 [n_f << sq_shift]  s_q; field f, replica r at (f << sq_shift) + r
  uint32_t off_dq;          // u32 [n_b]              demand quanta
  uint32_t image_bytes;

  // ---- image C (byte offsets inside image C)
  uint32_t offc_dtri;       // f64 [(n_f+1) n_f / 2]  strict lower triangle over {HQ, fields}      (mode 0)
  uint32_t offc_dfb;        // f64 [n_f][n_b]         field -> BP legs                              (modes 0, 2)
  uint32_t offc_xy;         // f64x2 [1 + n_b + n_f]  vertex coordinates                            (modes 1, 2)
  uint32_t offc_bxy;        // f64x2 [n_b][8]         BP coordinates, replica r of BP b at 8 b + r (lane l reads replica l & 7:
                            //                        the 16-byte loads of a quarter-warp never share a bank group)  (mode 1)
  uint32_t offc_dhq;        // f64 [n_f]              field -> HQ legs (the closing leg of a tour)  (modes 1, 2)
  uint32_t offc_sh;         // u32x2 [n_f]            {s_q, h_q}
  uint32_t offc_suinit;     // u32 [..]    initial array of the SU partition: capacity ranks of units 0.., right-aligned bytes
  uint32_t offc_cs;         // u32 [n_su]  SU capacity quanta by rank (ascending (capacity, unit)); the move kernels copy image C from here on
  uint32_t offc_rcp;        // f64 [..]    RN(1/k)
  uint32_t offc_unit;       // u8  [n_su]  rank -> SU
  uint32_t offc_rq;         // u32 [n_hu]  HU rate quanta
  uint32_t offc_rank;       // u8  [n_su]  SU -> rank
  uint32_t offc_hrs;        // u32 [n_hu]  HU rate quanta by rank (ascending (rate, unit)): the embedded HU assignment (N2)
  uint32_t offc_hunit;      // u8  [n_hu]  rank -> HU
  uint32_t offc_hrank;      // u8  [n_hu]  HU -> rank
  uint32_t flags;           // lgx_instance_desc.flags
  uint32_t imagec_bytes;

  // ---- state rows of the decode/cut kernel (32-bit rows only)
  uint32_t a32_perm, a32_bpseq, a32_ds, a32_scra, a32_scrb, a32_cnt, a32_rows;
  uint32_t a32_scru, a32_rows_dec;      // diagnostic decode mode: scratch of the unit partitions, appended

  // ---- state rows of the walk/finish kernel
  uint32_t c64_w, c64_e, c64_mask, c64_sd, c64_tp, c64_rows;
  uint32_t c32_s, c32_hn, c32_r, c32_hq, c32_ent, c32_rows;

  // ---- queue record (32-bit words, stored transposed: word w of slot q at queue[w*cap + q])
  //   0,1 index i | bpseq words | segend words | perm words
  uint32_t rec_bpseq, rec_segend, rec_perm, rec_words;
  uint32_t n_bpseq_words, n_segend_words, n_perm_words;
};
static_assert(sizeof(ImgHdr) % 16 == 0, "image header must keep 16-byte alignment");

}  // namespace lgx
