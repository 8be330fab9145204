// lgx_image.h — layout of the instance images that live in shared memory,
// of the per-candidate state rows, and of the queue record that carries a feasible
// candidate from the decode/walk kernel to the finish kernel.
// Product code (CUDA path).  Shares nothing with oracle/.
//
// Image AB (decode + pass 1):   distance tables or coordinates | {s_q,h_q} per field | demand quanta
// Image C  (Alg. 2 + pass 2):   field x BP table or coordinates | s_q per field | HU rate quanta |
//                               SU capacities by rank | RN(1/k) table | unit<->rank maps
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

namespace lgx {

constexpr int      kQ           = 1024;          // quanta per t / ha / (ha/h)   (R18)
constexpr uint32_t kPhiloxM0    = 0xD2511F53u;   // Philox4x32 multipliers (Salmon et al., SC'11)
constexpr uint32_t kPhiloxM1    = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0    = 0x9E3779B9u;   // key increments
constexpr uint32_t kPhiloxW1    = 0xBB67AE85u;
constexpr int      kMaxSmem     = 227 * 1024;    // opt-in dynamic shared memory per block, sm_100a
constexpr int      kMaxThreads  = 512;           // __launch_bounds__ of the finish kernel
constexpr int      kMaxThreadsA = 640;           // __launch_bounds__ of the decode/walk kernel (<= 96 registers)
constexpr int      kFinishBlocksPerSM = 2;       // the finish kernel's image is small: two blocks share an SM

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

  // ---- image AB (byte offsets)
  uint32_t off_dtri;        // f64 [(n_f+1) n_f / 2]  strict lower triangle over {HQ, fields}
  uint32_t off_dfb;         // f64 [n_f][n_b]         field -> BP legs
  uint32_t off_xy;          // f64x2 [1 + n_b + n_f]  vertex coordinates (coords mode)
  uint32_t off_sh;          // u32x2 [n_f]            {s_q, h_q}
  uint32_t off_dq;          // u32 [n_b]              demand quanta
  uint32_t image_bytes;

  // ---- image C (byte offsets inside image C)
  uint32_t offc_dfb, offc_xy, offc_s, offc_cs, offc_rcp, offc_unit;
  uint32_t offc_rq;         // u32 [n_hu]  HU rate quanta
  uint32_t offc_rank;       // u8  [n_su]  unit -> rank
  uint32_t offc_hrs;        // u32 [n_hu]  HU rate quanta by rank (ascending (rate, unit)): the embedded HU assignment (N2)
  uint32_t offc_hunit;      // u8  [n_hu]  rank -> HU
  uint32_t offc_hrank;      // u8  [n_hu]  HU -> rank
  uint32_t flags;           // lgx_instance_desc.flags (bit 1: Algorithm 1's workers embed the HU assignment)
  uint32_t imagec_bytes;

  // ---- state rows of the decode/walk kernel
  uint32_t a64_sd, a64_lt, a64_ent, a64_rows;
  uint32_t a32_perm, a32_bpseq, a32_segend, a32_scra, a32_scrb, a32_hq, a32_rows;

  // ---- state rows of the finish kernel
  uint32_t c64_w, c64_e, c64_mask, c64_rows;
  uint32_t c32_s, c32_nhu, c32_r, c32_ng, c32_magic, c32_ent, c32_scra, c32_rows;

  // ---- queue record (32-bit words, stored transposed: word w of slot q at queue[w*cap + q])
  //   0,1 index i | per tour g at rec_tour + g*rec_tw: LT lo,hi, H_q |
  //   SD[j] lo,hi at rec_sd + 2j | bpseq words | segend words | perm words
  uint32_t rec_tour, rec_tw, rec_sd, rec_bpseq, rec_segend, rec_perm, rec_words;
  uint32_t n_bpseq_words, n_segend_words, n_perm_words;
  uint32_t pad_[2];
};
static_assert(sizeof(ImgHdr) % 16 == 0, "image header must keep 16-byte alignment");

}  // namespace lgx
