// lgx_api.cu — C ABI of lgx (include/lgx.h): instance encoder (host side) and launchers.
// Product code (CUDA path); shares nothing with oracle/.  No CPU fallback: every compute
// entry point fails with LGX_ECUDA when there is no usable CUDA device.
#include "../../include/lgx.h"
#include "lgx_image.h"
#include "lgx_dispatch.h"
#include "lgx_moves.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <mutex>
#include <vector>

using namespace lgx;

struct lgx_instance {
  ImgHdr hdr{};
  std::vector<uint8_t> image, image_c;       // host copies of the two images
  std::vector<uint32_t> s_q, d_q;            // supply / demand quanta (image A is rebuilt when its replication changes)
  uint8_t *d_image = nullptr, *d_image_c = nullptr;
  size_t d_image_cap = 0;                    // bytes allocated behind d_image
  int device = 0, sm_count = 0;
  int64_t smem_budget = 0;                   // dynamic shared memory one block may take
  // launch configuration of the persistent kernels (lgx_decode_cut: a, its diagnostic decode mode: a_dec; lgx_walk_finish: b)
  int threads_a = 0, threads_a_dec = 0, threads_b = 0, grid = 0;
  int walk_lockstep = 0;                            // lgx_walk_finish: block-synchronous work fetch (default with coordinates)
  uint64_t a_state = 0, a_state_dec = 0, b_state = 0;   // per-candidate shared-memory bytes
  uint64_t chunk = 0;                          // candidates per decode/finish kernel pair
  cudaMemPool_t pool = nullptr;                // the device's workspace pool (owned by the library, not by the instance)
  mutable std::atomic<long long> launches{0};
  // optional per-kernel timing (lgx_instance_set_timing): CUDA events around every launch of a search
  mutable std::atomic<int> timing{0};
  mutable std::atomic<long long> ns_a{0}, ns_c{0}, timed_pairs{0};
  // move kernels (Algorithm 1: lgx_init_plan, lgx_move_eval_batch, lgx_local_search)
  MvHdr mv{};
  double2 *d_xy = nullptr;                     // vertex coordinates, every distance mode (lgx_init_plan)
  int threads_mv = 0, max_threads_mv = 0; size_t smem_mv = 0; int64_t mv_state = 0;
};

namespace {

thread_local std::string g_cuda_msg = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char *where)
{
  g_cuda_msg = std::string(where) + ": " + cudaGetErrorString(e);
  cudaGetLastError();
  return LGX_ECUDA;
}
#define CU(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__, #call); } while (0)

inline bool fin_nonneg(double v) { return std::isfinite(v) && v >= 0.0; }
inline int64_t quantise(double v) { return (int64_t)std::llrint(v * (double)kQ); }   // round-half-even (R18)
inline uint32_t align16(uint32_t v) { return (v + 15u) & ~15u; }
inline uint32_t cdiv(uint32_t a, uint32_t b) { return (a + b - 1u) / b; }

// Straight-line edge, one rounding per operation (compiled with -ffp-contract=off).
inline double edge(double ax, double ay, double bx, double by)
{
  const double dx = ax - bx, dy = ay - by;
  const double xx = dx * dx, yy = dy * dy;
  const double ss = xx + yy;
  return std::sqrt(ss);
}

template <int MODE> void pick_kernels(const ImgHdr &h, KernelFn &ka, KernelFn &kb)
{
  ka = pick_decode_cut(h, MODE);
  kb = h.coords == 0 ? pick_walk_finish_dm0(h, MODE) : (h.coords == 1 ? pick_walk_finish_dm1(h, MODE) : pick_walk_finish_dm2(h, MODE));
}

void fill_round_keys(KParams &P, uint64_t seed)
{
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { P.rk[2 * r] = k0; P.rk[2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
}

// Every compute entry point runs on the device the instance was created on (its images live there).
int check_device(const lgx_instance *I)
{
  int cur = -1;
  CU(cudaGetDevice(&cur));
  if (cur != I->device) { g_cuda_msg = "the current CUDA device is not the one the instance was created on"; return LGX_EINVAL; }
  return LGX_OK;
}

// Image A: s_q replicated 2^sq_shift times (replica r of field f at (f << sq_shift) + r: lanes of a warp read
// different banks whatever field they hold) and the demand quanta.  Built and uploaded into a NEW device buffer; the
// instance (header offsets, host copy, device pointer) changes only once the upload has succeeded, so a failure
// leaves it exactly as it was, still usable with its previous image.
int build_image_a(lgx_instance *I, uint32_t sq_shift)
{
  ImgHdr &H = I->hdr;
  const uint32_t nf = (uint32_t)H.n_f, nb = (uint32_t)H.n_b;
  uint32_t off = 0;
  const uint32_t off_sq = off; off = align16(off + 4u * (nf << sq_shift));
  const uint32_t off_dq = off; off = align16(off + 4u * nb);
  const uint32_t bytes = off;
  std::vector<uint8_t> img(bytes, 0);
  uint32_t *sq = reinterpret_cast<uint32_t *>(img.data() + off_sq);
  for (uint32_t f = 0; f < nf; ++f)
    for (uint32_t r = 0; r < (1u << sq_shift); ++r) sq[(f << sq_shift) + r] = I->s_q[f];
  uint32_t *dq = reinterpret_cast<uint32_t *>(img.data() + off_dq);
  for (uint32_t b = 0; b < nb; ++b) dq[b] = I->d_q[b];
  uint8_t *d_new = nullptr;
  CU(cudaMalloc((void **)&d_new, bytes));
  cudaError_t e = cudaMemcpy(d_new, img.data(), bytes, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(d_new); return cuda_fail(e, "cudaMemcpy(image A)"); }
  if (I->d_image) cudaFree(I->d_image);
  I->d_image = d_new; I->d_image_cap = bytes;
  I->image.swap(img);
  H.sq_shift = sq_shift; H.off_sq = off_sq; H.off_dq = off_dq; H.image_bytes = bytes;
  return LGX_OK;
}

int64_t fit_threads(int64_t budget, int64_t image, int64_t state, int64_t cap)
{
  const int64_t t = (budget - image) / std::max<int64_t>(state, 1);
  return std::min<int64_t>(t, cap) / 32 * 32;
}

// Launch configuration of the decode/cut kernel as a function of image A's size: the create-time defaults.  Used by
// lgx_instance_create and again whenever LGX_OPT_SQ_SHIFT has rebuilt the image (it resets LGX_OPT_THREADS_A to
// this default; nothing is derived from the values in place before).
void config_decode_cut(lgx_instance *I)
{
  const ImgHdr &H = I->hdr;
  const int64_t budget = I->smem_budget;
  I->threads_a     = (int)fit_threads(budget, H.image_bytes, (int64_t)I->a_state, H.perm16 ? kMaxThreadsA16 : kMaxThreadsA);
  I->threads_a_dec = (int)fit_threads(budget, H.image_bytes, (int64_t)I->a_state_dec, H.perm16 ? kMaxThreadsA16 : kMaxThreadsA);
}

// Stream-ordered workspace memory (the queue of feasible candidates, a few hundred bytes of counters) comes from ONE
// memory pool per device, created on first use and kept for the life of the process with its release threshold at the
// maximum: a freed workspace stays mapped, so creating an instance and searching with it does not pay for mapping
// the queue again (measured: ~150 ms per 2 GiB).  lgx_workspace_trim() hands the cached memory back.
constexpr int kMaxDevices = 64;
std::mutex g_pool_mutex;
cudaMemPool_t g_pools[kMaxDevices] = {};

int device_pool(int device, cudaMemPool_t *out)
{
  if (device < 0 || device >= kMaxDevices) return LGX_EINVAL;
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pools[device]) {
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = device;
    cudaMemPool_t pool = nullptr;
    CU(cudaMemPoolCreate(&pool, &props));
    // without the threshold every freed workspace goes back to the driver at the next synchronisation and each call
    // maps its queue again (correct, but several times slower end to end): treat a refusal as an error, not as a detail
    uint64_t keep = ~0ull;
    cudaError_t e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    if (e != cudaSuccess) { cudaMemPoolDestroy(pool); return cuda_fail(e, "cudaMemPoolSetAttribute(release threshold)"); }
    g_pools[device] = pool;
  }
  *out = g_pools[device];
  return LGX_OK;
}

void free_instance(lgx_instance *I)
{
  if (I->d_xy) cudaFree(I->d_xy);
  if (I->d_image) cudaFree(I->d_image);
  if (I->d_image_c) cudaFree(I->d_image_c);
  delete I;
}

// The kernels take up to 227 KB of dynamic shared memory: the opt-in attribute is set ONCE per kernel, to the
// device maximum, when an instance that uses the kernel is created — never per call, so concurrent calls on
// instances of different sizes cannot race on it.
int allow_max_smem(const void *fn, int smem_optin)
{
  cudaFuncAttributes fa{};
  CU(cudaFuncGetAttributes(&fa, fn));                      // the kernel's static shared memory counts against the limit
  CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, std::min(smem_optin, kMaxSmem) - (int)fa.sharedSizeBytes));
  return LGX_OK;
}

void pick_move_kernels(const ImgHdr &h, MvKernelFn &kb, MvKernelFn &ks);

}  // namespace

namespace lgx { int pipe_bench(int what, uint64_t iters, uint64_t *h_out); }   // lgx_pipes.cu

extern "C" {

const char *lgx_strerror(int code)
{
  switch (code) {
    case LGX_OK:      return "ok";
    case LGX_EINVAL:  return "invalid argument or instance outside the documented ranges";
    case LGX_ETOOBIG: return "instance image or per-candidate state does not fit (shared memory / 32-bit quanta / kernel limits)";
    case LGX_ECUDA:   return g_cuda_msg.c_str();
    case LGX_ENOMEM:  return "out of memory";
    case LGX_ESTATIC: return "lgx_eval_batch_static: n is larger than the library's fixed device scratch holds for this instance (lgx_eval_batch_static_max)";
    default:          return "unknown lgx error code";
  }
}

int lgx_instance_create(const lgx_instance_desc *d, lgx_instance **out)
{
  if (!d || !out) return LGX_EINVAL;
  *out = nullptr;
  // ---- validation (same documented rules as the header; PAPER.md:L69 N_T <= N_HU^total)
  if (d->n_fields < 1 || d->n_bps < 1 || d->n_hu_total < 1 || d->n_su_total < 1) return LGX_EINVAL;
  if (d->n_tours < 1 || d->n_tours > d->n_bps || d->n_tours > d->n_hu_total || d->n_tours > d->n_su_total) return LGX_EINVAL;
  if (d->n_fields > 65535 || d->n_bps > 255 || d->n_tours > 255 || d->n_hu_total > 255 || d->n_su_total > 255) return LGX_EINVAL;
  if (!d->field_x || !d->field_y || !d->field_supply_t || !d->field_area_ha || !d->bp_x || !d->bp_y ||
      !d->bp_demand_t || !d->hu_rate_ha_per_h || !d->su_capacity_t) return LGX_EINVAL;
  if (!std::isfinite(d->hq_x) || !std::isfinite(d->hq_y)) return LGX_EINVAL;
  if (!(std::isfinite(d->v_hu_road_kmh) && d->v_hu_road_kmh > 0.0)) return LGX_EINVAL;
  if (!(std::isfinite(d->v_su_road_kmh) && d->v_su_road_kmh > 0.0)) return LGX_EINVAL;
  if (!fin_nonneg(d->su_fill_h_per_t) || !fin_nonneg(d->w_path) || !fin_nonneg(d->w_time)) return LGX_EINVAL;
  const uint32_t known_flags = LGX_FLAG_HU_BALANCE | LGX_FLAG_MAKESPAN_FILTER | LGX_FLAG_FIX_FIELD_BP |
                               LGX_FLAG_DIST_COORDS | LGX_FLAG_DIST_MIXED;
  if ((d->flags & ~known_flags) != 0u) return LGX_EINVAL;
  if ((d->flags & LGX_FLAG_DIST_COORDS) && (d->flags & LGX_FLAG_DIST_MIXED)) return LGX_EINVAL;
  const int nf = d->n_fields, nb = d->n_bps, nhu = d->n_hu_total, nsu = d->n_su_total, nt = d->n_tours;
  for (int f = 0; f < nf; ++f)
    if (!std::isfinite(d->field_x[f]) || !std::isfinite(d->field_y[f]) || !fin_nonneg(d->field_supply_t[f]) ||
        !fin_nonneg(d->field_area_ha[f])) return LGX_EINVAL;
  for (int b = 0; b < nb; ++b)
    if (!std::isfinite(d->bp_x[b]) || !std::isfinite(d->bp_y[b]) || !fin_nonneg(d->bp_demand_t[b])) return LGX_EINVAL;
  for (int u = 0; u < nhu; ++u) if (!fin_nonneg(d->hu_rate_ha_per_h[u])) return LGX_EINVAL;
  for (int u = 0; u < nsu; ++u) if (!fin_nonneg(d->su_capacity_t[u])) return LGX_EINVAL;

  // ---- quantisation (Q = 1024) and the documented 32-bit ranges
  std::vector<int64_t> s_q(nf), h_q(nf), d_q(nb), r_q(nhu), c_q(nsu);
  int64_t s_max = 0, s_sum = 0, h_sum = 0, r_sum = 0, c_sum = 0;
  for (int f = 0; f < nf; ++f) {
    s_q[f] = quantise(d->field_supply_t[f]); h_q[f] = quantise(d->field_area_ha[f]);
    s_max = std::max(s_max, s_q[f]); s_sum += s_q[f]; h_sum += h_q[f];
  }
  for (int b = 0; b < nb; ++b) d_q[b] = quantise(d->bp_demand_t[b]);
  for (int u = 0; u < nhu; ++u) { r_q[u] = quantise(d->hu_rate_ha_per_h[u]); if (r_q[u] <= 0) return LGX_EINVAL; r_sum += r_q[u]; }
  for (int u = 0; u < nsu; ++u) { c_q[u] = quantise(d->su_capacity_t[u]); if (c_q[u] <= 0) return LGX_EINVAL; c_sum += c_q[u]; }
  const int64_t lim = (int64_t)1 << 32;
  // (sum s_q stays below 2^32 - 1: the decode/cut kernel marks the last BP of a plan with the demand 2^32 - 1)
  if (s_max * (int64_t)nsu + c_sum >= lim || s_sum >= lim - 1 || h_sum >= lim || r_sum >= lim) return LGX_ETOOBIG;
  for (int b = 0; b < nb; ++b) if (d_q[b] >= lim) return LGX_ETOOBIG;
  // kernel limits of this build (include/lgx.h): 7-bit BP ids in the plan entries, SU sets of 2 x 64 bits
  if (nb > LGX_MAX_BPS || nsu > LGX_MAX_SUS) return LGX_ETOOBIG;

  lgx_instance *I = new (std::nothrow) lgx_instance();
  if (!I) return LGX_ENOMEM;
  ImgHdr &H = I->hdr;
  H.n_f = nf; H.n_b = nb; H.n_hu = nhu; H.n_su = nsu; H.n_t = nt;
  H.thresh = d->extra_field_thresh;
  H.v_hu = d->v_hu_road_kmh; H.v_su = d->v_su_road_kmh; H.kappa = d->su_fill_h_per_t;
  H.w_path = d->w_path; H.w_time = d->w_time;
  H.flags = d->flags;
  H.perm16 = nf > 255 ? 1 : 0;
  H.mask_words = nsu > 64 ? 2u : 1u;
  const uint32_t MW = H.mask_words;
  // stream-4 draws taken up front: (N_B-1) failures + geometric extras, with slack; <= 60 (+ a sentinel bit)
  H.n_extra_blocks = (uint32_t)std::min(15, ((nb - 1) * 4 / 3 + 8 + 3) / 4);
  I->s_q.resize(nf); I->d_q.resize(nb);
  for (int f = 0; f < nf; ++f) I->s_q[f] = (uint32_t)s_q[f];
  H.zero_demand = 0u;
  for (int b = 0; b < nb; ++b) { I->d_q[b] = (uint32_t)d_q[b]; if (d_q[b] == 0) H.zero_demand = 1u; }

  // ---- permutation array: right-aligned inside its words so that consumption position
  //      p = EPW*q + t always sits in a static lane of word row wtop - q
  const uint32_t EPW = H.perm16 ? 2u : 4u;
  H.perm_pad = (EPW - (uint32_t)nf % EPW) % EPW;
  H.n_perm_words = ((uint32_t)nf + H.perm_pad) / EPW;
  {
    uint32_t w0 = 0;
    for (uint32_t t = 0; t < EPW; ++t) {
      const uint32_t v = (t >= H.perm_pad) ? (t - H.perm_pad) : 0u;
      w0 |= (v & (H.perm16 ? 0xFFFFu : 0xFFu)) << (t * (H.perm16 ? 16u : 8u));
    }
    H.perm_w0 = w0;
  }
  H.n_bpseq_words  = cdiv((uint32_t)nb, 4u);
  H.n_segend_words = cdiv((uint32_t)nb, EPW);

  // ---- state rows of the decode/cut kernel: 32-bit rows only (the kernel touches no FP64)
  const uint32_t n_units = (uint32_t)std::max(nhu, nsu);
  {
    uint32_t r = 0;
    H.a32_perm = r;  r += H.n_perm_words;
    H.a32_bpseq = r; r += H.n_bpseq_words;
    H.a32_ds = r;    r += (uint32_t)nb;                    // demands in plan order; cut j overwrites demand j once consumed
    H.a32_scra = r;  r += ((uint32_t)nb + 3u) / 4u + 1u;   // BP partition: Fisher-Yates array
    H.a32_scrb = r;  r += cdiv((uint32_t)nb, 4u);          // bin of consumption position p
    H.a32_cnt = r;   r += cdiv((uint32_t)nt, 4u);          // counting sort cursors
    H.a32_rows = r;
    H.a32_scru = r;  r += (n_units + 3u) / 4u + 1u;        // diagnostic decode mode only: unit partitions
    H.a32_rows_dec = r;
  }
  // ---- state rows of the walk/finish kernel.  Rows are reused as their contents die (lgx_kernels.cuh): one block of
  //      64-bit rows holds SD per plan BP, then T_wait(g) | the walk's tour parameters; the 32-bit rows of H_q(g) and of
  //      the walk entries are the unit partitions' scratch before (a thread only ever aliases its OWN cells: warps of a
  //      block are in different phases).
  {
    const uint32_t scratch_rows = (n_units + 3u) / 4u + 1u;
    const uint32_t blk = std::max((uint32_t)nb, 2u * (uint32_t)nt);
    uint32_t r = 0;
    H.c64_w = r; H.c64_sd = r; H.c64_tp = r + (uint32_t)nt; r += blk;
    H.c64_e = r; r += (uint32_t)nt;                        // sumE(g), E(g); then L_tour(g)
    H.c64_mask = r; r += (uint32_t)nt * MW;
    H.c64_rows = r;
    r = 0;
    H.c32_s = r; r += (uint32_t)nt;
    H.c32_hn = r; r += (uint32_t)nt;                       // n_HU(g) | n_SU(g) << 8 | m(g) << 16
    H.c32_r = r; r += (uint32_t)nt;
    H.c32_hq = r; H.c32_ent = r + (uint32_t)nt;            // H_q(g); walk entries + sentinel
    r += std::max((uint32_t)nt + (uint32_t)nb + 1u, scratch_rows);
    H.c32_rows = r;
  }
  // ---- queue record
  {
    uint32_t w = 2;
    H.rec_bpseq = w;  w += H.n_bpseq_words;
    H.rec_segend = w; w += H.n_segend_words;
    H.rec_perm = w;   w += H.n_perm_words;
    H.rec_words = w;
  }
  I->a_state = 4ull * H.a32_rows;
  I->a_state_dec = 4ull * H.a32_rows_dec;
  I->b_state = 8ull * H.c64_rows + 4ull * H.c32_rows;

  // ---- image C: packed distance tables when they leave room for >= 256 candidates per SM, else the
  //      field x BP table + coordinates while the table is small, else coordinates only
  const uint64_t tri_bytes = (uint64_t)(nf + 1) * (uint64_t)nf / 2 * 8, dfb_bytes = (uint64_t)nf * nb * 8;
  const uint64_t xy_bytes = 16ull * (1 + nb + nf) + 128ull * nb, room = (uint64_t)kMaxSmem - 1024;   // (+ the BP replicas of mode 1)
  const int n_rcp = std::max(nf, std::max(nb, nhu)) + 1;
  const uint64_t tail_bytes = 8ull * nf + 8ull * nf + 6ull * nsu + 8ull * n_rcp + 2ull * nsu + 8ull * nhu + 2ull * nhu + 320;
  if (tail_bytes + tri_bytes + dfb_bytes + 256ull * I->b_state <= room) H.coords = 0;
  else if (dfb_bytes <= 32ull * 1024 && tail_bytes + dfb_bytes + xy_bytes + 128ull * I->b_state <= room) H.coords = 2;
  else H.coords = 1;
  if (d->flags & LGX_FLAG_DIST_COORDS) H.coords = 1;      // tuning flags: same D(u,v) bit for bit
  if ((d->flags & LGX_FLAG_DIST_MIXED) && tail_bytes + dfb_bytes + xy_bytes + 32ull * I->b_state <= room) H.coords = 2;
  uint32_t off = 0;
  H.offc_dtri = H.offc_dfb = H.offc_xy = 0;
  if (H.coords == 0) { H.offc_dtri = off; off = align16(off + (uint32_t)tri_bytes); }
  if (H.coords != 1) { H.offc_dfb = off; off = align16(off + (uint32_t)dfb_bytes); }
  if (H.coords != 0) { H.offc_xy = off; off = align16(off + 16u * (uint32_t)(1 + nb + nf)); }
  H.offc_bxy = 0;
  if (H.coords == 1) { H.offc_bxy = off; off = align16(off + 16u * 8u * (uint32_t)nb); }   // BP coordinates, 8 interleaved replicas
  H.offc_dhq = 0;
  if (H.coords != 0) { H.offc_dhq = off; off = align16(off + 8u * (uint32_t)nf); }
  H.offc_sh   = off; off = align16(off + 8u * (uint32_t)nf);
  H.offc_suinit = off; off = align16(off + 4u * (((uint32_t)nsu + 3u) / 4u));
  H.offc_cs   = off; off = align16(off + 4u * (uint32_t)nsu);
  H.offc_rcp  = off; off = align16(off + 8u * (uint32_t)n_rcp);
  H.offc_unit = off; off = align16(off + (uint32_t)nsu);
  H.offc_rank = off; off = align16(off + (uint32_t)nsu);
  H.offc_rq   = off; off = align16(off + 4u * (uint32_t)nhu);
  H.offc_hrs  = off; off = align16(off + 4u * (uint32_t)nhu);
  H.offc_hunit = off; off = align16(off + (uint32_t)nhu);
  H.offc_hrank = off; off = align16(off + (uint32_t)nhu);
  H.imagec_bytes = off;

  I->image_c.assign(H.imagec_bytes, 0);
  uint8_t *imc = I->image_c.data();
  if (H.coords == 0) {
    // strict lower triangle over {HQ = 0, field f = f + 1}: entry (hi, lo) at hi(hi-1)/2 + lo
    double *tri = reinterpret_cast<double *>(imc + H.offc_dtri);
    for (int hi = 1; hi <= nf; ++hi)
      for (int lo = 0; lo < hi; ++lo) {
        const double ax = d->field_x[hi - 1], ay = d->field_y[hi - 1];
        const double bx = lo ? d->field_x[lo - 1] : d->hq_x, by = lo ? d->field_y[lo - 1] : d->hq_y;
        tri[(size_t)hi * (hi - 1) / 2 + lo] = edge(ax, ay, bx, by);
      }
  }
  if (H.coords != 1) {
    double *dfc = reinterpret_cast<double *>(imc + H.offc_dfb);
    for (int f = 0; f < nf; ++f)
      for (int b = 0; b < nb; ++b)
        dfc[(size_t)f * nb + b] = edge(d->field_x[f], d->field_y[f], d->bp_x[b], d->bp_y[b]);
  }
  std::vector<double> xyv(2 * (size_t)(1 + nb + nf));
  xyv[0] = d->hq_x; xyv[1] = d->hq_y;
  for (int b = 0; b < nb; ++b) { xyv[2 * (1 + b)] = d->bp_x[b]; xyv[2 * (1 + b) + 1] = d->bp_y[b]; }
  for (int f = 0; f < nf; ++f) { xyv[2 * (1 + nb + f)] = d->field_x[f]; xyv[2 * (1 + nb + f) + 1] = d->field_y[f]; }
  if (H.coords != 0) {
    std::memcpy(imc + H.offc_xy, xyv.data(), xyv.size() * 8);
    if (H.coords == 1) {
      // replica r of BP b at entry 8 b + r: lane l of a warp reads replica l & 7, so the eight lanes of a quarter-warp
      // (one wavefront of a 16-byte load) always hit eight different groups of four banks, whatever BPs they hold
      double *bx = reinterpret_cast<double *>(imc + H.offc_bxy);
      for (int b = 0; b < nb; ++b)
        for (int r = 0; r < 8; ++r) { bx[2 * (8 * b + r)] = d->bp_x[b]; bx[2 * (8 * b + r) + 1] = d->bp_y[b]; }
    }
    double *dh = reinterpret_cast<double *>(imc + H.offc_dhq);
    for (int f = 0; f < nf; ++f) dh[f] = edge(d->field_x[f], d->field_y[f], d->hq_x, d->hq_y);
  }
  uint32_t *shc = reinterpret_cast<uint32_t *>(imc + H.offc_sh);
  for (int f = 0; f < nf; ++f) { shc[2 * f] = (uint32_t)s_q[f]; shc[2 * f + 1] = (uint32_t)h_q[f]; }
  uint32_t *rq = reinterpret_cast<uint32_t *>(imc + H.offc_rq);
  for (int u = 0; u < nhu; ++u) rq[u] = (uint32_t)r_q[u];
  // SUs ascending by (capacity quanta, unit index): "rising fill times" (R16, R17)
  std::vector<int> order(nsu);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return c_q[a] < c_q[b]; });
  uint32_t *cc = reinterpret_cast<uint32_t *>(imc + H.offc_cs);
  for (int r = 0; r < nsu; ++r) {
    cc[r] = (uint32_t)c_q[order[r]];
    imc[H.offc_unit + r] = (uint8_t)order[r]; imc[H.offc_rank + order[r]] = (uint8_t)r;
  }
  {   // initial Fisher-Yates array of the SU partition: element i (byte i + pad of the right-aligned words) = rank of unit i
    const uint32_t padu = (4u - ((uint32_t)nsu & 3u)) & 3u;
    for (int u = 0; u < nsu; ++u) imc[H.offc_suinit + (uint32_t)u + padu] = imc[H.offc_rank + u];
  }
  {   // HUs ascending by (rate quanta, unit index): "sorted according to rising in-field working rates"
    std::vector<int> ho(nhu);
    std::iota(ho.begin(), ho.end(), 0);
    std::stable_sort(ho.begin(), ho.end(), [&](int a, int b) { return r_q[a] < r_q[b]; });
    uint32_t *hrs = reinterpret_cast<uint32_t *>(imc + H.offc_hrs);
    for (int r = 0; r < nhu; ++r) { hrs[r] = (uint32_t)r_q[ho[r]]; imc[H.offc_hunit + r] = (uint8_t)ho[r]; imc[H.offc_hrank + ho[r]] = (uint8_t)r; }
  }
  double *rcp = reinterpret_cast<double *>(imc + H.offc_rcp);
  rcp[0] = 0.0;
  for (int k = 1; k < n_rcp; ++k) rcp[k] = 1.0 / (double)k;          // correctly rounded reciprocals

  // ---- device: launch configuration and upload
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev < 1) { delete I; return cuda_fail(e != cudaSuccess ? e : cudaErrorNoDevice, "cudaGetDeviceCount"); }
  if ((e = cudaGetDevice(&I->device)) != cudaSuccess) { delete I; return cuda_fail(e, "cudaGetDevice"); }
  int smem_optin = 0;
  cudaDeviceGetAttribute(&I->sm_count, cudaDevAttrMultiProcessorCount, I->device);
  cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, I->device);
  I->smem_budget = std::min<int64_t>(smem_optin, kMaxSmem) - 1024;   // static smem of the reduction
  const int64_t budget = I->smem_budget;
  // s_q replication of image A: as many replicas (<= 32, a power of two) as 16 KB hold
  uint32_t sq_shift = 0;
  while (sq_shift < 5u && 4ull * ((uint64_t)nf << (sq_shift + 1u)) <= 16ull * 1024) ++sq_shift;
  int rc = build_image_a(I, sq_shift);
  if (rc != LGX_OK) { free_instance(I); return rc; }
  config_decode_cut(I);
  I->threads_b     = (int)fit_threads(budget, H.imagec_bytes, (int64_t)I->b_state, H.coords == 0 ? kMaxThreadsB : kMaxThreadsBC);
  if (I->threads_a < 32 || I->threads_a_dec < 32 || I->threads_b < 32) { free_instance(I); return LGX_ETOOBIG; }
  I->grid = I->sm_count;                       // one persistent block per SM
  // block-synchronous work fetch of lgx_walk_finish: measured -6 % (Large) and -10 % (Sweep) kernel time with coordinates, where warps
  // in different phases evict each other's code; +3.6 % with the tables (Medium) and +1.7 % on paper_scale, whose warps spend
  // all their time in the same two loops anyway
  I->walk_lockstep = (H.coords != 0 && nf < 1024) ? 1 : 0;
  // candidates per kernel pair: the queue holds a whole chunk (every candidate may pass eq. (2)); <= 2 GiB, <= 2^24
  // (measured: Medium gains 1.4 % from 2^22 -> 2^24, Toy 7 %; the big-record configs are flat between 2^18 and 2^21)
  {
    uint64_t cap = (2048ull << 20) / (4ull * H.rec_words);
    cap = std::min<uint64_t>(cap, 1ull << 24);
    I->chunk = std::max<uint64_t>(cap / 1024, 1) * 1024;
  }
  if ((e = cudaMalloc((void **)&I->d_image_c, H.imagec_bytes)) != cudaSuccess) { free_instance(I); return cuda_fail(e, "cudaMalloc(image C)"); }
  if ((e = cudaMemcpy(I->d_image_c, imc, H.imagec_bytes, cudaMemcpyHostToDevice)) != cudaSuccess) { free_instance(I); return cuda_fail(e, "cudaMemcpy(image C)"); }
  // workspaces come from the library's per-device pool, which keeps its memory between calls and between instances
  if ((rc = device_pool(I->device, &I->pool)) != LGX_OK) { I->pool = nullptr; free_instance(I); return rc; }
  {
    KernelFn ka, kb;
    pick_kernels<MODE_EVAL>(H, ka, kb);
    if (!kb) { free_instance(I); return LGX_EINVAL; }
    rc = allow_max_smem((const void *)ka, smem_optin); if (rc == LGX_OK) rc = allow_max_smem((const void *)kb, smem_optin);
    pick_kernels<MODE_SEARCH>(H, ka, kb);
    if (rc == LGX_OK) rc = allow_max_smem((const void *)ka, smem_optin); if (rc == LGX_OK) rc = allow_max_smem((const void *)kb, smem_optin);
    pick_kernels<MODE_DECODE>(H, ka, kb);
    if (rc == LGX_OK) rc = allow_max_smem((const void *)ka, smem_optin); if (rc == LGX_OK) rc = allow_max_smem((const void *)kb, smem_optin);
    if (rc != LGX_OK) { free_instance(I); return rc; }
  }
  // ---- move kernels: shared-memory layout (lgx_moves.cuh) and vertex coordinates for lgx_init_plan
  {
    MvHdr &M = I->mv;
    uint32_t o = 0;
    M.off_xy = o;    o = align16(o + 16u * (uint32_t)(1 + nb + nf));
    M.off_dq = o;    o = align16(o + 4u * (uint32_t)nb);
    M.off_c = o;     o = align16(o + (H.imagec_bytes - H.offc_cs));
    M.off_pfb = o;   o = align16(o + 4u * (uint32_t)nf);
    M.off_psq = o;   o = align16(o + 4u * (uint32_t)nf);
    M.off_phq = o;   o = align16(o + 4u * (uint32_t)nf);
    M.off_term = o;  o = align16(o + 8u * (uint32_t)nf);
    M.off_legx = o;  o = align16(o + 8u * (uint32_t)nf);
    M.off_legy = o;  o = align16(o + 8u * (uint32_t)nf);
    M.off_prex = o;  o = align16(o + 8u * (uint32_t)nf);
    M.off_prey = o;  o = align16(o + 8u * (uint32_t)nf);
    M.off_posf = o;  o = align16(o + 2u * (uint32_t)nf);
    M.off_bp = o;    o = align16(o + 8u * (uint32_t)nb);
    M.off_bsh = o;   o = align16(o + 8u * (uint32_t)nb);
    M.off_bpq = o;   o = align16(o + 8u * (uint32_t)nb);
    M.off_pre = o;   o = align16(o + 2u * ((uint32_t)nb + 1u));
    M.off_bpat = o;  o = align16(o + (uint32_t)nb);
    M.off_cnt = o;   o = align16(o + 4u * (uint32_t)nb);
    M.off_tpl = o;   o = align16(o + 4u * (uint32_t)nt);
    M.off_thu = o;   o = align16(o + 8u * (uint32_t)nt);
    M.off_thm = o;   o = align16(o + 8u * (uint32_t)nt);
    M.off_tsn = o;   o = align16(o + 8u * (uint32_t)nt);
    M.off_tmask = o; o = align16(o + 8u * (uint32_t)nt * MW);
    M.off_trng = o;  o = align16(o + 8u * (uint32_t)nt);
    M.off_tst = o;   o = align16(o + 56u * (uint32_t)nt);
    M.off_thq = o;   o = align16(o + 4u * (uint32_t)nt);
    M.off_sv = o;    o = align16(o + 16u * (uint32_t)nt * (uint32_t)nsu);
    M.off_misc = o;  o = align16(o + 64u);
    M.off_sort = o;  o = align16(o + 4u * (kSortKeys + 2u));
    M.off_order = o; o = align16(o + 2u * kSuper * (uint32_t)kMvThreads);
    uint32_t q = 0;
    q += (uint32_t)nb; M.pl_bpos = q; q += (uint32_t)nb; q = (q + 1u) & ~1u;
    M.pl_fbp = q; q += 2u * (uint32_t)nf; M.pl_fpos = q; q += 2u * (uint32_t)nf; q = (q + 7u) & ~7u;
    M.pl_mask = q; q += 8u * (uint32_t)nt * MW;
    M.pl_hmask = q; q += 8u * (uint32_t)nt;
    M.plan_bytes = align16(q);
    M.off_plans = o; o += 3u * M.plan_bytes;
    M.off_state = o;
    uint32_t r = 0;
    M.m64_w = r; r += (uint32_t)nt;
    M.m64_mask = r; r += (uint32_t)nt * MW; M.m64_bmask = r; r += (uint32_t)nt * MW;
    const bool hb = (H.flags & LGX_FLAG_HU_BALANCE) != 0u;
    if (hb) { M.m64_t = r; r += (uint32_t)nt; M.m64_hmask = r; r += (uint32_t)nt; M.m64_bhmask = r; r += (uint32_t)nt; }
    M.m64_rows = r;
    r = 0;
    M.m32_s = r; r += (uint32_t)nt;
    if (hb) { M.m32_r = r; r += (uint32_t)nt; }
    M.m32_rows = r;
    M.slot_words = 3u + (uint32_t)nt * MW + (uint32_t)nt;
    I->mv_state = 8ll * M.m64_rows + 4ll * M.m32_rows;
    int64_t tm = (budget - 256 - (int64_t)M.off_state) / I->mv_state;      // static smem of the reductions
    tm = std::min<int64_t>(tm, kMvThreads) / 32 * 32;
    if (nt > LGX_MAX_MOVE_TOURS || nhu > LGX_MAX_MOVE_HUS) tm = 0;        // 64-bit sets of tours and of HUs
    I->max_threads_mv = tm >= 64 ? (int)tm : 0;                           // 0: the move kernels do not fit (LGX_ETOOBIG there)
    I->threads_mv = I->max_threads_mv;
    I->smem_mv = (size_t)M.off_state + (size_t)I->mv_state * (size_t)I->threads_mv;
    if ((e = cudaMalloc((void **)&I->d_xy, xyv.size() * 8)) != cudaSuccess ||
        (e = cudaMemcpy(I->d_xy, xyv.data(), xyv.size() * 8, cudaMemcpyHostToDevice)) != cudaSuccess) {
      free_instance(I); return cuda_fail(e, "cudaMalloc/cudaMemcpy(xy)");
    }
    if (I->threads_mv) {
      MvKernelFn kb2, ks2; pick_move_kernels(H, kb2, ks2);
      rc = allow_max_smem((const void *)kb2, smem_optin); if (rc == LGX_OK) rc = allow_max_smem((const void *)ks2, smem_optin);
      if (rc != LGX_OK) { free_instance(I); return rc; }
    }
  }
  *out = I;
  return LGX_OK;
}

int lgx_instance_destroy(lgx_instance *I)
{
  if (!I) return LGX_EINVAL;
  free_instance(I);
  return LGX_OK;
}

int lgx_workspace_trim(void)
{
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  for (int dev = 0; dev < kMaxDevices; ++dev)
    if (g_pools[dev]) CU(cudaMemPoolTrimTo(g_pools[dev], 0));
  return LGX_OK;
}

int lgx_instance_set_option(lgx_instance *I, int key, int64_t value)
{
  if (!I) return LGX_EINVAL;
  const ImgHdr &H = I->hdr;
  const int64_t budget = I->smem_budget;
  auto threads_ok = [](int64_t v, int64_t lo, int64_t hi) { return v >= lo && v <= hi && v % 32 == 0; };
  switch (key) {
    case LGX_OPT_THREADS_A: {
      const int64_t hi = fit_threads(budget, H.image_bytes, (int64_t)I->a_state, H.perm16 ? kMaxThreadsA16 : kMaxThreadsA);
      if (!threads_ok(value, 32, hi)) return LGX_EINVAL;
      I->threads_a = (int)value; I->threads_a_dec = (int)std::min<int64_t>(value, fit_threads(budget, H.image_bytes, (int64_t)I->a_state_dec, H.perm16 ? kMaxThreadsA16 : kMaxThreadsA));
      return LGX_OK;
    }
    case LGX_OPT_THREADS_B: {
      const int64_t hi = fit_threads(budget, H.imagec_bytes, (int64_t)I->b_state, H.coords == 0 ? kMaxThreadsB : kMaxThreadsBC);
      if (!threads_ok(value, 32, hi)) return LGX_EINVAL;
      I->threads_b = (int)value;
      return LGX_OK;
    }
    case LGX_OPT_THREADS_MV: {
      if (!threads_ok(value, 64, I->max_threads_mv)) return LGX_EINVAL;
      I->threads_mv = (int)value;
      I->smem_mv = (size_t)I->mv.off_state + (size_t)I->mv_state * (size_t)I->threads_mv;
      return LGX_OK;
    }
    case LGX_OPT_CHUNK_LOG2: {
      if (value < 10 || value > 26) return LGX_EINVAL;
      I->chunk = 1ull << value;
      return LGX_OK;
    }
    case LGX_OPT_WALK_LOCKSTEP: {
      if (value != 0 && value != 1) return LGX_EINVAL;
      I->walk_lockstep = (int)value;
      return LGX_OK;
    }
    case LGX_OPT_SQ_SHIFT: {
      if (value < 0 || value > 5) return LGX_EINVAL;
      const int64_t img = 16 + 4ll * ((int64_t)H.n_f << value) + 16 + 4ll * H.n_b;
      if (fit_threads(budget, img, (int64_t)I->a_state_dec, H.perm16 ? kMaxThreadsA16 : kMaxThreadsA) < 32) return LGX_ETOOBIG;
      int rc = check_device(I);
      if (rc != LGX_OK) return rc;
      CU(cudaDeviceSynchronize());                       // no kernel may still be reading the image that is replaced
      rc = build_image_a(I, (uint32_t)value);            // on failure the instance keeps its previous image and configuration
      if (rc != LGX_OK) return rc;
      config_decode_cut(I);                              // create-time defaults for the new image size
      return LGX_OK;
    }
    default: return LGX_EINVAL;
  }
}

}  // extern "C"

namespace {

// One call = chunks of at most I->chunk candidates; per chunk the decode/cut kernel fills the
// queue and the walk/finish kernel drains it (same stream, so the pair is ordered).  The workspace
// is allocated stream-ordered per call, so concurrent calls on different streams are legal.
struct Workspace {
  uint8_t *base = nullptr;
  unsigned int *q_count = nullptr, *done = nullptr, *ctr_a = nullptr, *ctr_b = nullptr;
  unsigned long long *result = nullptr, *block_best = nullptr;
  uint32_t *queue = nullptr;
  uint64_t cap = 0;
};

int ws_alloc(const lgx_instance *I, uint64_t n, bool search, cudaStream_t st, Workspace &W)
{
  W.cap = std::min<uint64_t>(I->chunk, (n + 31) / 32 * 32);
  const size_t head = 64 + 16ull * (size_t)I->grid;
  const size_t qoff = (head + 255) & ~(size_t)255;
  const size_t bytes = qoff + 4ull * I->hdr.rec_words * W.cap;
  CU(cudaMallocFromPoolAsync((void **)&W.base, bytes, I->pool, st));
  W.q_count = reinterpret_cast<unsigned int *>(W.base);
  W.done = W.q_count + 1; W.ctr_a = W.q_count + 2; W.ctr_b = W.q_count + 3;
  W.result = reinterpret_cast<unsigned long long *>(W.base + 16);
  W.block_best = reinterpret_cast<unsigned long long *>(W.base + 64);
  W.queue = reinterpret_cast<uint32_t *>(W.base + qoff);
  cudaError_t e = cudaMemsetAsync(W.base, 0, 16, st);
  if (e == cudaSuccess && search) e = cudaMemsetAsync(W.result, 0xFF, 16, st);
  if (e != cudaSuccess) { cudaFreeAsync(W.base, st); W.base = nullptr; return cuda_fail(e, "cudaMemsetAsync(workspace)"); }
  return LGX_OK;
}

int run_chunks(const lgx_instance *I, KernelFn ka, KernelFn kb, KParams &P, uint64_t n, const Workspace &W, cudaStream_t st,
               bool decode_mode, std::vector<cudaEvent_t> *evs = nullptr)
{
  if (!ka || !kb) return LGX_EINVAL;
  const uint64_t ta = LGX_BLOCK_THREADS((uint64_t)(decode_mode ? I->threads_a_dec : I->threads_a));
  const uint64_t tb = LGX_BLOCK_THREADS((uint64_t)I->threads_b);
  const uint64_t cand_a = ta;                                            // candidates a block of kernel 1 holds
  const size_t smem_a = (size_t)I->hdr.image_bytes + (size_t)(decode_mode ? I->a_state_dec : I->a_state) * ta;
  const size_t smem_b = (size_t)I->hdr.imagec_bytes + (size_t)I->b_state * tb;
  P.H = I->hdr; P.image = I->d_image; P.image_c = I->d_image_c;
  P.queue = W.queue; P.cap = (uint32_t)W.cap; P.q_count = W.q_count; P.ctr_a = W.ctr_a; P.ctr_b = W.ctr_b;
  P.done_counter = W.done; P.block_best = W.block_best; P.result = W.result;
  P.lockstep = I->walk_lockstep ? 1u : 0u;
  void *args[] = { (void *)&P };
  for (uint64_t base = 0; base < n; base += W.cap) {
    P.base_i = base; P.n = std::min<uint64_t>(W.cap, n - base);
    const unsigned grid_a = (unsigned)std::min<uint64_t>((uint64_t)I->grid, (P.n + cand_a - 1) / cand_a);
    const unsigned grid_b = (unsigned)std::min<uint64_t>((uint64_t)I->grid, (P.n + tb - 1) / tb);
    cudaEvent_t e3[3] = {nullptr, nullptr, nullptr};
    if (evs) { for (auto &e : e3) { CU(cudaEventCreate(&e)); evs->push_back(e); } CU(cudaEventRecord(e3[0], st)); }
    CU(cudaLaunchKernel((const void *)ka, dim3(grid_a), dim3((unsigned)ta), args, smem_a, st));
    if (evs) CU(cudaEventRecord(e3[1], st));
    CU(cudaLaunchKernel((const void *)kb, dim3(grid_b), dim3((unsigned)tb), args, smem_b, st));
    if (evs) CU(cudaEventRecord(e3[2], st));
    I->launches.fetch_add(2);
  }
  return LGX_OK;
}

}  // namespace

extern "C" {

int lgx_instance_query(const lgx_instance *I, int what, int64_t *out)
{
  if (!I || !out) return LGX_EINVAL;
  switch (what) {
    case 0: *out = (int64_t)I->hdr.image_bytes + I->hdr.imagec_bytes; break;
    case 1: *out = I->threads_a; break;
    case 2: *out = I->grid; break;
    case 3: *out = (int64_t)I->hdr.image_bytes + (int64_t)I->a_state * I->threads_a; break;
    case 4: *out = I->hdr.coords; break;
    case 5: *out = (int64_t)I->a_state; break;
    case 6: *out = I->sm_count; break;
    case 7: *out = I->launches.load(); break;
    case 8: *out = I->threads_b; break;
    case 9: *out = (int64_t)I->hdr.imagec_bytes + (int64_t)I->b_state * I->threads_b; break;
    case 10: *out = (int64_t)I->chunk; break;
    case 11: *out = 4ll * I->hdr.rec_words; break;
    case 12: *out = I->ns_a.load(); break;
    case 13: *out = I->ns_c.load(); break;
    case 14: *out = I->timed_pairs.load(); break;
    case 15: *out = I->threads_mv; break;
    case 16: *out = (int64_t)I->smem_mv; break;
    case 17: *out = I->hdr.sq_shift; break;
    case 18: *out = I->threads_a_dec; break;
    case 19: *out = (int64_t)I->b_state; break;
    case 20: *out = I->device; break;
    case 24: *out = I->walk_lockstep; break;
    default: return LGX_EINVAL;
  }
  return LGX_OK;
}

int lgx_selftest(int what, uint64_t n, uint64_t seed, uint64_t *h_out)
{
  if (!h_out || n == 0) return LGX_EINVAL;
#ifndef LGX_EMU
  if (what >= 1 && what <= 5) {                          // pipe microbenchmarks (lgx_pipes.cu); n = loop iterations
    const int e = pipe_bench(what, n, h_out);
    return e == 0 ? LGX_OK : cuda_fail((cudaError_t)e, "lgx_selftest: pipe microbenchmark");
  }
#endif
  if (what != 0) return LGX_EINVAL;
  unsigned long long *d = nullptr;
  CU(cudaMalloc((void **)&d, 16));
  cudaError_t e = cudaMemset(d, 0, 16);
  if (e == cudaSuccess) {
    void *args[] = { (void *)&n, (void *)&seed, (void *)&d };
    e = cudaLaunchKernel(selftest_sqrt_kernel(), dim3(592), dim3(256), args, 0, nullptr);
  }
  unsigned long long r[2] = {0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(r, d, 16, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(e, "lgx_selftest");
  h_out[0] = r[0]; h_out[1] = r[1];
  return LGX_OK;
}

int lgx_instance_set_timing(lgx_instance *I, int enable)
{
  if (!I) return LGX_EINVAL;
  I->timing.store(enable ? 1 : 0);
  I->ns_a.store(0); I->ns_c.store(0); I->timed_pairs.store(0);
  return LGX_OK;
}

int lgx_eval_batch(const lgx_instance *I, uint64_t seed, const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                   double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible, void *stream)
{
  if (!I) return LGX_EINVAL;
  if (n == 0) return LGX_OK;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  KParams P{};
  fill_round_keys(P, seed);
  P.ids = d_ids; P.first_id = first_id;
  P.cost = d_cost; P.path_km = d_path_km; P.makespan_h = d_makespan_h; P.feasible = d_feasible;
  KernelFn ka, kb; pick_kernels<MODE_EVAL>(I->hdr, ka, kb);
  Workspace W;
  rc = ws_alloc(I, n, false, st, W);
  if (rc != LGX_OK) return rc;
  rc = run_chunks(I, ka, kb, P, n, W, st, false);
  cudaFreeAsync(W.base, st);
  return rc;
}

int lgx_decode_batch(const lgx_instance *I, uint64_t seed, const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                     uint8_t *d_bp_tour, uint8_t *d_bp_pos, uint16_t *d_field_bp, uint16_t *d_field_pos,
                     uint8_t *d_hu_tour, uint8_t *d_su_tour_init, uint8_t *d_su_tour_final, void *stream)
{
  if (!I) return LGX_EINVAL;
  if (n == 0) return LGX_OK;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  KParams P{};
  fill_round_keys(P, seed);
  P.ids = d_ids; P.first_id = first_id;
  P.bp_tour = d_bp_tour; P.bp_pos = d_bp_pos; P.field_bp = d_field_bp; P.field_pos = d_field_pos;
  P.hu_tour = d_hu_tour; P.su_init = d_su_tour_init; P.su_final = d_su_tour_final;
  KernelFn ka, kb; pick_kernels<MODE_DECODE>(I->hdr, ka, kb);
  Workspace W;
  rc = ws_alloc(I, n, false, st, W);
  if (rc != LGX_OK) return rc;
  rc = run_chunks(I, ka, kb, P, n, W, st, true);
  cudaFreeAsync(W.base, st);
  return rc;
}

int lgx_search_range(const lgx_instance *I, uint64_t seed, uint64_t first_id, uint64_t n,
                     double *h_best_cost, uint64_t *h_best_id, void *stream)
{
  if (!I || !h_best_cost || !h_best_id || n == 0) return LGX_EINVAL;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  KParams P{};
  fill_round_keys(P, seed);
  P.ids = nullptr; P.first_id = first_id;
  KernelFn ka, kb; pick_kernels<MODE_SEARCH>(I->hdr, ka, kb);
  Workspace W;
  rc = ws_alloc(I, n, true, st, W);
  if (rc != LGX_OK) return rc;
  std::vector<cudaEvent_t> evs;
  const bool timed = I->timing.load() != 0;
  rc = run_chunks(I, ka, kb, P, n, W, st, false, timed ? &evs : nullptr);
  unsigned long long res[2] = {0, 0};
  if (rc == LGX_OK) {
    cudaError_t e = cudaMemcpyAsync(res, W.result, sizeof res, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = cuda_fail(e, "lgx_search: copy/synchronize");
  }
  if (rc == LGX_OK) {
    for (size_t k = 0; k + 3 <= evs.size(); k += 3) {
      float ma = 0.f, mc = 0.f;
      if (cudaEventElapsedTime(&ma, evs[k], evs[k + 1]) == cudaSuccess &&
          cudaEventElapsedTime(&mc, evs[k + 1], evs[k + 2]) == cudaSuccess) {
        I->ns_a.fetch_add((long long)(ma * 1e6)); I->ns_c.fetch_add((long long)(mc * 1e6)); I->timed_pairs.fetch_add(1);
      }
    }
  }
  for (cudaEvent_t e : evs) cudaEventDestroy(e);
  cudaFreeAsync(W.base, st);
  if (rc != LGX_OK) return rc;
  if (res[0] == ~0ull && res[1] == ~0ull) {          // no feasible candidate: +inf, lowest id (R19, R29)
    res[0] = 0x7FF0000000000000ull; res[1] = first_id;
  }
  std::memcpy(h_best_cost, &res[0], 8);
  *h_best_id = res[1];
  return LGX_OK;
}

int lgx_search(const lgx_instance *I, uint64_t seed, uint64_t budget, double *h_best_cost, uint64_t *h_best_id, void *stream)
{
  return lgx_search_range(I, seed, 0, budget, h_best_cost, h_best_id, stream);
}

int lgx_eval_batch_host(const lgx_instance *I, uint64_t seed, const uint64_t *h_ids, uint64_t first_id, uint64_t n,
                        double *h_cost, double *h_path_km, double *h_makespan_h, uint8_t *h_feasible)
{
  if (!I) return LGX_EINVAL;
  if (n == 0) return LGX_OK;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  // Chunks of 2^21 candidates alternate between two streams, each with its own device buffers (from the cached pool):
  // with page-locked host buffers the copies of one chunk overlap the kernels of the next; with pageable buffers the
  // driver stages every copy and the chunks simply run one after the other.
  const uint64_t chunk = std::min<uint64_t>(n, 1ull << 21);
  cudaStream_t st[2] = {nullptr, nullptr};
  uint8_t *buf[2] = {nullptr, nullptr};
  const size_t o_c = 0, o_p = 8 * chunk, o_m = 16 * chunk, o_i = 24 * chunk, o_f = 32 * chunk, bytes = 33 * chunk + 256;
  cudaError_t e = cudaSuccess;
  auto cleanup = [&]() {
    for (int k = 0; k < 2; ++k) {
      if (buf[k]) cudaFreeAsync(buf[k], st[k]);
      if (st[k]) { cudaStreamSynchronize(st[k]); cudaStreamDestroy(st[k]); }
    }
  };
  for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
    e = cudaStreamCreateWithFlags(&st[k], cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaMallocFromPoolAsync((void **)&buf[k], bytes, I->pool, st[k]);
  }
  if (e != cudaSuccess) { cleanup(); return cuda_fail(e, "lgx_eval_batch_host: streams / buffers"); }
  uint64_t k = 0;
  for (uint64_t o = 0; o < n && rc == LGX_OK; o += chunk, ++k) {
    const uint64_t m = std::min<uint64_t>(chunk, n - o);
    cudaStream_t s = st[k & 1]; uint8_t *b = buf[k & 1];
    uint64_t *d_ids = reinterpret_cast<uint64_t *>(b + o_i);
    double *d_c = h_cost ? reinterpret_cast<double *>(b + o_c) : nullptr, *d_p = h_path_km ? reinterpret_cast<double *>(b + o_p) : nullptr;
    double *d_m = h_makespan_h ? reinterpret_cast<double *>(b + o_m) : nullptr; uint8_t *d_f = h_feasible ? b + o_f : nullptr;
    if (h_ids && (e = cudaMemcpyAsync(d_ids, h_ids + o, m * 8, cudaMemcpyHostToDevice, s)) != cudaSuccess) { rc = cuda_fail(e, "H2D ids"); break; }
    rc = lgx_eval_batch(I, seed, h_ids ? d_ids : nullptr, first_id + o, m, d_c, d_p, d_m, d_f, (void *)s);
    if (rc != LGX_OK) break;
    if (h_cost && (e = cudaMemcpyAsync(h_cost + o, d_c, m * 8, cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = cuda_fail(e, "D2H"); break; }
    if (h_path_km && (e = cudaMemcpyAsync(h_path_km + o, d_p, m * 8, cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = cuda_fail(e, "D2H"); break; }
    if (h_makespan_h && (e = cudaMemcpyAsync(h_makespan_h + o, d_m, m * 8, cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = cuda_fail(e, "D2H"); break; }
    if (h_feasible && (e = cudaMemcpyAsync(h_feasible + o, d_f, m, cudaMemcpyDeviceToHost, s)) != cudaSuccess) { rc = cuda_fail(e, "D2H"); break; }
  }
  for (int j = 0; j < 2; ++j)
    if ((e = cudaStreamSynchronize(st[j])) != cudaSuccess && rc == LGX_OK) rc = cuda_fail(e, "cudaStreamSynchronize");
  cleanup();
  return rc;
}

}  // extern "C"

// ================================================================== lgx_eval_batch_static: no allocation at call time
#ifndef LGX_EMU

namespace {

// The queue of feasible candidates and the kernels' counters for lgx_eval_batch_static.  It is part of the library's
// device image: the driver places it when the module is loaded on a GPU and it stays there until the process exits, so
// the entry point below never has to ask an allocator for memory.  One array per device, shared by every call: it keeps
// whatever the last call left in it.
static __device__ __align__(256) unsigned char g_static_scratch[LGX_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is only a handle for the runtime, not memory a kernel can use; the address the kernels
// get is looked up once per device, with that device current, and cached here.
std::mutex g_static_mutex;
unsigned char *g_static_ptr[kMaxDevices] = {};

int static_scratch(int device, unsigned char **out)
{
  if (device < 0 || device >= kMaxDevices) return LGX_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[device]) {
    unsigned char *p = nullptr;
    CU(cudaGetSymbolAddress((void **)&p, g_static_scratch));      // check_device() made `device` the current one
    if (!p) { g_cuda_msg = "cudaGetSymbolAddress returned a null address for the static scratch"; return LGX_ECUDA; }
    g_static_ptr[device] = p;
  }
  *out = g_static_ptr[device];
  return LGX_OK;
}

// Candidates one call can take: the array holds the counters, one 16-byte slot per block and one queue record each.
uint64_t static_capacity(const lgx_instance *I, size_t *qoff_out)
{
  const size_t head = 64 + 16ull * (size_t)I->grid;
  const size_t qoff = (head + 255) & ~(size_t)255;
  if (qoff_out) *qoff_out = qoff;
  if (qoff >= (size_t)LGX_STATIC_SCRATCH_BYTES) return 0;
  return ((size_t)LGX_STATIC_SCRATCH_BYTES - qoff) / (4ull * I->hdr.rec_words) / 32 * 32;
}

}  // namespace

extern "C" {

int lgx_eval_batch_static_max(const lgx_instance *I, uint64_t *max_n)
{
  if (!I || !max_n) return LGX_EINVAL;
  *max_n = static_capacity(I, nullptr);
  return LGX_OK;
}

int lgx_eval_batch_static(const lgx_instance *I, uint64_t seed, const uint64_t *d_ids, uint64_t first_id, uint64_t n,
                          double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible, void *stream)
{
  if (!I) return LGX_EINVAL;
  size_t qoff = 0;
  if (n > static_capacity(I, &qoff)) return LGX_ESTATIC;             // before anything is touched or launched
  if (n == 0) return LGX_OK;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  unsigned char *base = nullptr;
  rc = static_scratch(I->device, &base);                             // first call on this device: looks the address up
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  KParams P{};
  fill_round_keys(P, seed);
  P.ids = d_ids; P.first_id = first_id;
  P.cost = d_cost; P.path_km = d_path_km; P.makespan_h = d_makespan_h; P.feasible = d_feasible;
  KernelFn ka, kb; pick_kernels<MODE_EVAL>(I->hdr, ka, kb);
  Workspace W;                                                        // same layout as ws_alloc, inside the static array
  W.base = base;
  W.cap = (n + 31) / 32 * 32;                                         // one kernel pair takes the whole call
  W.q_count = reinterpret_cast<unsigned int *>(base);
  W.done = W.q_count + 1; W.ctr_a = W.q_count + 2; W.ctr_b = W.q_count + 3;
  W.result = reinterpret_cast<unsigned long long *>(base + 16);
  W.block_best = reinterpret_cast<unsigned long long *>(base + 64);
  W.queue = reinterpret_cast<uint32_t *>(base + qoff);
  // the array still holds the previous call's counters: the queue length and the work counters must start at zero
  CU(cudaMemsetAsync(base, 0, 64, st));
  return run_chunks(I, ka, kb, P, n, W, st, false);
}

}  // extern "C"

#endif  // LGX_EMU

// ================================================================== Algorithm 1

namespace {

void pick_move_kernels(const ImgHdr &h, MvKernelFn &kb, MvKernelFn &ks)
{
  if (h.mask_words == 1u) pick_move_kernels_mw1(h, kb, ks); else pick_move_kernels_mw2(h, kb, ks);
}

// A plan is valid when every BP sits on exactly one tour at a unique position 0..len-1, every field on exactly
// one BP likewise, and every tour has at least one HU and one SU (L69).
bool plan_valid(const ImgHdr &H, const uint8_t *bt, const uint8_t *bq, const uint16_t *fb, const uint16_t *fq,
                const uint8_t *hu, const uint8_t *su)
{
  const int nt = H.n_t, nb = H.n_b, nf = H.n_f;
  std::vector<int> tlen(nt, 0), blen(nb, 0), nhu(nt, 0), nsu(nt, 0);
  for (int b = 0; b < nb; ++b) { if (bt[b] >= nt) return false; ++tlen[bt[b]]; }
  for (int f = 0; f < nf; ++f) { if (fb[f] >= nb) return false; ++blen[fb[f]]; }
  std::vector<int> toff(nt + 1, 0), boff(nb + 1, 0);
  for (int g = 0; g < nt; ++g) toff[g + 1] = toff[g] + tlen[g];
  for (int b = 0; b < nb; ++b) boff[b + 1] = boff[b] + blen[b];
  std::vector<char> seen_b(nb, 0), seen_f(nf, 0);
  for (int b = 0; b < nb; ++b) { if (bq[b] >= tlen[bt[b]]) return false; char &c = seen_b[toff[bt[b]] + bq[b]]; if (c) return false; c = 1; }
  for (int f = 0; f < nf; ++f) { if (fq[f] >= blen[fb[f]]) return false; char &c = seen_f[boff[fb[f]] + fq[f]]; if (c) return false; c = 1; }
  for (int u = 0; u < H.n_hu; ++u) { if (hu[u] >= nt) return false; ++nhu[hu[u]]; }
  for (int u = 0; u < H.n_su; ++u) { if (su[u] >= nt) return false; ++nsu[su[u]]; }
  for (int g = 0; g < nt; ++g) if (nhu[g] < 1 || nsu[g] < 1) return false;
  return true;
}

struct PlanDev {
  uint8_t *base = nullptr;
  uint8_t *bt, *bq, *hu, *su; uint16_t *fb, *fq;
  size_t bytes = 0;
};

int plan_dev_alloc(const lgx_instance *I, cudaStream_t st, PlanDev &D)
{
  const ImgHdr &H = I->hdr;
  const size_t nb = H.n_b, nf = H.n_f, nhu = H.n_hu, nsu = H.n_su;
  size_t o = 0;
  const size_t o_fb = o; o += 2 * nf; const size_t o_fq = o; o += 2 * nf;
  const size_t o_bt = o; o += nb; const size_t o_bq = o; o += nb; const size_t o_hu = o; o += nhu; const size_t o_su = o; o += nsu;
  D.bytes = o;
  CU(cudaMallocFromPoolAsync((void **)&D.base, o, I->pool, st));        // the library's cached per-device pool
  D.fb = reinterpret_cast<uint16_t *>(D.base + o_fb); D.fq = reinterpret_cast<uint16_t *>(D.base + o_fq);
  D.bt = D.base + o_bt; D.bq = D.base + o_bq; D.hu = D.base + o_hu; D.su = D.base + o_su;
  return LGX_OK;
}

// The six host arrays are packed into ONE pageable buffer of the library's, in the device layout of plan_dev_alloc, and
// uploaded with one copy.  A copy from pageable memory has left its source when cudaMemcpyAsync returns (the driver stages
// it), so neither the caller's arrays (which may be page-locked: a direct copy from those would still be in flight after the
// return) nor the local buffer are read after this function.
int plan_upload(const ImgHdr &H, const PlanDev &D, const uint8_t *bt, const uint8_t *bq, const uint16_t *fb, const uint16_t *fq,
                const uint8_t *hu, const uint8_t *su, cudaStream_t st)
{
  std::vector<uint8_t> stage(D.bytes);
  uint8_t *s0 = stage.data();
  std::memcpy(s0 + ((uint8_t *)D.fb - D.base), fb, 2 * (size_t)H.n_f);
  std::memcpy(s0 + ((uint8_t *)D.fq - D.base), fq, 2 * (size_t)H.n_f);
  std::memcpy(s0 + (D.bt - D.base), bt, (size_t)H.n_b);
  std::memcpy(s0 + (D.bq - D.base), bq, (size_t)H.n_b);
  std::memcpy(s0 + (D.hu - D.base), hu, (size_t)H.n_hu);
  std::memcpy(s0 + (D.su - D.base), su, (size_t)H.n_su);
  CU(cudaMemcpyAsync(D.base, s0, D.bytes, cudaMemcpyHostToDevice, st));
  return LGX_OK;
}

int plan_download(const ImgHdr &H, const PlanDev &D, uint8_t *bt, uint8_t *bq, uint16_t *fb, uint16_t *fq, uint8_t *hu, uint8_t *su,
                  cudaStream_t st)
{
  CU(cudaMemcpyAsync(bt, D.bt, (size_t)H.n_b, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(bq, D.bq, (size_t)H.n_b, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(fb, D.fb, 2 * (size_t)H.n_f, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(fq, D.fq, 2 * (size_t)H.n_f, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(hu, D.hu, (size_t)H.n_hu, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(su, D.su, (size_t)H.n_su, cudaMemcpyDeviceToHost, st));
  return LGX_OK;
}

void mv_fill(const lgx_instance *I, MvParams &P, uint64_t seed, const PlanDev &D)
{
  P.H = I->hdr; P.M = I->mv; P.image = I->d_image; P.image_c = I->d_image_c; P.xy = I->d_xy;
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { P.rk[2 * r] = k0; P.rk[2 * r + 1] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
  P.bp_tour = D.bt; P.bp_pos = D.bq; P.field_bp = D.fb; P.field_pos = D.fq; P.hu_tour = D.hu; P.su_tour = D.su;
}

}  // namespace

extern "C" {

int lgx_init_plan(const lgx_instance *I, uint8_t *h_bp_tour, uint8_t *h_bp_pos, uint16_t *h_field_bp, uint16_t *h_field_pos,
                  uint8_t *h_hu_tour, uint8_t *h_su_tour, void *stream)
{
  if (!I || !h_bp_tour || !h_bp_pos || !h_field_bp || !h_field_pos || !h_hu_tour || !h_su_tour) return LGX_EINVAL;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const ImgHdr &H = I->hdr;
  PlanDev D;
  rc = plan_dev_alloc(I, st, D);
  if (rc != LGX_OK) return rc;
  const size_t nb = H.n_b, nf = H.n_f;
  const size_t scratch_bytes = 4 * (3 * nb + 1) + 2 * (nf + (nf & 1)) + 2 * nb + 16;
  uint32_t *scratch = nullptr;
  cudaError_t e = cudaMallocFromPoolAsync((void **)&scratch, scratch_bytes, I->pool, st);
  if (e != cudaSuccess) { cudaFreeAsync(D.base, st); return cuda_fail(e, "cudaMallocAsync(init scratch)"); }
  InitParams P{};
  P.n_f = H.n_f; P.n_b = H.n_b; P.n_t = H.n_t; P.n_hu = H.n_hu; P.n_su = H.n_su;
  P.xy = I->d_xy;
  P.sh = reinterpret_cast<const uint2 *>(I->d_image_c + H.offc_sh);
  P.dq = reinterpret_cast<const uint32_t *>(I->d_image + H.off_dq);
  P.unit_of = I->d_image_c + H.offc_unit;
  P.bp_tour = D.bt; P.bp_pos = D.bq; P.field_bp = D.fb; P.field_pos = D.fq; P.hu_tour = D.hu; P.su_tour = D.su;
  P.scratch = scratch;
  {
    void *args[] = { (void *)&P };
    e = cudaLaunchKernel(init_plan_kernel(), dim3(1), dim3(256), args, 0, st);
  }
  I->launches.fetch_add(1);
  if (e == cudaSuccess) rc = plan_download(H, D, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour, st);
  if (e == cudaSuccess && rc == LGX_OK) e = cudaStreamSynchronize(st);
  cudaFreeAsync(scratch, st); cudaFreeAsync(D.base, st);
  if (e != cudaSuccess) return cuda_fail(e, "lgx_init_plan");
  return rc;
}

int lgx_move_eval_batch(const lgx_instance *I,
                        const uint8_t *h_bp_tour, const uint8_t *h_bp_pos, const uint16_t *h_field_bp, const uint16_t *h_field_pos,
                        const uint8_t *h_hu_tour, const uint8_t *h_su_tour,
                        uint64_t seed, uint64_t first_id, uint64_t n,
                        double *d_cost, double *d_path_km, double *d_makespan_h, uint8_t *d_feasible, void *stream)
{
  if (!I || !h_bp_tour || !h_bp_pos || !h_field_bp || !h_field_pos || !h_hu_tour || !h_su_tour) return LGX_EINVAL;
  const ImgHdr &H = I->hdr;
  if (!plan_valid(H, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour)) return LGX_EINVAL;
  if (I->threads_mv < 64) return LGX_ETOOBIG;
  if (n == 0) return LGX_OK;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  MvKernelFn kb, ks; pick_move_kernels(H, kb, ks);
  if (!kb) return LGX_EINVAL;
  PlanDev D;
  rc = plan_dev_alloc(I, st, D);
  if (rc != LGX_OK) return rc;
  rc = plan_upload(H, D, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour, st);
  if (rc == LGX_OK) {
    MvParams P{};
    mv_fill(I, P, seed, D);
    P.first_id = first_id; P.n = n;
    P.cost = d_cost; P.path_km = d_path_km; P.makespan_h = d_makespan_h; P.feasible = d_feasible;
    cudaError_t e = cudaSuccess;
    {
      const uint64_t blocks = (n + (uint64_t)I->threads_mv - 1) / (uint64_t)I->threads_mv;
      const unsigned grid = (unsigned)std::min<uint64_t>((uint64_t)I->grid, blocks);
      void *args[] = { (void *)&P };
      e = cudaLaunchKernel((const void *)kb, dim3(grid), dim3((unsigned)I->threads_mv), args, I->smem_mv, st);
      I->launches.fetch_add(1);
    }
    if (e != cudaSuccess) rc = cuda_fail(e, "lgx_move_eval_batch: launch");
  }
  cudaFreeAsync(D.base, st);
  return rc;
}

int lgx_local_search(const lgx_instance *I,
                     uint8_t *h_bp_tour, uint8_t *h_bp_pos, uint16_t *h_field_bp, uint16_t *h_field_pos,
                     uint8_t *h_hu_tour, uint8_t *h_su_tour,
                     uint64_t seed, uint32_t n_iters, uint32_t n_workers, uint32_t eps_thresh,
                     double *h_best_cost, double *h_hist_cost, uint64_t *h_hist_id, void *stream)
{
  if (!I || !h_bp_tour || !h_bp_pos || !h_field_bp || !h_field_pos || !h_hu_tour || !h_su_tour || !h_best_cost) return LGX_EINVAL;
  if (n_workers == 0) return LGX_EINVAL;
  const ImgHdr &H = I->hdr;
  if (!plan_valid(H, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour)) return LGX_EINVAL;
  if (I->threads_mv < 64) return LGX_ETOOBIG;
  int rc = check_device(I);
  if (rc != LGX_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  MvKernelFn kb, ks; pick_move_kernels(H, kb, ks);
  if (!ks) return LGX_EINVAL;
  int coop = 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, I->device);
  if (!coop) { g_cuda_msg = "device does not support cooperative launches"; return LGX_ECUDA; }
  int per_sm = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void *)ks, I->threads_mv, I->smem_mv));
  if (per_sm < 1) return LGX_ETOOBIG;
  // one block per SM, fewer when the workers of an iteration do not fill them
  const uint64_t blocks = ((uint64_t)n_workers + (uint64_t)I->threads_mv - 1) / (uint64_t)I->threads_mv;
  const unsigned grid = (unsigned)std::min<uint64_t>((uint64_t)I->sm_count, blocks);
  PlanDev D;
  rc = plan_dev_alloc(I, st, D);
  if (rc != LGX_OK) return rc;
  uint8_t *ws = nullptr;
  const size_t slots_bytes = 2ull * grid * I->mv.slot_words * 8ull;
  const size_t hist_bytes = (size_t)n_iters * 8ull;
  const size_t ws_bytes = slots_bytes + 2 * hist_bytes + 16;
  cudaError_t e = cudaMallocFromPoolAsync((void **)&ws, ws_bytes, I->pool, st);
  if (e != cudaSuccess) { cudaFreeAsync(D.base, st); return cuda_fail(e, "cudaMallocAsync(search workspace)"); }
  rc = plan_upload(H, D, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour, st);
  double best = 0.0;
  if (rc == LGX_OK) {
    MvParams P{};
    mv_fill(I, P, seed, D);
    P.n_iters = n_iters; P.n_workers = n_workers; P.eps_thresh = eps_thresh;
    P.slots = reinterpret_cast<unsigned long long *>(ws);
    P.hist_cost = reinterpret_cast<double *>(ws + slots_bytes);
    P.hist_id = reinterpret_cast<unsigned long long *>(ws + slots_bytes + hist_bytes);
    P.best_cost = reinterpret_cast<double *>(ws + slots_bytes + 2 * hist_bytes);
    void *args[] = { (void *)&P };
    e = cudaLaunchCooperativeKernel((const void *)ks, dim3(grid), dim3((unsigned)I->threads_mv), args, I->smem_mv, st);
    I->launches.fetch_add(1);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&best, P.best_cost, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && h_hist_cost && n_iters) e = cudaMemcpyAsync(h_hist_cost, P.hist_cost, hist_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && h_hist_id && n_iters) e = cudaMemcpyAsync(h_hist_id, P.hist_id, hist_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) rc = plan_download(H, D, h_bp_tour, h_bp_pos, h_field_bp, h_field_pos, h_hu_tour, h_su_tour, st);
    if (e == cudaSuccess && rc == LGX_OK) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = cuda_fail(e, "lgx_local_search");
  }
  cudaFreeAsync(ws, st); cudaFreeAsync(D.base, st);
  if (rc == LGX_OK) *h_best_cost = best;
  return rc;
}

}  // extern "C"
