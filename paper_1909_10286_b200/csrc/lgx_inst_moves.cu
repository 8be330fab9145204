// lgx_inst_moves.cu — instantiations of the Algorithm-1 kernels for ONE SU-mask width (compiled twice:
// -DLGX_MASKW=1 | 2); the unit of MASKW = 1 also carries lgx_init_plan_k.
// Product code (CUDA path).  Shares nothing with oracle/.
#ifndef LGX_MASKW
#error "compile with -DLGX_MASKW=1 or 2"
#endif
#if LGX_MASKW == 1
#define LGX_INSTANTIATE_INIT_PLAN
#endif
#include "../../include/lgx.h"
#include "lgx_dispatch.h"
#include "lgx_moves.cuh"

#define LGX_CAT_(a, b) a##b
#define LGX_CAT(a, b) LGX_CAT_(a, b)

namespace lgx {

void LGX_CAT(pick_move_kernels_mw, LGX_MASKW)(const ImgHdr &h, MvKernelFn &batch, MvKernelFn &search)
{
  batch = search = nullptr;
  if (h.mask_words != (uint32_t)LGX_MASKW) return;
  if (h.flags & LGX_FLAG_HU_BALANCE) { batch = lgx_move_eval_k<LGX_MASKW, true>;  search = lgx_local_search_k<LGX_MASKW, true>; }
  else                               { batch = lgx_move_eval_k<LGX_MASKW, false>; search = lgx_local_search_k<LGX_MASKW, false>; }
}

#if LGX_MASKW == 1
const void *init_plan_kernel() { return (const void *)lgx_init_plan_k; }
#endif

}  // namespace lgx
