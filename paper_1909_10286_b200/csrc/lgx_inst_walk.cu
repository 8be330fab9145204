// lgx_inst_walk.cu — instantiations of lgx_walk_finish for ONE distance mode (compiled three times:
// -DLGX_DM=0 tables, 1 coordinates, 2 field x BP table + coordinates).
// Product code (CUDA path).  Shares nothing with oracle/.
#include "lgx_dispatch.h"

#ifndef LGX_DM
#error "compile with -DLGX_DM=0, 1 or 2"
#endif
#define LGX_CAT_(a, b) a##b
#define LGX_CAT(a, b) LGX_CAT_(a, b)

namespace lgx {

template <int MODE> static KernelFn pick_b(const ImgHdr &h)
{
  const bool p16 = h.perm16 != 0; const int mw = (int)h.mask_words;
  KernelFn k = nullptr;
#define LGX_PICK(P, M) if (p16 == P && mw == M) k = lgx_walk_finish<P, LGX_DM, M, MODE>;
  LGX_PICK(false, 1) LGX_PICK(false, 2) LGX_PICK(true, 1) LGX_PICK(true, 2)
#undef LGX_PICK
  return k;
}

KernelFn LGX_CAT(pick_walk_finish_dm, LGX_DM)(const ImgHdr &h, int mode)
{
  if (h.coords != LGX_DM) return nullptr;
  switch (mode) {
    case MODE_EVAL:   return pick_b<MODE_EVAL>(h);
    case MODE_SEARCH: return pick_b<MODE_SEARCH>(h);
    case MODE_DECODE: return pick_b<MODE_DECODE>(h);
    default:          return nullptr;
  }
}

}  // namespace lgx
