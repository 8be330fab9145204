// lgx_inst_decode.cu — instantiations of lgx_decode_cut (and the sqrt self-test kernel).
// Product code (CUDA path).  Shares nothing with oracle/.
#define LGX_INSTANTIATE_SELFTEST
#include "lgx_dispatch.h"

namespace lgx {

template <int MODE> static KernelFn pick_a(const ImgHdr &h)
{
  const bool p16 = h.perm16 != 0, zd = h.zero_demand != 0u, x64 = h.n_extra_blocks > 7u;
  KernelFn k = nullptr;
#define LGX_PICK_A(P, Z, X) if (p16 == P && zd == Z && x64 == X) k = lgx_decode_cut<P, Z, X, MODE>;
  LGX_PICK_A(false, false, false) LGX_PICK_A(false, false, true) LGX_PICK_A(false, true, false) LGX_PICK_A(false, true, true)
  LGX_PICK_A(true,  false, false) LGX_PICK_A(true,  false, true) LGX_PICK_A(true,  true, false) LGX_PICK_A(true,  true, true)
#undef LGX_PICK_A
  return k;
}

KernelFn pick_decode_cut(const ImgHdr &h, int mode)
{
  switch (mode) {
    case MODE_EVAL:   return pick_a<MODE_EVAL>(h);
    case MODE_SEARCH: return pick_a<MODE_SEARCH>(h);
    case MODE_DECODE: return pick_a<MODE_DECODE>(h);
    default:          return nullptr;
  }
}

const void *selftest_sqrt_kernel() { return (const void *)lgx_selftest_sqrt_k; }

}  // namespace lgx
