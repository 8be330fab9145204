// lgx_dispatch.h — which translation unit instantiates which kernel.  The kernel templates of lgx_kernels.cuh
// and lgx_moves.cuh are instantiated in small .cu files of their own (lgx_inst_*.cu) that nvcc compiles in
// parallel; the host code of lgx_api.cu only sees these pick functions.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include "lgx_kernels.cuh"

namespace lgx {

struct MvParams;
using KernelFn   = void (*)(const KParams);
using MvKernelFn = void (*)(const MvParams);

// lgx_decode_cut<P16, ZD, XB64, mode> for the instance (lgx_inst_decode.cu); mode = MODE_EVAL / _SEARCH / _DECODE
KernelFn pick_decode_cut(const ImgHdr &h, int mode);
// lgx_walk_finish<P16, DM, MASKW, mode>, one translation unit per distance mode DM (lgx_inst_walk.cu, -DLGX_DM=0|1|2)
KernelFn pick_walk_finish_dm0(const ImgHdr &h, int mode);
KernelFn pick_walk_finish_dm1(const ImgHdr &h, int mode);
KernelFn pick_walk_finish_dm2(const ImgHdr &h, int mode);
// lgx_move_eval_k / lgx_local_search_k<MASKW, HB>, one translation unit per MASKW (lgx_inst_moves.cu, -DLGX_MASKW=1|2)
void pick_move_kernels_mw1(const ImgHdr &h, MvKernelFn &batch, MvKernelFn &search);
void pick_move_kernels_mw2(const ImgHdr &h, MvKernelFn &batch, MvKernelFn &search);
const void *init_plan_kernel();        // lgx_init_plan_k (with MASKW = 1's unit)
const void *selftest_sqrt_kernel();    // lgx_selftest_sqrt_k (with the decode unit)

}  // namespace lgx
