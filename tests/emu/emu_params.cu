// emu_params.cu — TEST INFRASTRUCTURE (tests/emu): size of the kernel parameter block for the host shim's launcher.
#include "../../paper_1909_10286_b200/csrc/lgx_kernels.cuh"
size_t lgx_emu_param_bytes() { return sizeof(lgx::KParams); }
