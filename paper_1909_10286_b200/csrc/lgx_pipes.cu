// lgx_pipes.cu — issue-rate microbenchmarks of the execution pipes the sampling kernels lean on (lgx_selftest
// what = 1..5; "measure the pipe sub-limits before quoting a fraction").  Each kernel runs one kind of
// instruction in eight independent chains per thread at full occupancy (two blocks of 1024 threads per SM, <= 32
// registers) and reports the cycles of its slowest block (clock64 inside the kernel: no assumption about the clock):
//   1  IMAD.WIDE.U32   the 32x32->64 products of Philox4x32-10 (lgx_decode_cut)
//   2  LOP3            the ALU pipe: integer logic, selects and 3-input adds of the decoder and of the walks' cursors
//   3  LDS.U8 + STS.U8 byte accesses to per-thread shared-memory columns (the Fisher-Yates array)
//   4  DFMA            FP64 (distances, cost accumulation; DADD / DMUL issue on the same pipe)
//   5  MUFU.RSQ64H     the seed of the in-line correctly rounded square root
// Warp-instructions of the probed kind / cycles / SMs = the pipe's sustained issue rate per SM, the denominator
// bench.py prints as roofline.pipe_peaks beside the generic 4 warp-instructions/clk/SM of the schedulers.
// Product code (diagnostic entry point of the CUDA path); shares nothing with oracle/.
#include <cstdint>
#include <cuda_runtime.h>

namespace lgx {

constexpr int kPipeThreads = 1024, kChains = 8;

template <int WHAT>
__global__ void __launch_bounds__(kPipeThreads, 2) lgx_pipe_k(uint32_t iters, unsigned long long *out, uint32_t *sink)
{
  __shared__ uint8_t cols[kChains * 2 * kPipeThreads];         // (3): byte column of thread t = bytes t, t + 1024, ...
  const uint32_t tid = threadIdx.x;
  uint32_t a[kChains]; unsigned long long w[kChains]; double d[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) {
    a[c] = tid * 2654435761u + 40503u * (uint32_t)c + 1u; w[c] = a[c]; d[c] = 1.0 + 1e-9 * (double)(a[c] & 1023u);
    cols[(2 * c) * kPipeThreads + tid] = (uint8_t)a[c]; cols[(2 * c + 1) * kPipeThreads + tid] = (uint8_t)c;
  }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
    for (int rep = 0; rep < 4; ++rep) {
#pragma unroll
      for (int c = 0; c < kChains; ++c) {
        if (WHAT == 1) {       // both halves of the product feed the next step (as in a Philox round), or ptxas drops to a 32-bit IMAD;
                               // the XOR goes to the ALU pipe and is not counted
          asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[c]) : "r"(a[c]), "r"(0xD2511F53u));
          a[c] = (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32);
        }
        if (WHAT == 2) {       // (a 32-bit add would be moved to the FMA pipe as IMAD.IADD by ptxas: logic only)
          asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[c]) : "r"(tid), "r"(it));
          asm volatile("lop3.b32 %0, %0, %1, %2, 0xE8;" : "+r"(a[c]) : "r"(it), "r"(tid));
        }
        if (WHAT == 3) {
          uint32_t v;
          const uint32_t addr = (uint32_t)__cvta_generic_to_shared(cols + (2 * c) * kPipeThreads + tid);
          asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
          asm volatile("st.shared.u8 [%0], %1;" :: "r"(addr + kPipeThreads), "r"(v) : "memory");
          a[c] += v;
        }
        if (WHAT == 4) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(0.999999999), "d"(1e-12));
        if (WHAT == 5) asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(d[c]));
      }
    }
  }
  const long long t1 = clock64();
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) acc ^= a[c] ^ (uint32_t)w[c] ^ (uint32_t)(w[c] >> 32) ^ (uint32_t)__double_as_longlong(d[c]) ^ cols[(2 * c + 1) * kPipeThreads + tid];
  if (acc == 0x12345678u) sink[0] = acc;                        // keeps every chain alive; practically never taken
  if (tid == 0u) atomicMax(out, (unsigned long long)(t1 - t0));
}

// Host side: h_out[0] = warp-instructions of the probed kind issued by the whole grid, h_out[1] = cycles of the
// slowest block (all blocks are co-resident and start together: two per SM).  Returns a cudaError_t as int.
int pipe_bench(int what, uint64_t iters, uint64_t *h_out)
{
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return (int)e;
  unsigned long long *d = nullptr;
  if ((e = cudaMalloc((void **)&d, 16)) != cudaSuccess) return (int)e;
  e = cudaMemset(d, 0, 16);
  const uint32_t it = (uint32_t)(iters > 0xFFFFFFFFull ? 0xFFFFFFFFull : iters);
  const dim3 grid(2u * (unsigned)n_sm), block(kPipeThreads);
  uint32_t *sink = reinterpret_cast<uint32_t *>(d + 1);
  if (e == cudaSuccess) {
    switch (what) {
      case 1: lgx_pipe_k<1><<<grid, block>>>(it, d, sink); break;
      case 2: lgx_pipe_k<2><<<grid, block>>>(it, d, sink); break;
      case 3: lgx_pipe_k<3><<<grid, block>>>(it, d, sink); break;
      case 4: lgx_pipe_k<4><<<grid, block>>>(it, d, sink); break;
      default: lgx_pipe_k<5><<<grid, block>>>(it, d, sink); break;
    }
    e = cudaGetLastError();
  }
  unsigned long long cyc = 0;
  if (e == cudaSuccess) e = cudaMemcpy(&cyc, d, 8, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return (int)e;
  const uint64_t per_chain_step = (what == 2 || what == 3) ? 2u : 1u;      // (2): two LOP3, (3): LDS + STS per step
  h_out[0] = (uint64_t)grid.x * (kPipeThreads / 32) * (uint64_t)it * 4u * kChains * per_chain_step;
  h_out[1] = cyc;
  return 0;
}

}  // namespace lgx
