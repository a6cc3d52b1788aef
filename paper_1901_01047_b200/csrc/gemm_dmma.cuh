// The FP64 tensor-core instruction of sm_100a: mma.sync m8n8k4 (SASS DMMA.8x8x4).  tcgen05.mma has no FP64 kind, so
// the FP64 GEMM tiles of gemm_tma.cuh keep their accumulators in registers and issue this instruction per warp.
// Fragment layout (PTX ISA, mma.m8n8k4 .f64): lane l holds A[row l/4][k l%4], B[k l%4][col l/4] and the two
// accumulator elements C[row l/4][cols 2(l%4), 2(l%4)+1].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctaux {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

}  // namespace ctaux
