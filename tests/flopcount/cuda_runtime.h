/* Stand-in for <cuda_runtime.h> when tests/flopcount/count_flops.cpp compiles csrc/hel_amp.cuh on the HOST with g++
 * (no CUDA involved: the routines are templates on the real type and are instantiated with a counting scalar). */
#pragma once
#define __device__
#define __host__
#define __forceinline__ inline
#define __restrict__
