// color_sum_tf32.cu — FP32 colour sum of the 120-flow process on the tensor cores (float and mixed mode;
// "FP32 ... TF32-split", §7 hard part 3).
//
//     Y = C X,   C [120 x 120] colour-matrix numerators (integers with <= 11 significant bits: EXACT in TF32),
//     X = (Re J, Im J) of one helicity, split as X = X_hi + X_lo with X_hi = tf32(X), X_lo = tf32(X - X_hi):
//     Y = C X_hi + C X_lo accumulated in FP32  ->  relative error ~2^-21 (the FP32 level), far below the 1e-4 bound.
//
// mma.sync.m16n8k8 tf32 (SASS HMMA.1688.F32.TF32): M = 16 colour rows, N = 8 events, K = 8 colour columns.  As in
// color_sum_dmma.cu a warp owns 8 events and both their Re and Im columns for ALL row tiles (8 tiles of 16 rows, the
// last half-tile zero padded): 16 accumulator tiles (64 floats) in registers; C fragments in shared memory in
// fragment order (conflict-free 128-bit loads), B fragments straight from the global staging buffer.
// Superseded as the default by color_sum_tcgen05.cu (3x faster); kept behind ME_COLOR_MMA_SYNC=1 as its A/B baseline.
#include "multi.h"

namespace me {

#define CT_NCOL 120
#define CT_RT 8                 // row tiles of 16 (128 rows, 120 used)
#define CT_KS (CT_NCOL / 8)     // 15 k-steps
#define CT_WARPS 8

__device__ __forceinline__ unsigned f2tf32(float x) {
  unsigned r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void mma16n8k8_tf32(float (&d)[4], const uint4& a, unsigned b0, unsigned b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
               : "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b0), "r"(b1));
}

// RJ: staging type (float in float mode, double in mixed mode: cast on load)
template <typename RJ>
__global__ void __launch_bounds__(32 * CT_WARPS, 1) k_color_sum_tf32(const float* __restrict__ cmat, const RJ* __restrict__ gj, long npad, long n,
                                                                    long hs, int nh, const unsigned char* __restrict__ hels, int first,
                                                                    double norm_hel, double inv_avg,
                                                                    double* __restrict__ me_out, double* __restrict__ me_hel) {
  extern __shared__ __align__(16) uint4 cfrag4[];          // [CT_RT][CT_KS][32] A fragments (a0..a3 per lane)
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < CT_RT * CT_KS * 32; i += blockDim.x) {
    const int l = i & 31, ks = (i >> 5) % CT_KS, rt = (i >> 5) / CT_KS;
    const int g = l >> 2, t = l & 3, r0 = rt * 16 + g, c0 = ks * 8 + t;
    // a0:(g, t)  a1:(g+8, t)  a2:(g, t+4)  a3:(g+8, t+4)
    const float a0 = r0 < CT_NCOL ? cmat[r0 * CT_NCOL + c0] : 0.f, a1 = r0 + 8 < CT_NCOL ? cmat[(r0 + 8) * CT_NCOL + c0] : 0.f;
    const float a2 = r0 < CT_NCOL ? cmat[r0 * CT_NCOL + c0 + 4] : 0.f, a3 = r0 + 8 < CT_NCOL ? cmat[(r0 + 8) * CT_NCOL + c0 + 4] : 0.f;
    cfrag4[i] = make_uint4(f2tf32(a0), f2tf32(a1), f2tf32(a2), f2tf32(a3));
  }
  __syncthreads();
  const long ntiles = (npad + 8 * CT_WARPS - 1) / (8 * CT_WARPS);
  const int t = lane & 3, g = lane >> 2;                   // B fragment: rows t, t+4 of the k-step, event column g
  for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long e0 = (tile * CT_WARPS + w) * 8;
    if (e0 >= npad) continue;
    double me_acc0 = 0, me_acc1 = 0;
    for (int hc = 0; hc < nh; ++hc) {
      const RJ* gp = gj + (long)hc * (2 * CT_NCOL) * npad + e0;
      float acc[CT_RT][2][4];
#pragma unroll
      for (int rt = 0; rt < CT_RT; ++rt)
#pragma unroll
        for (int c = 0; c < 2; ++c) { acc[rt][c][0] = acc[rt][c][1] = acc[rt][c][2] = acc[rt][c][3] = 0.f; }
#pragma unroll 3
      for (int ks = 0; ks < CT_KS; ++ks) {
        // B (8 x 8): b0 = X[8 ks + t][event g], b1 = X[8 ks + t + 4][event g]; re and im tiles, hi and lo parts
        const RJ* p0 = gp + (long)(2 * (8 * ks + t)) * npad + g;
        const RJ* p1 = gp + (long)(2 * (8 * ks + t + 4)) * npad + g;
        const float xr0 = (float)p0[0], xi0 = (float)p0[npad], xr1 = (float)p1[0], xi1 = (float)p1[npad];
        const unsigned hr0 = f2tf32(xr0), hi0 = f2tf32(xi0), hr1 = f2tf32(xr1), hi1 = f2tf32(xi1);
        const unsigned lr0 = f2tf32(xr0 - __uint_as_float(hr0)), li0 = f2tf32(xi0 - __uint_as_float(hi0));
        const unsigned lr1 = f2tf32(xr1 - __uint_as_float(hr1)), li1 = f2tf32(xi1 - __uint_as_float(hi1));
        const uint4* af = cfrag4 + ks * 32 + lane;
#pragma unroll
        for (int rt = 0; rt < CT_RT; ++rt) {
          const uint4 a = af[rt * CT_KS * 32];
          mma16n8k8_tf32(acc[rt][0], a, hr0, hr1);
          mma16n8k8_tf32(acc[rt][0], a, lr0, lr1);
          mma16n8k8_tf32(acc[rt][1], a, hi0, hi1);
          mma16n8k8_tf32(acc[rt][1], a, li0, li1);
        }
      }
      // epilogue: c0:(row g, col 2t) c1:(g, 2t+1) c2:(g+8, 2t) c3:(g+8, 2t+1) of every row tile
      float p0 = 0.f, p1 = 0.f;
#pragma unroll
      for (int rt = 0; rt < CT_RT; ++rt) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const int row = rt * 16 + g + 8 * half;
          if (row < CT_NCOL) {
            const RJ* x = gp + (long)(2 * row) * npad + 2 * t;
            const float xr0 = (float)x[0], xr1 = (float)x[1], xi0 = (float)x[npad], xi1 = (float)x[npad + 1];
            p0 += acc[rt][0][2 * half] * xr0 + acc[rt][1][2 * half] * xi0;
            p1 += acc[rt][0][2 * half + 1] * xr1 + acc[rt][1][2 * half + 1] * xi1;
          }
        }
      }
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) { p0 += __shfl_xor_sync(0xffffffffu, p0, o); p1 += __shfl_xor_sync(0xffffffffu, p1, o); }
      if (lane < 4) {
        const long e = e0 + 2 * lane;
        if (me_hel != nullptr && hels[hc] != 255) {
          if (e < n) me_hel[(long)hels[hc] * hs + e] = (double)p0 * norm_hel * 0.5;
          if (e + 1 < n) me_hel[(long)hels[hc] * hs + e + 1] = (double)p1 * norm_hel * 0.5;
        }
        me_acc0 += (double)p0; me_acc1 += (double)p1;
      }
    }
    if (lane < 4 && me_out != nullptr) {
      const long e = e0 + 2 * lane;
      const double s = norm_hel * 0.5 * inv_avg;
      if (e < n) me_out[e] = first ? me_acc0 * s : me_out[e] + me_acc0 * s;
      if (e + 1 < n) me_out[e + 1] = first ? me_acc1 * s : me_out[e + 1] + me_acc1 * s;
    }
  }
}

cudaError_t launch_color_sum_tf32(int sms, int staging_is_double, const float* cmat, const void* gj, long npad, long n, long hs, int nh,
                                  const unsigned char* hels, int first, double norm_hel, double inv_avg, double* me_out, double* me_hel,
                                  cudaStream_t stream) {
  const size_t smem = sizeof(uint4) * CT_RT * CT_KS * 32;
  const long ntiles = (npad + 8 * CT_WARPS - 1) / (8 * CT_WARPS);
  const unsigned grid = (unsigned)(ntiles < sms ? ntiles : sms);
  cudaError_t e;
  if (staging_is_double) {
    e = cudaFuncSetAttribute(k_color_sum_tf32<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_color_sum_tf32<double><<<grid, 32 * CT_WARPS, smem, stream>>>(cmat, (const double*)gj, npad, n, hs, nh, hels, first, norm_hel, inv_avg, me_out, me_hel);
  } else {
    e = cudaFuncSetAttribute(k_color_sum_tf32<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_color_sum_tf32<float><<<grid, 32 * CT_WARPS, smem, stream>>>(cmat, (const float*)gj, npad, n, hs, nh, hels, first, norm_hel, inv_avg, me_out, me_hel);
  }
  return cudaGetLastError();
}

}  // namespace me
