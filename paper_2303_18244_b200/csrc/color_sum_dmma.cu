// color_sum_dmma.cu — FP64 colour sum of the 120-flow process on the tensor cores (SURVEY.md §8(a) step a7,
// BASELINE.json north_star: "the colour sum is batched as a genuine dense contraction over events, on FP64 DMMA").
//
//     Y = L X,   L = lower triangle of the [120 x 120] colour-matrix numerators (off-diagonal entries doubled: C is
//     symmetric),  X [120 x (2 * events)] = (Re J, Im J) of one helicity,
//     ME_h(evt) = sum_i  X[i][evt,re] Y[i][evt,re] + X[i][evt,im] Y[i][evt,im]
// The 8 x 4 tiles of L above the diagonal are zero and are skipped: 240 of the 450 (row block, k-step) pairs remain.
//
// mma.sync.m8n8k4.f64 (DMMA): M = 8 colour rows, N = 8 events, K = 4 colour columns.  A warp owns 8 events and both
// their Re and Im columns (two N-tiles) for ALL 15 row blocks: 30 accumulator tiles (60 doubles) in registers, so each
// A fragment (from shared memory, stored in fragment order -> conflict-free) feeds two DMMAs and each B fragment
// (read straight from the global staging buffer, 64-byte segments) feeds fifteen.  The epilogue multiplies Y with X in
// the accumulator layout and reduces over the 8 lanes that share a column with shuffles.  Persistent CTAs (one per
// SM, 8 warps) keep the 115 KB of C fragments resident.
#include "multi.h"

namespace me {

#define CD_NCOL 120
#define CD_RB (CD_NCOL / 8)     // 15 row blocks
#define CD_KS (CD_NCOL / 4)     // 30 k-steps
#define CD_WARPS 8
#define CD_PF 5                 // k-steps of B fragments prefetched per batch

__device__ __forceinline__ void dmma8x8x4(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(32 * CD_WARPS, 1) k_color_sum_dmma(const double* __restrict__ cmat, const double* __restrict__ gj, long npad, long n, long hs, int nh,
                                                                    const unsigned char* __restrict__ hels, int first,
                                                                    double norm_hel, double inv_avg,
                                                                    double* __restrict__ me_out, double* __restrict__ me_hel) {
  extern __shared__ __align__(16) double cfrag[];          // [CD_RB][CD_KS][32] in A-fragment order
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < CD_RB * CD_KS * 32; i += blockDim.x) {
    const int l = i & 31, ks = (i >> 5) % CD_KS, rb = (i >> 5) / CD_KS;
    const int r = rb * 8 + (l >> 2), c = ks * 4 + (l & 3);
    // C is symmetric: x^T C x = sum_r x_r (C_rr x_r + 2 sum_{c<r} C_rc x_c), so only the lower triangle is contracted
    cfrag[i] = c < r ? 2.0 * cmat[r * CD_NCOL + c] : c == r ? cmat[r * CD_NCOL + c] : 0.0;
  }
  __syncthreads();
  const long ntiles = (npad + 8 * CD_WARPS - 1) / (8 * CD_WARPS);
  const int kr = lane & 3, ec = lane >> 2;                 // B fragment: row kr of the k-step, event column ec
  for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long e0 = (tile * CD_WARPS + w) * 8;
    if (e0 >= npad) continue;                              // npad is a multiple of 32: a warp is either fully in or out
    double me_acc0 = 0, me_acc1 = 0;
    double bre[CD_PF], bim[CD_PF];                         // B fragments of the next batch of k-steps, always one batch ahead (also across helicities)
#pragma unroll
    for (int j = 0; j < CD_PF; ++j) {
      const double* p = gj + e0 + (long)(2 * (4 * j + kr)) * npad + ec;
      bre[j] = p[0]; bim[j] = p[npad];
    }
    for (int hc = 0; hc < nh; ++hc) {
      const double* g = gj + (long)hc * (2 * CD_NCOL) * npad + e0;
      double acc[CD_RB][2][2];
#pragma unroll
      for (int rb = 0; rb < CD_RB; ++rb) { acc[rb][0][0] = acc[rb][0][1] = acc[rb][1][0] = acc[rb][1][1] = 0; }
#pragma unroll   // fully unrolled: the triangular skip below is then resolved at compile time (a predicated-off DMMA still costs its pipe slot)
      for (int kb = 0; kb < CD_KS; kb += CD_PF) {
        double nre[CD_PF], nim[CD_PF];
        const bool more = kb + CD_PF < CD_KS;              // (compile-time after unrolling)
        if (more || hc + 1 < nh) {                         // the last batch of a helicity fetches the first batch of the next one: its latency hides behind the epilogue
          const double* gn = more ? g + (long)(2 * 4 * (kb + CD_PF)) * npad : g + (long)(2 * CD_NCOL) * npad;
#pragma unroll
          for (int j = 0; j < CD_PF; ++j) {
            const double* p = gn + (long)(2 * (4 * j + kr)) * npad + ec;
            nre[j] = p[0]; nim[j] = p[npad];
          }
        }
#pragma unroll
        for (int j = 0; j < CD_PF; ++j) {
          const double* af = cfrag + (kb + j) * 32 + lane;
          const int rbmin = (kb + j) >> 1;                 // row blocks above this one hold only zeros in columns 4 (kb + j) ..
#pragma unroll
          for (int rb = 0; rb < CD_RB; ++rb) {
            if (rb < rbmin) continue;
            const double a = af[rb * CD_KS * 32];
            dmma8x8x4(acc[rb][0][0], acc[rb][0][1], a, bre[j]);
            dmma8x8x4(acc[rb][1][0], acc[rb][1][1], a, bim[j]);
          }
        }
        if (more || hc + 1 < nh) {
#pragma unroll
          for (int j = 0; j < CD_PF; ++j) { bre[j] = nre[j]; bim[j] = nim[j]; }
        }
      }
      // epilogue: accumulator element (row = rb*8 + lane/4, column = 2*(lane%4) + {0,1})
      double p0 = 0, p1 = 0;
#pragma unroll
      for (int rb = 0; rb < CD_RB; ++rb) {
        const double* x = g + (long)(2 * (rb * 8 + ec)) * npad + 2 * kr;
        const double2 xr = *reinterpret_cast<const double2*>(x), xi = *reinterpret_cast<const double2*>(x + npad);
        p0 += acc[rb][0][0] * xr.x + acc[rb][1][0] * xi.x;
        p1 += acc[rb][0][1] * xr.y + acc[rb][1][1] * xi.y;
      }
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) { p0 += __shfl_xor_sync(0xffffffffu, p0, o); p1 += __shfl_xor_sync(0xffffffffu, p1, o); }
      if (lane < 4) {
        const long e = e0 + 2 * lane;
        if (me_hel != nullptr && hels[hc] != 255) {
          if (e < n) me_hel[(long)hels[hc] * hs + e] = p0 * norm_hel * 0.5;
          if (e + 1 < n) me_hel[(long)hels[hc] * hs + e + 1] = p1 * norm_hel * 0.5;
        }
        me_acc0 += p0; me_acc1 += p1;
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

cudaError_t launch_color_sum_dmma(int sms, const double* cmat, const double* gj, long npad, long n, long hs, int nh, const unsigned char* hels, int first,
                                  double norm_hel, double inv_avg, double* me_out, double* me_hel, cudaStream_t stream) {
  const size_t smem = sizeof(double) * CD_RB * CD_KS * 32;
  cudaError_t e = cudaFuncSetAttribute(k_color_sum_dmma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const long ntiles = (npad + 8 * CD_WARPS - 1) / (8 * CD_WARPS);
  const unsigned grid = (unsigned)(ntiles < sms ? ntiles : sms);
  k_color_sum_dmma<<<grid, 32 * CD_WARPS, smem, stream>>>(cmat, gj, npad, n, hs, nh, hels, first, norm_hel, inv_avg, me_out, me_hel);
  return cudaGetLastError();
}

}  // namespace me
