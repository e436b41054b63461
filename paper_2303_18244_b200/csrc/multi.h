// multi.h — pipeline of the multi-kernel process (g g -> t t~ g g g): diagram kernels (each looping over the
// helicities of the chunk) add the
// colour-flow amplitudes of a chunk of helicities into a global staging buffer
//     gj[hc][ncol][2 (re,im)][npad]      (FP64 in double and mixed mode, FP32 in float mode)
// and the batched colour-sum kernel (color_sum.cu) contracts them with the colour matrix.
#pragma once
#include "kernels.h"

#define ME_HEL_CHUNK 32   // helicities staged per pass
#ifndef ME_HEL_PER_CTA
#define ME_HEL_PER_CTA 4   // helicities looped inside one CTA of a diagram kernel (grid.y covers the chunk)
#endif

namespace me {

struct MultiArgs {
  const double* mom; long npad; const unsigned char* hels; int nh; double mt; void* gj; cudaStream_t stream;
  const int* hel_per_event; long n;
  void* cache;      // sharing kernels: L2-resident region for currents parked across the helicities of a CTA (null: not available)
};
// zeroes_staging: bit p set = the kernel launched for precision p zeroes the staging rows of a helicity itself before it adds into them;
// when the first kernel of a pass says so the staging buffer is not zeroed (cudaMemsetAsync) in front of the pass
struct MultiKernel { cudaError_t (*launch)(int precision, const MultiArgs&); int zeroes_staging; };

cudaError_t launch_multi(int precision, const LaunchArgs& a, const MultiKernel* const* parts, int nparts, int ncol,
                         const double* color_num_host);
size_t multi_scratch_bytes(int precision, long npad, int ncol);
// bytes of the current cache behind the staging buffer: `vectors` four-vectors per thread and CTA of a diagram kernel (0: none)
size_t multi_cache_bytes(int precision, long npad, int vectors);
cudaError_t launch_multi(int precision, const LaunchArgs& a, const MultiKernel* const* parts, int nparts, int ncol,
                         const double* color_num_host, int cache_vectors);
// (colour-sum launchers: cmat = device pointer owned by the context, sms = multiprocessors of its device)
// FP32 colour sum on the tensor cores, TF32 hi/lo split (color_sum_tf32.cu); cmat = device pointer to float numerators
cudaError_t launch_color_sum_tf32(int sms, int staging_is_double, const float* cmat, const void* gj, long npad, long n, long hs, int nh,
                                  const unsigned char* hels, int first, double norm_hel, double inv_avg, double* me_out, double* me_hel,
                                  cudaStream_t stream);
// the same contraction on tcgen05 / TMEM (color_sum_tcgen05.cu): the default FP32 / mixed colour sum
cudaError_t launch_color_sum_tcgen05(int sms, int staging_is_double, const float* cmat, const void* gj, long npad, long n, long hs, int nh,
                                     const unsigned char* hels, int first, double norm_hel, double inv_avg, double* me_out, double* me_hel,
                                     cudaStream_t stream);
// FP64 colour sum on the tensor cores (color_sum_dmma.cu); cmat = device pointer to the [ncol*ncol] numerators
cudaError_t launch_color_sum_dmma(int sms, const double* cmat, const double* gj, long npad, long n, long hs, int nh, const unsigned char* hels, int first,
                                  double norm_hel, double inv_avg, double* me_out, double* me_hel, cudaStream_t stream);

}  // namespace me
