// color_sum.cu — batched colour sum for the multi-kernel process:
//     ME_h(evt) = sum_ij conj(J_i) C_ij J_j = Jr^T C Jr + Ji^T C Ji          (C real symmetric)
// evaluated as a dense contraction over a tile of events: Y = C X with X = [ncol x (2*events)],
// then the column-wise dot X.Y.  This file holds the plain-FMA version (FP64 or FP32):
// a CTA owns 32 events (one per lane); each of its 8 warps owns ncol/8 rows of C and keeps their
// 2*ncol/8 accumulators in registers, so every shared-memory load of X feeds ncol/8 FMAs whose
// C operand is a warp-uniform (broadcast) load.
#include "multi.h"

#include <cstdlib>

namespace me {

#define CS_NCOL 120
#define CS_WARPS 8
#define CS_ROWS (CS_NCOL / CS_WARPS)   // 15

// (the colour-matrix numerators, exact small integers, 115 KB in FP64, live in device buffers owned by the context: cm)
// RJ: staging type, RC: arithmetic type of the contraction
template <typename RJ, typename RC>
__global__ void __launch_bounds__(32 * CS_WARPS) k_color_sum(const RC* __restrict__ cm, const RJ* __restrict__ gj, long npad, long n, long hs, int nh,
                                                             const unsigned char* __restrict__ hels, int first,
                                                             double norm_hel, double inv_avg,
                                                             double* __restrict__ me_out, double* __restrict__ me_hel) {
  extern __shared__ __align__(16) unsigned char cs_smem[];
  RC (*sx)[32] = reinterpret_cast<RC (*)[32]>(cs_smem);                 // [2*CS_NCOL][32]
  RC (*red)[32] = sx + 2 * CS_NCOL;                                     // [CS_WARPS][32]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const long e = (long)blockIdx.x * 32 + lane;
  double acc = 0;
  for (int hc = 0; hc < nh; ++hc) {
    const RJ* g = gj + (long)hc * (2 * CS_NCOL) * npad + e;
    __syncthreads();
    for (int r = w; r < 2 * CS_NCOL; r += CS_WARPS) sx[r][lane] = (RC)g[(long)r * npad];
    __syncthreads();
    RC yr[CS_ROWS], yi[CS_ROWS];
#pragma unroll
    for (int r = 0; r < CS_ROWS; ++r) { yr[r] = 0; yi[r] = 0; }
    const int row0 = w * CS_ROWS;
#pragma unroll 4
    for (int j = 0; j < CS_NCOL; ++j) {
      const RC xr = sx[2 * j][lane], xi = sx[2 * j + 1][lane];
#pragma unroll
      for (int r = 0; r < CS_ROWS; ++r) {
        const RC c = __ldg(&cm[(row0 + r) * CS_NCOL + j]);
        yr[r] += c * xr; yi[r] += c * xi;
      }
    }
    RC part = 0;
#pragma unroll
    for (int r = 0; r < CS_ROWS; ++r) part += yr[r] * sx[2 * (row0 + r)][lane] + yi[r] * sx[2 * (row0 + r) + 1][lane];
    red[w][lane] = part;
    __syncthreads();
    if (w == 0) {
      RC s = 0;
#pragma unroll
      for (int k = 0; k < CS_WARPS; ++k) s += red[k][lane];
      const double meh = (double)s;
      if (me_hel != nullptr && e < n && hels[hc] != 255) me_hel[(long)hels[hc] * hs + e] = meh * norm_hel * 0.5;
      acc += meh;
    }
  }
  if (w == 0 && me_out != nullptr && e < n) {
    const double v = acc * norm_hel * 0.5 * inv_avg;
    me_out[e] = first ? v : me_out[e] + v;
  }
}

// events are processed in slices so that the staging buffer stays bounded (32 helicities x 240 rows x 65536 events: 3.8 GB in FP64) whatever n is
#define ME_EVENT_SLICE 65536L
size_t multi_scratch_bytes(int precision, long npad, int ncol) {
  const long np = npad < ME_EVENT_SLICE ? npad : ME_EVENT_SLICE;
  return (size_t)ME_HEL_CHUNK * ncol * 2 * np * (precision == 2 ? sizeof(float) : sizeof(double));
}

// tensor-core colour sums (FP64: DMMA, FP32: TF32 split); ME_COLOR_FMA=1 in the environment selects the plain-FMA kernels (A/B timing)
static const bool g_use_dmma = getenv("ME_COLOR_FMA") == nullptr;
// ME_COLOR_MMA_SYNC=1 selects the warp-level TF32 kernel (color_sum_tf32.cu) instead of the tcgen05 one (A/B timing)
static const bool g_use_tcgen05 = getenv("ME_COLOR_MMA_SYNC") == nullptr;

// one region per CTA of a diagram kernel: grid = (slice / 128 threads) x (chunk / ME_HEL_PER_CTA helicity groups)
size_t multi_cache_bytes(int precision, long npad, int vectors) {
  const long np = npad < ME_EVENT_SLICE ? npad : ME_EVENT_SLICE;
  const long ctas = (np + 127) / 128 * (ME_HEL_CHUNK / ME_HEL_PER_CTA);
  return (size_t)ctas * vectors * 8 * 128 * (precision == 2 ? sizeof(float) : sizeof(double));
}

static cudaError_t launch_multi_slice(int precision, const LaunchArgs& a, long hs, const MultiKernel* const* parts, int nparts, int ncol,
                                      const double* color_num_host, void* cache);

cudaError_t launch_multi(int precision, const LaunchArgs& a, const MultiKernel* const* parts, int nparts, int ncol,
                         const double* color_num_host) {
  return launch_multi(precision, a, parts, nparts, ncol, color_num_host, 0);
}

cudaError_t launch_multi(int precision, const LaunchArgs& a, const MultiKernel* const* parts, int nparts, int ncol,
                         const double* color_num_host, int cache_vectors) {
  const int npar = 7;   // g g -> t t~ g g g
  // the current cache of the sharing kernels sits behind the staging buffer of the batch (sizes as scratch_bytes of the process table)
  void* cache = nullptr;
  if (cache_vectors > 0) {
    const size_t off = (multi_scratch_bytes(precision, a.npad, ncol) + 255) / 256 * 256;
    if (a.scratch == nullptr || a.scratch_bytes < off + multi_cache_bytes(precision, a.npad, cache_vectors)) return cudaErrorInvalidValue;
    cache = (char*)a.scratch + off;
  }
  for (long start = 0; start < a.n; start += ME_EVENT_SLICE) {
    LaunchArgs s = a;
    s.n = a.n - start < ME_EVENT_SLICE ? a.n - start : ME_EVENT_SLICE;
    s.npad = (s.n + ME_PAGE - 1) / ME_PAGE * ME_PAGE;
    s.mom = a.mom + (start / ME_PAGE) * (npar * 4 * ME_PAGE);
    if (a.me_out != nullptr) s.me_out = a.me_out + start;
    if (a.me_hel != nullptr) s.me_hel = a.me_hel + start;
    if (a.jamp_out != nullptr) s.jamp_out = a.jamp_out + start;
    if (a.hel_per_event != nullptr) s.hel_per_event = a.hel_per_event + start;
    cudaError_t e = launch_multi_slice(precision, s, a.n, parts, nparts, ncol, color_num_host, cache);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

static cudaError_t launch_multi_slice(int precision, const LaunchArgs& a, long hs, const MultiKernel* const* parts, int nparts, int ncol,
                                      const double* color_num_host, void* cache) {
  if (ncol != CS_NCOL) return cudaErrorInvalidValue;
  if (a.color_d == nullptr || a.color_f == nullptr) return cudaErrorInvalidValue;   // uploaded by me_create on the context's device
  const unsigned cgrid = (unsigned)(a.npad / 32);
  for (int base = 0; base < a.nhel; base += ME_HEL_CHUNK) {
    const int nh = a.nhel - base < ME_HEL_CHUNK ? a.nhel - base : ME_HEL_CHUNK;
    MultiArgs m{a.mom, a.npad, a.hels + base, nh, a.mt, a.scratch, a.stream, a.hel_per_event, a.n, cache};
    if (!((parts[0]->zeroes_staging >> precision) & 1)) {   // every diagram kernel ADDS its colour flows into the staging buffer
      const size_t esz = precision == 2 ? sizeof(float) : sizeof(double);
      cudaError_t e = cudaMemsetAsync(a.scratch, 0, (size_t)nh * ncol * 2 * a.npad * esz, a.stream);
      if (e != cudaSuccess) return e;
    }
    for (int k = 0; k < nparts; ++k) {
      cudaError_t e = parts[k]->launch(precision, m);
      if (e != cudaSuccess) return e;
    }
    if (a.jamp_out != nullptr && base == 0) {
      const size_t esz = precision == 2 ? sizeof(float) : sizeof(double);
      if (esz != sizeof(double)) return cudaErrorInvalidValue;   // jamp hook is FP64 only
      cudaError_t e = cudaMemcpy2DAsync(a.jamp_out, hs * sizeof(double), a.scratch, a.npad * sizeof(double), a.n * sizeof(double),
                                        2 * ncol, cudaMemcpyDeviceToDevice, a.stream);
      if (e != cudaSuccess) return e;
    }
    const int first = base == 0;
    const size_t smd = sizeof(double) * (2 * CS_NCOL + CS_WARPS) * 32, smf = sizeof(float) * (2 * CS_NCOL + CS_WARPS) * 32;
    cudaFuncSetAttribute(k_color_sum<double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smd);
    if (precision == 0 && g_use_dmma) {
      cudaError_t e2 = launch_color_sum_dmma(a.nsm, a.color_d, (const double*)a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.stream);
      if (e2 != cudaSuccess) return e2;
    } else if (precision != 0 && g_use_dmma) {      // FP32 colour sum (float and mixed mode) on the tensor cores, TF32 hi/lo split
      const float* cf = a.color_f;
      cudaError_t e2 = cudaSuccess;
      if (g_use_tcgen05)
        e2 = launch_color_sum_tcgen05(a.nsm, precision == 1, cf, a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.stream);
      else e2 = launch_color_sum_tf32(a.nsm, precision == 1, cf, a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.stream);
      if (e2 != cudaSuccess) return e2;
    } else if (precision == 0)
      k_color_sum<double, double><<<cgrid, 32 * CS_WARPS, smd, a.stream>>>(a.color_d, (const double*)a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel);
    else if (precision == 1)
      k_color_sum<double, float><<<cgrid, 32 * CS_WARPS, smf, a.stream>>>(a.color_f, (const double*)a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel);
    else
      k_color_sum<float, float><<<cgrid, 32 * CS_WARPS, smf, a.stream>>>(a.color_f, (const float*)a.scratch, a.npad, a.n, hs, nh, a.hels + base, first, a.norm_hel, a.inv_avg, a.me_out, a.me_hel);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace me
