// rng_rambo.cu — support kernels of the standalone harness:
// Philox4x32-10 uniforms (Salmon et al. SC'11; reading Q14) and RAMBO flat phase space
// (Kleiss, Stirling, Ellis 1986; reading Q12), plus the FMA-chain peak microbenchmark that
// bench.py uses as the measured roofline denominator.
#include "kernels.h"

namespace me {

// ---------------------------------------------------------------------------------- Philox
__device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3, uint32_t k0, uint32_t k1) {
  const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
  const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
  const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
  c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    philox_round(c0, c1, c2, c3, k0, k1);
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ double u53(uint32_t a, uint32_t b) {
  // ((a>>5)*2^26 + (b>>6) + 0.5) * 2^-53 : exact in binary64, strictly inside (0,1)
  return ((double)(a >> 5) * 67108864.0 + (double)(b >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

__global__ void k_philox(uint64_t seed, uint64_t first_event, long n, int per_event, double* __restrict__ rnd) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n * per_event) return;
  const uint64_t ev = first_event + (uint64_t)(t / per_event);
  const uint32_t k = (uint32_t)(t % per_event);
  uint32_t w[8];
  philox4x32_10((uint32_t)ev, (uint32_t)(ev >> 32), k, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  philox4x32_10((uint32_t)ev, (uint32_t)(ev >> 32), k, 1u, (uint32_t)seed, (uint32_t)(seed >> 32), w + 4);
  double2* o = reinterpret_cast<double2*>(rnd + t * 4);
  o[0] = make_double2(u53(w[0], w[1]), u53(w[2], w[3]));
  o[1] = make_double2(u53(w[4], w[5]), u53(w[6], w[7]));
}

cudaError_t launch_philox(uint64_t seed, uint64_t first_event, long n, int per_event, double* d_rnd, cudaStream_t s) {
  const long total = n * per_event;
  if (total == 0) return cudaSuccess;
  k_philox<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(seed, first_event, n, per_event, d_rnd);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------- helicity / colour selection
// PAPER.md line 138 (section 5): "event-by-event random choice of leading colour and helicity".  Reading (DESIGN.md
// "Selection"): two uniforms per event from Philox counter (event lo, event hi, 'SELE', 0); helicity h drawn with
// probability ME_h / sum ME_h over the good helicities, colour flow s with probability |J_s(h)|^2 / sum |J|^2; inverse
// CDF in index order, FP64, left-to-right sums: pick the first k with cum_k >= u * total.
#define ME_SELECT_TAG 0x53454C45u
__device__ __forceinline__ void select_uniforms(uint64_t seed, uint64_t ev, double& u1, double& u2) {
  uint32_t w[4];
  philox4x32_10((uint32_t)ev, (uint32_t)(ev >> 32), ME_SELECT_TAG, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  u1 = u53(w[0], w[1]); u2 = u53(w[2], w[3]);
}
__device__ __forceinline__ int inverse_cdf(const double* __restrict__ w, int m, long stride, double u) {
  double tot = 0;
  for (int k = 0; k < m; ++k) tot += w[k * stride];
  const double target = u * tot;
  double cum = 0; int sel = -1, lastpos = 0;
  for (int k = 0; k < m; ++k) {
    const double x = w[k * stride];
    cum += x;
    if (x > 0) lastpos = k;
    if (sel < 0 && x > 0 && cum >= target) sel = k;
  }
  return sel < 0 ? lastpos : sel;
}
__global__ void k_select_hel(const double* __restrict__ me_hel, int ncomb, long n, uint64_t seed, uint64_t first_event, int* __restrict__ ihel) {
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  double u1, u2; select_uniforms(seed, first_event + (uint64_t)e, u1, u2);
  ihel[e] = inverse_cdf(me_hel + e, ncomb, n, u1);
}
__global__ void k_select_col(double* __restrict__ jamp, int ncol, long n, uint64_t seed, uint64_t first_event, int* __restrict__ icol) {
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  double u1, u2; select_uniforms(seed, first_event + (uint64_t)e, u1, u2);
  for (int s = 0; s < ncol; ++s) {          // |J_s|^2 in place (re slot)
    const double re = jamp[(2 * s) * n + e], im = jamp[(2 * s + 1) * n + e];
    jamp[(2 * s) * n + e] = re * re + im * im;
  }
  icol[e] = inverse_cdf(jamp + e, ncol, 2 * n, u2);
}
// me_filter_helicities (reading Q7): tot[i] = sum_h ME_h(i) in index order, then per helicity the maximum over the filter events of
// ME_h(i) / tot[i] (IEEE division; a maximum does not depend on the reduction order: bit-identical to the plain host loops)
__global__ void k_hel_total(const double* __restrict__ me_hel, int ncomb, long n, double* __restrict__ tot) {
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  double t = 0;
  for (int h = 0; h < ncomb; ++h) t += me_hel[(long)h * n + e];
  tot[e] = t;
}
__global__ void __launch_bounds__(256) k_hel_maxfrac(const double* __restrict__ me_hel, long n, const double* __restrict__ tot, double* __restrict__ maxfrac) {
  __shared__ double sh[8];
  const double* row = me_hel + (long)blockIdx.x * n;
  double m = 0;
  for (long e = threadIdx.x; e < n; e += 256) { const double f = row[e] / tot[e]; if (f > m) m = f; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_down_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) { for (int k = 1; k < 8; ++k) m = fmax(m, sh[k]); maxfrac[blockIdx.x] = m; }
}
cudaError_t launch_helicity_fractions(const double* me_hel, int ncomb, long n, double* tot, double* maxfrac, cudaStream_t s) {
  k_hel_total<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(me_hel, ncomb, n, tot);
  k_hel_maxfrac<<<ncomb, 256, 0, s>>>(me_hel, n, tot, maxfrac);
  return cudaGetLastError();
}
cudaError_t launch_select_hel(const double* me_hel, int ncomb, long n, uint64_t seed, uint64_t first_event, int* ihel, cudaStream_t s) {
  k_select_hel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(me_hel, ncomb, n, seed, first_event, ihel);
  return cudaGetLastError();
}
cudaError_t launch_select_col(double* jamp, int ncol, long n, uint64_t seed, uint64_t first_event, int* icol, cudaStream_t s) {
  k_select_col<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(jamp, ncol, n, seed, first_event, icol);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------- cross section + unweighting
// PAPER.md line 24 (section 2): "hit-or-miss unweighting, cross-section"; line 45: idea of offloading it.  Reading (DESIGN.md
// "Unweighting"): w_i = flux * W_i * ME_i; sigma = mean w; event i is kept iff u_i * wmax < w_i with u_i from Philox counter
// (event lo, event hi, 'UNWT', 0).  Reductions are fixed-order trees (no atomics): bit-identical run to run.
#define ME_UNWT_TAG 0x554E5754u
#define ME_RED_THREADS 256
__device__ __forceinline__ void block_reduce3(double& s, double& q, double& m, double* sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s += __shfl_down_sync(0xffffffffu, s, o); q += __shfl_down_sync(0xffffffffu, q, o);
    m = fmax(m, __shfl_down_sync(0xffffffffu, m, o));
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { sh[3 * w] = s; sh[3 * w + 1] = q; sh[3 * w + 2] = m; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < ME_RED_THREADS / 32; ++k) { s += sh[3 * k]; q += sh[3 * k + 1]; m = fmax(m, sh[3 * k + 2]); }
  }
}
__global__ void __launch_bounds__(ME_RED_THREADS) k_weight_partials(const double* __restrict__ wt, const double* __restrict__ me_, long n,
                                                                    double flux, double* __restrict__ w_out, double* __restrict__ part) {
  __shared__ double sh[3 * ME_RED_THREADS / 32];
  const long e = (long)blockIdx.x * ME_RED_THREADS + threadIdx.x;
  double w = 0;
  if (e < n) { w = flux * wt[e] * me_[e]; w_out[e] = w; }
  double s = w, q = w * w, m = w;
  block_reduce3(s, q, m, sh);
  if (threadIdx.x == 0) { part[3 * blockIdx.x] = s; part[3 * blockIdx.x + 1] = q; part[3 * blockIdx.x + 2] = m; }
}
__global__ void __launch_bounds__(ME_RED_THREADS) k_weight_final(const double* __restrict__ part, long nblocks, double* __restrict__ out) {
  __shared__ double sh[3 * ME_RED_THREADS / 32];
  double s = 0, q = 0, m = 0;
  for (long b = threadIdx.x; b < nblocks; b += ME_RED_THREADS) { s += part[3 * b]; q += part[3 * b + 1]; m = fmax(m, part[3 * b + 2]); }
  block_reduce3(s, q, m, sh);
  if (threadIdx.x == 0) { out[0] = s; out[1] = q; out[2] = m; }
}
__global__ void __launch_bounds__(ME_RED_THREADS) k_accept(const double* __restrict__ w, long n, double wmax, uint64_t seed, uint64_t first_event,
                                                           unsigned char* __restrict__ accept, unsigned long long* __restrict__ part) {
  __shared__ int sh[ME_RED_THREADS / 32];
  const long e = (long)blockIdx.x * ME_RED_THREADS + threadIdx.x;
  int a = 0;
  if (e < n) {
    const uint64_t ev = first_event + (uint64_t)e;
    uint32_t r[4];
    philox4x32_10((uint32_t)ev, (uint32_t)(ev >> 32), ME_UNWT_TAG, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), r);
    a = u53(r[0], r[1]) * wmax < w[e] ? 1 : 0;
    if (accept != nullptr) accept[e] = (unsigned char)a;
  }
  const unsigned b = __ballot_sync(0xffffffffu, a);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = __popc(b);
  __syncthreads();
  if (threadIdx.x == 0) { int c = 0; for (int k = 0; k < ME_RED_THREADS / 32; ++k) c += sh[k]; part[blockIdx.x] = (unsigned long long)c; }
}
// part[0] = sum of the per-block accept counts (integers: exact in any order)
__global__ void __launch_bounds__(ME_RED_THREADS) k_count_final(unsigned long long* __restrict__ part, long nblocks) {
  __shared__ unsigned long long sh[ME_RED_THREADS];
  unsigned long long c = 0;
  for (long b = threadIdx.x; b < nblocks; b += ME_RED_THREADS) c += part[b];
  sh[threadIdx.x] = c;
  __syncthreads();
  if (threadIdx.x == 0) { for (int k = 1; k < ME_RED_THREADS; ++k) c += sh[k]; part[0] = c; }
}
cudaError_t run_unweight(const double* d_wt, const double* d_me, long n, double flux, uint64_t seed, uint64_t first_event, double wmax_in,
                         double sums[3], unsigned char* d_accept, long long* naccept, cudaStream_t st) {
  const long nb = (n + ME_RED_THREADS - 1) / ME_RED_THREADS;
  double *d_w = nullptr, *d_part = nullptr, *d_out = nullptr; unsigned long long* d_cnt = nullptr;
  cudaError_t e = cudaMalloc(&d_w, sizeof(double) * n);
  if (e == cudaSuccess) e = cudaMalloc(&d_part, sizeof(double) * 3 * nb);
  if (e == cudaSuccess) e = cudaMalloc(&d_out, sizeof(double) * 3);
  if (e == cudaSuccess) e = cudaMalloc(&d_cnt, sizeof(unsigned long long) * nb);
  if (e == cudaSuccess) {
    k_weight_partials<<<(unsigned)nb, ME_RED_THREADS, 0, st>>>(d_wt, d_me, n, flux, d_w, d_part);
    k_weight_final<<<1, ME_RED_THREADS, 0, st>>>(d_part, nb, d_out);
    e = cudaMemcpyAsync(sums, d_out, sizeof(double) * 3, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  if (e == cudaSuccess && (d_accept != nullptr || naccept != nullptr)) {      // the count is produced with or without the flags
    const double wmax = wmax_in > 0 ? wmax_in : sums[2];
    k_accept<<<(unsigned)nb, ME_RED_THREADS, 0, st>>>(d_w, n, wmax, seed, first_event, d_accept, d_cnt);
    k_count_final<<<1, ME_RED_THREADS, 0, st>>>(d_cnt, nb);
    unsigned long long total = 0;
    e = cudaMemcpyAsync(&total, d_cnt, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (naccept != nullptr) *naccept = (long long)total;
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(d_w); cudaFree(d_part); cudaFree(d_out); cudaFree(d_cnt);
  return e;
}

// ---------------------------------------------------------------------------------- RAMBO
struct RamboMasses { double m[6]; };

template <int NF>
__global__ void k_rambo(RamboMasses masses, double sqs, const double* __restrict__ rnd, long n, long npad,
                        double* __restrict__ mom, double* __restrict__ wt, double w0, int massive) {
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= npad) return;
  const long e = t < n ? t : n - 1;   // lanes beyond n repeat the last event (finite padding)
  const double PI = 3.14159265358979323846;
  double q[NF][4], Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0;
#pragma unroll
  for (int k = 0; k < NF; ++k) {
    const double2 ra = reinterpret_cast<const double2*>(rnd + (e * NF + k) * 4)[0];
    const double2 rb = reinterpret_cast<const double2*>(rnd + (e * NF + k) * 4)[1];
    const double c = 2.0 * ra.x - 1.0, phi = 2.0 * PI * ra.y, q0 = -log(rb.x * rb.y), st = sqrt(1.0 - c * c);
    double sp, cp; sincos(phi, &sp, &cp);
    q[k][0] = q0; q[k][1] = q0 * st * cp; q[k][2] = q0 * st * sp; q[k][3] = q0 * c;
    Q0 += q[k][0]; Q1 += q[k][1]; Q2 += q[k][2]; Q3 += q[k][3];
  }
  const double M = sqrt(Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3);
  const double b1 = -Q1 / M, b2 = -Q2 / M, b3 = -Q3 / M, x = sqs / M, gam = Q0 / M, a = 1.0 / (1.0 + gam);
  double p[NF][4];
#pragma unroll
  for (int k = 0; k < NF; ++k) {
    const double bq = b1 * q[k][1] + b2 * q[k][2] + b3 * q[k][3];
    p[k][1] = x * (q[k][1] + b1 * q[k][0] + a * bq * b1);
    p[k][2] = x * (q[k][2] + b2 * q[k][0] + a * bq * b2);
    p[k][3] = x * (q[k][3] + b3 * q[k][0] + a * bq * b3);
    // massless energy as |p| rather than x (gam q0 + b.q): same number algebraically, on shell to rounding whatever the boost
    // amplifies (reading Q12a; the propagator denominators of the ME kernels assume on-shell legs)
    p[k][0] = sqrt(p[k][1] * p[k][1] + p[k][2] * p[k][2] + p[k][3] * p[k][3]);
  }
  double w = w0;
  if (massive) {
    double summ = 0;
#pragma unroll
    for (int k = 0; k < NF; ++k) summ += masses.m[k];
    double xi = sqrt(1.0 - (summ / sqs) * (summ / sqs));
    for (int it = 0; it < 100; ++it) {
      double f = -sqs, df = 0;
#pragma unroll
      for (int k = 0; k < NF; ++k) {
        const double en = sqrt(masses.m[k] * masses.m[k] + xi * xi * p[k][0] * p[k][0]);
        f += en; df += xi * p[k][0] * p[k][0] / en;
      }
      if (fabs(f) < 1e-14 * sqs) break;
      xi -= f / df;
    }
    double prod = 1, sum2 = 0;
#pragma unroll
    for (int k = 0; k < NF; ++k) {
      const double en = sqrt(masses.m[k] * masses.m[k] + xi * xi * p[k][0] * p[k][0]);
      p[k][1] *= xi; p[k][2] *= xi; p[k][3] *= xi; p[k][0] = en;
      const double k3 = sqrt(p[k][1] * p[k][1] + p[k][2] * p[k][2] + p[k][3] * p[k][3]);
      prod *= k3 / en; sum2 += k3 * k3 / en;
    }
    w *= pow(xi, (double)(2 * NF - 3)) * prod * sqs / sum2;
  }
  double* o = mom + (t >> 5) * ((NF + 2) * 4 * 32) + (t & 31);
  o[0 * 32] = 0.5 * sqs; o[1 * 32] = 0; o[2 * 32] = 0; o[3 * 32] = 0.5 * sqs;
  o[4 * 32] = 0.5 * sqs; o[5 * 32] = 0; o[6 * 32] = 0; o[7 * 32] = -0.5 * sqs;
#pragma unroll
  for (int k = 0; k < NF; ++k)
#pragma unroll
    for (int i = 0; i < 4; ++i) o[(4 * (2 + k) + i) * 32] = p[k][i];
  if (wt != nullptr && t < n) wt[t] = w;
}

cudaError_t launch_rambo(int nfinal, const double* masses, double sqrt_s, const double* d_rnd, long n,
                         double* d_mom, double* d_wt, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  RamboMasses m{}; int massive = 0;
  for (int k = 0; k < nfinal; ++k) { m.m[k] = masses[k]; if (masses[k] != 0.0) massive = 1; }
  const double PI = 3.14159265358979323846;
  double f1 = 1, f2 = 1;
  for (int i = 2; i <= nfinal - 1; ++i) f1 *= i;
  for (int i = 2; i <= nfinal - 2; ++i) f2 *= i;
  // massless RAMBO volume: (pi/2)^(n-1) s^(n-2) / ((n-1)!(n-2)!) * (2 pi)^(4-3n)
  double w0 = 1; for (int i = 0; i < nfinal - 1; ++i) w0 *= PI / 2;
  for (int i = 0; i < nfinal - 2; ++i) w0 *= sqrt_s * sqrt_s;
  w0 /= f1 * f2;
  for (int i = 0; i < 3 * nfinal - 4; ++i) w0 /= 2 * PI;
  const long npad = (n + ME_PAGE - 1) / ME_PAGE * ME_PAGE;
  const unsigned grid = (unsigned)((npad + 127) / 128);
  switch (nfinal) {
    case 2: k_rambo<2><<<grid, 128, 0, s>>>(m, sqrt_s, d_rnd, n, npad, d_mom, d_wt, w0, massive); break;
    case 3: k_rambo<3><<<grid, 128, 0, s>>>(m, sqrt_s, d_rnd, n, npad, d_mom, d_wt, w0, massive); break;
    case 4: k_rambo<4><<<grid, 128, 0, s>>>(m, sqrt_s, d_rnd, n, npad, d_mom, d_wt, w0, massive); break;
    case 5: k_rambo<5><<<grid, 128, 0, s>>>(m, sqrt_s, d_rnd, n, npad, d_mom, d_wt, w0, massive); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------- FMA peak
template <typename R>
__global__ void __launch_bounds__(256) k_fma_chain(R* out, int iters, R a, R b) {
  R x0 = (R)threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
      x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
    }
  }
  out[(long)blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

template <typename R>
static cudaError_t fma_peak_t(double* tflops) {
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = sms * 8, threads = 256, iters = sizeof(R) == 8 ? 4096 : 8192;
  R* d = nullptr;
  cudaError_t err = cudaMalloc(&d, sizeof(R) * (size_t)blocks * threads);
  if (err != cudaSuccess) return err;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    k_fma_chain<R><<<blocks, threads>>>(d, iters, (R)0.999999, (R)1e-3);
    cudaEventRecord(e1);
    err = cudaEventSynchronize(e1);
    if (err != cudaSuccess) break;
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (err != cudaSuccess) return err;
  const double flops = 2.0 * 64.0 * iters * (double)blocks * threads;
  *tflops = flops / (best * 1e-3) * 1e-12;
  return cudaSuccess;
}

cudaError_t run_fma_peak(int fp64, double* tflops) { return fp64 ? fma_peak_t<double>(tflops) : fma_peak_t<float>(tflops); }

}  // namespace me
