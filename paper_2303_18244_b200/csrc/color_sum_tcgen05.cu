// color_sum_tcgen05.cu — FP32 colour sum of the 120-flow process on the 5th-generation tensor cores (float and mixed mode;
// SURVEY.md §8(a) step a7, north_star: "FP32 tcgen05 tensor cores").
//
// For one helicity, one part P in (re, im) and a tile of 128 events the contraction is the GEMM
//     D[e][f] = sum_k X_P[e][k] C[f][k]                 (M = 128 events, N = 128 (120 flows + 8 zero rows), K = 120)
// followed by the per-event dot  sum_f D[e][f] X_P[e][f]  (C is symmetric); |M|^2_h ~ dot(re) + dot(im).
// C holds integers with <= 11 significant bits, exact in TF32.  X is split as X = X_hi + X_lo, X_hi = the upper 19 bits
// of X (a TF32 number), X_lo = X - X_hi (exact in FP32; the tensor core reads its upper 19 bits); both halves are
// accumulated into the same FP32 accumulator: relative error ~2^-20 per term, the FP32 level, far below the 1e-4 bound.
//
// tcgen05.mma.kind::tf32, cta_group::1, M = 128, N = 128, K = 8 per instruction, both operands from shared memory in the
// canonical K-major no-swizzle layout (8 x 16 B core matrices), accumulator D in tensor memory (128 columns).
// A CTA is 128 threads = 128 TMEM lanes = 128 events: thread t loads the staged jamps of event t (FP32, or FP64 in mixed
// mode; coalesced across the warp), writes the hi / lo operands, and also parks the FP32 value in its own TMEM lane
// (tcgen05.st, 120 more columns), so that the epilogue dot reads D and X from tensor memory and nothing is fetched twice.
// K is streamed in chunks of 24 through a two-stage shared-memory ring with two chunks of loads in flight in registers;
// completion is tracked with tcgen05.commit -> mbarrier.  Two CTAs per SM (109 KB of shared memory, 256 TMEM columns each)
// overlap each other's load / MMA / epilogue phases.
#include <cstdint>

#include "multi.h"

namespace me {

#define TC_NCOL 120
#define TC_M 128                                   // events per tile = TMEM lanes
#define TC_KC 24                                   // K per ring stage (3 MMA steps of 8)
#define TC_NCHUNK (TC_NCOL / TC_KC)                // 5 chunks per (re | im) part
#define TC_A_SBO (128 * (TC_KC / 4))               // byte step between 8-event groups of A: 768
#define TC_HALF_BYTES (16 * TC_A_SBO)              // one operand (hi or lo) of a stage: 12288 B
#define TC_STAGE_BYTES (2 * TC_HALF_BYTES)
#define TC_B_BYTES (128 * TC_NCOL * 4)             // colour matrix, 128 rows (8 of them zero): 61440 B
#define TC_B_SBO (128 * (TC_NCOL / 4))             // byte step between 8-flow groups of B: 3840
#define TC_LBO 128                                 // byte step between core matrices adjacent in K
#define TC_SMEM (TC_B_BYTES + 2 * TC_STAGE_BYTES + 64)
#define TC_TMEM_COLS 256                           // D: columns 0..127, parked X: columns 128..247
#define TC_XCOL 128

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared-memory matrix descriptor, no swizzle: start address, leading (K) and stride (M/N) byte offsets in 16 B units, version 1
__device__ __forceinline__ uint64_t tc_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | (1ull << 46);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, N = 128, M = 128
#define TC_IDESC ((1u << 4) | (2u << 7) | (2u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24))

__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "l"(adesc), "l"(bdesc), "r"(TC_IDESC), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool tc_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
               : "=r"(done)
               : "r"(bar), "r"(parity)
               : "memory");
  return done != 0;
}
__device__ __forceinline__ void tc_wait(uint32_t bar, uint32_t parity) {
  if (tc_try_wait(bar, parity)) return;
  const long long t0 = clock64();
  while (!tc_try_wait(bar, parity))
    if (clock64() - t0 > 8000000000LL) __trap();   // ~4 s: a lost completion must surface as an error, never as a hang
}
// 8 consecutive TMEM columns of this thread's lane
__device__ __forceinline__ void tc_st8(uint32_t taddr, const float* v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};\n" ::"r"(taddr), "r"(__float_as_uint(v[0])),
               "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])),
               "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7]))
               : "memory");
}
__device__ __forceinline__ void tc_ld8_nowait(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
}

// RJ: staging type (float in float mode, double in mixed mode: cast after load)
template <typename RJ>
__global__ void __launch_bounds__(TC_M, 2) k_color_sum_tcgen05(const float* __restrict__ cmat, const RJ* __restrict__ gj, long npad, long n,
                                                                long hs, int nh, const unsigned char* __restrict__ hels, int first,
                                                                double norm_hel, double inv_avg, double* __restrict__ me_out,
                                                                double* __restrict__ me_hel) {
  extern __shared__ __align__(128) unsigned char smem[];
  unsigned char* sB = smem;                                   // colour matrix, canonical K-major layout
  unsigned char* sA = smem + TC_B_BYTES;                      // 2 stages x (hi | lo)
  uint64_t* bars = (uint64_t*)(smem + TC_B_BYTES + 2 * TC_STAGE_BYTES);
  uint32_t* tptr = (uint32_t*)(bars + 2);
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t bar0 = smem_u32(bars), sA0 = smem_u32(sA), sB0 = smem_u32(sB);

  // B[f][k] = C[f][k]: flow f -> 8-row group f / 8, 16 B chunk j = k / 4
  for (int i = tid; i < 128 * (TC_NCOL / 4); i += TC_M) {
    const int f = i / (TC_NCOL / 4), j = i % (TC_NCOL / 4);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (f < TC_NCOL) v = make_float4(cmat[f * TC_NCOL + 4 * j], cmat[f * TC_NCOL + 4 * j + 1], cmat[f * TC_NCOL + 4 * j + 2], cmat[f * TC_NCOL + 4 * j + 3]);
    *(float4*)(sB + (f >> 3) * TC_B_SBO + j * TC_LBO + (f & 7) * 16) = v;
  }
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0 + 8));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tptr)), "r"(TC_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // B was written through the generic proxy
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tptr;
  const uint32_t tlane = tmem + ((uint32_t)(warp * 32) << 16);   // this warp's quarter of the 128 lanes

  const long ntiles = (npad + TC_M - 1) / TC_M;
  unsigned char* myA = sA + (tid >> 3) * TC_A_SBO + (tid & 7) * 16;   // this event's 16 B slot inside every core matrix
  const long np2 = 2 * npad;
  uint32_t g = 0;                                                     // running chunk counter: ring stage = g & 1
  for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const long e = tile * TC_M + tid;
    const RJ* ge = gj + (e < npad ? e : tile * TC_M);                 // lanes past the end read finite data; the result is dropped
    double me_acc = 0;
    float p = 0.f;
    // two chunks of staged jamps are in flight in registers (raw staging type: the conversion waits for the data, so it
    // is done at the point of use).  Chunk q = hc * 10 + part * 5 + c covers rows (hc * 120 + 24 c + i) * 2 + part.
    RJ curA[TC_KC], curB[TC_KC];
    const int nq = nh * 2 * TC_NCHUNK;
#define TC_LOAD_CHUNK(CUR, Q)                                                                                     \
  if ((Q) < nq) {                                                                                                 \
    const int hq = (Q) / (2 * TC_NCHUNK), pq = (Q) % (2 * TC_NCHUNK);                                             \
    const RJ* pc_ = ge + (((long)hq * TC_NCOL + (pq % TC_NCHUNK) * TC_KC) * 2 + pq / TC_NCHUNK) * npad;           \
    _Pragma("unroll") for (int i = 0; i < TC_KC; ++i) CUR[i] = pc_[i * np2];                                      \
  }
    // one ring step: operands of chunk (hc, PC) from CUR -> shared memory and TMEM, refill CUR with chunk + 2, issue the MMAs
#define TC_STEP(CUR, PC)                                                                                          \
  {                                                                                                               \
    const uint32_t s = g & 1;                                                                                     \
    const int c = (PC) % TC_NCHUNK;                                                                               \
    float x[TC_KC], hi[TC_KC];                                                                                    \
    _Pragma("unroll") for (int i = 0; i < TC_KC; ++i) {                                                           \
      x[i] = (float)CUR[i];                                                                                       \
      hi[i] = __uint_as_float(__float_as_uint(x[i]) & 0xffffe000u);                                               \
    }                                                                                                             \
    TC_LOAD_CHUNK(CUR, hc * 2 * TC_NCHUNK + (PC) + 2)                                                             \
    _Pragma("unroll") for (int j = 0; j < TC_KC / 8; ++j) tc_st8(tlane + TC_XCOL + c * TC_KC + 8 * j, x + 8 * j); \
    if (g >= 2) tc_wait(bar0 + 8 * s, ((g >> 1) - 1) & 1); /* the MMAs that read this stage two chunks ago are done */ \
    unsigned char* a = myA + s * TC_STAGE_BYTES;                                                                  \
    _Pragma("unroll") for (int j = 0; j < TC_KC / 4; ++j) {                                                       \
      *(float4*)(a + j * TC_LBO) = make_float4(hi[4 * j], hi[4 * j + 1], hi[4 * j + 2], hi[4 * j + 3]);           \
      *(float4*)(a + TC_HALF_BYTES + j * TC_LBO) =                                                                \
          make_float4(x[4 * j] - hi[4 * j], x[4 * j + 1] - hi[4 * j + 1], x[4 * j + 2] - hi[4 * j + 2], x[4 * j + 3] - hi[4 * j + 3]); \
    }                                                                                                             \
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");                                                  \
    __syncthreads();                                                                                              \
    if (tid == 0) {                                                                                               \
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");                                             \
      const uint32_t ah = sA0 + s * TC_STAGE_BYTES, al = ah + TC_HALF_BYTES, b = sB0 + c * (TC_KC / 4) * TC_LBO;  \
      _Pragma("unroll") for (int st = 0; st < TC_KC / 8; ++st) {                                                  \
        const uint64_t bd = tc_desc(b + st * 2 * TC_LBO, TC_LBO, TC_B_SBO);                                       \
        tc_mma(tmem, tc_desc(ah + st * 2 * TC_LBO, TC_LBO, TC_A_SBO), bd, (c | st) != 0);                         \
        tc_mma(tmem, tc_desc(al + st * 2 * TC_LBO, TC_LBO, TC_A_SBO), bd, 1u);                                    \
      }                                                                                                           \
      tc_commit(bar0 + 8 * s);                                                                                    \
    }                                                                                                             \
    ++g;                                                                                                          \
    if (c == TC_NCHUNK - 1) { /* part complete: p += sum_f D[e][f] X[e][f], both read from this thread's TMEM lane */ \
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");                                                \
      tc_wait(bar0 + 8 * s, ((g - 1) >> 1) & 1);                                                                  \
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");                                             \
      _Pragma("unroll") for (int f0 = 0; f0 < TC_NCOL; f0 += 24) {                                                \
        uint32_t d[3][8], xs[3][8];                                                                               \
        _Pragma("unroll") for (int j = 0; j < 3; ++j) {                                                           \
          tc_ld8_nowait(tlane + f0 + 8 * j, d[j]);                                                                \
          tc_ld8_nowait(tlane + TC_XCOL + f0 + 8 * j, xs[j]);                                                     \
        }                                                                                                         \
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");                                              \
        _Pragma("unroll") for (int j = 0; j < 3; ++j)                                                             \
          _Pragma("unroll") for (int i = 0; i < 8; ++i) p = fmaf(__uint_as_float(d[j][i]), __uint_as_float(xs[j][i]), p); \
      }                                                                                                           \
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); /* orders these loads before the next MMAs */ \
    }                                                                                                             \
  }
    TC_LOAD_CHUNK(curA, 0)
    TC_LOAD_CHUNK(curB, 1)
    for (int hc = 0; hc < nh; ++hc) {
#pragma unroll 1
      for (int pc = 0; pc < 2 * TC_NCHUNK; pc += 2) {
        TC_STEP(curA, pc)
        TC_STEP(curB, pc + 1)
      }
      if (e < n && me_hel != nullptr && hels[hc] != 255) me_hel[(long)hels[hc] * hs + e] = (double)p * norm_hel * 0.5;
      me_acc += (double)p;
      p = 0.f;
    }
    if (e < n && me_out != nullptr) {
      const double sc = norm_hel * 0.5 * inv_avg;
      me_out[e] = first ? me_acc * sc : me_out[e] + me_acc * sc;
    }
  }
#undef TC_STEP
#undef TC_LOAD_CHUNK
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TC_TMEM_COLS) : "memory");
}

cudaError_t launch_color_sum_tcgen05(int sms, int staging_is_double, const float* cmat, const void* gj, long npad, long n, long hs, int nh,
                                     const unsigned char* hels, int first, double norm_hel, double inv_avg, double* me_out, double* me_hel,
                                     cudaStream_t stream) {
  const long ntiles = (npad + TC_M - 1) / TC_M;
  const unsigned grid = (unsigned)(ntiles < 2L * sms ? ntiles : 2L * sms);
  cudaError_t e;
  if (staging_is_double) {
    e = cudaFuncSetAttribute(k_color_sum_tcgen05<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM);
    if (e != cudaSuccess) return e;
    k_color_sum_tcgen05<double><<<grid, TC_M, TC_SMEM, stream>>>(cmat, (const double*)gj, npad, n, hs, nh, hels, first, norm_hel, inv_avg, me_out, me_hel);
  } else {
    e = cudaFuncSetAttribute(k_color_sum_tcgen05<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, TC_SMEM);
    if (e != cudaSuccess) return e;
    k_color_sum_tcgen05<float><<<grid, TC_M, TC_SMEM, stream>>>(cmat, (const float*)gj, npad, n, hs, nh, hels, first, norm_hel, inv_avg, me_out, me_hel);
  }
  return cudaGetLastError();
}

}  // namespace me
