// me_api.cu — the C-ABI boundary declared in include/me.h: context, helicity filtering, dispatch.
// Host logic only; every arithmetic step of the path runs in the kernels (hel_amp.cuh, epem.cu,
// gen_*.cu, rng_rambo.cu).  No CPU fallback: without a CUDA device every entry point returns ME_ECUDA.
#include <stdlib.h>
#include "../../include/me.h"
#include "kernels.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

struct me_ctx {
  me_process process;
  me_sm_params prm;
  me_info info;
  int device;
  const me::ProcTable* tab;      // null for e+e-
  me::EpemCouplings epem;
  double norm_hel, inv_avg;
  unsigned char* d_hels_all;     // [ncomb] 0..ncomb-1
  unsigned char* d_hels_good;    // [ngood]
  int ngood;
  unsigned char* d_hels_half;    // parity pairing: one helicity of every good pair {h, ~h}
  int nhalf;                     // 0 = pairing not applicable to the current mask
  bool pairing;                  // option ME_OPT_PARITY_PAIRING
  uint64_t mask[2];
  bool filtered;
  void* scratch; size_t scratch_bytes;
  // me_compute_host: two device slices of momenta / MEs, a stream per copy direction, events (all created on first use)
  double* h_mom[2]; double* h_me[2]; size_t h_slice;     // h_slice = events a slice buffer holds (0: nothing allocated)
  cudaStream_t s_h2d, s_d2h, s_comp;
  cudaEvent_t ev_start, ev_h2d[2], ev_comp[2], ev_d2h[2];
};

static thread_local char g_errbuf[256] = "CUDA error (none recorded)";
static me_status cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", where, cudaGetErrorString(e));
  return ME_ECUDA;
}
#define ME_CUDA(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

extern "C" const char* me_strerror(me_status s) {
  switch (s) {
    case ME_OK: return "ok";
    case ME_EINVAL: return "invalid argument";
    case ME_EPROCESS: return "unknown process";
    case ME_ENOTFILTERED: return "helicities not filtered: call me_filter_helicities or me_set_helicities first";
    case ME_EALIGN: return "device buffer not 16-byte aligned";
    case ME_ENOMEM: return "out of memory";
    case ME_ECUDA: return g_errbuf;
  }
  return "unknown status";
}

static const me::ProcTable* table_of(me_process p) {
  switch (p) {
    case ME_GG_TTX: return &me::tab_gg_ttx;
    case ME_GG_TTXG: return &me::tab_gg_ttxg;
    case ME_GG_TTXGG: return &me::tab_gg_ttxgg;
    case ME_GG_TTXGGG: return &me::tab_gg_ttxggg;
    default: return nullptr;
  }
}

extern "C" me_status me_create(me_process process, const me_sm_params* prm, me_ctx** out) {
  if (prm == nullptr || out == nullptr) return ME_EINVAL;
  if ((int)process < 0 || (int)process > (int)ME_GG_TTXGGG) return ME_EPROCESS;
  me_ctx* c = new (std::nothrow) me_ctx();
  if (c == nullptr) return ME_ENOMEM;
  c->process = process; c->prm = *prm; c->filtered = false; c->ngood = 0; c->mask[0] = c->mask[1] = 0;
  c->scratch = nullptr; c->scratch_bytes = 0; c->h_slice = 0; c->h_mom[0] = c->h_mom[1] = c->h_me[0] = c->h_me[1] = nullptr; c->s_h2d = c->s_d2h = nullptr; c->d_hels_all = c->d_hels_good = c->d_hels_half = nullptr; c->nhalf = 0; c->pairing = false;
  me_info& I = c->info; memset(&I, 0, sizeof(I));
  I.page = ME_PAGE; I.ninitial = 2;
  const double PI = 3.14159265358979323846;
  if (process == ME_EPEM_MUPMUM) {
    if (!(prm->aewm1 > 0) || !(prm->sw2 > 0 && prm->sw2 < 1) || !(prm->mz > 0)) { delete c; return ME_EINVAL; }
    c->tab = nullptr;
    I.npar = 4; I.ndiagrams = 2; I.ncomb = 16; I.ncolor = 1; I.color_denom = 1; I.avg_denom = 4; I.nkernels = 1; I.namplitudes = 2;
    const double sw = std::sqrt(prm->sw2), cw = std::sqrt(1.0 - prm->sw2);
    c->epem.gL = (-0.5 + prm->sw2) / (sw * cw); c->epem.gR = prm->sw2 / (sw * cw); c->epem.mz = prm->mz; c->epem.wz = prm->wz;
    const double e2 = 4.0 * PI / prm->aewm1;
    c->norm_hel = e2 * e2;
    for (int k = 0; k < 3; ++k) { I.flops_per_helicity[k] = I.flops_executed_per_helicity[k] = me::epem_flops_per_helicity; I.flops_per_event_fixed[k] = 60; }
  } else {
    if (!(prm->mt > 0) || prm->wt != 0.0 || !(prm->alpha_s > 0)) { delete c; return ME_EINVAL; }
    const me::ProcTable* t = table_of(process);
    c->tab = t;
    const int n = t->nglu;
    I.npar = n + 2; I.ndiagrams = t->ndiagrams; I.ncomb = 1 << (n + 2); I.ncolor = t->ncol; I.color_denom = t->color_denom;
    int fact = 1; for (int i = 2; i <= n - 2; ++i) fact *= i;
    I.avg_denom = 4 * 64 * fact; I.nkernels = t->nkernels; I.namplitudes = t->namplitudes;
    I.mass[2] = I.mass[3] = prm->mt;
    const double gs2 = 4.0 * PI * prm->alpha_s;
    // |M|^2 carries g_s^(2n); the generated colour sum returns half the numerator of J^dagger C J
    c->norm_hel = std::pow(gs2, n) * 2.0 / t->color_denom;
    for (int k = 0; k < 3; ++k) { I.flops_per_helicity[k] = t->flops_per_helicity[k]; I.flops_executed_per_helicity[k] = t->flops_executed[k]; I.flops_per_event_fixed[k] = t->fixed_flops; }
  }
  c->inv_avg = 1.0 / I.avg_denom;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_all, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_good, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_half, 128);
  if (e == cudaSuccess) {
    unsigned char all[128]; for (int i = 0; i < 128; ++i) all[i] = (unsigned char)i;
    e = cudaMemcpy(c->d_hels_all, all, 128, cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) { cudaFree(c->d_hels_all); cudaFree(c->d_hels_good); cudaFree(c->d_hels_half); delete c; return cuda_fail(e, "me_create"); }
  *out = c;
  return ME_OK;
}

extern "C" me_status me_destroy(me_ctx* c) {
  if (c == nullptr) return ME_EINVAL;
  cudaDeviceSynchronize();
  cudaFree(c->d_hels_all); cudaFree(c->d_hels_good); cudaFree(c->d_hels_half); cudaFree(c->scratch);
  if (c->s_h2d != nullptr) {
    for (int b = 0; b < 2; ++b) { cudaFree(c->h_mom[b]); cudaFree(c->h_me[b]); cudaEventDestroy(c->ev_h2d[b]); cudaEventDestroy(c->ev_comp[b]); cudaEventDestroy(c->ev_d2h[b]); }
    cudaEventDestroy(c->ev_start); cudaStreamDestroy(c->s_h2d); cudaStreamDestroy(c->s_d2h); cudaStreamDestroy(c->s_comp);
  }
  delete c;
  return ME_OK;
}

extern "C" me_status me_get_info(const me_ctx* c, me_info* out) {
  if (c == nullptr || out == nullptr) return ME_EINVAL;
  *out = c->info;
  return ME_OK;
}

extern "C" me_status me_color_matrix(const me_ctx* c, double* out) {
  if (c == nullptr || out == nullptr) return ME_EINVAL;
  if (c->tab == nullptr) { out[0] = 1.0; return ME_OK; }
  memcpy(out, c->tab->color_num, sizeof(double) * c->tab->ncol * c->tab->ncol);
  return ME_OK;
}

static me_status run(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, const unsigned char* hels, int nhel,
                     double* d_me, double* d_me_hel, double* d_jamp, void* stream, const int* hel_per_event = nullptr) {
  if ((int)prec < 0 || (int)prec > 2) return ME_EINVAL;
  if (((uintptr_t)d_mom & 15) || ((uintptr_t)d_me & 7) || ((uintptr_t)d_me_hel & 7)) return ME_EALIGN;
  me::LaunchArgs a;
  a.mom = d_mom; a.n = n; a.npad = (n + ME_PAGE - 1) / ME_PAGE * ME_PAGE; a.hels = hels; a.nhel = nhel;
  a.mt = c->prm.mt; a.norm_hel = c->norm_hel; a.inv_avg = c->inv_avg;
  a.me_out = d_me; a.me_hel = d_me_hel; a.jamp_out = d_jamp; a.stream = (cudaStream_t)stream;
  a.scratch = nullptr; a.scratch_bytes = 0; a.hel_per_event = hel_per_event;
  if (c->tab != nullptr && c->tab->scratch_bytes != nullptr) {
    const size_t need = c->tab->scratch_bytes((int)prec, a.npad);
    if (need > c->scratch_bytes) {
      ME_CUDA(cudaStreamSynchronize(a.stream), "scratch sync");
      cudaFree(c->scratch); c->scratch = nullptr; c->scratch_bytes = 0;
      cudaError_t e = cudaMalloc(&c->scratch, need);
      if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
      ME_CUDA(e, "scratch alloc");
      c->scratch_bytes = need;
    }
    a.scratch = c->scratch; a.scratch_bytes = c->scratch_bytes;
  }
  cudaError_t e = c->tab != nullptr ? c->tab->launch((int)prec, a) : me::launch_epem((int)prec, a, c->epem);
  if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
  return ME_OK;
}

extern "C" me_status me_set_helicities(me_ctx* c, const uint64_t mask[2]) {
  if (c == nullptr || mask == nullptr) return ME_EINVAL;
  unsigned char good[128]; int ng = 0;
  for (int h = 0; h < c->info.ncomb; ++h) if (mask[h >> 6] >> (h & 63) & 1) good[ng++] = (unsigned char)h;
  if (ng == 0) return ME_EINVAL;
  ME_CUDA(cudaMemcpy(c->d_hels_good, good, ng, cudaMemcpyHostToDevice), "me_set_helicities");
  c->ngood = ng; c->mask[0] = mask[0]; c->mask[1] = c->info.ncomb > 64 ? mask[1] : 0; c->filtered = true;
  // parity pairing (pure-QCD processes): ME_h = ME_{~h}, ~h = all helicities flipped.  Usable only if the mask is
  // closed under h -> ~h; then the helicities with particle 0 at -1 represent every pair.
  c->nhalf = 0;
  if (c->tab != nullptr) {
    const int full = c->info.ncomb - 1, top = c->info.ncomb >> 1;
    unsigned char half[64]; int nh = 0; bool closed = true;
    for (int i = 0; i < ng && closed; ++i) {
      const int h = good[i], hb = full ^ h;
      if (!(mask[hb >> 6] >> (hb & 63) & 1)) closed = false;
      else if (!(h & top)) half[nh++] = (unsigned char)h;
    }
    if (closed && 2 * nh == ng) {
      ME_CUDA(cudaMemcpy(c->d_hels_half, half, nh, cudaMemcpyHostToDevice), "me_set_helicities");
      c->nhalf = nh;
    }
  }
  return ME_OK;
}

extern "C" me_status me_set_option(me_ctx* c, me_option opt, int value) {
  if (c == nullptr) return ME_EINVAL;
  switch (opt) {
    case ME_OPT_PARITY_PAIRING: c->pairing = value != 0; return ME_OK;
  }
  return ME_EINVAL;
}

extern "C" me_status me_filter_helicities(me_ctx* c, const double* d_mom, int64_t n, uint64_t mask_out[2], int* ngood_out, void* stream) {
  if (c == nullptr || d_mom == nullptr || mask_out == nullptr || n < 1) return ME_EINVAL;
  const int nc = c->info.ncomb;
  double* d_mh = nullptr;
  cudaError_t e = cudaMalloc(&d_mh, sizeof(double) * (size_t)nc * n);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
  ME_CUDA(e, "filter alloc");
  me_status st = run(c, d_mom, n, ME_FP64, c->d_hels_all, nc, nullptr, d_mh, nullptr, stream);
  if (st != ME_OK) { cudaFree(d_mh); return st; }
  std::vector<double> mh((size_t)nc * n);
  e = cudaMemcpyAsync(mh.data(), d_mh, sizeof(double) * mh.size(), cudaMemcpyDeviceToHost, (cudaStream_t)stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
  cudaFree(d_mh);
  if (e != cudaSuccess) return cuda_fail(e, "me_filter_helicities");
  // reading Q7: good <=> max_evt ME_h / sum_h' ME_h' > 1e-12
  uint64_t mask[2] = {0, 0};
  std::vector<double> tot(n, 0.0);
  for (int h = 0; h < nc; ++h) for (int64_t i = 0; i < n; ++i) tot[i] += mh[(size_t)h * n + i];
  for (int h = 0; h < nc; ++h) {
    double mx = 0;
    for (int64_t i = 0; i < n; ++i) { const double f = mh[(size_t)h * n + i] / tot[i]; if (f > mx) mx = f; }
    if (mx > 1e-12) mask[h >> 6] |= (uint64_t)1 << (h & 63);
  }
  st = me_set_helicities(c, mask);
  if (st != ME_OK) return st;
  mask_out[0] = mask[0]; mask_out[1] = mask[1];
  if (ngood_out != nullptr) *ngood_out = c->ngood;
  return ME_OK;
}

extern "C" me_status me_compute(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, double* d_me, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_me == nullptr) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  if (c->pairing && c->nhalf > 0) {           // half the helicities, each counted twice
    const double keep = c->inv_avg;
    c->inv_avg = 2.0 * keep;
    const me_status st = run(c, d_mom, n, prec, c->d_hels_half, c->nhalf, d_me, nullptr, nullptr, stream);
    c->inv_avg = keep;
    return st;
  }
  return run(c, d_mom, n, prec, c->d_hels_good, c->ngood, d_me, nullptr, nullptr, stream);
}

// Host-buffer entry (include/me.h): the batch is cut in slices of whole waves of CTAs; slice k + 1 travels host -> device on a
// copy stream while slice k is computed on the caller's stream, and the MEs of slice k travel back on a second copy stream.
extern "C" me_status me_compute_host(me_ctx* c, const double* h_mom, int64_t n, me_precision prec, double* h_me, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (h_mom == nullptr || h_me == nullptr || (int)prec < 0 || (int)prec > 2) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  cudaStream_t st = (cudaStream_t)stream;
  if (c->s_h2d == nullptr) {
    ME_CUDA(cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking), "host stream");
    ME_CUDA(cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking), "host stream");
    ME_CUDA(cudaStreamCreateWithFlags(&c->s_comp, cudaStreamNonBlocking), "host stream");
    ME_CUDA(cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming), "host event");
    for (int b = 0; b < 2; ++b) {
      ME_CUDA(cudaEventCreateWithFlags(&c->ev_h2d[b], cudaEventDisableTiming), "host event");
      ME_CUDA(cudaEventCreateWithFlags(&c->ev_comp[b], cudaEventDisableTiming), "host event");
      ME_CUDA(cudaEventCreateWithFlags(&c->ev_d2h[b], cudaEventDisableTiming), "host event");
    }
  }
  // slice = 6 CTAs of ME_BLOCK events on every SM (whole waves for 1, 2, 3 or 6 resident CTAs per SM), a multiple of the page
  // (ME_HOST_SLICE_UNITS = k: k times that; measured equal for 1, 2 and 4 on the headline workload, 1 needs the least copy bandwidth:
  // a slice of g g -> t t~ g g is 22 MB against 5.5 ms of kernel).  Every kernel ends with a drain phase in which SMs idle, so odd slices are
  // computed on a second stream: the CTAs of slice k + 1 fill the drain of slice k.  Processes with a library-owned staging buffer
  // (g g -> t t~ g g g) keep all slices on one stream.
  int dev = 0, nsm = 0;
  ME_CUDA(cudaGetDevice(&dev), "device");
  ME_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev), "device");
  static const int slice_units = getenv("ME_HOST_SLICE_UNITS") != nullptr ? atoi(getenv("ME_HOST_SLICE_UNITS")) : 1;
  const int64_t unit = (int64_t)nsm * ME_BLOCK * 6, slice = (slice_units > 0 ? slice_units : 1) * unit;
  const bool one_stream = c->tab != nullptr && c->tab->scratch_bytes != nullptr;
  const size_t ev_words = (size_t)c->info.npar * 4;            // doubles per event
  if (c->h_slice < (size_t)slice) {
    ME_CUDA(cudaStreamSynchronize(c->s_h2d), "host sync"); ME_CUDA(cudaStreamSynchronize(c->s_d2h), "host sync");
    for (int b = 0; b < 2; ++b) {
      cudaFree(c->h_mom[b]); cudaFree(c->h_me[b]); c->h_mom[b] = c->h_me[b] = nullptr;
    }
    c->h_slice = 0;
    for (int b = 0; b < 2; ++b) {
      cudaError_t e = cudaMalloc(&c->h_mom[b], sizeof(double) * ev_words * slice);
      if (e == cudaSuccess) e = cudaMalloc(&c->h_me[b], sizeof(double) * slice);
      if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
      ME_CUDA(e, "host slice alloc");
    }
    c->h_slice = (size_t)slice;
  }
  ME_CUDA(cudaEventRecord(c->ev_start, st), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_h2d, c->ev_start, 0), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_d2h, c->ev_start, 0), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_comp, c->ev_start, 0), "host start");
  int k = 0;
  for (int64_t first = 0; first < n; ++k) {
    const int b = k & 1;
    const int64_t cap = slice;
    const int64_t m = n - first < cap ? n - first : cap;
    const int64_t mpad = (m + ME_PAGE - 1) / ME_PAGE * ME_PAGE;
    cudaStream_t cs = (b == 1 && !one_stream) ? c->s_comp : st;
    if (k >= 2) ME_CUDA(cudaStreamWaitEvent(c->s_h2d, c->ev_comp[b], 0), "host wait");      // slice k - 2 no longer reads this buffer
    ME_CUDA(cudaMemcpyAsync(c->h_mom[b], h_mom + (size_t)first * ev_words, sizeof(double) * ev_words * mpad, cudaMemcpyHostToDevice, c->s_h2d), "host h2d");
    ME_CUDA(cudaEventRecord(c->ev_h2d[b], c->s_h2d), "host h2d");
    ME_CUDA(cudaStreamWaitEvent(cs, c->ev_h2d[b], 0), "host wait");
    if (k >= 2) ME_CUDA(cudaStreamWaitEvent(cs, c->ev_d2h[b], 0), "host wait");             // the MEs of slice k - 2 have left
    const me_status ms = me_compute(c, c->h_mom[b], m, prec, c->h_me[b], (void*)cs);
    if (ms != ME_OK) return ms;
    ME_CUDA(cudaEventRecord(c->ev_comp[b], cs), "host compute");
    ME_CUDA(cudaStreamWaitEvent(c->s_d2h, c->ev_comp[b], 0), "host wait");
    ME_CUDA(cudaMemcpyAsync(h_me + first, c->h_me[b], sizeof(double) * m, cudaMemcpyDeviceToHost, c->s_d2h), "host d2h");
    ME_CUDA(cudaEventRecord(c->ev_d2h[b], c->s_d2h), "host d2h");
    first += m;
  }
  for (int b = 0; b < (k < 2 ? k : 2); ++b) ME_CUDA(cudaStreamWaitEvent(st, c->ev_d2h[b], 0), "host end");
  return ME_OK;
}

extern "C" me_status me_compute_helicities(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, double* d_me, double* d_me_hel, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_me_hel == nullptr) return ME_EINVAL;
  return run(c, d_mom, n, prec, c->d_hels_all, c->info.ncomb, d_me, d_me_hel, nullptr, stream);
}

extern "C" me_status me_compute_jamps(me_ctx* c, const double* d_mom, int64_t n, int ihel, double* d_jamp, void* stream) {
  if (c == nullptr || n < 0 || d_mom == nullptr || d_jamp == nullptr) return ME_EINVAL;
  if (c->tab == nullptr || ihel < 0 || ihel >= c->info.ncomb) return ME_EINVAL;
  if (n == 0) return ME_OK;
  return run(c, d_mom, n, ME_FP64, c->d_hels_all + ihel, 1, nullptr, nullptr, d_jamp, stream);
}

extern "C" me_status me_select_helicity_color(me_ctx* c, const double* d_mom, int64_t n, uint64_t seed, uint64_t first_event,
                                              int32_t* d_ihel, int32_t* d_icol, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_ihel == nullptr || d_icol == nullptr) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  const int nc = c->info.ncomb, ncol = c->info.ncolor;
  cudaStream_t st = (cudaStream_t)stream;
  double* buf = nullptr;
  const size_t words = (size_t)n * (nc > 2 * ncol ? nc : 2 * ncol);
  cudaError_t e = cudaMalloc(&buf, sizeof(double) * words);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
  ME_CUDA(e, "select alloc");
  me_status ms = ME_OK;
  e = cudaMemsetAsync(buf, 0, sizeof(double) * (size_t)nc * n, st);                      // masked helicities weigh 0
  if (e == cudaSuccess) ms = run(c, d_mom, n, ME_FP64, c->d_hels_good, c->ngood, nullptr, buf, nullptr, stream);
  if (e == cudaSuccess && ms == ME_OK) e = me::launch_select_hel(buf, nc, n, seed, first_event, d_ihel, st);
  if (e == cudaSuccess && ms == ME_OK) {
    if (c->tab == nullptr) e = cudaMemsetAsync(d_icol, 0, sizeof(int32_t) * n, st);       // one colour structure
    else {
      ms = run(c, d_mom, n, ME_FP64, c->d_hels_all, 1, nullptr, nullptr, buf, stream, d_ihel);   // jamps of each event's own helicity
      if (ms == ME_OK) e = me::launch_select_col(buf, ncol, n, seed, first_event, d_icol, st);
    }
  }
  cudaError_t e2 = cudaStreamSynchronize(st);
  cudaFree(buf);
  if (ms != ME_OK) return ms;
  if (e != cudaSuccess) return cuda_fail(e, "me_select_helicity_color");
  if (e2 != cudaSuccess) return cuda_fail(e2, "me_select_helicity_color");
  return ME_OK;
}

extern "C" me_status me_unweight(const double* d_weight, const double* d_me, int64_t n, double flux, uint64_t seed, uint64_t first_event,
                                 double wmax, double sums_out[3], uint8_t* d_accept, int64_t* naccept_out, void* stream) {
  if (n < 1 || d_weight == nullptr || d_me == nullptr || sums_out == nullptr || !(flux > 0)) return ME_EINVAL;
  long long na = 0;
  cudaError_t e = me::run_unweight(d_weight, d_me, n, flux, seed, first_event, wmax, sums_out, d_accept, &na, (cudaStream_t)stream);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
  if (e != cudaSuccess) return cuda_fail(e, "me_unweight");
  if (naccept_out != nullptr) *naccept_out = na;
  return ME_OK;
}

extern "C" me_status me_philox_uniform(uint64_t seed, uint64_t first_event, int64_t n, int per_event, double* d_rnd, void* stream) {
  if (n < 0 || per_event < 1 || (n > 0 && d_rnd == nullptr)) return ME_EINVAL;
  if ((uintptr_t)d_rnd & 15) return ME_EALIGN;
  ME_CUDA(me::launch_philox(seed, first_event, n, per_event, d_rnd, (cudaStream_t)stream), "philox");
  return ME_OK;
}

extern "C" me_status me_rambo(const me_ctx* c, double sqrt_s, const double* d_rnd, int64_t n, double* d_mom, double* d_wt, void* stream) {
  if (c == nullptr || n < 0 || !(sqrt_s > 0)) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_rnd == nullptr || d_mom == nullptr) return ME_EINVAL;
  if (((uintptr_t)d_rnd & 15) || ((uintptr_t)d_mom & 15)) return ME_EALIGN;
  const int nf = c->info.npar - 2;
  double msum = 0; for (int k = 0; k < nf; ++k) msum += c->info.mass[2 + k];
  if (!(msum < sqrt_s)) return ME_EINVAL;
  ME_CUDA(me::launch_rambo(nf, c->info.mass + 2, sqrt_s, d_rnd, n, d_mom, d_wt, (cudaStream_t)stream), "rambo");
  return ME_OK;
}

extern "C" me_status me_fma_peak(int fp64, double* out) {
  if (out == nullptr) return ME_EINVAL;
  ME_CUDA(me::run_fma_peak(fp64, out), "fma peak");
  return ME_OK;
}
