// me_api.cu — the C-ABI boundary declared in include/me.h: context, helicity filtering, dispatch.
// Host logic only; every arithmetic step of the path runs in the kernels (hel_amp.cuh, epem.cu,
// gen_*.cu, rng_rambo.cu).  No CPU fallback: without a CUDA device every entry point returns ME_ECUDA.
#include <stdlib.h>
#include "../../include/me.h"
#include "kernels.h"
#define ME_HEL_PER_CTA_HOST 4     // = ME_HEL_PER_CTA of csrc/multi.h (helicities one CTA of a staged diagram kernel loops over)

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

struct me_ctx {
  me_process process;
  me_sm_params prm;
  me_info info;
  int device;                    // the device that was current at me_create: every entry point runs there
  int nsm;                       // its multiprocessor count
  const me::ProcTable* tab;      // null for e+e-
  me::EpemCouplings epem;
  double norm_hel, inv_avg;
  unsigned char* d_hels_all;     // [ncomb] 0..ncomb-1
  unsigned char* d_hels_good;    // [ngood]
  int ngood;
  unsigned char* d_hels_half;    // parity pairing: one helicity of every good pair {h, ~h}
  int nhalf;                     // 0 = pairing not applicable to the current mask
  unsigned char* d_hels_gray;    // ME_OPT_SHARE_CURRENTS: the good helicities in the order the sharing kernels walk them (grouped and
  unsigned char* d_hels_gray_half;   // padded with 255 where the process groups by gluon helicities); ngray / ngray_half entries
  int ngray, ngray_half;
  bool pairing;                  // option ME_OPT_PARITY_PAIRING
  bool share;                    // option ME_OPT_SHARE_CURRENTS
  uint64_t mask[2];
  bool filtered;
  void* scratch; size_t scratch_bytes;   // jamp staging of the multi-kernel process / cached currents of the sharing kernel
  void* work; size_t work_bytes;         // workspace of me_filter_helicities / me_select_helicity_color (grown lazily)
  double* d_color_d; float* d_color_f;   // colour-matrix numerators on `device` (multi-kernel process only)
  // calls on one context share scratch / work: a call issued on another stream than the previous one first waits for it
  cudaEvent_t ev_run; cudaStream_t last_stream; bool ran;
  // me_compute_host: two device slices of momenta / MEs, a stream per copy direction, events (all created on first use)
  bool host_ready;
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

// Every entry point that takes a context runs on the context's device: if another device is current it is switched
// for the duration of the call and restored on return (include/me.h "Devices").
struct DeviceGuard {
  int prev; bool switched; cudaError_t err;
  explicit DeviceGuard(int want) : prev(-1), switched(false), err(cudaSuccess) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != want) { err = cudaSetDevice(want); switched = err == cudaSuccess; }
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define ME_ON_DEVICE(c) DeviceGuard guard_((c)->device); if (guard_.err != cudaSuccess) return cuda_fail(guard_.err, "device")

extern "C" const char* me_strerror(me_status s) {
  switch (s) {
    case ME_OK: return "ok";
    case ME_EINVAL: return "invalid argument";
    case ME_EPROCESS: return "unknown process";
    case ME_ENOTFILTERED: return "helicities not filtered: call me_filter_helicities or me_set_helicities first";
    case ME_EALIGN: return "device buffer not 16-byte aligned";
    case ME_ENOMEM: return "out of memory";
    case ME_ETOOLARGE: return g_errbuf;
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

static void free_device_members(me_ctx* c) {
  cudaFree(c->d_hels_all); cudaFree(c->d_hels_good); cudaFree(c->d_hels_half); cudaFree(c->d_hels_gray); cudaFree(c->d_hels_gray_half);
  cudaFree(c->scratch); cudaFree(c->work); cudaFree(c->d_color_d); cudaFree(c->d_color_f);
  if (c->ev_run != nullptr) cudaEventDestroy(c->ev_run);
}

extern "C" me_status me_create(me_process process, const me_sm_params* prm, me_ctx** out) {
  if (prm == nullptr || out == nullptr) return ME_EINVAL;
  if ((int)process < 0 || (int)process > (int)ME_GG_TTXGGG) return ME_EPROCESS;
  me_ctx* c = new (std::nothrow) me_ctx();      // value-initialised: every pointer null, every flag false
  if (c == nullptr) return ME_ENOMEM;
  c->process = process; c->prm = *prm;
  c->share = true;               // ME_OPT_SHARE_CURRENTS is on by default (exact, faster); it only acts where a sharing kernel exists
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
    I.flops_per_event_shared = t->flops_shared_event;
    I.flops_executed_per_event_shared = t->flops_executed_shared > 0 ? t->flops_executed_shared * I.ncomb + t->fixed_flops : t->flops_shared_event;
  }
  c->inv_avg = 1.0 / I.avg_denom;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, c->device);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_all, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_good, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_half, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_gray, 128);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_hels_gray_half, 128);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_run, cudaEventDisableTiming);
  if (e == cudaSuccess) {
    unsigned char all[128]; for (int i = 0; i < 128; ++i) all[i] = (unsigned char)i;
    e = cudaMemcpy(c->d_hels_all, all, 128, cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess && c->tab != nullptr && c->tab->needs_color_matrix) {
    // the colour matrix of the separate colour-sum kernels lives in buffers owned by the context, on the context's device
    const size_t nn = (size_t)I.ncolor * I.ncolor;
    float* cf = new (std::nothrow) float[nn];
    if (cf == nullptr) { free_device_members(c); delete c; return ME_ENOMEM; }
    for (size_t i = 0; i < nn; ++i) cf[i] = (float)c->tab->color_num[i];
    e = cudaMalloc(&c->d_color_d, sizeof(double) * nn);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_color_f, sizeof(float) * nn);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_color_d, c->tab->color_num, sizeof(double) * nn, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_color_f, cf, sizeof(float) * nn, cudaMemcpyHostToDevice);
    delete[] cf;
  }
  if (e != cudaSuccess) {
    free_device_members(c); delete c;
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
    return cuda_fail(e, "me_create");
  }
  *out = c;
  return ME_OK;
}

extern "C" me_status me_destroy(me_ctx* c) {
  if (c == nullptr) return ME_EINVAL;
  ME_ON_DEVICE(c);
  cudaDeviceSynchronize();
  free_device_members(c);
  if (c->host_ready) {
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

// grow a context-owned device buffer; the stream that may still use the old one is drained first
static me_status ensure_buffer(void** buf, size_t* have, size_t need, cudaStream_t last, const char* what) {
  if (need <= *have) return ME_OK;
  ME_CUDA(cudaStreamSynchronize(last), what);
  cudaFree(*buf); *buf = nullptr; *have = 0;
  cudaError_t e = cudaMalloc(buf, need);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return ME_ENOMEM; }
  ME_CUDA(e, what);
  *have = need;
  return ME_OK;
}

// a call on another stream than the previous call of this context waits for it: both use the context's scratch / workspace
// and helicity lists (include/me.h "Concurrency").  Same stream: stream order already serialises them.
static me_status order_after_previous(me_ctx* c, cudaStream_t st) {
  if (c->ran && c->last_stream != st) ME_CUDA(cudaStreamWaitEvent(st, c->ev_run, 0), "stream order");
  return ME_OK;
}
static me_status mark_ran(me_ctx* c, cudaStream_t st) {
  ME_CUDA(cudaEventRecord(c->ev_run, st), "stream order");
  c->last_stream = st; c->ran = true;
  return ME_OK;
}

// hels_gray != null selects the kernel that shares sub-tree currents across helicities (it walks the list in that order)
static me_status run(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, const unsigned char* hels, int nhel, double inv_avg,
                     double* d_me, double* d_me_hel, double* d_jamp, void* stream, const int* hel_per_event = nullptr, bool share = false,
                     bool ordered = true, size_t scratch_offset = 0, size_t scratch_total = 0) {
  if ((int)prec < 0 || (int)prec > 2) return ME_EINVAL;
  if (((uintptr_t)d_mom & 15) || ((uintptr_t)d_me & 7) || ((uintptr_t)d_me_hel & 7)) return ME_EALIGN;
  me::LaunchArgs a;
  a.mom = d_mom; a.n = n; a.npad = (n + ME_PAGE - 1) / ME_PAGE * ME_PAGE; a.hels = hels; a.nhel = nhel;
  a.mt = c->prm.mt; a.norm_hel = c->norm_hel; a.inv_avg = inv_avg;
  a.me_out = d_me; a.me_hel = d_me_hel; a.jamp_out = d_jamp; a.stream = (cudaStream_t)stream;
  a.scratch = nullptr; a.scratch_bytes = 0; a.hel_per_event = hel_per_event;
  a.color_d = c->d_color_d; a.color_f = c->d_color_f; a.nsm = c->nsm; a.share = share ? 1 : 0;
  me_status ms = ordered ? order_after_previous(c, a.stream) : ME_OK;
  if (ms != ME_OK) return ms;
  if (c->tab != nullptr && c->tab->scratch_bytes != nullptr) {
    // (me_compute_host runs alternate slices on two streams: it sizes a scratch of two slots and hands each slice its own)
    const size_t need = c->tab->scratch_bytes((int)prec, a.npad, a.share, c->nsm);
    if (need > 0) {
      if (scratch_offset + need > (scratch_total > 0 ? scratch_total : need)) return ME_EINVAL;
      ms = ensure_buffer(&c->scratch, &c->scratch_bytes, scratch_total > 0 ? scratch_total : need, c->ran ? c->last_stream : a.stream, "scratch alloc");
      if (ms != ME_OK) return ms;
      a.scratch = (char*)c->scratch + scratch_offset; a.scratch_bytes = need;
    }
  }
  cudaError_t e = c->tab != nullptr ? c->tab->launch((int)prec, a) : me::launch_epem((int)prec, a, c->epem);
  if (e != cudaSuccess) return cuda_fail(e, "kernel launch");
  return ordered ? mark_ran(c, a.stream) : ME_OK;
}

extern "C" me_status me_set_helicities(me_ctx* c, const uint64_t mask[2]) {
  if (c == nullptr || mask == nullptr) return ME_EINVAL;
  ME_ON_DEVICE(c);
  unsigned char good[128]; int ng = 0;
  for (int h = 0; h < c->info.ncomb; ++h) if (mask[h >> 6] >> (h & 63) & 1) good[ng++] = (unsigned char)h;
  if (ng == 0) return ME_EINVAL;
  // kernels of earlier calls may still read the lists (also on non-blocking streams): drain them before overwriting
  if (c->ran) ME_CUDA(cudaEventSynchronize(c->ev_run), "me_set_helicities");
  ME_CUDA(cudaMemcpy(c->d_hels_good, good, ng, cudaMemcpyHostToDevice), "me_set_helicities");
  c->ngood = ng; c->mask[0] = mask[0]; c->mask[1] = c->info.ncomb > 64 ? mask[1] : 0; c->filtered = true;
  // parity pairing (pure-QCD processes): ME_h = ME_{~h}, ~h = all helicities flipped.  Usable only if the mask is
  // closed under h -> ~h; then the helicities with particle 0 at -1 represent every pair.
  c->nhalf = 0;
  unsigned char half[64]; int nh = 0;
  if (c->tab != nullptr) {
    const int full = c->info.ncomb - 1, top = c->info.ncomb >> 1;
    bool closed = true;
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
  // current sharing (ME_OPT_SHARE_CURRENTS): the same lists in the walk order of the sharing kernel, a reflected Gray code
  // whose fastest bits are the two quark helicities (consecutive helicities differ in as few, and as rarely in gluon, bits as possible)
  c->ngray = c->ngray_half = 0;
  if (c->tab != nullptr && c->tab->gray_rank != nullptr) {
    unsigned char tmp[128], out[128];
    for (int pass = 0; pass < 2; ++pass) {
      const unsigned char* src = pass == 0 ? good : half; const int m = pass == 0 ? ng : c->nhalf;
      if (m == 0) continue;
      memcpy(tmp, src, m);
      for (int i = 1; i < m; ++i) {             // insertion sort by rank in the walk
        const unsigned char v = tmp[i]; int j = i - 1;
        while (j >= 0 && c->tab->gray_rank[tmp[j]] > c->tab->gray_rank[v]) { tmp[j + 1] = tmp[j]; --j; }
        tmp[j + 1] = v;
      }
      int len = 0;
      if (c->tab->group_mask == 0) { memcpy(out, tmp, m); len = m; }
      else {                                    // groups of equal gluon helicities, each padded with 255 to ME_HEL_PER_CTA entries
        const int keep = ~c->tab->group_mask;
        for (int i = 0; i < m; ++i) {
          if (i > 0 && (tmp[i] & keep) != (tmp[i - 1] & keep)) while (len % ME_HEL_PER_CTA_HOST) out[len++] = 255;
          out[len++] = tmp[i];
        }
        while (len % ME_HEL_PER_CTA_HOST) out[len++] = 255;
      }
      ME_CUDA(cudaMemcpy(pass == 0 ? c->d_hels_gray : c->d_hels_gray_half, out, len, cudaMemcpyHostToDevice), "me_set_helicities");
      (pass == 0 ? c->ngray : c->ngray_half) = len;
    }
  }
  return ME_OK;
}

extern "C" me_status me_set_option(me_ctx* c, me_option opt, int value) {
  if (c == nullptr) return ME_EINVAL;
  switch (opt) {
    case ME_OPT_PARITY_PAIRING: c->pairing = value != 0; return ME_OK;
    case ME_OPT_SHARE_CURRENTS: c->share = value != 0; return ME_OK;
  }
  return ME_EINVAL;
}

extern "C" me_status me_filter_helicities(me_ctx* c, const double* d_mom, int64_t n, uint64_t mask_out[2], int* ngood_out, void* stream) {
  if (c == nullptr || d_mom == nullptr || mask_out == nullptr || n < 1) return ME_EINVAL;
  ME_ON_DEVICE(c);
  const int nc = c->info.ncomb;
  cudaStream_t st = (cudaStream_t)stream;
  // workspace: ME_h [ncomb][n], then sum_h ME_h [n], then the per-helicity maxima [ncomb]
  const size_t words = (size_t)nc * n + (size_t)n + (size_t)nc;
  me_status ms = ensure_buffer(&c->work, &c->work_bytes, sizeof(double) * words, c->ran ? c->last_stream : st, "filter alloc");
  if (ms != ME_OK) return ms;
  double* d_mh = (double*)c->work; double* d_tot = d_mh + (size_t)nc * n; double* d_max = d_tot + n;
  ms = run(c, d_mom, n, ME_FP64, c->d_hels_all, nc, c->inv_avg, nullptr, d_mh, nullptr, stream);
  if (ms != ME_OK) return ms;
  // reading Q7: good <=> max_evt ME_h / sum_h' ME_h' > 1e-12; the fractions are reduced on the device (sum over h in index
  // order, IEEE division, max over events: independent of the reduction order), only ncomb doubles travel to the host
  double frac[128];
  cudaError_t e = me::launch_helicity_fractions(d_mh, nc, n, d_tot, d_max, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(frac, d_max, sizeof(double) * nc, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(e, "me_filter_helicities");
  uint64_t mask[2] = {0, 0};
  for (int h = 0; h < nc; ++h) if (frac[h] > 1e-12) mask[h >> 6] |= (uint64_t)1 << (h & 63);
  ms = me_set_helicities(c, mask);
  if (ms != ME_OK) return ms;
  mask_out[0] = mask[0]; mask_out[1] = mask[1];
  if (ngood_out != nullptr) *ngood_out = c->ngood;
  return ME_OK;
}

// the helicity list, averaging factor and kernel variant of a pass: with parity pairing half the helicities, each counted
// twice; with current sharing (processes that have such a kernel) the list in walk order
static void hel_list(const me_ctx* c, const unsigned char** hels, int* nhel, double* inv_avg, bool* share) {
  *share = c->share && c->tab != nullptr && c->tab->gray_rank != nullptr;
  if (c->pairing && c->nhalf > 0) { *hels = *share ? c->d_hels_gray_half : c->d_hels_half; *nhel = *share ? c->ngray_half : c->nhalf; *inv_avg = 2.0 * c->inv_avg; }
  else { *hels = *share ? c->d_hels_gray : c->d_hels_good; *nhel = *share ? c->ngray : c->ngood; *inv_avg = c->inv_avg; }
}

extern "C" me_status me_compute(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, double* d_me, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_me == nullptr) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  ME_ON_DEVICE(c);
  const unsigned char* hels; int nhel; double inv_avg; bool share;
  hel_list(c, &hels, &nhel, &inv_avg, &share);
  return run(c, d_mom, n, prec, hels, nhel, inv_avg, d_me, nullptr, nullptr, stream, nullptr, share);
}

// The hot path for callers that must not allocate (include/me.h): g g -> t t~ g g, currents shared across helicities, the current cache in
// a file-scope device array of the generated kernel file.  Touches no buffer of the context except its helicity list (read) and creates,
// grows or frees nothing; does not take part in the context's stream ordering (it does not use the context's scratch).
extern "C" me_status me_compute_static(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, double* d_me, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (c->process != ME_GG_TTXGG) return ME_EPROCESS;
  if ((int)prec < 0 || (int)prec > 2) return ME_EINVAL;
  if (n > (int64_t)me::static_max_events_gg_ttxgg) {
    snprintf(g_errbuf, sizeof(g_errbuf), "me_compute_static: n = %lld exceeds ME_STATIC_MAX_EVENTS = %ld (the static scratch is sized for that)",
             (long long)n, me::static_max_events_gg_ttxgg);
    return ME_ETOOLARGE;
  }
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_me == nullptr) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  if (((uintptr_t)d_mom & 15) || ((uintptr_t)d_me & 7)) return ME_EALIGN;
  ME_ON_DEVICE(c);
  me::LaunchArgs a;
  a.mom = d_mom; a.n = n; a.npad = (n + ME_PAGE - 1) / ME_PAGE * ME_PAGE;
  const bool half = c->pairing && c->nhalf > 0;           // the helicity list in walk order, as me_compute takes it with sharing on
  a.hels = half ? c->d_hels_gray_half : c->d_hels_gray; a.nhel = half ? c->ngray_half : c->ngray;
  a.mt = c->prm.mt; a.norm_hel = c->norm_hel; a.inv_avg = half ? 2.0 * c->inv_avg : c->inv_avg;
  a.me_out = d_me; a.me_hel = nullptr; a.jamp_out = nullptr; a.stream = (cudaStream_t)stream;
  a.scratch = nullptr; a.scratch_bytes = 0; a.hel_per_event = nullptr;
  a.color_d = nullptr; a.color_f = nullptr; a.nsm = c->nsm; a.share = 1;
  cudaError_t e = me::launch_gg_ttxgg_static((int)prec, a);
  if (e != cudaSuccess) return cuda_fail(e, "me_compute_static");
  return ME_OK;
}

static me_status host_init(me_ctx* c) {
  // everything is created into locals and committed to the context only when all of it exists
  cudaStream_t s[3] = {nullptr, nullptr, nullptr}; cudaEvent_t ev[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaStreamCreateWithFlags(&s[i], cudaStreamNonBlocking);
  for (int i = 0; i < 7 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming);
  if (e != cudaSuccess) {
    for (int i = 0; i < 3; ++i) if (s[i] != nullptr) cudaStreamDestroy(s[i]);
    for (int i = 0; i < 7; ++i) if (ev[i] != nullptr) cudaEventDestroy(ev[i]);
    return cuda_fail(e, "host streams");
  }
  c->s_h2d = s[0]; c->s_d2h = s[1]; c->s_comp = s[2];
  c->ev_start = ev[0];
  for (int b = 0; b < 2; ++b) { c->ev_h2d[b] = ev[1 + b]; c->ev_comp[b] = ev[3 + b]; c->ev_d2h[b] = ev[5 + b]; }
  c->host_ready = true;
  return ME_OK;
}

// Host-buffer entry (include/me.h): the batch is cut in slices of whole waves of CTAs; slice k + 1 travels host -> device on a
// copy stream while slice k is computed on the caller's stream, and the MEs of slice k travel back on a second copy stream.
extern "C" me_status me_compute_host(me_ctx* c, const double* h_mom, int64_t n, me_precision prec, double* h_me, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (h_mom == nullptr || h_me == nullptr || (int)prec < 0 || (int)prec > 2) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  ME_ON_DEVICE(c);
  cudaStream_t st = (cudaStream_t)stream;
  if (!c->host_ready) { const me_status ms = host_init(c); if (ms != ME_OK) return ms; }
  // slice = 6 CTAs of ME_BLOCK events on every SM (whole waves for 1, 2, 3 or 6 resident CTAs per SM), a multiple of the page
  // (ME_HOST_SLICE_UNITS = k: k times that; measured equal for 1, 2 and 4 on the headline workload, 1 needs the least copy bandwidth:
  // a slice of g g -> t t~ g g is 22 MB against 5.5 ms of kernel).  Every kernel ends with a drain phase in which SMs idle, so odd slices are
  // computed on a second stream: the CTAs of slice k + 1 fill the drain of slice k.  Processes whose kernels share a library-owned
  // scratch buffer (g g -> t t~ g g g; current sharing) keep all slices on one stream.
  static const int slice_units = getenv("ME_HOST_SLICE_UNITS") != nullptr ? atoi(getenv("ME_HOST_SLICE_UNITS")) : 1;
  const int64_t unit = (int64_t)c->nsm * ME_BLOCK * 6, slice = (slice_units > 0 ? slice_units : 1) * unit;
  const unsigned char* hels; int nhel; double inv_avg; bool share;
  hel_list(c, &hels, &nhel, &inv_avg, &share);
  // the staged process (scratch used by several kernels in sequence) keeps its slices on one stream; the sharing kernel only
  // needs a private scratch per slice in flight: two slots
  const bool one_stream = c->tab != nullptr && c->tab->scratch_bytes != nullptr && c->tab->scratch_bytes((int)prec, slice, 0, c->nsm) > 0;
  size_t slot_bytes = 0;
  if (!one_stream && c->tab != nullptr && c->tab->scratch_bytes != nullptr)      // one slot = what a full slice needs
    slot_bytes = (c->tab->scratch_bytes((int)prec, slice, share, c->nsm) + 255) / 256 * 256;
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
  me_status ms = order_after_previous(c, st);
  if (ms != ME_OK) return ms;
  ME_CUDA(cudaEventRecord(c->ev_start, st), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_h2d, c->ev_start, 0), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_d2h, c->ev_start, 0), "host start");
  ME_CUDA(cudaStreamWaitEvent(c->s_comp, c->ev_start, 0), "host start");
  // a failure in the middle leaves copies in flight on the caller's buffers: the internal streams are drained before the
  // error is returned, so that the caller may release its buffers
  cudaError_t e = cudaSuccess; const char* where = "";
#define HOST_TRY(call, w) if (e == cudaSuccess && ms == ME_OK) { e = (call); where = (w); }
  int k = 0;
  for (int64_t first = 0; first < n && e == cudaSuccess && ms == ME_OK; ++k) {
    const int b = k & 1;
    // the first slice is a third of a unit (one wave of two CTAs per SM): the kernels start after 1/9 of the copy time of a full slice
    const int64_t want = (k == 0 && n > slice) ? unit / 3 : slice;
    const int64_t m = n - first < want ? n - first : want;
    const int64_t mpad = (m + ME_PAGE - 1) / ME_PAGE * ME_PAGE;
    cudaStream_t cs = (b == 1 && !one_stream) ? c->s_comp : st;
    if (k >= 2) HOST_TRY(cudaStreamWaitEvent(c->s_h2d, c->ev_comp[b], 0), "host wait");      // slice k - 2 no longer reads this buffer
    HOST_TRY(cudaMemcpyAsync(c->h_mom[b], h_mom + (size_t)first * ev_words, sizeof(double) * ev_words * mpad, cudaMemcpyHostToDevice, c->s_h2d), "host h2d");
    HOST_TRY(cudaEventRecord(c->ev_h2d[b], c->s_h2d), "host h2d");
    HOST_TRY(cudaStreamWaitEvent(cs, c->ev_h2d[b], 0), "host wait");
    if (k >= 2) HOST_TRY(cudaStreamWaitEvent(cs, c->ev_d2h[b], 0), "host wait");             // the MEs of slice k - 2 have left
    if (e == cudaSuccess && ms == ME_OK)          // the slices are ordered by the events of this function (ordered = false)
      ms = run(c, c->h_mom[b], m, prec, hels, nhel, inv_avg, c->h_me[b], nullptr, nullptr, (void*)cs, nullptr, share, false, b * slot_bytes, 2 * slot_bytes);
    HOST_TRY(cudaEventRecord(c->ev_comp[b], cs), "host compute");
    HOST_TRY(cudaStreamWaitEvent(c->s_d2h, c->ev_comp[b], 0), "host wait");
    HOST_TRY(cudaMemcpyAsync(h_me + first, c->h_me[b], sizeof(double) * m, cudaMemcpyDeviceToHost, c->s_d2h), "host d2h");
    HOST_TRY(cudaEventRecord(c->ev_d2h[b], c->s_d2h), "host d2h");
    first += m;
  }
#undef HOST_TRY
  if (e != cudaSuccess || ms != ME_OK) {
    cudaStreamSynchronize(c->s_h2d); cudaStreamSynchronize(c->s_d2h); cudaStreamSynchronize(c->s_comp);
    return ms != ME_OK ? ms : cuda_fail(e, where);
  }
  // `stream` ends after everything this call enqueued: the D2H stream follows every compute event
  ME_CUDA(cudaEventRecord(c->ev_start, c->s_d2h), "host end");
  ME_CUDA(cudaStreamWaitEvent(st, c->ev_start, 0), "host end");
  return mark_ran(c, st);
}

extern "C" me_status me_compute_helicities(me_ctx* c, const double* d_mom, int64_t n, me_precision prec, double* d_me, double* d_me_hel, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_me_hel == nullptr) return ME_EINVAL;
  ME_ON_DEVICE(c);
  return run(c, d_mom, n, prec, c->d_hels_all, c->info.ncomb, c->inv_avg, d_me, d_me_hel, nullptr, stream);
}

extern "C" me_status me_compute_jamps(me_ctx* c, const double* d_mom, int64_t n, int ihel, double* d_jamp, void* stream) {
  if (c == nullptr || n < 0 || d_mom == nullptr || d_jamp == nullptr) return ME_EINVAL;
  if (c->tab == nullptr || ihel < 0 || ihel >= c->info.ncomb) return ME_EINVAL;
  if (n == 0) return ME_OK;
  ME_ON_DEVICE(c);
  return run(c, d_mom, n, ME_FP64, c->d_hels_all + ihel, 1, c->inv_avg, nullptr, nullptr, d_jamp, stream);
}

extern "C" me_status me_select_helicity_color(me_ctx* c, const double* d_mom, int64_t n, uint64_t seed, uint64_t first_event,
                                              int32_t* d_ihel, int32_t* d_icol, void* stream) {
  if (c == nullptr || n < 0) return ME_EINVAL;
  if (n == 0) return ME_OK;
  if (d_mom == nullptr || d_ihel == nullptr || d_icol == nullptr) return ME_EINVAL;
  if (!c->filtered) return ME_ENOTFILTERED;
  ME_ON_DEVICE(c);
  const int nc = c->info.ncomb, ncol = c->info.ncolor;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t words = (size_t)n * (nc > 2 * ncol ? nc : 2 * ncol);
  me_status ms = ensure_buffer(&c->work, &c->work_bytes, sizeof(double) * words, c->ran ? c->last_stream : st, "select alloc");
  if (ms != ME_OK) return ms;
  double* buf = (double*)c->work;
  ms = order_after_previous(c, st);                                                       // the workspace is shared with earlier calls
  if (ms != ME_OK) return ms;
  if (c->ngood < nc) ME_CUDA(cudaMemsetAsync(buf, 0, sizeof(double) * (size_t)nc * n, st), "select");      // masked helicities weigh 0
  ms = run(c, d_mom, n, ME_FP64, c->d_hels_good, c->ngood, c->inv_avg, nullptr, buf, nullptr, stream, nullptr, false, false);
  if (ms != ME_OK) return ms;
  ME_CUDA(me::launch_select_hel(buf, nc, n, seed, first_event, d_ihel, st), "select");
  if (c->tab == nullptr) ME_CUDA(cudaMemsetAsync(d_icol, 0, sizeof(int32_t) * n, st), "select");       // one colour structure
  else {
    ms = run(c, d_mom, n, ME_FP64, c->d_hels_all, 1, c->inv_avg, nullptr, nullptr, buf, stream, d_ihel, false, false);   // jamps of each event's own helicity
    if (ms != ME_OK) return ms;
    ME_CUDA(me::launch_select_col(buf, ncol, n, seed, first_event, d_icol, st), "select");
  }
  return mark_ran(c, st);
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
  ME_ON_DEVICE(c);
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
