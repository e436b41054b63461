// kernels.h — internal launch interface between the C-ABI layer (me_api.cu) and the per-process
// kernels (hand-written epem.cu, generated gen_*.cu).  Not part of the public boundary.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define ME_BLOCK 128   // threads per CTA of the diagram kernels (one event per thread)
#define ME_PAGE 32     // events per AoSoA page

namespace me {

// arguments common to every per-process launcher
struct LaunchArgs {
  const double* mom;          // device AoSoA momenta
  long n, npad;               // events, events rounded up to a whole page
  const unsigned char* hels;  // device list of helicity indices to evaluate
  int nhel;
  const int* hel_per_event;    // device [n] or null: if set, every event evaluates ITS OWN single helicity (nhel must be 1)
  double mt;                  // quark mass (QCD) — unused for e+e-
  double norm_hel;            // per-helicity normalisation (couplings, colour denominator)
  double inv_avg;             // 1 / averaging denominator
  double* me_out;             // [n] or null
  double* me_hel;             // [ncomb][n] or null
  double* jamp_out;           // [ncol][2][n] or null (single helicity expected)
  void* scratch;              // process-specific device scratch (gg->tt~ggg jamp staging; cached currents of the sharing kernel)
  size_t scratch_bytes;
  const double* color_d;      // device colour-matrix numerators [ncol*ncol] (processes with a separate colour-sum kernel), else null
  const float* color_f;
  int nsm;                    // multiprocessors of the context's device
  int share;                  // 1: kernel variant that shares sub-tree currents across helicities (hels is then in walk order)
  cudaStream_t stream;
};

// static description of a generated process
struct ProcTable {
  int nglu, ndiagrams, namplitudes, ncol, color_denom, nkernels;
  double flops_per_helicity[3];   // algorithmic (single pass), by me_precision
  double flops_executed[3];       // as emitted (with recomputation)
  double fixed_flops;
  const double* color_num;        // [ncol*ncol] host
  cudaError_t (*launch)(int precision, const LaunchArgs&);
  size_t (*scratch_bytes)(int precision, long npad, int share, int nsm);   // may be null; may return 0
  bool needs_color_matrix;        // the context uploads color_num for a separate colour-sum kernel
  const unsigned char* gray_rank; // [ncomb] position of every helicity in the walk of the current-sharing kernel, or null (no such kernel)
  double flops_shared_event;      // algorithmic flops per event of the sharing kernel over the full helicity set (0: none)
  int group_mask;                 // != 0: helicity bits (the quark helicities) that vary WITHIN a group of the sharing list; the entries with equal
                                  // remaining (gluon) bits are adjacent and padded with 255 to ME_HEL_PER_CTA entries (one CTA loops over one group)
  double flops_executed_shared;   // flops per helicity the sharing kernels issue over the full helicity set (0: as flops_executed)
};

extern const ProcTable tab_gg_ttx, tab_gg_ttxg, tab_gg_ttxgg, tab_gg_ttxggg;
// g g -> t t~ g g, sharing kernel on a file-scope device array instead of a.scratch (include/me.h me_compute_static): no allocation;
// a.hels in walk order (gray_rank), a.npad <= static_max_events_gg_ttxgg, only a.me_out is written
cudaError_t launch_gg_ttxgg_static(int precision, const LaunchArgs& a);
extern const long static_max_events_gg_ttxgg;

// e+ e- -> mu+ mu-: couplings passed explicitly
struct EpemCouplings { double gL, gR, mz, wz; };
cudaError_t launch_epem(int precision, const LaunchArgs&, const EpemCouplings&);
extern const double epem_flops_per_helicity;

cudaError_t launch_philox(uint64_t seed, uint64_t first_event, long n, int per_event, double* d_rnd, cudaStream_t s);
cudaError_t launch_rambo(int nfinal, const double* masses /*host, nfinal*/, double sqrt_s, const double* d_rnd, long n,
                         double* d_mom, double* d_wt, cudaStream_t s);
cudaError_t run_fma_peak(int fp64, double* tflops);
cudaError_t run_unweight(const double* d_wt, const double* d_me, long n, double flux, uint64_t seed, uint64_t first_event, double wmax_in,
                         double sums[3], unsigned char* d_accept, long long* naccept, cudaStream_t st);
cudaError_t launch_select_hel(const double* me_hel, int ncomb, long n, uint64_t seed, uint64_t first_event, int* ihel, cudaStream_t s);
// fractions of me_filter_helicities: tot[i] = sum_h me_hel[h][i] (index order), maxfrac[h] = max_i me_hel[h][i] / tot[i]
cudaError_t launch_helicity_fractions(const double* me_hel, int ncomb, long n, double* tot, double* maxfrac, cudaStream_t s);
cudaError_t launch_select_col(double* jamp, int ncol, long n, uint64_t seed, uint64_t first_event, int* icol, cudaStream_t s);

}  // namespace me
