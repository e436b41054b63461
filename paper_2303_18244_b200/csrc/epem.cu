// epem.cu — e+ e- -> mu+ mu-, s-channel photon + Z (BASELINE.json config 1).
// Hand-written: 2 diagrams, 16 helicities, 1 colour.  Particle order e+(0) e-(1) mu+(2) mu-(3), massless.
//   amp_h = (Je.Jm)/s + (JeZ.JmZ)/(s - MZ^2 + i MZ GZ),   J = L + R chiral currents, JZ = gL L + gR R
//   ME    = e^4/4 * sum_h |amp_h|^2      (relative sign of the two diagrams: DESIGN.md "cfg 1 phases")
#include "hel_amp.cuh"
#include "kernels.h"

namespace me {

const double epem_flops_per_helicity = 4 * 8 + 4 * 72 + 16 + 2 * 30 + 20;

template <typename R>
__global__ void __launch_bounds__(ME_BLOCK) k_epem(const double* __restrict__ mom, long n, long npad, const unsigned char* __restrict__ hels,
                                                   int nhel, double gL_d, double gR_d, double mz, double wz, double norm_hel, double inv_avg,
                                                   double* __restrict__ me_out, double* __restrict__ me_hel, const int* __restrict__ helpe) {
  const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= npad) return;
  const double* pm = mom + (e >> 5) * (4 * 4 * 32) + (e & 31);
  P4<double> pd[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) pd[k] = {pm[(4 * k) * 32], pm[(4 * k + 1) * 32], pm[(4 * k + 2) * 32], pm[(4 * k + 3) * 32]};
  const double s = 2.0 * pdot(pd[0], pd[1]);
  // propagators: 1/s and 1/(s - mz^2 + i mz wz)
  const double dz = s - mz * mz, gz = mz * wz, idz = 1.0 / (dz * dz + gz * gz);
  const R ps = (R)(1.0 / s), zr = (R)(dz * idz), zi = (R)(-gz * idz);
  const R gL = (R)gL_d, gR = (R)gR_d;
  SpinorBasis<R> sb[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) sb[k] = spinor_basis(pcast<R>(pd[k]), (R)0);
  double acc = 0;
  for (int ih = 0; ih < nhel; ++ih) {
    const int h = helpe != nullptr ? helpe[e < n ? e : n - 1] : hels[ih];
    const R l0 = (h & 8) ? (R)1 : (R)-1, l1 = (h & 4) ? (R)1 : (R)-1, l2 = (h & 2) ? (R)1 : (R)-1, l3 = (h & 1) ? (R)1 : (R)-1;
    const W4<R> vb = dirac_bar(spinor_v(sb[0], l0));   // incoming e+
    const W4<R> u = spinor_u(sb[1], l1);               // incoming e-
    const W4<R> v = spinor_v(sb[2], l2);               // outgoing mu+
    const W4<R> ub = spinor_ubar(sb[3], l3);           // outgoing mu-
    // chiral projections of the column spinors: P_L keeps components 0,1; P_R keeps 2,3
    const W4<R> uL = {u.r0, u.i0, u.r1, u.i1, 0, 0, 0, 0}, uR = {0, 0, 0, 0, u.r2, u.i2, u.r3, u.i3};
    const W4<R> vL = {v.r0, v.i0, v.r1, v.i1, 0, 0, 0, 0}, vR = {0, 0, 0, 0, v.r2, v.i2, v.r3, v.i3};
    const W4<R> JeL = bilinear(vb, uL), JeR = bilinear(vb, uR), JmL = bilinear(ub, vL), JmR = bilinear(ub, vR);
    W4<R> Je, Jm, JeZ, JmZ;
#define ME_COMB(o, a, b, ca, cb) \
    o.r0 = ca * a.r0 + cb * b.r0; o.i0 = ca * a.i0 + cb * b.i0; o.r1 = ca * a.r1 + cb * b.r1; o.i1 = ca * a.i1 + cb * b.i1; \
    o.r2 = ca * a.r2 + cb * b.r2; o.i2 = ca * a.i2 + cb * b.i2; o.r3 = ca * a.r3 + cb * b.r3; o.i3 = ca * a.i3 + cb * b.i3;
    ME_COMB(Je, JeL, JeR, (R)1, (R)1) ME_COMB(Jm, JmL, JmR, (R)1, (R)1)
    ME_COMB(JeZ, JeL, JeR, gL, gR) ME_COMB(JmZ, JmL, JmR, gL, gR)
#undef ME_COMB
    const Cx<R> ag = wdot(Je, Jm), az = wdot(JeZ, JmZ);
    const R ar = ag.re * ps + (az.re * zr - az.im * zi), ai = ag.im * ps + (az.re * zi + az.im * zr);
    const double meh = (double)(ar * ar + ai * ai);
    if (me_hel != nullptr && e < n) me_hel[(long)h * n + e] = meh * norm_hel;
    acc += meh;
  }
  if (me_out != nullptr && e < n) me_out[e] = acc * norm_hel * inv_avg;
}

cudaError_t launch_epem(int precision, const LaunchArgs& a, const EpemCouplings& c) {
  const int grid = (int)((a.npad + ME_BLOCK - 1) / ME_BLOCK);
  if (precision == 2)
    k_epem<float><<<grid, ME_BLOCK, 0, a.stream>>>(a.mom, a.n, a.npad, a.hels, a.nhel, c.gL, c.gR, c.mz, c.wz, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.hel_per_event);
  else
    k_epem<double><<<grid, ME_BLOCK, 0, a.stream>>>(a.mom, a.n, a.npad, a.hels, a.nhel, c.gL, c.gR, c.mz, c.wz, a.norm_hel, a.inv_avg, a.me_out, a.me_hel, a.hel_per_event);
  return cudaGetLastError();
}

}  // namespace me
