// Device functions shared by the stage kernels: geometry of an affine simplex, the Hermite-moment system matrices,
// the upwind flux in closed form, the collocated relaxation and the SARK output combination.
#pragma once
#include "alegb_internal.h"

namespace alegb {

#define ALEGB_SQRT2 1.4142135623730950488
#define ALEGB_SQRT3 1.7320508075688772935

// Geometric factors of one affine simplex from its moved vertices (L193).
//   vg = (d xi_a / d x_d, a-major) then J;   sg[f] = (unit outward normal, sJ, Fscale = sJ/J)
// 2-D faces: f1 v1->v2, f2 v2->v3, f3 v3->v1.  3-D faces: f1 t=-1, f2 s=-1, f3 r+s+t=-1, f4 r=-1.
template <int DIM>
__device__ __forceinline__ void element_geometry(const double (*X)[DIM], double* vg, double* sg) {
  if constexpr (DIM == 2) {
    const double xr = 0.5 * (X[1][0] - X[0][0]), yr = 0.5 * (X[1][1] - X[0][1]);
    const double xs = 0.5 * (X[2][0] - X[0][0]), ys = 0.5 * (X[2][1] - X[0][1]);
    const double J = xr * ys - xs * yr;
    const double iJ = 1.0 / J;
    vg[0] = ys * iJ; vg[1] = -xs * iJ;   // r_x r_y
    vg[2] = -yr * iJ; vg[3] = xr * iJ;   // s_x s_y
    vg[4] = J;
    const double nx[3] = {yr, ys - yr, -ys}, ny[3] = {-xr, xr - xs, xs};
#pragma unroll
    for (int f = 0; f < 3; ++f) {
      const double sJ = sqrt(nx[f] * nx[f] + ny[f] * ny[f]);
      sg[f * 4 + 0] = nx[f] / sJ; sg[f * 4 + 1] = ny[f] / sJ; sg[f * 4 + 2] = sJ; sg[f * 4 + 3] = sJ * iJ;
    }
  } else {
    const double xr = 0.5 * (X[1][0] - X[0][0]), yr = 0.5 * (X[1][1] - X[0][1]), zr = 0.5 * (X[1][2] - X[0][2]);
    const double xs = 0.5 * (X[2][0] - X[0][0]), ys = 0.5 * (X[2][1] - X[0][1]), zs = 0.5 * (X[2][2] - X[0][2]);
    const double xt = 0.5 * (X[3][0] - X[0][0]), yt = 0.5 * (X[3][1] - X[0][1]), zt = 0.5 * (X[3][2] - X[0][2]);
    const double c00 = ys * zt - zs * yt, c01 = xs * zt - zs * xt, c02 = xs * yt - ys * xt;
    const double J = xr * c00 - yr * c01 + zr * c02;
    const double iJ = 1.0 / J;
    const double rx = c00 * iJ, ry = -c01 * iJ, rz = c02 * iJ;
    const double sx = -(yr * zt - zr * yt) * iJ, sy = (xr * zt - zr * xt) * iJ, sz = -(xr * yt - yr * xt) * iJ;
    const double tx = (yr * zs - zr * ys) * iJ, ty = -(xr * zs - zr * xs) * iJ, tz = (xr * ys - yr * xs) * iJ;
    vg[0] = rx; vg[1] = ry; vg[2] = rz; vg[3] = sx; vg[4] = sy; vg[5] = sz; vg[6] = tx; vg[7] = ty; vg[8] = tz;
    vg[9] = J;
    const double nx[4] = {-tx, -sx, rx + sx + tx, -rx};
    const double ny[4] = {-ty, -sy, ry + sy + ty, -ry};
    const double nz[4] = {-tz, -sz, rz + sz + tz, -rz};
#pragma unroll
    for (int f = 0; f < 4; ++f) {
      const double nn = sqrt(nx[f] * nx[f] + ny[f] * ny[f] + nz[f] * nz[f]);
      sg[f * 5 + 0] = nx[f] / nn; sg[f * 5 + 1] = ny[f] / nn; sg[f * 5 + 2] = nz[f] / nn;
      sg[f * 5 + 3] = nn * J; sg[f * 5 + 4] = nn;
    }
  }
}

// P1 interpolation of the element's vertex velocities to a node: v_G = sum_v lambda_v v_v.
template <int DIM>
__device__ __forceinline__ void node_velocity(const double* lam, const double* vvel, double* vG) {
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    double s = 0.0;
#pragma unroll
    for (int v = 0; v <= DIM; ++v) s = fma(lam[v], vvel[v * DIM + d], s);
    vG[d] = s;
  }
}

// y_k = sum_d sum_j (A^_d)_{kj} in(d, j): the Hermite-recurrence matrices of the moment system (readings R1, R3;
// PAPER.md:L36-43 with the blank A_x reconstructed from v h_i = sqrt(i+1) h_{i+1} + sqrt(i) h_{i-1}).
template <int DIM, class In>
__device__ __forceinline__ void hermite_apply(In in, double* y) {
  if constexpr (DIM == 2) {
    y[0] = in(0, 1) + in(1, 2);
    y[1] = in(0, 0) + ALEGB_SQRT2 * in(0, 4) + in(1, 3);
    y[2] = in(0, 3) + in(1, 0) + ALEGB_SQRT2 * in(1, 5);
    y[3] = in(0, 2) + in(1, 1);
    y[4] = ALEGB_SQRT2 * in(0, 1);
    y[5] = ALEGB_SQRT2 * in(1, 2);
  } else {
    y[0] = in(0, 1) + in(1, 2) + in(2, 3);
    y[1] = in(0, 0) + ALEGB_SQRT2 * in(0, 7) + in(1, 4) + in(2, 5);
    y[2] = in(0, 4) + in(1, 0) + ALEGB_SQRT2 * in(1, 8) + in(2, 6);
    y[3] = in(0, 5) + in(1, 6) + in(2, 0) + ALEGB_SQRT2 * in(2, 9);
    y[4] = in(0, 2) + in(1, 1);
    y[5] = in(0, 3) + in(2, 1);
    y[6] = in(1, 3) + in(2, 2);
    y[7] = ALEGB_SQRT2 * in(0, 1);
    y[8] = ALEGB_SQRT2 * in(1, 2);
    y[9] = ALEGB_SQRT2 * in(2, 3);
  }
}

template <int DIM>
__device__ __forceinline__ void normal_apply(const double* nh, const double* x, double* y) {
  hermite_apply<DIM>([&](int d, int j) { return nh[d] * x[j]; }, y);
}

// N~(q) of PAPER.md:L115 evaluated at a node (collocation, reading R8); invtau = 1/tau.
template <int DIM>
__device__ __forceinline__ void relaxation(const double* q, double invtau, double* nt) {
  const double s = invtau / q[0];
  const double r = s * (1.0 / ALEGB_SQRT2);
  if constexpr (DIM == 2) {
    nt[0] = nt[1] = nt[2] = 0.0;
    nt[3] = q[1] * q[2] * s;
    nt[4] = q[1] * q[1] * r;
    nt[5] = q[2] * q[2] * r;
  } else {
    nt[0] = nt[1] = nt[2] = nt[3] = 0.0;
    nt[4] = q[1] * q[2] * s;
    nt[5] = q[1] * q[3] * s;
    nt[6] = q[2] * q[3] * s;
    nt[7] = q[1] * q[1] * r;
    nt[8] = q[2] * q[2] * r;
    nt[9] = q[3] * q[3] * r;
  }
}

// a4 at node n of element e: the collocated N~(q) (reading R8), or -- alegb_set_relaxation(CUBATURE) -- the
// cubature-projected term R = P N~(I q) that cubature.cu left in a.relax_cub (eq. 9 last term, L197).
template <int DIM>
__device__ __forceinline__ void relaxation_term(const StageArgs& a, const double* q, int64_t e, int n, int Np, double* nt) {
  if (a.relax_cub == nullptr) {
    relaxation<DIM>(q, a.invtau, nt);
  } else {
    constexpr int NS = DIM * (DIM + 1) / 2;
    const double* r = a.relax_cub + e * NS * Np + n;
#pragma unroll
    for (int k = 0; k <= DIM; ++k) nt[k] = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s) nt[DIM + 1 + s] = __ldg(r + s * Np);
  }
}

// Even-moment rows of A^_n applied to a vector w that lives in the first-moment (momentum) slots only.
template <int DIM>
__device__ __forceinline__ void normal_apply_odd_to_even(const double* nh, const double* w, double* y) {
  if constexpr (DIM == 2) {
    y[0] = fma(nh[0], w[0], nh[1] * w[1]);
    y[3] = fma(nh[0], w[1], nh[1] * w[0]);
    y[4] = ALEGB_SQRT2 * (nh[0] * w[0]);
    y[5] = ALEGB_SQRT2 * (nh[1] * w[1]);
  } else {
    y[0] = fma(nh[0], w[0], fma(nh[1], w[1], nh[2] * w[2]));
    y[4] = fma(nh[0], w[1], nh[1] * w[0]);
    y[5] = fma(nh[0], w[2], nh[2] * w[0]);
    y[6] = fma(nh[1], w[2], nh[2] * w[1]);
    y[7] = ALEGB_SQRT2 * (nh[0] * w[0]);
    y[8] = ALEGB_SQRT2 * (nh[1] * w[1]);
    y[9] = ALEGB_SQRT2 * (nh[2] * w[2]);
  }
}

// |A_n| [q] in closed form (reading R7).  A^_n couples the first moments (fields 1..DIM, "odd") only to the zeroth
// and second moments ("even"): A^_n = [[0, B^T], [B, 0]] with B^T B = I + 2 n n^T for every unit n (its spectrum
// {1, 1(,1), 3} is the squared non-zero spectrum {+-1, +-sqrt3} of A^_n).  Hence
//   |A^_n| odd  = (B^T B)^{1/2}  x_odd       = x_odd + (sqrt3 - 1)(n . x_odd) n
//   |A^_n| even = B (B^T B)^{-1/2} B^T x_even = B ( y + (1/sqrt3 - 1)(n . y) n ),   y = B^T x_even = (A^_n x)_odd
// which equals the polynomial form a A^_n^2 + b A^_n^4, a = (9 - sqrt3)/6, b = (sqrt3 - 3)/6, at a third of the work.
// Returns y1 = A^_n dq too.
template <int DIM>
__device__ __forceinline__ void abs_normal_apply(const double* nh, const double* dq, double* y1, double* absA) {
  normal_apply<DIM>(nh, dq, y1);
  double nm = 0.0, ny = 0.0;
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    nm = fma(nh[d], dq[1 + d], nm);
    ny = fma(nh[d], y1[1 + d], ny);
  }
  nm *= ALEGB_SQRT3 - 1.0;
  ny *= 1.0 / ALEGB_SQRT3 - 1.0;
  double w[DIM];
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    absA[1 + d] = fma(nm, nh[d], dq[1 + d]);
    w[d] = fma(ny, nh[d], y1[1 + d]);
  }
  normal_apply_odd_to_even<DIM>(nh, w, absA);
}

// Lifted-flux integrand at one face node (eq. 7 in the physical sign of reading R2, split upwinding R7):
//   Fscale ( -A_n^- [q] + max(v_n, 0) [q] ),  [q] = q+ - q-,  A_n^- = (A_n - |A_n|)/2,  A_n = c A^_n.
template <int DIM>
__device__ __forceinline__ void upwind_flux(const double* qM, const double* qP, const double* nh, double c, double vn,
                                            double Fscale, double* fl) {
  constexpr int Nf = DIM == 2 ? 6 : 10;
  // (|A^_n| - A^_n)[q] without forming either: with y = (A^_n [q])_odd = B^T [q]_even (see abs_normal_apply)
  //   odd rows :  [q]_odd + (sqrt3 - 1)(n . [q]_odd) n - y
  //   even rows:  B ( y + (1/sqrt3 - 1)(n . y) n ) - B [q]_odd  =  B ( y + (1/sqrt3 - 1)(n . y) n - [q]_odd )
  double dq[Nf], y1[Nf], r[Nf];
#pragma unroll
  for (int k = 0; k < Nf; ++k) dq[k] = qP[k] - qM[k];
  normal_apply<DIM>(nh, dq, y1);   // only the odd rows 1..DIM are used; the rest is dead code
  double nm = 0.0, ny = 0.0;
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    nm = fma(nh[d], dq[1 + d], nm);
    ny = fma(nh[d], y1[1 + d], ny);
  }
  nm *= ALEGB_SQRT3 - 1.0;
  ny *= 1.0 / ALEGB_SQRT3 - 1.0;
  double z[DIM];
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    r[1 + d] = fma(nm, nh[d], dq[1 + d]) - y1[1 + d];
    z[d] = fma(ny, nh[d], y1[1 + d]) - dq[1 + d];
  }
  normal_apply_odd_to_even<DIM>(nh, z, r);
  const double hcF = Fscale * (0.5 * c), vpF = Fscale * fmax(vn, 0.0);
#pragma unroll
  for (int k = 0; k < Nf; ++k) fl[k] = fma(hcF, r[k], vpF * dq[k]);
}

// Directional piece of the flux for the absorbing layer (reading R12):
//   Fscale ( -1/2 n_d c A^_d [q] + 1/2 n_d^2 |A_n| [q] )
template <int DIM>
__device__ __forceinline__ void directional_flux(int dd, const double* qM, const double* qP, const double* nh, double c,
                                                 double Fscale, double* fl) {
  constexpr int Nf = DIM == 2 ? 6 : 10;
  double dq[Nf], y1[Nf], absA[Nf], ad[Nf];
#pragma unroll
  for (int k = 0; k < Nf; ++k) dq[k] = qP[k] - qM[k];
  abs_normal_apply<DIM>(nh, dq, y1, absA);
  hermite_apply<DIM>([&](int d, int j) { return d == dd ? dq[j] : 0.0; }, ad);
  double nd = 0.0;
#pragma unroll
  for (int d = 0; d < DIM; ++d) if (d == dd) nd = nh[d];
  const double hc = 0.5 * c;
#pragma unroll
  for (int k = 0; k < Nf; ++k) fl[k] = Fscale * hc * (nd * nd * absA[k] - nd * ad[k]);
}

// a6: outputs of one fused stage for one degree of freedom (StageCoef).
__device__ __forceinline__ void stage_update(const StageArgs& a, int k, int64_t idx, double F) {
  if (a.F_out) a.F_out[idx] = F;
  if (a.q_out == nullptr && a.acc_out == nullptr) return;
  const double qn = a.q_n ? a.q_n[idx] : 0.0;
  const double f0 = a.F0_in ? a.F0_in[idx] : 0.0;
  const double ac = a.acc_in ? a.acc_in[idx] : 0.0;
  if (a.q_out) {
    double v = a.coef.cq_n[k] * qn;
    v = fma(a.coef.cq_f0[k], f0, v);
    v = fma(a.coef.cq_acc, ac, v);
    a.q_out[idx] = fma(a.coef.cq_f[k], F, v);
  }
  if (a.acc_out) {
    double v = a.coef.ca_n[k] * qn;
    v = fma(a.coef.ca_f0[k], f0, v);
    v = fma(a.coef.ca_acc, ac, v);
    a.acc_out[idx] = fma(a.coef.ca_f[k], F, v);
  }
}

}  // namespace alegb
