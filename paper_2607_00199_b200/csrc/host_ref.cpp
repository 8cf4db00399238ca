// Host-side setup: reference element, face connectivity, SARK coefficients.  Compiled with g++.
//
// The element matrices are the ones PAPER.md:L94-103 defines,
//     M_ij = int l_i l_j,  S^a_ij = int l_i dl_j/da,  D_a = M^-1 S^a,  LIFT = M^-1 M^f,
// for the Lagrange polynomials l_i of the Warp & Blend nodes (L75).  They are built here from a monomial basis in
// the unit-simplex coordinates u_d = (1 + r_d)/2 with closed-form simplex integrals
//     int_{unit simplex} u^a v^b w^c = a! b! c! / (a+b+c+dim)!,
// in __float128 arithmetic and rounded once to fp64.  (oracle/ uses a product-Legendre basis and Gauss-Jacobi
// quadrature in extended precision; the two constructions share nothing.)
#include "host_ref.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>

namespace alegb {

typedef __float128 qreal;

// Optimised blend parameters of the Warp & Blend construction (ref. [34] of the paper; reading R10).
static const double kAlpha2D[6] = {0.0, 0.0, 0.0, 1.4152, 0.1001, 0.2751};
static const double kAlpha3D[6] = {0.0, 0.0, 0.0, 0.0, 0.1002, 1.1332};

static const int kFaceVerts2D[3][3] = {{0, 1, -1}, {1, 2, -1}, {2, 0, -1}};
static const int kFaceVerts3D[4][3] = {{0, 1, 2}, {0, 1, 3}, {1, 2, 3}, {0, 2, 3}};

static qreal qabs(qreal x) { return x < 0 ? -x : x; }

// Legendre P_n(x), P_n'(x), P_n''(x) by the three-term recurrence.
static void legendre(int n, qreal x, qreal& p, qreal& dp, qreal& ddp) {
  qreal p0 = 1, p1 = x;
  if (n == 0) { p = 1; dp = 0; ddp = 0; return; }
  for (int k = 2; k <= n; ++k) {
    qreal pk = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
    p0 = p1; p1 = pk;
  }
  p = p1;
  // (1-x^2) P_n' = n (P_{n-1} - x P_n);  (1-x^2) P_n'' = 2 x P_n' - n(n+1) P_n
  dp = n * (p0 - x * p1) / (1 - x * x);
  ddp = (2 * x * dp - (qreal)n * (n + 1) * p1) / (1 - x * x);
}

// Legendre-Gauss-Lobatto points of order N: +-1 and the zeros of P_N'.
static std::vector<qreal> lgl_points(int N) {
  std::vector<qreal> x(N + 1);
  x[0] = -1; x[N] = 1;
  for (int i = 1; i < N; ++i) {
    qreal xi = -(qreal)cosl(M_PIl * i / N);
    for (int it = 0; it < 100; ++it) {
      qreal p, dp, ddp;
      legendre(N, xi, p, dp, ddp);
      qreal dx = dp / ddp;
      xi -= dx;
      if (qabs(dx) < (qreal)1e-32L) break;
    }
    x[i] = xi;
  }
  return x;
}

// 1-D warp: interpolant through the equispaced points of (LGL - equispaced).
static qreal warp_1d(int N, const std::vector<qreal>& lgl, qreal rho) {
  qreal w = 0;
  for (int i = 0; i <= N; ++i) {
    qreal ri = -1 + (qreal)2 * i / N, li = 1;
    for (int j = 0; j <= N; ++j)
      if (j != i) { qreal rj = -1 + (qreal)2 * j / N; li *= (rho - rj) / (ri - rj); }
    w += (lgl[i] - ri) * li;
  }
  return w;
}

// In-place Gauss-Jordan inverse with partial pivoting.
static bool invert(std::vector<qreal>& A, int n) {
  std::vector<qreal> B(n * n, 0);
  for (int i = 0; i < n; ++i) B[i * n + i] = 1;
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (qabs(A[r * n + c]) > qabs(A[piv * n + c])) piv = r;
    if (qabs(A[piv * n + c]) < (qreal)1e-60L) return false;
    if (piv != c) for (int k = 0; k < n; ++k) { std::swap(A[piv * n + k], A[c * n + k]); std::swap(B[piv * n + k], B[c * n + k]); }
    qreal inv = 1 / A[c * n + c];
    for (int k = 0; k < n; ++k) { A[c * n + k] *= inv; B[c * n + k] *= inv; }
    for (int r = 0; r < n; ++r) {
      if (r == c) continue;
      qreal f = A[r * n + c];
      if (f == 0) continue;
      for (int k = 0; k < n; ++k) { A[r * n + k] -= f * A[c * n + k]; B[r * n + k] -= f * B[c * n + k]; }
    }
  }
  A.swap(B);
  return true;
}

static qreal factorial(int n) { qreal f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }
static qreal qpow(qreal x, int e) { qreal r = 1; for (int i = 0; i < e; ++i) r *= x; return r; }

// exponents of the monomials of total degree <= N in nd variables
static std::vector<std::vector<int>> exponents(int nd, int N) {
  std::vector<std::vector<int>> ex;
  if (nd == 0) { ex.push_back({}); return ex; }
  if (nd == 1) { for (int a = 0; a <= N; ++a) ex.push_back({a}); return ex; }
  if (nd == 2) { for (int a = 0; a <= N; ++a) for (int b = 0; a + b <= N; ++b) ex.push_back({a, b}); return ex; }
  for (int a = 0; a <= N; ++a) for (int b = 0; a + b <= N; ++b) for (int c = 0; a + b + c <= N; ++c) ex.push_back({a, b, c});
  return ex;
}

// Gram matrix of the monomials on the simplex {u >= 0, sum u <= 1} scaled to the [-1,1]-vertex simplex: 2^nd * int.
static std::vector<qreal> gram(int nd, const std::vector<std::vector<int>>& ex) {
  int n = (int)ex.size();
  std::vector<qreal> G(n * n);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      qreal num = 1; int tot = nd;
      for (int d = 0; d < nd; ++d) { int e = ex[i][d] + ex[j][d]; num *= factorial(e); tot += e; }
      G[i * n + j] = qpow(2, nd) * num / factorial(tot);
    }
  return G;
}

// C = A(n x k) * B(k x m)
static std::vector<qreal> matmul(const std::vector<qreal>& A, const std::vector<qreal>& B, int n, int k, int m) {
  std::vector<qreal> C(n * m, 0);
  for (int i = 0; i < n; ++i) for (int l = 0; l < k; ++l) { qreal a = A[i * k + l]; for (int j = 0; j < m; ++j) C[i * m + j] += a * B[l * m + j]; }
  return C;
}
static std::vector<qreal> transpose(const std::vector<qreal>& A, int n, int m) {
  std::vector<qreal> T(n * m);
  for (int i = 0; i < n; ++i) for (int j = 0; j < m; ++j) T[j * n + i] = A[i * m + j];
  return T;
}

// Jacobi polynomial P_n^{(a,0)}(x) and its derivative: three-term recurrence and
// (2n+a)(1-x^2) P_n' = n (a - (2n+a) x) P_n + 2 (n+a) n P_{n-1}   (Abramowitz & Stegun 22.7.1, 22.8.1 with beta = 0)
static void jacobi_a0(int n, int a, qreal x, qreal& p, qreal& dp) {
  if (n == 0) { p = 1; dp = 0; return; }
  qreal p0 = 1, p1 = ((qreal)a + (qreal)(a + 2) * x) / 2;
  for (int k = 1; k < n; ++k) {
    const qreal c = 2 * k + a;
    const qreal A1 = 2 * (qreal)(k + 1) * (k + a + 1) * c;
    const qreal A2 = (c + 1) * (qreal)(a * a);
    const qreal A3 = c * (c + 1) * (c + 2);
    const qreal A4 = 2 * (qreal)(k + a) * k * (c + 2);
    const qreal pk = ((A2 + A3 * x) * p1 - A4 * p0) / A1;
    p0 = p1; p1 = pk;
  }
  p = p1;
  dp = (n * ((qreal)a - (qreal)(2 * n + a) * x) * p1 + 2 * (qreal)(n + a) * n * p0) / ((qreal)(2 * n + a) * (1 - x * x));
}

// n-point Gauss-Jacobi rule for the weight (1-x)^a on [-1,1]: zeros of P_n^{(a,0)} by Newton iteration with
// deflation, weights w_i = 2^{a+1} / ((1 - x_i^2) P_n'(x_i)^2).  Exact to degree 2n-1.
static void gauss_jacobi_a0(int n, int a, std::vector<qreal>& x, std::vector<qreal>& w) {
  x.assign(n, 0); w.assign(n, 0);
  for (int k = 0; k < n; ++k) {
    qreal r = -(qreal)cosl(M_PIl * (2 * k + 1) / (2.0L * n));
    if (k > 0) r = (r + x[k - 1]) / 2;
    for (int it = 0; it < 200; ++it) {
      qreal s = 0;
      for (int j = 0; j < k; ++j) s += 1 / (r - x[j]);
      qreal p, dp;
      jacobi_a0(n, a, r, p, dp);
      const qreal dx = -p / (dp - s * p);
      r += dx;
      if (qabs(dx) < (qreal)1e-30L) break;
    }
    x[k] = r;
  }
  for (int k = 0; k < n; ++k) {
    qreal p, dp;
    jacobi_a0(n, a, x[k], p, dp);
    w[k] = qpow(2, a + 1) / ((1 - x[k] * x[k]) * dp * dp);
  }
}

bool build_cubature(const RefElement& ref, int degree, Cubature& out, std::string& err) {
  const int dim = ref.dim, N = ref.N, Np = ref.Np, nv = dim + 1;
  if (Np == 0) { err = "reference element not built"; return false; }
  if (degree < 2 * N) { err = "cubature degree must be at least 2N"; return false; }
  const int n = degree / 2 + 1;
  std::vector<qreal> xa, wa, xb, wb, xc, wc;
  gauss_jacobi_a0(n, 0, xa, wa);
  gauss_jacobi_a0(n, 1, xb, wb);
  if (dim == 3) gauss_jacobi_a0(n, 2, xc, wc);
  // collapsed coordinates: 2-D r = (1+a)(1-b)/2 - 1, s = b, dr ds = (1-b)/2 da db;
  // 3-D r = (1+a)(1-b)(1-c)/4 - 1, s = (1+b)(1-c)/2 - 1, t = c, dr ds dt = (1-b)(1-c)^2/8 da db dc
  const int Nc = dim == 2 ? n * n : n * n * n;
  std::vector<qreal> pts(Nc * dim), wts(Nc);
  int q = 0;
  for (int ia = 0; ia < n; ++ia)
    for (int ib = 0; ib < n; ++ib) {
      if (dim == 2) {
        pts[q * 2 + 0] = (1 + xa[ia]) * (1 - xb[ib]) / 2 - 1;
        pts[q * 2 + 1] = xb[ib];
        wts[q++] = wa[ia] * wb[ib] / 2;
      } else {
        for (int ic = 0; ic < n; ++ic) {
          pts[q * 3 + 0] = (1 + xa[ia]) * (1 - xb[ib]) * (1 - xc[ic]) / 4 - 1;
          pts[q * 3 + 1] = (1 + xb[ib]) * (1 - xc[ic]) / 2 - 1;
          pts[q * 3 + 2] = xc[ic];
          wts[q++] = wa[ia] * wb[ib] * wc[ic] / 8;
        }
      }
    }
  // monomial basis in u = (1 + r)/2 as in build_reference: V at the nodes, Vc at the cubature points
  auto ex = exponents(dim, N);
  std::vector<qreal> V(Np * Np), Vc(Nc * Np);
  for (int i = 0; i < Np; ++i)
    for (int m = 0; m < Np; ++m) {
      qreal v = 1;
      for (int d = 0; d < dim; ++d) v *= qpow((qreal)ref.lam[i * nv + d + 1], ex[m][d]);
      V[i * Np + m] = v;
    }
  for (int c = 0; c < Nc; ++c)
    for (int m = 0; m < Np; ++m) {
      qreal v = 1;
      for (int d = 0; d < dim; ++d) v *= qpow((1 + pts[c * dim + d]) / 2, ex[m][d]);
      Vc[c * Np + m] = v;
    }
  std::vector<qreal> Vinv = V;
  if (!invert(Vinv, Np)) { err = "singular Vandermonde"; return false; }
  std::vector<qreal> Ginv = gram(dim, ex);
  if (!invert(Ginv, Np)) { err = "singular Gram matrix"; return false; }
  std::vector<qreal> Minv = matmul(matmul(V, Ginv, Np, Np, Np), transpose(V, Np, Np), Np, Np, Np);
  std::vector<qreal> I = matmul(Vc, Vinv, Nc, Np, Np);                      // [Nc][Np]
  std::vector<qreal> ItW = transpose(I, Nc, Np);                            // [Np][Nc]
  for (int j = 0; j < Np; ++j) for (int c = 0; c < Nc; ++c) ItW[j * Nc + c] *= wts[c];
  std::vector<qreal> P = matmul(Minv, ItW, Np, Np, Nc);                     // [Np][Nc]
  out.degree = degree; out.Nc = Nc;
  out.rst.resize(dim * Nc); out.w.resize(Nc); out.I.resize(Nc * Np); out.P.resize(Np * Nc);
  for (int c = 0; c < Nc; ++c) {
    out.w[c] = (double)wts[c];
    for (int d = 0; d < dim; ++d) out.rst[d * Nc + c] = (double)pts[c * dim + d];
  }
  for (int x = 0; x < Nc * Np; ++x) { out.I[x] = (double)I[x]; out.P[x] = (double)P[x]; }
  return true;
}

int RefElement::node_of(const int* wts) const {
  for (int i = 0; i < Np; ++i) {
    bool same = true;
    for (int v = 0; v <= dim; ++v) if (lattice[i * (dim + 1) + v] != wts[v]) { same = false; break; }
    if (same) return i;
  }
  return -1;
}

bool build_reference(int dim, int N, RefElement& ref, std::string& err) {
  if ((dim != 2 && dim != 3) || N < 1 || N > 5) { err = "dim must be 2 or 3 and 1 <= N <= 5"; return false; }
  ref.dim = dim; ref.N = N; ref.Nfaces = dim + 1;
  const int nv = dim + 1;
  // ---- lattice, order: weight of vertex 2 fastest, then vertex 3, then vertex 4
  ref.lattice.clear();
  if (dim == 2) {
    for (int j = 0; j <= N; ++j) for (int i = 0; i + j <= N; ++i) { ref.lattice.push_back(N - i - j); ref.lattice.push_back(i); ref.lattice.push_back(j); }
  } else {
    for (int k = 0; k <= N; ++k) for (int j = 0; j + k <= N; ++j) for (int i = 0; i + j + k <= N; ++i) {
      ref.lattice.push_back(N - i - j - k); ref.lattice.push_back(i); ref.lattice.push_back(j); ref.lattice.push_back(k);
    }
  }
  const int Np = (int)ref.lattice.size() / nv;
  ref.Np = Np;
  // ---- Warp & Blend in barycentric form (L75): every edge (a,b) pushes along itself by
  //      4 la lb w(rho)/(1-rho^2) (1 + (alpha l_rest)^2), rho = lb - la; lambda_b += push/2, lambda_a -= push/2
  const double alpha = dim == 2 ? kAlpha2D[N] : kAlpha3D[N];
  std::vector<qreal> lgl = lgl_points(N);
  std::vector<qreal> lam0(Np * nv), lam(Np * nv);
  for (int i = 0; i < Np * nv; ++i) lam0[i] = lam[i] = (qreal)ref.lattice[i] / N;
  for (int a = 0; a < nv; ++a)
    for (int b = a + 1; b < nv; ++b)
      for (int i = 0; i < Np; ++i) {
        qreal la = lam0[i * nv + a], lb = lam0[i * nv + b];
        qreal rho = lb - la, den = 1 - rho * rho;
        if (qabs(den) <= (qreal)1e-12L) continue;
        qreal rest = 1 - la - lb;
        qreal push = 4 * la * lb * warp_1d(N, lgl, rho) / den * (1 + (alpha * rest) * (alpha * rest));
        lam[i * nv + b] += push / 2;
        lam[i * nv + a] -= push / 2;
      }
  ref.lam.resize(Np * nv);
  for (int i = 0; i < Np * nv; ++i) ref.lam[i] = (double)lam[i];
  ref.rst.resize(dim * Np);
  for (int d = 0; d < dim; ++d) for (int i = 0; i < Np; ++i) ref.rst[d * Np + i] = (double)(2 * lam[i * nv + d + 1] - 1);

  // ---- volume matrices
  auto ex = exponents(dim, N);
  if ((int)ex.size() != Np) { err = "internal: basis size"; return false; }
  std::vector<qreal> V(Np * Np), Vd[3];
  for (int a = 0; a < dim; ++a) Vd[a].assign(Np * Np, 0);
  for (int i = 0; i < Np; ++i)
    for (int m = 0; m < Np; ++m) {
      qreal v = 1;
      for (int d = 0; d < dim; ++d) v *= qpow(lam[i * nv + d + 1], ex[m][d]);
      V[i * Np + m] = v;
      for (int a = 0; a < dim; ++a) {
        if (ex[m][a] == 0) continue;
        qreal g = ex[m][a] * qpow(lam[i * nv + a + 1], ex[m][a] - 1);
        for (int d = 0; d < dim; ++d) if (d != a) g *= qpow(lam[i * nv + d + 1], ex[m][d]);
        Vd[a][i * Np + m] = g / 2;   // d/dr = (1/2) d/du
      }
    }
  std::vector<qreal> Vinv = V;
  if (!invert(Vinv, Np)) { err = "singular Vandermonde"; return false; }
  for (int a = 0; a < dim; ++a) {
    auto Da = matmul(Vd[a], Vinv, Np, Np, Np);
    ref.D[a].resize(Np * Np);
    for (int i = 0; i < Np * Np; ++i) ref.D[a][i] = (double)Da[i];
  }
  std::vector<qreal> G = gram(dim, ex);
  std::vector<qreal> VinvT = transpose(Vinv, Np, Np);
  std::vector<qreal> M = matmul(matmul(VinvT, G, Np, Np, Np), Vinv, Np, Np, Np);
  ref.w.assign(Np, 0);
  for (int j = 0; j < Np; ++j) { qreal s = 0; for (int i = 0; i < Np; ++i) s += M[i * Np + j]; ref.w[j] = (double)s; }
  std::vector<qreal> Ginv = G;
  if (!invert(Ginv, Np)) { err = "singular Gram matrix"; return false; }
  std::vector<qreal> Minv = matmul(matmul(V, Ginv, Np, Np, Np), transpose(V, Np, Np), Np, Np, Np);

  // ---- faces: fmask (ascending node index), face mass matrices on the face's own reference simplex, LIFT
  for (int f = 0; f < dim + 1; ++f) for (int j = 0; j < 3; ++j) ref.face_verts[f][j] = dim == 2 ? kFaceVerts2D[f][j] : kFaceVerts3D[f][j];
  ref.fmask.clear();
  for (int f = 0; f < ref.Nfaces; ++f) {
    int opp = 0;
    for (int v = 0; v < nv; ++v) { bool on = false; for (int j = 0; j < dim; ++j) if (ref.face_verts[f][j] == v) on = true; if (!on) opp = v; }
    for (int i = 0; i < Np; ++i) if (ref.lattice[i * nv + opp] == 0) ref.fmask.push_back(i);
  }
  const int Nfp = (int)ref.fmask.size() / ref.Nfaces;
  ref.Nfp = Nfp;
  auto fex = exponents(dim - 1, N);
  if ((int)fex.size() != Nfp) { err = "internal: face basis size"; return false; }
  std::vector<qreal> Gf = gram(dim - 1, fex);
  const int ncol = ref.Nfaces * Nfp;
  ref.LIFT.assign(Np * ncol, 0.0);
  ref.wface.assign(ncol, 0.0);
  for (int f = 0; f < ref.Nfaces; ++f) {
    std::vector<qreal> Vf(Nfp * Nfp);
    for (int i = 0; i < Nfp; ++i) {
      int node = ref.fmask[f * Nfp + i];
      for (int m = 0; m < Nfp; ++m) {
        qreal v = 1;
        for (int d = 0; d < dim - 1; ++d) v *= qpow(lam[node * nv + ref.face_verts[f][d + 1]], fex[m][d]);
        Vf[i * Nfp + m] = v;
      }
    }
    std::vector<qreal> Vfinv = Vf;
    if (!invert(Vfinv, Nfp)) { err = "singular face Vandermonde"; return false; }
    std::vector<qreal> Mf = matmul(matmul(transpose(Vfinv, Nfp, Nfp), Gf, Nfp, Nfp, Nfp), Vfinv, Nfp, Nfp, Nfp);
    for (int j = 0; j < Nfp; ++j) {
      qreal s = 0;
      for (int i = 0; i < Nfp; ++i) s += Mf[i * Nfp + j];
      ref.wface[f * Nfp + j] = (double)s;
    }
    for (int r = 0; r < Np; ++r)
      for (int j = 0; j < Nfp; ++j) {
        qreal s = 0;
        for (int i = 0; i < Nfp; ++i) s += Minv[r * Np + ref.fmask[f * Nfp + i]] * Mf[i * Nfp + j];
        ref.LIFT[r * ncol + f * Nfp + j] = (double)s;
      }
  }
  return true;
}

// ---------------------------------------------------------------------------------------------------------------
int build_connectivity(const RefElement& ref, int64_t K, const int32_t* EToV, const int32_t* vertex_equiv,
                       const int8_t* EToB, Connectivity& out, std::string& err) {
  const int dim = ref.dim, nv = dim + 1, Nfaces = ref.Nfaces, Nfp = ref.Nfp, Np = ref.Np;
  if (K * (int64_t)Np >= (int64_t)1 << 31) { err = "mesh too large for int32 node indices"; return -2; }
  std::vector<int32_t> ids((size_t)K * nv);
  for (int64_t i = 0; i < K * nv; ++i) ids[i] = vertex_equiv ? vertex_equiv[EToV[i]] : EToV[i];
  for (int64_t e = 0; e < K; ++e)
    for (int a = 0; a < nv; ++a)
      for (int b = a + 1; b < nv; ++b)
        if (ids[e * nv + a] == ids[e * nv + b]) {
          err = "an element touches the same (periodic class of a) vertex twice: a periodic direction needs at least 3 cells";
          return -2;
        }
  struct FaceKey { int32_t v[3]; int64_t ef; };
  std::vector<FaceKey> keys((size_t)K * Nfaces);
  for (int64_t e = 0; e < K; ++e)
    for (int f = 0; f < Nfaces; ++f) {
      FaceKey& k = keys[e * Nfaces + f];
      k.v[2] = -1;
      for (int j = 0; j < dim; ++j) k.v[j] = ids[e * nv + ref.face_verts[f][j]];
      std::sort(k.v, k.v + dim);
      k.ef = e * Nfaces + f;
    }
  std::sort(keys.begin(), keys.end(), [](const FaceKey& a, const FaceKey& b) {
    if (a.v[0] != b.v[0]) return a.v[0] < b.v[0];
    if (a.v[1] != b.v[1]) return a.v[1] < b.v[1];
    if (a.v[2] != b.v[2]) return a.v[2] < b.v[2];
    return a.ef < b.ef;
  });
  auto same = [](const FaceKey& a, const FaceKey& b) { return a.v[0] == b.v[0] && a.v[1] == b.v[1] && a.v[2] == b.v[2]; };
  out.EToE.resize((size_t)K * Nfaces); out.EToF.resize((size_t)K * Nfaces);
  for (int64_t e = 0; e < K; ++e) for (int f = 0; f < Nfaces; ++f) { out.EToE[e * Nfaces + f] = (int32_t)e; out.EToF[e * Nfaces + f] = f; }
  std::vector<char> interior((size_t)K * Nfaces, 0);
  for (size_t i = 0; i < keys.size();) {
    size_t j = i + 1;
    while (j < keys.size() && same(keys[i], keys[j])) ++j;
    if (j - i > 2) { err = "a face is shared by more than two elements (non-conforming mesh or periodic direction < 3 cells)"; return -2; }
    if (j - i == 2) {
      int64_t a = keys[i].ef, b = keys[i + 1].ef;
      out.EToE[a] = (int32_t)(b / Nfaces); out.EToF[a] = (int32_t)(b % Nfaces);
      out.EToE[b] = (int32_t)(a / Nfaces); out.EToF[b] = (int32_t)(a % Nfaces);
      interior[a] = interior[b] = 1;
    }
    i = j;
  }
  for (int64_t i = 0; i < K * Nfaces; ++i) {
    int tag = EToB ? EToB[i] : 0;
    if (interior[i] && tag != 0) { err = "EToB tags an interior face"; return -2; }
    if (!interior[i] && tag == 0) { err = "unmatched face without a boundary tag"; return -2; }
    if (tag < 0 || tag > 2) { err = "unknown boundary tag"; return -2; }
  }
  out.vmapM.resize((size_t)K * Nfaces * Nfp); out.vmapP.resize((size_t)K * Nfaces * Nfp);
  // partner tables cached per (own face, placement of the own-face vertices in the neighbour)
  std::map<int, std::vector<int>> cache;
  for (int64_t e = 0; e < K; ++e)
    for (int f = 0; f < Nfaces; ++f) {
      const int64_t ef = e * Nfaces + f;
      for (int m = 0; m < Nfp; ++m) out.vmapM[ef * Nfp + m] = (int32_t)(e * Np + ref.fmask[f * Nfp + m]);
      if (!interior[ef]) { for (int m = 0; m < Nfp; ++m) out.vmapP[ef * Nfp + m] = out.vmapM[ef * Nfp + m]; continue; }
      const int64_t en = out.EToE[ef];
      int loc[3] = {0, 0, 0}, code = f;
      for (int j = 0; j < dim; ++j) {
        int32_t id = ids[e * nv + ref.face_verts[f][j]];
        int l = -1;
        for (int v = 0; v < nv; ++v) if (ids[en * nv + v] == id) l = v;
        if (l < 0) { err = "internal: face vertex not found in neighbour"; return -2; }
        loc[j] = l; code = code * nv + l;
      }
      auto it = cache.find(code);
      if (it == cache.end()) {
        std::vector<int> partner(Nfp);
        for (int m = 0; m < Nfp; ++m) {
          int n = ref.fmask[f * Nfp + m];
          int wn[4] = {0, 0, 0, 0};
          for (int j = 0; j < dim; ++j) wn[loc[j]] = ref.lattice[n * nv + ref.face_verts[f][j]];
          partner[m] = ref.node_of(wn);
          if (partner[m] < 0) { err = "internal: partner node not found"; return -2; }
        }
        it = cache.emplace(code, partner).first;
      }
      for (int m = 0; m < Nfp; ++m) out.vmapP[ef * Nfp + m] = (int32_t)(en * Np + it->second[m]);
    }
  return 0;
}

// ---------------------------------------------------------------------------------------------------------------
// phi_k(z) = (e^z - sum_{j<k} z^j/j!) / z^k, k = 1,2,3: Taylor series for |z| < 1, closed form otherwise.
static void phi_functions(long double z, long double phi[4]) {
  if (fabsl(z) < 1.0L) {
    for (int k = 1; k <= 3; ++k) {
      long double term = 1.0L, s = 0.0L;
      for (int j = 1; j <= k; ++j) term /= j;       // 1/k!
      for (int n = 0; n < 40; ++n) { s += term; term *= z / (n + k + 1); }
      phi[k] = s;
    }
  } else {
    long double e = expl(z);
    phi[1] = (e - 1.0L) / z;
    phi[2] = (e - 1.0L - z) / (z * z);
    phi[3] = (e - 1.0L - z - z * z / 2.0L) / (z * z * z);
  }
}

void sark_coefficients(double gamma, double a[6], double b[4]) {
  // classic RK4 (Table 1, blank in PAPER.md:L119; reading R4)
  if (gamma == 0.0) {
    a[0] = 0.5; a[1] = 0.0; a[2] = 0.5; a[3] = 0.0; a[4] = 0.0; a[5] = 1.0;
    b[0] = 1.0 / 6.0; b[1] = b[2] = 1.0 / 3.0; b[3] = 1.0 / 6.0;
    return;
  }
  long double g = gamma;
  if (fabsl(g) < 2.0L) {
    // the printed formulas of L148 rewritten through phi-functions (algebraically identical, no cancellation):
    // a10 = phi1(g/2)/2; a21 = phi2(g/2); a20 = a10 - a21; a32 = 2 phi2(g); a30 = phi1(g) - a32;
    // b0 = phi1 - 3 phi2 + 4 phi3; b1 = b2 = 2 phi2 - 4 phi3; b3 = 4 phi3 - phi2   (all at g)
    long double ph[4], pf[4];
    phi_functions(g / 2.0L, ph);
    phi_functions(g, pf);
    a[0] = (double)(ph[1] / 2.0L);
    a[2] = (double)(ph[2]);
    a[1] = (double)(ph[1] / 2.0L - ph[2]);
    a[5] = (double)(2.0L * pf[2]);
    a[3] = (double)(pf[1] - 2.0L * pf[2]);
    a[4] = 0.0;
    b[0] = (double)(pf[1] - 3.0L * pf[2] + 4.0L * pf[3]);
    b[1] = b[2] = (double)(2.0L * pf[2] - 4.0L * pf[3]);
    b[3] = (double)(4.0L * pf[3] - pf[2]);
  } else {
    // the formulas exactly as printed at L148, in extended precision (no small-gamma cancellation here)
    long double eh = expl(g / 2.0L), e = expl(g), g2 = g * g, g3 = g2 * g;
    a[0] = (double)((eh - 1.0L) / g);
    a[1] = (double)((4.0L + g + eh * (g - 4.0L)) / g2);
    a[2] = (double)((-4.0L - 2.0L * g + 4.0L * eh) / g2);
    a[3] = (double)((2.0L + g + e * (g - 2.0L)) / g2);
    a[4] = 0.0;
    a[5] = (double)((-2.0L - 2.0L * g + 2.0L * e) / g2);
    b[0] = (double)((-4.0L - g + e * (g2 - 3.0L * g + 4.0L)) / g3);
    b[1] = b[2] = (double)((4.0L + 2.0L * g + e * (2.0L * g - 4.0L)) / g3);
    b[3] = (double)((-4.0L - 3.0L * g - g2 + e * (4.0L - g)) / g3);
  }
}

}  // namespace alegb
