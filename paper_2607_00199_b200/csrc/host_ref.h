// Host-side setup of the library: reference element, connectivity, SARK coefficients.
// Independent of oracle/ (shares no code with it); compiled with g++ (uses __float128).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace alegb {

// Constant per-(dim, N) data of the nodal DG discretisation.
struct RefElement {
  int dim = 0, N = 0, Np = 0, Nfp = 0, Nfaces = 0;
  std::vector<int> lattice;    // [Np][dim+1] integer barycentric weights (sum N)
  std::vector<double> lam;     // [Np][dim+1] barycentric coordinates of the Warp & Blend nodes (L192 matrix)
  std::vector<double> rst;     // [dim][Np] reference coordinates
  std::vector<double> D[3];    // [Np][Np] row-major differentiation matrices D_a = M^-1 S_a
  std::vector<double> LIFT;    // [Np][Nfaces*Nfp]
  std::vector<double> w;       // [Np] 1^T M
  std::vector<double> wface;   // [Nfaces][Nfp] 1^T M^f on the nodes of each face (face quadrature weights, sum 2)
  std::vector<int> fmask;      // [Nfaces][Nfp]
  int face_verts[4][3];        // local vertex numbers of each face
  int node_of(const int* weights) const;  // lattice tuple -> node index
};

// Builds everything; returns false and fills err on failure.
bool build_reference(int dim, int N, RefElement& ref, std::string& err);

struct Connectivity {
  std::vector<int32_t> EToE, EToF;      // [K][Nfaces]
  std::vector<int32_t> vmapM, vmapP;    // [K][Nfaces][Nfp], flattened node index e*Np+n
};

// Cubature rule and the interpolation / projection operators of PAPER.md:L84-86, L103:
// conical-product Gauss-Jacobi rule exact to total degree `degree` on the reference simplex,
// I_cj = phi_j(x_c), P = M^-1 I^T diag(w) (reference element: the J^e of eq. 9 cancels against (M^e)^-1).
struct Cubature {
  int degree = 0, Nc = 0;
  std::vector<double> rst;   // [dim][Nc]
  std::vector<double> w;     // [Nc], sum = measure of the reference simplex
  std::vector<double> I;     // [Nc][Np]
  std::vector<double> P;     // [Np][Nc]
};
bool build_cubature(const RefElement& ref, int degree, Cubature& out, std::string& err);

// Faces matched by (periodic classes of) vertex ids, face nodes by the vertex permutation (never by coordinates).
// Returns 0, or -2 (BAD_MESH) with err filled.
int build_connectivity(const RefElement& ref, int64_t K, const int32_t* EToV, const int32_t* vertex_equiv,
                       const int8_t* EToB, Connectivity& out, std::string& err);

// SARK4 coefficients of PAPER.md:L148 for gamma = -dt/tau, evaluated cancellation-free (reading R6).
// a = (a10, a20, a21, a30, a31, a32); gamma == 0 gives the classic RK4 tableau (reading R4).
void sark_coefficients(double gamma, double a[6], double b[4]);

}  // namespace alegb
