// Reference elements of the nodal DG scheme (host side, extended precision).
//
// PAPER.md:L489 (§3.2): Warp & Blend nodes on the reference tetrahedron [68]; the triangle and line nodes
// are the tetrahedron's face and edge nodes.  PAPER.md:L529: differentiation and lifting matrices "defined
// in [42]": with an orthonormal modal basis psi_m and V_nm = psi_m(x_n),  D_a = (d_a V) V^-1,
// M^-1 = V V^T,  LIFT = M^-1 E  (E = face mass matrices scattered to the face nodes).
//
// All of it is evaluated in `long double` and rounded once, so that the operators are correct to ~1 ulp
// of double (needed for the 1e-11 parity bound after thousands of stages).
#pragma once
#include <vector>

namespace dg {

typedef long double ld;

struct RefElem {
    int dim = 0, N = 0, Np = 0, Nfp = 0, Nfaces = 0;
    std::vector<ld> rst;                 // [Np][dim] reference coordinates
    std::vector<double> D[3];            // D[a][n*Np+m]   (row n, column m)
    std::vector<double> LIFT;            // [Np][Nfaces*Nfp]
    std::vector<int> Fmask;              // [Nfaces][Nfp] node indices, increasing
    std::vector<ld> bary;                // [Np][dim+1] barycentric coordinates w.r.t. vertices 0..dim
};

// Local vertex lists of the faces, in the order of Fmask:
//   tet:      {0,1,2} (t=-1), {0,1,3} (s=-1), {1,2,3} (r+s+t=-1), {0,2,3} (r=-1)
//   triangle: {0,1} (s=-1),   {1,2} (r+s=0),  {0,2} (r=-1)
//   line:     {0} (r=-1),     {1} (r=+1)
extern const int TET_FACE_VERTS[4][3];
extern const int TRI_FACE_VERTS[3][2];

// Reference outward normals (un-normalised gradients of the face level sets), rows = faces.
extern const int TET_NHAT[4][3];
extern const int TRI_NHAT[3][2];

RefElem make_refelem(int dim, int N);

// Weights (M^-1 l(x))_n of a Dirac delta at the reference point x[dim] (point source).
std::vector<double> delta_weights(const RefElem& e, const ld* x);

// Dense helpers shared by the host setup (long double Gauss-Jordan inverse with partial pivoting).
std::vector<ld> invert(const std::vector<ld>& A, int n);

}  // namespace dg
