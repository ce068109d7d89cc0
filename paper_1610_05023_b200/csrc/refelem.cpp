// Reference elements in long double; see refelem.hpp for the citations.
#include "refelem.hpp"

#include <algorithm>
#include <cmath>
#include <stdexcept>

namespace dg {

const int TET_FACE_VERTS[4][3] = {{0, 1, 2}, {0, 1, 3}, {1, 2, 3}, {0, 2, 3}};
const int TRI_FACE_VERTS[3][2] = {{0, 1}, {1, 2}, {0, 2}};
const int TET_NHAT[4][3] = {{0, 0, -1}, {0, -1, 0}, {1, 1, 1}, {-1, 0, 0}};
const int TRI_NHAT[3][2] = {{0, -1}, {1, 1}, {-1, 0}};

// Warp & Blend optimised blending parameter for the tetrahedron, degrees 1..8 ([68]; reading R13).
static const double ALPHA_TET[9] = {0.0, 0.0, 0.0, 0.0, 0.1002, 1.1332, 1.5608, 1.3413, 1.2577};

// ------------------------------------------------------------------ dense inverse
std::vector<ld> invert(const std::vector<ld>& A, int n) {
    std::vector<ld> W(A), I((size_t)n * n, 0.0L);
    for (int i = 0; i < n; ++i) I[(size_t)i * n + i] = 1.0L;
    for (int c = 0; c < n; ++c) {
        int p = c;
        for (int r = c + 1; r < n; ++r)
            if (fabsl(W[(size_t)r * n + c]) > fabsl(W[(size_t)p * n + c])) p = r;
        if (W[(size_t)p * n + c] == 0.0L) throw std::runtime_error("singular matrix in reference-element setup");
        if (p != c)
            for (int k = 0; k < n; ++k) {
                std::swap(W[(size_t)p * n + k], W[(size_t)c * n + k]);
                std::swap(I[(size_t)p * n + k], I[(size_t)c * n + k]);
            }
        ld piv = 1.0L / W[(size_t)c * n + c];
        for (int k = 0; k < n; ++k) { W[(size_t)c * n + k] *= piv; I[(size_t)c * n + k] *= piv; }
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            ld f = W[(size_t)r * n + c];
            if (f == 0.0L) continue;
            for (int k = 0; k < n; ++k) {
                W[(size_t)r * n + k] -= f * W[(size_t)c * n + k];
                I[(size_t)r * n + k] -= f * I[(size_t)c * n + k];
            }
        }
    }
    return I;
}

// ------------------------------------------------------------------ Jacobi polynomials (orthonormal)
static ld jacobi(ld x, int a, int b, int n) {
    ld g0 = powl(2.0L, a + b + 1) / (a + b + 1) * tgammal(a + 1.0L) * tgammal(b + 1.0L) / tgammal(a + b + 1.0L);
    ld p0 = 1.0L / sqrtl(g0);
    if (n == 0) return p0;
    ld g1 = (ld)(a + 1) * (b + 1) / (a + b + 3) * g0;
    ld p1 = ((a + b + 2) * x / 2 + (ld)(a - b) / 2) / sqrtl(g1);
    if (n == 1) return p1;
    ld aold = 2.0L / (2 + a + b) * sqrtl((ld)(a + 1) * (b + 1) / (a + b + 3));
    for (int i = 1; i < n; ++i) {
        ld h1 = 2 * i + a + b;
        ld anew = 2.0L / (h1 + 2) * sqrtl((ld)(i + 1) * (i + 1 + a + b) * (i + 1 + a) * (i + 1 + b) / ((h1 + 1) * (h1 + 3)));
        ld bnew = -(ld)(a * a - b * b) / (h1 * (h1 + 2));
        ld p2 = (-aold * p0 + (x - bnew) * p1) / anew;
        p0 = p1; p1 = p2; aold = anew;
    }
    return p1;
}

static ld djacobi(ld x, int a, int b, int n) {
    if (n == 0) return 0.0L;
    return sqrtl((ld)n * (n + a + b + 1)) * jacobi(x, a + 1, b + 1, n - 1);
}

// Legendre-Gauss-Lobatto points: +-1 and the zeros of P^{(1,1)}_{N-1} (Newton with deflation).
static std::vector<ld> lgl(int N) {
    std::vector<ld> x(N + 1);
    x[0] = -1.0L; x[N] = 1.0L;
    int n = N - 1;
    const ld pi = acosl(-1.0L);
    std::vector<ld> z(n);
    for (int k = 0; k < n; ++k) {
        ld r = -cosl(pi * (2 * k + 1) / (2.0L * n));           // Chebyshev start
        for (int it = 0; it < 100; ++it) {
            ld s = 0.0L;
            for (int j = 0; j < k; ++j) s += 1.0L / (r - z[j]);
            ld f = jacobi(r, 1, 1, n), df = djacobi(r, 1, 1, n);
            ld d = f / (df - s * f);
            r -= d;
            if (fabsl(d) < 1e-19L) break;
        }
        z[k] = r;
    }
    std::sort(z.begin(), z.end());
    for (int k = 0; k < n; ++k) x[k + 1] = (z[k] - z[n - 1 - k]) / 2;    // exact symmetry
    return x;
}

// 1D warp function of [68] divided by (1 - x^2): w~(x) = sum_i (x_i^LGL - x_i^eq) l_i^eq(x) / (1 - x^2)
static ld scaled_warp(int N, const std::vector<ld>& gl, ld x) {
    ld den = 1.0L - x * x;
    if (fabsl(den) < 1e-12L) return 0.0L;
    ld w = 0.0L;
    for (int i = 0; i <= N; ++i) {
        ld xi = -1.0L + 2.0L * i / N, li = 1.0L;
        for (int j = 0; j <= N; ++j)
            if (j != i) { ld xj = -1.0L + 2.0L * j / N; li *= (x - xj) / (xi - xj); }
        w += (gl[i] - xi) * li;
    }
    return w / den;
}

// Warp & Blend nodes of the tetrahedron, lattice order t-major, then s, r fastest.
static void nodes_tet(int N, std::vector<ld>& rst, std::vector<ld>& bary) {
    const ld alpha = ALPHA_TET[N];
    const ld s3 = sqrtl(3.0L), s6 = sqrtl(6.0L);
    const ld VT[4][3] = {{-1, -1 / s3, -1 / s6}, {1, -1 / s3, -1 / s6}, {0, 2 / s3, -1 / s6}, {0, 0, 3 / s6}};
    std::vector<ld> gl = lgl(N);
    const ld tol = 1e-10L;
    rst.clear(); bary.clear();
    for (int n = 0; n <= N; ++n)
        for (int m = 0; m <= N - n; ++m)
            for (int q = 0; q <= N - n - m; ++q) {
                ld lam[4] = {(ld)(N - n - m - q) / N, (ld)q / N, (ld)m / N, (ld)n / N};
                ld X[3] = {0, 0, 0};
                for (int v = 0; v < 4; ++v)
                    for (int d = 0; d < 3; ++d) X[d] += lam[v] * VT[v][d];
                int nnz = 0;
                for (int v = 0; v < 4; ++v) nnz += lam[v] > tol;
                // sum over the four faces (a = opposite vertex) of blend_a * (sum over the face's three edges of
                // the 1D warp along the edge); nodes on a tet edge keep the pure 1D warp of that edge.
                ld sh[3] = {0, 0, 0};
                for (int a = 0; a < 4; ++a) {
                    int fv[3], c = 0;
                    for (int v = 0; v < 4; ++v) if (v != a) fv[c++] = v;
                    ld blend;
                    if (nnz >= 3) {
                        ld la = lam[a];
                        ld num = lam[fv[0]] * lam[fv[1]] * lam[fv[2]];
                        ld den = (lam[fv[0]] + la / 2) * (lam[fv[1]] + la / 2) * (lam[fv[2]] + la / 2);
                        blend = (1 + alpha * la * alpha * la) * num / den;
                    } else if (nnz == 2) {
                        // pure edge warp: take it once, from the lowest-numbered face that contains the edge
                        bool on_face = lam[a] <= tol;
                        bool first = true;
                        for (int a2 = 0; a2 < a; ++a2) if (lam[a2] <= tol) first = false;
                        blend = (on_face && first) ? 1.0L : 0.0L;
                    } else {
                        blend = 0.0L;
                    }
                    if (blend == 0.0L) continue;
                    for (int e = 0; e < 3; ++e) {
                        int mm = fv[e], nn = fv[(e + 1) % 3], oo = fv[(e + 2) % 3];
                        ld amp = 4 * lam[mm] * lam[nn] * scaled_warp(N, gl, lam[nn] - lam[mm]) *
                                 (1 + alpha * lam[oo] * alpha * lam[oo]);
                        for (int d = 0; d < 3; ++d) sh[d] += blend * amp * (VT[nn][d] - VT[mm][d]) / 2;
                    }
                }
                for (int d = 0; d < 3; ++d) X[d] += sh[d];
                // back to (r,s,t): X = V0 + (1+r)/2 (V1-V0) + (1+s)/2 (V2-V0) + (1+t)/2 (V3-V0)
                std::vector<ld> A(9);
                for (int d = 0; d < 3; ++d)
                    for (int v = 0; v < 3; ++v) A[d * 3 + v] = (VT[v + 1][d] - VT[0][d]) / 2;
                std::vector<ld> Ai = invert(A, 3);
                ld c3[3];
                for (int v = 0; v < 3; ++v) {
                    c3[v] = -1.0L;
                    for (int d = 0; d < 3; ++d) c3[v] += Ai[v * 3 + d] * (X[d] - VT[0][d]);
                }
                // snap lattice-exact coordinates so that faces / edges / vertices are exact
                for (int v = 0; v < 3; ++v) if (lam[v + 1] < tol) c3[v] = -1.0L;
                if (lam[0] < tol) c3[2] = -1.0L - c3[0] - c3[1];
                for (int v = 0; v < 3; ++v) rst.push_back(c3[v]);
                bary.push_back(-(1 + c3[0] + c3[1] + c3[2]) / 2);
                for (int v = 0; v < 3; ++v) bary.push_back((1 + c3[v]) / 2);
            }
}

// ------------------------------------------------------------------ orthonormal simplex bases ([42])
static void basis1d(ld r, int i, ld& v, ld& dr) { v = jacobi(r, 0, 0, i); dr = djacobi(r, 0, 0, i); }

static void basis2d(ld r, ld s, int i, int j, ld& v, ld& dr, ld& ds) {
    ld a = (fabsl(1 - s) > 1e-14L) ? 2 * (1 + r) / (1 - s) - 1 : -1.0L, b = s;
    ld fa = jacobi(a, 0, 0, i), dfa = djacobi(a, 0, 0, i);
    ld gb = jacobi(b, 2 * i + 1, 0, j), dgb = djacobi(b, 2 * i + 1, 0, j);
    ld hb = (1 - b) / 2;
    ld hbi = powl(hb, i), hbi1 = (i > 0) ? powl(hb, i - 1) : 1.0L;
    ld sc = powl(2.0L, i + 0.5L);
    v = sqrtl(2.0L) * fa * gb * powl(1 - b, i);
    dr = dfa * gb;
    if (i > 0) dr *= hbi1;
    ds = dfa * (gb * ((1 + a) / 2));
    if (i > 0) ds *= hbi1;
    ld tmp = dgb * hbi;
    if (i > 0) tmp -= 0.5L * i * gb * hbi1;
    ds += fa * tmp;
    dr *= sc; ds *= sc;
}

static void basis3d(ld r, ld s, ld t, int i, int j, int k, ld& v, ld& dr, ld& ds, ld& dt) {
    ld a = (fabsl(s + t) > 1e-14L) ? 2 * (1 + r) / (-s - t) - 1 : -1.0L;
    ld b = (fabsl(1 - t) > 1e-14L) ? 2 * (1 + s) / (1 - t) - 1 : -1.0L;
    ld c = t;
    ld fa = jacobi(a, 0, 0, i), dfa = djacobi(a, 0, 0, i);
    ld gb = jacobi(b, 2 * i + 1, 0, j), dgb = djacobi(b, 2 * i + 1, 0, j);
    ld hc = jacobi(c, 2 * (i + j) + 2, 0, k), dhc = djacobi(c, 2 * (i + j) + 2, 0, k);
    ld hb = (1 - b) / 2, hcc = (1 - c) / 2;
    int ij = i + j;
    ld pb_i = powl(hb, i), pb_i1 = (i > 0) ? powl(hb, i - 1) : 1.0L;
    ld pc_ij = powl(hcc, ij), pc_ij1 = (ij > 0) ? powl(hcc, ij - 1) : 1.0L;
    v = 2 * sqrtl(2.0L) * fa * gb * powl(1 - b, i) * hc * powl(1 - c, ij);
    ld vr = dfa * (gb * hc);
    if (i > 0) vr *= pb_i1;
    if (ij > 0) vr *= pc_ij1;
    ld vs = (1 + a) / 2 * vr;
    ld tmp = dgb * pb_i;
    if (i > 0) tmp += (-0.5L * i) * (gb * pb_i1);
    if (ij > 0) tmp *= pc_ij1;
    tmp = fa * (tmp * hc);
    vs += tmp;
    ld vt = (1 + a) / 2 * vr + (1 + b) / 2 * tmp;
    ld tmp2 = dhc * pc_ij;
    if (ij > 0) tmp2 -= 0.5L * ij * (hc * pc_ij1);
    tmp2 = fa * (gb * tmp2) * pb_i;
    vt += tmp2;
    ld sc = powl(2.0L, 2 * i + j + 1.5L);
    dr = vr * sc; ds = vs * sc; dt = vt * sc;
}

// Vandermonde V [n][Np] and its reference gradients for points given as [n][dim]
static void vandermonde(int dim, int N, const std::vector<ld>& x, int n, std::vector<ld>& V, std::vector<ld> G[3]) {
    int Np = (dim == 1) ? N + 1 : (dim == 2) ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
    V.assign((size_t)n * Np, 0);
    for (int a = 0; a < dim; ++a) G[a].assign((size_t)n * Np, 0);
    for (int p = 0; p < n; ++p) {
        int m = 0;
        if (dim == 1) {
            for (int i = 0; i <= N; ++i, ++m) basis1d(x[p], i, V[(size_t)p * Np + m], G[0][(size_t)p * Np + m]);
        } else if (dim == 2) {
            for (int i = 0; i <= N; ++i)
                for (int j = 0; j <= N - i; ++j, ++m)
                    basis2d(x[p * 2], x[p * 2 + 1], i, j, V[(size_t)p * Np + m], G[0][(size_t)p * Np + m],
                            G[1][(size_t)p * Np + m]);
        } else {
            for (int i = 0; i <= N; ++i)
                for (int j = 0; j <= N - i; ++j)
                    for (int k = 0; k <= N - i - j; ++k, ++m)
                        basis3d(x[p * 3], x[p * 3 + 1], x[p * 3 + 2], i, j, k, V[(size_t)p * Np + m],
                                G[0][(size_t)p * Np + m], G[1][(size_t)p * Np + m], G[2][(size_t)p * Np + m]);
        }
    }
}

static std::vector<ld> matmul(const std::vector<ld>& A, const std::vector<ld>& B, int n, int k, int m, bool transB) {
    std::vector<ld> C((size_t)n * m, 0);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < m; ++j) {
            ld s = 0;
            for (int q = 0; q < k; ++q) s += A[(size_t)i * k + q] * (transB ? B[(size_t)j * k + q] : B[(size_t)q * m + j]);
            C[(size_t)i * m + j] = s;
        }
    return C;
}

// (M^-1 l(x))_n = sum_m V_nm psi_m(x): the Galerkin weights of a Dirac delta at reference point x
std::vector<double> delta_weights(const RefElem& e, const ld* x) {
    std::vector<ld> V, Vx, G[3], Gx[3];
    vandermonde(e.dim, e.N, e.rst, e.Np, V, G);
    std::vector<ld> xs(x, x + e.dim);
    vandermonde(e.dim, e.N, xs, 1, Vx, Gx);
    std::vector<double> w(e.Np);
    for (int n = 0; n < e.Np; ++n) {
        ld s = 0;
        for (int m = 0; m < e.Np; ++m) s += V[(size_t)n * e.Np + m] * Vx[m];
        w[n] = (double)s;
    }
    return w;
}

RefElem make_refelem(int dim, int N) {
    if (dim < 1 || dim > 3 || N < 1 || N > 8) throw std::runtime_error("make_refelem: need dim in 1..3, N in 1..8");
    RefElem e;
    e.dim = dim; e.N = N;
    const ld tol = 1e-10L;
    std::vector<ld> r3, b3;
    nodes_tet(N, r3, b3);
    int Np3 = (int)r3.size() / 3;
    if (dim == 3) {
        e.rst = r3; e.bary = b3; e.Np = Np3; e.Nfaces = 4;
    } else if (dim == 2) {               // nodes of the tet face t = -1, coordinates (r,s)
        for (int n = 0; n < Np3; ++n)
            if (fabsl(1 + r3[n * 3 + 2]) < tol) {
                ld r = r3[n * 3], s = r3[n * 3 + 1];
                e.rst.push_back(r); e.rst.push_back(s);
                e.bary.push_back(-(r + s) / 2); e.bary.push_back((1 + r) / 2); e.bary.push_back((1 + s) / 2);
            }
        e.Np = (int)e.rst.size() / 2; e.Nfaces = 3;
    } else {                             // nodes of the tet edge s = t = -1: the LGL points
        e.rst = lgl(N);
        for (int n = 0; n <= N; ++n) { e.bary.push_back((1 - e.rst[n]) / 2); e.bary.push_back((1 + e.rst[n]) / 2); }
        e.Np = N + 1; e.Nfaces = 2;
    }
    const int Np = e.Np;
    e.Nfp = (dim == 3) ? (N + 1) * (N + 2) / 2 : (dim == 2) ? N + 1 : 1;
    // face masks: nodes whose barycentric coordinate of the opposite vertex vanishes
    static const int opp3[4] = {3, 2, 0, 1}, opp2[3] = {2, 0, 1}, opp1[2] = {1, 0};
    const int* opp = (dim == 3) ? opp3 : (dim == 2) ? opp2 : opp1;
    for (int f = 0; f < e.Nfaces; ++f) {
        int cnt = 0;
        for (int n = 0; n < Np; ++n)
            if (fabsl(e.bary[(size_t)n * (dim + 1) + opp[f]]) < tol) { e.Fmask.push_back(n); ++cnt; }
        if (cnt != e.Nfp) throw std::runtime_error("make_refelem: unexpected number of face nodes");
    }
    std::vector<ld> V, G[3];
    vandermonde(dim, N, e.rst, Np, V, G);
    std::vector<ld> Vi = invert(V, Np);
    for (int a = 0; a < dim; ++a) {
        std::vector<ld> D = matmul(G[a], Vi, Np, Np, Np, false);
        e.D[a].resize((size_t)Np * Np);
        for (size_t q = 0; q < D.size(); ++q) e.D[a][q] = (double)D[q];
    }
    std::vector<ld> Minv = matmul(V, V, Np, Np, Np, true);            // V V^T
    int nfn = e.Nfaces * e.Nfp;
    std::vector<ld> E((size_t)Np * nfn, 0);
    for (int f = 0; f < e.Nfaces; ++f) {
        if (dim == 1) { E[(size_t)e.Fmask[f] * nfn + f] = 1; continue; }
        // chart of the face onto the (dim-1)-simplex through its barycentric coordinates (vertex order of
        // TET_FACE_VERTS / TRI_FACE_VERTS): xi_a = 2 lambda_{a+1} - 1
        std::vector<ld> xf;
        for (int j = 0; j < e.Nfp; ++j) {
            int n = e.Fmask[f * e.Nfp + j];
            for (int a = 1; a < dim; ++a) {
                int v = (dim == 3) ? TET_FACE_VERTS[f][a] : TRI_FACE_VERTS[f][a];
                xf.push_back(2 * e.bary[(size_t)n * (dim + 1) + v] - 1);
            }
        }
        std::vector<ld> Vf, Gf[3];
        vandermonde(dim - 1, N, xf, e.Nfp, Vf, Gf);
        std::vector<ld> Mf = invert(matmul(Vf, Vf, e.Nfp, e.Nfp, e.Nfp, true), e.Nfp);
        for (int a = 0; a < e.Nfp; ++a)
            for (int b = 0; b < e.Nfp; ++b)
                E[(size_t)e.Fmask[f * e.Nfp + a] * nfn + f * e.Nfp + b] = Mf[(size_t)a * e.Nfp + b];
    }
    std::vector<ld> L = matmul(Minv, E, Np, Np, nfn, false);
    e.LIFT.resize(L.size());
    for (size_t q = 0; q < L.size(); ++q) e.LIFT[q] = (double)L[q];
    return e;
}

}  // namespace dg
