// Host mesh hierarchy; see mesh.hpp.
#include "mesh.hpp"

#include <algorithm>
#include <array>
#include <cmath>
#include <map>
#include <stdexcept>

namespace dg {

namespace {

const int PERMS3[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};

struct FaceKey {
    int32_t v[3];
    int32_t id;
    bool operator<(const FaceKey& o) const {
        if (v[0] != o.v[0]) return v[0] < o.v[0];
        if (v[1] != o.v[1]) return v[1] < o.v[1];
        if (v[2] != o.v[2]) return v[2] < o.v[2];
        return id < o.id;
    }
    bool same(const FaceKey& o) const { return v[0] == o.v[0] && v[1] == o.v[1] && v[2] == o.v[2]; }
};

[[noreturn]] void fail(const std::string& s) { throw std::runtime_error(s); }

// index j' such that weights w' of candidate j' on the permuted vertices equal the weights w of j
int match_bary(const std::vector<ld>& bary, int nv, const int* cand, int ncand, const ld* w, const int* sigma) {
    for (int c = 0; c < ncand; ++c) {
        const ld* wc = &bary[(size_t)cand[c] * nv];
        bool ok = true;
        for (int i = 0; i < nv && ok; ++i) ok = fabsl(wc[sigma[i]] - w[i]) < 1e-9L;
        if (ok) return c;
    }
    fail("EMESH: internal node matching failed");
}

}  // namespace

void build_mesh(HostMesh& m, int N, int nverts, const double* xyz, int ntets, const int32_t* tets, const int* face_bc) {
    for (int q = 0; q < 6; ++q) {
        m.face_bc[q] = face_bc ? face_bc[q] : 0;
        if (m.face_bc[q] < 0 || m.face_bc[q] > 2) throw std::runtime_error("EINVAL: face_bc codes are 0 (HABC), 1 (p = 0), 2 (rigid)");
    }
    if (nverts < 4 || ntets < 1 || !xyz || !tets) fail("EINVAL: empty mesh");
    m.N = N; m.K = ntets;
    m.r3 = make_refelem(3, N); m.r2 = make_refelem(2, N); m.r1 = make_refelem(1, N);
    m.Np = m.r3.Np; m.Nfp = m.r3.Nfp; m.N1 = N + 1;
    const int K = ntets, Np = m.Np, Nfp = m.Nfp, N1 = m.N1;
    (void)Np;
    m.verts.assign(xyz, xyz + (size_t)nverts * 3);
    m.tets.assign(tets, tets + (size_t)ntets * 4);
    for (size_t i = 0; i < m.tets.size(); ++i)
        if (m.tets[i] < 0 || m.tets[i] >= nverts) fail("EMESH: vertex index out of range");
    for (int d = 0; d < 3; ++d) { m.lo[d] = 1e300; m.hi[d] = -1e300; }
    for (int v = 0; v < nverts; ++v)
        for (int d = 0; d < 3; ++d) {
            m.lo[d] = std::min(m.lo[d], xyz[v * 3 + d]);
            m.hi[d] = std::max(m.hi[d], xyz[v * 3 + d]);
        }
    const double size = std::max({m.hi[0] - m.lo[0], m.hi[1] - m.lo[1], m.hi[2] - m.lo[2]});
    const double tol = 1e-9 * size;
    auto X = [&](int v, int d) { return m.verts[(size_t)v * 3 + d]; };
    // plane code of a vertex set: returns list of (axis, sign) planes containing all of them
    auto planes_of = [&](const int32_t* vs, int n, int (*out)[2]) {
        int cnt = 0;
        for (int a = 0; a < 3; ++a) {
            bool l = true, h = true;
            for (int i = 0; i < n; ++i) {
                l = l && std::fabs(X(vs[i], a) - m.lo[a]) < tol;
                h = h && std::fabs(X(vs[i], a) - m.hi[a]) < tol;
            }
            if (l) { out[cnt][0] = a; out[cnt][1] = -1; ++cnt; }
            if (h) { out[cnt][0] = a; out[cnt][1] = 1; ++cnt; }
        }
        return cnt;
    };

    // ---------------------------------------------------------------- volume geometry
    m.G3.resize((size_t)K * 9); m.J3.resize(K); m.Fs3.resize((size_t)K * 4);
    for (int k = 0; k < K; ++k) {
        int32_t* t = &m.tets[(size_t)k * 4];
        ld A[9], det = 0;
        for (int pass = 0; pass < 2; ++pass) {
            for (int d = 0; d < 3; ++d)
                for (int a = 0; a < 3; ++a) A[d * 3 + a] = ((ld)X(t[a + 1], d) - (ld)X(t[0], d)) / 2;
            det = A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) + A[2] * (A[3] * A[7] - A[4] * A[6]);
            if (det > 0) break;
            if (pass == 0) std::swap(t[2], t[3]);
        }
        if (!(det > 1e-14L * size * size * size)) fail("EMESH: degenerate tetrahedron");
        std::vector<ld> Ai = invert(std::vector<ld>(A, A + 9), 3);     // Ai[a*3+d] = d ref_a / d x_d
        for (int q = 0; q < 9; ++q) m.G3[(size_t)k * 9 + q] = (double)Ai[q];
        m.J3[k] = (double)det;
        for (int f = 0; f < 4; ++f) {
            ld s = 0;
            for (int d = 0; d < 3; ++d) {
                ld c = 0;
                for (int a = 0; a < 3; ++a) c += TET_NHAT[f][a] * Ai[a * 3 + d];
                s += c * c;
            }
            m.Fs3[(size_t)k * 4 + f] = (double)sqrtl(s);
        }
    }

    // ---------------------------------------------------------------- face-node permutation tables
    // all four tet faces list their nodes in the reference triangle's order (checked here)
    for (int f = 0; f < 4; ++f)
        for (int j = 0; j < Nfp; ++j) {
            int n = m.r3.Fmask[f * Nfp + j];
            for (int i = 0; i < 3; ++i)
                if (fabsl(m.r3.bary[(size_t)n * 4 + TET_FACE_VERTS[f][i]] - m.r2.bary[(size_t)j * 3 + i]) > 1e-12L)
                    fail("EMESH: internal face-node ordering mismatch");
        }
    m.perm3.resize(6 * Nfp);
    {
        std::vector<int> all(Nfp);
        for (int j = 0; j < Nfp; ++j) all[j] = j;
        for (int p = 0; p < 6; ++p)
            for (int j = 0; j < Nfp; ++j)
                m.perm3[p * Nfp + j] = (uint8_t)match_bary(m.r2.bary, 3, all.data(), Nfp, &m.r2.bary[(size_t)j * 3], PERMS3[p]);
    }

    // ---------------------------------------------------------------- volume connectivity
    std::vector<FaceKey> keys((size_t)K * 4);
    for (int k = 0; k < K; ++k)
        for (int f = 0; f < 4; ++f) {
            FaceKey& q = keys[(size_t)k * 4 + f];
            for (int i = 0; i < 3; ++i) q.v[i] = m.tets[(size_t)k * 4 + TET_FACE_VERTS[f][i]];
            std::sort(q.v, q.v + 3);
            if (q.v[0] == q.v[1] || q.v[1] == q.v[2]) fail("EMESH: repeated vertex in a tetrahedron");
            q.id = k * 4 + f;
        }
    std::sort(keys.begin(), keys.end());
    m.nbr3.assign((size_t)K * 4, INT32_MIN); m.nbrface3.assign((size_t)K * 4, 0); m.nbrperm3.assign((size_t)K * 4, 0);
    std::vector<int32_t> bfaces;
    for (size_t i = 0; i < keys.size();) {
        size_t j = i + 1;
        while (j < keys.size() && keys[j].same(keys[i])) ++j;
        if (j - i > 2) fail("EMESH: a face is shared by more than two tetrahedra");
        if (j - i == 1) {
            bfaces.push_back(keys[i].id);
        } else {
            for (int s = 0; s < 2; ++s) {
                int a = keys[i + s].id, b = keys[i + 1 - s].id;
                int ka = a / 4, fa = a % 4, kb = b / 4, fb = b % 4;
                int sigma[3];
                for (int q = 0; q < 3; ++q) {
                    int va = m.tets[(size_t)ka * 4 + TET_FACE_VERTS[fa][q]];
                    sigma[q] = -1;
                    for (int r = 0; r < 3; ++r)
                        if (m.tets[(size_t)kb * 4 + TET_FACE_VERTS[fb][r]] == va) sigma[q] = r;
                }
                int p = -1;
                for (int c = 0; c < 6; ++c)
                    if (PERMS3[c][0] == sigma[0] && PERMS3[c][1] == sigma[1] && PERMS3[c][2] == sigma[2]) p = c;
                if (p < 0) fail("EMESH: inconsistent shared face");
                m.nbr3[a] = kb; m.nbrface3[a] = (uint8_t)fb; m.nbrperm3[a] = (uint8_t)p;
            }
        }
        i = j;
    }

    // ---------------------------------------------------------------- surface mesh
    std::sort(bfaces.begin(), bfaces.end());
    m.bc3.assign((size_t)K * 4, 0);
    {
        std::vector<int32_t> habc_faces, wall_faces;
        for (int32_t bf : bfaces) {
            int k = bf / 4, f = bf % 4;
            int32_t v3[3];
            for (int i = 0; i < 3; ++i) v3[i] = m.tets[(size_t)k * 4 + TET_FACE_VERTS[f][i]];
            int pl[6][2];
            if (planes_of(v3, 3, pl) != 1) fail("EINVAL: a boundary cell face does not lie on exactly one face of the bounding cuboid");
            const int code = m.face_bc[pl[0][0] * 2 + (pl[0][1] > 0)];
            if (code == 0) habc_faces.push_back(bf);
            else { m.bc3[bf] = (uint8_t)code; wall_faces.push_back(bf); }
        }
        for (int32_t bf : wall_faces) m.nbr3[bf] = -1 - (int32_t)habc_faces.size();     // the zero ghost row
        bfaces.swap(habc_faces);
    }
    const int T = (int)bfaces.size();
    m.T = T;
    m.tri_tet.resize(T); m.tri_face.resize(T); m.tri_axis.resize(T); m.tri_sign.resize(T); m.tri_ax.resize((size_t)T * 2);
    m.G2.resize((size_t)T * 4); m.J2.resize(T); m.n2.resize((size_t)T * 6); m.Fs2.resize((size_t)T * 3);
    std::vector<std::array<int32_t, 3>> tv(T);
    for (int t = 0; t < T; ++t) {
        int k = bfaces[t] / 4, f = bfaces[t] % 4;
        m.nbr3[bfaces[t]] = -1 - t;
        m.tri_tet[t] = k; m.tri_face[t] = f;
        for (int i = 0; i < 3; ++i) tv[t][i] = m.tets[(size_t)k * 4 + TET_FACE_VERTS[f][i]];
        int pl[6][2];
        int np = planes_of(tv[t].data(), 3, pl);
        if (np != 1) fail("EINVAL: a boundary cell face does not lie on exactly one face of the bounding cuboid");
        m.tri_axis[t] = pl[0][0]; m.tri_sign[t] = pl[0][1];
        int ax[2], c = 0;
        for (int d = 0; d < 3; ++d) if (d != pl[0][0]) ax[c++] = d;
        m.tri_ax[t * 2] = ax[0]; m.tri_ax[t * 2 + 1] = ax[1];
        ld A[4];                                   // A[d*2+a] = d x_d / d ref_a
        for (int d = 0; d < 2; ++d)
            for (int a = 0; a < 2; ++a) A[d * 2 + a] = ((ld)X(tv[t][a + 1], ax[d]) - (ld)X(tv[t][0], ax[d])) / 2;
        ld det = A[0] * A[3] - A[1] * A[2];
        if (fabsl(det) < 1e-14L * size * size) fail("EMESH: degenerate boundary triangle");
        ld Gi[4] = {A[3] / det, -A[1] / det, -A[2] / det, A[0] / det};    // Gi[a*2+d] = d ref_a / d x_d
        for (int q = 0; q < 4; ++q) m.G2[(size_t)t * 4 + q] = (double)Gi[q];
        m.J2[t] = (double)fabsl(det);
        for (int e = 0; e < 3; ++e) {
            ld nv[2];
            for (int d = 0; d < 2; ++d) nv[d] = TRI_NHAT[e][0] * Gi[d] + TRI_NHAT[e][1] * Gi[2 + d];
            ld mag = sqrtl(nv[0] * nv[0] + nv[1] * nv[1]);
            m.Fs2[(size_t)t * 3 + e] = (double)mag;
            m.n2[(size_t)t * 6 + e * 2] = (double)(nv[0] / mag);
            m.n2[(size_t)t * 6 + e * 2 + 1] = (double)(nv[1] / mag);
        }
    }
    // triangle connectivity inside each domain face; unmatched edges lie on domain edges
    std::vector<FaceKey> ek((size_t)T * 3);
    for (int t = 0; t < T; ++t)
        for (int e = 0; e < 3; ++e) {
            FaceKey& q = ek[(size_t)t * 3 + e];
            int a = tv[t][TRI_FACE_VERTS[e][0]], b = tv[t][TRI_FACE_VERTS[e][1]];
            q.v[0] = std::min(a, b); q.v[1] = std::max(a, b); q.v[2] = m.tri_axis[t] * 2 + (m.tri_sign[t] > 0);
            q.id = t * 3 + e;
        }
    std::sort(ek.begin(), ek.end());
    m.nbr2.assign((size_t)T * 3, INT32_MIN); m.nbrnode2.assign((size_t)T * 3 * N1, 0);
    std::vector<int32_t> bedges;
    for (size_t i = 0; i < ek.size();) {
        size_t j = i + 1;
        while (j < ek.size() && ek[j].same(ek[i])) ++j;
        if (j - i > 2) fail("EMESH: non-manifold boundary surface");
        if (j - i == 1) {
            bedges.push_back(ek[i].id);
        } else {
            for (int s = 0; s < 2; ++s) {
                int a = ek[i + s].id, b = ek[i + 1 - s].id;
                int ta = a / 3, ea = a % 3, tb = b / 3, eb = b % 3;
                bool same_dir = tv[ta][TRI_FACE_VERTS[ea][0]] == tv[tb][TRI_FACE_VERTS[eb][0]];
                m.nbr2[a] = tb;
                for (int q = 0; q < N1; ++q)
                    m.nbrnode2[(size_t)a * N1 + q] = m.r2.Fmask[eb * N1 + (same_dir ? q : N - q)];
            }
        }
        i = j;
    }
    // edge nodes of the reference triangle run from the first to the second vertex of TRI_FACE_VERTS (checked)
    for (int e = 0; e < 3; ++e)
        for (int q = 0; q < N1; ++q) {
            int n = m.r2.Fmask[e * N1 + q];
            if (fabsl(m.r2.bary[(size_t)n * 3 + TRI_FACE_VERTS[e][1]] - m.r1.bary[(size_t)q * 2 + 1]) > 1e-12L)
                fail("EMESH: internal edge-node ordering mismatch");
        }

    // ---------------------------------------------------------------- line mesh
    std::sort(bedges.begin(), bedges.end());
    m.bc2.assign((size_t)T * 3, 0);
    std::map<std::pair<int32_t, int32_t>, int> line_of;
    std::vector<std::array<int32_t, 2>> lin_te;
    for (size_t q = 0; q < bedges.size(); ++q) {
        int t = bedges[q] / 3, e = bedges[q] % 3;
        int32_t vs[2] = {tv[t][TRI_FACE_VERTS[e][0]], tv[t][TRI_FACE_VERTS[e][1]]};
        int pl[6][2];
        int np = planes_of(vs, 2, pl);
        int oth = -1;
        for (int c = 0; c < np; ++c)
            if (pl[c][0] != m.tri_axis[t]) { if (oth >= 0) oth = -2; else oth = c; }
        if (np != 2 || oth < 0) fail("EINVAL: a boundary triangle edge without neighbour is not on an edge of the cuboid");
        if (m.face_bc[pl[oth][0] * 2 + (pl[oth][1] > 0)] != 0) {       // the other face carries no HABC: wall condition, no line
            m.bc2[bedges[q]] = (uint8_t)m.face_bc[pl[oth][0] * 2 + (pl[oth][1] > 0)];
            continue;
        }
        int a_own = m.tri_axis[t], a_oth = pl[oth][0];
        int side = a_own < a_oth ? 0 : 1;
        auto key = std::make_pair(std::min(vs[0], vs[1]), std::max(vs[0], vs[1]));
        auto it = line_of.find(key);
        int ell;
        if (it == line_of.end()) {
            ell = (int)lin_te.size();
            line_of[key] = ell;
            int tang = 3 - a_own - a_oth;
            int v0 = key.first, v1 = key.second;
            if (X(v0, tang) > X(v1, tang)) std::swap(v0, v1);
            m.lin_v.push_back(v0); m.lin_v.push_back(v1);
            m.lin_axis.push_back(tang);
            int sA = side == 0 ? m.tri_sign[t] : pl[oth][1], sB = side == 0 ? pl[oth][1] : m.tri_sign[t];
            m.lin_ab.push_back(std::min(a_own, a_oth)); m.lin_ab.push_back(std::max(a_own, a_oth));
            m.lin_sign.push_back(sA); m.lin_sign.push_back(sB);
            m.lin_tri.push_back(-1); m.lin_tri.push_back(-1);
            lin_te.push_back({-1, -1});
            m.J1.push_back(std::fabs(X(v1, tang) - X(v0, tang)) / 2);
            if (m.J1.back() < 1e-14 * size) fail("EMESH: degenerate boundary line");
        } else {
            ell = it->second;
        }
        if (m.lin_tri[ell * 2 + side] >= 0) fail("EMESH: a domain-edge cell has two parent triangles on one face");
        m.lin_tri[ell * 2 + side] = t;
        lin_te[ell][side] = e;
        m.nbr2[bedges[q]] = -1 - (2 * ell + side);
    }
    const int E = (int)lin_te.size();
    m.E = E;
    for (size_t q = 0; q < m.bc2.size(); ++q)
        if (m.bc2[q]) m.nbr2[q] = -1 - 2 * E;                           // the zero ghost row
    m.lin_trinode.assign((size_t)E * 2 * N1, 0);
    for (int ell = 0; ell < E; ++ell)
        for (int side = 0; side < 2; ++side) {
            int t = m.lin_tri[ell * 2 + side], e = lin_te[ell][side];
            if (t < 0) fail("EMESH: a domain-edge cell has only one parent triangle (F_bnd^tri = 2 K^lin violated)");
            bool same_dir = tv[t][TRI_FACE_VERTS[e][0]] == m.lin_v[ell * 2];
            for (int q = 0; q < N1; ++q) {
                int qe = same_dir ? q : N - q;                         // position on the triangle edge
                m.lin_trinode[((size_t)ell * 2 + side) * N1 + q] = m.r2.Fmask[e * N1 + qe];
                m.nbrnode2[((size_t)t * 3 + e) * N1 + qe] = q;
            }
        }
    // line connectivity along each domain edge; unmatched ends are corners
    m.nbr1.assign((size_t)E * 2, INT32_MIN);
    m.bc1.assign((size_t)E * 2, 0);
    std::vector<FaceKey> pk((size_t)E * 2);
    for (int ell = 0; ell < E; ++ell)
        for (int e = 0; e < 2; ++e) {
            FaceKey& q = pk[(size_t)ell * 2 + e];
            q.v[0] = m.lin_v[ell * 2 + e];
            q.v[1] = m.lin_ab[ell * 2] * 16 + m.lin_ab[ell * 2 + 1] * 4 + (m.lin_sign[ell * 2] > 0) * 2 + (m.lin_sign[ell * 2 + 1] > 0);
            q.v[2] = 0; q.id = ell * 2 + e;
        }
    std::sort(pk.begin(), pk.end());
    std::map<int32_t, int> corner_of;
    for (size_t i = 0; i < pk.size();) {
        size_t j = i + 1;
        while (j < pk.size() && pk[j].same(pk[i])) ++j;
        if (j - i > 2) fail("EMESH: non-manifold boundary line");
        if (j - i == 2) {
            m.nbr1[pk[i].id] = pk[i + 1].id / 2;
            m.nbr1[pk[i + 1].id] = pk[i].id / 2;
            if (pk[i].id % 2 == pk[i + 1].id % 2) fail("EMESH: inconsistent line orientation");
        } else {
            int ell = pk[i].id / 2, e = pk[i].id % 2, v = pk[i].v[0], tang = m.lin_axis[ell];
            int s = 0;
            if (std::fabs(X(v, tang) - m.lo[tang]) < tol) s = -1;
            else if (std::fabs(X(v, tang) - m.hi[tang]) < tol) s = 1;
            else fail("EINVAL: a boundary line ends away from a corner of the cuboid");
            if (m.face_bc[tang * 2 + (s > 0)] != 0) {                   // the third face carries no HABC: wall condition, no corner
                m.bc1[pk[i].id] = (uint8_t)m.face_bc[tang * 2 + (s > 0)];
                i = j;
                continue;
            }
            auto it = corner_of.find(v);
            int c;
            if (it == corner_of.end()) {
                c = (int)m.cor_vertex.size();
                corner_of[v] = c;
                m.cor_vertex.push_back(v);
                for (int d = 0; d < 3; ++d) { m.cor_line.push_back(-1); m.cor_end.push_back(0); m.cor_sign.push_back(0); }
            } else {
                c = it->second;
            }
            m.cor_line[c * 3 + tang] = ell; m.cor_end[c * 3 + tang] = e; m.cor_sign[c * 3 + tang] = s;
            m.nbr1[pk[i].id] = -1 - (3 * c + tang);
        }
        i = j;
    }
    m.C = (int)m.cor_vertex.size();
    for (size_t q = 0; q < m.bc1.size(); ++q)
        if (m.bc1[q]) m.nbr1[q] = -1 - 3 * m.C;                         // the zero ghost row
    for (size_t q = 0; q < m.cor_line.size(); ++q)
        if (m.cor_line[q] < 0) fail("EMESH: a corner is not the end of three boundary lines (F_bnd^lin = 3 K^pnt violated)");
}

}  // namespace dg
