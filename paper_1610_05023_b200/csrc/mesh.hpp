// Host mesh hierarchy of the multidimensional solver: volume mesh -> surface mesh (cell faces
// on the domain faces carrying the HABC) -> line mesh (cell edges on the domain edges) -> corners, with the
// connectivity of each level and the inter-level maps (PAPER.md:L581 `map`, L668).
//
// Node matching is combinatorial: two cells sharing a face agree on the global vertex ids of that face, and a
// face node is identified by its barycentric weights on those vertices, so the neighbour's node is found by
// permuting the weights (exact, no coordinate tolerance).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "refelem.hpp"

namespace dg {

struct HostMesh {
    int N = 0, K = 0, T = 0, E = 0, C = 0;
    int Np = 0, Nfp = 0, N1 = 0;
    RefElem r3, r2, r1;
    std::vector<double> verts;           // [nv][3]
    std::vector<int32_t> tets;           // [K][4] positively oriented
    double lo[3], hi[3];                 // bounding box = the cuboid
    int face_bc[6] = {0, 0, 0, 0, 0, 0}; // per domain face (axis * 2 + (outward sign > 0)): 0 HABC, 1 p = 0, 2 rigid wall

    // ---- volume level
    std::vector<double> G3;              // [K][9]  rx ry rz sx sy sz tx ty tz
    std::vector<double> J3;              // [K]     |det|
    std::vector<double> Fs3;             // [K][4]  sJ/J per face
    std::vector<int32_t> nbr3;           // [K][4]  neighbour tet, or -1-t for the boundary triangle t (t = T: wall face)
    std::vector<uint8_t> bc3;            // [K][4]  0, or the wall type (1 p = 0, 2 rigid) of a boundary face without HABC
    std::vector<uint8_t> nbrface3;       // [K][4]  neighbour's local face
    std::vector<uint8_t> nbrperm3;       // [K][4]  index into perm3: neighbour face node = perm3[p][my face node]
    std::vector<uint8_t> perm3;          // [6][Nfp]

    // ---- surface level (triangle t = boundary face (tri_tet, tri_face); its node j = tet node Fmask[face][j])
    std::vector<int32_t> tri_tet, tri_face, tri_axis, tri_sign;
    std::vector<int32_t> tri_ax;         // [T][2] in-plane Cartesian axes, increasing
    std::vector<double> G2;              // [T][4]  r_xi r_eta s_xi s_eta
    std::vector<double> J2;              // [T]
    std::vector<double> n2;              // [T][3][2] outward unit normals of the three edges (in-plane components)
    std::vector<double> Fs2;             // [T][3]
    std::vector<int32_t> nbr2;           // [T][3]  neighbour triangle, or -1-(2*line+side) on a domain edge (line = E: wall)
    std::vector<uint8_t> bc2;            // [T][3]  wall type of a triangle edge that meets a domain face without HABC
    std::vector<int32_t> nbrnode2;       // [T][3][N1] neighbour's node (0..Nfp-1), or the line node (0..N) on a domain edge

    // ---- line level
    std::vector<int32_t> lin_v;          // [E][2] vertices, ordered along the tangent axis
    std::vector<int32_t> lin_axis;       // [E]
    std::vector<int32_t> lin_ab;         // [E][2] normal axes of faces A (lower axis) and B
    std::vector<int32_t> lin_sign;       // [E][2]
    std::vector<int32_t> lin_tri;        // [E][2] parent triangles on A, B
    std::vector<int32_t> lin_trinode;    // [E][2][N1] node of the parent triangle under each line node
    std::vector<double> J1;              // [E] length/2
    std::vector<int32_t> nbr1;           // [E][2] neighbour line, or -1-(3*corner+axis) at a corner (corner = C: wall)
    std::vector<uint8_t> bc1;            // [E][2] wall type of a line end that meets a domain face without HABC

    // ---- corners
    std::vector<int32_t> cor_vertex;     // [C]
    std::vector<int32_t> cor_line;       // [C][3] line along x,y,z
    std::vector<int32_t> cor_end;        // [C][3] 0: r=-1 end, 1: r=+1 end
    std::vector<int32_t> cor_sign;       // [C][3]
};

// Throws std::runtime_error with a message starting "EMESH:" (degenerate / non-conforming mesh) or "EINVAL:"
// (non-cuboid boundary).
// face_bc: NULL (HABC on all six faces) or 6 codes indexed axis * 2 + (outward sign > 0): 0 HABC, 1 p = 0
// (PAPER.md:L516-518), 2 rigid wall.  Only faces with code 0 get triangles; lines exist between two HABC faces and
// corners where three meet (the K^pnt = 4 case of the paper's runs).
void build_mesh(HostMesh& m, int N, int nverts, const double* xyz, int ntets, const int32_t* tets,
                const int* face_bc = nullptr);

}  // namespace dg
