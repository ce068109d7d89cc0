// CUDA kernels of the DG + HABC time step (sm_100a).  One LSRK stage =
//   k_vol3d   fused volume + surface + update of the 3D solver                (Alg. 2, eq (41)-(43))
//   k_face2d  fused volume + surface + update of the J face solvers           (eq (31a-c), Alg. 3 first half)
//   k_edge1d  fused volume + surface + update of the J^2 edge solvers         (eq (34a-b), Alg. 4 first half)
//   k_close_face / k_close_edge / k_close_corner: the closure chain           (eq (28)-(30), (32)-(33), (35); Alg. 3-5)
// in that order (3D -> 2D -> 1D -> 0D).  Every solver reads the stage-(n-1) state from one buffer
// and writes stage n into the other (ping-pong), which is what lets volume, surface and update fuse: neighbours
// still see the old traces.  See DESIGN.md §6 for the layouts and the roofline of each kernel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dg {

constexpr int GEO3 = 24;   // per-tet record: G[9] | A[4] | B[4] | Fs[4] | rho c^2 | 1/rho | c | pad
constexpr int GEO2 = 24;   // per-triangle: G2[4] | n[3][2] | Fs[3] | A[3] | B[3] | rho c^2 | 1/rho | c | Z | pad
constexpr int GEO1 = 8;    // per-line: 1/J | A[2] | B[2] | rho c^2 | 1/rho | c
constexpr int JMAX = 12;

template <typename T> struct Q4 { T p, u, v, w; };
template <> struct __align__(32) Q4<double> { double p, u, v, w; };
template <> struct __align__(16) Q4<float> { float p, u, v, w; };

template <typename T>
struct Dev {
    int N, J, K, Tn, E, C, Np, Nfp, N1;
    // ---- 3D
    T* q[2]; T* res;                 // [K][Np][4]
    const T* geo3;                   // [K][GEO3]
    const int* nbr3;                 // [K][4]  neighbour tet or -1-triangle
    const uint32_t* finfo3;          // [K]     byte f: neighbour face | perm << 2
    const uint32_t* conn3;           // [K][4]  packed (kernel_vol3d_mma.cuh): boundary flag | id << 5 | perm << 2 | face
    const T* Dt3;                    // [3][Np][Np]  Dt3[a][m][n] = D_a[n][m]
    const T* Lt3;                    // [4 Nfp][Np]  Lt3[j][n]   = LIFT[n][j]
    const T* Dfrag; const T* Lfrag;  // the same operators in MMA-fragment order, zero-padded (N >= 6 tensor-pipe kernels
                                     // only; layouts in kernel_vol3d_mmag.cuh / kernel_vol3d_tf32g.cuh), else NULL
    const short* fmask3;             // [4][Nfp]
    const uint8_t* perm3;            // [6][Nfp]
    // ---- 2D
    T* fa[2]; T* fres;               // [T][J][3][Nfp]   p*_i, U_xi, U_eta
    T* S2;                           // [T][Nfp]   r^- + r^+ of the 3D field (q0^tet of the paper)
    T* qb3;                          // [T][Nfp]   r^- for the 3D solver     (qb^tet)
    T* ghost3;                       // [T][Nfp][4] ghost state (2 r^-, 0, 0, 0) behind an HABC face (tensor-pipe kernel)
    const T* geo2;                   // [T][GEO2]
    const int* nbr2;                 // [T][3]
    const int* nbrnode2;             // [T][3][N1]
    const int* tri_tet; const int* tri_face; const int* tri_axis; const int* tri_sign;
    const T* D2;                     // [2][Nfp][Nfp] row-major
    const T* L2;                     // [Nfp][3 N1]
    const short* fmask2;             // [3][N1]
    // ---- 1D
    T* ea[2]; T* eres;               // [E][J*J][2][N1]  p*_ij, w_ij
    T* S1;                           // [E][2][J][N1]    S^a_j , S^b_i          (q0^tri)
    T* qb2;                          // [E][2][J][N1]    side A: r^{-b}_i, side B: r^{-a}_j   (qb^tri)
    const T* geo1;                   // [E][GEO1]
    const int* nbr1;                 // [E][2]
    const int* lin_tri;              // [E][2]
    const int* lin_trinode;          // [E][2][N1]
    const int* lin_slot;             // [E][2]  which tangential velocity of the parent triangle is normal to the edge
    const int* lin_osign;            // [E][2]  outward sign of the OTHER face (the in-plane normal of this side)
    const T* D1;                     // [N1][N1]
    const T* L1;                     // [N1][2]
    // ---- 0D
    T* qb1;                          // [3 C][J*J]       r^- for the line solver (qb^lin)
    const int* cor_line; const int* cor_end; const int* cor_sign;   // [C][3]
    // ---- HABC algebra
    const T* cn;                     // [J]
    const T* Cij;                    // [J][J]  (1+c_i)/(1+c_i+c_j)
    const T* PeT; const T* QeT;      // [2J][2J] edge: r^- = Pe b + Qe r^+, stored transposed ([k][r])
    const T* Gc;                     // [3J^2][3J^2] corner: r^- = Gc r^+
    T invM;                          // 1/(2J+1)
};

// =====================================================================================================
// 3D: fused volume + surface + update.  Persistent CTAs; operators staged once in shared memory.
// Thread t < G*Np owns node n = t % Np of the ET elements of group g = t / Np  (EPB = G*ET per batch).
// =====================================================================================================
template <int N> struct Deg {
    static constexpr int Np = (N + 1) * (N + 2) * (N + 3) / 6;
    static constexpr int Nfp = (N + 1) * (N + 2) / 2;
    static constexpr int Nfn = 4 * Nfp;
};

template <typename T, int N, int G, int ET, bool OPS_IN_SMEM>
struct Vol3dCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EPB = G * ET;
    static constexpr int NT = ((G * Np + 31) / 32) * 32;
    static constexpr int ops_elems = OPS_IN_SMEM ? ((3 * Np * Np + Nfn * Np + 3) / 4) * 4 : 0;   // keeps sQ 32 B aligned
    static constexpr size_t ops_bytes = sizeof(T) * ops_elems;
    static constexpr size_t smem_bytes = ops_bytes + sizeof(T) * (EPB * Np * 4 + Nfn * EPB) + 16;
};

template <typename T, int N, int G, int ET, bool OPS_IN_SMEM>
__global__ void __launch_bounds__(Vol3dCfg<T, N, G, ET, OPS_IN_SMEM>::NT)
k_vol3d(Dev<T> d, int src, T rka, T rkb, T dt) {
    using Cfg = Vol3dCfg<T, N, G, ET, OPS_IN_SMEM>;
    constexpr int Np = Cfg::Np, Nfp = Cfg::Nfp, Nfn = Cfg::Nfn, EPB = Cfg::EPB, NT = Cfg::NT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const T* sD;
    const T* sL;
    if (OPS_IN_SMEM) {
        T* w = sm;
        for (int i = threadIdx.x; i < 3 * Np * Np; i += NT) w[i] = d.Dt3[i];
        for (int i = threadIdx.x; i < Nfn * Np; i += NT) w[3 * Np * Np + i] = d.Lt3[i];
        sD = w; sL = w + 3 * Np * Np;
        sm += Cfg::ops_elems;
    } else {
        sD = d.Dt3; sL = d.Lt3;
    }
    Q4<T>* sQ = reinterpret_cast<Q4<T>*>(sm);           // [EPB][Np]  (p, U^r, U^s, U^t)
    T* sG = sm + EPB * Np * 4;                          // [Nfn][EPB] flux jump g per face node
    const Q4<T>* __restrict__ qold = reinterpret_cast<const Q4<T>*>(d.q[src]);
    Q4<T>* __restrict__ qnew = reinterpret_cast<Q4<T>*>(d.q[src ^ 1]);
    Q4<T>* __restrict__ res = reinterpret_cast<Q4<T>*>(d.res);
    const int tid = threadIdx.x;
    const int grp = tid / Np, n = tid - grp * Np;
    const bool active = tid < G * Np;
    const int nbatch = (d.K + EPB - 1) / EPB;
    __syncthreads();

    for (int batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        const int e0 = batch * EPB;
        const int ne = min(EPB, d.K - e0);
        Q4<T> own[ET];
        // ---- phase 1: own nodes -> registers; (p, contravariant velocity) -> shared
        if (active) {
#pragma unroll
            for (int i = 0; i < ET; ++i) {
                const int e = grp * ET + i;
                if (e < ne) {
                    const T* g = d.geo3 + (size_t)(e0 + e) * GEO3;
                    Q4<T> v = qold[(size_t)(e0 + e) * Np + n];
                    own[i] = v;
                    Q4<T> c;
                    c.p = v.p;
                    c.u = g[0] * v.u + g[1] * v.v + g[2] * v.w;
                    c.v = g[3] * v.u + g[4] * v.v + g[5] * v.w;
                    c.w = g[6] * v.u + g[7] * v.v + g[8] * v.w;
                    sQ[e * Np + n] = c;
                } else {
                    own[i] = Q4<T>{0, 0, 0, 0};
                    sQ[e * Np + n] = Q4<T>{0, 0, 0, 0};
                }
            }
        }
        __syncthreads();
        // ---- phase 2: flux jump g at every face node (PAPER.md:L499-512 reduced to one scalar)
        for (int idx = tid; idx < EPB * Nfn; idx += NT) {
            const int e = idx / Nfn, fj = idx - e * Nfn;
            T gval = 0;
            if (e < ne) {
                const int f = fj / Nfp, j = fj - f * Nfp;
                const int k = e0 + e;
                const T* g = d.geo3 + (size_t)k * GEO3;
                const Q4<T> m = sQ[e * Np + d.fmask3[fj]];
                // Fs * n.u^- = nhat . U^-  (nhat: 0:(0,0,-1) 1:(0,-1,0) 2:(1,1,1) 3:(-1,0,0))
                const T unM = (f == 0) ? -m.w : (f == 1) ? -m.v : (f == 2) ? (m.u + m.v + m.w) : -m.u;
                const int nb = d.nbr3[k * 4 + f];
                T pP, unP;
                if (nb >= 0) {
                    const uint32_t info = (d.finfo3[k] >> (8 * f)) & 0xffu;
                    const int fp = info & 3, pm = info >> 2;
                    const int np_ = d.fmask3[fp * Nfp + d.perm3[pm * Nfp + j]];
                    const Q4<T> x = qold[(size_t)nb * Np + np_];
                    // Fs * n_f = nhat_f . G
                    T nx, ny, nz;
                    if (f == 0) { nx = -g[6]; ny = -g[7]; nz = -g[8]; }
                    else if (f == 1) { nx = -g[3]; ny = -g[4]; nz = -g[5]; }
                    else if (f == 2) { nx = g[0] + g[3] + g[6]; ny = g[1] + g[4] + g[7]; nz = g[2] + g[5] + g[8]; }
                    else { nx = -g[0]; ny = -g[1]; nz = -g[2]; }
                    pP = x.p;
                    unP = nx * x.u + ny * x.v + nz * x.w;
                } else {
                    pP = T(2) * d.qb3[(size_t)(-1 - nb) * Nfp + j];     // ghost state: p+ = 2 r^-, u+ = 0
                    unP = 0;
                }
                gval = g[9 + f] * (unP - unM) - g[13 + f] * (pP - m.p);
            }
            sG[fj * EPB + e] = gval;
        }
        __syncthreads();
        // ---- phase 3: D_r, D_s, D_t contraction, LIFT, update
        if (active) {
            T dpr[ET], dps[ET], dpt[ET], dvg[ET];
#pragma unroll
            for (int i = 0; i < ET; ++i) dpr[i] = dps[i] = dpt[i] = dvg[i] = 0;
            const Q4<T>* q0 = sQ + grp * ET * Np;
#pragma unroll 2
            for (int m = 0; m < Np; ++m) {
                const T dr = sD[m * Np + n], ds = sD[Np * Np + m * Np + n], dtt = sD[2 * Np * Np + m * Np + n];
#pragma unroll
                for (int i = 0; i < ET; ++i) {
                    const Q4<T> c = q0[i * Np + m];
                    dpr[i] += dr * c.p;
                    dps[i] += ds * c.p;
                    dpt[i] += dtt * c.p;
                    dvg[i] += dr * c.u;
                    dvg[i] += ds * c.v;
                    dvg[i] += dtt * c.w;
                }
            }
            T lp[ET], lx[ET], ly[ET], lz[ET];
#pragma unroll
            for (int i = 0; i < ET; ++i) lp[i] = lx[i] = ly[i] = lz[i] = 0;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                T acc[ET];
#pragma unroll
                for (int i = 0; i < ET; ++i) acc[i] = 0;
                for (int j = 0; j < Nfp; ++j) {
                    const T l = sL[(f * Nfp + j) * Np + n];
                    const T* gg = sG + (f * Nfp + j) * EPB + grp * ET;
#pragma unroll
                    for (int i = 0; i < ET; ++i) acc[i] += l * gg[i];
                }
#pragma unroll
                for (int i = 0; i < ET; ++i) {
                    const int e = grp * ET + i;
                    if (e < ne) {
                        const T* g = d.geo3 + (size_t)(e0 + e) * GEO3;
                        T nx, ny, nz;
                        if (f == 0) { nx = -g[6]; ny = -g[7]; nz = -g[8]; }
                        else if (f == 1) { nx = -g[3]; ny = -g[4]; nz = -g[5]; }
                        else if (f == 2) { nx = g[0] + g[3] + g[6]; ny = g[1] + g[4] + g[7]; nz = g[2] + g[5] + g[8]; }
                        else { nx = -g[0]; ny = -g[1]; nz = -g[2]; }
                        lp[i] += g[17 + f] * acc[i];
                        lx[i] += nx * acc[i];
                        ly[i] += ny * acc[i];
                        lz[i] += nz * acc[i];
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < ET; ++i) {
                const int e = grp * ET + i;
                if (e < ne) {
                    const size_t o = (size_t)(e0 + e) * Np + n;
                    const T* g = d.geo3 + (size_t)(e0 + e) * GEO3;
                    const T rc2 = g[21], irho = g[22], cc = g[23];
                    Q4<T> r = res[o];
                    Q4<T> v = own[i];
                    const T rp = -rc2 * (dvg[i] + lp[i]);
                    const T ru = -irho * (g[0] * dpr[i] + g[3] * dps[i] + g[6] * dpt[i]) + cc * lx[i];
                    const T rv = -irho * (g[1] * dpr[i] + g[4] * dps[i] + g[7] * dpt[i]) + cc * ly[i];
                    const T rw = -irho * (g[2] * dpr[i] + g[5] * dps[i] + g[8] * dpt[i]) + cc * lz[i];
                    r.p = rka * r.p + dt * rp;  v.p += rkb * r.p;
                    r.u = rka * r.u + dt * ru;  v.u += rkb * r.u;
                    r.v = rka * r.v + dt * rv;  v.v += rkb * r.v;
                    r.w = rka * r.w + dt * rw;  v.w += rkb * r.w;
                    res[o] = r;
                    qnew[o] = v;
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace dg
