// HABC kernels: 2D face solvers, 1D edge solvers and the face / edge / corner closures.
// These levels hold ~7 % of the unknowns at the headline size and a few per cent of the time (the paper:
// 2-4 %, Table 5), so they are written for clarity: run-time N and J, operators read through L1.
#pragma once
#include "kernels.cuh"

namespace dg {

// ---------------------------------------------------------------------------------------------------
// 2D: the J face solvers (operators reused across sets, L631).
// eq (31a-c): (1+c_i) dt p*_i + rho c^2 div_par U_i = 0 ; rho dt U_i + grad_par p_i = 0, p_i = p*_i + S.
// ---------------------------------------------------------------------------------------------------
// Threads <-> (pair, node), pair = (triangle t, set i): FACE2D_NT / max(Nfp, 3 N1) pairs per pass of a persistent CTA, the
// operators D_r, D_s, LIFT2D staged once per CTA in shared memory (transposed: lanes <-> consecutive nodes).
constexpr int FACE2D_NT = 128;

template <typename T>
__global__ void __launch_bounds__(FACE2D_NT) k_face2d(Dev<T> d, int src, T rka, T rkb, T dt) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Nfp = d.Nfp, N1 = d.N1, J = d.J, Nf = 3 * d.N1;
    const int W = max(Nfp, Nf);                   // thread slots per pair (3 N1 > Nfp for N <= 3)
    const int PB = max(1, FACE2D_NT / W);
    T* sD = reinterpret_cast<T*>(smem_raw);       // [2][Nfp(k)][Nfp(n)]
    T* sL = sD + 2 * Nfp * Nfp;                   // [3 N1 (j)][Nfp(n)]
    T* sp = sL + Nf * Nfp;                        // [PB][Nfp]
    T* su = sp + PB * Nfp;
    T* sv = su + PB * Nfp;
    T* sg = sv + PB * Nfp;                        // [PB][3 N1]
    const int tid = threadIdx.x;
    for (int idx = tid; idx < 2 * Nfp * Nfp; idx += FACE2D_NT) {
        const int a = idx / (Nfp * Nfp), r = idx - a * Nfp * Nfp, k = r / Nfp, n = r - k * Nfp;
        sD[idx] = d.D2[(size_t)a * Nfp * Nfp + n * Nfp + k];
    }
    for (int idx = tid; idx < Nf * Nfp; idx += FACE2D_NT) {
        const int j = idx / Nfp, n = idx - j * Nfp;
        sL[idx] = d.L2[n * Nf + j];
    }
    const int pl = tid / W, n = tid - pl * W;
    const bool active = pl < PB;
    const int npairs = d.Tn * J, nchunk = (npairs + PB - 1) / PB;
    const T* fold = d.fa[src];
    T* fnew = d.fa[src ^ 1];
    T* mp = sp + pl * Nfp; T* mu = su + pl * Nfp; T* mv = sv + pl * Nfp; T* mg = sg + pl * Nf;
    __syncthreads();
    for (int chunk = blockIdx.x; chunk < nchunk; chunk += gridDim.x) {
        const int pair = chunk * PB + pl;
        const bool valid = active && pair < npairs;
        const int t = valid ? pair / J : 0, i = valid ? pair - t * J : 0;
        const size_t o = (size_t)pair * 3 * Nfp;
        const T* g = d.geo2 + (size_t)t * GEO2;
        T ps = 0, u = 0, v = 0;
        if (valid && n < Nfp) {
            ps = fold[o + n]; u = fold[o + Nfp + n]; v = fold[o + 2 * Nfp + n];
            mp[n] = ps + d.S2[(size_t)t * Nfp + n]; mu[n] = u; mv[n] = v;
        }
        __syncthreads();
        if (valid && n < Nf) {
            // flux jump at edge node (e, m) of the triangle: neighbour triangle of the same domain face, or the
            // ghost state (2 r^-, 0) behind a domain edge (qb2 from the edge closure)
            const int e = n / N1, m = n - e * N1;
            const int a = d.fmask2[n];
            const int nb = d.nbr2[t * 3 + e];
            const int bnode = d.nbrnode2[(t * 3 + e) * N1 + m];
            const T nxe = g[4 + 2 * e], nye = g[5 + 2 * e];
            const T pM = mp[a], unM = nxe * mu[a] + nye * mv[a];
            T pP, unP;
            if (nb >= 0) {
                const size_t on = ((size_t)nb * J + i) * 3 * Nfp;
                pP = fold[on + bnode] + d.S2[(size_t)nb * Nfp + bnode];
                unP = nxe * fold[on + Nfp + bnode] + nye * fold[on + 2 * Nfp + bnode];
            } else {
                pP = T(2) * d.qb2[((size_t)(-1 - nb) * J + i) * N1 + bnode];
                unP = 0;
            }
            mg[n] = g[13 + e] * (unP - unM) - g[16 + e] * (pP - pM);
        }
        __syncthreads();
        if (valid && n < Nfp) {
            T pr = 0, pss = 0, ur = 0, us = 0, vr = 0, vs = 0;
            const T* Dr = sD + n;
            const T* Ds = sD + Nfp * Nfp + n;
            for (int k = 0; k < Nfp; ++k) {
                const T a_ = Dr[k * Nfp], b_ = Ds[k * Nfp];
                const T pk = mp[k], uk = mu[k], vk = mv[k];
                pr += a_ * pk; pss += b_ * pk;
                ur += a_ * uk; us += b_ * uk;
                vr += a_ * vk; vs += b_ * vk;
            }
            // G2 = (r_xi, r_eta, s_xi, s_eta)
            const T dpx = g[0] * pr + g[2] * pss, dpy = g[1] * pr + g[3] * pss;
            const T div = g[0] * ur + g[2] * us + g[1] * vr + g[3] * vs;
            T lp = 0, lx = 0, ly = 0;
            for (int ee = 0; ee < 3; ++ee) {
                T acc = 0;
                for (int k = 0; k < N1; ++k) acc += sL[(ee * N1 + k) * Nfp + n] * mg[ee * N1 + k];
                const T fs = g[10 + ee];
                lp += fs * acc; lx += fs * g[4 + 2 * ee] * acc; ly += fs * g[5 + 2 * ee] * acc;
            }
            const T rc2 = g[19], irho = g[20], cc = g[21];
            const T rp = -rc2 * (div + lp) / (T(1) + d.cn[i]);
            const T ru = -irho * dpx + cc * lx;
            const T rv = -irho * dpy + cc * ly;
            T r0 = d.fres[o + n], r1 = d.fres[o + Nfp + n], r2 = d.fres[o + 2 * Nfp + n];
            r0 = rka * r0 + dt * rp; r1 = rka * r1 + dt * ru; r2 = rka * r2 + dt * rv;
            d.fres[o + n] = r0; d.fres[o + Nfp + n] = r1; d.fres[o + 2 * Nfp + n] = r2;
            fnew[o + n] = ps + rkb * r0; fnew[o + Nfp + n] = u + rkb * r1; fnew[o + 2 * Nfp + n] = v + rkb * r2;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------
// 1D: one CTA per boundary line; thread <-> (set ij, node n).  eq (34a-b), p_ij0 by eq (32).
// ---------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T edge_pressure(const Dev<T>& d, const T* ea, int ell, int i, int j, int n) {
    const int J = d.J, N1 = d.N1;
    const T ps = ea[(((size_t)ell * J * J + i * J + j) * 2) * N1 + n];
    const T Sa = d.S1[(((size_t)ell * 2 + 0) * J + j) * N1 + n];
    const T Sb = d.S1[(((size_t)ell * 2 + 1) * J + i) * N1 + n];
    return ps + d.Cij[j * J + i] * Sb + d.Cij[i * J + j] * Sa;
}

template <typename T>
__global__ void k_edge1d(Dev<T> d, int src, T rka, T rkb, T dt) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int J = d.J, N1 = d.N1, JJ = J * J;
    T* sp = reinterpret_cast<T*>(smem_raw);       // [JJ][N1]
    T* sw = sp + JJ * N1;
    const int ell = blockIdx.x;
    const T* eold = d.ea[src];
    T* enew = d.ea[src ^ 1];
    const T* g = d.geo1 + (size_t)ell * GEO1;
    for (int idx = threadIdx.x; idx < JJ * N1; idx += blockDim.x) {
        const int ij = idx / N1, n = idx - ij * N1;
        sp[idx] = edge_pressure(d, eold, ell, ij / J, ij % J, n);
        sw[idx] = eold[(((size_t)ell * JJ + ij) * 2 + 1) * N1 + n];
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < JJ * N1; idx += blockDim.x) {
        const int ij = idx / N1, n = idx - ij * N1, i = ij / J, j = ij % J;
        T dp = 0, dw = 0;
        for (int k = 0; k < N1; ++k) {
            const T a = d.D1[n * N1 + k];
            dp += a * sp[ij * N1 + k]; dw += a * sw[ij * N1 + k];
        }
        const T rx = g[0];                        // 1/J = Fscale
        T lp = 0, lw = 0;
        for (int e = 0; e < 2; ++e) {
            const int own = e ? N1 - 1 : 0;
            const T nn = e ? T(1) : T(-1);
            const int nb = d.nbr1[ell * 2 + e];
            const T pM = sp[ij * N1 + own], unM = nn * sw[ij * N1 + own];
            T pP, unP;
            if (nb >= 0) {
                const int on = e ? 0 : N1 - 1;
                pP = edge_pressure(d, eold, nb, i, j, on);
                unP = nn * eold[(((size_t)nb * JJ + ij) * 2 + 1) * N1 + on];
            } else {
                pP = T(2) * d.qb1[(size_t)(-1 - nb) * JJ + ij];
                unP = 0;
            }
            const T gj = g[1 + e] * (unP - unM) - g[3 + e] * (pP - pM);
            const T acc = d.L1[n * 2 + e] * gj;
            lp += rx * acc; lw += rx * nn * acc;
        }
        const T rc2 = g[5], irho = g[6], cc = g[7];
        const T rp = -rc2 * (rx * dw + lp) / (T(1) + d.cn[i] + d.cn[j]);
        const T rw = -irho * rx * dp + cc * lw;
        const size_t o = (((size_t)ell * JJ + ij) * 2) * N1 + n;
        T r0 = d.eres[o], r1 = d.eres[o + N1];
        r0 = rka * r0 + dt * rp; r1 = rka * r1 + dt * rw;
        d.eres[o] = r0; d.eres[o + N1] = r1;
        enew[o] = eold[o] + rkb * r0;
        enew[o + N1] = sw[idx] + rkb * r1;
    }
}

// ---------------------------------------------------------------------------------------------------
// Closures (Algorithm 1): evaluated on the freshly updated buffers `cur`.
// ---------------------------------------------------------------------------------------------------
// face: r^+ from the 3D trace (28a), r^- = (1/M) sum c_i p*_i (30), S = r^- + r^+ (for (29))
template <typename T>
__global__ void k_close_face(Dev<T> d, int cur) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= d.Tn * d.Nfp) return;
    const int t = idx / d.Nfp, n = idx - t * d.Nfp;
    const Q4<T> q = reinterpret_cast<const Q4<T>*>(d.q[cur])[(size_t)d.tri_tet[t] * d.Np + d.fmask3[d.tri_face[t] * d.Nfp + n]];
    const int ax = d.tri_axis[t];
    const T un = T(d.tri_sign[t]) * (ax == 0 ? q.u : ax == 1 ? q.v : q.w);
    const T Z = d.geo2[(size_t)t * GEO2 + 22];
    const T rp = T(0.5) * (q.p + Z * un);
    T rm = 0;
    const T* f = d.fa[cur] + (size_t)t * d.J * 3 * d.Nfp + n;
    for (int i = 0; i < d.J; ++i) rm += d.cn[i] * f[(size_t)i * 3 * d.Nfp];
    rm *= d.invM;
    d.qb3[idx] = rm;
    d.ghost3[(size_t)idx * 4] = T(2) * rm;
    d.S2[idx] = rp + rm;
}

// edge: r^+ of both faces' 2D fields across the edge, the 2J x 2J system (33a-b) through its inverse
template <typename T>
__global__ void k_close_edge(Dev<T> d, int cur) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = d.J, N1 = d.N1, Nfp = d.Nfp;
    if (idx >= d.E * N1) return;
    const int ell = idx / N1, m = idx - ell * N1;
    T b[2 * JMAX], rp[2 * JMAX];
    // side 0 = face A supplies r^{+b}_i (stored at J+i), side 1 = face B supplies r^{+a}_j (stored at j)
    for (int side = 0; side < 2; ++side) {
        const int t = d.lin_tri[ell * 2 + side];
        const int a = d.lin_trinode[(ell * 2 + side) * N1 + m];
        const T S = d.S2[(size_t)t * Nfp + a];
        const T Z = d.geo2[(size_t)t * GEO2 + 22];
        const int slot = d.lin_slot[ell * 2 + side];
        const T sg = T(d.lin_osign[ell * 2 + side]);
        const T* f = d.fa[cur] + (size_t)t * J * 3 * Nfp;
        for (int i = 0; i < J; ++i) {
            const T p = f[(size_t)i * 3 * Nfp + a] + S;
            const T u = sg * f[(size_t)i * 3 * Nfp + (1 + slot) * Nfp + a];
            rp[(side == 0 ? J : 0) + i] = T(0.5) * (p + Z * u);
        }
    }
    const T* ea = d.ea[cur] + (size_t)ell * J * J * 2 * N1 + m;
    for (int k = 0; k < 2 * J; ++k) b[k] = 0;
    for (int i = 0; i < J; ++i)
        for (int j = 0; j < J; ++j) {
            const T ps = ea[(size_t)(i * J + j) * 2 * N1];
            b[j] += d.cn[i] * ps;            // b^a_j = sum_i c_i p*_ij
            b[J + i] += d.cn[j] * ps;        // b^b_i = sum_j c_j p*_ij
        }
    for (int r = 0; r < 2 * J; ++r) {
        T acc = 0;
        for (int k = 0; k < 2 * J; ++k) acc += d.Pe[r * 2 * J + k] * b[k] + d.Qe[r * 2 * J + k] * rp[k];
        // r < J: r^{-a}_j (for face B's fields, side 1); r >= J: r^{-b}_i (for face A's fields, side 0)
        const int side = r < J ? 1 : 0, s = r < J ? r : r - J;
        d.qb2[(((size_t)ell * 2 + side) * J + s) * N1 + m] = acc;
        d.S1[(((size_t)ell * 2 + (r < J ? 0 : 1)) * J + s) * N1 + m] = acc + rp[r];
    }
}

// corner: r^+ of the three edges' 1D fields at the corner, the 3J^2 system (35a-c) through Gc = L^-1 T
template <typename T>
__global__ void k_close_corner(Dev<T> d, int cur) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* srp = reinterpret_cast<T*>(smem_raw);      // [3 J^2]
    const int J = d.J, JJ = J * J, N1 = d.N1, c = blockIdx.x;
    for (int r = threadIdx.x; r < 3 * JJ; r += blockDim.x) {
        const int ax = r / JJ, ij = r - ax * JJ;
        const int ell = d.cor_line[c * 3 + ax];
        const int node = d.cor_end[c * 3 + ax] ? N1 - 1 : 0;
        const T p = edge_pressure(d, d.ea[cur], ell, ij / J, ij % J, node);
        const T w = d.ea[cur][(((size_t)ell * JJ + ij) * 2 + 1) * N1 + node];
        const T Z = d.geo1[(size_t)ell * GEO1 + 5] / d.geo1[(size_t)ell * GEO1 + 7];      // rho c^2 / c
        srp[r] = T(0.5) * (p + Z * T(d.cor_sign[c * 3 + ax]) * w);
    }
    __syncthreads();
    for (int r = threadIdx.x; r < 3 * JJ; r += blockDim.x) {
        T acc = 0;
        const T* row = d.Gc + (size_t)r * 3 * JJ;
        for (int k = 0; k < 3 * JJ; ++k) acc += row[k] * srp[k];
        d.qb1[(size_t)(c * 3 + r / JJ) * JJ + (r % JJ)] = acc;
    }
}

// physical auxiliary fields for dg_get_fields: p_i00 = p*_i00 + S (29), p_ij0 by (32)
template <typename T>
__global__ void k_export_aux(Dev<T> d, int cur, double* face_aux, double* edge_aux) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int J = d.J, Nfp = d.Nfp, N1 = d.N1;
    const size_t nf = (size_t)d.Tn * J * 3 * Nfp, nE = (size_t)d.E * J * J * 2 * N1;
    if (idx < nf) {
        const int n = idx % Nfp, fld = (idx / Nfp) % 3;
        const int t = idx / ((size_t)J * 3 * Nfp);
        T v = d.fa[cur][idx];
        if (fld == 0) v += d.S2[(size_t)t * Nfp + n];
        face_aux[idx] = (double)v;
    } else if (idx < nf + nE) {
        const size_t k = idx - nf;
        const int n = k % N1, fld = (k / N1) % 2, ij = (k / (2 * N1)) % (J * J);
        const int ell = k / ((size_t)J * J * 2 * N1);
        T v = d.ea[cur][k];
        if (fld == 0) v = edge_pressure(d, d.ea[cur], ell, ij / J, ij % J, n);
        edge_aux[k] = (double)v;
    }
}

}  // namespace dg
