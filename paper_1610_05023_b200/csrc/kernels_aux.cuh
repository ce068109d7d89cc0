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
// Work item = (triangle t, group of FACE2D_SB = 4 consecutive sets i); thread <-> (item, node), FACE2D_NT /
// max(Nfp, 3 N1) items per pass of a persistent CTA.  The operators D_r, D_s, LIFT2D are staged once per CTA in
// shared memory (transposed: lanes <-> consecutive nodes) and every operator entry a thread fetches is used for the
// four sets of its item (fields stored [node][set], one 32-byte broadcast load per field): 2 + 3 shared loads
// per 16 FMA instead of 5 per 6, which is what moves the kernel from the shared-memory pipe (profiles/
// r02_face2d_ncu.md: L1 data pipe 66 %, 657 us) to the FMA pipe.  The sets of one triangle also share its
// geometry, its cached closure S and its neighbour lookups.
constexpr int FACE2D_NT = 128;
constexpr int FACE2D_SB = 4;

template <typename T> __device__ __forceinline__ void ld4(const T* p, T (&v)[4]);
template <> __device__ __forceinline__ void ld4<double>(const double* p, double (&v)[4]) {
    const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
template <> __device__ __forceinline__ void ld4<float>(const float* p, float (&v)[4]) {
    const float4 a = *reinterpret_cast<const float4*>(p);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
}
template <typename T> __device__ __forceinline__ void st4(T* p, const T (&v)[4]);
template <> __device__ __forceinline__ void st4<double>(double* p, const double (&v)[4]) {
    *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    *reinterpret_cast<double2*>(p + 2) = make_double2(v[2], v[3]);
}
template <> __device__ __forceinline__ void st4<float>(float* p, const float (&v)[4]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}

__host__ __device__ inline int face2d_ops_elems(int Nfp, int N1) {          // operators + 1/(1+c_i), padded to 4
    return ((2 * Nfp * Nfp + 3 * N1 * Nfp + 3) / 4) * 4 + 16;
}

constexpr int FACE2D_MINB = 4;        // resident CTAs per SM the register budget is set for
template <typename T>
__global__ void __launch_bounds__(FACE2D_NT, FACE2D_MINB) k_face2d(Dev<T> d, int src, T rka, T rkb, T dt) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int SB = FACE2D_SB;
    const int Nfp = d.Nfp, N1 = d.N1, J = d.J, Nf = 3 * d.N1;
    const int W = max(Nfp, Nf);                   // thread slots per item (3 N1 > Nfp for N <= 3)
    const int PB = max(1, FACE2D_NT / W);
    const int NG = (J + SB - 1) / SB;             // set groups per triangle
    T* sD = reinterpret_cast<T*>(smem_raw);       // [2][Nfp(k)][Nfp(n)]
    T* sL = sD + 2 * Nfp * Nfp;                   // [3 N1 (j)][Nfp(n)]
    T* sIc = sD + face2d_ops_elems(Nfp, N1) - 16; // [J] 1 / (1 + c_i)   (eq (31a))
    T* sp = sD + face2d_ops_elems(Nfp, N1);       // [PB][Nfp][SB]  p_i00 = p*_i + S   (eq (29))
    T* sr = sp + PB * Nfp * SB;                   //                contravariant velocity U^r
    T* ss = sr + PB * Nfp * SB;                   //                U^s
    T* su = ss + PB * Nfp * SB;                   //                u, v (for the traces)
    T* sv = su + PB * Nfp * SB;
    T* sg = sv + PB * Nfp * SB;                   // [PB][3 N1][SB] flux jumps
    const int tid = threadIdx.x;
    for (int idx = tid; idx < 2 * Nfp * Nfp; idx += FACE2D_NT) {
        const int a = idx / (Nfp * Nfp), r = idx - a * Nfp * Nfp, k = r / Nfp, n = r - k * Nfp;
        sD[idx] = d.D2[(size_t)a * Nfp * Nfp + n * Nfp + k];
    }
    for (int idx = tid; idx < Nf * Nfp; idx += FACE2D_NT) {
        const int j = idx / Nfp, n = idx - j * Nfp;
        sL[idx] = d.L2[n * Nf + j];
    }
    for (int i = tid; i < 16; i += FACE2D_NT) sIc[i] = i < J ? T(1) / (T(1) + d.cn[i]) : T(0);
    const int pl = tid / W, n = tid - pl * W;
    const bool active = pl < PB;
    const int nitems = d.Tn * NG, nchunk = (nitems + PB - 1) / PB;
    const T* __restrict__ fold = d.fa[src];
    T* __restrict__ fnew = d.fa[src ^ 1];
    T* mp = sp + pl * Nfp * SB; T* mr = sr + pl * Nfp * SB; T* ms = ss + pl * Nfp * SB;
    T* mu = su + pl * Nfp * SB; T* mv = sv + pl * Nfp * SB; T* mg = sg + pl * Nf * SB;
    __syncthreads();
    // fields of this thread's (item, node) for the current chunk; loaded one chunk ahead (global latency is the
    // cost of this kernel: the same warps load, exchange through shared memory, gather and compute)
    T ps[SB], u[SB], v[SB];
    auto load_fields = [&](int chunk_, T (&a_)[SB], T (&b_)[SB], T (&c_)[SB]) {
        const int item_ = chunk_ * PB + pl;
        const bool ok_ = active && chunk_ < nchunk && item_ < nitems && n < Nfp;
        const int t_ = ok_ ? item_ / NG : 0, i0_ = ok_ ? (item_ - t_ * NG) * SB : 0;
        const size_t o_ = ((size_t)t_ * J + i0_) * 3 * Nfp + n;
#pragma unroll
        for (int q = 0; q < SB; ++q) {
            const bool okq = ok_ && i0_ + q < J;
            a_[q] = okq ? fold[o_ + (size_t)q * 3 * Nfp] : T(0);
            b_[q] = okq ? fold[o_ + (size_t)q * 3 * Nfp + Nfp] : T(0);
            c_[q] = okq ? fold[o_ + (size_t)q * 3 * Nfp + 2 * Nfp] : T(0);
        }
    };
    load_fields(blockIdx.x, ps, u, v);
    for (int chunk = blockIdx.x; chunk < nchunk; chunk += gridDim.x) {
        const int item = chunk * PB + pl;
        const bool valid = active && item < nitems;
        const int t = valid ? item / NG : 0, i0 = valid ? (item - t * NG) * SB : 0;
        const int ns = min(SB, J - i0);
        const size_t o = ((size_t)t * J + i0) * 3 * Nfp;          // set q of the item at o + q * 3 Nfp
        const T* g = d.geo2 + (size_t)t * GEO2;                   // G2 = (r_xi, r_eta, s_xi, s_eta) | n[3][2] | ...
        if (valid && n < Nfp) {
            const T S = d.S2[(size_t)t * Nfp + n];
            const T g0 = g[0], g1 = g[1], g2 = g[2], g3 = g[3];
            T pp[SB], ur[SB], us[SB];
#pragma unroll
            for (int q = 0; q < SB; ++q) {
                pp[q] = ps[q] + S;
                ur[q] = g0 * u[q] + g1 * v[q];
                us[q] = g2 * u[q] + g3 * v[q];
            }
            st4<T>(mp + n * SB, pp); st4<T>(mr + n * SB, ur); st4<T>(ms + n * SB, us);
            st4<T>(mu + n * SB, u); st4<T>(mv + n * SB, v);
        }
        __syncthreads();
        if (valid && n < Nf) {
            // flux jump at edge node (e, m) of the triangle: neighbour triangle of the same domain face, or the
            // ghost state (2 r^-, 0) behind a domain edge (qb2 from the edge closure)
            const int e = n / N1, m = n - e * N1;
            const int a = d.fmask2[n];
            const int nb = d.nbr2[t * 3 + e];
            const int bnode = d.nbrnode2[(t * 3 + e) * N1 + m];
            const T nxe = g[4 + 2 * e], nye = g[5 + 2 * e], Ae = g[13 + e], Be = g[16 + e];
            T pM[SB], uM[SB], vM[SB], gj[SB];
            ld4<T>(mp + a * SB, pM); ld4<T>(mu + a * SB, uM); ld4<T>(mv + a * SB, vM);
            if (nb >= 0) {
                const T Sn = d.S2[(size_t)nb * Nfp + bnode];
                const size_t on = ((size_t)nb * J + i0) * 3 * Nfp + bnode;
#pragma unroll
                for (int q = 0; q < SB; ++q) {
                    const bool ok = q < ns;
                    const T pP = (ok ? fold[on + (size_t)q * 3 * Nfp] : T(0)) + Sn;
                    const T uP = ok ? fold[on + (size_t)q * 3 * Nfp + Nfp] : T(0);
                    const T vP = ok ? fold[on + (size_t)q * 3 * Nfp + 2 * Nfp] : T(0);
                    gj[q] = Ae * ((nxe * uP + nye * vP) - (nxe * uM[q] + nye * vM[q])) - Be * (pP - pM[q]);
                }
            } else {
                const T* qb = d.qb2 + ((size_t)(-1 - nb) * J + i0) * N1 + bnode;
#pragma unroll
                for (int q = 0; q < SB; ++q) {
                    const T pP = q < ns ? T(2) * qb[(size_t)q * N1] : T(0);
                    gj[q] = Ae * (T(0) - (nxe * uM[q] + nye * vM[q])) - Be * (pP - pM[q]);
                }
            }
            st4<T>(mg + n * SB, gj);
        }
        __syncthreads();
        T nps[SB], nu[SB], nv[SB];
        load_fields(chunk + gridDim.x, nps, nu, nv);
        if (valid && n < Nfp) {
            T f0[SB], f1[SB], f2[SB];                             // res of this (item, node): loaded before the contraction
#pragma unroll
            for (int q = 0; q < SB; ++q) {
                const size_t oq = o + (size_t)q * 3 * Nfp + n;
                f0[q] = q < ns ? d.fres[oq] : T(0); f1[q] = q < ns ? d.fres[oq + Nfp] : T(0); f2[q] = q < ns ? d.fres[oq + 2 * Nfp] : T(0);
            }
            T pr[SB], pq[SB], dv[SB];
#pragma unroll
            for (int q = 0; q < SB; ++q) pr[q] = pq[q] = dv[q] = T(0);
            const T* Dr = sD + n;
            const T* Ds = sD + Nfp * Nfp + n;
            for (int k = 0; k < Nfp; ++k) {
                const T a_ = Dr[k * Nfp], b_ = Ds[k * Nfp];
                T pk[SB], rk[SB], sk[SB];
                ld4<T>(mp + k * SB, pk); ld4<T>(mr + k * SB, rk); ld4<T>(ms + k * SB, sk);
#pragma unroll
                for (int q = 0; q < SB; ++q) {
                    pr[q] += a_ * pk[q]; pq[q] += b_ * pk[q];
                    dv[q] += a_ * rk[q]; dv[q] += b_ * sk[q];
                }
            }
            T lp[SB], lx[SB], ly[SB];
#pragma unroll
            for (int q = 0; q < SB; ++q) lp[q] = lx[q] = ly[q] = T(0);
            for (int ee = 0; ee < 3; ++ee) {
                T acc[SB];
#pragma unroll
                for (int q = 0; q < SB; ++q) acc[q] = T(0);
                for (int k = 0; k < N1; ++k) {
                    const T l = sL[(ee * N1 + k) * Nfp + n];
                    T gk[SB];
                    ld4<T>(mg + (ee * N1 + k) * SB, gk);
#pragma unroll
                    for (int q = 0; q < SB; ++q) acc[q] += l * gk[q];
                }
                const T fs = g[10 + ee], fx = fs * g[4 + 2 * ee], fy = fs * g[5 + 2 * ee];
#pragma unroll
                for (int q = 0; q < SB; ++q) { lp[q] += fs * acc[q]; lx[q] += fx * acc[q]; ly[q] += fy * acc[q]; }
            }
            const T g0 = g[0], g1 = g[1], g2 = g[2], g3 = g[3];
            const T rc2 = g[19], irho = g[20], cc = g[21];
#pragma unroll
            for (int q = 0; q < SB; ++q) {
                if (q < ns) {
                    const size_t oq = o + (size_t)q * 3 * Nfp + n;
                    const T dpx = g0 * pr[q] + g2 * pq[q], dpy = g1 * pr[q] + g3 * pq[q];
                    const T rp = -rc2 * (dv[q] + lp[q]) * sIc[i0 + q];
                    const T ru = -irho * dpx + cc * lx[q];
                    const T rv = -irho * dpy + cc * ly[q];
                    T r0 = f0[q], r1 = f1[q], r2 = f2[q];
                    r0 = rka * r0 + dt * rp; r1 = rka * r1 + dt * ru; r2 = rka * r2 + dt * rv;
                    d.fres[oq] = r0; d.fres[oq + Nfp] = r1; d.fres[oq + 2 * Nfp] = r2;
                    fnew[oq] = ps[q] + rkb * r0; fnew[oq + Nfp] = u[q] + rkb * r1; fnew[oq + 2 * Nfp] = v[q] + rkb * r2;
                }
            }
        }
#pragma unroll
        for (int q = 0; q < SB; ++q) { ps[q] = nps[q]; u[q] = nu[q]; v[q] = nv[q]; }
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
    extern __shared__ __align__(128) unsigned char smem_raw[];
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

// edge: r^+ of both faces' 2D fields across the edge, the 2J x 2J system (33a-b) through its inverse.
// One WARP per edge node, lane k <-> unknown k of (r^{-a}_j ; r^{-b}_i): every lane gathers its own r^+ and
// right-hand side b, the vectors are exchanged through shared memory and lane r takes row r of the inverse
// (stored transposed: coalesced).  The first version ran one THREAD per node (~600 dependent loads, 60 us of
// pure latency whatever the mesh size).
constexpr int CLOSE_EDGE_WARPS = 4;
template <typename T>
__global__ void __launch_bounds__(32 * CLOSE_EDGE_WARPS) k_close_edge(Dev<T> d, int cur) {
    __shared__ T sb[CLOSE_EDGE_WARPS][2 * JMAX], srp[CLOSE_EDGE_WARPS][2 * JMAX];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int node = blockIdx.x * CLOSE_EDGE_WARPS + wl;
    const int J = d.J, N1 = d.N1, Nfp = d.Nfp, J2 = 2 * J;
    if (node >= d.E * N1) return;
    const int ell = node / N1, m = node - ell * N1;
    T rpk = 0;
    if (lane < J2) {
        // unknown k < J: r^{-a}_j, its r^{+a}_j comes from face B (side 1); k >= J: r^{-b}_i, r^{+b}_i from face A (side 0)
        const int side = lane < J ? 1 : 0, sidx = lane < J ? lane : lane - J;
        const int t = d.lin_tri[ell * 2 + side];
        const int a = d.lin_trinode[(ell * 2 + side) * N1 + m];
        const T S = d.S2[(size_t)t * Nfp + a];
        const T Z = d.geo2[(size_t)t * GEO2 + 22];
        const int slot = d.lin_slot[ell * 2 + side];
        const T sg = T(d.lin_osign[ell * 2 + side]);
        const T* f = d.fa[cur] + ((size_t)t * J + sidx) * 3 * Nfp;
        const T p = f[a] + S;
        const T u = sg * f[(1 + slot) * Nfp + a];
        rpk = T(0.5) * (p + Z * u);
        // b^a_j = sum_i c_i p*_ij ; b^b_i = sum_j c_j p*_ij
        const T* ea = d.ea[cur] + (size_t)ell * J * J * 2 * N1 + m;
        T bk = 0;
        for (int q = 0; q < J; ++q) {
            const int ij = lane < J ? q * J + sidx : sidx * J + q;
            bk += d.cn[q] * ea[(size_t)ij * 2 * N1];
        }
        sb[wl][lane] = bk;
        srp[wl][lane] = rpk;
    }
    __syncwarp();
    if (lane < J2) {
        T acc0 = 0, acc1 = 0;
        for (int k = 0; k < J2; ++k) {
            acc0 += d.PeT[k * J2 + lane] * sb[wl][k];
            acc1 += d.QeT[k * J2 + lane] * srp[wl][k];
        }
        const T acc = acc0 + acc1;
        // r < J: r^{-a}_j (for face B's fields, side 1); r >= J: r^{-b}_i (for face A's fields, side 0)
        const int r = lane, side = r < J ? 1 : 0, sidx = r < J ? r : r - J;
        d.qb2[(((size_t)ell * 2 + side) * J + sidx) * N1 + m] = acc;
        d.S1[(((size_t)ell * 2 + (r < J ? 0 : 1)) * J + sidx) * N1 + m] = acc + rpk;
    }
}

// corner: r^+ of the three edges' 1D fields at the corner, the 3J^2 system (35a-c) through Gc = L^-1 T.
// One CTA per corner; one WARP per row of Gc at a time, lanes across the columns (coalesced row reads, all loads
// independent), shuffle reduction.
template <typename T>
__global__ void k_close_corner(Dev<T> d, int cur) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* srp = reinterpret_cast<T*>(smem_raw);      // [3 J^2]
    const int J = d.J, JJ = J * J, N1 = d.N1, c = blockIdx.x, n3 = 3 * JJ;
    for (int r = threadIdx.x; r < n3; r += blockDim.x) {
        const int ax = r / JJ, ij = r - ax * JJ;
        const int ell = d.cor_line[c * 3 + ax];
        const int node = d.cor_end[c * 3 + ax] ? N1 - 1 : 0;
        const T p = edge_pressure(d, d.ea[cur], ell, ij / J, ij % J, node);
        const T w = d.ea[cur][(((size_t)ell * JJ + ij) * 2 + 1) * N1 + node];
        const T Z = d.geo1[(size_t)ell * GEO1 + 5] / d.geo1[(size_t)ell * GEO1 + 7];      // rho c^2 / c
        srp[r] = T(0.5) * (p + Z * T(d.cor_sign[c * 3 + ax]) * w);
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int r = wl; r < n3; r += nw) {
        const T* row = d.Gc + (size_t)r * n3;
        T acc = 0;
        for (int k = lane; k < n3; k += 32) acc += row[k] * srp[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) d.qb1[(size_t)(c * 3 + r / JJ) * JJ + (r % JJ)] = acc;
    }
}

// Point source delta(x - xs) S(t) in the pressure equation (S = integral of the Ricker wavelet (44)).
// Runs right after the 3D kernel of a stage: the fused kernel has applied res = a res + dt F, q += b res, and F
// is linear in the source, so the source's share is res_p += dt f, q_p += b dt f on the nodes of the source cell.
// The simulated time lives on the device (the step is replayed as a CUDA graph): *t_dev is the time at the start of
// the step, the last stage's launch advances it.
template <typename T>
__global__ void k_source(T* __restrict__ qnew, T* __restrict__ res, const T* __restrict__ w, int k, int Np, double* t_dev,
                         double rkc_dt, double dt, double rkb, double fpeak, double ts, double amp, int last) {
    const double t = *t_dev + rkc_dt;
    __syncthreads();
    const double tau = t - ts, a = 3.14159265358979323846 * fpeak * tau;
    const double S = amp * tau * exp(-a * a);
    for (int n = threadIdx.x; n < Np; n += blockDim.x) {
        const double f = S * (double)w[n];
        const size_t o = ((size_t)k * Np + n) * 4;
        res[o] = (T)((double)res[o] + dt * f);
        qnew[o] = (T)((double)qnew[o] + rkb * dt * f);
    }
    if (last && threadIdx.x == 0) *t_dev = *t_dev + dt;
}

// dg_set_initial / dg_get_fields: interface arrays are fp64 [K][Np] per field; the device state is [K][Np][4] of T
template <typename T>
__global__ void k_pack_field(const double* __restrict__ stage, T* __restrict__ q, int fld, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) q[i * 4 + fld] = (T)stage[i];
}
template <typename T>
__global__ void k_unpack_field(const T* __restrict__ q, double* __restrict__ stage, int fld, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) stage[i] = (double)q[i * 4 + fld];
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
