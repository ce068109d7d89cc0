// 2D: the J face solvers of the HABC on the fp64 tensor pipe (operators reused across the sets;
// eq (31a-c):  (1+c_i) dt p*_i + rho c^2 div_par U_i = 0 ;  rho dt U_i + grad_par p_i = 0,  p_i = p*_i + S
// (eq (29)); fused volume + surface + LSRK update, Alg. 3 first half, L633-666), one launch per stage.  fp64, N <= 5;
// other cases run k_face2d (kernels_aux.cuh).
//
// Why: the scalar kernel is bound by the shared-memory pipe, not by HBM or the fp64 unit (profiles/r03_face2d.md):
// a broadcast 16-byte operand load costs four wavefronts whatever the number of distinct addresses, i.e. about one
// wavefront per DFMA instruction, and register blocking over two nodes does not change that.  With the operator rows
// register-resident as DMMA A fragments (mma.sync.m8n8k4.f64, as in kernel_vol3d_mma.cuh) one conflict-free LDS.64 per
// lane feeds 256 FMA.
//
// Work item = (triangle t, group of 4 consecutive sets i) = 4 columns of the contraction; a persistent CTA of four
// warps takes PB = 8 items (32 columns) per pass ("chunk"), warp w the n-tile of columns 8w..8w+7 (two items) with
// ALL m-tiles of D_r, D_s and LIFT2D (N = 5: 54 doubles per lane).  Nothing is loaded from global memory into
// registers ahead of its use: the raw fields of the NEXT chunk and the LSRK residual of THIS chunk travel with
// cp.async (every lane copies the residual values it will update itself), so a chunk's global latency hides under
// the previous chunk's arithmetic.  Phases of a chunk: (1) unit (item, node): p_i00 = p*_i + S, contravariant
// velocity -> operand rows [k][column]; (2) unit (item, edge node): upwind flux jump against the neighbour triangle
// of the same domain face, or the ghost state (2 r^-, 0) behind a domain edge (qb2, from the edge closure);
// (3) per warp: contractions, right-hand side and update from the accumulator fragments.
#pragma once
#include "kernel_vol3d_mma.cuh"
#include "kernels_aux.cuh"

namespace dg {

template <int N>
struct Face2dMmaCfg {
    static constexpr int Nfp = (N + 1) * (N + 2) / 2, N1 = N + 1, Nf = 3 * N1, SB = 4;
    static constexpr int MT = (Nfp + 7) / 8;            // m-tiles (8 nodes)
    static constexpr int KD = (Nfp + 3) / 4, KPD = 4 * KD;   // k-steps of D_r, D_s
    static constexpr int KL = (N1 + 3) / 4, KPL = 4 * KL;    // k-steps of one edge of LIFT2D
    static constexpr int NT = 128, PB = 8, NC = PB * SB;     // 32 columns per chunk
    static constexpr int RS = NC + 4;                   // row stride in doubles: the four k-rows of a B fragment fall 8 banks apart
    // operand rows: p_i00 [KPD] | U^r [KPD] | U^s [KPD] | flux jump [3][KPL] | u [Nfp] | v [Nfp] | p* [Nfp]
    static constexpr int rP = 0, rR = KPD, rS = 2 * KPD, rG = 3 * KPD, rU = rG + 3 * KPL, rV = rU + Nfp, rQ = rV + Nfp;
    static constexpr int ROWS = rQ + Nfp;
    static constexpr int RAW = SB * 3 * Nfp;            // staged raw fields of an item [4][3][Nfp]
    static constexpr int NRES = MT * 2 * 3;             // residual values per lane: [m-tile][column][field]
    static constexpr int oRaw = ROWS * RS;
    static constexpr int oRes = oRaw + PB * RAW;
    static constexpr int oIc = oRes + NRES * NT;
    // per-item records staged with the fields (double-buffered: phases 2 and 3 still read them while the next chunk's
    // arrive): geo2 [24] | S2 row [Nfp, padded to even] | ints: nbr2 [3], nbrnode2 [3][N1]
    static constexpr int mS = GEO2, mI = mS + Nfp + (Nfp & 1), NMI = 3 + Nf, META = mI + (NMI + 1) / 2 + ((NMI + 1) / 2 & 1);
    static constexpr int oMeta = oIc + 16;
    static constexpr size_t smem_bytes = sizeof(double) * (oMeta + 2 * PB * META);
    static_assert(GEO2 / 2 + Nfp + NMI <= 64, "metadata copy units per item");
    static constexpr int regsA = 2 * MT * (2 * KD + 3 * KL);
    static_assert(regsA <= 150, "operator fragments do not fit the register file: use k_face2d");
};

__device__ __forceinline__ void cp_async8(double* smem, const double* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NKEEP> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NKEEP) : "memory"); }

template <int N>
__global__ void __launch_bounds__(Face2dMmaCfg<N>::NT, 2) k_face2d_mma(Dev<double> d, int src, double rka, double rkb, double dt) {
    using C = Face2dMmaCfg<N>;
    constexpr int Nfp = C::Nfp, N1 = C::N1, Nf = C::Nf, SB = C::SB, MT = C::MT, KD = C::KD, KL = C::KL, KPL = C::KPL,
                  NT = C::NT, PB = C::PB, RS = C::RS, RAW = C::RAW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sOp = reinterpret_cast<double*>(smem_raw);     // [ROWS][RS]
    double* sRaw = sOp + C::oRaw;                          // [PB][4][3][Nfp]
    double* sRes = sOp + C::oRes;                          // [NRES][NT]: lane-private residual values
    double* sIc = sOp + C::oIc;                            // [J] 1 / (1 + c_i)   (eq (31a))
    double* sMeta = sOp + C::oMeta;                        // [2][PB][META]
    constexpr int META = C::META;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, t = lane & 3;
    const int J = d.J;
    const int NG = (J + SB - 1) / SB;                      // set groups per triangle
    const int nitems = d.Tn * NG, nchunk = (nitems + PB - 1) / PB;
    const double* __restrict__ fold = d.fa[src];
    double* __restrict__ fnew = d.fa[src ^ 1];
    double* __restrict__ fres = d.fres;

    for (int i = tid; i < C::ROWS * RS; i += NT) sOp[i] = 0.0;     // the k-padding rows stay zero for ever
    for (int i = tid; i < 16; i += NT) sIc[i] = i < J ? 1.0 / (1.0 + d.cn[i]) : 0.0;
    // operator rows of nodes 8 m + g as A fragments (row g, k = 4 s + t)
    double Ar[MT][KD], As[MT][KD], AL[MT][3][KL];
#pragma unroll
    for (int m = 0; m < MT; ++m) {
        const int n = 8 * m + g;
#pragma unroll
        for (int s = 0; s < KD; ++s) {
            const int k = 4 * s + t;
            const bool ok = n < Nfp && k < Nfp;
            Ar[m][s] = ok ? d.D2[(size_t)n * Nfp + k] : 0.0;
            As[m][s] = ok ? d.D2[(size_t)Nfp * Nfp + n * Nfp + k] : 0.0;
        }
#pragma unroll
        for (int e = 0; e < 3; ++e)
#pragma unroll
            for (int s = 0; s < KL; ++s) {
                const int k = 4 * s + t;
                AL[m][e][s] = (n < Nfp && k < N1) ? d.L2[n * Nf + e * N1 + k] : 0.0;
            }
    }

    // raw fields of a chunk -> sRaw (set q of item pl at [pl][q][field][node]); sets beyond J read as zero;
    // the items' records (geometry, closure S of the triangle, neighbour tables) -> sMeta[buf]
    auto issue_fields = [&](int chunk_, int buf) {
        if (chunk_ >= nchunk) return;
        for (int u = tid; u < PB * 64; u += NT) {
            const int pl = u >> 6, k = u & 63, item = chunk_ * PB + pl;
            if (item >= nitems) continue;
            const int tt = item / NG;
            double* mt = sMeta + (buf * PB + pl) * META;
            if (k < GEO2 / 2) cp_async16(mt + 2 * k, d.geo2 + (size_t)tt * GEO2 + 2 * k);
            else if (k < GEO2 / 2 + Nfp) cp_async8(mt + C::mS + (k - GEO2 / 2), d.S2 + (size_t)tt * Nfp + (k - GEO2 / 2));
            else if (k < GEO2 / 2 + Nfp + 3) cp_async4(reinterpret_cast<int*>(mt + C::mI) + (k - GEO2 / 2 - Nfp), d.nbr2 + tt * 3 + (k - GEO2 / 2 - Nfp));
            else if (k < GEO2 / 2 + Nfp + C::NMI)
                cp_async4(reinterpret_cast<int*>(mt + C::mI) + (k - GEO2 / 2 - Nfp), d.nbrnode2 + (size_t)tt * Nf + (k - GEO2 / 2 - Nfp - 3));
        }
        for (int u = tid; u < PB * Nfp; u += NT) {
            const int pl = u / Nfp, n = u - pl * Nfp, item = chunk_ * PB + pl;
            if (item >= nitems) continue;
            const int tt = item / NG, i0 = (item - tt * NG) * SB;
            const double* gp = fold + ((size_t)tt * J + i0) * 3 * Nfp + n;
            double* sp = sRaw + pl * RAW + n;
#pragma unroll
            for (int q = 0; q < SB; ++q)
#pragma unroll
                for (int f = 0; f < 3; ++f) {
                    if (i0 + q < J) cp_async8(sp + (q * 3 + f) * Nfp, gp + (size_t)(q * 3 + f) * Nfp);
                    else sp[(q * 3 + f) * Nfp] = 0.0;
                }
        }
    };
    // the accumulator fragment of lane (g, t) holds columns 2t, 2t+1 of the warp's n-tile: item pl3, sets q0, q0 + 1
    const int pl3 = 2 * wid + (t >> 1), q0 = 2 * (t & 1), col3 = 8 * wid + 2 * t;

    issue_fields(blockIdx.x, 0);
    cp_async_commit();
    int par = 0;
    for (int chunk = blockIdx.x; chunk < nchunk; chunk += gridDim.x, par ^= 1) {
        cp_async_wait<0>();
        __syncthreads();                                   // this chunk's raw fields are in; the operand rows are free
        // ---- residual values of this lane: land under phases 1-3
        const int item3 = chunk * PB + pl3;
        const bool valid3 = item3 < nitems;
        const int t3 = valid3 ? item3 / NG : 0, i03 = valid3 ? (item3 - t3 * NG) * SB : 0;
        const int ns3 = valid3 ? min(SB, J - i03) : 0;
        const size_t o3 = ((size_t)t3 * J + i03) * 3 * Nfp;
#pragma unroll
        for (int m = 0; m < MT; ++m)
#pragma unroll
            for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                for (int f = 0; f < 3; ++f)
                    if (8 * m + g < Nfp && q0 + cc < ns3)
                        cp_async8(sRes + ((m * 2 + cc) * 3 + f) * NT + tid, fres + o3 + (size_t)((q0 + cc) * 3 + f) * Nfp + 8 * m + g);
        cp_async_commit();
        // ---- phase 1: operand rows
        for (int u = tid; u < PB * Nfp; u += NT) {
            const int pl = u / Nfp, n = u - pl * Nfp, item = chunk * PB + pl;
            if (item >= nitems) continue;
            const double* gg = sMeta + (par * PB + pl) * META;   // G2 = (r_xi, r_eta, s_xi, s_eta) | n[3][2] | ...
            const double S = gg[C::mS + n];
            const double g0 = gg[0], g1 = gg[1], g2 = gg[2], g3 = gg[3];
            const double* r = sRaw + pl * RAW + n;
            double ps[SB], uu[SB], vv[SB], pp[SB], ur[SB], us[SB];
#pragma unroll
            for (int q = 0; q < SB; ++q) {
                ps[q] = r[(q * 3) * Nfp]; uu[q] = r[(q * 3 + 1) * Nfp]; vv[q] = r[(q * 3 + 2) * Nfp];
                pp[q] = ps[q] + S;
                ur[q] = g0 * uu[q] + g1 * vv[q];
                us[q] = g2 * uu[q] + g3 * vv[q];
            }
            double* mrow = sOp + n * RS + pl * SB;
            st4<double>(mrow + C::rP * RS, pp); st4<double>(mrow + C::rR * RS, ur); st4<double>(mrow + C::rS * RS, us);
            st4<double>(mrow + C::rU * RS, uu); st4<double>(mrow + C::rV * RS, vv); st4<double>(mrow + C::rQ * RS, ps);
        }
        __syncthreads();
        issue_fields(chunk + gridDim.x, par ^ 1);          // the raw buffer is free again
        cp_async_commit();
        // ---- phase 2: flux jump at edge node (e, m) of the triangle
        for (int u = tid; u < PB * Nf; u += NT) {
            const int pl = u / Nf, n = u - pl * Nf, item = chunk * PB + pl;
            if (item >= nitems) continue;
            const int tt = item / NG, i0 = (item - tt * NG) * SB, ns = min(SB, J - i0);
            const double* gg = sMeta + (par * PB + pl) * META;
            const int* gi = reinterpret_cast<const int*>(gg + C::mI);
            const int e = n / N1, m = n - e * N1;
            const int a = d.fmask2[n];
            const int nb = gi[e];
            const int bnode = gi[3 + n];
            const double nxe = gg[4 + 2 * e], nye = gg[5 + 2 * e], Ae = gg[13 + e], Be = gg[16 + e];
            const double* mo = sOp + a * RS + pl * SB;
            double pM[SB], uM[SB], vM[SB], gj[SB];
            ld4<double>(mo + C::rP * RS, pM); ld4<double>(mo + C::rU * RS, uM); ld4<double>(mo + C::rV * RS, vM);
            if (nb >= 0) {
                const double Sn = d.S2[(size_t)nb * Nfp + bnode];
                const double* fn = fold + ((size_t)nb * J + i0) * 3 * Nfp + bnode;
#pragma unroll
                for (int q = 0; q < SB; ++q) {
                    const bool ok = q < ns;
                    const double pP = (ok ? fn[(size_t)q * 3 * Nfp] : 0.0) + Sn;
                    const double uP = ok ? fn[(size_t)q * 3 * Nfp + Nfp] : 0.0;
                    const double vP = ok ? fn[(size_t)q * 3 * Nfp + 2 * Nfp] : 0.0;
                    gj[q] = Ae * ((nxe * uP + nye * vP) - (nxe * uM[q] + nye * vM[q])) - Be * (pP - pM[q]);
                }
            } else {
                const double* qb = d.qb2 + ((size_t)(-1 - nb) * J + i0) * N1 + bnode;
#pragma unroll
                for (int q = 0; q < SB; ++q) {
                    const double pP = q < ns ? 2.0 * qb[(size_t)q * N1] : 0.0;
                    gj[q] = Ae * (0.0 - (nxe * uM[q] + nye * vM[q])) - Be * (pP - pM[q]);
                }
            }
            st4<double>(sOp + (C::rG + e * KPL + m) * RS + pl * SB, gj);
        }
        __syncthreads();
        // ---- phase 3: contractions (DMMA), right-hand side and LSRK update from the accumulator fragments
        const double* gg = sMeta + (par * PB + pl3) * META;
        const double g0 = gg[0], g1 = gg[1], g2 = gg[2], g3 = gg[3];
        const double rc2 = gg[19], irho = gg[20], cc_ = gg[21];
        const double fs0 = gg[10], fs1 = gg[11], fs2 = gg[12];
        const double fx0 = fs0 * gg[4], fy0 = fs0 * gg[5], fx1 = fs1 * gg[6], fy1 = fs1 * gg[7], fx2 = fs2 * gg[8], fy2 = fs2 * gg[9];
        const double* bp = sOp + t * RS + 8 * wid + g;     // B fragment: row 4 s + t, column 8 w + g
        cp_async_wait<1>();                                // this lane's residual values (the newer group is the next chunk's fields)
#pragma unroll
        for (int m = 0; m < MT; ++m) {
            double pr[2] = {0, 0}, pq[2] = {0, 0}, dv[2] = {0, 0}, dw[2] = {0, 0}, e0[2] = {0, 0}, e1[2] = {0, 0}, e2[2] = {0, 0};
#pragma unroll
            for (int s = 0; s < KD; ++s) {
                const double b0 = bp[(C::rP + 4 * s) * RS], b1 = bp[(C::rR + 4 * s) * RS], b2 = bp[(C::rS + 4 * s) * RS];
                dmma884(pr, Ar[m][s], b0);
                dmma884(pq, As[m][s], b0);
                dmma884(dv, Ar[m][s], b1);
                dmma884(dw, As[m][s], b2);
            }
#pragma unroll
            for (int s = 0; s < KL; ++s) {
                dmma884(e0, AL[m][0][s], bp[(C::rG + 4 * s) * RS]);
                dmma884(e1, AL[m][1][s], bp[(C::rG + KPL + 4 * s) * RS]);
                dmma884(e2, AL[m][2][s], bp[(C::rG + 2 * KPL + 4 * s) * RS]);
            }
            const int n = 8 * m + g;
            if (n < Nfp && ns3 > q0) {
                const double2 ps = *reinterpret_cast<const double2*>(sOp + (C::rQ + n) * RS + col3);
                const double2 uu = *reinterpret_cast<const double2*>(sOp + (C::rU + n) * RS + col3);
                const double2 vv = *reinterpret_cast<const double2*>(sOp + (C::rV + n) * RS + col3);
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int q = q0 + c;
                    if (q < ns3) {
                        const double dpx = g0 * pr[c] + g2 * pq[c], dpy = g1 * pr[c] + g3 * pq[c];
                        const double lp = fs0 * e0[c] + fs1 * e1[c] + fs2 * e2[c];
                        const double lx = fx0 * e0[c] + fx1 * e1[c] + fx2 * e2[c];
                        const double ly = fy0 * e0[c] + fy1 * e1[c] + fy2 * e2[c];
                        const double rp = -rc2 * ((dv[c] + dw[c]) + lp) * sIc[i03 + q];
                        const double ru = -irho * dpx + cc_ * lx;
                        const double rv = -irho * dpy + cc_ * ly;
                        const double* rs = sRes + ((m * 2 + c) * 3) * NT + tid;
                        const double a0 = rka * rs[0] + dt * rp, a1 = rka * rs[NT] + dt * ru, a2 = rka * rs[2 * NT] + dt * rv;
                        const size_t oq = o3 + (size_t)q * 3 * Nfp + n;
                        fres[oq] = a0; fres[oq + Nfp] = a1; fres[oq + 2 * Nfp] = a2;
                        fnew[oq] = (c ? ps.y : ps.x) + rkb * a0;
                        fnew[oq + Nfp] = (c ? uu.y : uu.x) + rkb * a1;
                        fnew[oq + 2 * Nfp] = (c ? vv.y : vv.x) + rkb * a2;
                    }
                }
            }
        }
    }
    cp_async_wait<0>();
}

}  // namespace dg
