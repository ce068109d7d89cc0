// 3D solver, fp64, tensor-pipe kernel for the degrees whose operator rows do not fit the register file (N >= 6):
// fused volume + surface + update of one LSRK stage (Alg. 2, eq (41)-(43)).
// Same mathematics and the same DMMA fragments as kernel_vol3d_mma.cuh (m-tile = 8 nodes, n-tile = 8 elements, k = 4),
// but the A fragments (rows of D_r, D_s, D_t, LIFT) are fetched per use from global memory, where the host has laid
// the operators out in FRAGMENT ORDER, zero-padded: Dfrag [3][MT][KD][32], Lfrag [4][MT][KL][32], entry (a, mt, s, lane
// = 4 g + t) = D_a[n = 8 mt + g][m = 4 s + t].  A fragment is then one unconditional, fully coalesced 256-byte load per
// warp (two wavefronts; the transposed operator array cost four 64-byte row segments and a bounds check per value),
// and the arrays stay L1/L2-resident (N = 8: 0.9 MB).  An A fragment feeds NTILE n-tiles (NTILE * 8 elements per
// batch), which divides the operator traffic per element by NTILE.
//   phase 1  all threads: (p, contravariant velocity) of every node of the batch -> B operand rows [k][8] per n-tile
//   phase 2  all threads: one upwind flux jump per face node  -> B operand rows of the LIFT part
//   phase 3  warp w loops over the m-tiles w, w+W, ...: 6 KD + 4 KL DMMA per n-tile, then the right-hand side and
//            the LSRK update of its 8 nodes x NTILE*8 elements straight from the accumulators (q, res from global)
#pragma once
#include "kernel_vol3d_mma.cuh"

namespace dg {

template <int N, int NTILE, int W>
struct MmagCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EPB = 8 * NTILE;
    static constexpr int MT = (Np + 7) / 8;
    static constexpr int KD = (Np + 3) / 4, KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4, KPL = KL * 4;
    static constexpr int NT = 32 * W;
    static constexpr int szT = (4 * KPD + 4 * KPL) * 8;             // operand rows of one n-tile, in doubles
    static constexpr size_t smem_bytes = sizeof(double) * NTILE * szT + 16;
};

template <int N, int NTILE, int W>
__global__ void __launch_bounds__(MmagCfg<N, NTILE, W>::NT)
k_vol3d_mmag(Dev<double> d, int src, double rka, double rkb, double dt) {
    using C = MmagCfg<N, NTILE, W>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EPB = C::EPB, MT = C::MT, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  KPL = C::KPL, NT = C::NT, szT = C::szT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sB = reinterpret_cast<double*>(smem_raw);       // [NTILE][p | U^r | U^s | U^t : KPD rows each | g_f : KPL rows each][8]
    const double* __restrict__ qold = d.q[src];
    double* __restrict__ qnew = d.q[src ^ 1];
    double* __restrict__ res = d.res;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int K = d.K;
    const int nbatch = (K + EPB - 1) / EPB;

    // padding rows (k >= Np, j >= Nfp) stay zero for ever
    for (int i = tid; i < NTILE * szT; i += NT) sB[i] = 0.0;
    __syncthreads();

    for (int batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        const int e0 = batch * EPB;
        // ---- phase 1: operands (one column per element, columns swizzled as in kernel_vol3d_mma.cuh)
        for (int idx = tid; idx < EPB * Np; idx += NT) {
            const int e = idx / Np, n = idx - e * Np;
            const int k = min(e0 + e, K - 1);               // elements past the end repeat the last one (never stored)
            const double* ge = d.geo3 + (size_t)k * GEO3;
            const double2 v0 = *reinterpret_cast<const double2*>(qold + ((size_t)k * Np + n) * 4);
            const double2 v1 = *reinterpret_cast<const double2*>(qold + ((size_t)k * Np + n) * 4 + 2);
            double* o = sB + (e >> 3) * szT + n * 8 + ((e & 7) ^ swz(n));
            o[0] = v0.x;
            o[KPD * 8] = ge[0] * v0.y + ge[1] * v1.x + ge[2] * v1.y;
            o[2 * KPD * 8] = ge[3] * v0.y + ge[4] * v1.x + ge[5] * v1.y;
            o[3 * KPD * 8] = ge[6] * v0.y + ge[7] * v1.x + ge[8] * v1.y;
        }
        __syncthreads();
        // ---- phase 2: g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-); Fs n.u- = nhat . U- from the operands
        for (int idx = tid; idx < EPB * Nfn; idx += NT) {
            const int e = idx / Nfn, fj = idx - e * Nfn;
            const int f = fj / Nfp, j = fj - f * Nfp;
            const int k = min(e0 + e, K - 1);
            const double* ge = d.geo3 + (size_t)k * GEO3;
            const int nm = d.fmask3[fj];
            const double* om = sB + (e >> 3) * szT + nm * 8 + ((e & 7) ^ swz(nm));
            const double pM = om[0], Ur = om[KPD * 8], Us = om[2 * KPD * 8], Ut = om[3 * KPD * 8];
            const double unM = (f == 0) ? -Ut : (f == 1) ? -Us : (f == 2) ? (Ur + Us + Ut) : -Ur;
            const int nb = d.nbr3[k * 4 + f];
            double pP, unP;
            if (nb >= 0) {
                const uint32_t info = (d.finfo3[k] >> (8 * f)) & 0xffu;
                const int fp = info & 3, pm = info >> 2;
                const int np_ = d.fmask3[fp * Nfp + d.perm3[pm * Nfp + j]];
                const double2 x0 = *reinterpret_cast<const double2*>(qold + ((size_t)nb * Np + np_) * 4);
                const double2 x1 = *reinterpret_cast<const double2*>(qold + ((size_t)nb * Np + np_) * 4 + 2);
                double nx, ny, nz;
                if (f == 0) { nx = -ge[6]; ny = -ge[7]; nz = -ge[8]; }
                else if (f == 1) { nx = -ge[3]; ny = -ge[4]; nz = -ge[5]; }
                else if (f == 2) { nx = ge[0] + ge[3] + ge[6]; ny = ge[1] + ge[4] + ge[7]; nz = ge[2] + ge[5] + ge[8]; }
                else { nx = -ge[0]; ny = -ge[1]; nz = -ge[2]; }
                pP = x0.x;
                unP = nx * x0.y + ny * x1.x + nz * x1.y;
            } else {
                pP = 2.0 * d.qb3[(size_t)(-1 - nb) * Nfp + j];          // ghost state: p+ = 2 r^-, u+ = 0
                unP = 0;
            }
            sB[(e >> 3) * szT + (4 * KPD + f * KPL + j) * 8 + ((e & 7) ^ swz(j))] = ge[9 + f] * (unP - unM) - ge[13 + f] * (pP - pM);
        }
        __syncthreads();
        // ---- phase 3: contractions and update, one m-tile at a time
        for (int mt = w; mt < MT; mt += W) {
            const int n = 8 * mt + g;
            const bool nok = n < Np;
            double acc[NTILE][10][2];
#pragma unroll
            for (int q = 0; q < NTILE; ++q)
#pragma unroll
                for (int v = 0; v < 10; ++v) acc[q][v][0] = acc[q][v][1] = 0.0;
            const double* bp = sB + t * 8 + (g ^ swz(t));
            // operator fragments one k-step ahead: their L1/L2 latency is the cost of this kernel
            const double* fD = d.Dfrag + (size_t)mt * KD * 32 + lane;
            auto loadD = [&](int s_, double& ar, double& as, double& at) {
                ar = fD[s_ * 32];
                as = fD[(MT * KD + s_) * 32];
                at = fD[(2 * MT * KD + s_) * 32];
            };
            double ar, as, at;
            loadD(0, ar, as, at);
#pragma unroll 2
            for (int s_ = 0; s_ < KD; ++s_) {
                double nr, ns, nt_;
                loadD(min(s_ + 1, KD - 1), nr, ns, nt_);
#pragma unroll
                for (int q = 0; q < NTILE; ++q) {
                    const double* b = bp + q * szT + (4 * s_) * 8;
                    const double b0 = b[0];
                    dmma884(acc[q][0], ar, b0);
                    dmma884(acc[q][1], as, b0);
                    dmma884(acc[q][2], at, b0);
                    dmma884(acc[q][3], ar, b[KPD * 8]);
                    dmma884(acc[q][4], as, b[2 * KPD * 8]);
                    dmma884(acc[q][5], at, b[3 * KPD * 8]);
                }
                ar = nr; as = ns; at = nt_;
            }
            const double* fL = d.Lfrag + (size_t)mt * KL * 32 + lane;
            for (int s_ = 0; s_ < KL; ++s_) {
#pragma unroll
                for (int f = 0; f < 4; ++f) {
                    const double al = fL[(f * MT * KL + s_) * 32];
#pragma unroll
                    for (int q = 0; q < NTILE; ++q)
                        dmma884(acc[q][6 + f], al, bp[q * szT + (4 * KPD + f * KPL + 4 * s_) * 8]);
                }
            }
            // right-hand side and LSRK update (eq (41)-(43)) of node n, elements 8 q + 2 t + ee
            if (nok) {
#pragma unroll
                for (int q = 0; q < NTILE; ++q)
#pragma unroll
                    for (int ee = 0; ee < 2; ++ee) {
                        const int k = e0 + 8 * q + 2 * t + ee;
                        if (k < K) {
                            const double* ge = d.geo3 + (size_t)k * GEO3;
                            const double a0 = acc[q][6][ee], a1 = acc[q][7][ee], a2 = acc[q][8][ee], a3 = acc[q][9][ee];
                            const double lp = ge[17] * a0 + ge[18] * a1 + ge[19] * a2 + ge[20] * a3;
                            const double rc2 = ge[21], irho = ge[22], cc = ge[23];
                            const double xr = cc * (a2 - a3) - irho * acc[q][0][ee];
                            const double xs = cc * (a2 - a1) - irho * acc[q][1][ee];
                            const double xt = cc * (a2 - a0) - irho * acc[q][2][ee];
                            const double rp = -rc2 * ((acc[q][3][ee] + acc[q][4][ee]) + acc[q][5][ee] + lp);
                            const double ru = ge[0] * xr + ge[3] * xs + ge[6] * xt;
                            const double rv = ge[1] * xr + ge[4] * xs + ge[7] * xt;
                            const double rw = ge[2] * xr + ge[5] * xs + ge[8] * xt;
                            const size_t o = ((size_t)k * Np + n) * 4;
                            double2 q0 = *reinterpret_cast<const double2*>(qold + o);
                            double2 q1 = *reinterpret_cast<const double2*>(qold + o + 2);
                            double2 r0 = *reinterpret_cast<const double2*>(res + o);
                            double2 r1 = *reinterpret_cast<const double2*>(res + o + 2);
                            r0.x = rka * r0.x + dt * rp;  q0.x += rkb * r0.x;
                            r0.y = rka * r0.y + dt * ru;  q0.y += rkb * r0.y;
                            r1.x = rka * r1.x + dt * rv;  q1.x += rkb * r1.x;
                            r1.y = rka * r1.y + dt * rw;  q1.y += rkb * r1.y;
                            __stcs(reinterpret_cast<double2*>(res + o), r0);
                            __stcs(reinterpret_cast<double2*>(res + o + 2), r1);
                            __stcs(reinterpret_cast<double2*>(qnew + o), q0);
                            __stcs(reinterpret_cast<double2*>(qnew + o + 2), q1);
                        }
                    }
            }
        }
        __syncthreads();
    }
}

}  // namespace dg
