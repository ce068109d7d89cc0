// 3D solver, fp32, tensor-core kernel for N >= 6: fused volume + surface + update of one LSRK stage (PAPER.md:L623-624,
// Alg. 2, eq (41)-(43)) with the contractions as error-compensated 3xTF32 (kernel_vol3d_tf32.cuh) and the
// phase structure of kernel_vol3d_mmag.cuh: the operator fragments (B of mma.m16n8k8: D[n = 8w+g][k = 8s+t, +4]) do
// not fit the register file at these degrees, so they are read per use through L1/L2 -- from arrays the host has laid
// out in FRAGMENT ORDER, zero-padded and already split: Dfrag [3][NTL][KD][32][4], Lfrag [4][NTL][KL][32][4], entry
// (a, nt, s, lane = 4 g + t) = (hi, hi', lo, lo') of D_a[n = 8 nt + g][k = 8 s + t] and [k + 4]: one unconditional,
// coalesced 16-byte load per lane replaces two scalar loads, two bounds checks and two splits.
// A batch is 16 elements (MMA m); warp w loops over the n-tiles (8 nodes) w, w+W, ...
#pragma once
#include "kernel_vol3d_tf32.cuh"

namespace dg {

template <int N, int W>
struct TfgCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EPB = 16;
    static constexpr int NTL = (Np + 7) / 8;            // n-tiles
    static constexpr int KD = (Np + 7) / 8, KPD = KD * 8;
    static constexpr int KL = (Nfp + 7) / 8, KPL = KL * 8;
    static constexpr int XS = 24;                       // operand row stride in floats (16 elements + 8: bank spread)
    static constexpr int NT = 32 * W;
    static constexpr int szT = (4 * KPD + 4 * KPL) * XS;
    static constexpr size_t smem_bytes = sizeof(float) * szT + 16;
};

template <int N, int W>
__global__ void __launch_bounds__(TfgCfg<N, W>::NT)
k_vol3d_tf32g(Dev<float> d, int src, float rka, float rkb, float dt) {
    using C = TfgCfg<N, W>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EPB = C::EPB, NTL = C::NTL, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  KPL = C::KPL, NT = C::NT, szT = C::szT, XS = C::XS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sB = reinterpret_cast<float*>(smem_raw);         // [p | U^r | U^s | U^t : KPD rows each | g_f : KPL rows each][XS]
    const float* __restrict__ qold = d.q[src];
    float* __restrict__ qnew = d.q[src ^ 1];
    float* __restrict__ res = d.res;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int K = d.K;
    const int nbatch = (K + EPB - 1) / EPB;

    for (int i = tid; i < szT; i += NT) sB[i] = 0.f;        // padding rows stay zero for ever
    __syncthreads();

    for (int batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
        const int e0 = batch * EPB;
        // ---- phase 1: operands [k][element]
        for (int idx = tid; idx < EPB * Np; idx += NT) {
            const int e = idx / Np, n = idx - e * Np;
            const int k = min(e0 + e, K - 1);               // elements past the end repeat the last one (never stored)
            const float* ge = d.geo3 + (size_t)k * GEO3;
            const float4 v = *reinterpret_cast<const float4*>(qold + ((size_t)k * Np + n) * 4);
            float* o = sB + n * XS + e;
            o[0] = v.x;
            o[KPD * XS] = ge[0] * v.y + ge[1] * v.z + ge[2] * v.w;
            o[2 * KPD * XS] = ge[3] * v.y + ge[4] * v.z + ge[5] * v.w;
            o[3 * KPD * XS] = ge[6] * v.y + ge[7] * v.z + ge[8] * v.w;
        }
        __syncthreads();
        // ---- phase 2: g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-); Fs n.u- = nhat . U- from the operands
        for (int idx = tid; idx < EPB * Nfn; idx += NT) {
            const int e = idx / Nfn, fj = idx - e * Nfn;
            const int f = fj / Nfp, j = fj - f * Nfp;
            const int k = min(e0 + e, K - 1);
            const float* ge = d.geo3 + (size_t)k * GEO3;
            const float* om = sB + d.fmask3[fj] * XS + e;
            const float pM = om[0], Ur = om[KPD * XS], Us = om[2 * KPD * XS], Ut = om[3 * KPD * XS];
            const float unM = (f == 0) ? -Ut : (f == 1) ? -Us : (f == 2) ? (Ur + Us + Ut) : -Ur;
            const int nb = d.nbr3[k * 4 + f];
            float pP, unP;
            if (nb >= 0) {
                const uint32_t info = (d.finfo3[k] >> (8 * f)) & 0xffu;
                const int fp = info & 3, pm = info >> 2;
                const int np_ = d.fmask3[fp * Nfp + d.perm3[pm * Nfp + j]];
                const float4 x = *reinterpret_cast<const float4*>(qold + ((size_t)nb * Np + np_) * 4);
                float nx, ny, nz;
                if (f == 0) { nx = -ge[6]; ny = -ge[7]; nz = -ge[8]; }
                else if (f == 1) { nx = -ge[3]; ny = -ge[4]; nz = -ge[5]; }
                else if (f == 2) { nx = ge[0] + ge[3] + ge[6]; ny = ge[1] + ge[4] + ge[7]; nz = ge[2] + ge[5] + ge[8]; }
                else { nx = -ge[0]; ny = -ge[1]; nz = -ge[2]; }
                pP = x.x;
                unP = nx * x.y + ny * x.z + nz * x.w;
            } else {
                pP = 2.f * d.qb3[(size_t)(-1 - nb) * Nfp + j];          // ghost state: p+ = 2 r^-, u+ = 0
                unP = 0;
            }
            sB[(4 * KPD + f * KPL + j) * XS + e] = ge[9 + f] * (unP - unM) - ge[13 + f] * (pP - pM);
        }
        __syncthreads();
        // ---- phase 3: contractions (3xTF32) and update, one n-tile of 8 nodes at a time
        for (int nt = w; nt < NTL; nt += W) {
            const uint4* fD = reinterpret_cast<const uint4*>(d.Dfrag) + (size_t)nt * KD * 32 + lane;
            const uint4* fL = reinterpret_cast<const uint4*>(d.Lfrag) + (size_t)nt * KL * 32 + lane;
            float cpr[4] = {0, 0, 0, 0}, cps[4] = {0, 0, 0, 0}, cpt[4] = {0, 0, 0, 0};
            float cvr[4] = {0, 0, 0, 0}, cvs[4] = {0, 0, 0, 0}, cvt[4] = {0, 0, 0, 0};
            float cl[4][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
            const float* ap = sB + t * XS + g;
            auto loadA = [&](const float* r0, uint32_t (&ah)[4], uint32_t (&al)[4]) {
                const float x0 = r0[0], x1 = r0[8], x2 = r0[4 * XS], x3 = r0[4 * XS + 8];
                split_tf32(x0, ah[0], al[0]);
                split_tf32(x1, ah[1], al[1]);
                split_tf32(x2, ah[2], al[2]);
                split_tf32(x3, ah[3], al[3]);
            };
#pragma unroll 1
            for (int s_ = 0; s_ < KD; ++s_) {
                uint32_t brh[2], brl[2], bsh[2], bsl[2], bth[2], btl[2];
                {
                    const uint4 vr = fD[s_ * 32], vs = fD[(NTL * KD + s_) * 32], vt = fD[(2 * NTL * KD + s_) * 32];
                    brh[0] = vr.x; brh[1] = vr.y; brl[0] = vr.z; brl[1] = vr.w;
                    bsh[0] = vs.x; bsh[1] = vs.y; bsl[0] = vs.z; bsl[1] = vs.w;
                    bth[0] = vt.x; bth[1] = vt.y; btl[0] = vt.z; btl[1] = vt.w;
                }
                uint32_t ph[4], pl[4], rh[4], rl[4], sh[4], sl[4], th[4], tl[4];
                loadA(ap + (8 * s_) * XS, ph, pl);
                loadA(ap + (KPD + 8 * s_) * XS, rh, rl);
                loadA(ap + (2 * KPD + 8 * s_) * XS, sh, sl);
                loadA(ap + (3 * KPD + 8 * s_) * XS, th, tl);
                mma_tf32(cpr, pl, brh[0], brh[1]); mma_tf32(cps, pl, bsh[0], bsh[1]); mma_tf32(cpt, pl, bth[0], bth[1]);
                mma_tf32(cvr, rl, brh[0], brh[1]); mma_tf32(cvs, sl, bsh[0], bsh[1]); mma_tf32(cvt, tl, bth[0], bth[1]);
                mma_tf32(cpr, ph, brl[0], brl[1]); mma_tf32(cps, ph, bsl[0], bsl[1]); mma_tf32(cpt, ph, btl[0], btl[1]);
                mma_tf32(cvr, rh, brl[0], brl[1]); mma_tf32(cvs, sh, bsl[0], bsl[1]); mma_tf32(cvt, th, btl[0], btl[1]);
                mma_tf32(cpr, ph, brh[0], brh[1]); mma_tf32(cps, ph, bsh[0], bsh[1]); mma_tf32(cpt, ph, bth[0], bth[1]);
                mma_tf32(cvr, rh, brh[0], brh[1]); mma_tf32(cvs, sh, bsh[0], bsh[1]); mma_tf32(cvt, th, bth[0], bth[1]);
            }
            const float* gp = ap + 4 * KPD * XS;
#pragma unroll 1
            for (int s_ = 0; s_ < KL; ++s_) {
#pragma unroll
                for (int f = 0; f < 4; ++f) {
                    uint32_t bh[2], bl[2], ah[4], al[4];
                    {
                        const uint4 v = fL[(f * NTL * KL + s_) * 32];
                        bh[0] = v.x; bh[1] = v.y; bl[0] = v.z; bl[1] = v.w;
                    }
                    loadA(gp + (f * KPL + 8 * s_) * XS, ah, al);
                    mma_3x(cl[f], ah, al, bh, bl);
                }
            }
            // right-hand side and LSRK update (eq (41)-(43)): accumulator index 2 r + c: element g + 8 r, node 8 nt + 2 t + c
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int k = e0 + g + 8 * r;
                if (k < K) {
                    const float* ge = d.geo3 + (size_t)k * GEO3;
                    const float rc2 = ge[21], irho = ge[22], cc = ge[23];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const int n = 8 * nt + 2 * t + c, i = 2 * r + c;
                        if (n < Np) {
                            const float a0 = cl[0][i], a1 = cl[1][i], a2 = cl[2][i], a3 = cl[3][i];
                            const float lp = ge[17] * a0 + ge[18] * a1 + ge[19] * a2 + ge[20] * a3;
                            const float xr = cc * (a2 - a3) - irho * cpr[i];
                            const float xs = cc * (a2 - a1) - irho * cps[i];
                            const float xt = cc * (a2 - a0) - irho * cpt[i];
                            const float rp = -rc2 * ((cvr[i] + cvs[i]) + cvt[i] + lp);
                            const float ru = ge[0] * xr + ge[3] * xs + ge[6] * xt;
                            const float rv = ge[1] * xr + ge[4] * xs + ge[7] * xt;
                            const float rw = ge[2] * xr + ge[5] * xs + ge[8] * xt;
                            const size_t o = ((size_t)k * Np + n) * 4;
                            float4 q = *reinterpret_cast<const float4*>(qold + o);
                            float4 rr = *reinterpret_cast<const float4*>(res + o);
                            rr.x = rka * rr.x + dt * rp;  q.x += rkb * rr.x;
                            rr.y = rka * rr.y + dt * ru;  q.y += rkb * rr.y;
                            rr.z = rka * rr.z + dt * rv;  q.z += rkb * rr.z;
                            rr.w = rka * rr.w + dt * rw;  q.w += rkb * rr.w;
                            __stcs(reinterpret_cast<float4*>(res + o), rr);
                            __stcs(reinterpret_cast<float4*>(qnew + o), q);
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace dg
