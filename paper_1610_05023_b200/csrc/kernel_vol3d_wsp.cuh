// 3D solver, fp64, warp-specialised tensor-pipe version with a SOFTWARE-PIPELINED MMA loop: fused volume +
// surface + update of one LSRK stage (Alg. 2, eq (41)-(43)).  Same mathematics, DMMA
// tiling, roles and per-tet record as kernel_vol3d_ws.cuh.
//
// What changes (profiles/r02_vol3d_ws_ncu.md): in k_vol3d_ws an MMA warp alternates between its 108 DMMA and the
// right-hand side + update of its accumulators, and the two MMA warps of an SM sub-partition pass a token so that
// one warp's update runs under the other's DMMAs; the fp64 unit of the busy sub-partitions is still idle 35 % of the
// time.  Here every MMA warp keeps TWO accumulator sets: while it issues the DMMAs of batch it into one, the update
// of batch it-1 (a branch-free block of loads, ~90 DFMA and predicated stores) sits in the same basic block and
// ptxas interleaves it with the DMMA stream.  No token, no phase in which a warp has no DMMA to issue.
// Stages of q / res / records are held one batch longer, so that ring is 4 deep; the neighbour traces (needed by
// PREP only) get their own 2-deep ring.
// Status (profiles/r02_vol3d_ws2.md): correct (parity tests) but 4.0 ms per launch at N = 5 against 3.63 ms of
// k_vol3d_ws -- a warp issues in order, so a DFMA of the update that waits for its operand also holds back the
// DMMAs behind it.  Kept as dg_options.kernel = 6 for the record; the library's default stays k_vol3d_ws.
#pragma once
#include "kernel_vol3d_ws.cuh"

namespace dg {

template <int N>
struct WspCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EB = 8;
    static constexpr int MT = (Np + 7) / 8;            // MMA warps
    static constexpr int KD = (Np + 3) / 4, KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4, KPL = KL * 4;
    static constexpr int LPAD = KPL * EB + 8;          // stride of one face block of the flux operand (bank spread)
    static constexpr int NT = 384;
    static constexpr int NS = 4;                       // staging depth of q / res / records
    static constexpr int QS = Np * 4 + 2;              // staged element stride of q / res (16 B skew)
    static constexpr int GS = GX3 + 2;
    static constexpr int szB = 4 * KPD * EB + 4 * LPAD;
    static constexpr int oB = 0;                       // [2][szB]        operand buffers
    static constexpr int oQ = oB + 2 * szB;            // [NS][8][QS]
    static constexpr int oR = oQ + NS * EB * QS;       // [NS][8][QS]
    static constexpr int oGeo = oR + NS * EB * QS;     // [NS][8][GS]
    static constexpr int oN = oGeo + NS * EB * GS;     // [2][Nfn][8][4] neighbour traces (halves of elements 4..7 swapped)
    static constexpr int oBar = oN + 2 * Nfn * EB * 4; // full[NS], empty[NS], ready[2], opfree[2], nfree[2]
    static constexpr int oEnd = oBar + 2 * NS + 6;
    static constexpr size_t smem_bytes = sizeof(double) * oEnd + sizeof(int) * (33 * Nfp + Nfn) + 32;
    static constexpr uint32_t tx_bytes = 2 * EB * Np * 32 + EB * GX3 * 8;
    static constexpr int NJ = (Nfp + 3) / 4;           // face nodes per PREP thread (j = pw + 4 r)
#ifndef WSP_REG_MMA
#define WSP_REG_MMA 208
#endif
    static constexpr int REG_BASE = 168, REG_MMA = WSP_REG_MMA, REG_PREP = REG_BASE - 2 * (REG_MMA - REG_BASE);
    static_assert((REG_BASE - REG_PREP) * 128 >= (REG_MMA - REG_BASE) * 256, "setmaxnreg pool would deadlock");
    static_assert(MT <= 7, "the warp-specialised kernels cover N <= 5");
    static_assert(smem_bytes <= 227 * 1024, "shared memory");
};

template <int N>
__global__ void __launch_bounds__(WspCfg<N>::NT, 1)
k_vol3d_wsp(Dev<double> d, const double* __restrict__ geox, int src, double rka, double rkb) {
    using C = WspCfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  NT = C::NT, QS = C::QS, MT = C::MT, NS = C::NS, LPAD = C::LPAD, NJ = C::NJ, GS = C::GS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sm = reinterpret_cast<double*>(smem_raw);
    double* sQ = sm + C::oQ;
    double* sR = sm + C::oR;
    double* sGeo = sm + C::oGeo;
    double* sN = sm + C::oN;
    uint64_t* full = reinterpret_cast<uint64_t*>(sm + C::oBar);
    uint64_t* empty = full + NS;
    uint64_t* ready = empty + NS;
    uint64_t* opfree = ready + 2;
    uint64_t* nfree = opfree + 2;
    int* sNode = reinterpret_cast<int*>(sm + C::oEnd);       // [33][Nfp]: (face | perm << 2, j) -> 4 * neighbour node
    int* sFm = sNode + 33 * Nfp;                             // [4][Nfp] own face node

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const double* __restrict__ qold = d.q[src];
    const int K = d.K;
    const int nbatch = (K + EB - 1) / EB;                    // arrays are padded to nbatch * EB elements

    // ---- one-time: tables, zeroed operand buffers (their padding rows stay zero for ever), barriers
    for (int i = tid; i < C::oQ; i += NT) sm[i] = 0.0;
    for (int i = tid; i < 33 * Nfp; i += NT) {               // entries are offsets in doubles (4 per node)
        const int fp = i / Nfp, j = i - fp * Nfp, pm = fp >> 2;
        sNode[i] = fp == 32 ? 4 * j : pm < 6 ? 4 * d.fmask3[(fp & 3) * Nfp + d.perm3[pm * Nfp + j]] : 0;
    }
    for (int i = tid; i < Nfn; i += NT) sFm[i] = d.fmask3[i];
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 33); mbar_init(&empty[s], MT); }
        for (int o = 0; o < 2; ++o) { mbar_init(&ready[o], 4); mbar_init(&opfree[o], MT); mbar_init(&nfree[o], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async;" ::: "memory");
    }
    __syncthreads();

    if (w >= 8) {
        // =============================================================== PREP warps
        reg_dec<C::REG_PREP>();
        const int pw = w - 8;
        const int ie = lane & 7, f = lane >> 3;
        const int slot = f + 4 * pw;                         // phase A: nodes slot + 16 r of element ie
        int it = 0;
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it % NS, o = it & 1;
            const double* bq = sQ + (s * EB + ie) * QS;
            const double* ge = sGeo + (s * EB + ie) * GS;
            const double* bn = sN + o * (Nfn * EB * 4) + f * (Nfp * 32) + ie * 4;
            const int h0 = 2 * ((ie >> 2) & 1);
            double* sB = sm + C::oB + o * C::szB;
            double* sG = sB + 4 * KPD * EB + f * LPAD;
            mbar_wait(&full[s], (it / NS) & 1);
            if (it >= 2) mbar_wait(&opfree[o], ((it >> 1) - 1) & 1);
            // ---- phase A: (p, contravariant velocity) -> operand rows (one column per element)
            {
                const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                              g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6);
                const double g8 = ge[8];
#pragma unroll
                for (int r = 0; r < (Np + 15) / 16; ++r) {
                    const int n = slot + 16 * r;
                    if (n < Np) {
                        const double2 v0 = *reinterpret_cast<const double2*>(bq + n * 4);
                        const double2 v1 = *reinterpret_cast<const double2*>(bq + n * 4 + 2);
                        double* op = sB + n * EB + (ie ^ swz(n));
                        op[0] = v0.x;
                        op[KPD * EB] = g01.x * v0.y + g01.y * v1.x + g23.x * v1.y;
                        op[2 * KPD * EB] = g23.y * v0.y + g45.x * v1.x + g45.y * v1.y;
                        op[3 * KPD * EB] = g67.x * v0.y + g67.y * v1.x + g8 * v1.y;
                    }
                }
            }
            // ---- phase B: one scalar flux jump per face node (upwind flux PAPER.md:L499-512):
            //      g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-)
            {
                const double2 nxy = *reinterpret_cast<const double2*>(ge + 12 + 4 * f);
                const double2 nzA = *reinterpret_cast<const double2*>(ge + 14 + 4 * f);
                const double Bf = ge[28 + f];
#pragma unroll
                for (int r = 0; r < NJ; ++r) {
                    const int j = pw + 4 * r;
                    if (j < Nfp) {
                        const int fm = 4 * sFm[f * Nfp + j];
                        const double2 m0 = *reinterpret_cast<const double2*>(bq + fm);
                        const double2 m1 = *reinterpret_cast<const double2*>(bq + fm + 2);
                        const double2 x0 = *reinterpret_cast<const double2*>(bn + j * 32 + h0);
                        const double2 x1 = *reinterpret_cast<const double2*>(bn + j * 32 + (2 - h0));
                        const double dn = nxy.x * (x0.y - m0.y) + nxy.y * (x1.x - m1.x) + nzA.x * (x1.y - m1.y);
                        sG[j * EB + (ie ^ swz(j))] = nzA.y * dn - Bf * (x0.x - m0.x);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(&ready[o]); mbar_arrive(&nfree[o]); }
        }
        return;
    }

    reg_inc<C::REG_MMA>();
    if (w == 7) {
        // =============================================================== LOADER warp
        // gather role: lanes 2k, 2k+1 fetch the two 16-byte halves of one node's (p,u,v,w): one 32-byte sector
        const int ie = (lane >> 1) & 7, h = lane & 1, hw = lane >> 4;
        const int hsw = 2 * (h ^ ((ie >> 2) & 1));           // halves of elements 4..7 are swapped (bank spread)
        const uint4* conn = reinterpret_cast<const uint4*>(d.conn3);
        int it = 0;
        uint4 cnext = conn[(size_t)blockIdx.x * EB + ie];
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it % NS, o = it & 1;
            const uint4 cw4 = cnext;                         // connectivity of element ie, one word per face
            if (b + (int)gridDim.x < nbatch) cnext = conn[(size_t)(b + gridDim.x) * EB + ie];
            if (it >= NS) mbar_wait(&empty[s], ((it / NS) - 1) & 1);
            const size_t e0 = (size_t)b * EB;
            if (lane == 0) mbar_arrive_expect_tx(&full[s], C::tx_bytes);
            __syncwarp();
            if (lane < EB) bulk_g2s(sQ + (s * EB + lane) * QS, qold + (e0 + lane) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 2 * EB) bulk_g2s(sR + (s * EB + lane - EB) * QS, d.res + (e0 + lane - EB) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 3 * EB) bulk_g2s(sGeo + (s * EB + lane - 2 * EB) * GS, geox + (e0 + lane - 2 * EB) * GX3, GX3 * 8, &full[s]);
            // neighbour traces (16-byte cp.async gathers), or the ghost state (2 r^-, 0, 0, 0) behind an HABC face;
            // this half-warp serves faces 2 hw and 2 hw + 1 of element ie
            if (it >= 2) mbar_wait(&nfree[o], ((it >> 1) - 1) & 1);
            double* dn = sN + o * (Nfn * EB * 4) + hw * (2 * Nfp * 32) + ie * 4 + hsw;
#pragma unroll
            for (int fl = 0; fl < 2; ++fl) {
                const uint32_t c = hw ? (fl ? cw4.w : cw4.z) : (fl ? cw4.y : cw4.x);
                const size_t id = (c >> 5) & CONN_MAX_ID;
                const bool bnd = (c & CONN_BND) != 0;
                const double* base = (bnd ? d.ghost3 + id * (Nfp * 4) : qold + id * (Np * 4)) + 2 * h;
                const int* tab = sNode + (bnd ? 32 : (int)(c & 31)) * Nfp;     // row 32 is the identity
                int off[Nfp];                                // all table reads first: cp.async is a compiler barrier
#pragma unroll
                for (int j = 0; j < Nfp; ++j) off[j] = tab[j];
#pragma unroll
                for (int j = 0; j < Nfp; ++j) cp_async16(dn + (fl * Nfp + j) * 32, base + off[j]);
            }
            cp_async_arrive_noinc(&full[s]);
        }
        return;
    }
    if (w >= MT) return;

    // =================================================================== MMA warps
    const int g = lane >> 2, t = lane & 3;
    const int n = 8 * w + g;                                 // the node this lane owns in the accumulators
    const bool nok = n < Np;
    double* __restrict__ qnew = d.q[src ^ 1];
    double* __restrict__ res = d.res;
    double Ar[KD], As[KD], At[KD], AL[4][KL];
#pragma unroll
    for (int s = 0; s < KD; ++s) {
        const int m = 4 * s + t;
        const bool ok = n < Np && m < Np;
        Ar[s] = ok ? d.Dt3[(0 * Np + m) * Np + n] : 0.0;     // Dt3[a][m][n] = D_a[n][m]
        As[s] = ok ? d.Dt3[(1 * Np + m) * Np + n] : 0.0;
        At[s] = ok ? d.Dt3[(2 * Np + m) * Np + n] : 0.0;
    }
#pragma unroll
    for (int f = 0; f < 4; ++f)
#pragma unroll
        for (int s = 0; s < KL; ++s) {
            const int j = 4 * s + t;
            AL[f][s] = (n < Np && j < Nfp) ? d.Lt3[(f * Nfp + j) * Np + n] : 0.0;   // Lt3[j][n] = LIFT[n][j]
        }

    // accumulators: 0..2 d_r p, d_s p, d_t p; 3..5 the three terms of div U; 6..9 LIFT_f g; [.][ee] = element 2t + ee
    double acc[10][2];
#pragma unroll
    for (int v = 0; v < 10; ++v) acc[v][0] = acc[v][1] = 0.0;

    // right-hand side and LSRK update (eq (41)-(43)) of node n, elements 2t, 2t+1 of the batch staged in `sp`
    // (dt folded into the record).  Branch-free: everything is computed, only the stores are predicated.
    auto update = [&](const double (&P)[10][2], int sp, int e0p, bool valid) {
        const double* bq = sQ + sp * (EB * QS);
        const double* br = sR + sp * (EB * QS);
        const double* bgeo = sGeo + sp * EB * GS;
        const int nn = nok ? n : 0;
#pragma unroll
        for (int ee = 0; ee < 2; ++ee) {
            const int e = 2 * t + ee;
            const bool ok = valid && nok && e0p + e < K;
            const double* ge = bgeo + e * GS;
            const double2 f01 = *reinterpret_cast<const double2*>(ge + 32), f23 = *reinterpret_cast<const double2*>(ge + 34);
            const double2 g8r = *reinterpret_cast<const double2*>(ge + 8), irc = *reinterpret_cast<const double2*>(ge + 10);
            const double a0 = P[6][ee], a1 = P[7][ee], a2 = P[8][ee], a3 = P[9][ee];
            const double lp = f01.x * a0 + f01.y * a1 + f23.x * a2 + f23.y * a3;
            const double rc2 = g8r.y, irho = irc.x, cc = irc.y;        // each already times dt
            // -1/rho grad p + c * sum_f (Fs n)_f LIFT_f g, both through G^T:  G^T (c*l - irho*dp)
            const double xr = cc * (a2 - a3) - irho * P[0][ee];
            const double xs = cc * (a2 - a1) - irho * P[1][ee];
            const double xt = cc * (a2 - a0) - irho * P[2][ee];
            const double rp = -rc2 * ((P[3][ee] + P[4][ee]) + P[5][ee] + lp);
            const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                          g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6);
            const double ru = g01.x * xr + g23.y * xs + g67.x * xt;
            const double rv = g01.y * xr + g45.x * xs + g67.y * xt;
            const double rw = g23.x * xr + g45.y * xs + g8r.x * xt;
            double2 q0 = *reinterpret_cast<const double2*>(bq + e * QS + nn * 4);
            double2 q1 = *reinterpret_cast<const double2*>(bq + e * QS + nn * 4 + 2);
            double2 r0 = *reinterpret_cast<const double2*>(br + e * QS + nn * 4);
            double2 r1 = *reinterpret_cast<const double2*>(br + e * QS + nn * 4 + 2);
            r0.x = rka * r0.x + rp;  q0.x += rkb * r0.x;
            r0.y = rka * r0.y + ru;  q0.y += rkb * r0.y;
            r1.x = rka * r1.x + rv;  q1.x += rkb * r1.x;
            r1.y = rka * r1.y + rw;  q1.y += rkb * r1.y;
            const size_t off = ((size_t)(e0p + e) * Np + nn) * 4;
            if (ok) {
                __stcs(reinterpret_cast<double2*>(res + off), r0);
                __stcs(reinterpret_cast<double2*>(res + off + 2), r1);
                __stcs(reinterpret_cast<double2*>(qnew + off), q0);
                __stcs(reinterpret_cast<double2*>(qnew + off + 2), q1);
            }
        }
    };

#ifndef WSP_UPD_AT
#define WSP_UPD_AT 6
#endif
    int it = 0, sp = 0, e0p = 0;
    for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
        const int s = it % NS, o = it & 1;
        const double* sB = sm + C::oB + o * C::szB;
        const double* sG = sB + 4 * KPD * EB;
        double P[10][2];                                     // the previous batch's results, updated under this batch's DMMAs
#pragma unroll
        for (int v = 0; v < 10; ++v) { P[v][0] = acc[v][0]; P[v][1] = acc[v][1]; acc[v][0] = acc[v][1] = 0.0; }
        mbar_wait(&ready[o], (it >> 1) & 1);
        mbar_wait(&full[s], (it / NS) & 1);                  // already complete: makes the async-proxy writes visible here
        {
            const double* bp = sB + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KD; ++s_) {
                const double b0 = bp[(0 * KPD + 4 * s_) * EB];
                dmma884v(acc[0], Ar[s_], b0);
                dmma884v(acc[1], As[s_], b0);
                dmma884v(acc[2], At[s_], b0);
                dmma884v(acc[3], Ar[s_], bp[(1 * KPD + 4 * s_) * EB]);
                dmma884v(acc[4], As[s_], bp[(2 * KPD + 4 * s_) * EB]);
                dmma884v(acc[5], At[s_], bp[(3 * KPD + 4 * s_) * EB]);
                if (s_ == WSP_UPD_AT) update(P, sp, e0p, it >= 1);
            }
            const double* gp = sG + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KL; ++s_)
#pragma unroll
                for (int f = 0; f < 4; ++f) dmma884v(acc[6 + f], AL[f][s_], gp[f * LPAD + 4 * s_ * EB]);
        }
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&opfree[o]);
            if (it >= 1) mbar_arrive(&empty[sp]);
        }
        sp = s; e0p = b * EB;
    }
    if (it >= 1) update(acc, sp, e0p, true);                 // the last batch
}

}  // namespace dg
