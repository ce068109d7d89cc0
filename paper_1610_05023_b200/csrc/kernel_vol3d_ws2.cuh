// 3D solver, fp64, warp-specialised tensor-pipe version 2: fused volume + surface + update of one LSRK stage
// (Alg. 2, eq (41)-(43)).  Same mathematics, DMMA tiling, staging and per-tet record
// as kernel_vol3d_ws.cuh; what changes is that the MMA warps do NOTHING but DMMA, and that the remaining fp64
// arithmetic is placed on the SM sub-partition whose fp64 unit has time for it.
//
// Why (profiles/r02_vol3d_ws_ncu.md, profiles/r02_dmma_issue.md).  DMMA and DFMA share one fp64 unit per SM
// sub-partition (SP); a DMMA.8x8x4 holds it for 16 cycles, a DFMA for 2.  Np = 56 gives 7 m-tiles for 4 SPs:
// SP0..2 run two MMA warps (216 DMMA = 3456 unit-cycles per batch), SP3 one (1728).  In k_vol3d_ws every MMA warp
// also ran the update of its accumulators and the four operand-preparation warps sat one per SP, so SP0..2 carried
// 3456 + ~400 cycles of unit work per batch plus the stalls of warps that alternate between DMMA and dependent DFMA
// chains (each DFMA queues behind the other warp's DMMAs): 5360 cycles per batch measured, DMMA sub-pipe 65 % busy.
// Two warps that only issue DMMA (+ one LDS.64 operand each) keep the unit 91-96 % busy (microbenchmark).  So:
//
//   warps 0..6    MMA      wait ready[o] -> 84 DMMA (D_r, D_s, D_t on p; divergence) -> results to H ->
//                          24 DMMA (LIFT on the flux jumps) -> release opfree[o] -> results to H -> signal hfull
//   warp 8        LOADER   bulk async copies (cp.async.bulk) of q, res, records into stage s of 3; 16-byte
//                          cp.async gathers of the neighbours' face traces into trace buffer it & 1
//   warps 7,11,15 HELPERS on SP3 (heavy) and warps 12,13,14 on SP0..2 (light): per batch
//                          PREP(it): operands (p, contravariant velocity) and one upwind flux jump per face node
//                           into operand buffer o; signal ready[o], release the trace buffer;
//                          UPDATE(it-1): wait hfull; right-hand side + LSRK update (eq (41)-(43)) as a stream over
//                          the 8 x Np (element, node) items of the batch, lane <-> node (1 KB coalesced stores);
//                          release H and stage s.
//                          Work is dealt in rows of 32 items, 4 of every 18 rows to each SP3 helper, 2 to each light one.
// Status (profiles/r02_vol3d_ws2.md): correct (parity tests), but at N = 5 it runs 4.17 ms per launch against the
// 3.63 ms of k_vol3d_ws: the shared-memory pipe (64-73 % busy: every MMA warp re-reads the whole operand, plus the H
// exchange) and the helpers' DFMA chains queueing behind DMMAs eat what the MMA warps gain.  Kept as
// dg_options.kernel = 4 for the record; the library's default stays k_vol3d_ws.
// Registers (setmaxnreg; 512 threads start at 128): warpgroups 0, 1 (MMA + helper 7) 176, of which 132 hold the
// operator fragments; warpgroups 2, 3 (loader, helpers) 80.
#pragma once
#include "kernel_vol3d_ws.cuh"

namespace dg {

template <int N>
struct Ws2Cfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EB = 8;
    static constexpr int MT = (Np + 7) / 8;            // MMA warps
    static constexpr int KD = (Np + 3) / 4, KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4, KPL = KL * 4;
    static constexpr int LPAD = KPL * EB + 8;          // stride of one face block of the flux operand (bank spread)
    static constexpr int NT = 512;
    static constexpr int NS = 3;                       // staging depth of q / res / records
    static constexpr int NH = 6;                       // helper warps
    static constexpr int QS = Np * 4 + 2;              // staged element stride of q / res (16 B skew)
    static constexpr int GS = GX3 + 2;
    static constexpr int HS = ((Np + 3) / 8) * 8 + 4;  // element stride of H: = 4 mod 8, so that the accumulator
                                                       // stores of a warp (node g, elements 2t / 2t+1) spread over all banks
    static constexpr int HV = EB * HS;                 // stride of one of the 8 result arrays of H
    static constexpr int szB = 4 * KPD * EB + 4 * LPAD;
    static constexpr int oB = 0;                       // [2][szB]        operand buffers
    static constexpr int oQ = oB + 2 * szB;            // [NS][8][QS]
    static constexpr int oR = oQ + NS * EB * QS;       // [NS][8][QS]
    static constexpr int oGeo = oR + NS * EB * QS;     // [NS][8][GS]
    static constexpr int oN = oGeo + NS * EB * GS;     // [2][Nfn][8][4] neighbour traces (halves of elements 4..7 swapped)
    static constexpr int oH = oN + 2 * Nfn * EB * 4;   // [8][8][HS]   d_r p, d_s p, d_t p, div U, LIFT_f g (f = 0..3)
    static constexpr int oBar = oH + 8 * HV;           // full[NS], empty[NS], ready[2], opfree[2], nfree[2], hfull, hfree
    static constexpr int NBAR = 2 * NS + 8;
    static constexpr int oEnd = oBar + NBAR;
    static constexpr size_t smem_bytes = sizeof(double) * oEnd + sizeof(int) * (33 * Nfp + Nfn) + 32;
    static constexpr uint32_t tx_bytes = 2 * EB * Np * 32 + EB * GX3 * 8;
    static constexpr int NROWA = (Np + 3) / 4;         // PREP phase A rows: 4 nodes x 8 elements
    static constexpr int NROWB = Nfp;                  // PREP phase B rows: 4 faces x 8 elements of face node j
    static constexpr int NROWU = (EB * Np + 31) / 32;  // UPDATE rows: 32 consecutive (element, node) items
    static constexpr int REG_LOW = 80, REG_MMA = 176;
    static_assert(2 * (128 - REG_LOW) * 128 >= (REG_MMA - 128) * 256, "setmaxnreg pool would deadlock");
    static_assert(MT <= 7, "the warp-specialised kernels cover N <= 5");
    static_assert(HS >= Np && HS % 8 == 4, "H stride");
    static_assert(smem_bytes <= 227 * 1024, "shared memory");
};

// shared-memory view + loop invariants handed to the helper role
struct Ws2Ctx {
    double *sm, *sQ, *sR, *sGeo, *sN, *sH;
    uint64_t *full, *empty, *ready, *opfree, *nfree, *hfull, *hfree;
    const int* sFm;
    double *qnew, *res;
    double rka, rkb;
    int K, nbatch;
};

// Rows of a phase are dealt to the helpers in rounds of 3 (HV + LT): heavy helper h (0..2, on SP3) takes HV rows
// of each round, light helper h (3..5, on SP0..2) takes LT.
#ifndef WS2_HV
#define WS2_HV 4
#endif
#ifndef WS2_LT
#define WS2_LT 2
#endif
// k is the iteration state of a helper's row loop (start with k = 0).  The loops are deliberately NOT unrolled:
// six helpers with unrolled row loops overflow the instruction cache (measured: 4.8 ms against 3.75 ms per launch).
__device__ __forceinline__ bool ws2_next_row(int& r, int& k, int hi, int nrows) {
    constexpr int HV = WS2_HV, LT = WS2_LT, ROUND = 3 * (HV + LT);
    const bool heavy = hi < 3;
    const int per = heavy ? HV : LT;
    const int round = heavy ? k / HV : k / LT, j = k - round * per;
    r = round * ROUND + (heavy ? hi : 3 * HV + (hi - 3)) + 3 * j;
    ++k;
    return r < nrows;
}

// ---- helper role, PREP half: operands of batch (stage s, operand buffer o)
template <int N>
__device__ __forceinline__ void ws2_prep(const Ws2Ctx& c, int hi, int lane, int s, int o) {
    using C = Ws2Cfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KPD = C::KPD, QS = C::QS, GS = C::GS, LPAD = C::LPAD;
    const int ie = lane & 7, f = lane >> 3;
    const double* bq = c.sQ + (s * EB + ie) * QS;
    const double* ge = c.sGeo + (s * EB + ie) * GS;
    double* sB = c.sm + C::oB + o * C::szB;
    // ---- phase A: (p, contravariant velocity) of node 4 row + f, element ie -> operand rows (one column per element)
    {
        const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                      g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6);
        const double g8 = ge[8];
        int row, k = 0;
#pragma unroll 1
        while (ws2_next_row(row, k, hi, C::NROWA)) {
            const int n = 4 * row + f;
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
    //      g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-);  row = face node j, lane = (face f, element ie)
    {
        const double2 nxy = *reinterpret_cast<const double2*>(ge + 12 + 4 * f);
        const double2 nzA = *reinterpret_cast<const double2*>(ge + 14 + 4 * f);
        const double Bf = ge[28 + f];
        const double* bn = c.sN + o * (Nfn * EB * 4) + f * (Nfp * 32) + ie * 4;
        const int h0 = 2 * ((ie >> 2) & 1);
        double* sG = sB + 4 * KPD * EB + f * LPAD;
        int j, k = 0;
#pragma unroll 1
        while (ws2_next_row(j, k, hi, C::NROWB)) {
            const int fm = 4 * c.sFm[f * Nfp + j];
            const double2 m0 = *reinterpret_cast<const double2*>(bq + fm);
            const double2 m1 = *reinterpret_cast<const double2*>(bq + fm + 2);
            const double2 x0 = *reinterpret_cast<const double2*>(bn + j * 32 + h0);
            const double2 x1 = *reinterpret_cast<const double2*>(bn + j * 32 + (2 - h0));
            const double dn = nxy.x * (x0.y - m0.y) + nxy.y * (x1.x - m1.x) + nzA.x * (x1.y - m1.y);
            sG[j * EB + (ie ^ swz(j))] = nzA.y * dn - Bf * (x0.x - m0.x);
        }
    }
}

// ---- helper role, UPDATE half: right-hand side and LSRK update (eq (41)-(43)); dt is folded into the record.
// Item idx = e * Np + n of the batch lives at global offset (e0 * Np + idx) * 4: a row of 32 items is 1 KB
// contiguous in q and in res.
template <int N>
__device__ __forceinline__ void ws2_update(const Ws2Ctx& c, int hi, int lane, int s, int e0) {
    using C = Ws2Cfg<N>;
    constexpr int Np = C::Np, EB = C::EB, QS = C::QS, GS = C::GS, HS = C::HS, HV = C::HV;
    const double* bq = c.sQ + s * (EB * QS);
    const double* br = c.sR + s * (EB * QS);
    const double* bgeo = c.sGeo + s * EB * GS;
    const double rka = c.rka, rkb = c.rkb;
    int row, k = 0;
#pragma unroll 1
    while (ws2_next_row(row, k, hi, C::NROWU)) {
        const int idx = row * 32 + lane;
        const int e = idx / Np, n = idx - e * Np;
        if (idx < EB * Np && e0 + e < c.K) {
            const double* hp = c.sH + e * HS + n;
            const double cpr = hp[0], cps = hp[HV], cpt = hp[2 * HV], dv = hp[3 * HV];
            const double a0 = hp[4 * HV], a1 = hp[5 * HV], a2 = hp[6 * HV], a3 = hp[7 * HV];
            double2 q0 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4);
            double2 q1 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4 + 2);
            double2 r0 = *reinterpret_cast<const double2*>(br + e * QS + n * 4);
            double2 r1 = *reinterpret_cast<const double2*>(br + e * QS + n * 4 + 2);
            const double* ge = bgeo + e * GS;
            const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                          g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6),
                          g8r = *reinterpret_cast<const double2*>(ge + 8), irc = *reinterpret_cast<const double2*>(ge + 10),
                          f01 = *reinterpret_cast<const double2*>(ge + 32), f23 = *reinterpret_cast<const double2*>(ge + 34);
            const double lp = (f01.x * a0 + f01.y * a1) + (f23.x * a2 + f23.y * a3);
            const double rc2 = g8r.y, irho = irc.x, cc = irc.y;        // each already times dt
            // -1/rho grad p + c * sum_f (Fs n)_f LIFT_f g, both through G^T:  G^T (c*l - irho*dp)
            const double xr = cc * (a2 - a3) - irho * cpr;
            const double xs = cc * (a2 - a1) - irho * cps;
            const double xt = cc * (a2 - a0) - irho * cpt;
            const double rp = -rc2 * (dv + lp);
            const double ru = g01.x * xr + g23.y * xs + g67.x * xt;
            const double rv = g01.y * xr + g45.x * xs + g67.y * xt;
            const double rw = g23.x * xr + g45.y * xs + g8r.x * xt;
            r0.x = rka * r0.x + rp;  q0.x += rkb * r0.x;
            r0.y = rka * r0.y + ru;  q0.y += rkb * r0.y;
            r1.x = rka * r1.x + rv;  q1.x += rkb * r1.x;
            r1.y = rka * r1.y + rw;  q1.y += rkb * r1.y;
            const size_t off = ((size_t)e0 * Np + idx) * 4;
            __stcs(reinterpret_cast<double2*>(c.res + off), r0);
            __stcs(reinterpret_cast<double2*>(c.res + off + 2), r1);
            __stcs(reinterpret_cast<double2*>(c.qnew + off), q0);
            __stcs(reinterpret_cast<double2*>(c.qnew + off + 2), q1);
        }
    }
}

template <int N>
__device__ __forceinline__ void ws2_helper(const Ws2Ctx& c, int hi, int lane) {
    using C = Ws2Cfg<N>;
    constexpr int NS = C::NS, EB = C::EB;
    int it = 0, bprev = 0;
    for (int b = blockIdx.x; b < c.nbatch; b += gridDim.x, ++it) {
        const int s = it % NS, o = it & 1;
        mbar_wait(&c.full[s], (it / NS) & 1);
        if (it >= 2) mbar_wait(&c.opfree[o], ((it >> 1) - 1) & 1);
        ws2_prep<N>(c, hi, lane, s, o);
        __syncwarp();
        if (lane == 0) { mbar_arrive(&c.ready[o]); mbar_arrive(&c.nfree[o]); }
        if (it >= 1) {
            const int sp = (it - 1) % NS;
            mbar_wait(c.hfull, (it - 1) & 1);
            ws2_update<N>(c, hi, lane, sp, bprev * EB);
            __syncwarp();
            if (lane == 0) { mbar_arrive(c.hfree); mbar_arrive(&c.empty[sp]); }
        }
        bprev = b;
    }
    if (it >= 1) {                                           // the last batch's update
        const int sp = (it - 1) % NS;
        mbar_wait(c.hfull, (it - 1) & 1);
        ws2_update<N>(c, hi, lane, sp, bprev * EB);
    }
}

template <int N>
__global__ void __launch_bounds__(Ws2Cfg<N>::NT, 1)
k_vol3d_ws2(Dev<double> d, const double* __restrict__ geox, int src, double rka, double rkb) {
    using C = Ws2Cfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  NT = C::NT, QS = C::QS, MT = C::MT, NS = C::NS, LPAD = C::LPAD, GS = C::GS, HS = C::HS, HV = C::HV;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sm = reinterpret_cast<double*>(smem_raw);
    Ws2Ctx c;
    c.sm = sm; c.sQ = sm + C::oQ; c.sR = sm + C::oR; c.sGeo = sm + C::oGeo; c.sN = sm + C::oN; c.sH = sm + C::oH;
    c.full = reinterpret_cast<uint64_t*>(sm + C::oBar);
    c.empty = c.full + NS; c.ready = c.empty + NS; c.opfree = c.ready + 2; c.nfree = c.opfree + 2;
    c.hfull = c.nfree + 2; c.hfree = c.hfull + 1;
    int* sNode = reinterpret_cast<int*>(sm + C::oEnd);       // [33][Nfp]: (face | perm << 2, j) -> 4 * neighbour node
    int* sFm = sNode + 33 * Nfp;                             // [4][Nfp] own face node
    c.sFm = sFm;
    c.qnew = d.q[src ^ 1]; c.res = d.res; c.rka = rka; c.rkb = rkb;
    c.K = d.K; c.nbatch = (d.K + EB - 1) / EB;               // arrays are padded to nbatch * EB elements

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const double* __restrict__ qold = d.q[src];
    const int nbatch = c.nbatch;

    // ---- one-time: tables, zeroed operand buffers (their padding rows stay zero for ever), barriers
    for (int i = tid; i < C::oQ; i += NT) sm[i] = 0.0;
    for (int i = tid; i < 33 * Nfp; i += NT) {               // entries are offsets in doubles (4 per node)
        const int fp = i / Nfp, j = i - fp * Nfp, pm = fp >> 2;
        sNode[i] = fp == 32 ? 4 * j : pm < 6 ? 4 * d.fmask3[(fp & 3) * Nfp + d.perm3[pm * Nfp + j]] : 0;
    }
    for (int i = tid; i < Nfn; i += NT) sFm[i] = d.fmask3[i];
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&c.full[s], 33); mbar_init(&c.empty[s], C::NH); }
        for (int o = 0; o < 2; ++o) { mbar_init(&c.ready[o], C::NH); mbar_init(&c.opfree[o], MT); mbar_init(&c.nfree[o], C::NH); }
        mbar_init(c.hfull, MT); mbar_init(c.hfree, C::NH);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async;" ::: "memory");
    }
    __syncthreads();

    if (w >= 8) {
        // =============================================================== warpgroups 2, 3: loader and helpers
        reg_dec<C::REG_LOW>();
        if (w >= 11) return ws2_helper<N>(c, w == 11 ? 1 : w == 15 ? 2 : w - 9, lane);   // light helpers 3, 4, 5 on SP0, 1, 2
        if (w != 8) return;
        // ----------------------------------------------------------- LOADER warp
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
            if (it >= NS) mbar_wait(&c.empty[s], ((it / NS) - 1) & 1);
            const size_t e0 = (size_t)b * EB;
            if (lane == 0) mbar_arrive_expect_tx(&c.full[s], C::tx_bytes);
            __syncwarp();
            if (lane < EB) bulk_g2s(c.sQ + (s * EB + lane) * QS, qold + (e0 + lane) * (Np * 4), Np * 32, &c.full[s]);
            else if (lane < 2 * EB) bulk_g2s(c.sR + (s * EB + lane - EB) * QS, d.res + (e0 + lane - EB) * (Np * 4), Np * 32, &c.full[s]);
            else if (lane < 3 * EB) bulk_g2s(c.sGeo + (s * EB + lane - 2 * EB) * GS, geox + (e0 + lane - 2 * EB) * GX3, GX3 * 8, &c.full[s]);
            // neighbour traces (16-byte cp.async gathers), or the ghost state (2 r^-, 0, 0, 0) behind an HABC face;
            // this half-warp serves faces 2 hw and 2 hw + 1 of element ie
            if (it >= 2) mbar_wait(&c.nfree[o], ((it >> 1) - 1) & 1);
            double* dn = c.sN + o * (Nfn * EB * 4) + hw * (2 * Nfp * 32) + ie * 4 + hsw;
#pragma unroll
            for (int fl = 0; fl < 2; ++fl) {
                const uint32_t cw = hw ? (fl ? cw4.w : cw4.z) : (fl ? cw4.y : cw4.x);
                const size_t id = (cw >> 5) & CONN_MAX_ID;
                const bool bnd = (cw & CONN_BND) != 0;
                const double* base = (bnd ? d.ghost3 + id * (Nfp * 4) : qold + id * (Np * 4)) + 2 * h;
                const int* tab = sNode + (bnd ? 32 : (int)(cw & 31)) * Nfp;    // row 32 is the identity
                int off[Nfp];                                // all table reads first: cp.async is a compiler barrier
#pragma unroll
                for (int j = 0; j < Nfp; ++j) off[j] = tab[j];
#pragma unroll
                for (int j = 0; j < Nfp; ++j) cp_async16(dn + (fl * Nfp + j) * 32, base + off[j]);
            }
            cp_async_arrive_noinc(&c.full[s]);
        }
        return;
    }

    // =================================================================== warpgroups 0, 1: MMA warps and helper 0
    reg_inc<C::REG_MMA>();
    if (w == 7) return ws2_helper<N>(c, 0, lane);
    if (w >= MT) return;

    const int g = lane >> 2, t = lane & 3;
    const int n = 8 * w + g;                                 // the node this lane owns in the accumulators
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
    double* hq = c.sH + (2 * t) * HS + n;                    // H[v][2t][n]; element 2t+1 at + HS
    const bool nok = n < Np;
    int it = 0;
    for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
        const int o = it & 1;
        const double* sB = sm + C::oB + o * C::szB;
        const double* sG = sB + 4 * KPD * EB;
        mbar_wait(&c.ready[o], (it >> 1) & 1);
        // ---- contractions (eq (41)): D_r p, D_s p, D_t p, div of the contravariant velocity
        double cpr[2] = {0, 0}, cps[2] = {0, 0}, cpt[2] = {0, 0}, cvr[2] = {0, 0}, cvs[2] = {0, 0}, cvt[2] = {0, 0};
        {
            const double* bp = sB + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KD; ++s_) {
                const double b0 = bp[(0 * KPD + 4 * s_) * EB];
                dmma884v(cpr, Ar[s_], b0);
                dmma884v(cps, As[s_], b0);
                dmma884v(cpt, At[s_], b0);
                dmma884v(cvr, Ar[s_], bp[(1 * KPD + 4 * s_) * EB]);
                dmma884v(cvs, As[s_], bp[(2 * KPD + 4 * s_) * EB]);
                dmma884v(cvt, At[s_], bp[(3 * KPD + 4 * s_) * EB]);
            }
        }
        if (it >= 1) mbar_wait(c.hfree, (it - 1) & 1);       // the helpers have consumed the previous batch's H
        if (nok) {
            hq[0] = cpr[0];          hq[HS] = cpr[1];
            hq[HV] = cps[0];         hq[HV + HS] = cps[1];
            hq[2 * HV] = cpt[0];     hq[2 * HV + HS] = cpt[1];
            hq[3 * HV] = (cvr[0] + cvs[0]) + cvt[0];
            hq[3 * HV + HS] = (cvr[1] + cvs[1]) + cvt[1];
        }
        // ---- LIFT_f g
        double cl[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
        {
            const double* gp = sG + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KL; ++s_)
#pragma unroll
                for (int f = 0; f < 4; ++f) dmma884v(cl[f], AL[f][s_], gp[f * LPAD + 4 * s_ * EB]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&c.opfree[o]);
        if (nok) {
#pragma unroll
            for (int f = 0; f < 4; ++f) { hq[(4 + f) * HV] = cl[f][0]; hq[(4 + f) * HV + HS] = cl[f][1]; }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(c.hfull);
    }
}

}  // namespace dg
