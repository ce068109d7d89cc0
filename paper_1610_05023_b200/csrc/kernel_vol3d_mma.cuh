// 3D solver, fp64, tensor-pipe version: fused volume + surface + update of one LSRK stage (PAPER.md:L623-624,
// Alg. 2, eq (41)-(43)) with the three dense contractions of eq (41) -- D_r/D_s/D_t applied to p, the
// divergence of the contravariant velocity, and LIFT applied to the upwind flux jump -- issued as fp64
// mma.sync.m8n8k4 (SASS DMMA.8x8x4) tiles.
//
// Why DMMA: on B200 DMMA and DFMA run on the same fp64 units (37.1 TFLOP/s each, 33 TFLOP/s when mixed;
// profiles/r01_peaks.md), so the tensor form buys no flops -- it buys issue slots and shared-memory bandwidth:
// one DMMA replaces 8 DFMA per lane and needs one 8-byte operand per lane from shared memory, where the
// scalar kernel needs a 16-byte broadcast per 2 DFMA and is bound by the 128 B/clk shared-memory port.
//
// Tiling.  A batch is EB = 8 consecutive elements = one n-tile of the MMA.  MMA warp w owns
// the m-tile of nodes 8w..8w+7 for every contraction, and keeps ITS rows of D_r, D_s, D_t and LIFT as register-
// resident A fragments for the life of the persistent CTA (N=5: 66 doubles per lane).  The B operands
// (p, U^r, U^s, U^t per node; flux jump g per face node), one column per element, are staged in shared memory
// as [k][8] (columns swizzled) so that a B fragment is one conflict-free LDS.64.  The accumulator fragment of
// lane (g,t) holds node 8w+g of elements 2t, 2t+1 for all eight results (d_r p, d_s p, d_t p, div U, LIFT_f g
// for f = 0..3), so the update stage runs in registers without any exchange.
//
// Data movement.  One extra PRODUCER warp runs one batch ahead of the MMA warps: it moves the batch's q, res
// and geometric records with bulk async copies (cp.async.bulk, the TMA engine: no LSU wavefronts) and gathers
// the neighbours' face traces with 16-byte cp.async, all completing on one mbarrier per buffer (full[s]); the
// MMA warps hand a buffer back through empty[s].  Neighbour traces come from the stage-(n-1) buffer
// (ping-pong q), which is what makes the fusion race-free; on boundary faces the "neighbour" is the ghost
// state (2 r^-, 0, 0, 0) that k_close_face stores (eq (30)), so the flux code has no branch.
#pragma once
#include "kernels.cuh"

namespace dg {

// conn3 word per (element, face): bit 31 = boundary face; bits 5..30 = neighbour tet | boundary triangle;
// bits 0..1 = neighbour's local face; bits 2..4 = face-node permutation id.
constexpr uint32_t CONN_BND = 0x80000000u;
constexpr int CONN_MAX_ID = (1 << 26) - 1;

template <int N>
struct MmaCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EB = 8;                       // elements per batch = MMA n
    static constexpr int MT = (Np + 7) / 8;            // m-tiles = MMA warps
    static constexpr int NPAD = MT * 8;
    static constexpr int KD = (Np + 3) / 4;            // k-steps of the D contractions
    static constexpr int KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4;           // k-steps of one face of LIFT
    static constexpr int KPL = KL * 4;
    static constexpr int NTM = MT * 32;                // MMA threads
    static constexpr int NT = NTM + 32;                // + the producer warp
    static constexpr int GEO_S = 26;                   // staged geometric record stride (16 B aligned, bank-spread)
    static constexpr int NITEM = (Nfn * EB + NTM - 1) / NTM;   // face-node items per MMA thread
    static constexpr int PITEM = (Nfn * EB + 31) / 32;         // face-node items per producer lane
    static constexpr int QS = Np * 4 + 2;              // staged element stride of q / res ([e][node][4], 16 B skew)
    // shared memory, in doubles
    static constexpr int szB = 4 * KPD * EB + 4 * KPL * EB;  // one operand buffer: p,U^r,U^s,U^t [4][KPD][8] + g [4][KPL][8]
    static constexpr int oB = 0;                             // [2] operand buffers (columns swizzled)
    static constexpr int oQ = oB + 2 * szB;                  // [2][8][QS]
    static constexpr int oR = oQ + 2 * EB * QS;              // [2][8][QS]
    static constexpr int oN = oR + 2 * EB * QS;              // [2][Nfn][2][8][2] neighbour traces
    static constexpr int oGeo = oN + 2 * Nfn * EB * 4;       // [2][8][GEO_S]
    static constexpr int oBar = oGeo + 2 * EB * GEO_S;       // full[2], empty[2]
    static constexpr int oEnd = oBar + 4;
    static constexpr size_t smem_bytes = sizeof(double) * oEnd + sizeof(int) * (32 * Nfp) + 32;
    static constexpr uint32_t tx_bytes = 2 * EB * Np * 32 + EB * GEO3 * 8;
    static constexpr int regs_A = 2 * (3 * KD + 4 * KL);
    static constexpr int min_ctas = regs_A > 100 ? 1 : (regs_A > 60 ? 2 : 3);
};

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
// the mbarrier gets one arrival when all cp.async issued so far by this thread have landed
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem, const void* gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
template <int NTHREADS>
__device__ __forceinline__ void bar_mma_warps() { asm volatile("bar.sync 1, %0;" ::"n"(NTHREADS) : "memory"); }

// column swizzle of the [k][8] operand arrays: makes both the B-fragment LDS.64 (lanes (g,t) -> row 4s+t,
// column g) and the 16-byte operand stores (row n, columns 2t..2t+1) bank-conflict free
__device__ __forceinline__ int swz(int row) { return ((row >> 1) & 1) << 2; }

template <int N>
__global__ void __launch_bounds__(MmaCfg<N>::NT, MmaCfg<N>::min_ctas)
k_vol3d_mma(Dev<double> d, int src, double rka, double rkb, double dt) {
    using C = MmaCfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  KPL = C::KPL, NTM = C::NTM, NT = C::NT, GS = C::GEO_S, NITEM = C::NITEM, QS = C::QS, MT = C::MT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sm = reinterpret_cast<double*>(smem_raw);
    double* sQ = sm + C::oQ;
    double* sR = sm + C::oR;
    double* sN = sm + C::oN;
    double* sGeo = sm + C::oGeo;
    uint64_t* full = reinterpret_cast<uint64_t*>(sm + C::oBar);
    uint64_t* empty = full + 2;
    int* sNode = reinterpret_cast<int*>(sm + C::oEnd);       // [32][Nfp]: (face | perm << 2, j) -> neighbour node

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const double* __restrict__ qold = d.q[src];
    const int K = d.K;
    const int nbatch = (K + EB - 1) / EB;                    // arrays are padded to nbatch * EB elements

    // ---- one-time: tables, zeroed operand buffers (their padding rows stay zero for ever), barriers
    for (int i = tid; i < C::oQ; i += NT) sm[i] = 0.0;
    for (int i = tid; i < 32 * Nfp; i += NT) {
        const int fp = i / Nfp, j = i - fp * Nfp, pm = fp >> 2;
        sNode[i] = pm < 6 ? d.fmask3[(fp & 3) * Nfp + d.perm3[pm * Nfp + j]] : 0;
    }
    if (tid == 0) {
        mbar_init(&full[0], 33); mbar_init(&full[1], 33);    // 32 cp.async arrivals + 1 expect_tx arrival
        mbar_init(&empty[0], MT); mbar_init(&empty[1], MT);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async;" ::: "memory");
    }
    __syncthreads();

    if (w == MT) {
        // =============================================================== producer warp
        constexpr int PITEM = C::PITEM;
        const int ie = lane & 7;
        int it = 0;
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it & 1;
            // connectivity words of this lane's items (independent loads, issued before the wait)
            uint32_t cn[PITEM];
#pragma unroll
            for (int r = 0; r < PITEM; ++r) {
                const int fj = (lane >> 3) + 4 * r;
                cn[r] = fj < Nfn ? d.conn3[((size_t)b * EB + ie) * 4 + fj / Nfp] : 0u;
            }
            if (it >= 2) mbar_wait(&empty[s], ((it >> 1) - 1) & 1);
            const size_t e0 = (size_t)b * EB;
            if (lane == 0) mbar_arrive_expect_tx(&full[s], C::tx_bytes);
            __syncwarp();
            if (lane < EB) bulk_g2s(sQ + (s * EB + lane) * QS, qold + (e0 + lane) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 2 * EB) bulk_g2s(sR + (s * EB + lane - EB) * QS, d.res + (e0 + lane - EB) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 3 * EB) bulk_g2s(sGeo + (s * EB + lane - 2 * EB) * GS, d.geo3 + (e0 + lane - 2 * EB) * GEO3, GEO3 * 8, &full[s]);
            // neighbour traces, or the ghost state on boundary faces
            double* dn = sN + s * (Nfn * EB * 4);
#pragma unroll
            for (int r = 0; r < PITEM; ++r) {
                const int fj = (lane >> 3) + 4 * r;
                if (fj < Nfn) {
                    const int j = fj % Nfp;
                    const uint32_t c = cn[r];
                    const size_t id = (c >> 5) & CONN_MAX_ID;
                    const double* sp = (c & CONN_BND) ? d.ghost3 + (id * Nfp + j) * 4
                                                      : qold + (id * Np + sNode[(c & 31) * Nfp + j]) * 4;
                    double* dst = dn + fj * 32 + ie * 2;
                    cp_async16(dst, sp);
                    cp_async16(dst + 16, sp + 2);
                }
            }
            cp_async_arrive_noinc(&full[s]);
        }
        return;
    }

    // =================================================================== MMA warps
    const int g = lane >> 2, t = lane & 3;
    const int n = 8 * w + g;                                 // the node this lane owns in the accumulators
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
    // face-node role: item r = (face node fj, element ie); packed f | j << 2 | fmask << 10
    const int ie = tid & 7;
    int item[NITEM];
#pragma unroll
    for (int r = 0; r < NITEM; ++r) {
        const int fj = (tid >> 3) + (NTM >> 3) * r;
        const int f = fj / Nfp, j = fj - f * Nfp;
        item[r] = fj < Nfn ? (f | (j << 2) | ((int)d.fmask3[fj] << 10)) : -1;
    }

    int it = 0;
    for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
        const int s = it & 1;
        const int e0 = b * EB;
        const double* bq = sQ + s * (EB * QS);
        const double* br = sR + s * (EB * QS);
        const double* bgeo = sGeo + s * EB * GS;
        const double* bn = sN + s * (Nfn * EB * 4);
        double* sB = sm + C::oB + s * C::szB;                // operand buffers alternate: one barrier per batch
        double* sG = sB + 4 * KPD * EB;
        mbar_wait(&full[s], (it >> 1) & 1);
        // ---- phase A: (p, contravariant velocity) of my node for elements 2t, 2t+1 -> B operands
        if (n < Np) {
            double P[2], UR[2], US[2], UT[2];
#pragma unroll
            for (int ee = 0; ee < 2; ++ee) {
                const int e = 2 * t + ee;
                const double2 v0 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4);
                const double2 v1 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4 + 2);
                const double* ge = bgeo + e * GS;
                P[ee] = v0.x;
                UR[ee] = ge[0] * v0.y + ge[1] * v1.x + ge[2] * v1.y;
                US[ee] = ge[3] * v0.y + ge[4] * v1.x + ge[5] * v1.y;
                UT[ee] = ge[6] * v0.y + ge[7] * v1.x + ge[8] * v1.y;
            }
            double* o = sB + n * EB + ((2 * t) ^ swz(n));
            *reinterpret_cast<double2*>(o) = make_double2(P[0], P[1]);
            *reinterpret_cast<double2*>(o + KPD * EB) = make_double2(UR[0], UR[1]);
            *reinterpret_cast<double2*>(o + 2 * KPD * EB) = make_double2(US[0], US[1]);
            *reinterpret_cast<double2*>(o + 3 * KPD * EB) = make_double2(UT[0], UT[1]);
        }
        // ---- phase B: one scalar flux jump per face node (upwind flux PAPER.md:L499-512):
        //      g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-), in physical components straight from the staged q
        {
            const double* ge = bgeo + ie * GS;
            const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                          g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6);
            const double g8 = ge[8];
#pragma unroll
            for (int r = 0; r < NITEM; ++r) {
                if (item[r] >= 0) {
                    const int f = item[r] & 3, j = (item[r] >> 2) & 255, fm = item[r] >> 10;
                    const int fj = (tid >> 3) + (NTM >> 3) * r;
                    const double2 m0 = *reinterpret_cast<const double2*>(bq + ie * QS + fm * 4);
                    const double2 m1 = *reinterpret_cast<const double2*>(bq + ie * QS + fm * 4 + 2);
                    const double2 x0 = *reinterpret_cast<const double2*>(bn + fj * 32 + ie * 2);
                    const double2 x1 = *reinterpret_cast<const double2*>(bn + fj * 32 + 16 + ie * 2);
                    // MINUS the scaled outward normal, Fs n = nhat . G  (nhat: f0 (0,0,-1), f1 (0,-1,0), f2 (1,1,1), f3 (-1,0,0))
                    double nx = (f == 0) ? g67.x : (f == 1) ? g23.y : g01.x;
                    double ny = (f == 0) ? g67.y : (f == 1) ? g45.x : g01.y;
                    double nz = (f == 0) ? g8 : (f == 1) ? g45.y : g23.x;
                    if (f == 2) { nx = -(g01.x + g23.y + g67.x); ny = -(g01.y + g45.x + g67.y); nz = -(g23.x + g45.y + g8); }
                    const double dn = -(nx * (x0.y - m0.y) + ny * (x1.x - m1.x) + nz * (x1.y - m1.y));
                    sG[(f * KPL + j) * EB + (ie ^ swz(j))] = ge[9 + f] * dn - ge[13 + f] * (x0.x - m0.x);
                }
            }
        }
        bar_mma_warps<NTM>();
        // ---- phase C: contractions
        double cpr[2] = {0, 0}, cps[2] = {0, 0}, cpt[2] = {0, 0}, cvr[2] = {0, 0}, cvs[2] = {0, 0}, cvt[2] = {0, 0};
        double cl[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
        {
            const double* bp = sB + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KD; ++s_) {
                const double b0 = bp[(0 * KPD + 4 * s_) * EB];
                dmma884(cpr, Ar[s_], b0);
                dmma884(cps, As[s_], b0);
                dmma884(cpt, At[s_], b0);
                dmma884(cvr, Ar[s_], bp[(1 * KPD + 4 * s_) * EB]);
                dmma884(cvs, As[s_], bp[(2 * KPD + 4 * s_) * EB]);
                dmma884(cvt, At[s_], bp[(3 * KPD + 4 * s_) * EB]);
            }
            const double* gp = sG + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KL; ++s_)
#pragma unroll
                for (int f = 0; f < 4; ++f) dmma884(cl[f], AL[f][s_], gp[(f * KPL + 4 * s_) * EB]);
        }
        // ---- phase D: right-hand side and LSRK update (eq (41)-(43)) of node n, elements 2t, 2t+1
        if (n < Np) {
#pragma unroll
            for (int ee = 0; ee < 2; ++ee) {
                const int e = 2 * t + ee;
                if (e0 + e < K) {
                    const double* ge = bgeo + e * GS;
                    const double2 g01 = *reinterpret_cast<const double2*>(ge), g23 = *reinterpret_cast<const double2*>(ge + 2),
                                  g45 = *reinterpret_cast<const double2*>(ge + 4), g67 = *reinterpret_cast<const double2*>(ge + 6),
                                  g8_ = *reinterpret_cast<const double2*>(ge + 8), f01 = *reinterpret_cast<const double2*>(ge + 16),
                                  f23 = *reinterpret_cast<const double2*>(ge + 18), f4r = *reinterpret_cast<const double2*>(ge + 20),
                                  irc = *reinterpret_cast<const double2*>(ge + 22);
                    const double a0 = cl[0][ee], a1 = cl[1][ee], a2 = cl[2][ee], a3 = cl[3][ee];
                    const double lp = f01.y * a0 + f23.x * a1 + f23.y * a2 + f4r.x * a3;
                    const double rc2 = f4r.y, irho = irc.x, cc = irc.y;
                    // -1/rho grad p + c * sum_f (Fs n)_f LIFT_f g, both through G^T:  G^T (c*l - irho*dp)
                    const double xr = cc * (a2 - a3) - irho * cpr[ee];
                    const double xs = cc * (a2 - a1) - irho * cps[ee];
                    const double xt = cc * (a2 - a0) - irho * cpt[ee];
                    const double rp = -rc2 * ((cvr[ee] + cvs[ee]) + cvt[ee] + lp);
                    const double ru = g01.x * xr + g23.y * xs + g67.x * xt;
                    const double rv = g01.y * xr + g45.x * xs + g67.y * xt;
                    const double rw = g23.x * xr + g45.y * xs + g8_.x * xt;
                    double2 q0 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4);
                    double2 q1 = *reinterpret_cast<const double2*>(bq + e * QS + n * 4 + 2);
                    double2 r0 = *reinterpret_cast<const double2*>(br + e * QS + n * 4);
                    double2 r1 = *reinterpret_cast<const double2*>(br + e * QS + n * 4 + 2);
                    r0.x = rka * r0.x + dt * rp;  q0.x += rkb * r0.x;
                    r0.y = rka * r0.y + dt * ru;  q0.y += rkb * r0.y;
                    r1.x = rka * r1.x + dt * rv;  q1.x += rkb * r1.x;
                    r1.y = rka * r1.y + dt * rw;  q1.y += rkb * r1.y;
                    const size_t o = ((size_t)(e0 + e) * Np + n) * 4;
                    __stcs(reinterpret_cast<double2*>(res + o), r0);
                    __stcs(reinterpret_cast<double2*>(res + o + 2), r1);
                    __stcs(reinterpret_cast<double2*>(qnew + o), q0);
                    __stcs(reinterpret_cast<double2*>(qnew + o + 2), q1);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }
}

}  // namespace dg
