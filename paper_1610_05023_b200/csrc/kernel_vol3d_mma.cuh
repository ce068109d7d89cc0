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
// Tiling.  A batch is EB = 8 consecutive elements = one n-tile of the MMA.  Warp w owns the
// m-tile of nodes 8w..8w+7 for every contraction, and keeps ITS rows of D_r, D_s, D_t and LIFT as register-
// resident A fragments for the life of the persistent CTA (N=5: 66 doubles per lane).  The B operands
// (p, U^r, U^s, U^t per node; flux jump g per face node), one column per element, are staged in shared memory
// as [k][8] so that a B fragment is one conflict-free LDS.64.  The accumulator fragment of lane (g,t) holds
// node 8w+g of elements 2t, 2t+1 for all eight results (d_r p, d_s p, d_t p, div U, LIFT_f g for f = 0..3),
// so the update stage runs in registers without any exchange.
//
// Data movement.  Next batch's q, res, geometric record and the neighbours' face traces are fetched with
// cp.async (LDGSTS) straight into shared memory while the current batch is in its DMMA phase; q and res are
// transposed on the fly to [node][element] so every later shared-memory access is conflict-free.  Neighbour
// traces come from the stage-(n-1) buffer (ping-pong), which is what makes the fusion race-free.
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
    static constexpr int MT = (Np + 7) / 8;            // m-tiles = warps
    static constexpr int NPAD = MT * 8;
    static constexpr int KD = (Np + 3) / 4;            // k-steps of the D contractions
    static constexpr int KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4;           // k-steps of one face of LIFT
    static constexpr int KPL = KL * 4;
    static constexpr int NT = MT * 32;
    static constexpr int GEO_S = 26;                   // padded geometric record (16 B aligned, bank-spread)
    static constexpr int NITEM = (Nfn * EB + NT - 1) / NT;   // face-node items per thread
    // shared memory, in doubles
    static constexpr int oB = 0;                             // [4][KPD][8]   p, U^r, U^s, U^t
    static constexpr int oG = oB + 4 * KPD * EB;             // [4][KPL][8]   flux jump
    static constexpr int oQ = oG + 4 * KPL * EB;             // [2][NPAD][8][4]
    static constexpr int oR = oQ + 2 * NPAD * EB * 4;        // [2][NPAD][8][4]
    static constexpr int oN = oR + 2 * NPAD * EB * 4;        // [Nfn][8][4]   neighbour traces
    static constexpr int oGeo = oN + Nfn * EB * 4;           // [2][8][GEO_S]
    static constexpr int oEnd = oGeo + 2 * EB * GEO_S;
    static constexpr size_t smem_bytes = sizeof(double) * oEnd + sizeof(int) * (Nfn + 6 * Nfp) + 32;
    static constexpr int regs_A = 2 * (3 * KD + 4 * KL);
    static constexpr int min_ctas = regs_A > 100 ? 1 : (regs_A > 60 ? 2 : 3);
};

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int N>
__global__ void __launch_bounds__(MmaCfg<N>::NT, MmaCfg<N>::min_ctas)
k_vol3d_mma(Dev<double> d, int src, double rka, double rkb, double dt) {
    using C = MmaCfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KD = C::KD, KPD = C::KPD, KL = C::KL,
                  KPL = C::KPL, NT = C::NT, NPAD = C::NPAD, GS = C::GEO_S, NITEM = C::NITEM;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* sm = reinterpret_cast<double*>(smem_raw);
    double* sB = sm + C::oB;
    double* sG = sm + C::oG;
    double* sQ = sm + C::oQ;
    double* sR = sm + C::oR;
    double* sN = sm + C::oN;
    double* sGeo = sm + C::oGeo;
    int* sFmask = reinterpret_cast<int*>(sm + C::oEnd);      // [Nfn]
    int* sPerm = sFmask + Nfn;                               // [6][Nfp]

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g = lane >> 2, t = lane & 3;
    const int n = 8 * w + g;                                 // the node this lane owns in the accumulators
    const double* __restrict__ qold = d.q[src];
    double* __restrict__ qnew = d.q[src ^ 1];
    double* __restrict__ res = d.res;
    const int K = d.K;
    const int nbatch = (K + EB - 1) / EB;

    // ---- one-time: tables, zeroed operand padding, register-resident A fragments
    for (int i = tid; i < C::oQ; i += NT) sm[i] = 0.0;       // sB, sG (padding rows stay zero for ever)
    for (int i = tid; i < Nfn; i += NT) sFmask[i] = d.fmask3[i];
    for (int i = tid; i < 6 * Nfp; i += NT) sPerm[i] = d.perm3[i];
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

    // ---- loop-invariant roles of this thread in the face-node passes: item = (face node fj, element e)
    // (recomputed from idx where needed; kept out of registers)
    auto prefetch = [&](int b, int buf, const uint32_t (&cn)[NITEM]) {
        const int e0 = b * EB;
        // own q, res: 16-byte chunks, transposed to [node][element]
        double* dq = sQ + buf * (NPAD * EB * 4);
        double* dr = sR + buf * (NPAD * EB * 4);
        for (int c = tid; c < EB * Np * 2; c += NT) {
            const int e = c / (Np * 2), r = c - e * (Np * 2), nn = r >> 1, h = r & 1;
            const int k = min(e0 + e, K - 1);
            const size_t so = ((size_t)k * Np + nn) * 4 + 2 * h;
            const int dof = (nn * EB + e) * 4 + 2 * h;
            cp_async16(dq + dof, qold + so);
            cp_async16(dr + dof, res + so);
        }
        for (int c = tid; c < EB * (GEO3 / 2); c += NT) {
            const int e = c / (GEO3 / 2), r = c - e * (GEO3 / 2);
            const int k = min(e0 + e, K - 1);
            cp_async16(sGeo + (buf * EB + e) * GS + 2 * r, d.geo3 + (size_t)k * GEO3 + 2 * r);
        }
        // neighbour traces (or r^- of the HABC on boundary faces, PAPER.md:L514 / eq (30))
#pragma unroll
        for (int r = 0; r < NITEM; ++r) {
            const int idx = tid + NT * r;
            if (idx < Nfn * EB) {
                const int fj = idx >> 3, e = idx & 7;
                const int f = fj / Nfp, j = fj - f * Nfp;
                const uint32_t c = cn[r];
                const int id = (c >> 5) & CONN_MAX_ID;
                double* dst = sN + idx * 4;
                if (c & CONN_BND) {
                    cp_async8(dst, d.qb3 + (size_t)id * Nfp + j);
                } else {
                    const int node = sFmask[(c & 3) * Nfp + sPerm[((c >> 2) & 7) * Nfp + j]];
                    const double* s = qold + ((size_t)id * Np + node) * 4;
                    cp_async16(dst, s);
                    cp_async16(dst + 2, s + 2);
                }
            }
        }
        cp_async_commit();
    };
    auto load_conn = [&](int b, uint32_t (&cn)[NITEM]) {
#pragma unroll
        for (int r = 0; r < NITEM; ++r) {
            const int idx = tid + NT * r;
            cn[r] = 0;
            if (idx < Nfn * EB && b < nbatch) {
                const int fj = idx >> 3, e = idx & 7;
                const int k = min(b * EB + e, K - 1);
                cn[r] = d.conn3[(size_t)k * 4 + fj / Nfp];
            }
        }
    };

    uint32_t ccur[NITEM], cnext[NITEM];
    __syncthreads();                                         // tables visible before the first prefetch
    int b = blockIdx.x, buf = 0;
    if (b < nbatch) {
        load_conn(b, ccur);
        prefetch(b, 0, ccur);
        load_conn(b + gridDim.x, cnext);
    }

    for (; b < nbatch; b += gridDim.x, buf ^= 1) {
        const int e0 = b * EB;
        const double* bq = sQ + buf * (NPAD * EB * 4);
        const double* br = sR + buf * (NPAD * EB * 4);
        const double* bgeo = sGeo + buf * EB * GS;
        cp_async_wait_all();
        __syncthreads();
        // ---- phase A: (p, contravariant velocity) of my node for elements 2t, 2t+1 -> B operands
        if (n < Np) {
            double P[2], UR[2], US[2], UT[2];
#pragma unroll
            for (int ee = 0; ee < 2; ++ee) {
                const int e = 2 * t + ee;
                const double4 v = *reinterpret_cast<const double4*>(bq + (n * EB + e) * 4);
                const double* ge = bgeo + e * GS;
                P[ee] = v.x;
                UR[ee] = ge[0] * v.y + ge[1] * v.z + ge[2] * v.w;
                US[ee] = ge[3] * v.y + ge[4] * v.z + ge[5] * v.w;
                UT[ee] = ge[6] * v.y + ge[7] * v.z + ge[8] * v.w;
            }
            double* o = sB + n * EB + 2 * t;
            *reinterpret_cast<double2*>(o) = make_double2(P[0], P[1]);
            *reinterpret_cast<double2*>(o + KPD * EB) = make_double2(UR[0], UR[1]);
            *reinterpret_cast<double2*>(o + 2 * KPD * EB) = make_double2(US[0], US[1]);
            *reinterpret_cast<double2*>(o + 3 * KPD * EB) = make_double2(UT[0], UT[1]);
        }
        __syncthreads();
        // ---- phase B: one scalar flux jump per face node (upwind flux PAPER.md:L499-512)
#pragma unroll
        for (int r = 0; r < NITEM; ++r) {
            const int idx = tid + NT * r;
            if (idx < Nfn * EB) {
                const int fj = idx >> 3, e = idx & 7;
                const int f = fj / Nfp, j = fj - f * Nfp;
                const double* ge = bgeo + e * GS;
                const int o = sFmask[fj] * EB + e;
                const double pM = sB[o], ur = sB[o + KPD * EB], us = sB[o + 2 * KPD * EB], ut = sB[o + 3 * KPD * EB];
                // Fs n.u^- = nhat . U^-   (nhat: f0 (0,0,-1), f1 (0,-1,0), f2 (1,1,1), f3 (-1,0,0))
                const double unM = (f == 0) ? -ut : (f == 1) ? -us : (f == 2) ? (ur + us + ut) : -ur;
                const double4 x = *reinterpret_cast<const double4*>(sN + idx * 4);
                double pP, unP;
                if (ccur[r] & CONN_BND) {
                    pP = 2.0 * x.x;                          // ghost state p+ = 2 r^-, u+ = 0
                    unP = 0.0;
                } else {
                    double nx, ny, nz;                       // Fs n = nhat . G
                    if (f == 0) { nx = -ge[6]; ny = -ge[7]; nz = -ge[8]; }
                    else if (f == 1) { nx = -ge[3]; ny = -ge[4]; nz = -ge[5]; }
                    else if (f == 2) { nx = ge[0] + ge[3] + ge[6]; ny = ge[1] + ge[4] + ge[7]; nz = ge[2] + ge[5] + ge[8]; }
                    else { nx = -ge[0]; ny = -ge[1]; nz = -ge[2]; }
                    pP = x.x;
                    unP = nx * x.y + ny * x.z + nz * x.w;
                }
                sG[(f * KPL + j) * EB + e] = ge[9 + f] * (unP - unM) - ge[13 + f] * (pP - pM);
            }
        }
        __syncthreads();
        // ---- next batch's data starts moving while this one is in the tensor pipe
        if (b + (int)gridDim.x < nbatch) {
#pragma unroll
            for (int r = 0; r < NITEM; ++r) ccur[r] = cnext[r];
            prefetch(b + gridDim.x, buf ^ 1, ccur);
            load_conn(b + 2 * gridDim.x, cnext);
        }
        // ---- phase C: contractions
        double cpr[2] = {0, 0}, cps[2] = {0, 0}, cpt[2] = {0, 0}, cvr[2] = {0, 0}, cvs[2] = {0, 0}, cvt[2] = {0, 0};
        double cl[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
        {
            const double* bp = sB + t * EB + g;
#pragma unroll
            for (int s = 0; s < KD; ++s) {
                const double b0 = bp[(0 * KPD + 4 * s) * EB];
                dmma884(cpr, Ar[s], b0);
                dmma884(cps, As[s], b0);
                dmma884(cpt, At[s], b0);
                dmma884(cvr, Ar[s], bp[(1 * KPD + 4 * s) * EB]);
                dmma884(cvs, As[s], bp[(2 * KPD + 4 * s) * EB]);
                dmma884(cvt, At[s], bp[(3 * KPD + 4 * s) * EB]);
            }
            const double* gp = sG + t * EB + g;
#pragma unroll
            for (int s = 0; s < KL; ++s)
#pragma unroll
                for (int f = 0; f < 4; ++f) dmma884(cl[f], AL[f][s], gp[(f * KPL + 4 * s) * EB]);
        }
        // ---- phase D: right-hand side and LSRK update (eq (41)-(43)) of node n, elements 2t, 2t+1
        if (n < Np) {
#pragma unroll
            for (int ee = 0; ee < 2; ++ee) {
                const int e = 2 * t + ee;
                if (e0 + e < K) {
                    const double* ge = bgeo + e * GS;
                    const double a0 = cl[0][ee], a1 = cl[1][ee], a2 = cl[2][ee], a3 = cl[3][ee];
                    const double lp = ge[17] * a0 + ge[18] * a1 + ge[19] * a2 + ge[20] * a3;
                    const double rc2 = ge[21], irho = ge[22], cc = ge[23];
                    // -1/rho grad p + c * sum_f (Fs n)_f LIFT_f g, both through G^T:  G^T (c*l - irho*dp)
                    const double xr = cc * (a2 - a3) - irho * cpr[ee];
                    const double xs = cc * (a2 - a1) - irho * cps[ee];
                    const double xt = cc * (a2 - a0) - irho * cpt[ee];
                    const double rp = -rc2 * ((cvr[ee] + cvs[ee]) + cvt[ee] + lp);
                    const double ru = ge[0] * xr + ge[3] * xs + ge[6] * xt;
                    const double rv = ge[1] * xr + ge[4] * xs + ge[7] * xt;
                    const double rw = ge[2] * xr + ge[5] * xs + ge[8] * xt;
                    double4 q = *reinterpret_cast<const double4*>(bq + (n * EB + e) * 4);
                    double4 rr = *reinterpret_cast<const double4*>(br + (n * EB + e) * 4);
                    rr.x = rka * rr.x + dt * rp;  q.x += rkb * rr.x;
                    rr.y = rka * rr.y + dt * ru;  q.y += rkb * rr.y;
                    rr.z = rka * rr.z + dt * rv;  q.z += rkb * rr.z;
                    rr.w = rka * rr.w + dt * rw;  q.w += rkb * rr.w;
                    const size_t o = ((size_t)(e0 + e) * Np + n) * 4;
                    __stcs(reinterpret_cast<double2*>(res + o), make_double2(rr.x, rr.y));
                    __stcs(reinterpret_cast<double2*>(res + o + 2), make_double2(rr.z, rr.w));
                    __stcs(reinterpret_cast<double2*>(qnew + o), make_double2(q.x, q.y));
                    __stcs(reinterpret_cast<double2*>(qnew + o + 2), make_double2(q.z, q.w));
                }
            }
        }
    }
    cp_async_wait_all();
}

}  // namespace dg
