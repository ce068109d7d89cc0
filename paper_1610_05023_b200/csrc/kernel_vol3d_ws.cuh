// 3D solver, fp64, warp-specialised tensor-pipe version: fused volume + surface + update of one LSRK stage
// (Alg. 2, eq (41)-(43)).  Same mathematics and the same DMMA tiling as
// kernel_vol3d_mma.cuh (m-tile of 8 nodes per MMA warp, operator rows register-resident, batch of 8 elements =
// MMA n); what changes is WHO does what, so that the fp64 unit never waits (profiles/r01a_*: in the batch-
// synchronous kernel the DMMA sub-pipe was busy 45 % of the time because operand build, contraction and update
// ran back to back behind a CTA-wide barrier).
//
// 12 warps, three roles, decoupled by mbarriers:
//   warps 0..MT-1  MMA      wait ready[o] -> 108 DMMA (N=5) from operand buffer o -> release opfree[o] ->
//                           right-hand side + LSRK update of their 8 nodes x 8 elements -> release empty[s]
//   warp 7         LOADER   bulk async copies (cp.async.bulk, the TMA engine) of q, res and the geometric
//                           records of a batch, plus 16-byte cp.async gathers of the neighbours' face traces,
//                           into stage s of NS, all completing on full[s]
//   warps 8..11    PREP     wait full[s]; build the operands (p, contravariant velocity; one upwind flux jump per
//                           face node) into operand buffer o; signal ready[o]
// With at most three m-tiles (N <= 3) the same roles are packed into two warpgroups -- MMA 0..MT-1, LOADER 3, PREP
// 4..7, 256 threads -- and two CTAs share an SM (WsCfg::COMPACT): in the 12-warp layout four warps would only hold
// registers and an SM would run three MMA warps (N = 3 on the SEAM-shaped workload: 1075 -> 753 us per launch).
// PREP runs one batch ahead of MMA, LOADER up to NS-1 batches ahead.  Register budget (setmaxnreg): the two
// MMA warpgroups take 208 registers per thread (132 of them hold the operator fragments), PREP 88.
#pragma once
#include "kernel_vol3d_mma.cuh"

namespace dg {

constexpr int GX3 = 44;   // per-tet record of this kernel, in values of T.  Every constant of the stage is folded in on
                          // the host, so that the update needs no scaling of its own (Z = rho c of the cell):
                          //  0..8   Ga = -dt rho c^2 G, G = (r,s,t)_(x,y,z): the operand rows are -dt rho c^2 (G u)
                          //  9..11, 36..41  Gb = -dt/rho G: the velocity right-hand side is Gb^T y
                          // 12+4f   (Fs n)_x, (Fs n)_y, (Fs n)_z, Z A_f   (f = 0..3; scaled OUTWARD normal)
                          // 28+f    Z B_f          32+f  dt c Fs_f          42, 43 pad
                          // A_f = Z+/((Z+ + Z-) Fs_f), B_f = 1/(Z+ + Z-)   (upwind flux)

template <int N>
struct WsCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EB = 8;
    static constexpr int MT = (Np + 7) / 8;            // MMA warps
    static constexpr int KD = (Np + 3) / 4, KPD = KD * 4;
    static constexpr int KL = (Nfp + 3) / 4, KPL = KL * 4;
    static constexpr int LPAD = KPL * EB + 8;          // stride of one face block of the flux operand (bank spread)
    // warp roles: MMA warps 0..MT-1, LOADER warp LW, PREP warps PW0..PW0+3.  With MT <= 3 (N <= 3) the roles fit two
    // warpgroups and two CTAs share an SM; otherwise three warpgroups, one CTA per SM
    static constexpr bool COMPACT = MT <= 3;
    static constexpr int NT = COMPACT ? 256 : 384, LW = COMPACT ? 3 : 7, PW0 = COMPACT ? 4 : 8, MINB = COMPACT ? 2 : 1;
    static constexpr int NS = 3;                       // staging depth
    // staged q / res: element e sits at e * QS + 2 * slot(e) doubles, QS a multiple of 128 bytes and slot(e) a
    // permutation of the eight 16-byte bank groups chosen so that BOTH access patterns are conflict-free: PREP
    // (8 elements, one node per quarter-warp) and the update of the MMA warps (4 elements of equal parity x 2
    // adjacent nodes per quarter-warp: elements {0,2,4,6} -> slots {0,1,4,5}, {1,3,5,7} -> {2,3,6,7})
    static constexpr int QS = ((Np * 4 + 15) / 16) * 16 + 16;
    static constexpr int GS = GX3 + 2;                 // staged stride of the geometric record: 368 B = 23 x 16 B, so that
                                                       // the records of elements 0..7 fall in distinct 16-byte bank groups
    static constexpr int szB = 4 * KPD * EB + 4 * LPAD;
    static constexpr int oB = 0;                       // [2][szB]        operand buffers
    static constexpr int oQ = oB + 2 * szB;            // [NS][8][QS]
    static constexpr int oR = oQ + NS * EB * QS;       // [NS][8][QS]
    static constexpr int oGeo = oR + NS * EB * QS;     // [NS][8][GX3]
    static constexpr int oN = oGeo + NS * EB * GS;     // [NS][Nfn][8][4] neighbour traces (halves of elements 4..7 swapped)
    static constexpr int oBar = oN + NS * Nfn * EB * 4;  // full[NS], empty[NS], ready[2], opfree[2]
    static constexpr int oEnd = oBar + 2 * NS + 4;
    static constexpr size_t smem_bytes = sizeof(double) * oEnd + sizeof(int) * (33 * Nfp + Nfn) + 32;
    static_assert(smem_bytes <= 227 * 1024, "shared memory");
    static constexpr uint32_t tx_bytes = 2 * EB * Np * 32 + EB * GX3 * 8;
    static constexpr int NJ = (Nfp + 3) / 4;           // face nodes per PREP thread (j = pw + 4 r)
    static constexpr int PITEM = (Nfn + 3) / 4;        // face nodes per LOADER lane
    // setmaxnreg: the kernel is compiled for 168 registers (65536 / 384 rounded down to a multiple of 8); the
    // registers the PREP warpgroup gives back are the only pool the two MMA warpgroups can grow from
    static constexpr int REG_BASE = COMPACT ? 128 : 168, REG_PREP = 88, REG_MMA = COMPACT ? 168 : 208;
    static_assert((REG_BASE - REG_PREP) * 128 >= (REG_MMA - REG_BASE) * (NT - 128), "setmaxnreg pool would deadlock");
    static_assert(REG_BASE * NT * MINB <= 65536, "register file");
    static_assert(MT <= 7, "the warp-specialised kernel covers N <= 5");
};

__device__ __forceinline__ int ws_eoff(int e, int QS) {
    const int a = e >> 1;
    return e * QS + 2 * (2 * (e & 1) + (a & 1) + 4 * (a >> 1));
}

__device__ __forceinline__ double2 ldg_nc2(const double* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
template <int R> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(R)); }
template <int R> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(R)); }

// volatile: keeps the written issue order (independent accumulators interleaved) and pins the hand-over point
__device__ __forceinline__ void dmma884v(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ void bar_sync64(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void bar_arrive64(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

template <int N>
__global__ void __launch_bounds__(WsCfg<N>::NT, WsCfg<N>::MINB)
k_vol3d_ws(Dev<double> d, const double* __restrict__ geox, int src, double rka, double rkb) {
    using C = WsCfg<N>;
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
        for (int o = 0; o < 2; ++o) { mbar_init(&ready[o], 4); mbar_init(&opfree[o], MT); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async;" ::: "memory");
    }
    __syncthreads();

    if (w >= C::PW0) {
        // =============================================================== PREP warps
        reg_dec<C::REG_PREP>();
        const int pw = w - C::PW0;
        const int ie = lane & 7, f = lane >> 3;
        const int slot = f + 4 * pw;                         // phase A: nodes slot + 16 r of element ie
        int fmo[NJ];                                         // phase B: own node of face node j = pw + 4 r of face f
#pragma unroll
        for (int r = 0; r < NJ; ++r) fmo[r] = (pw + 4 * r < Nfp) ? 4 * sFm[f * Nfp + pw + 4 * r] : 0;
        int it = 0;
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it % NS, o = it & 1;
            const double* bq = sQ + s * EB * QS + ws_eoff(ie, QS);
            const double* ge = sGeo + (s * EB + ie) * GS;
            const double* bn = sN + s * (Nfn * EB * 4) + f * (Nfp * 32) + ie * 4;
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
                        const double2 m0 = *reinterpret_cast<const double2*>(bq + fmo[r]);
                        const double2 m1 = *reinterpret_cast<const double2*>(bq + fmo[r] + 2);
                        const double2 x0 = *reinterpret_cast<const double2*>(bn + j * 32 + h0);
                        const double2 x1 = *reinterpret_cast<const double2*>(bn + j * 32 + (2 - h0));
                        const double dn = nxy.x * (x0.y - m0.y) + nxy.y * (x1.x - m1.x) + nzA.x * (x1.y - m1.y);
                        sG[j * EB + (ie ^ swz(j))] = nzA.y * dn - Bf * (x0.x - m0.x);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready[o]);
        }
        return;
    }

    reg_inc<C::REG_MMA>();
    if (w == C::LW) {
        // =============================================================== LOADER warp
        // gather role: lanes 2k, 2k+1 fetch the two 16-byte halves of one node's (p,u,v,w): one 32-byte sector
        const int ie = (lane >> 1) & 7, h = lane & 1, hw = lane >> 4;
        const int hsw = 2 * (h ^ ((ie >> 2) & 1));           // halves of elements 4..7 are swapped (bank spread)
        const uint4* conn = reinterpret_cast<const uint4*>(d.conn3);
        int it = 0;
        uint4 cnext = conn[(size_t)blockIdx.x * EB + ie];
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it % NS;
            const uint4 cw4 = cnext;                         // connectivity of element ie, one word per face
            if (b + (int)gridDim.x < nbatch) cnext = conn[(size_t)(b + gridDim.x) * EB + ie];
            if (it >= NS) mbar_wait(&empty[s], ((it / NS) - 1) & 1);
            const size_t e0 = (size_t)b * EB;
            if (lane == 0) mbar_arrive_expect_tx(&full[s], C::tx_bytes);
            __syncwarp();
            if (lane < EB) bulk_g2s(sQ + s * EB * QS + ws_eoff(lane, QS), qold + (e0 + lane) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 2 * EB) bulk_g2s(sR + s * EB * QS + ws_eoff(lane - EB, QS), d.res + (e0 + lane - EB) * (Np * 4), Np * 32, &full[s]);
            else if (lane < 3 * EB) bulk_g2s(sGeo + (s * EB + lane - 2 * EB) * GS, geox + (e0 + lane - 2 * EB) * GX3, GX3 * 8, &full[s]);
            // neighbour traces (16-byte cp.async gathers), or the ghost state (2 r^-, 0, 0, 0) behind an HABC face;
            // this half-warp serves faces 2 hw and 2 hw + 1 of element ie
            double* dn = sN + s * (Nfn * EB * 4) + hw * (2 * Nfp * 32) + ie * 4 + hsw;
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

    // Ping-pong: the two MMA warps that share an SM sub-partition (w and w ^ 4) take turns on the fp64 unit, so
    // that one warp's update phase runs under the other's 108 DMMA instead of both idling the unit together.
    // Named barriers 1..6 carry the token (bar.sync by the waiter + bar.arrive by the partner = 64 threads).
    const bool paired = (w ^ 4) < MT;
    const int my_turn = 1 + 2 * (w & 3) + (w >> 2), partner_turn = 1 + 2 * (w & 3) + ((w >> 2) ^ 1);
    if (paired && w >= 4) bar_arrive64(partner_turn);       // the lower warp goes first
    int it = 0;
    for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
        const int s = it % NS, o = it & 1;
        const int e0 = b * EB;
        const double* bq = sQ + s * (EB * QS);
        const double* br = sR + s * (EB * QS);
        const double* bgeo = sGeo + s * EB * GS;
        const double* sB = sm + C::oB + o * C::szB;
        const double* sG = sB + 4 * KPD * EB;
        mbar_wait(&ready[o], (it >> 1) & 1);
        mbar_wait(&full[s], (it / NS) & 1);                  // already complete: makes the async-proxy writes visible here
        if (paired) bar_sync64(my_turn);                     // the pair's DMMA token
        // ---- contractions (eq (41)): D_r p, D_s p, D_t p, div of the contravariant velocity, LIFT_f g
        double cpr[2] = {0, 0}, cps[2] = {0, 0}, cpt[2] = {0, 0}, cvr[2] = {0, 0}, cvs[2] = {0, 0}, cvt[2] = {0, 0};
        double cl[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
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
                // half-way: let the partner start, so that the two DMMA streams overlap by about half (one warp
                // alone can issue a DMMA every ~24 cycles, the unit takes one every 16)
                if (s_ == KD / 2 && paired && !(w >= 4 && b + (int)gridDim.x >= nbatch)) bar_arrive64(partner_turn);
            }
            const double* gp = sG + t * EB + (g ^ swz(t));
#pragma unroll
            for (int s_ = 0; s_ < KL; ++s_)
#pragma unroll
                for (int f = 0; f < 4; ++f) dmma884v(cl[f], AL[f][s_], gp[f * LPAD + 4 * s_ * EB]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&opfree[o]);
        // ---- right-hand side and LSRK update (eq (41)-(43)) of node n, elements 2t, 2t+1 (dt folded into the record)
        if (n < Np) {
#pragma unroll
            for (int ee = 0; ee < 2; ++ee) {
                const int e = 2 * t + ee;
                if (e0 + e < K) {
                    const double* ge = bgeo + e * GS;
                    const double2 b01 = *reinterpret_cast<const double2*>(ge + 8), b12 = *reinterpret_cast<const double2*>(ge + 10),
                                  b34 = *reinterpret_cast<const double2*>(ge + 36), b56 = *reinterpret_cast<const double2*>(ge + 38),
                                  b78 = *reinterpret_cast<const double2*>(ge + 40),
                                  f01 = *reinterpret_cast<const double2*>(ge + 32), f23 = *reinterpret_cast<const double2*>(ge + 34);
                    const double a0 = cl[0][ee], a1 = cl[1][ee], a2 = cl[2][ee], a3 = cl[3][ee];
                    // the record carries every scale factor (GX3 above): the accumulators are -dt rho c^2 div u,
                    // D p and Z LIFT_f g; the reference normals (0,0,-1), (0,-1,0), (1,1,1), (-1,0,0) combine the lifts
                    const double yr = (cpr[ee] - a2) + a3;
                    const double ys = (cps[ee] - a2) + a1;
                    const double yt = (cpt[ee] - a2) + a0;
                    const double rp = (((((cvr[ee] + cvs[ee]) + cvt[ee]) - f01.x * a0) - f01.y * a1) - f23.x * a2) - f23.y * a3;
                    const double ru = b01.y * yr + b34.x * ys + b56.y * yt;       // Gb^T y: Gb[0], Gb[3], Gb[6]
                    const double rv = b12.x * yr + b34.y * ys + b78.x * yt;       //         Gb[1], Gb[4], Gb[7]
                    const double rw = b12.y * yr + b56.x * ys + b78.y * yt;       //         Gb[2], Gb[5], Gb[8]
                    const int eo = ws_eoff(e, QS) + n * 4;
                    double2 q0 = *reinterpret_cast<const double2*>(bq + eo);
                    double2 q1 = *reinterpret_cast<const double2*>(bq + eo + 2);
                    double2 r0 = *reinterpret_cast<const double2*>(br + eo);
                    double2 r1 = *reinterpret_cast<const double2*>(br + eo + 2);
                    r0.x = rka * r0.x + rp;  q0.x += rkb * r0.x;
                    r0.y = rka * r0.y + ru;  q0.y += rkb * r0.y;
                    r1.x = rka * r1.x + rv;  q1.x += rkb * r1.x;
                    r1.y = rka * r1.y + rw;  q1.y += rkb * r1.y;
                    const size_t off = ((size_t)(e0 + e) * Np + n) * 4;
                    __stcs(reinterpret_cast<double2*>(res + off), r0);
                    __stcs(reinterpret_cast<double2*>(res + off + 2), r1);
                    __stcs(reinterpret_cast<double2*>(qnew + off), q0);
                    __stcs(reinterpret_cast<double2*>(qnew + off + 2), q1);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }
}

}  // namespace dg
