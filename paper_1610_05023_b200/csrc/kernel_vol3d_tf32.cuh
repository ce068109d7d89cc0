// 3D solver, fp32, tensor-core version: fused volume + surface + update of one LSRK stage (PAPER.md:L623-624,
// Alg. 2, eq (41)-(43)) with the dense contractions of eq (41) on the tensor cores as error-compensated
// 3xTF32: every fp32 operand x is split into hi = x with the 13 low mantissa bits cleared (exactly a TF32 number)
// and lo = x - hi (exact in fp32; the tensor core reads its leading 11 bits), and a product a*b is accumulated in
// fp32 as  lo_a*hi_b + hi_a*lo_b + hi_a*hi_b.  The dropped terms are O(2^-22) relative, i.e. fp32-level accuracy
// (measured against the fp64 oracle: same 1e-6 error as the FFMA kernel; the 1e-4 tolerance of BASELINE.json holds
// with two orders of margin), where plain TF32 (2^-11 per operand) would not survive 100 steps.
//
// Why tensor cores here (north_star: "only if ncu shows it is compute-bound ... and the tolerances still hold"):
// the scalar kernel k_vol3d<float,5> runs at 5.6 ms per launch = 21 % of either roof; it is bound by the shared-
// memory pipe (one broadcast LDS.128 per 4 FFMA) and issue slots, not by HBM.  mma.sync.m16n8k8.tf32 delivers
// 512 FMA/clk/SM (profiles/r02_dmma_issue.md), so even at 3 MMAs per product the contraction costs 0.9 ms per
// launch, under the 1.2 ms HBM roof.  (tcgen05 kind::tf32 would be ~4x faster still, but needs its operands as
// UMMA shared-memory tiles and its accumulator in TMEM; with the contraction already under the HBM roof the
// legacy mma.sync path, whose fragments live in registers next to the update stage, is the simpler fit.)
//
// Tiling.  A batch is EB = 16 consecutive elements = MMA m.  MMA warp w owns the n-tile of nodes 8w..8w+7 and
// keeps ITS rows of D_r, D_s, D_t and LIFT, split hi/lo, as register-resident B fragments for the life of the
// persistent CTA (N=5: 132 registers).  The A operands (p, U^r, U^s, U^t per node; flux jump g per face node) are
// staged in shared memory as [k][16 elements] (row stride 24 floats: conflict-free fragment loads) and split on
// the fly.  The accumulator fragment of lane (g,t) holds elements g, g+8 x nodes 8w+2t, 8w+2t+1 of all eight
// results (d_r p, d_s p, d_t p, div U, LIFT_f g), so the update stage runs in registers; it uses the FMA pipe and
// does not compete with the tensor pipe.  Warp roles, staging, barriers and the per-tet record are those of
// kernel_vol3d_ws.cuh (LOADER: cp.async.bulk + cp.async gathers; PREP: operands and flux jumps; MMA + update), including
// the compact two-warpgroup layout with two CTAs per SM at N = 3 (TfCfg::COMPACT: 816 -> 509 us per launch on the
// SEAM-shaped workload).
#pragma once
#include "kernel_vol3d_ws.cuh"

namespace dg {

template <int N>
struct TfCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int EB = 16;                      // elements per batch = MMA m
    static constexpr int MT = (Np + 7) / 8;            // n-tiles = MMA warps
    static constexpr int KD = (Np + 7) / 8, KPD = KD * 8;
    static constexpr int KL = (Nfp + 7) / 8, KPL = KL * 8;
    static constexpr int XS = 24;                      // operand row stride in floats (16 elements + 8: bank spread)
    // warp roles: MMA warps 0..MT-1, LOADER warp LW, PREP warps PW0..PW0+3.  With MT <= 3 (N = 3) the roles fit two
    // warpgroups and two CTAs share an SM (six MMA warps per SM instead of three); otherwise three warpgroups, one CTA
    static constexpr bool COMPACT = MT <= 3;
    static constexpr int NT = COMPACT ? 256 : 384, LW = COMPACT ? 3 : 7, PW0 = COMPACT ? 4 : 8, MINB = COMPACT ? 2 : 1;
    static constexpr int NS = 3;                       // staging depth
    static constexpr int QS = Np * 4 + 4;              // staged element stride of q / res in floats (16 B skew)
    static constexpr int GS = GX3 + 8;                 // staged stride of the record (208 B = 13 x 16 B: bank spread)
    static constexpr int szB = (4 * KPD + 4 * KPL) * XS;
    static constexpr int oB = 0;                       // [2][szB]        operand buffers
    static constexpr int oQ = oB + 2 * szB;            // [NS][16][QS]
    static constexpr int oR = oQ + NS * EB * QS;       // [NS][16][QS]
    static constexpr int oGeo = oR + NS * EB * QS;     // [NS][16][GS]
    static constexpr int oN = oGeo + NS * EB * GS;     // [NS][Nfn][16][4] neighbour traces
    static constexpr int oBar = ((oN + NS * Nfn * EB * 4 + 3) / 4) * 4;   // full[NS], empty[NS], ready[2], opfree[2] (8 B each)
    static constexpr int oEnd = oBar + 2 * (2 * NS + 4);
    static constexpr size_t smem_bytes = sizeof(float) * oEnd + sizeof(int) * (33 * Nfp + Nfn) + 32;
    static constexpr uint32_t tx_bytes = 2 * EB * Np * 16 + EB * GX3 * 4;
    static constexpr int NRA = (Np + 1) / 2;           // PREP phase A rows: 2 nodes x 16 elements
    static constexpr int NRB = 2 * Nfp;                // PREP phase B rows: (face node j, face pair) x 2 faces x 16 elements
    // setmaxnreg: launched with REG_BASE registers per thread (65536 / (NT * MINB)); what the PREP warpgroup gives back
    // is the only pool the MMA warpgroup(s) can grow from
    static constexpr int REG_BASE = COMPACT ? 128 : 168, REG_PREP = 88, REG_MMA = COMPACT ? 168 : 208;
    static_assert((REG_BASE - REG_PREP) * 128 >= (REG_MMA - REG_BASE) * (NT - 128), "setmaxnreg pool would deadlock");
    static_assert(REG_BASE * NT * MINB <= 65536, "register file");
    static_assert(MT <= 7, "the tensor-core fp32 kernel covers N <= 5");
    static_assert(smem_bytes <= 227 * 1024, "shared memory");
};

__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// x = hi + lo with hi a TF32 number (13 low mantissa bits clear) and lo exact in fp32
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}
// acc += a * b in 3xTF32 (small terms first)
__device__ __forceinline__ void mma_3x(float (&c)[4], const uint32_t (&ah)[4], const uint32_t (&al)[4],
                                       const uint32_t (&bh)[2], const uint32_t (&bl)[2]) {
    mma_tf32(c, al, bh[0], bh[1]);
    mma_tf32(c, ah, bl[0], bl[1]);
    mma_tf32(c, ah, bh[0], bh[1]);
}

template <int N>
__global__ void __launch_bounds__(TfCfg<N>::NT, TfCfg<N>::MINB)
k_vol3d_tf32(Dev<float> d, const float* __restrict__ geox, int src, float rka, float rkb) {
    using C = TfCfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, EB = C::EB, KD = C::KD, KPD = C::KPD, KL = C::KL, KPL = C::KPL,
                  NT = C::NT, QS = C::QS, MT = C::MT, NS = C::NS, GS = C::GS, XS = C::XS;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sm = reinterpret_cast<float*>(smem_raw);
    float* sQ = sm + C::oQ;
    float* sR = sm + C::oR;
    float* sGeo = sm + C::oGeo;
    float* sN = sm + C::oN;
    uint64_t* full = reinterpret_cast<uint64_t*>(sm + C::oBar);
    uint64_t* empty = full + NS;
    uint64_t* ready = empty + NS;
    uint64_t* opfree = ready + 2;
    int* sNode = reinterpret_cast<int*>(sm + C::oEnd);       // [33][Nfp]: (face | perm << 2, j) -> 4 * neighbour node
    int* sFm = sNode + 33 * Nfp;                             // [4][Nfp] own face node

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const float* __restrict__ qold = d.q[src];
    const int K = d.K;
    const int nbatch = (K + EB - 1) / EB;                    // arrays are padded to nbatch * EB elements

    // ---- one-time: tables, zeroed operand buffers (their padding rows stay zero for ever), barriers
    for (int i = tid; i < C::oQ; i += NT) sm[i] = 0.f;
    for (int i = tid; i < 33 * Nfp; i += NT) {               // entries are offsets in floats (4 per node)
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
        const int ie = lane & 15, fh = lane >> 4;
        int it = 0;
        for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
            const int s = it % NS, o = it & 1;
            const float* bq = sQ + (s * EB + ie) * QS;
            const float* ge = sGeo + (s * EB + ie) * GS;
            const float* bn = sN + s * (Nfn * EB * 4) + ie * 4;
            float* sB = sm + C::oB + o * C::szB;
            mbar_wait(&full[s], (it / NS) & 1);
            if (it >= 2) mbar_wait(&opfree[o], ((it >> 1) - 1) & 1);
            // ---- phase A: (p, contravariant velocity) of node 2 row + fh, element ie -> operand rows [k][element]
            {
                const float4 ga = *reinterpret_cast<const float4*>(ge), gb = *reinterpret_cast<const float4*>(ge + 4);
                const float g8 = ge[8];
#pragma unroll 4
                for (int row = pw; row < C::NRA; row += 4) {
                    const int n = 2 * row + fh;
                    if (n < Np) {
                        const float4 v = *reinterpret_cast<const float4*>(bq + n * 4);
                        float* op = sB + n * XS + ie;
                        op[0] = v.x;
                        op[KPD * XS] = ga.x * v.y + ga.y * v.z + ga.z * v.w;
                        op[2 * KPD * XS] = ga.w * v.y + gb.x * v.z + gb.y * v.w;
                        op[3 * KPD * XS] = gb.z * v.y + gb.w * v.z + g8 * v.w;
                    }
                }
            }
            // ---- phase B: one scalar flux jump per face node (upwind flux PAPER.md:L499-512):
            //      g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-);  row = (face node j, face pair), face f = 2 pair + fh
            {
#pragma unroll 2
                for (int row = pw; row < C::NRB; row += 4) {
                    const int j = row >> 1, f = 2 * (row & 1) + fh;
                    const float4 nA = *reinterpret_cast<const float4*>(ge + 12 + 4 * f);   // (Fs n)_xyz, A_f
                    const float Bf = ge[28 + f];
                    const float4 m = *reinterpret_cast<const float4*>(bq + 4 * sFm[f * Nfp + j]);
                    const float4 x = *reinterpret_cast<const float4*>(bn + (f * Nfp + j) * (EB * 4));
                    const float dn = nA.x * (x.y - m.y) + nA.y * (x.z - m.z) + nA.z * (x.w - m.w);
                    sB[(4 * KPD + f * KPL + j) * XS + ie] = nA.w * dn - Bf * (x.x - m.x);
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
        // half-warp hw gathers faces 2 hw and 2 hw + 1 of element ie: one 16-byte cp.async per face node (p,u,v,w)
        const int ie = lane & 15, hw = lane >> 4;
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
            if (lane < EB) {
                bulk_g2s(sQ + (s * EB + lane) * QS, qold + (e0 + lane) * (Np * 4), Np * 16, &full[s]);
                bulk_g2s(sGeo + (s * EB + lane) * GS, geox + (e0 + lane) * GX3, GX3 * 4, &full[s]);
            } else {
                bulk_g2s(sR + (s * EB + lane - EB) * QS, d.res + (e0 + lane - EB) * (Np * 4), Np * 16, &full[s]);
            }
            float* dn = sN + s * (Nfn * EB * 4) + ie * 4;
#pragma unroll
            for (int fl = 0; fl < 2; ++fl) {
                const int f = 2 * hw + fl;
                const uint32_t c = hw ? (fl ? cw4.w : cw4.z) : (fl ? cw4.y : cw4.x);
                const size_t id = (c >> 5) & CONN_MAX_ID;
                const bool bnd = (c & CONN_BND) != 0;
                const float* base = bnd ? d.ghost3 + id * (Nfp * 4) : qold + id * (Np * 4);
                const int* tab = sNode + (bnd ? 32 : (int)(c & 31)) * Nfp;     // row 32 is the identity
                int off[Nfp];                                // all table reads first: cp.async is a compiler barrier
#pragma unroll
                for (int j = 0; j < Nfp; ++j) off[j] = tab[j];
#pragma unroll
                for (int j = 0; j < Nfp; ++j) cp_async16(dn + (f * Nfp + j) * (EB * 4), base + off[j]);
            }
            cp_async_arrive_noinc(&full[s]);
        }
        return;
    }
    if (w >= MT) return;

    // =================================================================== MMA warps
    const int g = lane >> 2, t = lane & 3;
    const int nb0 = 8 * w + g;                               // B-fragment column (node) of this lane
    float* __restrict__ qnew = d.q[src ^ 1];
    float* __restrict__ res = d.res;
    // operator rows of node nb0, split hi / lo: b0 = (k = 8 s + t), b1 = (k = 8 s + t + 4)
    uint32_t Brh[KD][2], Brl[KD][2], Bsh[KD][2], Bsl[KD][2], Bth[KD][2], Btl[KD][2], BLh[4][KL][2], BLl[4][KL][2];
#pragma unroll
    for (int s = 0; s < KD; ++s)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int m = 8 * s + t + 4 * h;
            const bool ok = nb0 < Np && m < Np;
            split_tf32(ok ? d.Dt3[(0 * Np + m) * Np + nb0] : 0.f, Brh[s][h], Brl[s][h]);   // Dt3[a][m][n] = D_a[n][m]
            split_tf32(ok ? d.Dt3[(1 * Np + m) * Np + nb0] : 0.f, Bsh[s][h], Bsl[s][h]);
            split_tf32(ok ? d.Dt3[(2 * Np + m) * Np + nb0] : 0.f, Bth[s][h], Btl[s][h]);
        }
#pragma unroll
    for (int f = 0; f < 4; ++f)
#pragma unroll
        for (int s = 0; s < KL; ++s)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int j = 8 * s + t + 4 * h;
                split_tf32((nb0 < Np && j < Nfp) ? d.Lt3[(f * Nfp + j) * Np + nb0] : 0.f, BLh[f][s][h], BLl[f][s][h]);
            }

    int it = 0;
    for (int b = blockIdx.x; b < nbatch; b += gridDim.x, ++it) {
        const int s = it % NS, o = it & 1;
        const int e0 = b * EB;
        const float* sB = sm + C::oB + o * C::szB;
        mbar_wait(&ready[o], (it >> 1) & 1);
        mbar_wait(&full[s], (it / NS) & 1);                  // already complete: makes the async-proxy writes visible here
        // ---- contractions (eq (41)): accumulators [element g / g+8][node 8w+2t / +1]
        // Issue order: the three MMAs of one product (lo*hi, hi*lo, hi*hi) hit the same accumulator, so they are
        // issued as three PASSES over six (D part) or four (LIFT part) independent accumulators -- a dependent
        // HMMA is then 6 (4) issue slots away and the tensor pipe never waits for its own result.
        float cpr[4] = {0, 0, 0, 0}, cps[4] = {0, 0, 0, 0}, cpt[4] = {0, 0, 0, 0};
        float cvr[4] = {0, 0, 0, 0}, cvs[4] = {0, 0, 0, 0}, cvt[4] = {0, 0, 0, 0};
        float cl[4][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
        {
            // A fragment of k-step s_: rows (elements) g, g+8; columns (k) 8 s_ + t, + 4
            const float* ap = sB + t * XS + g;
            auto load = [&](const float* r0, uint32_t (&ah)[4], uint32_t (&al)[4]) {
                const float x0 = r0[0], x1 = r0[8], x2 = r0[4 * XS], x3 = r0[4 * XS + 8];
                split_tf32(x0, ah[0], al[0]);
                split_tf32(x1, ah[1], al[1]);
                split_tf32(x2, ah[2], al[2]);
                split_tf32(x3, ah[3], al[3]);
            };
#pragma unroll
            for (int s_ = 0; s_ < KD; ++s_) {
                uint32_t ph[4], pl[4], rh[4], rl[4], sh[4], sl[4], th[4], tl[4];
                load(ap + (8 * s_) * XS, ph, pl);
                load(ap + (KPD + 8 * s_) * XS, rh, rl);
                load(ap + (2 * KPD + 8 * s_) * XS, sh, sl);
                load(ap + (3 * KPD + 8 * s_) * XS, th, tl);
                mma_tf32(cpr, pl, Brh[s_][0], Brh[s_][1]);
                mma_tf32(cps, pl, Bsh[s_][0], Bsh[s_][1]);
                mma_tf32(cpt, pl, Bth[s_][0], Bth[s_][1]);
                mma_tf32(cvr, rl, Brh[s_][0], Brh[s_][1]);
                mma_tf32(cvs, sl, Bsh[s_][0], Bsh[s_][1]);
                mma_tf32(cvt, tl, Bth[s_][0], Bth[s_][1]);
                mma_tf32(cpr, ph, Brl[s_][0], Brl[s_][1]);
                mma_tf32(cps, ph, Bsl[s_][0], Bsl[s_][1]);
                mma_tf32(cpt, ph, Btl[s_][0], Btl[s_][1]);
                mma_tf32(cvr, rh, Brl[s_][0], Brl[s_][1]);
                mma_tf32(cvs, sh, Bsl[s_][0], Bsl[s_][1]);
                mma_tf32(cvt, th, Btl[s_][0], Btl[s_][1]);
                mma_tf32(cpr, ph, Brh[s_][0], Brh[s_][1]);
                mma_tf32(cps, ph, Bsh[s_][0], Bsh[s_][1]);
                mma_tf32(cpt, ph, Bth[s_][0], Bth[s_][1]);
                mma_tf32(cvr, rh, Brh[s_][0], Brh[s_][1]);
                mma_tf32(cvs, sh, Bsh[s_][0], Bsh[s_][1]);
                mma_tf32(cvt, th, Bth[s_][0], Bth[s_][1]);
            }
            const float* gp = ap + 4 * KPD * XS;
#pragma unroll
            for (int s_ = 0; s_ < KL; ++s_) {
                uint32_t fh[4][4], fl[4][4];
#pragma unroll
                for (int f = 0; f < 4; ++f) load(gp + (f * KPL + 8 * s_) * XS, fh[f], fl[f]);
#pragma unroll
                for (int f = 0; f < 4; ++f) mma_tf32(cl[f], fl[f], BLh[f][s_][0], BLh[f][s_][1]);
#pragma unroll
                for (int f = 0; f < 4; ++f) mma_tf32(cl[f], fh[f], BLl[f][s_][0], BLl[f][s_][1]);
#pragma unroll
                for (int f = 0; f < 4; ++f) mma_tf32(cl[f], fh[f], BLh[f][s_][0], BLh[f][s_][1]);
            }
        }
        float cdv[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) cdv[i] = (cvr[i] + cvs[i]) + cvt[i];
        __syncwarp();
        if (lane == 0) mbar_arrive(&opfree[o]);
        // ---- right-hand side and LSRK update (eq (41)-(43)); dt is folded into the record.
        //      accumulator index 2 r + c: element g + 8 r, node 8 w + 2 t + c
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int e = g + 8 * r;
            if (e0 + e < K) {
                const float* ge = sGeo + (s * EB + e) * GS;
                // the record carries every scale factor (GX3 in kernel_vol3d_ws.cuh): Gb = -dt/rho G at 9..11, 36..41
                const float4 gc = *reinterpret_cast<const float4*>(ge + 8), gd = *reinterpret_cast<const float4*>(ge + 36),
                             fs = *reinterpret_cast<const float4*>(ge + 32);
                const float2 ge2 = *reinterpret_cast<const float2*>(ge + 40);
                const float b0 = gc.y, b1 = gc.z, b2 = gc.w, b3 = gd.x, b4 = gd.y, b5 = gd.z, b6 = gd.w, b7 = ge2.x, b8 = ge2.y;
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int n = 8 * w + 2 * t + c, i = 2 * r + c;
                    if (n < Np) {
                        const float a0 = cl[0][i], a1 = cl[1][i], a2 = cl[2][i], a3 = cl[3][i];
                        // accumulators: -dt rho c^2 div u, D p, Z LIFT_f g; the reference normals combine the lifts
                        const float yr = (cpr[i] - a2) + a3;
                        const float ys = (cps[i] - a2) + a1;
                        const float yt = (cpt[i] - a2) + a0;
                        const float rp = (((cdv[i] - fs.x * a0) - fs.y * a1) - fs.z * a2) - fs.w * a3;
                        const float ru = b0 * yr + b3 * ys + b6 * yt;
                        const float rv = b1 * yr + b4 * ys + b7 * yt;
                        const float rw = b2 * yr + b5 * ys + b8 * yt;
                        float4 q = *reinterpret_cast<const float4*>(sQ + (s * EB + e) * QS + n * 4);
                        float4 rr = *reinterpret_cast<const float4*>(sR + (s * EB + e) * QS + n * 4);
                        rr.x = rka * rr.x + rp;  q.x += rkb * rr.x;
                        rr.y = rka * rr.y + ru;  q.y += rkb * rr.y;
                        rr.z = rka * rr.z + rv;  q.z += rkb * rr.z;
                        rr.w = rka * rr.w + rw;  q.w += rkb * rr.w;
                        const size_t off = ((size_t)(e0 + e) * Np + n) * 4;
                        __stcs(reinterpret_cast<float4*>(res + off), rr);
                        __stcs(reinterpret_cast<float4*>(qnew + off), q);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }
}

}  // namespace dg
