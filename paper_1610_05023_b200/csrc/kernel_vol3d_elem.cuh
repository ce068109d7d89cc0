// 3D solver, fp32, N = 1, 2: fused volume + surface + update of one LSRK stage (Alg. 2,
// eq (41)-(43)) with ONE THREAD PER ELEMENT.  At these degrees an element is 4 or 10 nodes: a thread-per-node kernel
// spends its time in barriers and shared-memory exchanges for a contraction of 16 or 100 terms, and the tensor-core
// kernels have nothing to tile.  Here the whole element lives in the registers of its thread, every loop is unrolled,
// and the operators D_r, D_s, D_t, LIFT sit in constant memory: all lanes read the same entry at the same time, so an
// operator value is an instruction operand (FFMA with a constant-bank source), not a load.  The only dynamically
// indexed accesses (own face nodes, the neighbour's permuted face nodes) go through a thread-private column of
// shared memory and two small index tables.  Same flux (one scalar jump per face node), same
// per-tet record `geo3` and the same ghost / wall convention as k_vol3d (kernels.cuh).
#pragma once
#include "kernels.cuh"

namespace dg {

constexpr int ELEM_MAXN = 2;
constexpr int ELEM_OPS = 3 * 10 * 10 + 10 * 24;              // D[3][Np][Np] | LIFT[Np][4 Nfp] at N = 2
__constant__ float c_elem_ops[ELEM_MAXN][ELEM_OPS];

template <int N>
struct ElemCfg {
    static constexpr int Np = Deg<N>::Np, Nfp = Deg<N>::Nfp, Nfn = Deg<N>::Nfn;
    static constexpr int NT = 128;
    static constexpr size_t smem_bytes = sizeof(float) * 4 * Np * NT + sizeof(int) * (24 * Nfp + Nfn);
};

template <int N>
__global__ void __launch_bounds__(ElemCfg<N>::NT) k_vol3d_elem(Dev<float> d, int src, float rka, float rkb, float dt) {
    using C = ElemCfg<N>;
    constexpr int Np = C::Np, Nfp = C::Nfp, Nfn = C::Nfn, NT = C::NT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sX = reinterpret_cast<float*>(smem_raw);          // [4][Np][NT]: p, U^r, U^s, U^t of this thread's element
    int* sNb = reinterpret_cast<int*>(sX + 4 * Np * NT);     // [24][Nfp]: (neighbour face | perm << 2, j) -> neighbour node
    int* sFm = sNb + 24 * Nfp;                               // [4][Nfp] own face node
    const int tid = threadIdx.x;
    for (int i = tid; i < 24 * Nfp; i += NT) {
        const int fp = i / Nfp, j = i - fp * Nfp;
        sNb[i] = d.fmask3[(fp & 3) * Nfp + d.perm3[(fp >> 2) * Nfp + j]];
    }
    for (int i = tid; i < Nfn; i += NT) sFm[i] = d.fmask3[i];
    __syncthreads();
    const int k = blockIdx.x * NT + tid;
    if (k >= d.K) return;
    const float* __restrict__ cD = c_elem_ops[N - 1];
    const float* __restrict__ cL = c_elem_ops[N - 1] + 3 * Np * Np;
    const float4* __restrict__ qold = reinterpret_cast<const float4*>(d.q[src]);
    float4* __restrict__ qnew = reinterpret_cast<float4*>(d.q[src ^ 1]);
    float4* __restrict__ res = reinterpret_cast<float4*>(d.res);

    float g[GEO3];
    {
        const float4* gp = reinterpret_cast<const float4*>(d.geo3 + (size_t)k * GEO3);
#pragma unroll
        for (int i = 0; i < GEO3 / 4; ++i) { const float4 v = gp[i]; g[4 * i] = v.x; g[4 * i + 1] = v.y; g[4 * i + 2] = v.z; g[4 * i + 3] = v.w; }
    }
    // ---- own nodes; (p, contravariant velocity) to registers and to the thread-private shared column
    float4 q[Np];
    float Ur[Np], Us[Np], Ut[Np];
    float* mx = sX + tid;
#pragma unroll
    for (int n = 0; n < Np; ++n) {
        q[n] = qold[(size_t)k * Np + n];
        Ur[n] = g[0] * q[n].y + g[1] * q[n].z + g[2] * q[n].w;
        Us[n] = g[3] * q[n].y + g[4] * q[n].z + g[5] * q[n].w;
        Ut[n] = g[6] * q[n].y + g[7] * q[n].z + g[8] * q[n].w;
        mx[(0 * Np + n) * NT] = q[n].x; mx[(1 * Np + n) * NT] = Ur[n]; mx[(2 * Np + n) * NT] = Us[n]; mx[(3 * Np + n) * NT] = Ut[n];
    }
    // ---- volume (eq (41)): D_r p, D_s p, D_t p, div of the contravariant velocity
    float dpr[Np], dps[Np], dpt[Np], dvg[Np];
#pragma unroll
    for (int n = 0; n < Np; ++n) {
        float a = 0.f, b = 0.f, c = 0.f, e = 0.f;
#pragma unroll
        for (int m = 0; m < Np; ++m) {
            const float dr = cD[n * Np + m], ds = cD[Np * Np + n * Np + m], dtt = cD[2 * Np * Np + n * Np + m];
            a += dr * q[m].x; b += ds * q[m].x; c += dtt * q[m].x;
            e += dr * Ur[m]; e += ds * Us[m]; e += dtt * Ut[m];
        }
        dpr[n] = a; dps[n] = b; dpt[n] = c; dvg[n] = e;
    }
    // ---- surface: one flux jump per face node, g = A_f (Fs n).(u+ - u-) - B_f (p+ - p-)
    float gj[Nfn];
    const uint32_t finfo = d.finfo3[k];
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        const int nb = d.nbr3[k * 4 + f];
        const int* tab = sNb + ((finfo >> (8 * f)) & 0xffu) * Nfp;
        // Fs n_f = nhat_f . G  (nhat: 0:(0,0,-1) 1:(0,-1,0) 2:(1,1,1) 3:(-1,0,0)); Fs n.u^- = nhat . U^-
        float nx, ny, nz;
        if (f == 0) { nx = -g[6]; ny = -g[7]; nz = -g[8]; }
        else if (f == 1) { nx = -g[3]; ny = -g[4]; nz = -g[5]; }
        else if (f == 2) { nx = g[0] + g[3] + g[6]; ny = g[1] + g[4] + g[7]; nz = g[2] + g[5] + g[8]; }
        else { nx = -g[0]; ny = -g[1]; nz = -g[2]; }
#pragma unroll
        for (int j = 0; j < Nfp; ++j) {
            const int nm = sFm[f * Nfp + j];
            const float pM = mx[nm * NT], ur = mx[(Np + nm) * NT], us = mx[(2 * Np + nm) * NT], ut = mx[(3 * Np + nm) * NT];
            const float unM = (f == 0) ? -ut : (f == 1) ? -us : (f == 2) ? (ur + us + ut) : -ur;
            float pP, unP;
            if (nb >= 0) {
                const float4 x = qold[(size_t)nb * Np + tab[j]];
                pP = x.x;
                unP = nx * x.y + ny * x.z + nz * x.w;
            } else {
                pP = 2.f * d.qb3[(size_t)(-1 - nb) * Nfp + j];          // ghost state: p+ = 2 r^-, u+ = 0 (zero row: walls)
                unP = 0.f;
            }
            gj[f * Nfp + j] = g[9 + f] * (unP - unM) - g[13 + f] * (pP - pM);
        }
    }
    // ---- LIFT, right-hand side and LSRK update (eq (41)-(43))
    const float rc2 = g[21], irho = g[22], cc = g[23];
#pragma unroll
    for (int n = 0; n < Np; ++n) {
        float a[4];
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            float s = 0.f;
#pragma unroll
            for (int j = 0; j < Nfp; ++j) s += cL[n * Nfn + f * Nfp + j] * gj[f * Nfp + j];
            a[f] = s;
        }
        const float lp = g[17] * a[0] + g[18] * a[1] + g[19] * a[2] + g[20] * a[3];
        const float xr = cc * (a[2] - a[3]) - irho * dpr[n];
        const float xs = cc * (a[2] - a[1]) - irho * dps[n];
        const float xt = cc * (a[2] - a[0]) - irho * dpt[n];
        const float rp = -rc2 * (dvg[n] + lp);
        const float ru = g[0] * xr + g[3] * xs + g[6] * xt;
        const float rv = g[1] * xr + g[4] * xs + g[7] * xt;
        const float rw = g[2] * xr + g[5] * xs + g[8] * xt;
        float4 r = res[(size_t)k * Np + n];
        r.x = rka * r.x + dt * rp; r.y = rka * r.y + dt * ru; r.z = rka * r.z + dt * rv; r.w = rka * r.w + dt * rw;
        float4 o = q[n];
        o.x += rkb * r.x; o.y += rkb * r.y; o.z += rkb * r.z; o.w += rkb * r.w;
        res[(size_t)k * Np + n] = r;
        qnew[(size_t)k * Np + n] = o;
    }
}

}  // namespace dg
