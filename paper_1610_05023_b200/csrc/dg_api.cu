// C ABI of the DG + HABC time stepper (include/dg_habc.h): host setup, device upload, stage sequencing.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <set>
#include <stdexcept>
#include <type_traits>
#include <string>
#include <vector>

#include "../../include/dg_habc.h"
#include "habc_coef.hpp"
#include "kernels.cuh"
#include "kernels_aux.cuh"
#include "kernel_face2d.cuh"
#include "kernel_vol3d_mma.cuh"
#include "kernel_vol3d_ws.cuh"
#include "kernel_vol3d_tf32.cuh"
#include "kernel_vol3d_mmag.cuh"
#include "kernel_vol3d_tf32g.cuh"
#include "kernel_vol3d_elem.cuh"
#include "mesh.hpp"

namespace {

thread_local std::string g_err;

int set_err(int code, const std::string& msg) { g_err = msg; return code; }

int err_from_exception(const std::exception& e) {
    std::string m = e.what();
    if (m.rfind("EMESH", 0) == 0) return set_err(DG_EMESH, m);
    if (m.rfind("ECUDA", 0) == 0) return set_err(DG_ECUDA, m);
    if (m.rfind("ENOMEM", 0) == 0) return set_err(DG_ENOMEM, m);
    return set_err(DG_EINVAL, m);
}

void cu(cudaError_t e, const char* what) {
    if (e != cudaSuccess) throw std::runtime_error(std::string("ECUDA: ") + what + ": " + cudaGetErrorString(e));
}

// LSRK4(5) of Carpenter & Kennedy (ref. [10] of the paper; eq (42)-(43))
const double RKA[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                       -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
const double RKC[5] = {0.0, 1432997174477.0 / 9575080441755.0, 2526269341429.0 / 6820363962896.0,
                       2006345519317.0 / 3224310063776.0, 2802321613138.0 / 2924317926251.0};
const double RKB[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                       1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                       2277821191437.0 / 14882151754819.0};

struct Arena {
    char* base = nullptr;
    size_t size = 0, used = 0;
    bool dry = true;
    void* take(size_t bytes) {
        size_t o = (used + 255) & ~size_t(255);
        used = o + bytes;
        if (dry) return nullptr;
        if (used > size) throw std::runtime_error("ENOMEM: workspace too small");
        return base + o;
    }
};

}  // namespace

struct dg_solver {
    dg::HostMesh m;
    dg::HabcCoef hc;
    int N = 0, J = 0, precision = 64, device = 0;
    double dt = 0;
    cudaStream_t stream = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    bool own_ws = false;
    dg::Dev<double> d64{};
    dg::Dev<float> d32{};
    int cur = 0;
    int grid3 = 0;
    int face_grid = 1;              // persistent CTAs of the 2D solver kernel (from the occupancy calculator, dg_create)
    size_t smem3 = 0;
    int kern3 = 0;                  // the 3D kernel in use (enum Kern3, resolved from dg_options.kernel in dg_create)
    const void* geox3 = nullptr;    // [Kp][GX3] per-tet record of the warp-specialised kernels (dt folded in), fp64 or fp32
    bool use_graph = true;
    cudaGraphExec_t graph[2] = {nullptr, nullptr};
    std::vector<double> rho, c;
    // point source (dg_set_source): cell, Ricker parameters, device copies of the weights and of the simulated time
    bool src_on = false;
    int src_k = 0;
    double src_f = 0, src_ts = 0, src_amp = 0;
    void* src_w = nullptr;          // [Np] of T
    double* t_dev = nullptr;        // simulated time at the start of the current step (advanced by k_source while a source is on)
    double t_host = 0;              // the same clock kept on the host (dg_step adds dt per step), so that a source
                                    // switched on after some steps starts at the right time
    bool time_kernels = false;      // dg_options.time_kernels: events around the 3D kernel of every stage
    cudaEvent_t evk[2][5][2] = {};  // [parity of the step's first buffer][stage][before, after]
    int last_par = -1;              // parity of the last enqueued step (-1: none yet)
    double* export_buf = nullptr;   // device scratch for dg_get_fields (aux fields, fp64)
    size_t export_elems = 0;
};

namespace {

using namespace dg;

// The 3D kernels.  The values are dg_options.kernel (include/dg_habc.h); KERNELS says what each one covers and
// DEFAULT_KERNEL which one runs when the caller asks for 0.
enum Kern3 : int { K3_AUTO = 0, K3_SCALAR = 1, K3_MMA = 2, K3_WS = 3, K3_TF32 = 4, K3_TPG = 5, K3_ELEM = 6, K3_COUNT };

struct KernRow { int precision /* 0: both */, nmin, nmax; bool geox /* reads the extended per-tet record */; const char* what; };
const KernRow KERNELS[K3_COUNT] = {
    {0, 1, 8, false, "auto"},
    {0, 1, 8, false, "scalar-FMA kernel (kernel = 1): fp64/fp32, N = 1..8"},
    {64, 1, 5, false, "fp64 tensor-pipe kernel (kernel = 2): fp64, N = 1..5"},
    {64, 1, 5, true, "warp-specialised fp64 tensor-pipe kernel (kernel = 3): fp64, N = 1..5"},
    {32, 3, 5, true, "fp32 3xTF32 tensor-core kernel (kernel = 4): fp32, N = 3..5"},
    {0, 6, 8, false, "tensor-pipe kernels with operators read through L1/L2 (kernel = 5): N = 6..8"},
    {32, 1, 2, false, "thread-per-element fp32 kernel (kernel = 6): fp32, N = 1, 2"},
};
//                                    N =      1          2          3        4        5      6       7       8
const int DEFAULT_KERNEL_F64[9] = {0, K3_MMA,    K3_MMA,    K3_WS,   K3_MMA,  K3_WS,   K3_TPG, K3_TPG, K3_TPG};
const int DEFAULT_KERNEL_F32[9] = {0, K3_ELEM,   K3_ELEM,   K3_TF32, K3_TF32, K3_TF32, K3_TPG, K3_TPG, K3_TPG};

int resolve_kernel(int requested, int precision, int N) {
    if (requested < 0 || requested >= K3_COUNT) throw std::runtime_error("EINVAL: dg_options.kernel must be 0..6");
    const int k = requested != K3_AUTO ? requested : (precision == 64 ? DEFAULT_KERNEL_F64 : DEFAULT_KERNEL_F32)[N];
    const KernRow& r = KERNELS[k];
    if ((r.precision && r.precision != precision) || N < r.nmin || N > r.nmax)
        throw std::runtime_error(std::string("EINVAL: the ") + r.what + " does not cover this (precision, N)");
    return k;
}

// ---------------------------------------------------------------- device image of the problem
template <typename T>
struct Uploader {
    Arena& A;
    cudaStream_t st;
    template <typename S>
    const T* real(const std::vector<S>& h, size_t n) {
        T* p = (T*)A.take(sizeof(T) * std::max<size_t>(n, 1));
        if (!A.dry && h.size() != n) throw std::runtime_error("EINVAL: internal size mismatch");
        if (!A.dry && !h.empty()) {
            std::vector<T> t(h.begin(), h.end());
            cu(cudaMemcpy(p, t.data(), sizeof(T) * t.size(), cudaMemcpyHostToDevice), "upload");
        }
        return p;
    }
    template <typename I, typename S>
    const I* ints(const std::vector<S>& h, size_t n) {
        I* p = (I*)A.take(sizeof(I) * std::max<size_t>(n, 1));
        if (!A.dry && h.size() != n) throw std::runtime_error("EINVAL: internal size mismatch");
        if (!A.dry && !h.empty()) {
            std::vector<I> t(h.begin(), h.end());
            cu(cudaMemcpy(p, t.data(), sizeof(I) * t.size(), cudaMemcpyHostToDevice), "upload");
        }
        return p;
    }
    T* zeros(size_t n) {
        T* p = (T*)A.take(sizeof(T) * std::max<size_t>(n, 1));
        if (!A.dry) cu(cudaMemset(p, 0, sizeof(T) * std::max<size_t>(n, 1)), "memset");
        return p;
    }
};

// Sizes only (dry run) or the real upload.  `s` must hold the host mesh, coefficients, rho, c.
template <typename T>
void build_device(dg_solver* s, Arena& A, Dev<T>& d) {
    const HostMesh& m = s->m;
    const int K = m.K, Tn = s->J > 0 ? m.T : 0, E = s->J > 0 ? m.E : 0, C = s->J > 0 ? m.C : 0;
    const int Np = m.Np, Nfp = m.Nfp, N1 = m.N1, J = s->J;
    Uploader<T> U{A, s->stream};
    d.N = m.N; d.J = J; d.K = K; d.Tn = Tn; d.E = E; d.C = C; d.Np = Np; d.Nfp = Nfp; d.N1 = N1;
    d.invM = T(1.0 / (2 * J + 1));
    // ---- 3D state
    const size_t Kp = ((size_t)K + 15) / 16 * 16;  // the tensor-pipe kernels read whole batches of 8 (fp64) / 16 (fp32) elements
    const size_t n3 = Kp * Np * 4;
    d.q[0] = U.zeros(n3); d.q[1] = U.zeros(n3); d.res = U.zeros(n3);
    std::vector<double> geo, dt3, lt3;
    std::vector<int> fm3;
    std::vector<uint32_t> finfo, conn;
    if (!A.dry) {
        geo.assign(Kp * GEO3, 0.0);
        finfo.assign(K, 0);
        conn.assign(Kp * 4, 0);
        for (int k = 0; k < K; ++k) {
            double* g = &geo[(size_t)k * GEO3];
            for (int q = 0; q < 9; ++q) g[q] = m.G3[(size_t)k * 9 + q];
            const double Zm = s->rho[k] * s->c[k];
            for (int f = 0; f < 4; ++f) {
                const int nb = m.nbr3[(size_t)k * 4 + f];
                const double Zp = nb >= 0 ? s->rho[nb] * s->c[nb] : Zm;
                const double Fs = m.Fs3[(size_t)k * 4 + f];
                g[9 + f] = Zp / ((Zp + Zm) * Fs);
                g[13 + f] = 1.0 / (Zp + Zm);
                g[17 + f] = Fs;
                // wall faces: the "neighbour" is the all-zero ghost row, so (u+ - u-, p+ - p-) = -(u-, p-); doubling
                // one flux weight and dropping the other gives the mirror states p+ = -p- (p = 0)
                // resp. n.u+ = -n.u- (rigid wall) through the same branch-free flux code
                if (m.bc3[(size_t)k * 4 + f] == 1) { g[9 + f] = 0.0; g[13 + f] *= 2.0; }
                else if (m.bc3[(size_t)k * 4 + f] == 2) { g[9 + f] *= 2.0; g[13 + f] = 0.0; }
                const uint32_t fp = (uint32_t)(m.nbrface3[(size_t)k * 4 + f] | (m.nbrperm3[(size_t)k * 4 + f] << 2));
                finfo[k] |= fp << (8 * f);
                conn[(size_t)k * 4 + f] = nb >= 0 ? ((uint32_t)nb << 5) | fp : CONN_BND | ((uint32_t)(-1 - nb) << 5);
            }
            g[21] = s->rho[k] * s->c[k] * s->c[k];
            g[22] = 1.0 / s->rho[k];
            g[23] = s->c[k];
        }
        dt3.resize((size_t)3 * Np * Np);
        for (int a = 0; a < 3; ++a)
            for (int n = 0; n < Np; ++n)
                for (int q = 0; q < Np; ++q) dt3[((size_t)a * Np + q) * Np + n] = m.r3.D[a][(size_t)n * Np + q];
        lt3.resize((size_t)4 * Nfp * Np);
        for (int n = 0; n < Np; ++n)
            for (int j = 0; j < 4 * Nfp; ++j) lt3[(size_t)j * Np + n] = m.r3.LIFT[(size_t)n * 4 * Nfp + j];
        fm3.assign(m.r3.Fmask.begin(), m.r3.Fmask.end());
    }
    if (!A.dry && m.N <= ELEM_MAXN && std::is_same<T, float>::value) {
        // k_vol3d_elem reads its operators from constant memory: D[3][Np][Np] | LIFT[Np][4 Nfp], one slot per degree
        // (the values depend on N only, so solvers of the same degree write the same bytes)
        std::vector<float> ops((size_t)3 * Np * Np + (size_t)Np * 4 * Nfp);
        for (int a = 0; a < 3; ++a)
            for (size_t i = 0; i < (size_t)Np * Np; ++i) ops[(size_t)a * Np * Np + i] = (float)m.r3.D[a][i];
        for (size_t i = 0; i < (size_t)Np * 4 * Nfp; ++i) ops[(size_t)3 * Np * Np + i] = (float)m.r3.LIFT[i];
        cu(cudaMemcpyToSymbol(c_elem_ops, ops.data(), sizeof(float) * ops.size(), sizeof(float) * (size_t)(m.N - 1) * ELEM_OPS), "upload operators");
    }
    d.geo3 = U.real(geo, Kp * GEO3);
    if (KERNELS[s->kern3].geox) {
        // record of kernel_vol3d_ws.cuh (GX3): every scale factor of the stage folded in, Z = rho c of the cell:
        // Ga = -dt rho c^2 G | Gb = -dt/rho G | (Fs n, Z A)_f | Z B_f | dt c Fs_f
        std::vector<double> gx;
        if (!A.dry) {
            gx.assign(Kp * GX3, 0.0);
            static const double NH[4][3] = {{0, 0, -1}, {0, -1, 0}, {1, 1, 1}, {-1, 0, 0}};   // outward, in (r,s,t)
            for (int k = 0; k < K; ++k) {
                const double* g = &geo[(size_t)k * GEO3];
                double* x = &gx[(size_t)k * GX3];
                const double Z = s->rho[k] * s->c[k];
                for (int q = 0; q < 9; ++q) {
                    x[q] = -s->dt * g[21] * g[q];
                    x[q < 3 ? 9 + q : 33 + q] = -s->dt * g[22] * g[q];
                }
                for (int f = 0; f < 4; ++f) {
                    for (int c = 0; c < 3; ++c) x[12 + 4 * f + c] = NH[f][0] * g[c] + NH[f][1] * g[3 + c] + NH[f][2] * g[6 + c];
                    x[12 + 4 * f + 3] = Z * g[9 + f];
                    x[28 + f] = Z * g[13 + f];
                    x[32 + f] = s->dt * g[23] * g[17 + f];
                }
            }
        }
        s->geox3 = U.real(gx, Kp * GX3);
    }
    d.nbr3 = U.template ints<int>(m.nbr3, (size_t)K * 4);
    d.finfo3 = U.template ints<uint32_t>(finfo, K);
    d.conn3 = U.template ints<uint32_t>(conn, Kp * 4);
    d.Dt3 = U.real(dt3, (size_t)3 * Np * Np); d.Lt3 = U.real(lt3, (size_t)4 * Nfp * Np);
    d.Dfrag = nullptr; d.Lfrag = nullptr;
    if (s->kern3 == K3_TPG) {
        // operators in MMA-fragment order, zero-padded, for the kernels that fetch them per use (kernel_vol3d_mmag.cuh /
        // kernel_vol3d_tf32g.cuh).  fp64: A of mma.m8n8k4, one value per lane.  fp32: B of mma.m16n8k8, per lane the
        // two k-halves, split into (hi, hi', lo, lo') exactly as split_tf32 does on the device.
        const bool f64 = std::is_same<T, double>::value;
        const int MTn = (Np + 7) / 8, kstep = f64 ? 4 : 8, per = f64 ? 1 : 4;
        const int KDn = (Np + kstep - 1) / kstep, KLn = (Nfp + kstep - 1) / kstep;
        std::vector<T> df, lf;
        if (!A.dry) {
            df.assign((size_t)3 * MTn * KDn * 32 * per, T(0));
            lf.assign((size_t)4 * MTn * KLn * 32 * per, T(0));
            auto put = [&](std::vector<T>& out, size_t base, double v0, double v1) {
                if (f64) { out[base] = (T)v0; return; }
                const float x[2] = {(float)v0, (float)v1};
                for (int h = 0; h < 2; ++h) {
                    uint32_t bits; std::memcpy(&bits, &x[h], 4);
                    bits &= 0xffffe000u;
                    float hi; std::memcpy(&hi, &bits, 4);
                    out[base + h] = (T)hi; out[base + 2 + h] = (T)(x[h] - hi);
                }
            };
            for (int mt = 0; mt < MTn; ++mt)
                for (int lane = 0; lane < 32; ++lane) {
                    const int g = lane >> 2, t = lane & 3, n = 8 * mt + g;
                    if (n >= Np) continue;
                    for (int a = 0; a < 3; ++a)
                        for (int sx = 0; sx < KDn; ++sx) {
                            const int k0 = kstep * sx + t, k1 = k0 + 4;
                            const double v0 = k0 < Np ? m.r3.D[a][(size_t)n * Np + k0] : 0.0;
                            const double v1 = (!f64 && k1 < Np) ? m.r3.D[a][(size_t)n * Np + k1] : 0.0;
                            put(df, ((((size_t)a * MTn + mt) * KDn + sx) * 32 + lane) * per, v0, v1);
                        }
                    for (int f = 0; f < 4; ++f)
                        for (int sx = 0; sx < KLn; ++sx) {
                            const int j0 = kstep * sx + t, j1 = j0 + 4;
                            const double v0 = j0 < Nfp ? m.r3.LIFT[(size_t)n * 4 * Nfp + f * Nfp + j0] : 0.0;
                            const double v1 = (!f64 && j1 < Nfp) ? m.r3.LIFT[(size_t)n * 4 * Nfp + f * Nfp + j1] : 0.0;
                            put(lf, ((((size_t)f * MTn + mt) * KLn + sx) * 32 + lane) * per, v0, v1);
                        }
                }
        }
        d.Dfrag = U.real(df, (size_t)3 * MTn * KDn * 32 * per);
        d.Lfrag = U.real(lf, (size_t)4 * MTn * KLn * 32 * per);
    }
    d.fmask3 = U.template ints<short>(fm3, 4 * Nfp);
    d.perm3 = U.template ints<uint8_t>(m.perm3, 6 * Nfp);
    // ---- 2D
    const size_t n2 = (size_t)Tn * J * 3 * Nfp;
    d.fa[0] = U.zeros(n2); d.fa[1] = U.zeros(n2); d.fres = U.zeros(n2);
    d.S2 = U.zeros((size_t)std::max(m.T, 1) * Nfp);
    d.qb3 = U.zeros((size_t)(m.T + 1) * Nfp);               // row T stays zero: the ghost of wall faces
    d.ghost3 = U.zeros((size_t)(m.T + 1) * Nfp * 4);
    std::vector<double> geo2, d2, l2;
    std::vector<int> fm2;
    if (!A.dry) {
        geo2.assign((size_t)m.T * GEO2, 0.0); d2.resize((size_t)2 * Nfp * Nfp);
        for (int t = 0; t < m.T; ++t) {
            double* g = &geo2[(size_t)t * GEO2];
            const int k = m.tri_tet[t];
            const double Zm = s->rho[k] * s->c[k];
            for (int q = 0; q < 4; ++q) g[q] = m.G2[(size_t)t * 4 + q];
            for (int q = 0; q < 6; ++q) g[4 + q] = m.n2[(size_t)t * 6 + q];
            for (int e = 0; e < 3; ++e) {
                g[10 + e] = m.Fs2[(size_t)t * 3 + e];
                const int nb = m.nbr2[(size_t)t * 3 + e];
                double Zp = Zm;
                if (nb >= 0) { const int kn = m.tri_tet[nb]; Zp = s->rho[kn] * s->c[kn]; }
                g[13 + e] = Zp / (Zp + Zm);
                g[16 + e] = 1.0 / (Zp + Zm);
                if (m.bc2[(size_t)t * 3 + e] == 1) { g[13 + e] = 0.0; g[16 + e] *= 2.0; }
                else if (m.bc2[(size_t)t * 3 + e] == 2) { g[13 + e] *= 2.0; g[16 + e] = 0.0; }
            }
            g[19] = s->rho[k] * s->c[k] * s->c[k]; g[20] = 1.0 / s->rho[k]; g[21] = s->c[k]; g[22] = Zm;
        }
        for (int a = 0; a < 2; ++a)
            for (size_t q = 0; q < (size_t)Nfp * Nfp; ++q) d2[(size_t)a * Nfp * Nfp + q] = m.r2.D[a][q];
        l2 = m.r2.LIFT;
        fm2.assign(m.r2.Fmask.begin(), m.r2.Fmask.end());
    }
    d.geo2 = U.real(geo2, (size_t)m.T * GEO2);
    d.nbr2 = U.template ints<int>(m.nbr2, (size_t)m.T * 3);
    d.nbrnode2 = U.template ints<int>(m.nbrnode2, (size_t)m.T * 3 * N1);
    d.tri_tet = U.template ints<int>(m.tri_tet, m.T);
    d.tri_face = U.template ints<int>(m.tri_face, m.T);
    d.tri_axis = U.template ints<int>(m.tri_axis, m.T);
    d.tri_sign = U.template ints<int>(m.tri_sign, m.T);
    d.D2 = U.real(d2, (size_t)2 * Nfp * Nfp); d.L2 = U.real(l2, (size_t)Nfp * 3 * N1);
    d.fmask2 = U.template ints<short>(fm2, 3 * N1);
    // ---- 1D
    const size_t n1 = (size_t)E * J * J * 2 * N1;
    d.ea[0] = U.zeros(n1); d.ea[1] = U.zeros(n1); d.eres = U.zeros(n1);
    d.S1 = U.zeros((size_t)std::max(m.E, 1) * 2 * std::max(J, 1) * N1);
    d.qb2 = U.zeros((size_t)(2 * m.E + 1) * std::max(J, 1) * N1);    // row 2E stays zero
    std::vector<double> geo1;
    std::vector<int> slot, osign;
    if (!A.dry) {
        geo1.assign((size_t)m.E * GEO1, 0.0); slot.resize((size_t)m.E * 2); osign.resize((size_t)m.E * 2);
        for (int l = 0; l < m.E; ++l) {
            double* g = &geo1[(size_t)l * GEO1];
            const int k = m.tri_tet[m.lin_tri[l * 2]];                 // material of the triangle on face A (reading R9)
            const double Zm = s->rho[k] * s->c[k];
            g[0] = 1.0 / m.J1[l];
            for (int e = 0; e < 2; ++e) {
                const int nb = m.nbr1[l * 2 + e];
                double Zp = Zm;
                if (nb >= 0) { const int kn = m.tri_tet[m.lin_tri[nb * 2]]; Zp = s->rho[kn] * s->c[kn]; }
                g[1 + e] = Zp / (Zp + Zm);
                g[3 + e] = 1.0 / (Zp + Zm);
                if (m.bc1[(size_t)l * 2 + e] == 1) { g[1 + e] = 0.0; g[3 + e] *= 2.0; }
                else if (m.bc1[(size_t)l * 2 + e] == 2) { g[1 + e] *= 2.0; g[3 + e] = 0.0; }
            }
            g[5] = s->rho[k] * s->c[k] * s->c[k]; g[6] = 1.0 / s->rho[k]; g[7] = s->c[k];
            for (int side = 0; side < 2; ++side) {
                const int t = m.lin_tri[l * 2 + side], oth = m.lin_ab[l * 2 + 1 - side];
                slot[l * 2 + side] = (m.tri_ax[t * 2] == oth) ? 0 : 1;
                osign[l * 2 + side] = m.lin_sign[l * 2 + 1 - side];
            }
        }
    }
    d.geo1 = U.real(geo1, (size_t)m.E * GEO1);
    d.nbr1 = U.template ints<int>(m.nbr1, (size_t)m.E * 2);
    d.lin_tri = U.template ints<int>(m.lin_tri, (size_t)m.E * 2);
    d.lin_trinode = U.template ints<int>(m.lin_trinode, (size_t)m.E * 2 * N1);
    d.lin_slot = U.template ints<int>(slot, (size_t)m.E * 2);
    d.lin_osign = U.template ints<int>(osign, (size_t)m.E * 2);
    d.D1 = U.real(m.r1.D[0], (size_t)N1 * N1); d.L1 = U.real(m.r1.LIFT, (size_t)N1 * 2);
    // ---- 0D + algebra
    d.qb1 = U.zeros((size_t)(3 * m.C + 1) * std::max(J * J, 1));    // row 3C stays zero
    d.cor_line = U.template ints<int>(m.cor_line, (size_t)m.C * 3);
    d.cor_end = U.template ints<int>(m.cor_end, (size_t)m.C * 3);
    d.cor_sign = U.template ints<int>(m.cor_sign, (size_t)m.C * 3);
    const HabcCoef& h = s->hc;
    const size_t e2 = (size_t)4 * J * J, c2 = (size_t)9 * J * J * J * J;
    d.cn = U.real(h.cn, J);
    d.Cij = U.real(h.Cij, (size_t)J * J);
    auto transposed = [](const std::vector<double>& M, int n) {
        std::vector<double> Tm(M.size());
        if (M.size() != (size_t)n * n) return Tm;              // sizing pass: the coefficients are not built yet
        for (int r = 0; r < n; ++r)
            for (int k = 0; k < n; ++k) Tm[(size_t)k * n + r] = M[(size_t)r * n + k];
        return Tm;
    };
    d.PeT = U.real(transposed(h.Pe, 2 * J), e2);
    d.QeT = U.real(transposed(h.Qe, 2 * J), e2);
    d.Gc = U.real(h.Gc, c2);
    s->src_w = A.take(sizeof(T) * Np);
    s->t_dev = (double*)A.take(sizeof(double));
    if (!A.dry) {
        cu(cudaMemset(s->src_w, 0, sizeof(T) * Np), "memset");
        cu(cudaMemset(s->t_dev, 0, sizeof(double)), "memset");
    }
    // fp64 scratch for exporting the physical auxiliary fields
    s->export_elems = n2 + n1;
    s->export_buf = (double*)A.take(sizeof(double) * std::max<size_t>(s->export_elems, 1));
}

// ---------------------------------------------------------------- kernel dispatch
// Sizing (configure = true: shared-memory attribute, persistent grid) or launch of one 3D kernel instantiation.
// per_sm_max = 1 for the kernels that own an SM's register file, else what the occupancy calculator allows.
template <typename Kern, typename... Args>
void run_vol3d(dg_solver* s, Kern kern, int nthreads, size_t smem, int elems_per_batch, int K, bool one_per_sm,
               bool configure, Args... args) {
    if (configure) {
        cu(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "smem attr");
        int per_sm = 0, sms = 0;
        cu(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, nthreads, smem), "occupancy");
        cu(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device), "sm count");
        if (per_sm < 1) throw std::runtime_error("ECUDA: the 3D kernel does not fit on an SM");   // caught at dg_create
        if (one_per_sm) per_sm = 1;
        const int nbatch = (K + elems_per_batch - 1) / elems_per_batch;
        s->grid3 = std::max(1, std::min(nbatch, per_sm * sms));
        s->smem3 = smem;
        return;
    }
    kern<<<s->grid3, nthreads, smem, s->stream>>>(args...);
}

template <typename T, int N, int G, int ET, bool SM>
void vol3d_scalar(dg_solver* s, Dev<T>& d, int src, double a, double b, bool cfg) {
    using Cfg = Vol3dCfg<T, N, G, ET, SM>;
    run_vol3d(s, k_vol3d<T, N, G, ET, SM>, Cfg::NT, Cfg::smem_bytes, Cfg::EPB, d.K, false, cfg, d, src, (T)a, (T)b, (T)s->dt);
}
template <int N>
void vol3d_mma(dg_solver* s, Dev<double>& d, int src, double a, double b, bool cfg) {
    using Cfg = MmaCfg<N>;
    run_vol3d(s, k_vol3d_mma<N>, Cfg::NT, Cfg::smem_bytes, Cfg::EB, d.K, false, cfg, d, src, a, b, s->dt);
}
template <int N>
void vol3d_ws(dg_solver* s, Dev<double>& d, int src, double a, double b, bool cfg) {
    using Cfg = WsCfg<N>;
    run_vol3d(s, k_vol3d_ws<N>, Cfg::NT, Cfg::smem_bytes, Cfg::EB, d.K, Cfg::MINB == 1, cfg, d, (const double*)s->geox3, src, a, b);
}
template <int N>
void vol3d_tf32(dg_solver* s, Dev<float>& d, int src, double a, double b, bool cfg) {
    using Cfg = TfCfg<N>;
    run_vol3d(s, k_vol3d_tf32<N>, Cfg::NT, Cfg::smem_bytes, Cfg::EB, d.K, Cfg::MINB == 1, cfg, d, (const float*)s->geox3, src, (float)a, (float)b);
}
template <int N>
void vol3d_mmag(dg_solver* s, Dev<double>& d, int src, double a, double b, bool cfg) {
    using Cfg = MmagCfg<N, 2, 8>;                            // 2 n-tiles (16 elements) per batch, 8 warps
    run_vol3d(s, k_vol3d_mmag<N, 2, 8>, Cfg::NT, Cfg::smem_bytes, Cfg::EPB, d.K, false, cfg, d, src, a, b, s->dt);
}
template <int N>
void vol3d_tf32g(dg_solver* s, Dev<float>& d, int src, double a, double b, bool cfg) {
    constexpr int W = N == 6 ? 7 : N == 7 ? 8 : 11;          // warps per CTA, from the sweep in profiles/r02_degree_sweep.md
    using Cfg = TfgCfg<N, W>;
    run_vol3d(s, k_vol3d_tf32g<N, W>, Cfg::NT, Cfg::smem_bytes, Cfg::EPB, d.K, false, cfg, d, src, (float)a, (float)b, (float)s->dt);
}

template <int N>
void vol3d_elem(dg_solver* s, Dev<float>& d, int src, double a, double b, bool cfg) {
    using Cfg = ElemCfg<N>;
    if (cfg) {
        cu(cudaFuncSetAttribute(k_vol3d_elem<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem_bytes), "smem attr");
        s->grid3 = std::max(1, (d.K + Cfg::NT - 1) / Cfg::NT);     // one thread per element, not persistent
        s->smem3 = Cfg::smem_bytes;
        return;
    }
    k_vol3d_elem<N><<<s->grid3, Cfg::NT, Cfg::smem_bytes, s->stream>>>(d, src, (float)a, (float)b, (float)s->dt);
}

template <typename T> struct OpsFit;                         // scalar kernel: degrees whose operators fit shared memory
template <> struct OpsFit<double> { static constexpr int maxN = 5; };
template <> struct OpsFit<float> { static constexpr int maxN = 6; };

#define DG_CASE(n, call) case n: return call
template <typename T>
void launch_vol3d(dg_solver* s, Dev<T>& d, int src, double a, double b, bool cfg) {
    constexpr bool F64 = std::is_same<T, double>::value;
    constexpr int mx = OpsFit<T>::maxN;
    const int N = s->N;
    switch (s->kern3) {
        case K3_SCALAR:
            switch (N) {
                DG_CASE(1, (vol3d_scalar<T, 1, 32, 4, true>(s, d, src, a, b, cfg)));
                DG_CASE(2, (vol3d_scalar<T, 2, 16, 4, true>(s, d, src, a, b, cfg)));
                DG_CASE(3, (vol3d_scalar<T, 3, 8, 4, true>(s, d, src, a, b, cfg)));
                DG_CASE(4, (vol3d_scalar<T, 4, 8, 4, true>(s, d, src, a, b, cfg)));
                DG_CASE(5, (vol3d_scalar<T, 5, 4, 4, true>(s, d, src, a, b, cfg)));
                DG_CASE(6, (vol3d_scalar<T, 6, 4, 2, (6 <= mx)>(s, d, src, a, b, cfg)));
                DG_CASE(7, (vol3d_scalar<T, 7, 2, 4, false>(s, d, src, a, b, cfg)));
                DG_CASE(8, (vol3d_scalar<T, 8, 2, 2, false>(s, d, src, a, b, cfg)));
            }
            break;
        case K3_MMA:
            if constexpr (F64) switch (N) {
                DG_CASE(1, vol3d_mma<1>(s, d, src, a, b, cfg)); DG_CASE(2, vol3d_mma<2>(s, d, src, a, b, cfg));
                DG_CASE(3, vol3d_mma<3>(s, d, src, a, b, cfg)); DG_CASE(4, vol3d_mma<4>(s, d, src, a, b, cfg));
                DG_CASE(5, vol3d_mma<5>(s, d, src, a, b, cfg));
            }
            break;
        case K3_WS:
            if constexpr (F64) switch (N) {
                DG_CASE(1, vol3d_ws<1>(s, d, src, a, b, cfg)); DG_CASE(2, vol3d_ws<2>(s, d, src, a, b, cfg));
                DG_CASE(3, vol3d_ws<3>(s, d, src, a, b, cfg)); DG_CASE(4, vol3d_ws<4>(s, d, src, a, b, cfg));
                DG_CASE(5, vol3d_ws<5>(s, d, src, a, b, cfg));
            }
            break;
        case K3_TF32:
            if constexpr (!F64) switch (N) {
                DG_CASE(3, vol3d_tf32<3>(s, d, src, a, b, cfg)); DG_CASE(4, vol3d_tf32<4>(s, d, src, a, b, cfg));
                DG_CASE(5, vol3d_tf32<5>(s, d, src, a, b, cfg));
            }
            break;
        case K3_ELEM:
            if constexpr (!F64) switch (N) {
                DG_CASE(1, vol3d_elem<1>(s, d, src, a, b, cfg)); DG_CASE(2, vol3d_elem<2>(s, d, src, a, b, cfg));
            }
            break;
        case K3_TPG:
            if constexpr (F64) switch (N) {
                DG_CASE(6, vol3d_mmag<6>(s, d, src, a, b, cfg)); DG_CASE(7, vol3d_mmag<7>(s, d, src, a, b, cfg));
                DG_CASE(8, vol3d_mmag<8>(s, d, src, a, b, cfg));
            } else switch (N) {
                DG_CASE(6, vol3d_tf32g<6>(s, d, src, a, b, cfg)); DG_CASE(7, vol3d_tf32g<7>(s, d, src, a, b, cfg));
                DG_CASE(8, vol3d_tf32g<8>(s, d, src, a, b, cfg));
            }
            break;
    }
    throw std::runtime_error("EINVAL: no 3D kernel for this (kernel, precision, N)");     // resolve_kernel rules this out
}
#undef DG_CASE

// 2D solver.  fp64, N <= 5: the tensor-pipe kernel (kernel_face2d.cuh); otherwise the scalar kernel.
// configure = true: shared-memory attribute and persistent grid instead of a launch.
template <int N>
void face2d_mma_run(dg_solver* s, Dev<double>& d, int src, double a, double b, bool configure) {
    using Cfg = Face2dMmaCfg<N>;
    if (configure) {
        cu(cudaFuncSetAttribute(k_face2d_mma<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem_bytes), "smem attr");
        int per_sm = 0, sms = 0;
        cu(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_face2d_mma<N>, Cfg::NT, Cfg::smem_bytes), "occupancy");
        cu(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device), "sm count");
        if (per_sm < 1) throw std::runtime_error("ECUDA: the 2D kernel does not fit on an SM");
        const int nitems = d.Tn * ((d.J + Cfg::SB - 1) / Cfg::SB), nchunk = (nitems + Cfg::PB - 1) / Cfg::PB;
        s->face_grid = std::max(1, std::min(nchunk, per_sm * sms));
        return;
    }
    k_face2d_mma<N><<<s->face_grid, Cfg::NT, Cfg::smem_bytes, s->stream>>>(d, src, a, b, s->dt);
}

template <typename T>
void launch_face2d(dg_solver* s, Dev<T>& d, int src, double a, double b, bool configure = false) {
    if constexpr (std::is_same<T, double>::value) {
        switch (s->N) {
            case 1: return face2d_mma_run<1>(s, d, src, a, b, configure);
            case 2: return face2d_mma_run<2>(s, d, src, a, b, configure);
            case 3: return face2d_mma_run<3>(s, d, src, a, b, configure);
            case 4: return face2d_mma_run<4>(s, d, src, a, b, configure);
            case 5: return face2d_mma_run<5>(s, d, src, a, b, configure);
        }
    }
    if (configure) {
        int sms = 0;
        cu(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device), "sm count");
        s->face_grid = sms * 8;
        cu(cudaFuncSetAttribute(k_face2d<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024), "smem attr");
        return;
    }
    const int Nf = 3 * d.N1, PB = std::max(1, FACE2D_NT / std::max(d.Nfp, Nf));
    const size_t smem = sizeof(T) * (face2d_ops_elems(d.Nfp, d.N1) + (size_t)PB * (5 * d.Nfp + Nf) * FACE2D_SB);
    const int nitems = d.Tn * ((d.J + FACE2D_SB - 1) / FACE2D_SB);
    const int nchunk = (nitems + PB - 1) / PB;
    const int grid = std::max(1, std::min(nchunk, s->face_grid));
    k_face2d<T><<<grid, FACE2D_NT, smem, s->stream>>>(d, src, (T)a, (T)b, (T)s->dt);
}

// one LSRK stage: 3D, 2D, 1D solvers (independent), then the closure chain 2D -> 1D -> 0D
template <typename T>
void launch_closures(dg_solver* s, Dev<T>& d, int cur) {
    if (d.J == 0 || d.Tn == 0) return;
    const int nf = d.Tn * d.Nfp;
    k_close_face<T><<<(nf + 255) / 256, 256, 0, s->stream>>>(d, cur);
    if (d.E > 0) {
        const int ne = d.E * d.N1;
        k_close_edge<T><<<(ne + CLOSE_EDGE_WARPS - 1) / CLOSE_EDGE_WARPS, 32 * CLOSE_EDGE_WARPS, 0, s->stream>>>(d, cur);
    }
    if (d.C > 0) {
        const int JJ3 = 3 * d.J * d.J;
        k_close_corner<T><<<d.C, 1024, sizeof(T) * JJ3, s->stream>>>(d, cur);
    }
}

template <typename T>
void launch_source(dg_solver* s, Dev<T>& d, int src, int stage) {
    if (!s->src_on) return;
    k_source<T><<<1, 64, 0, s->stream>>>(d.q[src ^ 1], d.res, (const T*)s->src_w, s->src_k, d.Np, s->t_dev,
                                       RKC[stage] * s->dt, s->dt, RKB[stage], s->src_f, s->src_ts, s->src_amp, stage == 4);
}

template <typename T>
void launch_stage(dg_solver* s, Dev<T>& d, int src, int stage, int par) {
    const double a = RKA[stage], b = RKB[stage];
    // inside a stream capture an event only becomes a real record node of the graph with cudaEventRecordExternal
    // (the flag is invalid outside a capture)
    unsigned evflag = cudaEventRecordDefault;
    if (s->time_kernels) {
        cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
        cu(cudaStreamIsCapturing(s->stream, &st), "capture status");
        if (st == cudaStreamCaptureStatusActive) evflag = cudaEventRecordExternal;
        cu(cudaEventRecordWithFlags(s->evk[par][stage][0], s->stream, evflag), "event record");
    }
    launch_vol3d<T>(s, d, src, a, b, false);
    if (s->time_kernels) cu(cudaEventRecordWithFlags(s->evk[par][stage][1], s->stream, evflag), "event record");
    launch_source<T>(s, d, src, stage);
    if (d.J > 0 && d.Tn > 0) {
        launch_face2d<T>(s, d, src, a, b);
        if (d.E > 0) {
            const int work = d.J * d.J * d.N1;
            k_edge1d<T><<<d.E, std::min(512, ((work + 31) / 32) * 32), sizeof(T) * 2 * work, s->stream>>>(
                d, src, (T)a, (T)b, (T)s->dt);
        }
    }
    launch_closures<T>(s, d, src ^ 1);
}

int launches_per_stage(const dg_solver* s) {
    int n = 1 + (s->src_on ? 1 : 0);
    if (s->J > 0 && s->m.T > 0) {
        n += 2;                       // 2D solver + face closure
        if (s->m.E > 0) n += 2;       // 1D solver + edge closure
        if (s->m.C > 0) n += 1;       // corner closure
    }
    return n;
}

template <typename T>
void run_step_plain(dg_solver* s, Dev<T>& d) {
    const int par = s->cur;
    for (int st = 0; st < 5; ++st) {
        launch_stage<T>(s, d, s->cur, st, par);
        s->cur ^= 1;
    }
}

template <typename T>
void run_steps(dg_solver* s, Dev<T>& d, int nsteps) {
    if (!s->use_graph) {
        for (int i = 0; i < nsteps; ++i) {
            s->last_par = s->cur;
            run_step_plain<T>(s, d);
            cu(cudaGetLastError(), "kernel launch");
            s->t_host += s->dt;        // the host clock follows the steps that were really enqueued
        }
        return;
    }
    for (int i = 0; i < nsteps; ++i) {
        const int par = s->cur;
        if (!s->graph[par]) {
            cudaGraph_t g = nullptr;
            cu(cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal), "begin capture");
            try {
                run_step_plain<T>(s, d);
                cu(cudaGetLastError(), "kernel launch (capture)");
            } catch (...) {                // never leave the caller's stream in capture mode
                cudaStreamEndCapture(s->stream, &g);
                if (g) cudaGraphDestroy(g);
                cudaGetLastError();
                s->cur = par;
                throw;
            }
            cu(cudaStreamEndCapture(s->stream, &g), "end capture");
            const cudaError_t e = cudaGraphInstantiate(&s->graph[par], g, 0);
            cudaGraphDestroy(g);
            s->cur = par;              // capture did not execute anything
            cu(e, "graph instantiate");
        }
        cu(cudaGraphLaunch(s->graph[par], s->stream), "graph launch");
        s->last_par = par;
        s->cur = par ^ 1;              // five stages flip the parity once
        s->t_host += s->dt;
    }
}

size_t dry_bytes(dg_solver* s) {
    Arena A;
    A.dry = true;
    if (s->precision == 64) { Dev<double> d{}; build_device<double>(s, A, d); }
    else { Dev<float> d{}; build_device<float>(s, A, d); }
    return A.used + 256;
}

void check_args(const dg_mesh* mesh, int N, int J, int precision) {
    if (!mesh || !mesh->xyz || !mesh->tets) throw std::runtime_error("EINVAL: NULL mesh");
    if (N < 1 || N > 8) throw std::runtime_error("EINVAL: N must be in 1..8");
    if (J < 0 || J > JMAX) throw std::runtime_error("EINVAL: J must be in 0..12");
    if (precision != 64 && precision != 32) throw std::runtime_error("EINVAL: precision must be 64 or 32");
}

template <typename T>
void upload_initial(dg_solver* s, Dev<T>& d, const double* p, const double* u, const double* v, const double* w) {
    const size_t n = (size_t)d.K * d.Np;
    // each fp64 field goes to the device as it is (q[1] is free here and serves as the staging area: it holds
    // 4 n values of T >= n doubles) and is converted / interleaved into q[0] by a kernel
    const double* fields[4] = {p, u, v, w};
    double* stage = reinterpret_cast<double*>(d.q[1]);
    for (int f = 0; f < 4; ++f) {
        cu(cudaMemcpyAsync(stage, fields[f], sizeof(double) * n, cudaMemcpyHostToDevice, s->stream), "upload field");
        k_pack_field<T><<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(stage, d.q[0], f, n);
    }
    cu(cudaGetLastError(), "pack launch");
    cu(cudaMemsetAsync(d.q[1], 0, sizeof(T) * n * 4, s->stream), "memset");
    cu(cudaMemsetAsync(d.res, 0, sizeof(T) * n * 4, s->stream), "memset");
    const size_t n2 = (size_t)d.Tn * d.J * 3 * d.Nfp, n1 = (size_t)d.E * d.J * d.J * 2 * d.N1;
    for (int b = 0; b < 2; ++b) {
        if (n2) cu(cudaMemsetAsync(d.fa[b], 0, sizeof(T) * n2, s->stream), "memset");
        if (n1) cu(cudaMemsetAsync(d.ea[b], 0, sizeof(T) * n1, s->stream), "memset");
    }
    if (n2) cu(cudaMemsetAsync(d.fres, 0, sizeof(T) * n2, s->stream), "memset");
    if (n1) cu(cudaMemsetAsync(d.eres, 0, sizeof(T) * n1, s->stream), "memset");
    s->cur = 0;
    s->t_host = 0;
    cu(cudaMemsetAsync(s->t_dev, 0, sizeof(double), s->stream), "memset");
    launch_closures<T>(s, d, 0);        // reading R5: cached r^-, S consistent with the initial state
    cu(cudaStreamSynchronize(s->stream), "set_initial");
}

template <typename T>
void download_fields(dg_solver* s, Dev<T>& d, double* p, double* u, double* v, double* w, double* fa, double* ea) {
    const size_t n = (size_t)d.K * d.Np;
    {
        // one field at a time through the buffer the next stage will overwrite anyway (q[cur ^ 1])
        double* out[4] = {p, u, v, w};
        double* stage = reinterpret_cast<double*>(d.q[s->cur ^ 1]);
        for (int f = 0; f < 4; ++f) {
            if (!out[f]) continue;
            k_unpack_field<T><<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(d.q[s->cur], stage, f, n);
            cu(cudaMemcpyAsync(out[f], stage, sizeof(double) * n, cudaMemcpyDeviceToHost, s->stream), "download field");
        }
        cu(cudaGetLastError(), "unpack launch");
    }
    const size_t n2 = (size_t)d.Tn * d.J * 3 * d.Nfp, n1 = (size_t)d.E * d.J * d.J * 2 * d.N1;
    if ((fa || ea) && n2 + n1 > 0) {
        const size_t tot = n2 + n1;
        k_export_aux<T><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(d, s->cur, s->export_buf, s->export_buf + n2);
        cu(cudaGetLastError(), "export launch");
        if (fa && n2) cu(cudaMemcpyAsync(fa, s->export_buf, sizeof(double) * n2, cudaMemcpyDeviceToHost, s->stream), "download");
        if (ea && n1) cu(cudaMemcpyAsync(ea, s->export_buf + n2, sizeof(double) * n1, cudaMemcpyDeviceToHost, s->stream), "download");
    }
    cu(cudaStreamSynchronize(s->stream), "sync");
}

template <typename T>
void profile_step(dg_solver* s, Dev<T>& d, double* ms) {
    for (int i = 0; i < 6; ++i) ms[i] = 0;
    cudaEvent_t ev[2];
    cu(cudaEventCreate(&ev[0]), "event"); cu(cudaEventCreate(&ev[1]), "event");
    auto timed = [&](int slot, auto&& fn) {
        cu(cudaEventRecord(ev[0], s->stream), "record");
        fn();
        cu(cudaEventRecord(ev[1], s->stream), "record");
        cu(cudaEventSynchronize(ev[1]), "sync");
        float t = 0;
        cu(cudaEventElapsedTime(&t, ev[0], ev[1]), "elapsed");
        ms[slot] += t;
    };
    for (int st = 0; st < 5; ++st) {
        const int src = s->cur;
        const double a = RKA[st], b = RKB[st];
        timed(0, [&] { launch_vol3d<T>(s, d, src, a, b, false); launch_source<T>(s, d, src, st); });
        if (d.J > 0 && d.Tn > 0) {
            timed(1, [&] { launch_face2d<T>(s, d, src, a, b); });
            if (d.E > 0) {
                const int work = d.J * d.J * d.N1;
                timed(2, [&] {
                    k_edge1d<T><<<d.E, std::min(512, ((work + 31) / 32) * 32), sizeof(T) * 2 * work, s->stream>>>(
                        d, src, (T)a, (T)b, (T)s->dt);
                });
            }
            const int cur = src ^ 1;
            timed(3, [&] { k_close_face<T><<<(d.Tn * d.Nfp + 255) / 256, 256, 0, s->stream>>>(d, cur); });
            if (d.E > 0) timed(4, [&] { k_close_edge<T><<<(d.E * d.N1 + CLOSE_EDGE_WARPS - 1) / CLOSE_EDGE_WARPS, 32 * CLOSE_EDGE_WARPS, 0, s->stream>>>(d, cur); });
            if (d.C > 0) {
                const int JJ3 = 3 * d.J * d.J;
                timed(5, [&] {
                    k_close_corner<T><<<d.C, 1024, sizeof(T) * JJ3, s->stream>>>(d, cur);
                });
            }
        }
        s->cur ^= 1;
    }
    cudaEventDestroy(ev[0]); cudaEventDestroy(ev[1]);
    cu(cudaGetLastError(), "profile step");
}

}  // namespace

// ======================================================================================= C ABI
extern "C" {

const char* dg_last_error(void) { return g_err.c_str(); }

int dg_mesh_counts(const dg_mesh* mesh, const int32_t* face_bc, int32_t* counts) {
    try {
        if (!mesh || !counts) throw std::runtime_error("EINVAL: NULL argument");
        dg::HostMesh m;
        dg::build_mesh(m, 1, mesh->nverts, mesh->xyz, mesh->ntets, mesh->tets, face_bc);
        counts[0] = m.K; counts[1] = m.T; counts[2] = m.E; counts[3] = m.C;
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_reference_element(int dim, int N, double* rst, double* D, double* LIFT, int32_t* Fmask, int32_t* np_out) {
    try {
        dg::RefElem e = dg::make_refelem(dim, N);
        if (np_out) *np_out = e.Np;
        if (rst) for (size_t i = 0; i < e.rst.size(); ++i) rst[i] = (double)e.rst[i];
        if (D) for (int a = 0; a < dim; ++a) std::copy(e.D[a].begin(), e.D[a].end(), D + (size_t)a * e.Np * e.Np);
        if (LIFT) std::copy(e.LIFT.begin(), e.LIFT.end(), LIFT);
        if (Fmask) std::copy(e.Fmask.begin(), e.Fmask.end(), Fmask);
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

// Exact hierarchy sizes of a cuboid mesh without building connectivity: boundary cell faces are the faces whose
// three vertices share a bounding plane; boundary lines are the distinct cell edges lying on two bounding planes.
static void quick_counts(const dg_mesh* mesh, int& T, int& E) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int v = 0; v < mesh->nverts; ++v)
        for (int d = 0; d < 3; ++d) {
            lo[d] = std::min(lo[d], mesh->xyz[v * 3 + d]);
            hi[d] = std::max(hi[d], mesh->xyz[v * 3 + d]);
        }
    const double tol = 1e-9 * std::max({hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]});
    std::vector<uint8_t> code(mesh->nverts, 0);
    for (int v = 0; v < mesh->nverts; ++v)
        for (int d = 0; d < 3; ++d) {
            if (std::fabs(mesh->xyz[v * 3 + d] - lo[d]) < tol) code[v] |= 1 << (2 * d);
            if (std::fabs(mesh->xyz[v * 3 + d] - hi[d]) < tol) code[v] |= 2 << (2 * d);
        }
    T = 0;
    std::set<std::pair<int, int>> lines;
    for (int k = 0; k < mesh->ntets; ++k) {
        const int32_t* t = mesh->tets + (size_t)k * 4;
        for (int f = 0; f < 4; ++f) {
            int a = t[dg::TET_FACE_VERTS[f][0]], b = t[dg::TET_FACE_VERTS[f][1]], c = t[dg::TET_FACE_VERTS[f][2]];
            if (code[a] & code[b] & code[c]) ++T;
        }
        for (int i = 0; i < 4; ++i)
            for (int j = i + 1; j < 4; ++j)
                if (__builtin_popcount(code[t[i]] & code[t[j]]) >= 2)
                    lines.insert({std::min(t[i], t[j]), std::max(t[i], t[j])});
    }
    E = (int)lines.size();
}

int dg_workspace_bytes(const dg_mesh* mesh, int N, int J, int precision, uint64_t* bytes) {
    try {
        check_args(mesh, N, J, precision);
        if (!bytes) throw std::runtime_error("EINVAL: NULL argument");
        dg_solver s;
        s.N = N; s.J = J; s.precision = precision;
        s.m.N = N; s.m.K = mesh->ntets; s.m.C = 8;
        quick_counts(mesh, s.m.T, s.m.E);
        s.m.Np = (N + 1) * (N + 2) * (N + 3) / 6; s.m.Nfp = (N + 1) * (N + 2) / 2; s.m.N1 = N + 1;
        size_t need = 0;                                       // upper bound over every dg_options.kernel choice that
        for (int k = 1; k < K3_COUNT; ++k) {                   // covers (precision, N): some carry extra per-tet records
            if ((KERNELS[k].precision && KERNELS[k].precision != precision) || N < KERNELS[k].nmin || N > KERNELS[k].nmax) continue;
            s.kern3 = k;
            need = std::max(need, dry_bytes(&s));
        }
        *bytes = need + 4096;
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_create(const dg_mesh* mesh, int N, int J, const double* c, const double* rho, const dg_options* opt,
              dg_solver** out) {
    dg_solver* s = nullptr;
    try {
        const int precision = opt ? opt->precision : 64;
        check_args(mesh, N, J, precision);
        if (!c || !rho || !out) throw std::runtime_error("EINVAL: NULL argument");
        for (int k = 0; k < mesh->ntets; ++k)
            if (!(c[k] > 0) || !(rho[k] > 0)) throw std::runtime_error("EINVAL: c and rho must be positive");
        s = new dg_solver();
        s->N = N; s->J = J; s->precision = precision;
        s->device = opt ? opt->device : 0;
        s->stream = opt ? (cudaStream_t)opt->stream : nullptr;
        s->use_graph = opt ? opt->use_graph != 0 : true;
        s->kern3 = resolve_kernel(opt ? opt->kernel : 0, precision, N);
        s->time_kernels = opt && opt->time_kernels != 0;
        if (mesh->ntets > CONN_MAX_ID) throw std::runtime_error("EINVAL: more than 2^26 - 1 tetrahedra");
        if (!s->stream) s->use_graph = false;      // the legacy default stream cannot be captured
        s->rho.assign(rho, rho + mesh->ntets);
        s->c.assign(c, c + mesh->ntets);
        dg::build_mesh(s->m, N, mesh->nverts, mesh->xyz, mesh->ntets, mesh->tets, opt ? opt->face_bc : nullptr);
        s->hc = dg::make_habc(J);
        // eq (46), PAPER.md:L796 (reading R7): dt = cfl * min_k 1 / (c_k (N+1)^2 max_f Fscale_kf)
        double dtmin = 1e300;
        for (int k = 0; k < s->m.K; ++k) {
            double fs = 0;
            for (int f = 0; f < 4; ++f) fs = std::max(fs, s->m.Fs3[(size_t)k * 4 + f]);
            dtmin = std::min(dtmin, 1.0 / (c[k] * (N + 1) * (N + 1) * fs));
        }
        const double cfl = (opt && opt->cfl > 0) ? opt->cfl : 1.0;
        s->dt = (opt && opt->dt > 0) ? opt->dt : cfl * dtmin;
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->time_kernels)
            for (auto& par : s->evk) for (auto& st : par) for (auto& e : st) cu(cudaEventCreate(&e), "event create");
        const size_t need = dry_bytes(s);
        if (opt && opt->workspace_dev) {
            if (opt->workspace_bytes < need) throw std::runtime_error("ENOMEM: workspace_bytes is smaller than dg_workspace_bytes");
            s->ws = opt->workspace_dev; s->ws_bytes = opt->workspace_bytes; s->own_ws = false;
        } else {
            if (cudaMalloc(&s->ws, need) != cudaSuccess) { cudaGetLastError(); throw std::runtime_error("ENOMEM: cudaMalloc failed"); }
            s->ws_bytes = need; s->own_ws = true;
        }
        Arena A;
        A.base = (char*)s->ws; A.size = s->ws_bytes; A.dry = false;
        // align the arena base to 256 B
        size_t mis = (size_t)(uintptr_t)A.base & 255;
        if (mis) { A.base += 256 - mis; A.size -= 256 - mis; }
        if (precision == 64) {
            build_device<double>(s, A, s->d64);
            launch_vol3d<double>(s, s->d64, 0, 0, 0, true);
            if (s->d64.J > 0 && s->d64.Tn > 0) launch_face2d<double>(s, s->d64, 0, 0, 0, true);
        } else {
            build_device<float>(s, A, s->d32);
            launch_vol3d<float>(s, s->d32, 0, 0, 0, true);
            if (s->d32.J > 0 && s->d32.Tn > 0) launch_face2d<float>(s, s->d32, 0, 0, 0, true);
        }
        cu(cudaDeviceSynchronize(), "setup");
        *out = s;
        return DG_OK;
    } catch (const std::exception& e) {
        if (s) dg_destroy(s);
        return err_from_exception(e);
    }
}

void dg_destroy(dg_solver* s) {
    if (!s) return;
    int prev = -1;
    cudaGetDevice(&prev);                  // the caller's current device is left as it was
    if (cudaSetDevice(s->device) == cudaSuccess) {
        cudaStreamSynchronize(s->stream);  // dg_step is asynchronous: nothing may still be writing the workspace
        for (int i = 0; i < 2; ++i) if (s->graph[i]) cudaGraphExecDestroy(s->graph[i]);
        for (auto& par : s->evk) for (auto& st : par) for (auto& e : st) if (e) cudaEventDestroy(e);
        if (s->own_ws && s->ws) cudaFree(s->ws);
    }
    if (prev >= 0) cudaSetDevice(prev);
    cudaGetLastError();                    // the return codes above are ignored on purpose: leave no stale error behind
    delete s;
}

int dg_get_info(const dg_solver* s, dg_info* o) {
    if (!s || !o) return set_err(DG_EINVAL, "EINVAL: NULL argument");
    o->N = s->N; o->J = s->J; o->K = s->m.K; o->Np = s->m.Np; o->Nfp = s->m.Nfp;
    o->T = s->m.T; o->E = s->m.E; o->C = s->m.C; o->precision = s->precision;
    o->launches_per_step = 5 * launches_per_stage(s);
    o->dt = s->dt; o->device_bytes = s->ws_bytes;
    o->kernel = s->kern3;
    static const char* const NAMES[K3_COUNT][2] = {{"", ""}, {"k_vol3d", "k_vol3d"}, {"k_vol3d_mma", ""}, {"k_vol3d_ws", ""},
                                                   {"", "k_vol3d_tf32"}, {"k_vol3d_mmag", "k_vol3d_tf32g"}, {"", "k_vol3d_elem"}};
    snprintf(o->kernel_name, sizeof(o->kernel_name), "%s<%d>", NAMES[s->kern3][s->precision == 32], s->N);
    return DG_OK;
}

int dg_get_nodes(const dg_solver* s, double* x, double* y, double* z) {
    if (!s) return set_err(DG_EINVAL, "EINVAL: NULL argument");
    const dg::HostMesh& m = s->m;
    double* out[3] = {x, y, z};
    for (int k = 0; k < m.K; ++k)
        for (int n = 0; n < m.Np; ++n)
            for (int d = 0; d < 3; ++d) {
                if (!out[d]) continue;
                long double acc = 0;
                for (int v = 0; v < 4; ++v) acc += m.r3.bary[(size_t)n * 4 + v] * m.verts[(size_t)m.tets[(size_t)k * 4 + v] * 3 + d];
                out[d][(size_t)k * m.Np + n] = (double)acc;
            }
    return DG_OK;
}

int dg_set_initial(dg_solver* s, const double* p, const double* u, const double* v, const double* w) {
    try {
        if (!s || !p || !u || !v || !w) throw std::runtime_error("EINVAL: NULL argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->precision == 64) upload_initial<double>(s, s->d64, p, u, v, w);
        else upload_initial<float>(s, s->d32, p, u, v, w);
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_set_source(dg_solver* s, const double* xyz, double f_peak, double t_s, double amplitude) {
    try {
        if (!s || !xyz) throw std::runtime_error("EINVAL: NULL argument");
        if (!(f_peak > 0)) throw std::runtime_error("EINVAL: f_peak must be positive");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        const dg::HostMesh& m = s->m;
        typedef long double ld;
        int kfound = -1;
        ld lam[4] = {0, 0, 0, 0};
        for (int k = 0; k < m.K && kfound < 0; ++k) {
            const double* v[4];
            for (int i = 0; i < 4; ++i) v[i] = &m.verts[(size_t)m.tets[(size_t)k * 4 + i] * 3];
            ld A[3][3], b[3];
            for (int r = 0; r < 3; ++r) {
                for (int c = 0; c < 3; ++c) A[r][c] = (ld)v[c + 1][r] - (ld)v[0][r];
                b[r] = (ld)xyz[r] - (ld)v[0][r];
            }
            auto det3 = [](ld M[3][3]) {
                return M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0]) +
                       M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
            };
            const ld D = det3(A);
            ld l[4];
            l[0] = 1;
            for (int c = 0; c < 3; ++c) {
                ld B[3][3];
                for (int r = 0; r < 3; ++r)
                    for (int q = 0; q < 3; ++q) B[r][q] = q == c ? b[r] : A[r][q];
                l[c + 1] = det3(B) / D;
                l[0] -= l[c + 1];
            }
            if (std::min(std::min(l[0], l[1]), std::min(l[2], l[3])) >= -1e-12L) {
                kfound = k;
                for (int i = 0; i < 4; ++i) lam[i] = l[i];
            }
        }
        if (kfound < 0) throw std::runtime_error("EINVAL: the source point is outside the mesh");
        const ld rst[3] = {-1 + 2 * lam[1], -1 + 2 * lam[2], -1 + 2 * lam[3]};
        std::vector<double> w = dg::delta_weights(m.r3, rst);
        for (double& x : w) x /= m.J3[kfound];
        cu(cudaStreamSynchronize(s->stream), "sync");
        if (s->precision == 64) {
            cu(cudaMemcpy(s->src_w, w.data(), sizeof(double) * w.size(), cudaMemcpyHostToDevice), "upload weights");
        } else {
            std::vector<float> wf(w.begin(), w.end());
            cu(cudaMemcpy(s->src_w, wf.data(), sizeof(float) * wf.size(), cudaMemcpyHostToDevice), "upload weights");
        }
        // the device clock only runs while a source is on: bring it to the time reached so far
        cu(cudaMemcpy(s->t_dev, &s->t_host, sizeof(double), cudaMemcpyHostToDevice), "upload clock");
        s->src_k = kfound; s->src_f = f_peak; s->src_ts = t_s; s->src_amp = amplitude;
        s->src_on = amplitude != 0.0;
        for (int i = 0; i < 2; ++i)                 // the captured step no longer matches
            if (s->graph[i]) { cudaGraphExecDestroy(s->graph[i]); s->graph[i] = nullptr; }
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_step(dg_solver* s, int nsteps) {
    try {
        if (!s || nsteps < 0) throw std::runtime_error("EINVAL: bad argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->precision == 64) run_steps<double>(s, s->d64, nsteps);
        else run_steps<float>(s, s->d32, nsteps);
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_get_fields(dg_solver* s, double* p, double* u, double* v, double* w, double* face_aux, double* edge_aux) {
    try {
        if (!s) throw std::runtime_error("EINVAL: NULL argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->precision == 64) download_fields<double>(s, s->d64, p, u, v, w, face_aux, edge_aux);
        else download_fields<float>(s, s->d32, p, u, v, w, face_aux, edge_aux);
        cu(cudaGetLastError(), "device work");
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_get_face_map(const dg_solver* s, int32_t* tet, int32_t* face, int32_t* axis, int32_t* sign, double* xyz) {
    if (!s) return set_err(DG_EINVAL, "EINVAL: NULL argument");
    const dg::HostMesh& m = s->m;
    for (int t = 0; t < m.T; ++t) {
        if (tet) tet[t] = m.tri_tet[t];
        if (face) face[t] = m.tri_face[t];
        if (axis) axis[t] = m.tri_axis[t];
        if (sign) sign[t] = m.tri_sign[t];
        if (xyz)
            for (int j = 0; j < m.Nfp; ++j) {
                const int n = m.r3.Fmask[m.tri_face[t] * m.Nfp + j];
                for (int d = 0; d < 3; ++d) {
                    long double acc = 0;
                    for (int v = 0; v < 4; ++v)
                        acc += m.r3.bary[(size_t)n * 4 + v] * m.verts[(size_t)m.tets[(size_t)m.tri_tet[t] * 4 + v] * 3 + d];
                    xyz[((size_t)t * m.Nfp + j) * 3 + d] = (double)acc;
                }
            }
    }
    return DG_OK;
}

int dg_get_edge_map(const dg_solver* s, int32_t* axis, int32_t* normal_axes, int32_t* signs, double* xyz) {
    if (!s) return set_err(DG_EINVAL, "EINVAL: NULL argument");
    const dg::HostMesh& m = s->m;
    for (int l = 0; l < m.E; ++l) {
        if (axis) axis[l] = m.lin_axis[l];
        for (int q = 0; q < 2; ++q) {
            if (normal_axes) normal_axes[l * 2 + q] = m.lin_ab[l * 2 + q];
            if (signs) signs[l * 2 + q] = m.lin_sign[l * 2 + q];
        }
        if (xyz)
            for (int n = 0; n < m.N1; ++n)
                for (int d = 0; d < 3; ++d) {
                    long double acc = 0;
                    for (int v = 0; v < 2; ++v) acc += m.r1.bary[(size_t)n * 2 + v] * m.verts[(size_t)m.lin_v[l * 2 + v] * 3 + d];
                    xyz[((size_t)l * m.N1 + n) * 3 + d] = (double)acc;
                }
    }
    return DG_OK;
}

int dg_set_time_kernels(dg_solver* s, int on) {
    try {
        if (!s) throw std::runtime_error("EINVAL: NULL argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if ((on != 0) == s->time_kernels) return DG_OK;
        cu(cudaStreamSynchronize(s->stream), "sync");
        if (on)
            for (auto& par : s->evk) for (auto& st : par) for (auto& e : st)
                if (!e) cu(cudaEventCreate(&e), "event create");
        s->time_kernels = on != 0;
        s->last_par = -1;                          // no step has been timed under the new setting yet
        for (int i = 0; i < 2; ++i)                 // the captured step has (or lacks) the event nodes: capture again
            if (s->graph[i]) { cudaGraphExecDestroy(s->graph[i]); s->graph[i] = nullptr; }
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_last_step_kernel_ms(dg_solver* s, double* ms) {
    try {
        if (!s || !ms) throw std::runtime_error("EINVAL: NULL argument");
        if (!s->time_kernels) throw std::runtime_error("EINVAL: the solver was created without dg_options.time_kernels");
        if (s->last_par < 0) throw std::runtime_error("EINVAL: no step has been enqueued yet");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        cu(cudaStreamSynchronize(s->stream), "sync");
        for (int st = 0; st < 5; ++st) {
            float t = 0;
            cu(cudaEventElapsedTime(&t, s->evk[s->last_par][st][0], s->evk[s->last_par][st][1]), "elapsed");
            ms[st] = t;
        }
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

int dg_get_device_ptrs(const dg_solver* s, dg_device_view* o) {
    if (!s || !o) return set_err(DG_EINVAL, "EINVAL: NULL argument");
    const bool aux = s->J > 0;
    o->reserved = 0;
    if (s->precision == 64) {
        const dg::Dev<double>& d = s->d64;
        o->elem_bytes = 8; o->q = d.q[s->cur];
        o->face_aux = aux && d.Tn > 0 ? d.fa[s->cur] : nullptr; o->face_S = aux && d.Tn > 0 ? d.S2 : nullptr;
        o->edge_aux = aux && d.E > 0 ? d.ea[s->cur] : nullptr;
    } else {
        const dg::Dev<float>& d = s->d32;
        o->elem_bytes = 4; o->q = d.q[s->cur];
        o->face_aux = aux && d.Tn > 0 ? d.fa[s->cur] : nullptr; o->face_S = aux && d.Tn > 0 ? d.S2 : nullptr;
        o->edge_aux = aux && d.E > 0 ? d.ea[s->cur] : nullptr;
    }
    return DG_OK;
}

int dg_profile_step(dg_solver* s, double* ms) {
    try {
        if (!s || !ms) throw std::runtime_error("EINVAL: NULL argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->precision == 64) profile_step<double>(s, s->d64, ms);
        else profile_step<float>(s, s->d32, ms);
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}

}  // extern "C"

// ======================================================================================= allocation-free read-back
// dg_get_aux_fields_noalloc (include/dg_habc.h): k_export_aux staged through an array that is part of the library
// image, for callers that have no way to obtain device memory (see the header for who they are).
#include <mutex>

// The staging area.  One instance per CUDA context that loads this module, DG_NOALLOC_MAX_VALUES doubles = 4 MiB, held
// until the process exits.  In HOST code the name g_noalloc_stage is only a handle for the runtime's symbol calls: it
// is not a device address and must never be handed to a kernel or to cudaMemcpy as a pointer.
static __device__ __align__(256) double g_noalloc_stage[DG_NOALLOC_MAX_VALUES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_lock;                                   // set-up table and the array itself (one call at a time)
double* g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};            // device address of g_noalloc_stage, per device ordinal

// Device address of the staging array on `device`, which must be the current device.  Looked up on the first call
// for that device and remembered; every later call is a table read.  Caller holds g_noalloc_lock.
double* noalloc_stage_address(int device) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES)
        throw std::runtime_error("EINVAL: dg_get_aux_fields_noalloc supports device ordinals 0..63");
    if (!g_noalloc_addr[device]) {
        double* ptr = nullptr;
        cu(cudaGetSymbolAddress((void**)&ptr, g_noalloc_stage), "cudaGetSymbolAddress(staging array)");
        if (!ptr) throw std::runtime_error("ECUDA: the staging array has no address on this device");
        g_noalloc_addr[device] = ptr;
    }
    return g_noalloc_addr[device];
}

template <typename T>
void export_aux_noalloc(dg_solver* s, Dev<T>& d, double* fa, double* ea) {
    const size_t n2 = (size_t)d.Tn * d.J * 3 * d.Nfp, n1 = (size_t)d.E * d.J * d.J * 2 * d.N1, tot = n2 + n1;
    if (tot > (size_t)DG_NOALLOC_MAX_VALUES)
        throw std::runtime_error("ENOMEM: dg_get_aux_fields_noalloc: this solver has " + std::to_string(tot) +
                                 " auxiliary values, the built-in staging array holds " +
                                 std::to_string((size_t)DG_NOALLOC_MAX_VALUES) + "; use dg_get_fields");
    if (tot == 0 || (!fa && !ea)) {                          // J = 0 or no HABC face: nothing to export
        cu(cudaStreamSynchronize(s->stream), "sync");
        return;
    }
    std::lock_guard<std::mutex> hold(g_noalloc_lock);        // until the copy-out is complete: the array is shared
    double* stage = noalloc_stage_address(s->device);
    // every value in [0, tot) is written here before the copies below read it; values beyond tot (left by a
    // larger solver's call) are never read
    k_export_aux<T><<<(unsigned)((tot + 255) / 256), 256, 0, s->stream>>>(d, s->cur, stage, stage + n2);
    try {
        cu(cudaGetLastError(), "export launch");
        if (fa && n2) cu(cudaMemcpyAsync(fa, stage, sizeof(double) * n2, cudaMemcpyDeviceToHost, s->stream), "download");
        if (ea && n1) cu(cudaMemcpyAsync(ea, stage + n2, sizeof(double) * n1, cudaMemcpyDeviceToHost, s->stream), "download");
    } catch (...) {
        cudaStreamSynchronize(s->stream);                    // the lock must outlive whatever was enqueued
        throw;
    }
    cu(cudaStreamSynchronize(s->stream), "sync");
}

}  // namespace

extern "C" int dg_get_aux_fields_noalloc(dg_solver* s, double* face_aux, double* edge_aux) {
    try {
        if (!s) throw std::runtime_error("EINVAL: NULL argument");
        cu(cudaSetDevice(s->device), "cudaSetDevice");
        if (s->precision == 64) export_aux_noalloc<double>(s, s->d64, face_aux, edge_aux);
        else export_aux_noalloc<float>(s, s->d32, face_aux, edge_aux);
        return DG_OK;
    } catch (const std::exception& e) { return err_from_exception(e); }
}
