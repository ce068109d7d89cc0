// Algebra of the Padé HABC on the host (long double): coefficients c_n (eq (6)), the inverse of
// the 2J x 2J edge system (33a-b)/(36) (L406-408, L462-475) and of the 3J^2 x 3J^2 corner system (35a-c)
// (L447-451), precomputed once as the paper does (L475).
#pragma once
#include <cmath>
#include <vector>

#include "refelem.hpp"

namespace dg {

struct HabcCoef {
    int J = 0;
    std::vector<double> cn;      // [J]
    std::vector<double> Cij;     // [J][J] (1+c_i)/(1+c_i+c_j)
    std::vector<double> Pe, Qe;  // [2J][2J]: [r^{-a}; r^{-b}] = Pe [b^a; b^b] + Qe [r^{+a}; r^{+b}]
    std::vector<double> Gc;      // [3J^2][3J^2]: r^- = Gc r^+, unknown order X[j,k], Y[i,k], Z[i,j]
};

inline HabcCoef make_habc(int J) {
    HabcCoef h;
    h.J = J;
    if (J == 0) return h;
    const ld pi = acosl(-1.0L);
    const int M = 2 * J + 1;
    std::vector<ld> c(J);
    for (int n = 0; n < J; ++n) { ld t = tanl((n + 1) * pi / M); c[n] = t * t; }
    h.cn.resize(J); h.Cij.resize((size_t)J * J);
    for (int i = 0; i < J; ++i) {
        h.cn[i] = (double)c[i];
        for (int j = 0; j < J; ++j) h.Cij[i * J + j] = (double)((1 + c[i]) / (1 + c[i] + c[j]));
    }
    // ---- edge: (M + d_j) r^{-a}_j - sum_i A_ji r^{-b}_i = b^a_j - d_j r^{+a}_j + sum_i A_ji r^{+b}_i   and a<->b, i<->j
    //      d_j = sum_i c_i c_j / (1+c_i+c_j),  A_ji = c_i (1+c_j) / (1+c_i+c_j)
    const int n2 = 2 * J;
    std::vector<ld> L((size_t)n2 * n2, 0), Tm((size_t)n2 * n2, 0);
    for (int j = 0; j < J; ++j) {
        ld dj = 0;
        for (int i = 0; i < J; ++i) dj += c[i] * c[j] / (1 + c[i] + c[j]);
        for (int blk = 0; blk < 2; ++blk) {
            int r = blk * J + j;
            L[(size_t)r * n2 + r] = M + dj;
            Tm[(size_t)r * n2 + r] = -dj;
            for (int i = 0; i < J; ++i) {
                ld A = c[i] * (1 + c[j]) / (1 + c[i] + c[j]);
                int col = (1 - blk) * J + i;
                L[(size_t)r * n2 + col] = -A;
                Tm[(size_t)r * n2 + col] = A;
            }
        }
    }
    std::vector<ld> Li = invert(L, n2);
    h.Pe.resize((size_t)n2 * n2); h.Qe.resize((size_t)n2 * n2);
    for (int r = 0; r < n2; ++r)
        for (int k = 0; k < n2; ++k) {
            ld s = 0;
            for (int q = 0; q < n2; ++q) s += Li[(size_t)r * n2 + q] * Tm[(size_t)q * n2 + k];
            h.Pe[(size_t)r * n2 + k] = (double)Li[(size_t)r * n2 + k];
            h.Qe[(size_t)r * n2 + k] = (double)s;
        }
    // ---- corner: M r^-x_jk = sum_i c_i [ (C_ijk - 1) S^x_jk + C_jki S^y_ik + C_kij S^z_ij ] and cyclic,
    //      C_ijk = (1+c_i)/(1+c_i+c_j+c_k), S = r^- + r^+
    const int JJ = J * J, n3 = 3 * JJ;
    std::vector<ld> Tc((size_t)n3 * n3, 0);
    auto X = [&](int j, int k) { return j * J + k; };
    auto Y = [&](int i, int k) { return JJ + i * J + k; };
    auto Z = [&](int i, int j) { return 2 * JJ + i * J + j; };
    for (int i = 0; i < J; ++i)
        for (int j = 0; j < J; ++j)
            for (int k = 0; k < J; ++k) {
                ld s = 1 + c[i] + c[j] + c[k];
                ld Ci = (1 + c[i]) / s, Cj = (1 + c[j]) / s, Ck = (1 + c[k]) / s;
                Tc[(size_t)X(j, k) * n3 + X(j, k)] += c[i] * (Ci - 1);
                Tc[(size_t)X(j, k) * n3 + Y(i, k)] += c[i] * Cj;
                Tc[(size_t)X(j, k) * n3 + Z(i, j)] += c[i] * Ck;
                Tc[(size_t)Y(i, k) * n3 + X(j, k)] += c[j] * Ci;
                Tc[(size_t)Y(i, k) * n3 + Y(i, k)] += c[j] * (Cj - 1);
                Tc[(size_t)Y(i, k) * n3 + Z(i, j)] += c[j] * Ck;
                Tc[(size_t)Z(i, j) * n3 + X(j, k)] += c[k] * Ci;
                Tc[(size_t)Z(i, j) * n3 + Y(i, k)] += c[k] * Cj;
                Tc[(size_t)Z(i, j) * n3 + Z(i, j)] += c[k] * (Ck - 1);
            }
    std::vector<ld> Lc((size_t)n3 * n3);
    for (int r = 0; r < n3; ++r)
        for (int k = 0; k < n3; ++k) Lc[(size_t)r * n3 + k] = (r == k ? (ld)M : 0.0L) - Tc[(size_t)r * n3 + k];
    std::vector<ld> Lci = invert(Lc, n3);
    h.Gc.resize((size_t)n3 * n3);
    for (int r = 0; r < n3; ++r)
        for (int k = 0; k < n3; ++k) {
            ld s = 0;
            for (int q = 0; q < n3; ++q) s += Lci[(size_t)r * n3 + q] * Tc[(size_t)q * n3 + k];
            h.Gc[(size_t)r * n3 + k] = (double)s;
        }
    return h;
}

}  // namespace dg
