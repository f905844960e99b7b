// pole_search.cpp - host-side pole search of the resonant response (Eq. 6-10).
//
// xi(kappa) ~ sum_j zeta_j / (kappa - eta_j) + regular part (Eq. 6).  With P(kappa) = prod (kappa - eta_j) =
// kappa^Np + sum_{k<Np} p_k kappa^k (Eq. 7), P xi is analytic, so its Nd-th divided difference over any Nd+1 mesh
// points vanishes (Eq. 8): sum_k [sum_i kappa_i^k xi_i w_i] p_k = - sum_i kappa_i^Np xi_i w_i with
// w_i = 1 / prod_{j != i} (kappa_i - kappa_j) (Eq. 9; the paper prints xi_i in the denominator, which annihilates
// P/xi instead - DESIGN.md reading R11 puts it in the numerator).  One equation per sliding window; all
// npts - Nd windows are used, by least squares if more than Np (R13).  Roots = eigenvalues of the companion matrix
// by shifted QR.  Amplitudes by Eq. 10 (upper limit N_p, R12) over the window centred nearest the pole.
// kappa is mapped affinely to t in [-1, 1] before powers are formed (R16).
#include <cmath>
#include <complex>
#include <vector>

#include "gsm.h"

namespace {
typedef std::complex<double> cd;

// least squares min ||M p - r|| by Householder QR; M is rows x cols (row-major), rows >= cols
bool lstsq(std::vector<cd>& M, std::vector<cd>& r, int rows, int cols, std::vector<cd>& p) {
    for (int k = 0; k < cols; ++k) {
        double nrm = 0.0;
        for (int i = k; i < rows; ++i) nrm += std::norm(M[i * cols + k]);
        nrm = std::sqrt(nrm);
        if (nrm == 0.0) return false;
        const cd akk = M[k * cols + k];
        const cd phase = std::abs(akk) > 0.0 ? akk / std::abs(akk) : cd(1.0, 0.0);
        const cd alpha = -phase * nrm;
        std::vector<cd> v(rows - k);
        for (int i = k; i < rows; ++i) v[i - k] = M[i * cols + k];
        v[0] -= alpha;
        double vn = 0.0;
        for (auto& z : v) vn += std::norm(z);
        if (vn == 0.0) continue;
        for (int c = k; c < cols; ++c) {
            cd dot = 0.0;
            for (int i = k; i < rows; ++i) dot += std::conj(v[i - k]) * M[i * cols + c];
            dot *= 2.0 / vn;
            for (int i = k; i < rows; ++i) M[i * cols + c] -= dot * v[i - k];
        }
        cd dot = 0.0;
        for (int i = k; i < rows; ++i) dot += std::conj(v[i - k]) * r[i];
        dot *= 2.0 / vn;
        for (int i = k; i < rows; ++i) r[i] -= dot * v[i - k];
    }
    p.assign(cols, cd(0.0));
    for (int i = cols - 1; i >= 0; --i) {
        cd acc = r[i];
        for (int c = i + 1; c < cols; ++c) acc -= M[i * cols + c] * p[c];
        if (std::abs(M[i * cols + i]) == 0.0) return false;
        p[i] = acc / M[i * cols + i];
    }
    return true;
}

// eigenvalues of an upper Hessenberg complex matrix (n x n, row-major) by single-shift QR with deflation
bool hessenberg_eigs(std::vector<cd> H, int n, std::vector<cd>& ev) {
    ev.assign(n, cd(0.0));
    int hi = n - 1, iter = 0;
    const double eps = 2.220446049250313e-16;
    while (hi >= 0) {
        int l = 0;
        for (int k = hi; k >= 1; --k) {
            const double s = std::abs(H[k * n + k]) + std::abs(H[(k - 1) * n + k - 1]);
            if (std::abs(H[k * n + k - 1]) <= eps * (s > 0.0 ? s : 1.0)) { H[k * n + k - 1] = 0.0; l = k; break; }
        }
        if (l == hi) { ev[hi] = H[hi * n + hi]; --hi; iter = 0; continue; }
        if (++iter > 300) return false;
        // Wilkinson shift: eigenvalue of the trailing 2x2 closer to H[hi][hi]
        const cd a = H[(hi - 1) * n + hi - 1], b = H[(hi - 1) * n + hi], c = H[hi * n + hi - 1], d = H[hi * n + hi];
        const cd tr = a + d, det = a * d - b * c;
        const cd disc = std::sqrt(tr * tr - 4.0 * det);
        const cd m1 = 0.5 * (tr + disc), m2 = 0.5 * (tr - disc);
        cd mu = std::abs(m1 - d) < std::abs(m2 - d) ? m1 : m2;
        if (iter % 11 == 10) mu += cd(std::abs(c), 0.0);   // exceptional shift
        for (int k = l; k <= hi; ++k) H[k * n + k] -= mu;
        std::vector<double> cs(hi - l);
        std::vector<cd> sn(hi - l);
        for (int k = l; k < hi; ++k) {   // QR by Givens: rows k, k+1
            const cd x = H[k * n + k], y = H[(k + 1) * n + k];
            const double r = std::sqrt(std::norm(x) + std::norm(y));
            double cc = 1.0;
            cd ss = 0.0;
            if (r > 0.0) {
                if (std::abs(x) == 0.0) { cc = 0.0; ss = 1.0; }
                else { cc = std::abs(x) / r; ss = (x / std::abs(x)) * std::conj(y) / r; }
            }
            cs[k - l] = cc;
            sn[k - l] = ss;
            for (int col = k; col <= hi; ++col) {
                const cd u = H[k * n + col], v = H[(k + 1) * n + col];
                H[k * n + col] = cc * u + ss * v;
                H[(k + 1) * n + col] = -std::conj(ss) * u + cc * v;
            }
        }
        for (int k = l; k < hi; ++k) {   // RQ: columns k, k+1 times G^H
            const double cc = cs[k - l];
            const cd ss = sn[k - l];
            const int top = k + 1 < hi ? k + 2 : hi;
            for (int row = l; row <= top && row <= hi; ++row) {
                const cd u = H[row * n + k], v = H[row * n + k + 1];
                H[row * n + k] = cc * u + std::conj(ss) * v;
                H[row * n + k + 1] = -ss * u + cc * v;
            }
        }
        for (int k = l; k <= hi; ++k) H[k * n + k] += mu;
    }
    return true;
}
}  // namespace

extern "C" gsm_status gsm_pole_search(int npts, const double* kappa, const double* xi, int Np, int Nd, double kappa_lo,
                                      double kappa_hi, double* eta, double* zeta, int* best) {
    if (!kappa || !xi || !eta || !zeta || Np < 1 || Np > 32 || Nd <= Np || npts < Np + Nd) return GSM_E_INVALID;
    const int S = npts - Nd;
    const double mid = 0.5 * (kappa[0] + kappa[npts - 1]), half = 0.5 * (kappa[npts - 1] - kappa[0]);
    if (!(half > 0.0)) return GSM_E_INVALID;
    std::vector<double> t(npts);
    std::vector<cd> x(npts);
    for (int i = 0; i < npts; ++i) { t[i] = (kappa[i] - mid) / half; x[i] = cd(xi[2 * i], xi[2 * i + 1]); }
    std::vector<cd> M((size_t)S * Np), rhs(S), p;
    double scale = 0.0;
    for (int s = 0; s < S; ++s) {
        rhs[s] = 0.0;
        for (int i = 0; i <= Nd; ++i) {
            double w = 1.0;
            for (int j = 0; j <= Nd; ++j) if (j != i) w *= t[s + i] - t[s + j];
            const cd xw = x[s + i] / w;
            double pw = 1.0;
            for (int k = 0; k < Np; ++k) { M[(size_t)s * Np + k] += pw * xw; pw *= t[s + i]; }
            rhs[s] -= pw * xw;
        }
        for (int k = 0; k < Np; ++k) scale = std::fmax(scale, std::abs(M[(size_t)s * Np + k]));
    }
    if (!(scale > 0.0)) return GSM_E_INVALID;
    for (auto& z : M) z /= scale;
    for (auto& z : rhs) z /= scale;
    if (!lstsq(M, rhs, S, Np, p)) return GSM_E_INVALID;
    std::vector<cd> comp((size_t)Np * Np, cd(0.0)), et;
    for (int i = 1; i < Np; ++i) comp[(size_t)i * Np + i - 1] = 1.0;
    for (int i = 0; i < Np; ++i) comp[(size_t)i * Np + Np - 1] = -p[i];
    if (!hessenberg_eigs(comp, Np, et)) return GSM_NOT_CONVERGED;
    int bidx = -1;
    double bamp = -1.0;
    for (int k = 0; k < Np; ++k) {
        // Eq. 10 over the window whose centre is nearest to Re eta_k
        int near = 0;
        for (int i = 1; i < npts; ++i) if (std::fabs(t[i] - et[k].real()) < std::fabs(t[near] - et[k].real())) near = i;
        int s = near - Nd / 2;
        if (s < 0) s = 0;
        if (s > S - 1) s = S - 1;
        cd acc = 0.0;
        for (int i = 0; i <= Nd; ++i) {
            cd Pi = 1.0, lag = 1.0;
            for (int j = 0; j < Np; ++j) Pi *= t[s + i] - et[j];
            for (int j = 0; j <= Nd; ++j) if (j != i) lag *= (et[k] - t[s + j]) / (t[s + i] - t[s + j]);
            acc += x[s + i] * Pi * lag;
        }
        cd den = 1.0;
        for (int j = 0; j < Np; ++j) if (j != k) den *= et[k] - et[j];
        const cd zt = acc / den;
        const cd e = mid + half * et[k], z = half * zt;
        eta[2 * k] = e.real(); eta[2 * k + 1] = e.imag();
        zeta[2 * k] = z.real(); zeta[2 * k + 1] = z.imag();
        if (e.real() >= kappa_lo && e.real() <= kappa_hi && std::abs(z) > bamp) { bamp = std::abs(z); bidx = k; }
    }
    if (best) *best = bidx;
    return GSM_OK;
}
