// arkcos_split.cpp - include/arkcos_split.h: the specified arithmetic of the paper's kernel split
// (Eq. 2.1-2.4).  Host, FP64, no device.  Product code; shares
// nothing with oracle/ or tests/.
#include <cmath>
#include <cstddef>
#include <new>
#include <vector>

#include "../../include/arkcos_split.h"

namespace {
constexpr double kPi = 3.14159265358979323846264338327950288;

// Gauss-Legendre nodes and weights on [-1, 1] by Newton iteration on P_n (n <= 64).
void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
    x.assign(n, 0.0); w.assign(n, 0.0);
    for (int i = 0; i < (n + 1) / 2; i++) {
        double z = std::cos(kPi * (i + 0.75) / (n + 0.5));
        double pp = 1.0;
        for (int it = 0; it < 100; it++) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; j++) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            const double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = -z; x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

bool finite_all(const double* v, size_t n) {
    for (size_t i = 0; i < n; i++) if (!std::isfinite(v[i])) return false;
    return true;
}

// sigma of Eq. 2.2 for one (b_l, l_cut); optionally writes Khat_l, Ktilde_l.
double split_sigma(const double* k_l, const double* b_l, int l_max, int l_cut, int compensate, double alpha,
                   double* khat_l, double* ktilde_l) {
    long double num = 0.0L, den = 0.0L;
    for (int l = 0; l <= l_max; l++) {
        double khat = 0.0;
        if (l <= l_cut) khat = compensate ? k_l[l] - b_l[l] : k_l[l];
        const double ktilde = khat + b_l[l];                         // Eq. 2.1
        const double d = ktilde - k_l[l];
        num += (long double)(2 * l + 1) * d * d;
        den += (long double)(2 * l + 1) * k_l[l] * k_l[l];
        if (khat_l) khat_l[l] = khat;
        if (ktilde_l) ktilde_l[l] = ktilde;
    }
    if (!(den > 0.0L)) return num > 0.0L ? INFINITY : 0.0;
    return alpha * std::sqrt((double)(num / den));                   // Eq. 2.2 (the 1/4pi factors cancel)
}
}  // namespace

extern "C" {

arkcos_status arkcos_table_legendre(const double* k_table, int n_table, double theta_cut, int m_split, double theta_split,
                                    int l_max, double* b_l) {
    if (!k_table || !b_l || n_table < 2 || l_max < 0) return ARKCOS_EINVAL;
    if (!(theta_cut > 0.0) || !(theta_cut <= kPi * (1.0 + 1e-15)) || !finite_all(k_table, (size_t)n_table)) return ARKCOS_EINVAL;
    if (m_split < 0) return ARKCOS_EINVAL;
    if (m_split > 0 && (m_split > n_table - 2 || !(theta_split > 0.0) || !(theta_split < theta_cut))) return ARKCOS_EINVAL;
    try {
        std::vector<long double> acc((size_t)l_max + 1, 0.0L);
        std::vector<double> gx, gw;
        int order_built = 0;
        for (int m = 0; m + 1 < n_table; m++) {
            // cell [ta, tb] between nodes m and m+1 (uniform or two-zone nodes, include/arkcos.h)
            double ta, tb;
            if (m_split == 0) {
                const double h = theta_cut / (n_table - 1);
                ta = m * h; tb = (m + 1) * h;
            } else if (m < m_split) {
                const double h = theta_split / m_split;
                ta = m * h; tb = (m + 1) * h;
            } else {
                const double h = (theta_cut - theta_split) / (n_table - 1 - m_split);
                ta = theta_split + (m - m_split) * h; tb = theta_split + (m + 1 - m_split) * h;
            }
            if (m + 2 == n_table) tb = theta_cut;
            const double h = tb - ta;
            // P_l(cos t) sin t * (linear) has ~ l_max * h / pi half-waves on the cell
            int order = 4 + (int)std::ceil(0.75 * l_max * h);
            if (order > 64) order = 64;
            if (order != order_built) { gauss_legendre(order, gx, gw); order_built = order; }
            // cells wider than the quadrature can resolve are subdivided
            const int sub = 1 + (int)(0.75 * l_max * h / 56.0);
            for (int s = 0; s < sub; s++) {
                const double sa = ta + h * s / sub, sb = ta + h * (s + 1) / sub;
                for (int q = 0; q < order; q++) {
                    const double t = 0.5 * (sa + sb) + 0.5 * (sb - sa) * gx[q];
                    const double f = (t - ta) / h;
                    const double k = (1.0 - f) * k_table[m] + f * k_table[m + 1];
                    const double wq = 0.5 * (sb - sa) * gw[q] * k * std::sin(t);
                    const double x = std::cos(t);
                    double p0 = 1.0, p1 = x;
                    acc[0] += wq;
                    if (l_max >= 1) acc[1] += wq * x;
                    for (int l = 1; l < l_max; l++) {
                        const double p2 = ((2.0 * l + 1.0) * x * p1 - l * p0) / (l + 1.0);
                        acc[(size_t)l + 1] += wq * p2;
                        p0 = p1; p1 = p2;
                    }
                }
            }
        }
        for (int l = 0; l <= l_max; l++) b_l[l] = (double)(2.0L * (long double)kPi * acc[(size_t)l]);
    } catch (const std::bad_alloc&) { return ARKCOS_ENOMEM; }
    return ARKCOS_OK;
}

arkcos_status arkcos_split_error(const double* k_l, const double* b_l, int l_max, int l_cut, int compensate, double alpha,
                                 double* sigma, double* khat_l, double* ktilde_l) {
    if (!k_l || !b_l || !sigma || l_max < 0 || l_cut < -1 || l_cut > l_max || !(alpha >= 0.0) || !std::isfinite(alpha)) return ARKCOS_EINVAL;
    if (compensate != 0 && compensate != 1) return ARKCOS_EINVAL;
    if (!finite_all(k_l, (size_t)l_max + 1) || !finite_all(b_l, (size_t)l_max + 1)) return ARKCOS_EINVAL;
    *sigma = split_sigma(k_l, b_l, l_max, l_cut, compensate, alpha, khat_l, ktilde_l);
    return ARKCOS_OK;
}

arkcos_status arkcos_split_search(const double* k_l, int l_max, int n_cand, const double* theta_cut_arcmin, const double* b_l_cand,
                                  int compensate, double alpha, double bound, const arkcos_cost_model* cost, int* best_cand,
                                  int* best_l_cut, double* best_time_s, double* best_sigma) {
    if (!k_l || !theta_cut_arcmin || !b_l_cand || !cost || !best_cand || !best_l_cut || l_max < 0 || n_cand < 1) return ARKCOS_EINVAL;
    if (compensate != 0 && compensate != 1) return ARKCOS_EINVAL;
    if (!(bound > 0.0) || !(alpha >= 0.0) || !std::isfinite(alpha) || !(cost->cpu_l_ref > 0.0)) return ARKCOS_EINVAL;
    if (!finite_all(k_l, (size_t)l_max + 1) || !finite_all(theta_cut_arcmin, (size_t)n_cand) ||
        !finite_all(b_l_cand, (size_t)n_cand * ((size_t)l_max + 1))) return ARKCOS_EINVAL;
    *best_cand = -1; *best_l_cut = -1;
    double t_best = INFINITY, s_best = INFINITY;
    for (int c = 0; c < n_cand; c++) {
        const double* b = b_l_cand + (size_t)c * ((size_t)l_max + 1);
        const double th = theta_cut_arcmin[c];
        const double t_gpu = cost->gpu_a2 * th * th + cost->gpu_a1 * th + cost->gpu_c;                 // Eq. 2.3 (generalised)
        // smallest l_cut within the bound: the error is not monotone in l_cut in general, so scan
        for (int l_cut = -1; l_cut <= l_max; l_cut++) {
            const double s = split_sigma(k_l, b, l_max, l_cut, compensate, alpha, nullptr, nullptr);
            if (!(s <= bound)) continue;
            const double lc = l_cut < 0 ? 0.0 : (double)l_cut;
            const double t_cpu = cost->cpu_full_s * lc * lc * (double)l_max / (cost->cpu_l_ref * cost->cpu_l_ref * cost->cpu_l_ref);   // Eq. 2.4
            const double t = t_gpu > t_cpu ? t_gpu : t_cpu;                                          // the halves run in parallel (L74)
            if (t < t_best) { t_best = t; s_best = s; *best_cand = c; *best_l_cut = l_cut; }
            break;
        }
    }
    if (best_time_s) *best_time_s = t_best;
    if (best_sigma) *best_sigma = s_best;
    return ARKCOS_OK;
}

}  // extern "C"
