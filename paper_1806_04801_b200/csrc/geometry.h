// Host-side preparation of the plan geometry ("preparation step"): image-cell tables,
// monitoring points, integration nodes.  Plain C++; results are uploaded once to the device.
#pragma once
#include <cmath>
#include <vector>

#include "common.cuh"
#include "hsma.h"

namespace hsma {

inline void reflecting_axes(int kind, bool refl[3]) {
    refl[0] = refl[1] = refl[2] = false;
    if (kind == HSMA_BC_MIRROR_CAVITY) refl[0] = refl[1] = refl[2] = true;
    if (kind == HSMA_BC_SLAB_XY_PERIODIC_Z_MIRROR) refl[2] = true;
}

// Cells |k_a| <= shell[a], minus (if exclude) the cells with all |k_a| <= exclude[a].
// Periodic axis: image = r + kL (Eq.3).  Reflecting axis: image = (-1)^k r + kL,
// weight gamma^|k| with |k| summed over the reflecting axes only (Eq.4; reading G11).
inline std::vector<Cell> make_cells(int kind, const double L[3], const int shell[3], double gamma,
                                    const int* exclude) {
    bool refl[3];
    reflecting_axes(kind, refl);
    std::vector<Cell> out;
    for (int kx = -shell[0]; kx <= shell[0]; ++kx)
        for (int ky = -shell[1]; ky <= shell[1]; ++ky)
            for (int kz = -shell[2]; kz <= shell[2]; ++kz) {
                const int k[3] = {kx, ky, kz};
                if (exclude && std::abs(kx) <= exclude[0] && std::abs(ky) <= exclude[1] && std::abs(kz) <= exclude[2])
                    continue;
                Cell c;
                int order = 0, f[3];
                for (int a = 0; a < 3; ++a) {
                    f[a] = (refl[a] && (std::abs(k[a]) & 1)) ? 1 : 0;
                    if (refl[a]) order += std::abs(k[a]);
                }
                c.sx = k[0] * L[0]; c.sy = k[1] * L[1]; c.sz = k[2] * L[2];
                c.w = order > 0 ? std::pow(gamma, (double)order) : 1.0;
                c.fx = f[0]; c.fy = f[1]; c.fz = f[2];
                c.central = (kx == 0 && ky == 0 && kz == 0) ? 1 : 0;
                out.push_back(c);
            }
    return out;
}

// PAPER.md:82 (reading G7): K points on |x| = R0, latitude sin(theta_i) = (2i-1)/K - 1,
// azimuth 2 pi i omega, omega = (sqrt5 - 1)/2, i = 1..K.
inline std::vector<double> fibonacci_checkpoints(int K, double R0) {
    std::vector<double> x(3 * (size_t)K);
    const double om = (std::sqrt(5.0) - 1.0) / 2.0;
    for (int i = 1; i <= K; ++i) {
        const double s = (2.0 * i - 1.0) / K - 1.0;
        const double c = std::sqrt(1.0 - s * s);
        const double az = 2.0 * i * M_PI * om;
        x[3 * (size_t)(i - 1)] = R0 * c * std::cos(az);
        x[3 * (size_t)(i - 1) + 1] = R0 * c * std::sin(az);
        x[3 * (size_t)(i - 1) + 2] = R0 * s;
    }
    return x;
}

// Deterministic "nearly uniformly distributed" points on the faces normal to the listed axes
// (reading S5b): faces ordered (-x,+x,-y,+y,-z,+z); face f gets floor(K a_f/sum a)
// points, leftovers one each to the first faces; global point n has in-face coordinates
// (frac(1/2 + (n+1) g1) - 1/2) L_u, (frac(1/2 + (n+1) g2) - 1/2) L_v, g = 1/rho, 1/rho^2 (plastic number).
// lower_only: only the faces x_a = -L_a/2 (the face-pair closure).
inline std::vector<double> default_face_points(int K, const double L[3], const bool use_axis[3], bool lower_only = false) {
    const double rho = 1.32471795724474602596;
    const double g1 = 1.0 / rho, g2 = 1.0 / (rho * rho);
    std::vector<int> fa, fs;
    std::vector<double> area;
    double asum = 0.0;
    for (int a = 0; a < 3; ++a)
        if (use_axis[a])
            for (int s = -1; s <= (lower_only ? -1 : 1); s += 2) {
                fa.push_back(a); fs.push_back(s);
                const double ar = L[(a + 1) % 3] * L[(a + 2) % 3];
                area.push_back(ar); asum += ar;
            }
    std::vector<int> cnt(fa.size());
    int tot = 0;
    for (size_t f = 0; f < fa.size(); ++f) { cnt[f] = (int)std::floor(K * area[f] / asum); tot += cnt[f]; }
    for (int f = 0; f < K - tot; ++f) cnt[f] += 1;
    std::vector<double> pts(3 * (size_t)K, 0.0);
    int n = 0;
    for (size_t f = 0; f < fa.size(); ++f) {
        const int a = fa[f];
        int u_ax = -1, v_ax = -1;
        for (int b = 0; b < 3; ++b)
            if (b != a) { if (u_ax < 0) u_ax = b; else v_ax = b; }
        for (int t = 0; t < cnt[f]; ++t) {
            const double u = std::fmod(0.5 + (n + 1) * g1, 1.0), v = std::fmod(0.5 + (n + 1) * g2, 1.0);
            pts[3 * (size_t)n + a] = 0.5 * fs[f] * L[a];
            pts[3 * (size_t)n + u_ax] = (u - 0.5) * L[u_ax];
            pts[3 * (size_t)n + v_ax] = (v - 0.5) * L[v_ax];
            ++n;
        }
    }
    return pts;
}

// Integration nodes on the unit sphere (normals) and weights for radius R.  PAPER.md:122-126.
//   spiral (reading S10): z_j = -1 + (2j+1)/M, cos th = z + sin(pi z)/pi, phi = 2 pi j omega,
//                         w = (4 pi R^2/M)(1 + cos pi z), j = 0..M-1
//   lattice (reading G4): z_j = -1 + 2j/F2, phi_j = pi j F1/F2, nodes at phi_j and phi_j + pi,
//                         w = (2 pi R^2/F2)(1 + cos pi z_j), j = 0..F2;  M = 2(F2+1)
inline bool make_nodes(int M, double R, int rule, std::vector<double>& nrm, std::vector<double>& w) {
    nrm.assign(3 * (size_t)M, 0.0);
    w.assign((size_t)M, 0.0);
    auto put = [&](size_t j, double ct, double ph, double wt) {
        if (ct > 1.0) ct = 1.0;
        if (ct < -1.0) ct = -1.0;
        const double st = std::sqrt(1.0 - ct * ct);
        nrm[3 * j] = st * std::cos(ph); nrm[3 * j + 1] = st * std::sin(ph); nrm[3 * j + 2] = ct;
        w[j] = wt;
    };
    if (rule == HSMA_QUAD_LATTICE) {
        if (M % 2 || M < 4) return false;
        const long long F2 = M / 2 - 1;
        long long a = 1, b = 1;
        while (b < F2) { const long long c = a + b; a = b; b = c; }
        if (b != F2) return false;
        const long long F1 = a;
        for (long long j = 0; j <= F2; ++j) {
            const double z = -1.0 + 2.0 * (double)j / (double)F2;
            const double ct = z + std::sin(M_PI * z) / M_PI;
            const double ph = M_PI * (double)j * (double)F1 / (double)F2;
            const double wt = (2.0 * M_PI * R * R / (double)F2) * (1.0 + std::cos(M_PI * z));
            put(2 * (size_t)j, ct, ph, wt);
            put(2 * (size_t)j + 1, ct, ph + M_PI, wt);
        }
        return true;
    }
    const double om = (std::sqrt(5.0) - 1.0) / 2.0;
    for (int j = 0; j < M; ++j) {
        const double z = -1.0 + (2.0 * j + 1.0) / M;
        put((size_t)j, z + std::sin(M_PI * z) / M_PI, 2.0 * M_PI * j * om,
            (4.0 * M_PI * R * R / M) * (1.0 + std::cos(M_PI * z)));
    }
    return true;
}

}  // namespace hsma
