// md_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU oracle for the hot path of arXiv 1610.03343
// (Fan et al.): Tersoff / Stillinger-Weber energy, force, per-atom virial and
// per-atom heat current, periodic neighbour list, velocity-Verlet.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may call this.  It shares no code with the CUDA path
// (paper_1610_03343_b200/csrc): its own parameter structs, its own layouts
// (atom-major NL[i*K+m]), its own arithmetic.
//
// What is the definition and what is derived (citations are PAPER.md lines):
//  * U      : Eqs. (1)-(6); per-atom U_i = sum_j U_ij/2.
//  * F      : the CONVENTIONAL derivative, Algorithm 1 scatter with Eqs. (7)-(11),
//             NOT the pairwise form the GPU path uses.
//  * P_ij = dU_i/dr_ij : the paper defers the explicit expression to its Ref. [27]
//             (PAPER.md:176).  Here it is obtained by forward-mode automatic
//             differentiation (dual numbers) of the plain function U_i({r_ij}),
//             so no hand-derived formula is shared with the GPU kernels.
//  * W_i, J_i : Eqs. (29), (30), from P_ij.
//  * multi-element Tersoff ("more than one type of atom"): Tersoff's multicomponent form,
//             DESIGN.md reading A17 (per-element parameters, mixing rules, chi_ij); functions tersoff_multi_*.
//  * SW     : not written out in the paper (Ref. [18]); standard
//             Stillinger-Weber form, readings A6/S1-S2.
//  * neighbour predicate, minimum image: DESIGN.md reading A7.
//
// Pins (tests/test_oracle_*.py): Tersoff/SW textbook cohesive energies and
// lattice constants, dimer closed forms, zero force on the perfect lattice,
// sum F = 0, central finite differences of U (forces) and of U_i (P_ij),
// pairwise == conventional (Eqs. 15-16), strain-derivative virial, heat-current
// identities, NVE energy conservation, brute-force neighbour search.
//
// Templated on the real type: double ("f64") and long double ("f80", used to
// tell oracle rounding from GPU rounding).  Inputs/outputs are always double.
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC (see oracle/__init__.py).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---------------------------------------------------------------- parameters
struct TersoffPar { double A, B, lambda, mu, beta, n, c, d, h, R, S; };
struct SWPar { double epsilon, sigma, a, lambda, gamma, A, B, p, q, cos0; };

const long double PI_L = 3.14159265358979323846264338327950288L;

// ------------------------------------------------ minimum image (reading A7)
// Coordinates are in [0, L); |d| < L, so one conditional shift suffices.
inline double min_image(double d, double L) {
    const double h = 0.5 * L;
    if (d > h) d -= L;
    else if (d < -h) d += L;
    return d;
}

// --------------------------------------------------------------- dual numbers
// value + gradient w.r.t. up to NV independent variables (forward-mode AD).
constexpr int MAXM = 40;           // max in-range neighbours handled by the AD path
constexpr int MAXV = 3 * MAXM;

template <class R>
struct Dual {
    R v;
    R g[MAXV];
    int nv;
    Dual() : v(0), nv(0) {}
    Dual(R val, int nvars) : v(val), nv(nvars) { for (int a = 0; a < nv; ++a) g[a] = 0; }
    Dual(const Dual& o) : v(o.v), nv(o.nv) { for (int a = 0; a < nv; ++a) g[a] = o.g[a]; }
    Dual& operator=(const Dual& o) {
        v = o.v; nv = o.nv; for (int a = 0; a < nv; ++a) g[a] = o.g[a]; return *this;
    }
};

template <class R> Dual<R> variable(R val, int index, int nvars) {
    Dual<R> d(val, nvars); d.g[index] = 1; return d;
}
template <class R> Dual<R> operator+(const Dual<R>& a, const Dual<R>& b) {
    Dual<R> r(a.v + b.v, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] + b.g[i]; return r;
}
template <class R> Dual<R> operator-(const Dual<R>& a, const Dual<R>& b) {
    Dual<R> r(a.v - b.v, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] - b.g[i]; return r;
}
template <class R> Dual<R> operator*(const Dual<R>& a, const Dual<R>& b) {
    Dual<R> r(a.v * b.v, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] * b.v + a.v * b.g[i]; return r;
}
template <class R> Dual<R> operator/(const Dual<R>& a, const Dual<R>& b) {
    Dual<R> r(a.v / b.v, a.nv);
    for (int i = 0; i < r.nv; ++i) r.g[i] = (a.g[i] - r.v * b.g[i]) / b.v;
    return r;
}
template <class R> Dual<R> operator+(const Dual<R>& a, R s) { Dual<R> r = a; r.v += s; return r; }
template <class R> Dual<R> operator+(R s, const Dual<R>& a) { return a + s; }
template <class R> Dual<R> operator-(const Dual<R>& a, R s) { Dual<R> r = a; r.v -= s; return r; }
template <class R> Dual<R> operator-(R s, const Dual<R>& a) {
    Dual<R> r(s - a.v, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = -a.g[i]; return r;
}
template <class R> Dual<R> operator*(const Dual<R>& a, R s) {
    Dual<R> r(a.v * s, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] * s; return r;
}
template <class R> Dual<R> operator*(R s, const Dual<R>& a) { return a * s; }
template <class R> Dual<R> operator/(const Dual<R>& a, R s) {
    Dual<R> r(a.v / s, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] / s; return r;
}
template <class R> Dual<R> operator/(R s, const Dual<R>& a) {
    Dual<R> r(s / a.v, a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = -r.v * a.g[i] / a.v; return r;
}
template <class R> Dual<R> sqrt(const Dual<R>& a) {
    Dual<R> r(std::sqrt(a.v), a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] / (2 * r.v); return r;
}
template <class R> Dual<R> exp(const Dual<R>& a) {
    Dual<R> r(std::exp(a.v), a.nv); for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] * r.v; return r;
}
template <class R> Dual<R> cos(const Dual<R>& a) {
    Dual<R> r(std::cos(a.v), a.nv); const R s = -std::sin(a.v);
    for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] * s;
    return r;
}
// a^s for a.v > 0
template <class R> Dual<R> pow(const Dual<R>& a, R s) {
    Dual<R> r(std::pow(a.v, s), a.nv); const R d = s * std::pow(a.v, s - 1);
    for (int i = 0; i < r.nv; ++i) r.g[i] = a.g[i] * d;
    return r;
}
template <class R> inline R value(const Dual<R>& a) { return a.v; }
inline double value(double a) { return a; }
inline long double value(long double a) { return a; }

using std::sqrt; using std::exp; using std::cos; using std::pow;

// ======================================================================
//  Tersoff (Eqs. 1-6; f_C, f_R, f_A: DESIGN.md reading A1)
// ======================================================================
// f_C(r) = 1 (r <= R); 1/2 [1 + cos(pi (r-R)/(S-R))] (R < r < S); 0 (r >= S)
template <class T, class R> T tersoff_fc(const T& r, R Rc, R Sc) {
    if (value(r) <= Rc) return r * R(0) + R(1);
    if (value(r) >= Sc) return r * R(0);
    const R w = R(PI_L) / (Sc - Rc);
    return R(0.5) * (R(1) + cos((r - Rc) * w));
}
template <class R> R tersoff_fc_prime(R r, R Rc, R Sc) {
    if (r <= Rc || r >= Sc) return 0;
    const R w = R(PI_L) / (Sc - Rc);
    return R(-0.5) * w * std::sin((r - Rc) * w);
}
// Eq. (5): g = 1 + c^2/d^2 - c^2/(d^2 + (h - cos)^2)
template <class T, class R> T tersoff_g(const T& cs, R c, R d, R h) {
    const T x = h - cs;
    return (R(1) + c * c / (d * d)) - (c * c) / (d * d + x * x);
}
template <class R> R tersoff_g_prime(R cs, R c, R d, R h) {       // dg/dcos
    const R x = h - cs; const R q = d * d + x * x;
    return R(-2) * c * c * x / (q * q);
}
// Eq. (3): b = (1 + beta^n zeta^n)^(-1/(2n)); zeta = 0 -> b = 1 exactly (reading A8)
template <class T, class R> T tersoff_b(const T& zeta, R beta, R n) {
    if (value(zeta) <= R(0)) return zeta * R(0) + R(1);
    return pow(R(1) + pow(zeta * beta, n), R(-1) / (R(2) * n));
}
template <class R> R tersoff_b_prime(R zeta, R beta, R n) {        // db/dzeta
    if (zeta <= R(0)) return 0;
    const R t = std::pow(beta * zeta, n);
    const R b = std::pow(R(1) + t, R(-1) / (R(2) * n));
    return -b * t / (R(2) * zeta * (R(1) + t));
}

// U_i as a plain function of the M relative vectors r_ij (all of them within range S).
template <class T, class R>
T tersoff_Ui(const TersoffPar& pp, int M, const T* rx, const T* ry, const T* rz) {
    const R A = pp.A, B = pp.B, lam = pp.lambda, mu = pp.mu, beta = pp.beta, n = pp.n;
    const R c = pp.c, d = pp.d, h = pp.h, Rc = pp.R, Sc = pp.S;
    std::vector<T> r(M);
    for (int j = 0; j < M; ++j) r[j] = sqrt(rx[j] * rx[j] + ry[j] * ry[j] + rz[j] * rz[j]);
    T U = r.empty() ? T() : r[0] * R(0);
    for (int j = 0; j < M; ++j) {
        T zeta = r[j] * R(0);
        for (int k = 0; k < M; ++k) {
            if (k == j) continue;
            const T cs = (rx[j] * rx[k] + ry[j] * ry[k] + rz[j] * rz[k]) / (r[j] * r[k]);   // Eq. (6)
            zeta = zeta + tersoff_fc<T, R>(r[k], Rc, Sc) * tersoff_g<T, R>(cs, c, d, h);    // Eq. (4)
        }
        const T b = tersoff_b<T, R>(zeta, beta, n);                                          // Eq. (3)
        const T fR = A * exp(r[j] * (-lam));
        const T fA = B * exp(r[j] * (-mu));
        U = U + R(0.5) * (tersoff_fc<T, R>(r[j], Rc, Sc) * (fR - b * fA));                   // Eq. (2), U_i
    }
    return U;
}

// ======================================================================
//  Stillinger-Weber (S1-S2; per-atom partition: reading A6)
// ======================================================================
template <class T, class R> T sw_V2(const SWPar& pp, const T& r) {
    const R eps = pp.epsilon, sg = pp.sigma, rc = pp.a * pp.sigma;
    const T sr = sg / r;
    return (R(pp.A) * eps) * (R(pp.B) * pow(sr, R(pp.p)) - pow(sr, R(pp.q))) * exp(sg / (r - rc));
}
template <class T, class R> T sw_V3(const SWPar& pp, const T& r1, const T& r2, const T& cs) {
    const R eps = pp.epsilon, sg = pp.sigma, rc = pp.a * pp.sigma, gm = pp.gamma;
    const T dl = cs - R(pp.cos0);
    return (R(pp.lambda) * eps) * (dl * dl) * exp((gm * sg) / (r1 - rc) + (gm * sg) / (r2 - rc));
}
template <class T, class R>
T sw_Ui(const SWPar& pp, int M, const T* rx, const T* ry, const T* rz) {
    std::vector<T> r(M);
    for (int j = 0; j < M; ++j) r[j] = sqrt(rx[j] * rx[j] + ry[j] * ry[j] + rz[j] * rz[j]);
    T U = r.empty() ? T() : r[0] * R(0);
    for (int j = 0; j < M; ++j) U = U + R(0.5) * sw_V2<T, R>(pp, r[j]);
    for (int j = 0; j < M; ++j)
        for (int k = j + 1; k < M; ++k) {
            const T cs = (rx[j] * rx[k] + ry[j] * ry[k] + rz[j] * rz[k]) / (r[j] * r[k]);
            U = U + sw_V3<T, R>(pp, r[j], r[k], cs);
        }
    return U;
}

// ======================================================================
//  Multi-element Tersoff (reading A17 = Tersoff's multicomponent formulation):
//    U_i   = 1/2 sum_j f_C(r_ij; R_ij, S_ij) [ A_ij exp(-lambda_ij r_ij) - b_ij B_ij exp(-mu_ij r_ij) ]
//    b_ij  = chi_ij (1 + beta_i^n_i zeta_ij^n_i)^(-1/(2 n_i))
//    zeta_ij = sum_{k != j} f_C(r_ik; R_ik, S_ik) g_i(theta_ijk),  g_i with c_i, d_i, h_i of the CENTRAL atom
//    mixing: lambda_ij, mu_ij arithmetic means; A_ij, B_ij, R_ij, S_ij geometric means; chi_ii = 1.
// ======================================================================
constexpr int MAXT = 4;
struct TersoffMultiPar {
    int nt;
    TersoffPar el[MAXT];
    double chi[MAXT][MAXT];
};
// blob layout (ctypes): [nt, then nt x 11 element parameters, then nt x nt chi (row-major)]
inline TersoffMultiPar unpack_multi(const double* blob) {
    TersoffMultiPar p;
    p.nt = (int)blob[0];
    for (int t = 0; t < p.nt; ++t) std::memcpy(&p.el[t], blob + 1 + 11 * t, sizeof(TersoffPar));
    for (int a = 0; a < p.nt; ++a)
        for (int b = 0; b < p.nt; ++b) p.chi[a][b] = blob[1 + 11 * p.nt + a * p.nt + b];
    return p;
}
struct MixedPair { double A, B, lam, mu, R, S, chi; };
inline MixedPair mix(const TersoffMultiPar& p, int a, int b) {
    MixedPair m;
    m.A = std::sqrt(p.el[a].A * p.el[b].A); m.B = std::sqrt(p.el[a].B * p.el[b].B);
    m.lam = 0.5 * (p.el[a].lambda + p.el[b].lambda); m.mu = 0.5 * (p.el[a].mu + p.el[b].mu);
    m.R = std::sqrt(p.el[a].R * p.el[b].R); m.S = std::sqrt(p.el[a].S * p.el[b].S);
    m.chi = p.chi[a][b];
    return m;
}

// U_i as a plain function of the M relative vectors r_ij; ti = type of i, tj[a] = type of neighbour a.
// Neighbours beyond their pair's S contribute nothing (f_C = 0), so the caller may pass every listed one.
template <class T, class R>
T tersoff_multi_Ui(const TersoffMultiPar& pp, int ti, int M, const int* tj, const T* rx, const T* ry, const T* rz) {
    const TersoffPar& ci = pp.el[ti];
    std::vector<T> r(M);
    for (int j = 0; j < M; ++j) r[j] = sqrt(rx[j] * rx[j] + ry[j] * ry[j] + rz[j] * rz[j]);
    T U = r.empty() ? T() : r[0] * R(0);
    for (int j = 0; j < M; ++j) {
        const MixedPair mj = mix(pp, ti, tj[j]);
        T zeta = r[j] * R(0);
        for (int k = 0; k < M; ++k) {
            if (k == j) continue;
            const MixedPair mk = mix(pp, ti, tj[k]);
            const T cs = (rx[j] * rx[k] + ry[j] * ry[k] + rz[j] * rz[k]) / (r[j] * r[k]);
            zeta = zeta + tersoff_fc<T, R>(r[k], R(mk.R), R(mk.S)) * tersoff_g<T, R>(cs, R(ci.c), R(ci.d), R(ci.h));
        }
        const T b = R(mj.chi) * tersoff_b<T, R>(zeta, R(ci.beta), R(ci.n));
        const T fR = R(mj.A) * exp(r[j] * R(-mj.lam));
        const T fA = R(mj.B) * exp(r[j] * R(-mj.mu));
        U = U + R(0.5) * (tersoff_fc<T, R>(r[j], R(mj.R), R(mj.S)) * (fR - b * fA));
    }
    return U;
}

// ======================================================================
//  Neighbour lists (predicate: DESIGN.md reading A7)
// ======================================================================
// strict d2 < r_list^2 with d2 = fma(dz,dz, fma(dy,dy, dx*dx)), dx = min_image(xj - xi)
inline bool is_neighbour(const double* x, const double* y, const double* z, int64_t i, int64_t j,
                         const double* box, double rc2) {
    const double dx = min_image(x[j] - x[i], box[0]);
    const double dy = min_image(y[j] - y[i], box[1]);
    const double dz = min_image(z[j] - z[i], box[2]);
    const double d2 = std::fma(dz, dz, std::fma(dy, dy, dx * dx));
    return d2 < rc2;
}

// O(N^2) all pairs.  Rows sorted by j.  Returns the largest row length, or -1 if a row exceeds K.
int neighbours_brute(int64_t n, const double* x, const double* y, const double* z,
                     const double* box, double r_list, int K, int32_t* NN, int32_t* NL) {
    const double rc2 = r_list * r_list;
    int maxc = 0;
    for (int64_t i = 0; i < n; ++i) {
        int c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            if (is_neighbour(x, y, z, i, j, box, rc2)) {
                if (c >= K) return -1;
                NL[i * K + c++] = (int32_t)j;
            }
        }
        NN[i] = c;
        maxc = std::max(maxc, c);
    }
    return maxc;
}

// Plain cell list (cells of edge >= r_list, 27-cell search).  Falls back to all pairs when
// an axis has fewer than 3 cells.
int neighbours_cell(int64_t n, const double* x, const double* y, const double* z,
                    const double* box, double r_list, int K, int32_t* NN, int32_t* NL) {
    int nc[3];
    for (int a = 0; a < 3; ++a) nc[a] = (int)std::floor(box[a] / r_list);
    if (nc[0] < 3 || nc[1] < 3 || nc[2] < 3) return neighbours_brute(n, x, y, z, box, r_list, K, NN, NL);
    const double rc2 = r_list * r_list;
    const int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    std::vector<std::vector<int32_t>> cells(ncell);
    auto cell_of = [&](double c, int a) {
        int k = (int)std::floor(c / box[a] * nc[a]);
        if (k < 0) k = 0;
        if (k >= nc[a]) k = nc[a] - 1;
        return k;
    };
    for (int64_t i = 0; i < n; ++i) {
        const int cx = cell_of(x[i], 0), cy = cell_of(y[i], 1), cz = cell_of(z[i], 2);
        cells[((int64_t)cx * nc[1] + cy) * nc[2] + cz].push_back((int32_t)i);
    }
    int maxc = 0;
    for (int64_t i = 0; i < n; ++i) {
        const int cx = cell_of(x[i], 0), cy = cell_of(y[i], 1), cz = cell_of(z[i], 2);
        int c = 0;
        for (int ox = -1; ox <= 1; ++ox)
            for (int oy = -1; oy <= 1; ++oy)
                for (int oz = -1; oz <= 1; ++oz) {
                    const int ax = (cx + ox + nc[0]) % nc[0], ay = (cy + oy + nc[1]) % nc[1],
                              az = (cz + oz + nc[2]) % nc[2];
                    for (int32_t j : cells[((int64_t)ax * nc[1] + ay) * nc[2] + az]) {
                        if (j == i) continue;
                        if (is_neighbour(x, y, z, i, j, box, rc2)) {
                            if (c >= K) return -1;
                            NL[i * K + c++] = j;
                        }
                    }
                }
        std::sort(NL + i * K, NL + i * K + c);
        NN[i] = c;
        maxc = std::max(maxc, c);
    }
    return maxc;
}

// ======================================================================
//  Local geometry (O2): in-range neighbours of atom i
// ======================================================================
template <class R> struct Local {
    int M = 0;
    int slot[MAXM];        // position m in row i of the list
    int32_t idx[MAXM];     // atom index j
    int type[MAXM];        // element of j (multi-element Tersoff; 0 otherwise)
    R rx[MAXM], ry[MAXM], rz[MAXM], r[MAXM];
};

template <class R>
bool gather_local(Local<R>& loc, int64_t i, const double* x, const double* y, const double* z,
                  const double* box, const int32_t* NN, const int32_t* NL, int K, double r_force,
                  const int32_t* types = nullptr) {
    loc.M = 0;
    for (int m = 0; m < NN[i]; ++m) {
        const int32_t j = NL[i * K + m];
        const R dx = min_image(x[j] - x[i], box[0]);      // r_ij = r_j - r_i
        const R dy = min_image(y[j] - y[i], box[1]);
        const R dz = min_image(z[j] - z[i], box[2]);
        const R r = std::sqrt(dx * dx + dy * dy + dz * dz);
        if (!(r < R(r_force))) continue;
        if (loc.M >= MAXM) return false;
        const int a = loc.M++;
        loc.slot[a] = m; loc.idx[a] = j; loc.rx[a] = dx; loc.ry[a] = dy; loc.rz[a] = dz; loc.r[a] = r;
        loc.type[a] = types ? types[j] : 0;
    }
    return true;
}

// ======================================================================
//  Conventional forces: Algorithm 1 with Eqs. (7)-(11)
// ======================================================================
template <class R>
void tersoff_conventional_atom(const TersoffPar& pp, const Local<R>& L, int64_t i, R* F, int64_t n) {
    const R A = pp.A, B = pp.B, lam = pp.lambda, mu = pp.mu, beta = pp.beta, nn = pp.n;
    const R c = pp.c, d = pp.d, h = pp.h, Rc = pp.R, Sc = pp.S;
    for (int ja = 0; ja < L.M; ++ja) {
        const int64_t j = L.idx[ja];
        const R rij = L.r[ja];
        const R ex = L.rx[ja] / rij, ey = L.ry[ja] / rij, ez = L.rz[ja] / rij;
        const R fc = tersoff_fc<R, R>(rij, Rc, Sc), fcp = tersoff_fc_prime<R>(rij, Rc, Sc);
        const R fR = A * std::exp(-lam * rij), fA = B * std::exp(-mu * rij);
        R zeta = 0;
        for (int ka = 0; ka < L.M; ++ka) {
            if (ka == ja) continue;
            const R cs = (L.rx[ja] * L.rx[ka] + L.ry[ja] * L.ry[ka] + L.rz[ja] * L.rz[ka]) / (rij * L.r[ka]);
            zeta += tersoff_fc<R, R>(L.r[ka], Rc, Sc) * tersoff_g<R, R>(cs, c, d, h);
        }
        const R b = tersoff_b<R, R>(zeta, beta, nn), bp = tersoff_b_prime<R>(zeta, beta, nn);
        // Eqs. (7), (8): two-body part at fixed b; d/dr_i = -d/dr_ij, d/dr_j = +d/dr_ij
        const R D = R(0.5) * ((fcp * fR - lam * fc * fR) - b * (fcp * fA - mu * fc * fA));
        F[0 * n + i] += D * ex; F[1 * n + i] += D * ey; F[2 * n + i] += D * ez;
        F[0 * n + j] -= D * ex; F[1 * n + j] -= D * ey; F[2 * n + j] -= D * ez;
        // Eqs. (9)-(11): F_x^(ijk) = 1/2 fC(r_ij) fA(r_ij) b'_ij d/dr_x [ fC(r_ik) g_ijk ]
        const R qp = R(0.5) * fc * fA * bp;
        for (int ka = 0; ka < L.M; ++ka) {
            if (ka == ja) continue;
            const int64_t k = L.idx[ka];
            const R rik = L.r[ka];
            const R kx = L.rx[ka] / rik, ky = L.ry[ka] / rik, kz = L.rz[ka] / rik;
            const R cs = ex * kx + ey * ky + ez * kz;
            const R fck = tersoff_fc<R, R>(rik, Rc, Sc), fckp = tersoff_fc_prime<R>(rik, Rc, Sc);
            const R g = tersoff_g<R, R>(cs, c, d, h), gp = tersoff_g_prime<R>(cs, c, d, h);
            // d/dr_j [fC(r_ik) g] = fC(r_ik) g' dcos/dr_ij ; dcos/dr_ij = (e_ik - cos e_ij)/r_ij
            const R ajx = fck * gp * (kx - cs * ex) / rij, ajy = fck * gp * (ky - cs * ey) / rij,
                    ajz = fck * gp * (kz - cs * ez) / rij;
            // d/dr_k [fC(r_ik) g] = fC'(r_ik) g e_ik + fC(r_ik) g' (e_ij - cos e_ik)/r_ik
            const R ckx = fckp * g * kx + fck * gp * (ex - cs * kx) / rik,
                    cky = fckp * g * ky + fck * gp * (ey - cs * ky) / rik,
                    ckz = fckp * g * kz + fck * gp * (ez - cs * kz) / rik;
            F[0 * n + j] += qp * ajx; F[1 * n + j] += qp * ajy; F[2 * n + j] += qp * ajz;       // Eq. (10)
            F[0 * n + k] += qp * ckx; F[1 * n + k] += qp * cky; F[2 * n + k] += qp * ckz;       // Eq. (11)
            F[0 * n + i] -= qp * (ajx + ckx); F[1 * n + i] -= qp * (ajy + cky);                 // Eq. (9)
            F[2 * n + i] -= qp * (ajz + ckz);
        }
    }
}

// Algorithm 1 for the multi-element form: the same scatter, with the pair's mixed parameters in f_C, f_R, f_A
// (pair i-j for the bond, pair i-k inside zeta) and the central atom's in g and b.
template <class R>
void tersoff_multi_conventional_atom(const TersoffMultiPar& pp, int ti, const Local<R>& L, int64_t i, R* F, int64_t n) {
    const TersoffPar& ci = pp.el[ti];
    const R beta = ci.beta, nn = ci.n, c = ci.c, d = ci.d, h = ci.h;
    for (int ja = 0; ja < L.M; ++ja) {
        const MixedPair mj = mix(pp, ti, L.type[ja]);
        const int64_t j = L.idx[ja];
        const R rij = L.r[ja];
        const R ex = L.rx[ja] / rij, ey = L.ry[ja] / rij, ez = L.rz[ja] / rij;
        const R fc = tersoff_fc<R, R>(rij, R(mj.R), R(mj.S)), fcp = tersoff_fc_prime<R>(rij, R(mj.R), R(mj.S));
        const R fR = R(mj.A) * std::exp(-R(mj.lam) * rij), fA = R(mj.B) * std::exp(-R(mj.mu) * rij);
        R zeta = 0;
        for (int ka = 0; ka < L.M; ++ka) {
            if (ka == ja) continue;
            const MixedPair mk = mix(pp, ti, L.type[ka]);
            const R cs = (L.rx[ja] * L.rx[ka] + L.ry[ja] * L.ry[ka] + L.rz[ja] * L.rz[ka]) / (rij * L.r[ka]);
            zeta += tersoff_fc<R, R>(L.r[ka], R(mk.R), R(mk.S)) * tersoff_g<R, R>(cs, c, d, h);
        }
        const R b = R(mj.chi) * tersoff_b<R, R>(zeta, beta, nn), bp = R(mj.chi) * tersoff_b_prime<R>(zeta, beta, nn);
        const R D = R(0.5) * ((fcp * fR - R(mj.lam) * fc * fR) - b * (fcp * fA - R(mj.mu) * fc * fA));
        F[0 * n + i] += D * ex; F[1 * n + i] += D * ey; F[2 * n + i] += D * ez;
        F[0 * n + j] -= D * ex; F[1 * n + j] -= D * ey; F[2 * n + j] -= D * ez;
        const R qp = R(0.5) * fc * fA * bp;
        for (int ka = 0; ka < L.M; ++ka) {
            if (ka == ja) continue;
            const MixedPair mk = mix(pp, ti, L.type[ka]);
            const int64_t k = L.idx[ka];
            const R rik = L.r[ka];
            const R kx = L.rx[ka] / rik, ky = L.ry[ka] / rik, kz = L.rz[ka] / rik;
            const R cs = ex * kx + ey * ky + ez * kz;
            const R fck = tersoff_fc<R, R>(rik, R(mk.R), R(mk.S)), fckp = tersoff_fc_prime<R>(rik, R(mk.R), R(mk.S));
            const R g = tersoff_g<R, R>(cs, c, d, h), gp = tersoff_g_prime<R>(cs, c, d, h);
            const R ajx = fck * gp * (kx - cs * ex) / rij, ajy = fck * gp * (ky - cs * ey) / rij,
                    ajz = fck * gp * (kz - cs * ez) / rij;
            const R ckx = fckp * g * kx + fck * gp * (ex - cs * kx) / rik,
                    cky = fckp * g * ky + fck * gp * (ey - cs * ky) / rik,
                    ckz = fckp * g * kz + fck * gp * (ez - cs * kz) / rik;
            F[0 * n + j] += qp * ajx; F[1 * n + j] += qp * ajy; F[2 * n + j] += qp * ajz;
            F[0 * n + k] += qp * ckx; F[1 * n + k] += qp * cky; F[2 * n + k] += qp * ckz;
            F[0 * n + i] -= qp * (ajx + ckx); F[1 * n + i] -= qp * (ajy + cky);
            F[2 * n + i] -= qp * (ajz + ckz);
        }
    }
}

template <class R> R sw_V2_prime(const SWPar& pp, R r) {
    const R eps = pp.epsilon, sg = pp.sigma, rc = pp.a * pp.sigma, p = pp.p, q = pp.q;
    const R sp = std::pow(sg / r, p), sq = std::pow(sg / r, q);
    const R e = std::exp(sg / (r - rc));
    return R(pp.A) * eps * e * ((-p * R(pp.B) * sp + q * sq) / r - (R(pp.B) * sp - sq) * sg / ((r - rc) * (r - rc)));
}

// Conventional SW: differentiate sum V2 + sum V3 w.r.t. the atoms of each pair / triplet directly.
template <class R>
void sw_conventional_atom(const SWPar& pp, const Local<R>& L, int64_t i, R* F, int64_t n) {
    const R eps = pp.epsilon, sg = pp.sigma, rc = pp.a * pp.sigma, gm = pp.gamma;
    for (int ja = 0; ja < L.M; ++ja) {                       // ordered pairs: each carries V2/2
        const int64_t j = L.idx[ja];
        const R r = L.r[ja];
        const R D = R(0.5) * sw_V2_prime<R>(pp, r);
        const R ex = L.rx[ja] / r, ey = L.ry[ja] / r, ez = L.rz[ja] / r;
        F[0 * n + i] += D * ex; F[1 * n + i] += D * ey; F[2 * n + i] += D * ez;
        F[0 * n + j] -= D * ex; F[1 * n + j] -= D * ey; F[2 * n + j] -= D * ez;
    }
    for (int ja = 0; ja < L.M; ++ja)
        for (int ka = ja + 1; ka < L.M; ++ka) {              // triplet centred on i
            const int64_t j = L.idx[ja], k = L.idx[ka];
            const R r1 = L.r[ja], r2 = L.r[ka];
            const R ex = L.rx[ja] / r1, ey = L.ry[ja] / r1, ez = L.rz[ja] / r1;
            const R kx = L.rx[ka] / r2, ky = L.ry[ka] / r2, kz = L.rz[ka] / r2;
            const R cs = ex * kx + ey * ky + ez * kz;
            const R dl = cs - R(pp.cos0);
            const R E = R(pp.lambda) * eps * std::exp(gm * sg / (r1 - rc) + gm * sg / (r2 - rc));
            const R V3 = E * dl * dl;
            const R a1 = -gm * sg / ((r1 - rc) * (r1 - rc)), a2 = -gm * sg / ((r2 - rc) * (r2 - rc));
            // dV3/dr_ij and dV3/dr_ik (vectors)
            const R g1x = V3 * a1 * ex + R(2) * E * dl * (kx - cs * ex) / r1,
                    g1y = V3 * a1 * ey + R(2) * E * dl * (ky - cs * ey) / r1,
                    g1z = V3 * a1 * ez + R(2) * E * dl * (kz - cs * ez) / r1;
            const R g2x = V3 * a2 * kx + R(2) * E * dl * (ex - cs * kx) / r2,
                    g2y = V3 * a2 * ky + R(2) * E * dl * (ey - cs * ky) / r2,
                    g2z = V3 * a2 * kz + R(2) * E * dl * (ez - cs * kz) / r2;
            F[0 * n + j] -= g1x; F[1 * n + j] -= g1y; F[2 * n + j] -= g1z;
            F[0 * n + k] -= g2x; F[1 * n + k] -= g2y; F[2 * n + k] -= g2z;
            F[0 * n + i] += g1x + g2x; F[1 * n + i] += g1y + g2y; F[2 * n + i] += g1z + g2z;
        }
}

// ======================================================================
//  One evaluation: U_i, conventional F_i, P_ij (AD), pairwise F_i, W_i, J_i
// ======================================================================
enum { POT_TERSOFF = 0, POT_SW = 1, POT_TERSOFF_MULTI = 2 };

// Atoms i0 <= i < i1 only (the whole system: 0, n).  A proper sub-range serves bench.py's all-core timing
// entry: the same per-atom functions, called by several threads on disjoint ranges, each with its own
// force buffer because Algorithm 1 scatters to j and k; the per-pair outputs (f_pair,
// virial, heat, P_out), which need every atom's P, are then not available and must be NULL.
template <class R>
int evaluate(int pot, const void* par, int64_t n, const double* x, const double* y, const double* z,
             const double* vx, const double* vy, const double* vz, const double* box,
             const int32_t* NN, const int32_t* NL, int K,
             double* pe, double* f_conv, double* f_pair, double* virial, double* heat, double* P_out,
             int64_t i0, int64_t i1, const int32_t* types = nullptr) {
    const TersoffPar* tp = (const TersoffPar*)par;
    const SWPar* sp = (const SWPar*)par;
    TersoffMultiPar mp;
    double r_force = 0;
    if (pot == POT_TERSOFF) r_force = tp->S;
    else if (pot == POT_SW) r_force = sp->a * sp->sigma;
    else {                                                   // every pair inside the largest S; f_C sorts out the rest
        if (!types) return -6;
        mp = unpack_multi((const double*)par);
        for (int t = 0; t < mp.nt; ++t) r_force = std::max(r_force, mp.el[t].S);
    }
    const bool whole = i0 == 0 && i1 == n;
    const bool need_P = P_out || f_pair || virial || heat;
    if (need_P && !whole) return -4;
    std::vector<R> F((size_t)3 * n, R(0));
    std::vector<R> P(need_P ? (size_t)3 * n * K : (size_t)3 * K, R(0));   // P[(i*K+m)*3+a] = dU_i/dr_ij^a, j = NL[i*K+m]
    Local<R> L;
    std::vector<Dual<R>> vxr(MAXM), vyr(MAXM), vzr(MAXM);
    for (int64_t i = i0; i < i1; ++i) {
        if (!gather_local<R>(L, i, x, y, z, box, NN, NL, K, r_force, types)) return -2;
        // conventional forces (Algorithm 1)
        if (pot == POT_TERSOFF) tersoff_conventional_atom<R>(*tp, L, i, F.data(), n);
        else if (pot == POT_SW) sw_conventional_atom<R>(*sp, L, i, F.data(), n);
        else tersoff_multi_conventional_atom<R>(mp, types[i], L, i, F.data(), n);
        // U_i and P_ij = dU_i/dr_ij by forward-mode AD of the plain U_i({r_ij})
        const int nv = 3 * L.M;
        for (int a = 0; a < L.M; ++a) {
            vxr[a] = variable<R>(L.rx[a], 3 * a + 0, nv);
            vyr[a] = variable<R>(L.ry[a], 3 * a + 1, nv);
            vzr[a] = variable<R>(L.rz[a], 3 * a + 2, nv);
        }
        Dual<R> Ui = pot == POT_TERSOFF
            ? tersoff_Ui<Dual<R>, R>(*tp, L.M, vxr.data(), vyr.data(), vzr.data())
            : pot == POT_SW ? sw_Ui<Dual<R>, R>(*sp, L.M, vxr.data(), vyr.data(), vzr.data())
            : tersoff_multi_Ui<Dual<R>, R>(mp, types[i], L.M, L.type, vxr.data(), vyr.data(), vzr.data());
        if (pe) pe[i] = (double)Ui.v;
        const size_t row = need_P ? (size_t)i * K : 0;     // without per-pair outputs one row of scratch is reused
        for (int a = 0; a < L.M; ++a)
            for (int q = 0; q < 3; ++q) P[(row + L.slot[a]) * 3 + q] = Ui.g[3 * a + q];
    }
    if (f_conv) for (size_t q = 0; q < (size_t)3 * n; ++q) f_conv[q] = (double)F[q];
    if (P_out) for (size_t q = 0; q < (size_t)3 * n * K; ++q) P_out[q] = (double)P[q];
    if (!need_P) return 0;
    // per-atom outputs, Eqs. (28)-(30)
    for (int64_t i = 0; i < n; ++i) {
        R fp[3] = {0, 0, 0}, W[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, J[3] = {0, 0, 0};
        for (int m = 0; m < NN[i]; ++m) {
            const int32_t j = NL[i * K + m];
            int mm = -1;
            for (int q = 0; q < NN[j]; ++q) if (NL[j * K + q] == i) { mm = q; break; }
            if (mm < 0) return -3;                                     // list must be symmetric
            const R rij[3] = {R(min_image(x[j] - x[i], box[0])), R(min_image(y[j] - y[i], box[1])),
                              R(min_image(z[j] - z[i], box[2]))};
            const R* Pij = &P[((size_t)i * K + m) * 3];
            const R* Pji = &P[((size_t)j * K + mm) * 3];
            R Fij[3];
            for (int b = 0; b < 3; ++b) { Fij[b] = Pij[b] - Pji[b]; fp[b] += Fij[b]; }   // Eq. (28)
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) W[3 * a + b] -= R(0.5) * rij[a] * Fij[b];     // Eq. (29)
            if (vx) {
                const R dot = Pji[0] * R(vx[i]) + Pji[1] * R(vy[i]) + Pji[2] * R(vz[i]);
                for (int a = 0; a < 3; ++a) J[a] += rij[a] * dot;                         // Eq. (30)
            }
        }
        if (f_pair) for (int b = 0; b < 3; ++b) f_pair[b * n + i] = (double)fp[b];
        if (virial) for (int q = 0; q < 9; ++q) virial[q * n + i] = (double)W[q];
        if (heat) for (int a = 0; a < 3; ++a) heat[a * n + i] = (double)J[a];
    }
    return 0;
}

// velocity-Verlet half steps; kappa converts eV/A/amu to A/fs^2
const double KAPPA_ACC = 9.648533215665e-3;

void vv_kick_drift(int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                   const double* f, double mass, double dt, const double* box) {
    const double hk = 0.5 * dt * KAPPA_ACC / mass;
    double* X[3] = {x, y, z}; double* V[3] = {vx, vy, vz};
    for (int a = 0; a < 3; ++a)
        for (int64_t i = 0; i < n; ++i) {
            V[a][i] += hk * f[a * n + i];
            double c = X[a][i] + dt * V[a][i];
            c -= box[a] * std::floor(c / box[a]);
            if (c >= box[a] || c < 0.0) c = 0.0;          // reading A8
            X[a][i] = c;
        }
}
void vv_kick(int64_t n, double* vx, double* vy, double* vz, const double* f, double mass, double dt) {
    const double hk = 0.5 * dt * KAPPA_ACC / mass;
    double* V[3] = {vx, vy, vz};
    for (int a = 0; a < 3; ++a)
        for (int64_t i = 0; i < n; ++i) V[a][i] += hk * f[a * n + i];
}

}  // namespace

// ======================================================================
//  C exports (ctypes).  All arrays are host double / int32, SoA [3][n], [9][n].
// ======================================================================
extern "C" {

int oracle_neighbors_brute(int64_t n, const double* x, const double* y, const double* z, const double* box,
                           double r_list, int K, int32_t* NN, int32_t* NL) {
    return neighbours_brute(n, x, y, z, box, r_list, K, NN, NL);
}
int oracle_neighbors_cell(int64_t n, const double* x, const double* y, const double* z, const double* box,
                          double r_list, int K, int32_t* NN, int32_t* NL) {
    return neighbours_cell(n, x, y, z, box, r_list, K, NN, NL);
}

// pot: 0 Tersoff (par -> 11 doubles A,B,lambda,mu,beta,n,c,d,h,R,S), 1 SW (10 doubles
// epsilon,sigma,a,lambda,gamma,A,B,p,q,cos0).  precision: 0 double, 1 long double.
// Any output pointer may be NULL.  P_out is [n][K][3].
int oracle_evaluate(int pot, const double* par, int precision, int64_t n,
                    const double* x, const double* y, const double* z,
                    const double* vx, const double* vy, const double* vz, const double* box,
                    const int32_t* NN, const int32_t* NL, int K,
                    double* pe, double* f_conv, double* f_pair, double* virial, double* heat, double* P_out) {
    if (precision == 1)
        return evaluate<long double>(pot, par, n, x, y, z, vx, vy, vz, box, NN, NL, K,
                                     pe, f_conv, f_pair, virial, heat, P_out, 0, n);
    return evaluate<double>(pot, par, n, x, y, z, vx, vy, vz, box, NN, NL, K,
                            pe, f_conv, f_pair, virial, heat, P_out, 0, n);
}

// Multi-element Tersoff (pot = 2): par = [nt, nt x 11 element parameters, nt x nt chi], types[n] in 0..nt-1.
int oracle_evaluate_multi(const double* par, int precision, int64_t n,
                          const double* x, const double* y, const double* z,
                          const double* vx, const double* vy, const double* vz, const double* box,
                          const int32_t* types, const int32_t* NN, const int32_t* NL, int K,
                          double* pe, double* f_conv, double* f_pair, double* virial, double* heat, double* P_out) {
    if (precision == 1)
        return evaluate<long double>(POT_TERSOFF_MULTI, par, n, x, y, z, vx, vy, vz, box, NN, NL, K,
                                     pe, f_conv, f_pair, virial, heat, P_out, 0, n, types);
    return evaluate<double>(POT_TERSOFF_MULTI, par, n, x, y, z, vx, vy, vz, box, NN, NL, K,
                            pe, f_conv, f_pair, virial, heat, P_out, 0, n, types);
}
// U_i of one atom of element ti from explicit relative vectors and neighbour elements (finite-difference pin)
double oracle_atom_energy_multi(const double* par, int ti, int M, const int32_t* tj, const double* rx,
                                const double* ry, const double* rz) {
    std::vector<long double> a(rx, rx + M), b(ry, ry + M), c(rz, rz + M);
    std::vector<int> t(tj, tj + M);
    return (double)tersoff_multi_Ui<long double, long double>(unpack_multi(par), ti, M, t.data(), a.data(), b.data(), c.data());
}

// U_i (pe[i], i0 <= i < i1; other entries untouched) and the conventional forces these atoms' terms scatter
// (f_conv[3][n], overwritten: zero except where atoms of the range, their neighbours and their neighbours'
// partners receive a contribution).  For the threaded timing entry of bench.py; see evaluate().
int oracle_evaluate_range(int pot, const double* par, int64_t n, const double* x, const double* y, const double* z,
                          const double* box, const int32_t* NN, const int32_t* NL, int K,
                          int64_t i0, int64_t i1, double* pe, double* f_conv) {
    if (i0 < 0 || i1 > n || i0 > i1) return -5;
    return evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN, NL, K,
                            pe, f_conv, nullptr, nullptr, nullptr, nullptr, i0, i1);
}

// U_i of one atom from explicit relative vectors (for the finite-difference pin of P_ij)
double oracle_atom_energy(int pot, const double* par, int M, const double* rx, const double* ry, const double* rz) {
    std::vector<long double> a(rx, rx + M), b(ry, ry + M), c(rz, rz + M);
    if (pot == POT_TERSOFF)
        return (double)tersoff_Ui<long double, long double>(*(const TersoffPar*)par, M, a.data(), b.data(), c.data());
    return (double)sw_Ui<long double, long double>(*(const SWPar*)par, M, a.data(), b.data(), c.data());
}

void oracle_vv_kick_drift(int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                          const double* f, double mass, double dt, const double* box) {
    vv_kick_drift(n, x, y, z, vx, vy, vz, f, mass, dt, box);
}
void oracle_vv_kick(int64_t n, double* vx, double* vy, double* vz, const double* f, double mass, double dt) {
    vv_kick(n, vx, vy, vz, f, mass, dt);
}

// NVE loop: nsteps velocity-Verlet steps, list rebuilt every `rebuild_every` steps (cell list,
// r_list).  f must hold the forces of the incoming state if f_valid != 0.  Records the total
// potential energy after each step in pe_trace[nsteps] (may be NULL).  Returns 0 or <0.
int oracle_nve_run(int pot, const double* par, int64_t n, double* x, double* y, double* z,
                   double* vx, double* vy, double* vz, const double* box, double mass, double dt,
                   int nsteps, int rebuild_every, double r_list, int K, double* f, int f_valid,
                   double* pe, double* pe_trace) {
    std::vector<int32_t> NN(n), NL((size_t)n * K);
    std::vector<double> pe_loc(n);
    double* pe_use = pe ? pe : pe_loc.data();
    if (!f_valid) {
        if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        int rc = evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                                  pe_use, f, nullptr, nullptr, nullptr, nullptr, 0, n);
        if (rc) return rc;
    }
    for (int s = 0; s < nsteps; ++s) {
        vv_kick_drift(n, x, y, z, vx, vy, vz, f, mass, dt, box);
        if (s % rebuild_every == 0 || !f_valid)
            if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        f_valid = 1;
        int rc = evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                                  pe_use, f, nullptr, nullptr, nullptr, nullptr, 0, n);
        if (rc) return rc;
        vv_kick(n, vx, vy, vz, f, mass, dt);
        if (pe_trace) { long double s2 = 0; for (int64_t i = 0; i < n; ++i) s2 += pe_use[i]; pe_trace[s] = (double)s2; }
    }
    return 0;
}

// NVE with the total heat current sampled every `sample_every` steps (the Green-Kubo workload of the paper's
// Ref. [27]).  After the step's second half-kick:
//   J_pot = sum_i J_i,  J_i = sum_j r_ij (dU_j/dr_ji . v_i)                 (Eq. 30 / Eq. 25)
//   J_kin = sum_i (1/2 m v_i^2 + U_i) v_i                                    (convective part, reading A12)
// J_pot[ns][3], J_kin[ns][3] (either may be NULL), ns = number of steps s with (s + 1) % sample_every == 0.
int oracle_nve_heat_run(int pot, const double* par, int64_t n, double* x, double* y, double* z,
                        double* vx, double* vy, double* vz, const double* box, double mass, double dt,
                        int nsteps, int rebuild_every, double r_list, int K, double* f, int f_valid,
                        int sample_every, double* J_pot, double* J_kin) {
    std::vector<int32_t> NN(n), NL((size_t)n * K);
    std::vector<double> pe(n), J((size_t)3 * n);
    if (!f_valid) {
        if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        int rc = evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                                  pe.data(), f, nullptr, nullptr, nullptr, nullptr, 0, n);
        if (rc) return rc;
    }
    int ns = 0;
    for (int s = 0; s < nsteps; ++s) {
        vv_kick_drift(n, x, y, z, vx, vy, vz, f, mass, dt, box);
        if (s % rebuild_every == 0 || !f_valid)
            if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        f_valid = 1;
        const bool sample = (s + 1) % sample_every == 0;
        int rc;
        if (!sample) {
            rc = evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                                  pe.data(), f, nullptr, nullptr, nullptr, nullptr, 0, n);
            if (rc) return rc;
            vv_kick(n, vx, vy, vz, f, mass, dt);
            continue;
        }
        // Eq. (30) uses v_i of the state the forces belong to: kick first with the new forces, then evaluate J
        rc = evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                              pe.data(), f, nullptr, nullptr, nullptr, nullptr, 0, n);
        if (rc) return rc;
        vv_kick(n, vx, vy, vz, f, mass, dt);
        std::vector<double> f2((size_t)3 * n);
        rc = evaluate<double>(pot, par, n, x, y, z, vx, vy, vz, box, NN.data(), NL.data(), K,
                              pe.data(), f2.data(), nullptr, nullptr, J.data(), nullptr, 0, n);
        if (rc) return rc;
        long double jp[3] = {0, 0, 0}, jk[3] = {0, 0, 0};
        for (int64_t i = 0; i < n; ++i) {
            const double e = 0.5 * mass / KAPPA_ACC * (vx[i] * vx[i] + vy[i] * vy[i] + vz[i] * vz[i]) + pe[i];
            jp[0] += J[i]; jp[1] += J[n + i]; jp[2] += J[2 * n + i];
            jk[0] += e * vx[i]; jk[1] += e * vy[i]; jk[2] += e * vz[i];
        }
        for (int a = 0; a < 3; ++a) {
            if (J_pot) J_pot[3 * ns + a] = (double)jp[a];
            if (J_kin) J_kin[3 * ns + a] = (double)jk[a];
        }
        ++ns;
    }
    return 0;
}

// NPT by weak coupling (Berendsen thermostat and barostat: the paper's benchmark ensemble, PAPER.md:355;
// DESIGN.md reading A18).  One step = velocity-Verlet step, then
//   T = 2 KE / (3 N kB),  P = (2 KE + tr sum_i W_i) / (3 V)        (W = sum r_i (x) F_i, Eq. 17)
//   v *= lambda,  lambda = sqrt(1 + (dt/tau_T)(T0/T - 1))
//   x, box *= mu, mu = (1 - beta (dt/tau_P)(P0 - P))^(1/3)
// P in eV/A^3, beta in A^3/eV.  T_trace, P_trace [nsteps] receive the values measured BEFORE the scaling.
int oracle_npt_run(int pot, const double* par, int64_t n, double* x, double* y, double* z,
                   double* vx, double* vy, double* vz, double* box, double mass, double dt,
                   int nsteps, int rebuild_every, double r_list, int K, double* f, int f_valid,
                   double T0, double tau_T, double P0, double tau_P, double beta,
                   double* T_trace, double* P_trace) {
    const double KB = 8.617333262e-5;
    std::vector<int32_t> NN(n), NL((size_t)n * K);
    std::vector<double> pe(n), W((size_t)9 * n);
    auto forces = [&]() {
        return evaluate<double>(pot, par, n, x, y, z, nullptr, nullptr, nullptr, box, NN.data(), NL.data(), K,
                                pe.data(), f, nullptr, W.data(), nullptr, nullptr, 0, n);
    };
    if (!f_valid) {
        if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        int rc = forces();
        if (rc) return rc;
    }
    for (int s = 0; s < nsteps; ++s) {
        vv_kick_drift(n, x, y, z, vx, vy, vz, f, mass, dt, box);
        if (s % rebuild_every == 0 || !f_valid)
            if (neighbours_cell(n, x, y, z, box, r_list, K, NN.data(), NL.data()) < 0) return -1;
        f_valid = 1;
        int rc = forces();
        if (rc) return rc;
        vv_kick(n, vx, vy, vz, f, mass, dt);
        long double ke2 = 0, trw = 0;                                      // 2 KE and tr W
        for (int64_t i = 0; i < n; ++i) {
            ke2 += (long double)(vx[i] * vx[i] + vy[i] * vy[i] + vz[i] * vz[i]);
            trw += (long double)(W[0 * n + i] + W[4 * n + i] + W[8 * n + i]);
        }
        ke2 *= mass / KAPPA_ACC;
        const double V = box[0] * box[1] * box[2];
        const double T = (double)ke2 / (3.0 * n * KB), P = (double)(ke2 + trw) / (3.0 * V);
        if (T_trace) T_trace[s] = T;
        if (P_trace) P_trace[s] = P;
        const double lam = T > 0 ? std::sqrt(1.0 + dt / tau_T * (T0 / T - 1.0)) : 1.0;
        const double mu = std::cbrt(1.0 - beta * dt / tau_P * (P0 - P));
        for (int64_t i = 0; i < n; ++i) {
            vx[i] *= lam; vy[i] *= lam; vz[i] *= lam;
            x[i] *= mu; y[i] *= mu; z[i] *= mu;
        }
        for (int a = 0; a < 3; ++a) box[a] *= mu;
    }
    return 0;
}

}  // extern "C"
