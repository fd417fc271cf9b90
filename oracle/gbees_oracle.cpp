// GBEES prediction-step ORACLE  (test infrastructure, NOT product code)
// =====================================================================
// A plain, serial, obviously-correct CPU implementation of what the hot path of
// "GBEES-GPU" (arXiv 2508.13986, /root/reference/PAPER.md) computes, written from the
// paper and from the readings D1-D5 / A1-A18 in SURVEY.md section 8(c) (restated in DESIGN.md).
//
// * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
//   legs may load this. The product (paper_2508_13986_b200/) never does.
// * Shares NO code with the CUDA path: no common header, helper, packing or hashing.
//   Cells are keyed by their int32 coordinate vector in a std::unordered_map.
// * fp64 throughout; compile with -O2 -ffp-contract=off (no FMA contraction), so that
//   face velocities, grow/prune decisions and dt are IEEE-reproducible (reading A12).
// * Flux is the *scatter* form, in the paper's order: DCU (Eq. 7), then
//   Algorithm 1 with line 7 corrected (reading A2), then the
//   high-resolution term (reading A3, PAPER.md:112 defers it to ref. [11]).
//
// Parity pins (tests/test_oracle_pins.py): P1 telescoping/conservation, P2 Courant-1
// shift (bit exact), P3 n-D constant-velocity closed form for all sign patterns,
// P4 1-D binomial smear, P5 Lax-Wendroff, P6 TVD + order, P7 dense-array brute force
// (oracle/dense_ctu.py, gather form), P8 dt closed form, P9 linear-dynamics moments,
// P10 Bayes/Kalman, P12 grow/prune duality, P13 reflection; dynamics() ids 0-4 by what the paper
// and the mathematics fix (test_D_*: equilibria, "(F, ..., F) is an unstable equilibrium",
// energy conservation of the Lorenz '96 advection term, divergence, Jacobian structure of PAPER.md:303/319).
// PARITY UNPINNED against the paper's own software: the limiter family (A3), the exact
// edge-growth test (A10/A11), the normalisation cadence (A9). See DESIGN.md.
//
// C ABI: gbeeso_* (host pointers only). All functions return 0 on success, <0 on error.

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <unordered_map>
#include <vector>

namespace {

constexpr int MAXN = 6;
using Coord = std::array<int32_t, MAXN>;  // unused dims stay 0

struct CoordHash {
    size_t operator()(const Coord& c) const noexcept {
        // FNV-1a style mix over the coordinates (oracle-only; unrelated to the GPU hash)
        uint64_t h = 1469598103934665603ull;
        for (int j = 0; j < MAXN; ++j) {
            h ^= (uint64_t)(uint32_t)c[j];
            h *= 1099511628211ull;
            h ^= h >> 29;
        }
        return (size_t)h;
    }
};
using CellMap = std::unordered_map<Coord, int64_t, CoordHash>;

struct Oracle {
    int n = 0;
    double h[MAXN] = {0};
    double thresh = 0;
    int dyn = 0;
    std::vector<double> par;
    double cfl = 0.9;
    int hi_res = 1;
    int limiter = 0;     // 0 = monotonised central, 1 = none (phi == 1)
    int do_grow = 1;     // test switches (pins P1-P5 freeze the grid / skip normalisation)
    int do_norm = 1;
    double mu[MAXN] = {0};  // grid origin = mean passed to init_gaussian (reading A8)
    double t = 0;
    double last_dt = 0;
    double last_mass = 1;
    std::vector<Coord> key;
    std::vector<double> P;
    CellMap map;
};

inline double pos(double u) { return u > 0.0 ? u : 0.0; }  // f^+ = max(f,0)
inline double neg(double u) { return u < 0.0 ? u : 0.0; }  // f^- = min(f,0)

// Dynamics f_j(x), fixed operation order (reading A12). No FMA (-ffp-contract=off).
double dynamics(const Oracle& o, const double* x, int j) {
    const int n = o.n;
    const double* p = o.par.data();
    switch (o.dyn) {
        case 0:  // Lorenz '63 classic (sigma, beta, rho) -- BASELINE configs 0/1
            if (j == 0) return p[0] * (x[1] - x[0]);
            if (j == 1) return x[0] * (p[2] - x[2]) - x[1];
            return x[0] * x[1] - p[1] * x[2];
        case 1:  // Lorenz '63, paper's z-shifted form (sigma, b, r)
            if (j == 0) return p[0] * (x[1] - x[0]);
            if (j == 1) return (-x[1]) - x[0] * x[2];
            return (x[0] * x[1] - p[1] * x[2]) - p[1] * p[2];
        case 2: {  // Lorenz '96 (F), cyclic
            const int jp = (j + 1) % n, jm1 = (j + n - 1) % n, jm2 = (j + n - 2) % n;
            return ((x[jp] - x[jm2]) * x[jm1] - x[j]) + p[0];
        }
        case 3: {  // linear f = A x, A row-major, ascending m  (BASELINE config 3)
            double s = p[j * n + 0] * x[0];
            for (int m = 1; m < n; ++m) s = s + p[j * n + m] * x[m];
            return s;
        }
        case 4:  // constant f = v  (pins P2-P5)
            return p[j];
    }
    return 0.0;
}

// u_{c,j} = f_j at the centre of the LOWER j-face of cell c (paper's i - e^j/2).
// Face coordinate in dim j: mu_j + (double(c_j) - 0.5) * h_j ; other dims mu_m + double(c_m) * h_m
// (one multiply, one add; reading A12). The upper j-face of c is the lower j-face of c + e^j.
double face_velocity(const Oracle& o, const Coord& c, int j) {
    double x[MAXN];
    for (int m = 0; m < o.n; ++m) {
        const double cm = (m == j) ? ((double)c[m] - 0.5) : (double)c[m];
        x[m] = o.mu[m] + cm * o.h[m];
    }
    return dynamics(o, x, j);
}

inline Coord shifted(const Coord& c, int j, int s) {
    Coord r = c;
    r[j] += s;
    return r;
}

inline double probe(const Oracle& o, const Coord& c) {  // P reads as 0 outside I (reading A6)
    auto it = o.map.find(c);
    return it == o.map.end() ? 0.0 : o.P[it->second];
}

void insert_cell(Oracle& o, const Coord& c, double p) {
    auto it = o.map.find(c);
    if (it != o.map.end()) return;
    o.map.emplace(c, (int64_t)o.key.size());
    o.key.push_back(c);
    o.P.push_back(p);
}

// Targets(c) of D1.1 (readings A10/A11): downwind face neighbours and downwind pairwise-edge
// neighbours, decided by the SOURCE cell's own face velocities with strict sign tests.
void targets(const Oracle& o, const Coord& c, std::vector<Coord>& out) {
    out.clear();
    const int n = o.n;
    bool op[MAXN], om[MAXN];
    for (int j = 0; j < n; ++j) {
        op[j] = face_velocity(o, shifted(c, j, +1), j) > 0.0;  // outflow through upper face
        om[j] = face_velocity(o, c, j) < 0.0;                  // outflow through lower face
    }
    for (int j = 0; j < n; ++j) {
        if (op[j]) out.push_back(shifted(c, j, +1));
        if (om[j]) out.push_back(shifted(c, j, -1));
    }
    for (int j = 0; j < n; ++j)
        for (int l = j + 1; l < n; ++l)
            for (int sj = -1; sj <= 1; sj += 2)
                for (int sl = -1; sl <= 1; sl += 2) {
                    const bool oj = sj > 0 ? op[j] : om[j];
                    const bool ol = sl > 0 ? op[l] : om[l];
                    if (oj && ol) out.push_back(shifted(shifted(c, j, sj), l, sl));
                }
}

// monotonised-central limiter, division-free (reading A3)
inline double mc(double a, double b) {
    if (a * b <= 0.0) return 0.0;
    const double m = std::min(0.5 * std::fabs(a + b), std::min(2.0 * std::fabs(a), 2.0 * std::fabs(b)));
    return a > 0.0 ? m : -m;
}

}  // namespace

namespace {

// ---- D1.1 grow (206-216) ---------------------------------------------------
void grow(Oracle& o) {
    const int64_t n0 = (int64_t)o.key.size();  // all tests use the pre-grow state
    std::vector<Coord> tg;
    for (int64_t i = 0; i < n0; ++i) {
        if (!(o.P[i] >= o.thresh)) continue;
        const Coord c = o.key[i];
        targets(o, c, tg);
        for (const Coord& q : tg) insert_cell(o, q, 0.0);
    }
}

// ---- D1.2 dt, Eq. (8) (readings A1/A4) ------------------------------------
// s_c = sum_j abs(u_{c,j}) / h_j over the n lower faces of every active cell; dt = C / max s_c.
double cfl_smax(const Oracle& o) {
    double smax = 0.0;
    for (size_t i = 0; i < o.key.size(); ++i) {
        double s = 0.0;
        for (int j = 0; j < o.n; ++j) s = s + std::fabs(face_velocity(o, o.key[i], j)) / o.h[j];
        if (s > smax) smax = s;
    }
    return smax;
}

// ---- D1.3 flux, scatter form ----------------------------------------------------------------
// Face (c,j) = lower j-face of cell c. The face set is every face adjacent to >= 1 active cell,
// i.e. the lower faces of the "extended" cells E = I u {c + e^j : c in I}. Each extended cell
// carries n flux accumulators F[e][j]; only the valid faces are ever touched.
struct Ext {
    std::vector<Coord> key;
    std::vector<int64_t> act;  // index into the active pool or -1
    CellMap map;
    std::vector<double> F;     // [e * n + j]
    std::vector<double> U;     // face velocity u_{e,j}
    std::vector<char> valid;   // face (e,j) adjacent to >= 1 active cell
};

int64_t ext_get(Ext& x, const Coord& c) {
    auto it = x.map.find(c);
    if (it != x.map.end()) return it->second;
    const int64_t e = (int64_t)x.key.size();
    x.map.emplace(c, e);
    x.key.push_back(c);
    x.act.push_back(-1);
    return e;
}

void build_ext(const Oracle& o, Ext& x) {
    const int n = o.n;
    const int64_t N = (int64_t)o.key.size();
    x.key.reserve(2 * N);
    x.map.reserve(4 * N);
    for (int64_t i = 0; i < N; ++i) {
        const int64_t e = ext_get(x, o.key[i]);
        x.act[e] = i;
    }
    for (int64_t i = 0; i < N; ++i)
        for (int j = 0; j < n; ++j) ext_get(x, shifted(o.key[i], j, +1));
    const int64_t E = (int64_t)x.key.size();
    x.F.assign(E * n, 0.0);
    x.U.assign(E * n, 0.0);
    x.valid.assign(E * n, 0);
    for (int64_t e = 0; e < E; ++e)
        for (int j = 0; j < n; ++j) {
            const bool here = x.act[e] >= 0;
            const bool below = o.map.count(shifted(x.key[e], j, -1)) > 0;
            if (here || below) {
                x.valid[e * n + j] = 1;
                x.U[e * n + j] = face_velocity(o, x.key[e], j);
            }
        }
}

// index of face-owner cell q in the extended set (must exist for the faces Alg. 1 touches)
inline int64_t ext_find(const Ext& x, const Coord& q) {
    auto it = x.map.find(q);
    return it == x.map.end() ? -1 : it->second;
}

void compute_fluxes(const Oracle& o, Ext& x, double dt) {
    const int n = o.n;
    const int64_t E = (int64_t)x.key.size();
    // DCU, Eq. (7): F(c,j) = u+ P_{c-e^j} + u- P_c
    for (int64_t e = 0; e < E; ++e)
        for (int j = 0; j < n; ++j) {
            if (!x.valid[e * n + j]) continue;
            const double u = x.U[e * n + j];
            const double Pc = x.act[e] >= 0 ? o.P[x.act[e]] : 0.0;
            const double Pb = probe(o, shifted(x.key[e], j, -1));
            x.F[e * n + j] = pos(u) * Pb + neg(u) * Pc;
        }
    // CTU, Algorithm 1 (lines 3-8), applied per face (c,j); line 7 uses f+ (reading A2);
    // a correction whose carrier cell (c for lines 5-6, b = c - e^j for lines 7-8) is not
    // active is dropped (reading A6).
    for (int64_t e = 0; e < E; ++e)
        for (int j = 0; j < n; ++j) {
            if (!x.valid[e * n + j]) continue;
            const Coord c = x.key[e];
            const Coord b = shifted(c, j, -1);
            const double Pc = x.act[e] >= 0 ? o.P[x.act[e]] : 0.0;
            const double Pb = probe(o, b);
            const double Fs = 0.5 * (dt / o.h[j]) * (Pc - Pb);  // line 3
            const double u = x.U[e * n + j];
            const bool c_act = x.act[e] >= 0;
            const bool b_act = o.map.count(b) > 0;
            const int64_t eb = b_act ? ext_find(x, b) : -1;
            for (int l = 0; l < n; ++l) {
                if (l == j) continue;
                if (c_act) {
                    const int64_t eu = ext_find(x, shifted(c, l, +1));  // face c + e^l/2
                    x.F[eu * n + l] -= pos(u) * pos(x.U[eu * n + l]) * Fs;   // line 5
                    x.F[e * n + l] -= pos(u) * neg(x.U[e * n + l]) * Fs;     // line 6
                }
                if (b_act) {
                    const int64_t eu = ext_find(x, shifted(b, l, +1));  // face b + e^l/2
                    x.F[eu * n + l] -= neg(u) * pos(x.U[eu * n + l]) * Fs;   // line 7 (A2)
                    x.F[eb * n + l] -= neg(u) * neg(x.U[eb * n + l]) * Fs;   // line 8
                }
            }
        }
    // High-resolution term (reading A3): F(c,j) += 1/2 abs(u) (1 - tau_j abs(u)) W~,
    // W = P_c - P_{c-e^j}; W_up one cell upwind; all from time-level-k P.
    if (o.hi_res) {
        for (int64_t e = 0; e < E; ++e)
            for (int j = 0; j < n; ++j) {
                if (!x.valid[e * n + j]) continue;
                const double u = x.U[e * n + j];
                if (u == 0.0) continue;
                const Coord c = x.key[e];
                const double Pc = x.act[e] >= 0 ? o.P[x.act[e]] : 0.0;
                const double Pb = probe(o, shifted(c, j, -1));
                const double W = Pc - Pb;
                double Wl;
                if (o.limiter == 1) {
                    Wl = W;
                } else {
                    const double Wup = u > 0.0 ? Pb - probe(o, shifted(c, j, -2))
                                               : probe(o, shifted(c, j, +1)) - Pc;
                    Wl = mc(W, Wup);
                }
                const double au = std::fabs(u);
                x.F[e * n + j] += 0.5 * au * (1.0 - (dt / o.h[j]) * au) * Wl;
            }
    }
}

// ---- D1 one prediction step -------------------------------------------------------------------
int step(Oracle& o, double* dt_io) {
    if (o.key.empty()) return -7;
    if (o.do_grow) grow(o);
    const double cap = *dt_io;
    const bool capped = std::isfinite(cap) && cap > 0.0;
    const double smax = cfl_smax(o);
    double dt;
    if (smax > 0.0) {
        dt = o.cfl / smax;
        if (capped && cap < dt) dt = cap;
    } else {
        if (!capped) return -6;
        dt = cap;
    }
    Ext x;
    build_ext(o, x);
    compute_fluxes(o, x, dt);
    // D1.4 update: P_c <- P_c - sum_j tau_j (F(c+e^j, j) - F(c, j)); no clipping (A5)
    const int n = o.n;
    std::vector<double> Pn(o.P.size());
    for (size_t i = 0; i < o.key.size(); ++i) {
        const int64_t e = ext_find(x, o.key[i]);
        double p = o.P[i];
        for (int j = 0; j < n; ++j) {
            const int64_t eu = ext_find(x, shifted(o.key[i], j, +1));
            p -= (dt / o.h[j]) * (x.F[eu * n + j] - x.F[e * n + j]);
        }
        Pn[i] = p;
    }
    o.P.swap(Pn);
    // D1.5 normalise (serial, pool order)
    double M = 0.0;
    for (double p : o.P) M += p;
    o.last_mass = M;
    if (o.do_norm) {
        if (!(M > 0.0) || !std::isfinite(M)) return -6;
        for (double& p : o.P) p /= M;
    }
    o.t += dt;
    o.last_dt = dt;
    *dt_io = dt;
    return 0;
}

void rebuild(Oracle& o, const std::vector<char>& keep) {
    std::vector<Coord> k2;
    std::vector<double> p2;
    for (size_t i = 0; i < o.key.size(); ++i)
        if (keep[i]) {
            k2.push_back(o.key[i]);
            p2.push_back(o.P[i]);
        }
    o.key.swap(k2);
    o.P.swap(p2);
    o.map.clear();
    for (size_t i = 0; i < o.key.size(); ++i) o.map.emplace(o.key[i], (int64_t)i);
}

int normalise(Oracle& o) {
    double M = 0.0;
    for (double p : o.P) M += p;
    o.last_mass = M;
    if (!(M > 0.0) || !std::isfinite(M)) return -6;
    for (double& p : o.P) p /= M;
    return 0;
}

// ---- D3 prune (Alg. 3) --------------------------------------
int prune(Oracle& o) {
    std::vector<char> keep(o.key.size(), 0);
    std::vector<Coord> tg;
    for (size_t i = 0; i < o.key.size(); ++i) {
        if (!(o.P[i] >= o.thresh)) continue;
        keep[i] = 1;
        targets(o, o.key[i], tg);
        for (const Coord& q : tg) {
            auto it = o.map.find(q);
            if (it != o.map.end()) keep[it->second] = 1;
        }
    }
    rebuild(o, keep);
    if (o.key.empty()) return -6;
    return o.do_norm ? normalise(o) : 0;
}

// Cholesky-based inverse of an SPD matrix (n <= 6); returns false if not SPD. det via L.
bool spd_inverse(int n, const double* A, double* inv, double* det) {
    double L[MAXN][MAXN] = {{0}};
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = A[i * n + j];
            for (int k = 0; k < j; ++k) s -= L[i][k] * L[j][k];
            if (i == j) {
                if (!(s > 0.0)) return false;
                L[i][i] = std::sqrt(s);
            } else {
                L[i][j] = s / L[j][j];
            }
        }
    double Li[MAXN][MAXN] = {{0}};  // inverse of L (lower triangular)
    for (int i = 0; i < n; ++i) {
        Li[i][i] = 1.0 / L[i][i];
        for (int j = 0; j < i; ++j) {
            double s = 0.0;
            for (int k = j; k < i; ++k) s -= L[i][k] * Li[k][j];
            Li[i][j] = s / L[i][i];
        }
    }
    double d = 1.0;
    for (int i = 0; i < n; ++i) d *= L[i][i] * L[i][i];
    *det = d;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) {
            double s = 0.0;
            for (int k = std::max(i, j); k < n; ++k) s += Li[k][i] * Li[k][j];
            inv[i * n + j] = s;
        }
    return true;
}

inline double quad_form(int n, const double* Ainv, const double* d) {
    double q = 0.0;
    for (int i = 0; i < n; ++i) {
        double r = 0.0;
        for (int j = 0; j < n; ++j) r += Ainv[i * n + j] * d[j];
        q += d[i] * r;
    }
    return q;
}

// ---- D5 / A8 init_gaussian ---------------------------------------------------------------------
int init_gaussian(Oracle& o, const double* mean, const double* cov) {
    const int n = o.n;
    double inv[MAXN * MAXN], det;
    if (!spd_inverse(n, cov, inv, &det)) return -3;
    for (int j = 0; j < n; ++j) o.mu[j] = mean[j];
    o.key.clear();
    o.P.clear();
    o.map.clear();
    o.t = 0.0;
    double vol = 1.0;
    for (int j = 0; j < n; ++j) vol *= o.h[j];
    const double norm = vol / std::sqrt(std::pow(2.0 * M_PI, n) * det);  // P~ at the mean
    if (!(norm >= o.thresh)) return -6;
    // bounding box of the ellipsoid {q <= r2}: |d_j| <= sqrt(r2 * cov_jj)  (+1 cell of slack)
    const double r2 = 2.0 * std::log(norm / o.thresh);
    int64_t R[MAXN] = {0};
    for (int j = 0; j < n; ++j) R[j] = (int64_t)std::floor(std::sqrt(r2 * cov[j * n + j]) / o.h[j]) + 1;
    Coord c{};
    for (int j = 0; j < n; ++j) c[j] = (int32_t)(-R[j]);
    for (;;) {
        double d[MAXN];
        for (int j = 0; j < n; ++j) d[j] = (double)c[j] * o.h[j];  // x_c - mu = c o h exactly
        const double g = std::exp(-0.5 * quad_form(n, inv, d)) * norm;
        if (g >= o.thresh) insert_cell(o, c, g);
        int j = n - 1;
        while (j >= 0) {
            if (++c[j] <= R[j]) break;
            c[j] = (int32_t)(-R[j]);
            --j;
        }
        if (j < 0) break;
    }
    return normalise(o);
}

// ---- D4 correct, Eq. (4) with h(x) = x (reading A13) -----------------------------
int correct(Oracle& o, const double* z, const double* Rm) {
    const int n = o.n;
    double inv[MAXN * MAXN], det;
    if (!spd_inverse(n, Rm, inv, &det)) return -3;
    for (size_t i = 0; i < o.key.size(); ++i) {
        double d[MAXN];
        for (int j = 0; j < n; ++j) d[j] = z[j] - (o.mu[j] + (double)o.key[i][j] * o.h[j]);
        o.P[i] *= std::exp(-0.5 * quad_form(n, inv, d));
    }
    return normalise(o);
}

// ---- f2: Eq. (4) with a linear measurement model y = H x + v, v ~ N(0, R), H m x n.
// The paper's own scenario observes one state only (y = x3, sigma_y = 1): H = (0 0 1).
// P_c <- P_c * exp(-1/2 (y - H x_c)^T R^-1 (y - H x_c)), then normalise.
int correct_linear(Oracle& o, const double* H, int m, const double* y, const double* Rm) {
    const int n = o.n;
    if (m < 1 || m > MAXN) return -1;
    double inv[MAXN * MAXN], det;
    if (!spd_inverse(m, Rm, inv, &det)) return -3;
    for (size_t i = 0; i < o.key.size(); ++i) {
        double x[MAXN], d[MAXN];
        for (int j = 0; j < n; ++j) x[j] = o.mu[j] + (double)o.key[i][j] * o.h[j];
        for (int r = 0; r < m; ++r) {
            double hx = 0.0;
            for (int j = 0; j < n; ++j) hx += H[r * n + j] * x[j];
            d[r] = y[r] - hx;
        }
        o.P[i] *= std::exp(-0.5 * quad_form(m, inv, d));
    }
    return normalise(o);
}

// ---- f2, a NON-linear measurement: the range to a point s, y = ||x - s||_2 + v, v ~ N(0, sigma^2).
// Eq. (4): P_c <- P_c * exp(-1/2 ((y - ||x_c - s||) / sigma)^2), then normalise.
int correct_range(Oracle& o, const double* s, double y, double sigma) {
    if (!(sigma > 0.0)) return -3;
    for (size_t i = 0; i < o.key.size(); ++i) {
        double r2 = 0.0;
        for (int j = 0; j < o.n; ++j) {
            const double d = (o.mu[j] + (double)o.key[i][j] * o.h[j]) - s[j];
            r2 += d * d;
        }
        const double e = (y - std::sqrt(r2)) / sigma;
        o.P[i] *= std::exp(-0.5 * e * e);
    }
    return normalise(o);
}

}  // namespace

// ================================ C ABI (host pointers only) ====================================
extern "C" {

int gbeeso_create(void** out, int n, const double* dx, double threshold, int dynamics_id,
                  const double* params, int n_params, double cfl, int hi_res, int limiter) {
    if (!out || n < 1 || n > MAXN || !dx) return -1;
    if (dynamics_id < 0 || dynamics_id > 4) return -1;
    if ((dynamics_id == 0 || dynamics_id == 1) && (n != 3 || n_params < 3)) return -1;
    if (dynamics_id == 2 && (n < 4 || n_params < 1)) return -1;
    if (dynamics_id == 3 && n_params < n * n) return -1;
    if (dynamics_id == 4 && n_params < n) return -1;
    Oracle* o = new Oracle();
    o->n = n;
    for (int j = 0; j < n; ++j) {
        if (!(dx[j] > 0.0)) { delete o; return -1; }
        o->h[j] = dx[j];
    }
    o->thresh = threshold;
    o->dyn = dynamics_id;
    o->par.assign(params, params + n_params);
    o->cfl = cfl;
    o->hi_res = hi_res;
    o->limiter = limiter;
    *out = o;
    return 0;
}

int gbeeso_destroy(void* h) { delete (Oracle*)h; return 0; }

// test switches: grow on/off, normalise on/off (pins P1-P5 need the raw flux-form update)
int gbeeso_set_flags(void* h, int do_grow, int do_norm) {
    Oracle* o = (Oracle*)h;
    o->do_grow = do_grow;
    o->do_norm = do_norm;
    return 0;
}

int gbeeso_init_gaussian(void* h, const double* mean, const double* cov) {
    return init_gaussian(*(Oracle*)h, mean, cov);
}

// raw state import (tests): origin mu, count cells with int32 coords [count*n] and P as given
int gbeeso_import(void* h, const double* origin, const int32_t* keys, const double* p, int64_t count) {
    Oracle* o = (Oracle*)h;
    for (int j = 0; j < o->n; ++j) o->mu[j] = origin[j];
    o->key.clear(); o->P.clear(); o->map.clear();
    o->t = 0.0;
    for (int64_t i = 0; i < count; ++i) {
        Coord c{};
        for (int j = 0; j < o->n; ++j) c[j] = keys[i * o->n + j];
        if (o->map.count(c)) return -1;
        insert_cell(*o, c, p[i]);
    }
    return 0;
}

int gbeeso_step(void* h, double* dt) { return step(*(Oracle*)h, dt); }
int gbeeso_prune(void* h) { return prune(*(Oracle*)h); }
int gbeeso_correct(void* h, const double* z, const double* R) { return correct(*(Oracle*)h, z, R); }
int gbeeso_correct_range(void* h, const double* s, double y, double sigma) { return correct_range(*(Oracle*)h, s, y, sigma); }
int gbeeso_correct_linear(void* h, const double* H, int m, const double* y, const double* R) {
    return correct_linear(*(Oracle*)h, H, m, y, R);
}

int gbeeso_export(void* h, int32_t* keys, double* p, int64_t cap, int64_t* count) {
    Oracle* o = (Oracle*)h;
    const int64_t N = (int64_t)o->key.size();
    if (count) *count = N;
    if (!keys && !p) return 0;
    if (cap < N) return -5;
    for (int64_t i = 0; i < N; ++i) {
        if (keys) for (int j = 0; j < o->n; ++j) keys[i * o->n + j] = o->key[i][j];
        if (p) p[i] = o->P[i];
    }
    return 0;
}

int64_t gbeeso_count(void* h) { return (int64_t)((Oracle*)h)->key.size(); }
double gbeeso_time(void* h) { return ((Oracle*)h)->t; }
double gbeeso_last_mass(void* h) { return ((Oracle*)h)->last_mass; }
double gbeeso_last_dt(void* h) { return ((Oracle*)h)->last_dt; }

// u_{c,j}: velocity at the lower j-face of cell c (exposed so tests can pin A12 / Eq. 8)
double gbeeso_face_velocity(void* h, const int32_t* coords, int j) {
    Oracle* o = (Oracle*)h;
    Coord c{};
    for (int m = 0; m < o->n; ++m) c[m] = coords[m];
    return face_velocity(*o, c, j);
}

// test hook for the dynamics pins (tests/test_oracle_pins.py): out[j] = f_j(x) at an arbitrary point x,
// through the same dynamics() the face velocities use
int gbeeso_dynamics(void* h, const double* x, double* out) {
    Oracle* o = (Oracle*)h;
    for (int j = 0; j < o->n; ++j) out[j] = dynamics(*o, x, j);
    return 0;
}

// number of grow targets of cell `coords` and (optionally) their coordinates [<= 72 * n]
int gbeeso_targets(void* h, const int32_t* coords, int32_t* out) {
    Oracle* o = (Oracle*)h;
    Coord c{};
    for (int m = 0; m < o->n; ++m) c[m] = coords[m];
    std::vector<Coord> tg;
    targets(*o, c, tg);
    if (out)
        for (size_t i = 0; i < tg.size(); ++i)
            for (int m = 0; m < o->n; ++m) out[i * o->n + m] = tg[i][m];
    return (int)tg.size();
}

// ---- config 4: hashtable / compaction reference answers (std::unordered_map over u64) --------
// found[i] = 1 if query[i] is among keys[0..nk); used to check the GPU table's lookups.
int gbeeso_ht_lookup(const uint64_t* keys, int64_t nk, const uint64_t* query, int64_t nq, uint8_t* found) {
    std::unordered_map<uint64_t, int64_t> m;
    m.reserve((size_t)nk * 2);
    for (int64_t i = 0; i < nk; ++i) m.emplace(keys[i], i);
    for (int64_t i = 0; i < nq; ++i) found[i] = m.count(query[i]) ? 1 : 0;
    return 0;
}

}  // extern "C"
