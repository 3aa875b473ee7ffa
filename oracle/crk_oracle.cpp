// crk_oracle.cpp -- CPU ORACLE (FP64, brute-force neighbours) for the CRKSPH short-range gas pipeline.
// TEST INFRASTRUCTURE ONLY: see crk_oracle.h.  Shares no code with the CUDA library.
//
// Every function cites the PAPER.md passage it follows.  Notation follows the paper:
//   x_ij = x_i - x_j (minimum image),  r = |x_ij|,  eta = r/h,  h = SUPPORT radius (W=0 for eta>=1, l.91),
//   W_ij = W(r, h_i)  (Eq. 13, l.95),   D(r,h) = W'(r)/r  so that  grad_i W_ij = D(r,h_i) x_ij.
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -mavx2 -mfma   (see oracle/build.py)
//   -ffp-contract=off : the FP32 neighbour predicate (reading S3) must be evaluated exactly as written.
#include "crk_oracle.h"

#include <algorithm>
#include <cmath>
#include <limits>
#include <cstring>
#include <vector>
#include <omp.h>

namespace {

constexpr double PI = 3.14159265358979323846;
constexpr double SIGMA = 495.0 / (32.0 * PI);   // Eq. 12 normalisation (3-D Wendland C4, unit extent)
constexpr uint32_t FLAG_I = 0x80000000u;         // r < h_i : j is in the gather set of i
constexpr uint32_t FLAG_J = 0x40000000u;         // r < h_j : i is in the gather set of j
constexpr uint32_t IDX_MASK = 0x3fffffffu;

int g_threads = 0;

// ---------------------------------------------------------------------------------------------- kernel
// Eq. 12: W_C4(eta,h) = 495/(32 pi h^3) (1-eta)^6 (1 + 6 eta + 35/3 eta^2), 0 for eta >= 1
inline double W_c4(double r, double h) {
    const double eta = r / h;
    if (eta >= 1.0) return 0.0;
    const double t = 1.0 - eta;
    const double t2 = t * t;
    return SIGMA / (h * h * h) * (t2 * t2 * t2) * (1.0 + 6.0 * eta + (35.0 / 3.0) * eta * eta);
}
// radial derivative of Eq. 12 (derived): dW/dr = -(56/3) sigma h^-4 eta (1-eta)^5 (1+5 eta)
inline double dWdr_c4(double r, double h) {
    const double eta = r / h;
    if (eta >= 1.0) return 0.0;
    const double t = 1.0 - eta;
    const double t2 = t * t;
    return -(56.0 / 3.0) * SIGMA / (h * h * h * h) * eta * (t2 * t2 * t) * (1.0 + 5.0 * eta);
}
// D = W'/r = -(56/3) sigma h^-5 (1-eta)^5 (1+5 eta): finite at r = 0, so grad W = D x needs no division by r
inline double D_c4(double r, double h) {
    const double eta = r / h;
    if (eta >= 1.0) return 0.0;
    const double t = 1.0 - eta;
    const double t2 = t * t;
    return -(56.0 / 3.0) * SIGMA / (h * h * h * h * h) * (t2 * t2 * t) * (1.0 + 5.0 * eta);
}

struct Coef {          // first-order RK coefficients of one particle
    double A;
    double B[3];
    double dA[3];      // dA[c]    = d_c A
    double dB[3][3];   // dB[c][a] = d_c B^a
};

struct Moments {       // sums of step 4, all over the gather set of i; self term only in m0
    double m0, m1[3], m2[3][3];
    double dm0[3], dm1[3][3] /* [a][c] = d_c m1^a */, dm2[3][3][3] /* [a][b][c] = d_c m2^{ab} */;
};

}  // namespace

struct crk_oracle_ctx {
    crk_oracle_params p;
    int64_t n = 0;
    std::vector<float> x, y, z, h;               // the FP32 inputs, kept for the predicate
    std::vector<int64_t> off;                    // CSR offsets into nbr
    std::vector<uint32_t> nbr;                   // j | FLAG_I | FLAG_J
    std::vector<double> m, V, rho;
    std::vector<Coef> coef;
    std::vector<Moments> mom;
    std::vector<double> vx, vy, vz, u, P, cs;
    std::vector<double> ax, ay, az;              // dv/dt of the last crk_oracle_hydro_derivs (Eq. 17), for Eqs. 19-23
    std::vector<double> gradv;                   // [i][alpha][beta] = d_beta v^alpha  (Eq. 26, reading S9)
    int stage = 0;                               // 0 none, 1 built, 2 volumes, 3 coefficients, 4 hydro
};

namespace {

// minimum-image separation in double (values); reading step 1 of DESIGN.md
inline void sep(const crk_oracle_ctx* c, int64_t i, int64_t j, double d[3]) {
    const double L = c->p.box, half = 0.5 * c->p.box;
    d[0] = (double)c->x[i] - (double)c->x[j];
    d[1] = (double)c->y[i] - (double)c->y[j];
    d[2] = (double)c->z[i] - (double)c->z[j];
    for (int a = 0; a < 3; ++a) {
        if (d[a] > half) d[a] -= L;
        else if (d[a] < -half) d[a] += L;
    }
}

// Reading S3: the neighbour predicate in PRESCRIBED FP32:  d = xi - xj (float); wrap by +-L (float);
// r2 = fmaf(dz,dz, fmaf(dy,dy, dx*dx));  j in N(i)  iff  r2 < h_i*h_i  (float product).
inline float wrapf(float d, float L, float half) {
    if (d > half) d -= L;
    else if (d < -half) d += L;
    return d;
}
inline float r2_f32(float xi, float yi, float zi, float xj, float yj, float zj, float L, float half) {
    const float dx = wrapf(xi - xj, L, half);
    const float dy = wrapf(yi - yj, L, half);
    const float dz = wrapf(zi - zj, L, half);
    return std::fmaf(dz, dz, std::fmaf(dy, dy, dx * dx));
}

// Eqs. 15-16: WR_ij = A_i (1 + B_i.x) W ;
// (grad WR_ij)^c = d_c A_i s W + A_i (d_c B_i^a x^a + B_i^c) W + A_i s D x^c ,  s = 1 + B_i.x
inline double rk_kernel(const Coef& k, const double x[3], double W) {
    const double s = 1.0 + k.B[0] * x[0] + k.B[1] * x[1] + k.B[2] * x[2];
    return k.A * s * W;
}
inline void rk_grad(const Coef& k, const double x[3], double W, double D, double g[3]) {
    const double s = 1.0 + k.B[0] * x[0] + k.B[1] * x[1] + k.B[2] * x[2];
    for (int c = 0; c < 3; ++c) {
        const double dBx = k.dB[c][0] * x[0] + k.dB[c][1] * x[1] + k.dB[c][2] * x[2];
        g[c] = k.dA[c] * s * W + k.A * (dBx + k.B[c]) * W + k.A * s * D * x[c];
    }
}

inline bool inv3(const double m[3][3], double inv[3][3]) {
    const double c00 = m[1][1] * m[2][2] - m[1][2] * m[2][1];
    const double c01 = m[1][2] * m[2][0] - m[1][0] * m[2][2];
    const double c02 = m[1][0] * m[2][1] - m[1][1] * m[2][0];
    const double det = m[0][0] * c00 + m[0][1] * c01 + m[0][2] * c02;
    // reading S14: m2 counts as singular when det m2 <= 1e-4 (tr m2 / 3)^3, i.e. when the neighbours span less
    // than three dimensions up to rounding (fewer than 3 non-collinear, or coplanar, neighbours); an isotropic m2 has ratio 1
    const double tr3 = (m[0][0] + m[1][1] + m[2][2]) / 3.0;
    if (!(det > 1.0e-4 * tr3 * tr3 * tr3) || !std::isfinite(det)) return false;
    const double id = 1.0 / det;
    inv[0][0] = c00 * id;
    inv[0][1] = (m[0][2] * m[2][1] - m[0][1] * m[2][2]) * id;
    inv[0][2] = (m[0][1] * m[1][2] - m[0][2] * m[1][1]) * id;
    inv[1][0] = c01 * id;
    inv[1][1] = (m[0][0] * m[2][2] - m[0][2] * m[2][0]) * id;
    inv[1][2] = (m[0][2] * m[1][0] - m[0][0] * m[1][2]) * id;
    inv[2][0] = c02 * id;
    inv[2][1] = (m[0][1] * m[2][0] - m[0][0] * m[2][1]) * id;
    inv[2][2] = (m[0][0] * m[1][1] - m[0][1] * m[1][0]) * id;
    return true;
}

// enforce  sum_j V_j WR_ij = 1  and  sum_j V_j x_ij WR_ij = 0  (closed form derived in DESIGN.md):
//   B = -m2^-1 m1 ;  A = 1/(m0 + B.m1) ;
//   d_c A = -A^2 (d_c m0 + 2 B.d_c m1 + B^T (d_c m2) B) ;   d_c B = -m2^-1 (d_c m1 + (d_c m2) B)
inline void solve_coef(const Moments& M, Coef& k) {
    double inv[3][3];
    if (!inv3(M.m2, inv)) {   // reading S14: degenerate neighbourhood -> zeroth-order correction only
        k.A = 1.0 / M.m0;
        for (int a = 0; a < 3; ++a) {
            k.B[a] = 0.0;
            k.dA[a] = -k.A * k.A * M.dm0[a];
            for (int b = 0; b < 3; ++b) k.dB[a][b] = 0.0;
        }
        return;
    }
    for (int a = 0; a < 3; ++a)
        k.B[a] = -(inv[a][0] * M.m1[0] + inv[a][1] * M.m1[1] + inv[a][2] * M.m1[2]);
    k.A = 1.0 / (M.m0 + k.B[0] * M.m1[0] + k.B[1] * M.m1[1] + k.B[2] * M.m1[2]);
    for (int c = 0; c < 3; ++c) {
        double Bdm1 = 0.0, BdmB = 0.0, rhs[3];
        for (int a = 0; a < 3; ++a) {
            Bdm1 += k.B[a] * M.dm1[a][c];
            double t = 0.0;
            for (int b = 0; b < 3; ++b) t += M.dm2[a][b][c] * k.B[b];
            BdmB += k.B[a] * t;
            rhs[a] = M.dm1[a][c] + t;
        }
        k.dA[c] = -k.A * k.A * (M.dm0[c] + 2.0 * Bdm1 + BdmB);
        for (int a = 0; a < 3; ++a)
            k.dB[c][a] = -(inv[a][0] * rhs[0] + inv[a][1] * rhs[1] + inv[a][2] * rhs[2]);
    }
}

// moments of the kernel centred at point p (support h) over sources j with volumes V_j; x = p - x_j
inline void add_moment_term(Moments& M, const double x[3], double w, double g) {
    M.m0 += w;
    for (int a = 0; a < 3; ++a) {
        M.m1[a] += w * x[a];
        M.dm0[a] += g * x[a];
        for (int b = 0; b < 3; ++b) {
            M.m2[a][b] += w * x[a] * x[b];
            M.dm1[a][b] += g * x[a] * x[b];
            for (int cc = 0; cc < 3; ++cc) M.dm2[a][b][cc] += g * x[a] * x[b] * x[cc];
        }
    }
}
// product-rule terms: d_c m1^a += delta_ac m0 ;  d_c m2^{ab} += delta_ac m1^b + delta_bc m1^a
inline void finish_moments(Moments& M) {
    for (int a = 0; a < 3; ++a) {
        M.dm1[a][a] += M.m0;
        for (int b = 0; b < 3; ++b) {
            M.dm2[a][b][a] += M.m1[b];
            M.dm2[a][b][b] += M.m1[a];
        }
    }
}

// Eqs. 28-32 with reading S7 (division-free van Leer form)
inline double limiter(const crk_oracle_ctx* c, const double x[3], double r, double hi, double hj,
                      const double* gvi, const double* gvj, double gix[3], double gjx[3]) {
    for (int a = 0; a < 3; ++a) {
        gix[a] = gvi[3 * a + 0] * x[0] + gvi[3 * a + 1] * x[1] + gvi[3 * a + 2] * x[2];   // (grad v_i . x_ij)^a
        gjx[a] = gvj[3 * a + 0] * x[0] + gvj[3 * a + 1] * x[1] + gvj[3 * a + 2] * x[2];
    }
    const double N = x[0] * gix[0] + x[1] * gix[1] + x[2] * gix[2];    // numerator of Eq. 30
    const double Dn = x[0] * gjx[0] + x[1] * gjx[1] + x[2] * gjx[2];   // denominator of Eq. 30
    double phi_vl = 0.0;                                                 // Eq. 29 with r_ij = N/Dn
    if (N * Dn > 0.0) phi_vl = 4.0 * N * Dn / ((N + Dn) * (N + Dn));
    const double eta_crit = 1.0 / c->p.n_h, eta_fold = 0.2 / c->p.n_h;
    const double eta_ij = std::min(r / hi, r / hj);                      // Eq. 32
    double phi_ad = 1.0;                                                 // Eq. 31
    if (eta_ij < eta_crit) {
        const double q = (eta_ij - eta_crit) / eta_fold;
        phi_ad = std::exp(-q * q);
    }
    return phi_vl * phi_ad;                                              // Eq. 28
}

struct PairOut { double F[3]; double dE; double phi, Qi, Qj, mui, muj; };

// one neighbour's contribution to Eqs. 17-18 with P -> P+Q, a = 1, adot = 0
inline void pair_term(const crk_oracle_ctx* c, int64_t i, int64_t j, PairOut& o) {
    double x[3];
    sep(c, i, j, x);
    const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
    const double r = std::sqrt(r2);
    const double hi = c->h[i], hj = c->h[j];
    const double Wi = W_c4(r, hi), Di = D_c4(r, hi);
    const double Wj = W_c4(r, hj), Dj = D_c4(r, hj);
    double gij[3], gji[3], xm[3] = {-x[0], -x[1], -x[2]};
    rk_grad(c->coef[i], x, Wi, Di, gij);        // grad WR_ij
    rk_grad(c->coef[j], xm, Wj, Dj, gji);       // grad WR_ji  (x_ji = -x_ij, support h_j)
    const double G[3] = {gji[0] - gij[0], gji[1] - gij[1], gji[2] - gij[2]};

    double gix[3], gjx[3];
    const double phi = limiter(c, x, r, hi, hj, &c->gradv[9 * i], &c->gradv[9 * j], gix, gjx);
    // Eq. 27 (adot = 0):  uhat_ij = v_ij - (1/2) phi (grad v_i + grad v_j) . x_ij     (x_ji = -x_ij)
    const double vij[3] = {c->vx[i] - c->vx[j], c->vy[i] - c->vy[j], c->vz[i] - c->vz[j]};
    double ux = 0.0;
    for (int a = 0; a < 3; ++a) ux += (vij[a] - 0.5 * phi * (gix[a] + gjx[a])) * x[a];
    // Eq. 25 with uhat for u, a = 1:  mu_k = min(0, hhat_k (uhat.x) / (r^2 + hhat_k^2 eps^2))
    const double e2 = c->p.eps * c->p.eps;
    const double hhi = hi / c->p.n_h, hhj = hj / c->p.n_h;
    const double mui = std::min(0.0, hhi * ux / (r2 + hhi * hhi * e2));
    const double muj = std::min(0.0, hhj * ux / (r2 + hhj * hhj * e2));
    // Eq. 24: Q_k = rho_k (-C_l c_k mu_k + C_q mu_k^2)
    const double Qi = c->rho[i] * (-c->p.C_l * c->cs[i] * mui + c->p.C_q * mui * mui);
    const double Qj = c->rho[j] * (-c->p.C_l * c->cs[j] * muj + c->p.C_q * muj * muj);
    // Eq. 17:  m_i dv_i/dt += (1/2) V_i V_j (P_i+Q_i + P_j+Q_j) (grad WR_ji - grad WR_ij)
    const double half_vv = 0.5 * c->V[i] * c->V[j];
    const double pf = half_vv * (c->P[i] + Qi + c->P[j] + Qj);
    for (int a = 0; a < 3; ++a) o.F[a] = pf * G[a];
    // Eq. 18 (reading S6: sum over j, P_j as printed): m_i du_i/dt += (1/2) V_i V_j (P_j+Q_j) v_ji . (grad WR_ji - grad WR_ij)
    o.dE = half_vv * (c->P[j] + Qj) * (-(vij[0] * G[0] + vij[1] * G[1] + vij[2] * G[2]));
    o.phi = phi; o.Qi = Qi; o.Qj = Qj; o.mui = mui; o.muj = muj;
}

void set_threads() {
    if (g_threads > 0) omp_set_num_threads(g_threads);
}

}  // namespace

extern "C" {

crk_oracle_ctx* crk_oracle_create(const crk_oracle_params* p) {
    if (!p) return nullptr;
    crk_oracle_ctx* c = new crk_oracle_ctx();
    c->p = *p;
    return c;
}
void crk_oracle_destroy(crk_oracle_ctx* c) { delete c; }
void crk_oracle_set_threads(int n) { g_threads = n; if (n > 0) omp_set_num_threads(n); else omp_set_num_threads(omp_get_num_procs()); }
int crk_oracle_get_threads(void) { return g_threads > 0 ? g_threads : omp_get_max_threads(); }

double crk_oracle_W(double r, double h) { return W_c4(r, h); }
double crk_oracle_dWdr(double r, double h) { return dWdr_c4(r, h); }

// "a periodic neighbour search within each particle's smoothing support": brute force over all (i,j).
// Stores the symmetric set  r2 < max(h_i^2, h_j^2)  with flags for the two one-sided memberships (reading S3).
int crk_oracle_build(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h) {
    if (!c || n < 0 || n >= (int64_t)IDX_MASK || (n > 0 && (!x || !y || !z || !h))) return -1;
    set_threads();
    const float L = (float)c->p.box, half = 0.5f * L;
    for (int64_t i = 0; i < n; ++i) {
        if (!(h[i] > 0.0f) || !(h[i] < half)) return -1;                                  // reading S13
        if (!(x[i] >= 0.0f && x[i] < L && y[i] >= 0.0f && y[i] < L && z[i] >= 0.0f && z[i] < L)) return -1;
    }
    c->n = n;
    c->x.assign(x, x + n); c->y.assign(y, y + n); c->z.assign(z, z + n); c->h.assign(h, h + n);
    std::vector<std::vector<uint32_t>> rows((size_t)n);
#pragma omp parallel
    {
        std::vector<float> r2((size_t)n);
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n; ++i) {
            const float xi = x[i], yi = y[i], zi = z[i];
            const float hi2 = h[i] * h[i];
            for (int64_t j = 0; j < n; ++j) r2[j] = r2_f32(xi, yi, zi, x[j], y[j], z[j], L, half);
            std::vector<uint32_t>& row = rows[i];
            for (int64_t j = 0; j < n; ++j) {
                if (j == i) continue;
                const float hj2 = h[j] * h[j];
                uint32_t f = 0;
                if (r2[j] < hi2) f |= FLAG_I;
                if (r2[j] < hj2) f |= FLAG_J;
                if (f) row.push_back((uint32_t)j | f);
            }
        }
    }
    c->off.assign((size_t)n + 1, 0);
    for (int64_t i = 0; i < n; ++i) c->off[i + 1] = c->off[i] + (int64_t)rows[i].size();
    c->nbr.resize((size_t)c->off[n]);
    for (int64_t i = 0; i < n; ++i) std::copy(rows[i].begin(), rows[i].end(), c->nbr.begin() + c->off[i]);
    c->stage = 1;
    return 0;
}

// Eq. 14: V_i^-1 = n_i = sum_j W(|x_i - x_j|, h_i), self term included (reading S4);
// rho_i = m_i / V_i (reading S2).
int crk_oracle_volumes(crk_oracle_ctx* c, const float* m, double* V, double* rho, uint32_t* nbr_count) {
    if (!c || c->stage < 1 || !m) return -1;
    set_threads();
    const int64_t n = c->n;
    c->m.resize(n); c->V.resize(n); c->rho.resize(n);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const double hi = c->h[i];
        double ni = W_c4(0.0, hi);
        uint32_t cnt = 0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            if (!(c->nbr[k] & FLAG_I)) continue;
            const int64_t j = c->nbr[k] & IDX_MASK;
            double d[3];
            sep(c, i, j, d);
            ni += W_c4(std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]), hi);
            ++cnt;
        }
        c->m[i] = m[i];
        c->V[i] = 1.0 / ni;
        c->rho[i] = (double)m[i] * ni;
        if (V) V[i] = c->V[i];
        if (rho) rho[i] = c->rho[i];
        if (nbr_count) nbr_count[i] = cnt;
    }
    c->stage = 2;
    return 0;
}

// moments (DESIGN.md step 4) then solve
int crk_oracle_rk_coefficients(crk_oracle_ctx* c, double* A, double* B, double* gradA, double* gradB) {
    if (!c || c->stage < 2) return -1;
    set_threads();
    const int64_t n = c->n;
    c->coef.resize(n); c->mom.resize(n);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const double hi = c->h[i];
        Moments M;
        std::memset(&M, 0, sizeof(M));
        M.m0 = c->V[i] * W_c4(0.0, hi);                                  // self term: x = 0, only m0 sees it
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            if (!(c->nbr[k] & FLAG_I)) continue;
            const int64_t j = c->nbr[k] & IDX_MASK;
            double x[3];
            sep(c, i, j, x);
            const double r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
            add_moment_term(M, x, c->V[j] * W_c4(r, hi), c->V[j] * D_c4(r, hi));
        }
        finish_moments(M);
        c->mom[i] = M;
        solve_coef(M, c->coef[i]);
        const Coef& k = c->coef[i];
        if (A) A[i] = k.A;
        for (int a = 0; a < 3; ++a) {
            if (B) B[a * n + i] = k.B[a];
            if (gradA) gradA[a * n + i] = k.dA[a];
            for (int b = 0; b < 3; ++b)
                if (gradB) gradB[(3 * a + b) * n + i] = k.dB[a][b];
        }
    }
    c->stage = 3;
    return 0;
}

int crk_oracle_hydro_derivs(crk_oracle_ctx* c, const float* vx, const float* vy, const float* vz, const float* u,
                            double* ax, double* ay, double* az, double* dudt, uint32_t* pair_count) {
    if (!c || c->stage < 3 || !vx || !vy || !vz || !u) return -1;
    set_threads();
    const int64_t n = c->n;
    c->vx.assign(vx, vx + n); c->vy.assign(vy, vy + n); c->vz.assign(vz, vz + n); c->u.assign(u, u + n);
    c->P.resize(n); c->cs.resize(n); c->gradv.assign((size_t)9 * n, 0.0);
    c->ax.resize(n); c->ay.resize(n); c->az.resize(n);
    const double g = c->p.gamma;
    for (int64_t i = 0; i < n; ++i) {
        c->P[i] = (g - 1.0) * c->rho[i] * c->u[i];                        // Eq. 4 (unclamped, reading S12)
        c->cs[i] = std::sqrt(g * (g - 1.0) * std::max(c->u[i], 0.0));     // c_s = sqrt(gamma P / rho)
    }
    // Eq. 26: grad v_i = - sum_j V_j (v_i - v_j) (x) grad WR_ij   (gather set; self term is zero)
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const double hi = c->h[i];
        double gv[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            if (!(c->nbr[k] & FLAG_I)) continue;
            const int64_t j = c->nbr[k] & IDX_MASK;
            double x[3], gw[3];
            sep(c, i, j, x);
            const double r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
            rk_grad(c->coef[i], x, W_c4(r, hi), D_c4(r, hi), gw);
            const double vij[3] = {c->vx[i] - c->vx[j], c->vy[i] - c->vy[j], c->vz[i] - c->vz[j]};
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) gv[3 * a + b] -= c->V[j] * vij[a] * gw[b];
        }
        for (int q = 0; q < 9; ++q) c->gradv[9 * i + q] = gv[q];
    }
    // Eqs. 17-18 with limited viscosity
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double F[3] = {0, 0, 0}, dE = 0.0;
        uint32_t cnt = 0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            const int64_t j = c->nbr[k] & IDX_MASK;
            PairOut o;
            pair_term(c, i, j, o);
            F[0] += o.F[0]; F[1] += o.F[1]; F[2] += o.F[2]; dE += o.dE;
            ++cnt;
        }
        const double im = 1.0 / c->m[i];
        c->ax[i] = F[0] * im; c->ay[i] = F[1] * im; c->az[i] = F[2] * im;
        if (ax) ax[i] = F[0] * im;
        if (ay) ay[i] = F[1] * im;
        if (az) az[i] = F[2] * im;
        if (dudt) dudt[i] = dE * im;
        if (pair_count) pair_count[i] = cnt;
    }
    c->stage = 4;
    return 0;
}

// NEXT row 4b -- active / passive particles ("all ('active') gas leaves that require force updates will
// evaluate the necessary derivatives ... while the remaining ('passive') leaves are simply streamed").  The same sums as
// crk_oracle_hydro_derivs, restricted to the particles i with active[i] != 0; j ranges over everyone, and grad v (Eq. 26) is
// evaluated for every particle because a passive neighbour's grad v_j enters Eqs. 27-30 of an active i.  Outputs of passive
// particles are set to NaN (they are never evaluated).
int crk_oracle_hydro_derivs_active(crk_oracle_ctx* c, const uint8_t* active, const float* vx, const float* vy, const float* vz,
                                   const float* u, double* ax, double* ay, double* az, double* dudt) {
    if (!c || !active || !ax || !ay || !az || !dudt) return -1;
    const int64_t n = c->n;
    std::vector<double> fx((size_t)n), fy((size_t)n), fz((size_t)n), fe((size_t)n);
    const int rc = crk_oracle_hydro_derivs(c, vx, vy, vz, u, fx.data(), fy.data(), fz.data(), fe.data(), nullptr);
    if (rc) return rc;
    const double nan = std::numeric_limits<double>::quiet_NaN();
    for (int64_t i = 0; i < n; ++i) {
        const bool on = active[i] != 0;
        ax[i] = on ? fx[i] : nan; ay[i] = on ? fy[i] : nan; az[i] = on ? fz[i] : nan; dudt[i] = on ? fe[i] : nan;
    }
    return 0;
}

// ---- oracle at scale: neighbour COUNTS of a full configuration (SURVEY.md section 8(c) "oracle at scale") -------------
// The brute-force scan is O(N^2); for the 128^3 .. 512^3 configurations the counts of every particle come from this second
// formulation: particles are binned in a uniform periodic grid of cells no smaller than the largest h, so every j with
// r < max(h_i, h_j) sits in the 27 cells around i; the predicate is the same prescribed FP32 expression (r2_f32, S3).
// It is pinned by bit-exact agreement with crk_oracle_build on small sets (tests/test_oracle_pins.py).
int crk_oracle_grid_counts(double box, int64_t n, const float* x, const float* y, const float* z, const float* h,
                           uint32_t* nbr_count, uint32_t* pair_count) {
    if (n < 0 || (n > 0 && (!x || !y || !z || !h || !nbr_count || !pair_count))) return -1;
    set_threads();
    const float L = (float)box, half = 0.5f * L;
    float hmax = 0.0f;
    for (int64_t i = 0; i < n; ++i) {
        if (!(h[i] > 0.0f) || !(h[i] < half)) return -1;
        if (!(x[i] >= 0.0f && x[i] < L && y[i] >= 0.0f && y[i] < L && z[i] >= 0.0f && z[i] < L)) return -1;
        hmax = std::max(hmax, h[i]);
    }
    if (n == 0) return 0;
    // cells of side >= hmax (a little larger so that FP32 rounding of r cannot reach across two cells)
    int nc = (int)std::floor((double)L / ((double)hmax * 1.0001));
    nc = std::min(nc, 1024);
    if (nc < 3) return -2;                      // the 27-cell stencil would visit a cell twice: use the brute-force build
    const double inv = (double)nc / (double)L;
    auto cell_of = [&](float p) { int q = (int)std::floor((double)p * inv); return q < 0 ? 0 : (q >= nc ? nc - 1 : q); };
    const int64_t ncell = (int64_t)nc * nc * nc;
    std::vector<int64_t> start((size_t)ncell + 1, 0);
    std::vector<int64_t> cid((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        cid[i] = ((int64_t)cell_of(x[i]) * nc + cell_of(y[i])) * nc + cell_of(z[i]);
        ++start[cid[i] + 1];
    }
    for (int64_t q = 0; q < ncell; ++q) start[q + 1] += start[q];
    std::vector<int64_t> fill(start.begin(), start.end() - 1), order((size_t)n);
    for (int64_t i = 0; i < n; ++i) order[fill[cid[i]]++] = i;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) {
        const float xi = x[i], yi = y[i], zi = z[i], hi2 = h[i] * h[i];
        const int cx = cell_of(xi), cy = cell_of(yi), cz = cell_of(zi);
        uint32_t cg = 0, cs = 0;
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dz = -1; dz <= 1; ++dz) {
                    const int64_t q = ((int64_t)((cx + dx + nc) % nc) * nc + (cy + dy + nc) % nc) * nc + (cz + dz + nc) % nc;
                    for (int64_t k = start[q]; k < start[q + 1]; ++k) {
                        const int64_t j = order[k];
                        if (j == i) continue;
                        const float r2 = r2_f32(xi, yi, zi, x[j], y[j], z[j], L, half);
                        const float hj2 = h[j] * h[j];
                        if (r2 < hi2) ++cg;
                        if (r2 < std::max(hi2, hj2)) ++cs;
                    }
                }
        nbr_count[i] = cg;
        pair_count[i] = cs;
    }
    return 0;
}

// the same CSR neighbour structure as crk_oracle_build, found through the uniform grid of crk_oracle_grid_counts instead of
// the O(N^2) scan (so that volumes .. hydro_derivs can run on a full 128^3 / 256^3 configuration).  Entries of a row are
// sorted by j, which makes the structure identical to the brute-force one (pinned: tests/test_oracle_pins.py).
int crk_oracle_build_grid(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h) {
    if (!c || n < 0 || n >= (int64_t)IDX_MASK || (n > 0 && (!x || !y || !z || !h))) return -1;
    set_threads();
    const float L = (float)c->p.box, half = 0.5f * L;
    float hmax = 0.0f;
    for (int64_t i = 0; i < n; ++i) {
        if (!(h[i] > 0.0f) || !(h[i] < half)) return -1;                                  // reading S13
        if (!(x[i] >= 0.0f && x[i] < L && y[i] >= 0.0f && y[i] < L && z[i] >= 0.0f && z[i] < L)) return -1;
        hmax = std::max(hmax, h[i]);
    }
    int nc = n > 0 ? (int)std::floor((double)L / ((double)hmax * 1.0001)) : 3;
    nc = std::min(nc, 1024);
    if (nc < 3) return -2;
    c->n = n;
    c->x.assign(x, x + n); c->y.assign(y, y + n); c->z.assign(z, z + n); c->h.assign(h, h + n);
    const double inv = (double)nc / (double)L;
    auto cell_of = [&](float p) { int q = (int)std::floor((double)p * inv); return q < 0 ? 0 : (q >= nc ? nc - 1 : q); };
    const int64_t ncell = (int64_t)nc * nc * nc;
    std::vector<int64_t> start((size_t)ncell + 1, 0), cid((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        cid[i] = ((int64_t)cell_of(x[i]) * nc + cell_of(y[i])) * nc + cell_of(z[i]);
        ++start[cid[i] + 1];
    }
    for (int64_t q = 0; q < ncell; ++q) start[q + 1] += start[q];
    std::vector<int64_t> fill(start.begin(), start.end() - 1), order((size_t)n);
    for (int64_t i = 0; i < n; ++i) order[fill[cid[i]]++] = i;
    c->off.assign((size_t)n + 1, 0);
    for (int pass = 0; pass < 2; ++pass) {          // count, then fill
        if (pass == 1) {
            for (int64_t i = 0; i < n; ++i) c->off[i + 1] += c->off[i];
            c->nbr.resize((size_t)c->off[n]);
        }
#pragma omp parallel for schedule(dynamic, 256)
        for (int64_t i = 0; i < n; ++i) {
            const float xi = x[i], yi = y[i], zi = z[i], hi2 = h[i] * h[i];
            const int cx = cell_of(xi), cy = cell_of(yi), cz = cell_of(zi);
            int64_t w = pass == 1 ? c->off[i] : 0;
            for (int dx = -1; dx <= 1; ++dx)
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dz = -1; dz <= 1; ++dz) {
                        const int64_t q = ((int64_t)((cx + dx + nc) % nc) * nc + (cy + dy + nc) % nc) * nc + (cz + dz + nc) % nc;
                        for (int64_t k = start[q]; k < start[q + 1]; ++k) {
                            const int64_t j = order[k];
                            if (j == i) continue;
                            const float r2 = r2_f32(xi, yi, zi, x[j], y[j], z[j], L, half);
                            uint32_t f = 0;
                            if (r2 < hi2) f |= FLAG_I;
                            if (r2 < h[j] * h[j]) f |= FLAG_J;
                            if (!f) continue;
                            if (pass == 0) ++w;
                            else c->nbr[w++] = (uint32_t)j | f;
                        }
                    }
            if (pass == 0) c->off[i + 1] = w;
            else std::sort(c->nbr.begin() + c->off[i], c->nbr.begin() + w,
                           [](uint32_t p, uint32_t q2) { return (p & IDX_MASK) < (q2 & IDX_MASK); });
        }
    }
    c->stage = 1;
    return 0;
}

// ---- NEXT row 2a: time-step criteria, Eqs. 46-50, a = 1, adot = 0, dy/dt = 1, no gravity ----------
// Eq. 50 (sign garbled as printed; reading S17: the approach speed): v_sig,ij = max(-(v_ij . x_ij) / |x_ij|, 0),
//   v_sig,i = max_j v_sig,ij over the pairs of the momentum sweep (r < max(h_i, h_j)).
// Eq. 46: v_max,i = max(v_sig,i, c_s,i, c_sq,i, hhat_i |Tr grad v_i|), c_sq = sqrt(zeta Q_i / rho_i), zeta = 4, with
//   Q_i the largest viscous pressure of particle i over its pairs (reading S18: "maximum viscous sound speed").
// Eq. 47: dt_hyd = C_CFL hhat_i / v_max,i.   Eq. 48 (r_soft = infinity without gravity): dt_acc = sqrt(hhat_i / |dv_i/dt|).
// Eq. 49: dt_min = min(dt_hyd, dt_acc).
int crk_oracle_timestep(crk_oracle_ctx* c, double C_cfl, double* dt_min, double* dt_hyd_out, double* dt_acc_out) {
    if (!c || c->stage < 4 || !dt_min) return -1;
    set_threads();
    const int64_t n = c->n;
    const double inf = std::numeric_limits<double>::infinity();
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double vsig = 0.0, Qmax = 0.0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            const int64_t j = c->nbr[k] & IDX_MASK;
            double x[3];
            sep(c, i, j, x);
            const double r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
            const double vx = (c->vx[i] - c->vx[j]) * x[0] + (c->vy[i] - c->vy[j]) * x[1] + (c->vz[i] - c->vz[j]) * x[2];
            if (r > 0.0) vsig = std::max(vsig, std::max(-vx / r, 0.0));                     // Eq. 50
            PairOut o;
            pair_term(c, i, j, o);
            Qmax = std::max(Qmax, o.Qi);
        }
        const double hhat = (double)c->h[i] / c->p.n_h;
        const double* gv = &c->gradv[9 * i];
        const double div = std::fabs(gv[0] + gv[4] + gv[8]);
        const double csq = std::sqrt(4.0 * Qmax / c->rho[i]);
        const double vmax = std::max(std::max(vsig, c->cs[i]), std::max(csq, hhat * div));  // Eq. 46
        const double th = vmax > 0.0 ? C_cfl * hhat / vmax : inf;                           // Eq. 47
        const double amag = std::sqrt(c->ax[i] * c->ax[i] + c->ay[i] * c->ay[i] + c->az[i] * c->az[i]);
        const double ta = amag > 0.0 ? std::sqrt(hhat / amag) : inf;                        // Eq. 48
        dt_min[i] = std::min(th, ta);                                                       // Eq. 49
        if (dt_hyd_out) dt_hyd_out[i] = th;
        if (dt_acc_out) dt_acc_out[i] = ta;
    }
    return 0;
}

// ---- NEXT row 3: evolved smoothing length, Eqs. 51-53 ---------------------------------------------
// Eq. 51: N_i = (4/3) pi h_i^3 n_i with n_i the SPH number density of Eq. 14.  Target N_res = (4/3) pi n_h^3 (PAPER.md:336,
// reading S1: h is the support radius).  Delta_N = (N_res / N_i)^(1/3).  Eq. 53: lambda = 0.2 (1 + Delta_N^2) if Delta_N < 1,
// 0.2 (1 + 1/Delta_N^3) otherwise.  Eq. 52: h~ = h (1 - lambda + lambda Delta_N).
double crk_oracle_h_update(double h, double n_i, double n_h) {
    const double four_thirds_pi = 4.0 / 3.0 * 3.14159265358979323846;
    const double N_i = four_thirds_pi * h * h * h * n_i;
    const double N_res = four_thirds_pi * n_h * n_h * n_h;
    const double dN = std::cbrt(N_res / N_i);
    const double lambda = dN < 1.0 ? 0.2 * (1.0 + dN * dN) : 0.2 * (1.0 + 1.0 / (dN * dN * dN));
    return h * (1.0 - lambda + lambda * dN);
}

int crk_oracle_evolve_h(crk_oracle_ctx* c, double* h_new) {
    if (!c || c->stage < 2 || !h_new) return -1;
    for (int64_t i = 0; i < c->n; ++i) h_new[i] = crk_oracle_h_update((double)c->h[i], 1.0 / c->V[i], c->p.n_h);
    return 0;
}

// ---- NEXT row 1: compatible energy update, Eqs. 19-23, a = 1, adot = 0, p = v ----------------------
// Eq. 22: v'_i = v_i + (dv_i/dt) dt.   Eq. 20: du_ij = (f_ij / 2) (v_j + v'_j - v_i - v'_i) . a_ij with a_ij the pairwise
// acceleration of Eq. 17 (P -> P + Q).   Eq. 21: dE_ij = m_i du_ij + m_j du_ji; because m_i a_ij = -m_j a_ji
// and f_ij + f_ji = 1 this is (1/2) m_i a_ij . (v_j + v'_j - v_i - v'_i) whatever f is, which is how its sign is taken.
// Eq. 23 as printed is garbled; reading G1: f_ij = min(s_i,s_j)/(s_i+s_j) if (dE_ij >= 0 and s_i >= s_j) or
// (dE_ij < 0 and s_i < s_j), else max(s_i,s_j)/(s_i+s_j), s = P / rho^gamma  ("cooler nodes are heated or hotter nodes
// are cooled", f_ij + f_ji = 1).  Reading S16: if either entropy is not positive (u <= 0, config 2's unstable steps),
// f_ij = 1/2.   Eq. 19: Delta u_i = sum_j du_ij dt.
struct CompatOut { double du, dE, f; };
// kick = optional [3][n] array: the velocity change of each particle over the kick, v' - v, with v the velocities of the last
// crk_oracle_hydro_derivs.  nullptr: Eq. 22 as printed, v' - v = (dv/dt) dt.
inline void pair_compat(const crk_oracle_ctx* c, int64_t i, int64_t j, double dt, CompatOut& o, const double* kick = nullptr) {
    PairOut po;
    pair_term(c, i, j, po);                                   // po.F = m_i a_ij
    const double im = 1.0 / c->m[i];
    const double aij[3] = {po.F[0] * im, po.F[1] * im, po.F[2] * im};
    const double vi[3] = {c->vx[i], c->vy[i], c->vz[i]}, vj[3] = {c->vx[j], c->vy[j], c->vz[j]};
    const double ai[3] = {c->ax[i], c->ay[i], c->az[i]}, aj[3] = {c->ax[j], c->ay[j], c->az[j]};
    const int64_t n = c->n;
    double w = 0.0;
    for (int q = 0; q < 3; ++q) {
        const double vpi = vi[q] + (kick ? kick[q * n + i] : ai[q] * dt);         // Eq. 22
        const double vpj = vj[q] + (kick ? kick[q * n + j] : aj[q] * dt);
        w += (vj[q] + vpj - vi[q] - vpi) * aij[q];
    }
    o.dE = 0.5 * c->m[i] * w;                                                     // Eq. 21
    const double g = c->p.gamma;
    const double si = c->P[i] / std::pow(c->rho[i], g), sj = c->P[j] / std::pow(c->rho[j], g);
    double f = 0.5;
    if (si > 0.0 && sj > 0.0) {
        const bool small = (o.dE >= 0.0 && si >= sj) || (o.dE < 0.0 && si < sj);
        f = (small ? std::min(si, sj) : std::max(si, sj)) / (si + sj);            // Eq. 23 (reading G1)
    }
    o.f = f;
    o.du = 0.5 * f * w;                                                           // Eq. 20
}

int crk_oracle_compatible_energy(crk_oracle_ctx* c, double dt, double* delta_u) {
    if (!c || c->stage < 4 || !delta_u) return -1;
    set_threads();
    const int64_t n = c->n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double s = 0.0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            CompatOut o;
            pair_compat(c, i, (int64_t)(c->nbr[k] & IDX_MASK), dt, o);
            s += o.du;
        }
        delta_u[i] = s * dt;                                                      // Eq. 19 with adot = 0
    }
    return 0;
}

// Eqs. 19-21, 23 for a kick whose velocity change v' - v is given per particle (kick[3][n]) instead of Eq. 22's (dv/dt) dt:
// what the velocity-Verlet step needs, where the second half kick starts from v^1/2 while the derivatives were taken at
// the predicted velocities (crk_oracle.py:kdk_steps).  Reduces to crk_oracle_compatible_energy for kick = (dv/dt) dt.
// (v and v' enter only through v + v' = 2 v + kick, so a kick that starts from v - delta is passed as kick - 2 delta.)
int crk_oracle_compatible_energy_kick(crk_oracle_ctx* c, double dt, const double* kick, double* delta_u) {
    if (!c || c->stage < 4 || !delta_u || !kick) return -1;
    set_threads();
    const int64_t n = c->n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double s = 0.0;
        for (int64_t k = c->off[i]; k < c->off[i + 1]; ++k) {
            CompatOut o;
            pair_compat(c, i, (int64_t)(c->nbr[k] & IDX_MASK), dt, o, kick);
            s += o.du;
        }
        delta_u[i] = s * dt;
    }
    return 0;
}

int crk_oracle_pair_compat(crk_oracle_ctx* c, int64_t i, int64_t j, double dt, double out[3]) {
    if (!c || c->stage < 4 || i < 0 || j < 0 || i >= c->n || j >= c->n || i == j) return -1;
    CompatOut o;
    pair_compat(c, i, j, dt, o);
    out[0] = o.du; out[1] = o.dE; out[2] = o.f;
    return 0;
}

int crk_oracle_step_derivs(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z,
                           const float* h, const float* vx, const float* vy, const float* vz, const float* m,
                           const float* u, double* ax, double* ay, double* az, double* dudt) {
    int rc = crk_oracle_build(c, n, x, y, z, h);
    if (rc) return rc;
    rc = crk_oracle_volumes(c, m, nullptr, nullptr, nullptr);
    if (rc) return rc;
    rc = crk_oracle_rk_coefficients(c, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
    return crk_oracle_hydro_derivs(c, vx, vy, vz, u, ax, ay, az, dudt, nullptr);
}

// -------------------------------------------------------------------------------------- diagnostics
int crk_oracle_get_gradv(crk_oracle_ctx* c, double* gradv) {
    if (!c || c->stage < 4 || !gradv) return -1;
    const int64_t n = c->n;
    for (int64_t i = 0; i < n; ++i)
        for (int q = 0; q < 9; ++q) gradv[q * n + i] = c->gradv[9 * i + q];
    return 0;
}

int crk_oracle_get_moments(crk_oracle_ctx* c, double* m0, double* m1, double* m2) {
    if (!c || c->stage < 3) return -1;
    const int64_t n = c->n;
    for (int64_t i = 0; i < n; ++i) {
        if (m0) m0[i] = c->mom[i].m0;
        for (int a = 0; a < 3; ++a) {
            if (m1) m1[a * n + i] = c->mom[i].m1[a];
            for (int b = 0; b < 3; ++b)
                if (m2) m2[(3 * a + b) * n + i] = c->mom[i].m2[a][b];
        }
    }
    return 0;
}

int crk_oracle_rk_sums(crk_oracle_ctx* c, double* S0, double* S1, double* G0, double* G1) {
    if (!c || c->stage < 3) return -1;
    set_threads();
    const int64_t n = c->n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const double hi = c->h[i];
        const Coef& k = c->coef[i];
        const double zero[3] = {0, 0, 0};
        double g[3];
        double s0 = c->V[i] * rk_kernel(k, zero, W_c4(0.0, hi));
        double s1[3] = {0, 0, 0}, g0[3], g1[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        rk_grad(k, zero, W_c4(0.0, hi), D_c4(0.0, hi), g);
        for (int a = 0; a < 3; ++a) g0[a] = c->V[i] * g[a];
        for (int64_t q = c->off[i]; q < c->off[i + 1]; ++q) {
            if (!(c->nbr[q] & FLAG_I)) continue;
            const int64_t j = c->nbr[q] & IDX_MASK;
            double x[3];
            sep(c, i, j, x);
            const double r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
            const double W = W_c4(r, hi), D = D_c4(r, hi);
            const double wr = rk_kernel(k, x, W);
            rk_grad(k, x, W, D, g);
            s0 += c->V[j] * wr;
            for (int a = 0; a < 3; ++a) {
                s1[a] += c->V[j] * x[a] * wr;
                g0[a] += c->V[j] * g[a];
                for (int b = 0; b < 3; ++b) g1[3 * a + b] += c->V[j] * x[a] * g[b];
            }
        }
        if (S0) S0[i] = s0;
        for (int a = 0; a < 3; ++a) {
            if (S1) S1[a * n + i] = s1[a];
            if (G0) G0[a * n + i] = g0[a];
        }
        if (G1) for (int q = 0; q < 9; ++q) G1[q * n + i] = g1[q];
    }
    return 0;
}

int crk_oracle_eval_AB_at(crk_oracle_ctx* c, const double p[3], double h, double* A, double B[3]) {
    if (!c || c->stage < 2 || !p) return -1;
    const double L = c->p.box, half = 0.5 * L;
    Moments M;
    std::memset(&M, 0, sizeof(M));
    for (int64_t j = 0; j < c->n; ++j) {
        double x[3] = {p[0] - (double)c->x[j], p[1] - (double)c->y[j], p[2] - (double)c->z[j]};
        for (int a = 0; a < 3; ++a) {
            if (x[a] > half) x[a] -= L;
            else if (x[a] < -half) x[a] += L;
        }
        const double r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
        if (r >= h) continue;
        add_moment_term(M, x, c->V[j] * W_c4(r, h), c->V[j] * D_c4(r, h));
    }
    Coef k;
    finish_moments(M);
    solve_coef(M, k);
    if (A) *A = k.A;
    if (B) { B[0] = k.B[0]; B[1] = k.B[1]; B[2] = k.B[2]; }
    return 0;
}

int crk_oracle_pair_term(crk_oracle_ctx* c, int64_t i, int64_t j, double out[4]) {
    if (!c || c->stage < 4 || i < 0 || j < 0 || i >= c->n || j >= c->n || i == j) return -1;
    PairOut o;
    pair_term(c, i, j, o);
    out[0] = o.F[0]; out[1] = o.F[1]; out[2] = o.F[2]; out[3] = o.dE;
    return 0;
}

int crk_oracle_pair_visc(crk_oracle_ctx* c, int64_t i, int64_t j, double out[5]) {
    if (!c || c->stage < 4 || i < 0 || j < 0 || i >= c->n || j >= c->n || i == j) return -1;
    PairOut o;
    pair_term(c, i, j, o);
    out[0] = o.phi; out[1] = o.Qi; out[2] = o.Qj; out[3] = o.mui; out[4] = o.muj;
    return 0;
}

int64_t crk_oracle_neighbors(crk_oracle_ctx* c, int64_t i, uint32_t* buf, int64_t cap) {
    if (!c || c->stage < 1 || i < 0 || i >= c->n) return -1;
    const int64_t cnt = c->off[i + 1] - c->off[i];
    for (int64_t k = 0; k < cnt && k < cap; ++k) buf[k] = c->nbr[c->off[i] + k];
    return cnt;
}

}  // extern "C"
