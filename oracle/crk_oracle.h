/* crk_oracle.h -- CPU ORACLE for the CRKSPH short-range gas pipeline.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct FP64 implementation of what the hot path computes, written from
 * /root/reference/PAPER.md (arxiv 2202.02840) section 2.2, Eqs. 12-18 and 24-32, with the readings
 * listed in DESIGN.md ("Readings of the paper").  Neighbours are found by a brute-force O(N^2) periodic
 * minimum-image scan; sums run over exactly those sets.  No cells, no tiles, no fusion.
 *
 * It shares NO code with the CUDA library (paper_2202_02840_b200/csrc) and neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * All pointers are HOST pointers.  Inputs are the same float32 arrays the CUDA library receives; every
 * value is promoted to double -- except the neighbour predicate, which is evaluated in prescribed FP32
 * (reading S3) so that neighbour sets are a bit-exact contract rather than a rounding accident.
 *
 * Pin status (tests/test_oracle_pins.py): kernel, volumes, moments, A, B, gradA, gradB, RK gradient,
 * grad v, momentum/energy pair antisymmetry are pinned by invariants; the limiter (phi_VL off r = 1, phi_ad), mu, Q and
 * the pair terms of Eqs. 17-18 are pinned against the paper's PRINTED forms rebuilt in numpy with the golden constants
 * (C_l, C_q, eps, eta_fold/eta_crit), incl. closed-form pairs (head-on approach, close approach in a linear flow).
 * The zeroth-order fallback of solve_coef for a singular m2 (S14: B = 0, A = 1/m0, grad A = -A^2 grad m0) is pinned against
 * the zeroth-moment constraint of PAPER.md:116, its gradient and finite differences of A on sets that span fewer than three
 * dimensions; the position of the singularity line is pinned from both sides (first-moment condition holds above it, equals
 * A m1 below it) within a factor ten (test_S14_*).
 * PARITY UNPINNED
 * (fixed by DESIGN.md readings only): Eq. 18 P_j-vs-P_i choice (S6), rho = m/V for unequal masses (S2),
 * c_s clamp max(u,0) (S12), and the VALUE 1e-4 of S14's threshold det m2 <= 1e-4 (tr m2 / 3)^3: the paper gives no number.
 * A particle whose ratio lies within FP32 rounding of the line can take different branches here (FP64 sums) and in the CUDA
 * library (FP32 sums); the parity fixtures stay a factor two away from it (smallest ratio 2.0e-4).
 */
#ifndef CRK_ORACLE_H
#define CRK_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct crk_oracle_ctx crk_oracle_ctx;

typedef struct {
    double box;    /* cubic periodic box side L, positions in [0,L)                         */
    double gamma;  /* adiabatic index, Eq. 4                                                */
    double n_h;    /* hhat = h/n_h (Eq. 25); eta_crit = 1/n_h, eta_fold = 0.2/n_h (l.179)   */
    double C_l, C_q; /* (2,1)                                                 */
    double eps;    /* 0.1, enters as eps^2 * hhat^2 in Eq. 25                               */
} crk_oracle_params;

crk_oracle_ctx* crk_oracle_create(const crk_oracle_params* p);
void            crk_oracle_destroy(crk_oracle_ctx* c);
void            crk_oracle_set_threads(int nthreads);   /* 0 = all cores */
int             crk_oracle_get_threads(void);

/* neighbour search (brute force, periodic): returns 0, or -1 on bad input (h<=0, h>=L/2, x outside [0,L)) */
int crk_oracle_build(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h);
/* Eq. 14 + S2: V = 1/sum_j W(r_ij,h_i) (self included), rho = m/V; nbr_count = #{j!=i : r_ij < h_i}      */
int crk_oracle_volumes(crk_oracle_ctx* c, const float* m, double* V, double* rho, uint32_t* nbr_count);
/* PAPER.md:116 constraints: A[n], B[3][n], gradA[3][n] (d_c A), gradB[9][n] (index 3*c+a = d_c B^a)    */
int crk_oracle_rk_coefficients(crk_oracle_ctx* c, double* A, double* B, double* gradA, double* gradB);
/* Eqs. 26, 27-32, 24-25, 17-18: a = dv/dt [n] x3, dudt [n]; pair_count = #{j!=i : r_ij < max(h_i,h_j)}    */
int crk_oracle_hydro_derivs(crk_oracle_ctx* c, const float* vx, const float* vy, const float* vz, const float* u,
                            double* ax, double* ay, double* az, double* dudt, uint32_t* pair_count);
/* the four calls above in order */
int crk_oracle_step_derivs(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z,
                           const float* h, const float* vx, const float* vy, const float* vz, const float* m,
                           const float* u, double* ax, double* ay, double* az, double* dudt);

/* NEXT row 1 -- compatible energy update, Eqs. 19-23 with a = 1, adot = 0, after
 * crk_oracle_hydro_derivs: delta_u[i] = dt * sum_j (f_ij/2) (v_j + v'_j - v_i - v'_i) . a_ij, v' = v + (dv/dt) dt.
 * Pinned: sum_i m_i delta_u_i + Delta KE = 0 to roundoff, f_ij + f_ji = 1, the heating/cooling rule of PAPER.md:141.
 * PARITY UNPINNED: the exact form of the garbled Eq. 23 (reading G1) and f = 1/2 for s <= 0 (S16).      */
int crk_oracle_compatible_energy(crk_oracle_ctx* c, double dt, double* delta_u);
/* the same for a kick with a given velocity change per particle, kick[3][n] = v' - v (v = velocities of the last
 * hydro_derivs): delta_u[i] = dt * sum_j (f_ij/2) (2 (v_j - v_i) + kick_j - kick_i) . a_ij.  Pinned: equals the call above
 * for kick = (dv/dt) dt; makes the Verlet step of crk_oracle.py:kdk_steps(compatible=True) conserve energy to roundoff.   */
int crk_oracle_compatible_energy_kick(crk_oracle_ctx* c, double dt, const double* kick, double* delta_u);
/* one pair of the above: out = { du_ij (Eq. 20), dE_ij (Eq. 21), f_ij (Eq. 23) }                                 */
int crk_oracle_pair_compat(crk_oracle_ctx* c, int64_t i, int64_t j, double dt, double out[3]);

/* NEXT row 4b -- active / passive particles: crk_oracle_hydro_derivs restricted to the particles with
 * active[i] != 0 (j ranges over everyone; grad v is evaluated for all, a passive neighbour's grad v_j enters Eqs. 27-30 of an
 * active i).  Outputs of passive particles are NaN.  Pinned: mask = all gives the bits of crk_oracle_hydro_derivs; the
 * results of an active particle do not depend on which other particles are active.                                      */
int crk_oracle_hydro_derivs_active(crk_oracle_ctx* c, const uint8_t* active, const float* vx, const float* vy,
                                   const float* vz, const float* u, double* ax, double* ay, double* az, double* dudt);

/* Oracle at scale: nbr_count[i] = #{j != i : r_ij < h_i} and pair_count[i] = #{j != i : r_ij < max(h_i, h_j)} of a FULL
 * configuration through a uniform periodic grid of cells >= h_max (27-cell stencil) with the same FP32 predicate (S3).
 * Pinned by bit-exact agreement with crk_oracle_build / _volumes / _hydro_derivs counts on small sets.  Returns -2 if
 * the box holds fewer than 3 cells per side (use the brute-force build then), -1 on bad input.                        */
int crk_oracle_grid_counts(double box, int64_t n, const float* x, const float* y, const float* z, const float* h,
                           uint32_t* nbr_count, uint32_t* pair_count);

/* crk_oracle_build through the same uniform grid (identical neighbour structure, rows sorted by j): lets volumes ..
 * hydro_derivs run on a full 128^3 / 256^3 configuration.  -2 if the box holds fewer than 3 cells per side.          */
int crk_oracle_build_grid(crk_oracle_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h);

/* NEXT row 2a -- time-step criteria, Eqs. 46-50 with a = 1, adot = 0, no gravity, after
 * crk_oracle_hydro_derivs: dt_min = min(C_cfl hhat / max(v_sig, c_s, sqrt(4 Q_max / rho), hhat |Tr grad v|), sqrt(hhat / |a|)).
 * dt_hyd / dt_acc (nullable) return the two criteria separately.  Pinned: static gas closed form C hhat / c_s, linear
 * compression closed form, acceleration criterion from the Eq. 17 pair diagnostic.  PARITY UNPINNED: the sign reading
 * of the garbled Eq. 50 (S17) and "Q_i" = the maximum over pairs (S18).                                              */
int crk_oracle_timestep(crk_oracle_ctx* c, double C_cfl, double* dt_min, double* dt_hyd, double* dt_acc);

/* NEXT row 3 -- evolved smoothing length, Eqs. 51-53, after crk_oracle_volumes:
 * h_new[i] = h_i (1 - lambda + lambda Delta_N), Delta_N^3 = N_res / N_i, N_i = (4/3) pi h_i^3 / V_i, N_res = (4/3) pi n_h^3.
 * Pinned: hand-evaluated values of Eqs. 52-53 at Delta_N = 1/2, 1, 2; continuity of lambda at 1; iteration -> N_res.    */
int    crk_oracle_evolve_h(crk_oracle_ctx* c, double* h_new);
double crk_oracle_h_update(double h, double n_i, double n_h);   /* the per-particle rule on its own */

/* ---- diagnostics used by the pins (tests only) ---- */
double crk_oracle_W(double r, double h);        /* Eq. 12                                   */
double crk_oracle_dWdr(double r, double h);     /* its radial derivative                    */
/* raw moments after crk_oracle_rk_coefficients: m0[n], m1[3][n], m2[9][n] (index 3*a+b); any may be NULL */
int crk_oracle_get_moments(crk_oracle_ctx* c, double* m0, double* m1, double* m2);
/* after crk_oracle_hydro_derivs */
int crk_oracle_get_gradv(crk_oracle_ctx* c, double* gradv /* [9][n], index 3*alpha+beta = d_beta v^alpha */);
/* S0_i = sum_j V_j WR_ij ; S1_i = sum_j V_j x_ij WR_ij ; G0_i = sum_j V_j grad WR_ij ;
 * G1_i[3*a+c] = sum_j V_j x_ij^a (grad WR_ij)^c   (sums over the gather set incl. self)                */
int crk_oracle_rk_sums(crk_oracle_ctx* c, double* S0, double* S1, double* G0, double* G1);
/* A, B of the reproducing kernel centred at an arbitrary point p with support h, sources = all particles with
 * their V_j held fixed (reading S5); brute force over all particles                                     */
int crk_oracle_eval_AB_at(crk_oracle_ctx* c, const double p[3], double h, double* A, double B[3]);
/* contribution of neighbour j to particle i in Eqs. 17/18: out = { m_i a_{i<-j} (3), m_i du_{i<-j} }       */
int crk_oracle_pair_term(crk_oracle_ctx* c, int64_t i, int64_t j, double out[4]);
/* limiter phi_ij and viscous pressures Q_i, Q_j of a pair (Eqs. 24-32): out = {phi, Q_i, Q_j, mu_i, mu_j}  */
int crk_oracle_pair_visc(crk_oracle_ctx* c, int64_t i, int64_t j, double out[5]);
/* neighbour list of i: entries j | flags (bit31: r<h_i, bit30: r<h_j); returns count (may exceed cap)    */
int64_t crk_oracle_neighbors(crk_oracle_ctx* c, int64_t i, uint32_t* buf, int64_t cap);

#ifdef __cplusplus
}
#endif
#endif
