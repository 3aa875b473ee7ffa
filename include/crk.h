/* crk.h -- C ABI of libcrk: the CRKSPH short-range gas interaction pipeline of CRK-HACC (arxiv 2202.02840) on one
 * NVIDIA B200 (sm_100a).  Hand-written CUDA kernels behind plain pointers; no torch types cross this boundary.
 *
 * What the library computes (citations are lines of /root/reference/PAPER.md; readings S1..S15 are in DESIGN.md):
 *   crk_build_cells      neighbour search structure: space-filling-curve sort, 32-particle leaf buckets with
 *                        bounding boxes extended by the leaf's maximal smoothing length, and the leaf interaction
 *                        list that every hydro kernel reuses (section 3.3), periodic box.
 *   crk_volumes          V_i^-1 = n_i = sum_j W(|x_i-x_j|, h_i)            Eq. 14, Wendland C4 Eq. 12
 *                        rho_i = m_i / V_i (S2); neighbour count #{j != i : r_ij < h_i}
 *   crk_rk_coefficients  A_i, B_i and their gradients from  sum_j V_j WR_ij = 1,  sum_j V_j x_ij WR_ij = 0
 *                         with WR_ij = A_i (1 + B_i.x_ij) W_ij    Eqs. 15-16
 *   crk_hydro_derivs     grad v_i (Eq. 26), limiter phi_ij (Eqs. 28-32), viscous pressure Q (Eqs. 24-25 with the
 *                        midpoint projection of Eq. 27), then dv_i/dt (Eq. 17) and du_i/dt (Eq. 18) with P -> P+Q
 *                        (PAPER.md:120-122, 151); non-cosmological natural units a = 1, adot = 0
 *   crk_step_derivs      the four calls above in order (one "hydro sub-cycle" derivative evaluation)
 *
 * Conventions
 *   - h is the SUPPORT radius: W = 0 for |x| >= h.  n_h relates it to the inter-particle spacing.
 *   - Every array pointer is a DEVICE pointer owned by the caller (except in crk_step_derivs_host), SoA, length n,
 *     float32 / uint32.  Inputs are never modified.  Outputs are written in the caller's particle order.
 *   - Calls are asynchronous on the stream given to crk_create and ordered on it, except that crk_build_cells
 *     synchronises ONCE at its end: one 48-byte read-back carries the input-range flag, the smallest h (which fixes the
 *     width of the sort key), the largest leaf list, the pair totals and the size of the neighbour lists.  The build runs
 *     on what the previous build of the context found for these and is repeated if the data outgrew one of them, so the
 *     result never depends on the history of the context (crk_stats.rebuilds counts the repeats).  The first build of
 *     a context synchronises once more, up front, to learn the smallest h.  crk_hydro_derivs_active synchronises once
 *     (leaf counts); crk_step_derivs_host synchronises at its end; nothing else does.
 *   - State flows build -> volumes -> rk_coefficients -> hydro_derivs inside the context; calling out of order
 *     returns CRK_ESTATE.  The context owns all scratch memory (cudaMalloc, grown on demand, freed by crk_destroy).
 *   - Errors: every call returns CRK_OK (0) or a negative code; nothing aborts or throws across the boundary; there
 *     is no host fallback.  crk_last_error gives a message for the last failure on that context.
 *   - Neighbour predicate (bit-exact contract, S3): d = x_i - x_j in float, wrapped by -+L if |d| > L/2,
 *     r2 = fmaf(dz,dz,fmaf(dy,dy,dx*dx)); j is a neighbour of i iff r2 < h_i*h_i; the pair interacts in
 *     crk_hydro_derivs iff r2 < max(h_i*h_i, h_j*h_j).
 */
#ifndef CRK_H
#define CRK_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define CRK_OK       0
#define CRK_EINVAL  -1   /* null pointer, negative n, bad parameter                                            */
#define CRK_ERANGE  -2   /* some h <= 0 or h >= L/2, or a position outside [0, L)  (checked on the device)    */
#define CRK_ENOMEM  -3   /* device allocation failed                                                          */
#define CRK_ECUDA   -4   /* a CUDA call or kernel failed; see crk_last_error                                  */
#define CRK_ESTATE  -5   /* calls made out of order                                                           */

typedef struct crk_ctx crk_ctx;   /* opaque */

typedef struct {
    float box;        /* cubic periodic box side L; positions in [0, L)                                       */
    float gamma;      /* adiabatic index of Eq. 4                                                             */
    float n_h;        /* particles per support radius: hhat = h/n_h (Eq. 25), eta_crit = 1/n_h,
                         eta_fold = 0.2/n_h.  Paper default 4; the BASELINE configs use 2.4    */
    float C_l, C_q;   /* linear / quadratic viscosity coefficients, (2, 1) in the paper        */
    float eps;        /* 0.1; enters Eq. 25 as eps^2 * hhat^2                                                 */
    int   leaf_size;  /* particles per leaf bucket; must be 32 in this version (one warp lane per particle)   */
    int   flags;      /* 0 or an OR of CRK_FLAG_TIMESTEP (the momentum sweep also reduces what crk_timestep needs),
                         CRK_FLAG_KDK_REUSE and CRK_FLAG_KDK_COMPATIBLE (both about crk_kdk_step), CRK_FLAG_TREE_PER_LEAF, defined below */
} crk_params;

typedef struct {
    int64_t  n;               /* particles in the last build                                                  */
    int64_t  n_leaves;        /* leaf buckets                                                                 */
    int64_t  n_leaf_pairs;    /* entries of the leaf interaction list (symmetric criterion)                   */
    int64_t  n_leaf_pairs_gather; /* of which satisfy the one-sided (gather) criterion                        */
    int64_t  launches;        /* kernels launched by this context since crk_create / crk_reset_stats          */
    int64_t  scratch_bytes;   /* device memory currently owned by the context                                 */
    int64_t  list_bytes;      /* bytes of per-particle neighbour lists written by the last build              */
    float    ms_build, ms_volumes, ms_rk, ms_hydro;   /* mean device time per call of each entry point over the
                                                         steps since crk_reset_stats, when timing is on          */
    float    ms_sort, ms_tree, ms_gradv, ms_forces;   /* finer split: sort+pack | leaves+leaf list | Eq.26 | Eqs.17-18 */
    float    ms_lists;        /* per-particle neighbour lists (third part of crk_build_cells)                  */
    int32_t  timed_steps;     /* number of completed steps the ms_* fields average over (event ring of 64)    */
    int32_t  sort_passes;     /* 8-bit radix passes of the last build (key bits follow the smallest h)         */
    int64_t  n_active_leaves, n_halo_leaves;   /* of the last crk_hydro_derivs_active                                 */
    int32_t  rebuilds;        /* builds repeated since crk_create because the data outgrew the key width, the leaf-list
                                 capacity or the list arena the previous build had found (see crk_build_cells)        */
    int32_t  n_fallback;      /* particles of the last crk_rk_coefficients whose second moment counted as singular, det m2 <=
                                 1e-4 (tr m2 / 3)^3 (fewer than three dimensions spanned: thin sheets, n <= 3), and that therefore
                                 got the zeroth-order correction only (B = 0; reading S14).  0 before that call       */
} crk_stats;

/* stream: a cudaStream_t (0 = default stream).  Returns CRK_OK and *out, or an error.                       */
int  crk_create(crk_ctx** out, const crk_params* params, void* cuda_stream);
void crk_destroy(crk_ctx* c);

/* x, y, z, h: device float[n].  Builds the sorted particle order, leaves and the leaf interaction list.     */
int  crk_build_cells(crk_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h);
/* m: device float[n].  V, rho: device float[n] or NULL.  nbr_count: device uint32[n] or NULL.               */
int  crk_volumes(crk_ctx* c, const float* m, float* V, float* rho, uint32_t* nbr_count);
/* A: float[n]; B: float[3][n]; gradA: float[3][n] (index c: d_c A); gradB: float[9][n] (index 3*c+a: d_c B^a).
 * Any may be NULL (the coefficients are kept inside the context for crk_hydro_derivs either way).           */
int  crk_rk_coefficients(crk_ctx* c, float* A, float* B, float* gradA, float* gradB);
/* vx, vy, vz, u: device float[n] (u = specific internal energy).  ax, ay, az = dv/dt, dudt = du/dt: device
 * float[n].  pair_count: device uint32[n] or NULL = #{j != i : r_ij < max(h_i, h_j)}.                        */
int  crk_hydro_derivs(crk_ctx* c, const float* vx, const float* vy, const float* vz, const float* u,
                      float* ax, float* ay, float* az, float* dudt, uint32_t* pair_count);
/* build_cells + volumes + rk_coefficients + hydro_derivs.  All device pointers.                             */
int  crk_step_derivs(crk_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h,
                     const float* vx, const float* vy, const float* vz, const float* m, const float* u,
                     float* ax, float* ay, float* az, float* dudt);
/* Same, with HOST pointers (pinned memory recommended): copies the nine inputs to the device, evaluates, copies
 * the four outputs back and synchronises the stream.  This is the end-to-end entry bench.py's `e2e` times.  */
int  crk_step_derivs_host(crk_ctx* c, int64_t n, const float* x, const float* y, const float* z, const float* h,
                          const float* vx, const float* vy, const float* vz, const float* m, const float* u,
                          float* ax, float* ay, float* az, float* dudt);

/* ---- NEXT row 1: compatible energy update, Eqs. 19-23, PAPER.md:126-141 -------------
 * After crk_hydro_derivs (else CRK_ESTATE).  With a = 1, adot = 0, p = v:
 *   delta_u[i] = dt * sum_j (f_ij / 2) (v_j + v'_j - v_i - v'_i) . a_ij,   v' = v + (dv/dt) dt  (Eq. 22),
 * a_ij = the pairwise acceleration of Eq. 17 (with Q), f_ij the entropy-weighted partition of Eq. 23 (DESIGN.md reading
 * G1; 1/2 when an entropy P / rho^gamma is not positive).  sum_i m_i delta_u_i = -(kinetic energy change of v -> v').
 * delta_u: device float[n], caller order, written.  One more symmetric pair sweep on the resident state.          */
int  crk_compatible_energy(crk_ctx* c, float dt, float* delta_u);

/* ---- NEXT row 2b: hydro-only velocity-Verlet step U_V, Eq. 43, PAPER.md:232-241 (a = 1, dt/dy = 1, p = v) --------
 * Advances the caller's device arrays IN PLACE by one step dt (x, y, z wrapped into [0, box); h, m untouched):
 *   v^1/2 = v + a dt/2, u^1/2 = u + udot dt/2;  x^1 = x + v^1/2 dt;  predictions v_p = v^1/2 + a dt/2, u_p likewise;
 *   v^1 = v^1/2 + a(x^1, v_p, u_p) dt/2,  u^1 = u^1/2 + udot(x^1, v_p, u_p) dt/2,
 * a and udot from two full crk_step_derivs evaluations (udot = Eq. 18, reading S19).  Errors as
 * crk_step_derivs (CRK_ERANGE if the state leaves the admissible range).  The context is left in the state of the
 * second evaluation (predicted velocities), so crk_timestep / crk_compatible_energy afterwards refer to that state.
 * On failure of the SECOND evaluation (e.g. CRK_ERANGE: a predicted position left the admissible range) the arrays are
 * left at the predicted state x^1, v_p, u_p -- the step is not rolled back; keep a copy if a retry with a smaller dt is
 * wanted.                                                                                                            */
/* CRK_FLAG_KDK_REUSE (crk_params.flags): consecutive crk_kdk_step calls on the same arrays reuse sort, tree, neighbour
 * lists, volumes and RK coefficients of the previous step's second evaluation for their first one (same x, h, m).  Set it
 * only if nothing but crk_kdk_step changes x, y, z, h, m between the calls (the check is by array address): any
 * crk_build_cells / crk_volumes / crk_rk_coefficients call in between drops the reuse, and so does crk_evolve_h (its
 * caller is about to change h, possibly in place).                                                                  */
#define CRK_FLAG_KDK_REUSE 2
/* CRK_FLAG_KDK_COMPATIBLE: the two half kicks of crk_kdk_step advance u with the compatible energy of Eqs. 19-23 (each for
 * its own velocity change and pair accelerations, reading S20) instead of Eq. 18's rate: total energy is then
 * conserved to roundoff -- the paper's fiducial energy integration.  Two more pair sweeps per step.     */
#define CRK_FLAG_KDK_COMPATIBLE 4
/* CRK_FLAG_TREE_PER_LEAF: crk_build_cells builds every leaf interaction list with the per-leaf tree walk.  Without it, sets of
 * 2048 or more level-1 nodes whose supports span less than a factor four walk the tree once per node of 32 leaves (same
 * entries in the same order; tests compare the two).  */
#define CRK_FLAG_TREE_PER_LEAF 8
int  crk_kdk_step(crk_ctx* c, int64_t n, float* x, float* y, float* z, const float* h, float* vx, float* vy, float* vz,
                  const float* m, float* u, float dt);

/* ---- NEXT row 2a: time-step criteria, Eqs. 46-50, PAPER.md:262-276 (a = 1, adot = 0, no gravity) ----------------
 * Needs a context created with CRK_FLAG_TIMESTEP in crk_params.flags and a completed crk_hydro_derivs (else CRK_ESTATE):
 *   v_max = max(v_sig, c_s, sqrt(4 Q_max / rho), hhat |Tr grad v|),  v_sig = max_j max(-(v_ij.x_ij)/|x_ij|, 0)  (S17),
 *   Q_max = max over the particle's pairs of its Q of Eq. 24 (S18),   dt_min = min(C_cfl hhat / v_max, sqrt(hhat / |dv/dt|)).
 * dt_min: device float[n], caller order, written (inf where both criteria are unbounded).  One stream pass; the two
 * maxima ride on the momentum sweep (two fmax per pair).                                                           */
#define CRK_FLAG_TIMESTEP 1
int  crk_timestep(crk_ctx* c, float C_cfl, float* dt_min);

/* ---- NEXT row 3: evolved smoothing length, Eqs. 51-53, PAPER.md:340-354 -----------------------------------------
 * After crk_volumes (else CRK_ESTATE): h_new[i] = h_i (1 - lambda + lambda Delta_N) with Delta_N^3 = N_res / N_i,
 * N_i = (4/3) pi h_i^3 / V_i (Eq. 51), N_res = (4/3) pi n_h^3, lambda of Eq. 53.  h_new: device float[n], caller order,
 * written (may alias nothing the library reads later: the build keeps its own copy of h).  One stream pass that moves 40 B
 * per particle (two 16-byte packed records, the permutation, the result).                                            */
int  crk_evolve_h(crk_ctx* c, float* h_new);

/* ---- NEXT row 4b: active / passive particles, PAPER.md:282 ("all ('active') gas leaves that require force updates will
 * evaluate the necessary derivatives ... while the remaining ('passive') leaves are simply streamed") -----------------
 * After crk_rk_coefficients (else CRK_ESTATE).  active: device uint8[n], caller order.  Evaluates Eqs. 17-18 (with the
 * limited viscosity, as crk_hydro_derivs) for the particles with active[i] != 0 only and writes ax, ay, az, dudt THERE;
 * entries of passive particles are left untouched.  j ranges over all particles.  Internally a 32-particle leaf is active
 * when one of its particles is; the force sweep runs over the active leaves, the Eq. 26 sweep over the leaves of their
 * interaction lists (a passive neighbour's grad v_j enters Eqs. 27-30 of an active particle).  Synchronises once (leaf
 * counts).  The context is left at the stage of crk_rk_coefficients: crk_compatible_energy / crk_timestep need a full
 * crk_hydro_derivs.
 * What it saves.  The unit of work is the LEAF (32 consecutive particles of the curve order, crk_get_perm), and the stream
 * passes that pack v and u still run over all n particles.  A mask scattered at random over the box therefore saves
 * little: with 10 % of the particles of the 256^3 benchmark set active, half of the leaves hold an active particle and
 * nearly all are in some interaction list (10.9 ms against 16.3 ms for all particles); the same 10 % chosen as whole
 * leaves, or as a compact region, costs in proportion.  Choose the active set per leaf where the integrator allows it:
 * particles perm[32 q .. 32 q + 31] form leaf q.                                                                       */
int  crk_hydro_derivs_active(crk_ctx* c, const uint8_t* active, const float* vx, const float* vy, const float* vz,
                             const float* u, float* ax, float* ay, float* az, float* dudt);

/* ---- for callers that must not allocate device memory: the space-filling-curve order without a context ----------------
 * Who this is for.  A simulation code that claims nearly all of the device memory for its own arena at start-up (HACC-style
 * hosts do) leaves nothing for a library's cudaMalloc later on, and a time step that has gravity and hydro kernels in
 * flight on several streams cannot afford one either: cudaMalloc and cudaFree stall the whole device until everything
 * queued has drained.  Every other entry point of this header works on a crk_ctx, which grows its scratch buffers with
 * cudaMalloc on demand.  This one does not: it needs no context and makes no cudaMalloc / cudaFree / cudaMallocHost call,
 * now or later.
 * What it does.  The first half of crk_build_cells (section 3.3): validates the input as crk_build_cells
 * does, forms the Hilbert keys on the grid whose cells are half the smallest h (at most 16 bits per axis), sorts them
 * with the library's stable 8-bit LSD radix sort, and writes perm[k] = caller index of the k-th particle along the curve
 * -- bit for bit what crk_get_perm returns after a crk_build_cells of the same x, y, z, h on a fresh context with the same
 * box.  A caller can use it to put its own arrays in the order in which 32 consecutive particles form a compact leaf.
 * Arguments.  x, y, z, h: device float[n], read only.  perm: device int32[n], written.  box as in crk_params.  n from 0
 * (nothing is done) to CRK_NOALLOC_MAX_N; a larger n is refused with CRK_EINVAL before anything is launched.  errbuf:
 * host char[errbuf_len] or NULL; receives a one-line message when the return value is not CRK_OK.
 * Where the scratch lives.  The sort's working set (two key and two index buffers, the packed copy of the input that the
 * key kernel writes, the digit histograms and their scan, two status words; CRK_NOALLOC_SCRATCH_BYTES = about 10.3 MB for
 * CRK_NOALLOC_MAX_N = 262 144 particles) is a fixed array inside the library's device image.  Every GPU onto which the
 * library's device code is loaded holds those bytes until the process exits, whether or not this function is ever called
 * there.
 * First call on a device.  The first call made with a given device current looks up the device address of that array
 * (cudaGetSymbolAddress) and remembers it for that device; make this first call outside any stream capture, e.g. once
 * during start-up with n = 0.  Later calls on that device only launch kernels, two small device-to-host copies and one
 * device-to-device copy on `cuda_stream`.
 * Sharing.  All calls on one device use the same array, and it still holds what the previous call left there.  The function
 * clears the two status words it needs at zero itself, on the stream, at the start of each call; everything else is
 * overwritten before it is read.  Two calls whose GPU work can overlap (different streams, or different host threads) race
 * on the array and give garbage: serialise them.
 * Synchronisation and errors.  Synchronises `cuda_stream` twice (after measuring the smallest h, and at the end to read
 * the range flag), so perm is complete on return.  CRK_EINVAL: null pointer with n > 0, n < 0, n > CRK_NOALLOC_MAX_N or box
 * <= 0; CRK_ERANGE: a position outside [0, box) or an h outside (0, box/2) (perm is then unspecified); CRK_ECUDA: a CUDA call
 * failed.                                                                                                              */
#define CRK_NOALLOC_MAX_N 262144
#define CRK_NOALLOC_SCRATCH_BYTES 10765056
int  crk_sfc_order_noalloc(void* cuda_stream, int64_t n, const float* x, const float* y, const float* z, const float* h,
                           float box, int32_t* perm, char* errbuf, int errbuf_len);

/* ---- diagnostics ---- */
const char* crk_last_error(const crk_ctx* c);
int  crk_get_perm(crk_ctx* c, int32_t* perm);        /* device int32[n]: perm[k] = caller index of sorted slot k   */
int  crk_get_gradv(crk_ctx* c, float* gradv);         /* device float[9][n], index 3*a+b = d_b v^a (Eq. 26), caller order */
/* device uint32[n_leaves][4]: first neighbour-list segment of every leaf = {next segment (0 = none), C | 0x8000 if some entry
 * crosses the periodic boundary | K << 16, 0, arena unit}; C = candidate slots, K = rows of the entry block (layout:
 * csrc/crk_internal.cuh)                                                                                       */
int  crk_get_leaf_segments(crk_ctx* c, uint32_t* seg);
int  crk_get_stats(crk_ctx* c, crk_stats* out);       /* host struct; synchronises the stream (reads n_fallback, the timings) */
int  crk_reset_stats(crk_ctx* c);
int  crk_set_timing(crk_ctx* c, int on);              /* record CUDA events around each pass (adds stream syncs when read) */
/* leaf interaction list of leaf `leaf` (host buffer): entries leaf_index | bit31 (gather) | bit30 (periodic wrap);
 * returns the number of entries (may exceed cap) or a negative error.  Synchronises.                         */
int64_t crk_get_leaf_list(crk_ctx* c, int64_t leaf, uint32_t* host_buf, int64_t cap);

/* Measurement aid (not part of the method): runs a register-resident FFMA loop on every SM and returns the achieved
 * FP32 rate in flop/s (FMA = 2 flops) for bench.py's roofline denominator; *ms_out receives the kernel time.  */
double crk_measure_fp32_peak(void* cuda_stream, int repeats, float* ms_out);
/* The same loop with three register operands per FFMA (a = b * c + a, the form of every accumulated pair sum).  On B200 the
 * register file feeds such a stream at about 61 % of the rate of the forms with at most two register operands, so this is
 * the rate the accumulating part of the pair sweeps can reach; reported by bench.py beside the nominal peak.  */
double crk_measure_fp32_peak_3reg(void* cuda_stream, int repeats, float* ms_out);

#ifdef __cplusplus
}
#endif
#endif
