// crk_internal.cuh -- context, buffers and launch helpers shared by the translation units of libcrk.
// Product code (CUDA, sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include "../../include/crk.h"

#define CRK_LEAF 32              // particles per leaf bucket = one warp lane per particle
#define CRK_BVH_FAN 32           // children per node of the implicit wide tree over leaves
#define CRK_MAX_LEVELS 8
#define CRK_KEY_BITS 16          // space-filling-curve bits per dimension (48-bit keys)

#define CRK_EV_RING 64
#define CRK_EV_N 13
enum { EV_BUILD0 = 0, EV_SORTED, EV_TREE1, EV_BUILD1, EV_VOL0, EV_VOL1, EV_RK0, EV_GV0, EV_GV1, EV_F1, EV_RK1, EV_HY0, EV_PREP1 };

// ---- neighbour lists (lists.cu): per leaf a chain of segments in one arena of 16-byte units --------------------------
//   segment = header (5 units) | cand[C] u32, padded to 4 (not in a leaf's first segment) | ell[K][32] u16
//   header unit 0: {next segment (arena unit, 0 = none), C | CRK_SEG_WRAP | K << 16, 0, 0}; units 1-4: cnt[32] u16
//   the first segment's header is mirrored in dense per-leaf arrays, so that a sweep reaches the payload without a
//   pointer chase: seg_first[leaf] = {next, C | CRK_SEG_WRAP | K << 16, 0, own arena unit (0 = leaf has no segment)},
//   leaf_cnt[leaf][32] = cnt, and cand_first[leaf][CRK_CAND_STRIDE] = the first segment's candidate indices
//   cand[c]   = sorted-order index of candidate c (only candidates accepted by at least one lane of the leaf); in a
//               leaf's first segment cand[0..31] are the leaf's own 32 particles in lane order (always kept)
//   ell[k][l] = k-th entry of lane l: candidate index | CRK_ELL_SYM (h_i^2 <= r2 < h_j^2: a pair of the symmetric set that
//               is not in the lane's gather set; also the padding of rows beyond cnt[l]: CRK_ELL_SYM | slot 0) | CRK_ELL_WRAP
//               (pair crosses the periodic boundary); lane l owns cnt[l]
//               entries; CRK_SEG_WRAP: some entry of the segment may carry CRK_ELL_WRAP (a diagnostic of the builder, shown by
//               crk_get_leaf_segments; the sweeps test the per-entry flag and do not read it)
#define CRK_CCAP 384             // candidates per segment (tile capacity of the sweeps)
#define CRK_CAND_STRIDE 384      // u32 per leaf in cand_first (the sweeps read it in 16-byte groups)
#define CRK_QCAP 128             // entries per lane per segment
#define CRK_TCULL 32             // cull tile of the list builder
#define CRK_SEG_HDR_UNITS 5
#define CRK_ELL_WRAP 0x8000u
#define CRK_ELL_SYM  0x4000u
#define CRK_ELL_MASK 0x3fffu
#define CRK_SEG_WRAP 0x8000u

#define CRK_FLAG_GATHER 0x80000000u   // leaf-list entry: gap(a,b) < hmax(a)   (one-sided passes use it)
#define CRK_FLAG_WRAP   0x40000000u   // leaf pair may straddle the periodic boundary
#define CRK_LEAF_MASK   0x0fffffffu

// device status words (c->flag, mirrored in pinned host memory c->h_flag), read back with ONE copy at the end of a build
enum { FW_ERROR = 0,        // bit 0: input out of range (S13)
       FW_HMIN = 1,         // smallest h, encoded for atomicMax (sort.cu)
       FW_MAXLIST = 2,      // largest leaf interaction list (tree.cu)
       FW_CHECK = 3,        // CRK_CHECKED builds: bit mask of failed internal bound checks
       FW_SUM_GATHER = 4,   // u64: leaf pairs with the gather flag
       FW_SUM_ALL = 6,      // u64: leaf pairs
       FW_ARENA = 8,        // u64: arena units the neighbour lists need
       FW_SETMIXED = 10,    // 1: the supports of the set span more than a factor four (tree.cu: every leaf list built per leaf)
       FW_HOST_ACTIVE = 12, // host side only: crk_select_active
       FW_FALLBACK = 13,    // particles whose m2 counted as singular in the last coefficient sweep (S14), pairs.cu k_rk
       FW_WORDS = 16 };

// CRK_CHECKED builds (python -m paper_2202_02840_b200.build --checked -> libcrk_checked.so): every index the list builder and the
// sweeps form into shared memory, the arena and the particle arrays is range-checked on the device; a failed check sets a
// bit of the status word FW_CHECK (and the access is skipped or clamped), which the next entry point reports as CRK_ECUDA.
// compute-sanitizer is not available on the GPU pool this was developed on; this is the stand-in (profiles/r02_sanitizers.md).
#ifdef CRK_CHECKED
#define CRK_CHECK(flagp, cond, bit) do { if (!(cond)) atomicOr((int*)(flagp) + FW_CHECK, 1 << (bit)); } while (0)
#else
#define CRK_CHECK(flagp, cond, bit) do { } while (0)
#endif

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
};

struct crk_ctx {
    crk_params prm;
    cudaStream_t stream = 0;
    cudaStream_t copy_stream = nullptr;      // crk_step_derivs_host: second H2D stream (created on first use)
    cudaEvent_t ev_copy = nullptr;
    // crk_kdk_step with CRK_FLAG_KDK_REUSE: the arrays the last step's second evaluation was built for
    bool kdk_valid = false;
    const float *kdk_x = nullptr, *kdk_y = nullptr, *kdk_z = nullptr, *kdk_h = nullptr, *kdk_m = nullptr;
    int64_t n = 0, nl = 0;
    int stage = 0;                 // 0 none, 1 built, 2 volumes, 3 coefficients, 4 hydro
    char err[256];
    int64_t launches = 0;
    size_t scratch_bytes = 0;
    int timing = 0;
    cudaEvent_t ev[CRK_EV_RING][CRK_EV_N];   // one event set per step, so a timed loop can be read back afterwards
    bool ev_done[CRK_EV_RING];
    int ev_slot = 0;
    int64_t ev_steps = 0;
    bool ev_ok = false;
    crk_stats st;

    // sort
    DevBuf keys[2], vals[2], hist, scan_tmp;
    DevBuf posh_orig;              // float4 (x,y,z,h) in caller order
    DevBuf posh;                   // float4 (x,y,z,h) in sorted order
    int32_t* perm = nullptr;       // alias into vals[] after the sort
    // leaves + tree
    DevBuf leaf_lo, leaf_hi;       // float4 per node, all levels concatenated; lo.w = hmax of the subtree
    int n_levels = 0;
    int64_t level_off[CRK_MAX_LEVELS + 1];
    int64_t level_cnt[CRK_MAX_LEVELS + 1];
    DevBuf nbr_cnt, nbr_off, nbr_list, nbr_gcnt;   // leaf interaction list: leaf q owns nbr_list[q * leaf_list_cap ...], nbr_cnt[q] entries
    int64_t leaf_list_cap = 0;
    int key_bits = 0;              // space-filling-curve bits per axis of the last build (0 = not known yet)
    int64_t n_pairs = 0, n_pairs_gather = 0;
    DevBuf arena, seg_first;       // neighbour-list arena (16-byte units); per leaf a uint4 copy of its first segment's header
    DevBuf leaf_cnt;               // u16[nl][32]: per-lane entry counts of the first segment (dense, like cand_first)
    DevBuf cand_first;             // u32[nl][CRK_CAND_STRIDE]: candidate indices of the first segment (dense)
    DevBuf act_flags, act_offs, act_ids;   // crk_hydro_derivs_active: leaf flags (active | halo), their scan, compacted leaf ids
    int64_t n_active_leaves = 0, n_halo_leaves = 0;
    int64_t arena_units = 0;       // units used by the last build
    // per-particle state in sorted order
    DevBuf posV;                   // float4 (x,y,z,V)
    DevBuf rho_s;                  // float
    DevBuf coef;                   // 4 planes float4[n]: (A,Bx,By,Bz) (cx,cy,cz,M00) (M01,M02,M10,M11) (M12,M20,M21,M22)
    DevBuf fst;                    // force-sweep state, one 128-byte row per particle (layout at k_rk in pairs.cu)
    DevBuf xv;                     // float4[2] per particle: (x,y,z,1/h) (vx,vy,vz,V), written by the hydro preparation
    DevBuf facc;                   // float4 (dv/dt, s = P / rho^gamma) per particle, sorted, written by k_forces
    DevBuf ts_s;                   // float2 (max approach speed, max Q_i), sorted; only with CRK_FLAG_TIMESTEP
    DevBuf kick;                   // compatible-energy sweep: (v' - v, s) per particle, sorted
    DevBuf kdk;                    // crk_kdk_step scratch: derivatives [4][n] and half-step state [4][n]
    DevBuf u_s;                    // float, specific internal energy in sorted order
    DevBuf vel_orig;               // float4 (vx,vy,vz,u) caller order (packed for a 16-byte gather)
    DevBuf m_s;                    // float, sorted
    DevBuf flag;                   // int[4] device error / status flags
    DevBuf sched;                  // work counter of the persistent sweeps (pairs.cu)
    DevBuf host_stage;             // device staging for crk_step_derivs_host (13 float arrays)
    int* h_flag = nullptr;         // pinned host mirror
    // launch geometry of the persistent sweeps (pairs.cu: persistent_grid), one entry per (kernel, shared memory, threads, device)
    struct GridGeo { const void* kernel = nullptr; int smem = 0, threads = 0, dev = 0, per_sm = 0, sms = 0; };
    static constexpr int GEO_CAP = 16;
    GridGeo geo[GEO_CAP];
    int n_geo = 0;
};

#define CRK_CUDA(c, call)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (call);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            snprintf((c)->err, sizeof((c)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call,        \
                     cudaGetErrorString(e__));                                                     \
            return CRK_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)

#define CRK_TRY(expr)                \
    do {                             \
        int rc__ = (expr);           \
        if (rc__ != CRK_OK) return rc__; \
    } while (0)

static inline void crk_rec(crk_ctx* c, int e) {
    if (c->timing) cudaEventRecord(c->ev[c->ev_slot][e], c->stream);
}

static inline int crk_ensure(crk_ctx* c, DevBuf& b, size_t bytes) {
    if (bytes <= b.cap && b.p) return CRK_OK;
    if (b.p) {
        cudaFree(b.p);
        c->scratch_bytes -= b.cap;
        b.p = nullptr;
        b.cap = 0;
    }
    size_t want = bytes + bytes / 16 + 256;
    cudaError_t e = cudaMalloc(&b.p, want);
    if (e != cudaSuccess) {
        cudaGetLastError();
        snprintf(c->err, sizeof(c->err), "cudaMalloc(%zu bytes) failed: %s", want, cudaGetErrorString(e));
        b.p = nullptr;
        return CRK_ENOMEM;
    }
    b.cap = want;
    c->scratch_bytes += want;
    return CRK_OK;
}

static inline int crk_check_launch(crk_ctx* c, const char* what) {
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(c->err, sizeof(c->err), "launch of %s failed: %s", what, cudaGetErrorString(e));
        return CRK_ECUDA;
    }
    return CRK_OK;
}

// ---- translation-unit entry points (host side) ----
int crk_sort_particles(crk_ctx* c, const float* x, const float* y, const float* z, const float* h, int bits);   // sort.cu
int crk_key_bits_from_hmin(const crk_ctx* c, uint32_t hmin_enc);                                       // sort.cu
int crk_measure_hmin(crk_ctx* c, const float* h, bool sync, uint32_t* enc_out);                       // sort.cu
int crk_exclusive_scan_u32(crk_ctx* c, const uint32_t* in, uint32_t* out, int64_t n, DevBuf& tmp);    // sort.cu
int crk_build_tree_and_list(crk_ctx* c);                                                               // tree.cu
int crk_build_nbr_lists(crk_ctx* c);                                                                   // lists.cu
unsigned long long crk_arena_cap_units(const crk_ctx* c);                                              // lists.cu
int crk_launch_volumes(crk_ctx* c, const float* m, float* V, float* rho, uint32_t* nbr_count);        // pairs.cu
int crk_launch_hydro_prep(crk_ctx* c, const float* vx, const float* vy, const float* vz, const float* u);   // pairs.cu
int crk_launch_rk(crk_ctx* c, bool mom, bool gv, float* A, float* B, float* gradA, float* gradB, float* gradv_full,
                  const int32_t* ids = nullptr, int64_t n_ids = 0);   // pairs.cu
int crk_launch_forces(crk_ctx* c, float* ax, float* ay, float* az, float* dudt, uint32_t* pair_count, const int32_t* ids = nullptr,
                      int64_t n_ids = 0, const uint8_t* active = nullptr);   // pairs.cu
int crk_select_active(crk_ctx* c, const uint8_t* active, int64_t* n_active, int64_t* n_halo);   // pairs.cu
int crk_launch_timestep(crk_ctx* c, float C_cfl, float* dt_min);                                       // pairs.cu
int crk_launch_evolve_h(crk_ctx* c, float* h_new);                                                    // pairs.cu
int crk_launch_compat(crk_ctx* c, float dt, float c1, float c0, const float* bx, const float* by, const float* bz,
                      float* delta_u);                                          // pairs.cu                                                  // pairs.cu
