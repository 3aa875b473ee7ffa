// pairs.cu -- steps a1..a5: the four pair sweeps of one CRKSPH derivative evaluation (FP32 pair math on the FMA pipes).
//
// Common structure (one warp = one 32-particle leaf, one lane = one particle i, state of i in registers):
//   for each neighbour leaf b of the leaf interaction list (tree.cu):
//     cull    lane l takes particle l of b and tests it against the bounding box of the warp's own leaf (point-to-box gap
//             vs the leaf's hmax, same monotone float sequence as the predicate, so nothing is lost); survivors are
//             compacted (ballot + prefix popc) into a warp-private shared-memory tile of CAP slots, all planes
//   when the tile is full (and at the end):
//     test    every staged j against the lane's i with the prescribed FP32 predicate (S3); all lanes read the
//             same j (shared-memory broadcast); accepted slots are appended to a per-lane byte queue
//     drain   each lane walks its own queue and evaluates the pair math only for accepted pairs (lane divergence is
//             limited to the spread of queue lengths over one tile instead of the few-% acceptance rate)
// Equation numbers refer to /root/reference/PAPER.md; the closed forms of A, B, grad A, grad B are derived in DESIGN.md.
#include "crk_internal.cuh"

namespace {

constexpr int WPC = 4;                       // warps (= leaves) per CTA
constexpr float SIGMA_C4 = 4.923856051905513f;     // 495 / (32 pi), Eq. 12
constexpr float C35_3 = 35.0f / 3.0f;
constexpr float C56_3 = 56.0f / 3.0f;
constexpr float R2_TINY = 1.0e-37f;

struct SweepArgs {
    int64_t n, nl;
    float L, half;
    const uint32_t* __restrict__ off;     // leaf list CSR offsets [nl+1]
    const uint32_t* __restrict__ list;    // entries: leaf | flags
    const int32_t* __restrict__ perm;     // sorted slot -> caller index
    const float4* __restrict__ posh;      // (x,y,z,h)
    const float4* __restrict__ leaf_lo;   // per leaf: (xlo,ylo,zlo,hmax)
    const float4* __restrict__ leaf_hi;   // per leaf: (xhi,yhi,zhi,hmin)
    float4* __restrict__ posV;            // (x,y,z,V)
    float4* __restrict__ velV;            // (vx,vy,vz,V)
    float4* __restrict__ thermo;          // (P,rho,cs,1/h)
    float4* __restrict__ coef;            // 4 planes, stride np
    float4* __restrict__ gv;              // 3 planes, stride np
    float* __restrict__ rho_s;
    const float* __restrict__ m_s;
    int64_t np;                           // padded particle count nl*32 (plane stride)
    float gamma, n_h, C_l, C_q, eps2;
    // outputs in caller order (may be null)
    float* __restrict__ o0; float* __restrict__ o1; float* __restrict__ o2; float* __restrict__ o3;
    uint32_t* __restrict__ ocnt;
};

__device__ __forceinline__ float wrap1(float d, float L, float half) {
    return d > half ? __fsub_rn(d, L) : (d < -half ? __fadd_rn(d, L) : d);
}

// ---- culling helpers: lower bound of |wrap(x_i - x_j)| on one axis for x_i in [lo,hi] (monotone float ops) -------
__device__ __forceinline__ float gap1(float lo, float hi, float x) {
    return fmaxf(0.f, fmaxf(__fsub_rn(lo, x), __fsub_rn(x, hi)));
}
__device__ __forceinline__ float gap1_wrap(float lo, float hi, float x, float L) {
    const float dmin = __fsub_rn(lo, x), dmax = __fsub_rn(hi, x);     // d = x_i - x_j ranges over [dmin, dmax]
    const float g0 = fmaxf(0.f, fmaxf(dmin, -dmax));
    const float gp = fmaxf(0.f, fmaxf(__fsub_rn(L, dmax), __fsub_rn(dmin, L)));
    const float gm = fmaxf(0.f, fmaxf(__fadd_rn(dmin, L), __fsub_rn(-L, dmax)));
    return fminf(g0, fminf(gp, gm));
}

// ---- test phase: append accepted slots to the lane's byte queue; returns queue length -------------------------------
// SYM = false: gather predicate r2 < h_i^2 (Eqs. 13-14: W_ij = W(|x_i-x_j|, h_i));   SYM = true: r2 < max(h_i^2,h_j^2)
template <bool SYM>
__device__ __forceinline__ int test_slots(const SweepArgs& a, int fill4, bool wrap, int self_slot, int lane, float xi,
                                          float yi, float zi, float hi2, const float4* tile, uint8_t* queue) {
    uint8_t* qp = queue + lane;
    if (!wrap) {
#pragma unroll 1
        for (int s = 0; s < fill4; s += 4) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4 pj = tile[s + u];
                const float dx = __fsub_rn(xi, pj.x), dy = __fsub_rn(yi, pj.y), dz = __fsub_rn(zi, pj.z);
                const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                const float lim = SYM ? fmaxf(hi2, __fmul_rn(pj.w, pj.w)) : hi2;
                if (r2 < lim && (s + u) != self_slot) {
                    *qp = (uint8_t)(s + u);
                    qp += 32;
                }
            }
        }
    } else {
#pragma unroll 1
        for (int s = 0; s < fill4; ++s) {
            const float4 pj = tile[s];
            const float dx0 = __fsub_rn(xi, pj.x), dy0 = __fsub_rn(yi, pj.y), dz0 = __fsub_rn(zi, pj.z);
            const float dx = wrap1(dx0, a.L, a.half), dy = wrap1(dy0, a.L, a.half), dz = wrap1(dz0, a.L, a.half);
            const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const float lim = SYM ? fmaxf(hi2, __fmul_rn(pj.w, pj.w)) : hi2;
            if (r2 < lim && s != self_slot) {
                const bool wrapped = (dx != dx0) || (dy != dy0) || (dz != dz0);
                *qp = (uint8_t)(s | (wrapped ? 0x80 : 0));    // bit 7: pair crosses the periodic boundary
                qp += 32;
            }
        }
    }
    return (int)(qp - (queue + lane)) >> 5;
}

// ---- the sweep: cull + compact survivors of each neighbour leaf into the tile, test + drain when it fills ---------
template <int CAP, int PLANES, bool SYM, typename Drain>
__device__ __forceinline__ void sweep_loop(const SweepArgs& a, const float4* const (&planes)[PLANES], int64_t leaf,
                                           int lane, float xi, float yi, float zi, float hi2, float4* tile,
                                           uint8_t* queue, Drain drain) {
    static_assert(CAP <= 128 && CAP % 32 == 0, "queue entries keep bit 7 for the periodic-wrap mark");
    const float4 blo = a.leaf_lo[leaf], bhi = a.leaf_hi[leaf];
    const float hq2 = __fmul_rn(blo.w, blo.w);
    const uint32_t lt = (1u << lane) - 1u;
    int fill = 0, self_slot = -1;
    bool cwrap = false;
    const uint32_t e0 = a.off[leaf], e1 = a.off[leaf + 1];
    auto flush = [&]() {
        const int fill4 = (fill + 3) & ~3;
        if (lane < fill4 - fill) tile[fill + lane] = make_float4(3.0e30f, 3.0e30f, 3.0e30f, 0.0f);   // never accepted
        __syncwarp();
        const int cnt = test_slots<SYM>(a, fill4, cwrap, self_slot, lane, xi, yi, zi, hi2, tile, queue);
        drain(cnt);
        __syncwarp();
        fill = 0;
        self_slot = -1;
        cwrap = false;
    };
    uint32_t ent = (e0 < e1) ? a.list[e0] : 0u;
    float4 pj = (e0 < e1) ? planes[0][(int64_t)(ent & CRK_LEAF_MASK) * CRK_LEAF + lane] : make_float4(0, 0, 0, 0);
    for (uint32_t e = e0; e < e1; ++e) {
        const uint32_t cur = ent;
        const float4 pc = pj;
        if (e + 1 < e1) {   // prefetch the next leaf's positions
            ent = a.list[e + 1];
            pj = planes[0][(int64_t)(ent & CRK_LEAF_MASK) * CRK_LEAF + lane];
        }
        if (!SYM && !(cur & CRK_FLAG_GATHER)) continue;
        const int64_t b = (int64_t)(cur & CRK_LEAF_MASK);
        const int64_t g = b * CRK_LEAF + lane;
        const bool wrap = (cur & CRK_FLAG_WRAP) != 0;
        float gx, gy, gz;
        if (!wrap) {
            gx = gap1(blo.x, bhi.x, pc.x); gy = gap1(blo.y, bhi.y, pc.y); gz = gap1(blo.z, bhi.z, pc.z);
        } else {
            gx = gap1_wrap(blo.x, bhi.x, pc.x, a.L); gy = gap1_wrap(blo.y, bhi.y, pc.y, a.L); gz = gap1_wrap(blo.z, bhi.z, pc.z, a.L);
        }
        const float g2 = __fmaf_rn(gz, gz, __fmaf_rn(gy, gy, __fmul_rn(gx, gx)));
        const float lim = SYM ? fmaxf(hq2, __fmul_rn(pc.w, pc.w)) : hq2;
        const bool surv = g2 < lim;
        const uint32_t m = __ballot_sync(0xffffffffu, surv);
        const int cnt = __popc(m);
        if (cnt == 0) continue;
        if (fill + cnt > CAP) flush();
        const int slot = fill + __popc(m & lt);
        if (surv) {
            tile[slot] = pc;
#pragma unroll
            for (int p = 1; p < PLANES; ++p) tile[p * CAP + slot] = planes[p][g];
        }
        if (b == leaf) self_slot = surv ? slot : -1;
        cwrap = cwrap || wrap;
        fill += cnt;
    }
    if (fill > 0) flush();
}

// Wendland C4 (Eq. 12) without its sigma/h^3 prefactor, and D~ with W'/r = sigma h^-5 D~:
//   W~ = (1-eta)^6 (1 + 6 eta + 35/3 eta^2),   D~ = -(56/3) (1-eta)^5 (1 + 5 eta)
__device__ __forceinline__ void wendland(float eta, float& Wt, float& Dt) {
    const float t = fmaxf(1.0f - eta, 0.0f);
    const float t2 = t * t;
    const float t5 = t2 * t2 * t;
    Wt = t5 * t * fmaf(eta, fmaf(eta, C35_3, 6.0f), 1.0f);
    Dt = -C56_3 * t5 * fmaf(5.0f, eta, 1.0f);
}
__device__ __forceinline__ float wendland_w(float eta) {
    const float t = fmaxf(1.0f - eta, 0.0f);
    const float t2 = t * t;
    return t2 * t2 * t2 * fmaf(eta, fmaf(eta, C35_3, 6.0f), 1.0f);
}

// Separation of an accepted pair for the VALUES (the set membership was decided by the prescribed predicate above).
// Plain pairs: d = x_i - x_j.  Pairs that cross the periodic boundary (queue bit 7): shift the coordinate that lies in
// the upper half of the box by -L first (exact, Sterbenz) and subtract afterwards, so that the rounding error is
// relative to |d| and not to L  (fl(x_i - x_j) ~ 1 - 1e-3 would lose 1e-5 of a 4e-3 separation).
__device__ __forceinline__ float sep1_wrapped(float xi, float xj, float L, float half) {
    const float d = __fsub_rn(xi, xj);
    if (d > half) return __fsub_rn(__fsub_rn(xi, L), xj);
    if (d < -half) return __fsub_rn(xi, __fsub_rn(xj, L));
    return d;
}
__device__ __forceinline__ void sep3(const SweepArgs& a, bool wrapped, float xi, float yi, float zi, const float4& pj,
                                     float& dx, float& dy, float& dz, float& r2) {
    if (!wrapped) {
        dx = __fsub_rn(xi, pj.x);
        dy = __fsub_rn(yi, pj.y);
        dz = __fsub_rn(zi, pj.z);
    } else {
        dx = sep1_wrapped(xi, pj.x, a.L, a.half);
        dy = sep1_wrapped(yi, pj.y, a.L, a.half);
        dz = sep1_wrapped(zi, pj.z, a.L, a.half);
    }
    r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

template <int CAP, int PLANES>
struct Smem {
    static constexpr int TILE_F4 = PLANES * CAP;
    static constexpr int QUEUE_B = CAP * 32;
    static constexpr int PER_WARP = TILE_F4 * 16 + QUEUE_B;
};

// =================================================================================================== a1: volumes
// Eq. 14: V_i^-1 = n_i = sum_j W(|x_i - x_j|, h_i), self term included (S4); rho_i = m_i / V_i (S2).
constexpr int CH1 = 128;   // tile capacity (slots)
__global__ void __launch_bounds__(WPC * 32) k_volumes(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Smem<CH1, 1>;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t leaf = (int64_t)blockIdx.x * WPC + w;
    if (leaf >= a.nl) return;
    float4* tile = (float4*)(smem_raw + (size_t)w * S::PER_WARP);
    uint8_t* queue = (uint8_t*)(tile + S::TILE_F4);
    const int64_t i = leaf * CRK_LEAF + lane;
    const bool valid = i < a.n;
    const float4 pi = a.posh[i];
    const float xi = pi.x, yi = pi.y, zi = pi.z, hi = pi.w;
    const float hi2 = __fmul_rn(hi, hi);
    const float inv_h = valid ? 1.0f / hi : 0.0f;
    float acc = 0.0f;
    uint32_t count = 0;
    const float4* const planes[1] = {a.posh};
    sweep_loop<CH1, 1, false>(a, planes, leaf, lane, xi, yi, zi, hi2, tile, queue, [&](int cnt) {
        const int maxc = __reduce_max_sync(0xffffffffu, cnt);
        for (int s = 0; s < maxc; ++s) {
            if (s < cnt) {
                const int qe = queue[s * 32 + lane];
                const float4 pj = tile[qe & 0x7f];
                float dx, dy, dz, r2;
                sep3(a, (qe & 0x80) != 0, xi, yi, zi, pj, dx, dy, dz, r2);
                const float r = r2 * rsqrtf(fmaxf(r2, R2_TINY));
                acc += wendland_w(r * inv_h);
            }
        }
        count += cnt;
    });
    if (valid) {
        const float k3 = SIGMA_C4 * inv_h * inv_h * inv_h;
        const float ni = k3 * (acc + 1.0f);              // self term W~(0) = 1
        const float V = 1.0f / ni;
        const float mi = a.m_s[i];
        const float rho = mi * ni;
        a.posV[i] = make_float4(xi, yi, zi, V);
        a.rho_s[i] = rho;
        const int32_t p = a.perm[i];
        if (a.o0) a.o0[p] = V;
        if (a.o1) a.o1[p] = rho;
        if (a.ocnt) a.ocnt[p] = count;
    } else {
        a.posV[i] = make_float4(pi.x, pi.y, pi.z, 0.0f);
        a.rho_s[i] = 0.0f;
    }
}

// ========================================================================================== a2 + a3: RK coefficients
// A, B from  sum_j V_j WR_ij = 1,  sum_j V_j x_ij WR_ij = 0.  With moments over the gather set
//   m0 = sum w, m1 = sum w x, m2 = sum w x x  (w = V_j W_ij, self term in m0 only) and their gradients
//   d_c m0 = sum g x_c, d_c m1_a = sum g x_a x_c + delta_ac m0, d_c m2_ab = sum g x_a x_b x_c + delta_ac m1_b + delta_bc m1_a
//   (g = V_j W'_ij / r):   B = -m2^-1 m1,  A = 1/(m0 + B.m1),
//   d_c A = -A^2 (d_c m0 + 2 B.d_c m1 + B^T d_c m2 B),  d_c B = -m2^-1 (d_c m1 + d_c m2 B).
// 29 FP32 sums per particle in eta-normalised units, then an FP64 3x3 solve per particle.
constexpr int CH2 = 128;
__global__ void __launch_bounds__(WPC * 32) k_moments(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Smem<CH2, 1>;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t leaf = (int64_t)blockIdx.x * WPC + w;
    if (leaf >= a.nl) return;
    float4* tile = (float4*)(smem_raw + (size_t)w * S::PER_WARP);
    uint8_t* queue = (uint8_t*)(tile + S::TILE_F4);
    const int64_t i = leaf * CRK_LEAF + lane;
    const bool valid = i < a.n;
    const float4 ph = a.posh[i];
    const float xi = ph.x, yi = ph.y, zi = ph.z, hi = ph.w;
    const float hi2 = __fmul_rn(hi, hi);
    const float inv_h = valid ? 1.0f / hi : 0.0f;
    // accumulators: s0; s1[3]; s2[6] (xx,xy,xz,yy,yz,zz); t0[3]; t1[6]; t2[10] (xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz)
    float s0 = 0.f, s1x = 0.f, s1y = 0.f, s1z = 0.f;
    float sxx = 0.f, sxy = 0.f, sxz = 0.f, syy = 0.f, syz = 0.f, szz = 0.f;
    float t0x = 0.f, t0y = 0.f, t0z = 0.f;
    float txx = 0.f, txy = 0.f, txz = 0.f, tyy = 0.f, tyz = 0.f, tzz = 0.f;
    float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f, c4 = 0.f, c5 = 0.f, c6 = 0.f, c7 = 0.f, c8 = 0.f, c9 = 0.f;
    const float4* const planes[1] = {a.posV};
    sweep_loop<CH2, 1, false>(a, planes, leaf, lane, xi, yi, zi, hi2, tile, queue, [&](int cnt) {
        const int maxc = __reduce_max_sync(0xffffffffu, cnt);
        for (int s = 0; s < maxc; ++s) {
            if (s < cnt) {
                const int qe = queue[s * 32 + lane];
                const float4 pj = tile[qe & 0x7f];
                float dx, dy, dz, r2;
                sep3(a, (qe & 0x80) != 0, xi, yi, zi, pj, dx, dy, dz, r2);
                const float r = r2 * rsqrtf(fmaxf(r2, R2_TINY));
                float Wt, Dt;
                wendland(r * inv_h, Wt, Dt);
                const float wv = pj.w * Wt, gv = pj.w * Dt;
                const float x = dx * inv_h, y = dy * inv_h, z = dz * inv_h;
                const float xx = x * x, xy = x * y, xz = x * z, yy = y * y, yz = y * z, zz = z * z;
                s0 += wv;
                s1x = fmaf(wv, x, s1x); s1y = fmaf(wv, y, s1y); s1z = fmaf(wv, z, s1z);
                sxx = fmaf(wv, xx, sxx); sxy = fmaf(wv, xy, sxy); sxz = fmaf(wv, xz, sxz);
                syy = fmaf(wv, yy, syy); syz = fmaf(wv, yz, syz); szz = fmaf(wv, zz, szz);
                t0x = fmaf(gv, x, t0x); t0y = fmaf(gv, y, t0y); t0z = fmaf(gv, z, t0z);
                txx = fmaf(gv, xx, txx); txy = fmaf(gv, xy, txy); txz = fmaf(gv, xz, txz);
                tyy = fmaf(gv, yy, tyy); tyz = fmaf(gv, yz, tyz); tzz = fmaf(gv, zz, tzz);
                c0 = fmaf(gv, xx * x, c0); c1 = fmaf(gv, xx * y, c1); c2 = fmaf(gv, xx * z, c2);
                c3 = fmaf(gv, xy * y, c3); c4 = fmaf(gv, xy * z, c4); c5 = fmaf(gv, xz * z, c5);
                c6 = fmaf(gv, yy * y, c6); c7 = fmaf(gv, yy * z, c7); c8 = fmaf(gv, yz * z, c8);
                c9 = fmaf(gv, zz * z, c9);
            }
        }
    });
    float4 o0 = make_float4(0, 0, 0, 0), o1 = o0, o2 = o0, o3 = o0;
    if (valid) {
        // ---- a3: FP64 solve (dimensional quantities; k3 = sigma/h^3)
        const double h = (double)hi, ih = 1.0 / h;
        const double k3 = (double)SIGMA_C4 * ih * ih * ih;
        const double Vi = (double)a.posV[i].w;
        const double m0 = k3 * ((double)s0 + Vi);
        const double m1[3] = {k3 * h * s1x, k3 * h * s1y, k3 * h * s1z};
        const double k3h2 = k3 * h * h;
        const double m2[3][3] = {{k3h2 * sxx, k3h2 * sxy, k3h2 * sxz},
                                 {k3h2 * sxy, k3h2 * syy, k3h2 * syz},
                                 {k3h2 * sxz, k3h2 * syz, k3h2 * szz}};
        const double dm0[3] = {k3 * ih * t0x, k3 * ih * t0y, k3 * ih * t0z};
        // sum g x_a x_c (symmetric)
        const double q1[3][3] = {{k3 * txx, k3 * txy, k3 * txz}, {k3 * txy, k3 * tyy, k3 * tyz}, {k3 * txz, k3 * tyz, k3 * tzz}};
        const double k3h = k3 * h;
        const double cc[10] = {k3h * c0, k3h * c1, k3h * c2, k3h * c3, k3h * c4, k3h * c5, k3h * c6, k3h * c7, k3h * c8, k3h * c9};
        // inverse of m2 (adjugate)
        const double a00 = m2[1][1] * m2[2][2] - m2[1][2] * m2[1][2];
        const double a01 = m2[0][2] * m2[1][2] - m2[0][1] * m2[2][2];
        const double a02 = m2[0][1] * m2[1][2] - m2[0][2] * m2[1][1];
        const double a11 = m2[0][0] * m2[2][2] - m2[0][2] * m2[0][2];
        const double a12 = m2[0][1] * m2[0][2] - m2[0][0] * m2[1][2];
        const double a22 = m2[0][0] * m2[1][1] - m2[0][1] * m2[0][1];
        const double det = m2[0][0] * a00 + m2[0][1] * a01 + m2[0][2] * a02;
        double A, B[3], dA[3], dB[3][3];   // dB[c][a] = d_c B^a
        if (fabs(det) > 0.0 && isfinite(det)) {
            const double id = 1.0 / det;
            const double inv[3][3] = {{a00 * id, a01 * id, a02 * id}, {a01 * id, a11 * id, a12 * id}, {a02 * id, a12 * id, a22 * id}};
#pragma unroll
            for (int p = 0; p < 3; ++p) B[p] = -(inv[p][0] * m1[0] + inv[p][1] * m1[1] + inv[p][2] * m1[2]);
            A = 1.0 / (m0 + B[0] * m1[0] + B[1] * m1[1] + B[2] * m1[2]);
            // index of the symmetric cubic monomial x_a x_b x_c in cc[]
            const int cub[3][3][3] = {{{0, 1, 2}, {1, 3, 4}, {2, 4, 5}}, {{1, 3, 4}, {3, 6, 7}, {4, 7, 8}}, {{2, 4, 5}, {4, 7, 8}, {5, 8, 9}}};
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double Bdm1 = 0.0, BdmB = 0.0, rhs[3];
#pragma unroll
                for (int p = 0; p < 3; ++p) {
                    const double dm1_pc = q1[p][c] + (p == c ? m0 : 0.0);
                    Bdm1 += B[p] * dm1_pc;
                    double t = 0.0;
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        const double dm2_pqc = cc[cub[p][q][c]] + (p == c ? m1[q] : 0.0) + (q == c ? m1[p] : 0.0);
                        t += dm2_pqc * B[q];
                    }
                    BdmB += B[p] * t;
                    rhs[p] = dm1_pc + t;
                }
                dA[c] = -A * A * (dm0[c] + 2.0 * Bdm1 + BdmB);
#pragma unroll
                for (int p = 0; p < 3; ++p) dB[c][p] = -(inv[p][0] * rhs[0] + inv[p][1] * rhs[1] + inv[p][2] * rhs[2]);
            }
        } else {   // S14: degenerate neighbourhood -> zeroth-order correction only
            A = 1.0 / m0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                B[c] = 0.0;
                dA[c] = -A * A * dm0[c];
                dB[c][0] = dB[c][1] = dB[c][2] = 0.0;
            }
        }
        // pre-combined form used by the later sweeps:  (grad WR_ij)_c = W (cvec_c + M_ca x_a) + A s D x_c, s = 1 + B.x
        //   cvec_c = d_c A + A B_c,   M_ca = d_c A B_a + A d_c B_a
        o0 = make_float4((float)A, (float)B[0], (float)B[1], (float)B[2]);
        float Mf[9];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int p = 0; p < 3; ++p) Mf[3 * c + p] = (float)(dA[c] * B[p] + A * dB[c][p]);
        o1 = make_float4((float)(dA[0] + A * B[0]), (float)(dA[1] + A * B[1]), (float)(dA[2] + A * B[2]), Mf[0]);
        o2 = make_float4(Mf[1], Mf[2], Mf[3], Mf[4]);
        o3 = make_float4(Mf[5], Mf[6], Mf[7], Mf[8]);
        const int32_t p = a.perm[i];
        const int64_t n = a.n;
        if (a.o0) a.o0[p] = (float)A;
        if (a.o1) { a.o1[p] = (float)B[0]; a.o1[n + p] = (float)B[1]; a.o1[2 * n + p] = (float)B[2]; }
        if (a.o2) { a.o2[p] = (float)dA[0]; a.o2[n + p] = (float)dA[1]; a.o2[2 * n + p] = (float)dA[2]; }
        if (a.o3) {
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int q = 0; q < 3; ++q) a.o3[(3 * c + q) * n + p] = (float)dB[c][q];
        }
    }
    a.coef[i] = o0;
    a.coef[a.np + i] = o1;
    a.coef[2 * a.np + i] = o2;
    a.coef[3 * a.np + i] = o3;
}

// ---- hydro preparation: sorted (vx,vy,vz,V) and (P, rho, c_s, 1/h) ------------------------------------------------
__global__ void __launch_bounds__(256) k_pack_vel(const float* __restrict__ vx, const float* __restrict__ vy,
                                                  const float* __restrict__ vz, const float* __restrict__ u, int64_t n,
                                                  float4* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_float4(vx[i], vy[i], vz[i], u[i]);
}
// Eq. 4: P = (gamma-1) rho u (unclamped);  c_s = sqrt(gamma P / rho) = sqrt(gamma (gamma-1) max(u,0))  (S12)
__global__ void __launch_bounds__(256) k_hydro_prep(SweepArgs a, const float4* __restrict__ vel_orig) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.np) return;
    if (k < a.n) {
        const float4 v = vel_orig[a.perm[k]];
        const float V = a.posV[k].w;
        const float rho = a.rho_s[k];
        const float g = a.gamma;
        a.velV[k] = make_float4(v.x, v.y, v.z, V);
        a.thermo[k] = make_float4((g - 1.0f) * rho * v.w, rho, sqrtf(g * (g - 1.0f) * fmaxf(v.w, 0.0f)), 1.0f / a.posh[k].w);
    } else {
        a.velV[k] = make_float4(0, 0, 0, 0);
        a.thermo[k] = make_float4(0, 0, 0, 0);
    }
}

// per-particle RK coefficients in registers
struct Coef {
    float A, Bx, By, Bz, cx, cy, cz, M[9];
};
__device__ __forceinline__ Coef load_coef(const float4& q0, const float4& q1, const float4& q2, const float4& q3) {
    Coef k;
    k.A = q0.x; k.Bx = q0.y; k.By = q0.z; k.Bz = q0.w;
    k.cx = q1.x; k.cy = q1.y; k.cz = q1.z;
    k.M[0] = q1.w; k.M[1] = q2.x; k.M[2] = q2.y; k.M[3] = q2.z; k.M[4] = q2.w;
    k.M[5] = q3.x; k.M[6] = q3.y; k.M[7] = q3.z; k.M[8] = q3.w;
    return k;
}
// Eq. 16 in the pre-combined form.  Written with explicit round-to-nearest intrinsics so that the two
// lanes that evaluate the same (particle, separation) pair from opposite sides obtain bit-identical vectors, which makes
// G_ij = grad WR_ji - grad WR_ij exactly antisymmetric in floating point.
__device__ __forceinline__ void rk_grad(const Coef& k, float x, float y, float z, float W, float D, float& gx, float& gy,
                                        float& gz) {
    const float s = __fmaf_rn(k.Bz, z, __fmaf_rn(k.By, y, __fmaf_rn(k.Bx, x, 1.0f)));
    const float q = __fmul_rn(__fmul_rn(k.A, s), D);
    const float tx = __fmaf_rn(k.M[2], z, __fmaf_rn(k.M[1], y, __fmaf_rn(k.M[0], x, k.cx)));
    const float ty = __fmaf_rn(k.M[5], z, __fmaf_rn(k.M[4], y, __fmaf_rn(k.M[3], x, k.cy)));
    const float tz = __fmaf_rn(k.M[8], z, __fmaf_rn(k.M[7], y, __fmaf_rn(k.M[6], x, k.cz)));
    gx = __fmaf_rn(q, x, __fmul_rn(W, tx));
    gy = __fmaf_rn(q, y, __fmul_rn(W, ty));
    gz = __fmaf_rn(q, z, __fmul_rn(W, tz));
}
// Eq. 24: Q = rho (-C_l c_s mu + C_q mu^2); explicit intrinsics so both sides of a pair compute identical bits
__device__ __forceinline__ float visc_Q(float rho, float cs, float mu, float Cl, float Cq) {
    return __fmul_rn(__fmul_rn(rho, mu), __fmaf_rn(Cq, mu, -__fmul_rn(Cl, cs)));
}
// dimensional W and D = W'/r for support h (k3 = sigma/h^3, ih = 1/h)
__device__ __forceinline__ void wendland_dim(float r, float ih, float k3, float& W, float& D) {
    float Wt, Dt;
    wendland(__fmul_rn(r, ih), Wt, Dt);
    W = __fmul_rn(k3, Wt);
    D = __fmul_rn(__fmul_rn(__fmul_rn(k3, ih), ih), Dt);
}

// =============================================================================================== a4: velocity gradient
// Eq. 26: grad v_i = - sum_j V_j (v_i - v_j) (x) grad WR_ij   over the gather set; index [3a+b] = d_b v^a
constexpr int CH4 = 128;
__global__ void __launch_bounds__(WPC * 32) k_gradv(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Smem<CH4, 2>;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t leaf = (int64_t)blockIdx.x * WPC + w;
    if (leaf >= a.nl) return;
    float4* tile = (float4*)(smem_raw + (size_t)w * S::PER_WARP);
    uint8_t* queue = (uint8_t*)(tile + S::TILE_F4);
    const int64_t i = leaf * CRK_LEAF + lane;
    const bool valid = i < a.n;
    const float4 ph = a.posh[i];
    const float xi = ph.x, yi = ph.y, zi = ph.z, hi = ph.w;
    const float hi2 = __fmul_rn(hi, hi);
    const float ih = valid ? 1.0f / hi : 0.0f;
    const float k3 = SIGMA_C4 * ih * ih * ih;
    const float4 vi = a.velV[i];
    const Coef ci = load_coef(a.coef[i], a.coef[a.np + i], a.coef[2 * a.np + i], a.coef[3 * a.np + i]);
    float g[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    const float4* const planes[2] = {a.posh, a.velV};
    sweep_loop<CH4, 2, false>(a, planes, leaf, lane, xi, yi, zi, hi2, tile, queue, [&](int cnt) {
        const int maxc = __reduce_max_sync(0xffffffffu, cnt);
        for (int s = 0; s < maxc; ++s) {
            if (s < cnt) {
                const int qe = queue[s * 32 + lane];
                const int jj = qe & 0x7f;
                const float4 pj = tile[jj];
                const float4 vj = tile[CH4 + jj];
                float dx, dy, dz, r2;
                sep3(a, (qe & 0x80) != 0, xi, yi, zi, pj, dx, dy, dz, r2);
                const float r = r2 * rsqrtf(fmaxf(r2, R2_TINY));
                float W, D, gx, gy, gz;
                wendland_dim(r, ih, k3, W, D);
                rk_grad(ci, dx, dy, dz, W, D, gx, gy, gz);
                const float Vj = vj.w;
                const float ux = Vj * (vi.x - vj.x), uy = Vj * (vi.y - vj.y), uz = Vj * (vi.z - vj.z);
                g[0] = fmaf(-ux, gx, g[0]); g[1] = fmaf(-ux, gy, g[1]); g[2] = fmaf(-ux, gz, g[2]);
                g[3] = fmaf(-uy, gx, g[3]); g[4] = fmaf(-uy, gy, g[4]); g[5] = fmaf(-uy, gz, g[5]);
                g[6] = fmaf(-uz, gx, g[6]); g[7] = fmaf(-uz, gy, g[7]); g[8] = fmaf(-uz, gz, g[8]);
            }
        }
    });
    const float hhat = hi / a.n_h;
    a.gv[i] = make_float4(g[0], g[1], g[2], g[3]);
    a.gv[a.np + i] = make_float4(g[4], g[5], g[6], g[7]);
    a.gv[2 * a.np + i] = make_float4(g[8], k3, hhat, hhat * hhat * a.eps2);
}

// ============================================================================================ a5: momentum and energy
// Eq. 17:  m_i dv_i/dt = sum_j (1/2) V_i V_j (P_i+Q_i+P_j+Q_j) (grad WR_ji - grad WR_ij)
// Eq. 18:  m_i du_i/dt = sum_j (1/2) V_i V_j (P_j+Q_j) (v_j - v_i).(grad WR_ji - grad WR_ij)       (S6)
// Q from Eqs. 24-25 with the limited midpoint projection of Eqs. 27-32 (S7: division-free van Leer form).
// Sums over all j != i with r2 < max(h_i^2, h_j^2); each ordered pair is evaluated by the lane that owns i.
constexpr int CH5 = 64;
constexpr int PL5 = 10;
__global__ void __launch_bounds__(WPC * 32) k_forces(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using S = Smem<CH5, PL5>;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t leaf = (int64_t)blockIdx.x * WPC + w;
    if (leaf >= a.nl) return;
    float4* tile = (float4*)(smem_raw + (size_t)w * S::PER_WARP);
    uint8_t* queue = (uint8_t*)(tile + S::TILE_F4);
    const int64_t i = leaf * CRK_LEAF + lane;
    const bool valid = i < a.n;
    const float4 ph = a.posh[i];
    const float xi = ph.x, yi = ph.y, zi = ph.z, hi = ph.w;
    const float hi2 = __fmul_rn(hi, hi);
    const float4 vi = a.velV[i];        // vx,vy,vz,V
    const float4 ti = a.thermo[i];      // P,rho,cs,1/h
    const Coef ci = load_coef(a.coef[i], a.coef[a.np + i], a.coef[2 * a.np + i], a.coef[3 * a.np + i]);
    const float4 g0 = a.gv[i], g1 = a.gv[a.np + i], g2 = a.gv[2 * a.np + i];
    const float gi[9] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w, g2.x};
    const float k3i = g2.y, hhi = g2.z, he2i = g2.w;
    const float eta_crit = 1.0f / a.n_h, inv_fold = a.n_h / 0.2f;
    float Fx = 0.f, Fy = 0.f, Fz = 0.f, dE = 0.f;
    uint32_t count = 0;
    const float4* const planes[PL5] = {a.posh, a.velV, a.thermo, a.coef, a.coef + a.np, a.coef + 2 * a.np,
                                       a.coef + 3 * a.np, a.gv, a.gv + a.np, a.gv + 2 * a.np};
    constexpr int PS = CH5;        // plane stride in the tile
    sweep_loop<CH5, PL5, true>(a, planes, leaf, lane, xi, yi, zi, hi2, tile, queue, [&](int cnt) {
        const int maxc = __reduce_max_sync(0xffffffffu, cnt);
        for (int s = 0; s < maxc; ++s) {
            if (s < cnt) {
                const int qe = queue[s * 32 + lane];
                const int jj = qe & 0x7f;
                const float4 pj = tile[jj];
                const float4 vj = tile[PS + jj];
                const float4 tj = tile[2 * PS + jj];
                const Coef cj = load_coef(tile[3 * PS + jj], tile[4 * PS + jj], tile[5 * PS + jj], tile[6 * PS + jj]);
                const float4 h0 = tile[7 * PS + jj], h1 = tile[8 * PS + jj], h2 = tile[9 * PS + jj];
                float dx, dy, dz, r2;
                sep3(a, (qe & 0x80) != 0, xi, yi, zi, pj, dx, dy, dz, r2);
                const float r = __fmul_rn(r2, rsqrtf(fmaxf(r2, R2_TINY)));
                float Wi, Di, Wj, Dj;
                wendland_dim(r, ti.w, k3i, Wi, Di);
                wendland_dim(r, tj.w, h2.y, Wj, Dj);
                float aix, aiy, aiz, ajx, ajy, ajz;
                rk_grad(ci, dx, dy, dz, Wi, Di, aix, aiy, aiz);            // grad WR_ij
                rk_grad(cj, -dx, -dy, -dz, Wj, Dj, ajx, ajy, ajz);         // grad WR_ji  (x_ji = -x_ij)
                const float Gx = __fsub_rn(ajx, aix), Gy = __fsub_rn(ajy, aiy), Gz = __fsub_rn(ajz, aiz);
                // (grad v . x_ij) for both particles, written so that the mirrored lane forms the same numbers
                const float wix = __fmaf_rn(gi[2], dz, __fmaf_rn(gi[1], dy, __fmul_rn(gi[0], dx)));
                const float wiy = __fmaf_rn(gi[5], dz, __fmaf_rn(gi[4], dy, __fmul_rn(gi[3], dx)));
                const float wiz = __fmaf_rn(gi[8], dz, __fmaf_rn(gi[7], dy, __fmul_rn(gi[6], dx)));
                const float wjx = __fmaf_rn(h0.z, dz, __fmaf_rn(h0.y, dy, __fmul_rn(h0.x, dx)));
                const float wjy = __fmaf_rn(h1.y, dz, __fmaf_rn(h1.x, dy, __fmul_rn(h0.w, dx)));
                const float wjz = __fmaf_rn(h2.x, dz, __fmaf_rn(h1.w, dy, __fmul_rn(h1.z, dx)));
                const float Nn = __fmaf_rn(dz, wiz, __fmaf_rn(dy, wiy, __fmul_rn(dx, wix)));   // Eq. 30 numerator
                const float Dn = __fmaf_rn(dz, wjz, __fmaf_rn(dy, wjy, __fmul_rn(dx, wjx)));   // Eq. 30 denominator
                // Eq. 29 with r_ij = N/Dn:  phi_VL = 4 N Dn / (N + Dn)^2 if N Dn > 0 else 0  (S7)
                const float nd = __fmul_rn(Nn, Dn);
                const float sm = __fadd_rn(Nn, Dn);
                float phi = 0.0f;
                if (nd > 0.0f) phi = __fdividef(4.0f * nd, __fmul_rn(sm, sm));
                phi = fminf(phi, 1.0f);
                // Eqs. 31-32
                const float eta = __fmul_rn(r, fminf(ti.w, tj.w));
                if (eta < eta_crit) {
                    const float q = (eta - eta_crit) * inv_fold;
                    phi *= __expf(-q * q);
                }
                // Eq. 27 (adot = 0): uhat_ij = v_ij - (1/2) phi (grad v_i + grad v_j).x_ij ; then uhat_ij . x_ij
                const float hp = 0.5f * phi;
                const float ux = __fsub_rn(__fsub_rn(vi.x, vj.x), __fmul_rn(hp, __fadd_rn(wix, wjx)));
                const float uy = __fsub_rn(__fsub_rn(vi.y, vj.y), __fmul_rn(hp, __fadd_rn(wiy, wjy)));
                const float uz = __fsub_rn(__fsub_rn(vi.z, vj.z), __fmul_rn(hp, __fadd_rn(wiz, wjz)));
                const float udx = __fmaf_rn(uz, dz, __fmaf_rn(uy, dy, __fmul_rn(ux, dx)));
                // Eq. 25: mu_k = min(0, hhat_k (uhat.x) / (r^2 + hhat_k^2 eps^2));  Eq. 24: Q_k = rho_k (-C_l c_k mu_k + C_q mu_k^2)
                const float mui = fminf(0.0f, __fdividef(__fmul_rn(hhi, udx), __fadd_rn(r2, he2i)));
                const float muj = fminf(0.0f, __fdividef(__fmul_rn(h2.z, udx), __fadd_rn(r2, h2.w)));
                const float Qi = visc_Q(ti.y, ti.z, mui, a.C_l, a.C_q);
                const float Qj = visc_Q(tj.y, tj.z, muj, a.C_l, a.C_q);
                const float PQi = __fadd_rn(ti.x, Qi), PQj = __fadd_rn(tj.x, Qj);
                const float hvv = 0.5f * __fmul_rn(vi.w, vj.w);
                const float pf = __fmul_rn(hvv, __fadd_rn(PQi, PQj));
                Fx = fmaf(pf, Gx, Fx); Fy = fmaf(pf, Gy, Fy); Fz = fmaf(pf, Gz, Fz);
                const float vG = (vj.x - vi.x) * Gx + (vj.y - vi.y) * Gy + (vj.z - vi.z) * Gz;
                dE = fmaf(hvv * PQj, vG, dE);
            }
        }
        count += cnt;
    });
    if (valid) {
        const float im = 1.0f / a.m_s[i];
        const int32_t p = a.perm[i];
        a.o0[p] = Fx * im;
        a.o1[p] = Fy * im;
        a.o2[p] = Fz * im;
        a.o3[p] = dE * im;
        if (a.ocnt) a.ocnt[p] = count;
    }
}

__global__ void __launch_bounds__(256) k_gather_f32(const float* __restrict__ in, const int32_t* __restrict__ perm,
                                                    int64_t n, int64_t np, float* __restrict__ out) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < np) out[k] = (k < n) ? in[perm[k]] : 1.0f;
}

SweepArgs make_args(crk_ctx* c) {
    SweepArgs a;
    memset(&a, 0, sizeof(a));
    a.n = c->n; a.nl = c->nl; a.np = c->nl * CRK_LEAF;
    a.L = c->prm.box; a.half = 0.5f * c->prm.box;
    a.off = (const uint32_t*)c->nbr_off.p; a.list = (const uint32_t*)c->nbr_list.p;
    a.perm = c->perm;
    a.leaf_lo = (const float4*)c->leaf_lo.p; a.leaf_hi = (const float4*)c->leaf_hi.p;
    a.posh = (const float4*)c->posh.p; a.posV = (float4*)c->posV.p; a.velV = (float4*)c->velV.p;
    a.thermo = (float4*)c->thermo.p; a.coef = (float4*)c->coef.p; a.gv = (float4*)c->gv.p;
    a.rho_s = (float*)c->rho_s.p; a.m_s = (const float*)c->m_s.p;
    a.gamma = c->prm.gamma; a.n_h = c->prm.n_h; a.C_l = c->prm.C_l; a.C_q = c->prm.C_q;
    a.eps2 = c->prm.eps * c->prm.eps;
    return a;
}

template <typename K>
int set_smem(crk_ctx* c, K kernel, int bytes) {
    if (bytes > 48 * 1024) CRK_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    return CRK_OK;
}

}  // namespace

int crk_launch_volumes(crk_ctx* c, const float* m, float* V, float* rho, uint32_t* nbr_count) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->posV, (size_t)np * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->rho_s, (size_t)np * sizeof(float)));
    CRK_TRY(crk_ensure(c, c->m_s, (size_t)np * sizeof(float)));
    k_gather_f32<<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>(m, c->perm, c->n, np, (float*)c->m_s.p);
    CRK_TRY(crk_check_launch(c, "k_gather_f32"));
    SweepArgs a = make_args(c);
    a.o0 = V; a.o1 = rho; a.ocnt = nbr_count;
    const int smem = WPC * Smem<CH1, 1>::PER_WARP;
    CRK_TRY(set_smem(c, k_volumes, smem));
    k_volumes<<<(unsigned)((c->nl + WPC - 1) / WPC), WPC * 32, smem, c->stream>>>(a);
    return crk_check_launch(c, "k_volumes");
}

int crk_launch_moments(crk_ctx* c, float* A, float* B, float* gradA, float* gradB) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->coef, (size_t)np * 4 * sizeof(float4)));
    SweepArgs a = make_args(c);
    a.o0 = A; a.o1 = B; a.o2 = gradA; a.o3 = gradB;
    const int smem = WPC * Smem<CH2, 1>::PER_WARP;
    CRK_TRY(set_smem(c, k_moments, smem));
    k_moments<<<(unsigned)((c->nl + WPC - 1) / WPC), WPC * 32, smem, c->stream>>>(a);
    return crk_check_launch(c, "k_moments");
}

int crk_launch_hydro(crk_ctx* c, const float* vx, const float* vy, const float* vz, const float* u, float* ax,
                     float* ay, float* az, float* dudt, uint32_t* pair_count) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->vel_orig, (size_t)c->n * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->velV, (size_t)np * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->thermo, (size_t)np * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->gv, (size_t)np * 3 * sizeof(float4)));
    k_pack_vel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(vx, vy, vz, u, c->n, (float4*)c->vel_orig.p);
    CRK_TRY(crk_check_launch(c, "k_pack_vel"));
    SweepArgs a = make_args(c);
    k_hydro_prep<<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>(a, (const float4*)c->vel_orig.p);
    CRK_TRY(crk_check_launch(c, "k_hydro_prep"));
    crk_rec(c, EV_GV0);
    {
        const int smem = WPC * Smem<CH4, 2>::PER_WARP;
        CRK_TRY(set_smem(c, k_gradv, smem));
        k_gradv<<<(unsigned)((c->nl + WPC - 1) / WPC), WPC * 32, smem, c->stream>>>(a);
        CRK_TRY(crk_check_launch(c, "k_gradv"));
    }
    crk_rec(c, EV_GV1);
    a.o0 = ax; a.o1 = ay; a.o2 = az; a.o3 = dudt; a.ocnt = pair_count;
    {
        const int smem = WPC * Smem<CH5, PL5>::PER_WARP;
        CRK_TRY(set_smem(c, k_forces, smem));
        k_forces<<<(unsigned)((c->nl + WPC - 1) / WPC), WPC * 32, smem, c->stream>>>(a);
        CRK_TRY(crk_check_launch(c, "k_forces"));
    }
    crk_rec(c, EV_F1);
    return CRK_OK;
}
