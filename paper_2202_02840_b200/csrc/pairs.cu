// pairs.cu -- steps a1..a5: the four pair sweeps of one CRKSPH derivative evaluation (FP32 pair math on the FMA pipes),
// and the next rows that ride on them: compatible energy sweep, time-step criteria, evolved smoothing length.
//
// All sweeps walk the neighbour lists built once per crk_build_cells (lists.cu).  A leaf (32 particles) is served by a group
// of WPL warps; lane l of each of them holds particle i = 32*leaf + l in registers.  The kernels are persistent: a group takes
// leaves from a work counter until none is left.  Per segment of the leaf's chain:
//   meta    header, entry counts and candidate indices were copied to shared memory while the previous segment's rows ran
//   stage   the WPL warps copy the j-state of the segment's C candidates into a shared-memory tile, slot = candidate
//   drain   warp wl takes rows wl, wl+WPL, ... of the ELL block; row k holds the k-th entry of every lane, so each lane
//           evaluates one accepted pair per row with j-state fetched from the tile (entries are prefetched 4 rows ahead)
// and at the end the WPL partial sums of a lane are added in fixed warp order (deterministic) before the epilogue.
// No candidate is tested here: set membership was decided by the builder with the prescribed predicate (S3).
// Equation numbers refer to /root/reference/PAPER.md; the closed forms of A, B, grad A, grad B are derived in DESIGN.md.
#include "crk_internal.cuh"


namespace {

constexpr float SIGMA_C4 = 4.923856051905513f;     // 495 / (32 pi), Eq. 12
constexpr float C35_3 = 35.0f / 3.0f;
constexpr float C56_3 = 56.0f / 3.0f;
constexpr float R2_TINY = 1.0e-37f;
constexpr int FROW = 8;                            // float4 per force-sweep state row: one 128-byte line per particle
constexpr int CPL = FROW + 1;                      // + the kick plane (v' - v, s = P / rho^gamma) of the compatible-energy sweep
// shared-memory tile: plane-major, plane p of candidate slot c at p * PSTRIDE + c * 16 bytes.  The 16 bytes of padding per
// plane put the FROW pieces of one candidate row (written by eight neighbouring lanes of one LDGSTS) into different banks.
constexpr uint32_t PSTRIDE = CRK_CCAP * 16u + 16u;

struct SweepArgs {
    int64_t n, nl;
    float L, half;
    const uint4* __restrict__ arena;      // neighbour-list segments
    const uint4* __restrict__ seg_first;  // dense copy of each leaf's first segment header (.w = its arena unit, 0 = none)
    const uint16_t* __restrict__ leaf_cnt;  // [nl][32] per-lane entry counts of the first segment
    const uint32_t* __restrict__ cand_first; // [nl][CRK_CAND_STRIDE] candidate indices of the first segment
    const int32_t* __restrict__ perm;     // sorted slot -> caller index
    const float4* __restrict__ posh;      // (x,y,z,h)
    float4* __restrict__ posV;            // (x,y,z,V)
    float4* __restrict__ coef;            // 4 planes, stride np: (A,B) (c,M0) (M1..M4) (M5..M8)
    float4* __restrict__ fst;             // force-sweep state, one row of FROW float4 per particle (layout at k_rk)
    float4* __restrict__ facc;            // (dv/dt, s = P / rho^gamma) per particle, written by k_forces
    float4* __restrict__ xv;              // (x,y,z,1/h) (vx,vy,vz,V) per particle, 32 bytes: what the grad v sweep stages
    float* __restrict__ rho_s;
    float* __restrict__ m_s;              // masses in sorted order (written by k_volumes)
    const float* __restrict__ m_in;       // masses in caller order (crk_volumes)
    int64_t np;                           // padded particle count nl*32 (plane stride)
    float gamma, n_h, C_l, C_q, eps2;
    // outputs in caller order (may be null)
    float* __restrict__ o0; float* __restrict__ o1; float* __restrict__ o2; float* __restrict__ o3;
    uint32_t* __restrict__ ocnt;
    float2* __restrict__ ts;              // (max approach speed, max Q_i) per particle, sorted (time-step criteria), or null
    const int32_t* __restrict__ ids;      // compacted list of leaves to sweep (crk_hydro_derivs_active), or null = all nl leaves
    int64_t n_ids;
    const uint8_t* __restrict__ active;   // per particle, caller order: outputs are written where active[p] != 0 (null = everywhere)
    int* flag;                            // status words (CRK_CHECKED builds write FW_CHECK)
    unsigned int* sched;                  // work counter of the persistent groups (zeroed before every launch)
};

struct Seg {
    const uint16_t* ell;
    int C, K, ct;
    uint32_t next;
};

// Metadata of the segment a group stages next, in shared memory: the same 105 16-byte chunks a segment carries in the arena
// (header | cnt[32] u16 | cand[CRK_CCAP] u32; a leaf's first segment keeps them in the dense per-leaf arrays).
// It is fetched with cp.async while the group is still evaluating the rows of the previous segment, so the three dependent
// loads (header -> candidate indices -> state) that used to open every leaf shrink to the last one.
struct __align__(16) Meta {
    uint4 hdr;                    // {next segment unit, C | CRK_SEG_WRAP | K << 16, 0, own unit (first segments only)}
    uint16_t cnt[32];
    uint32_t cand[CRK_CCAP];
    long long next_leaf;          // sweep_begin: the group's first leaf (-1 = none)
    long long next2;              // the leaf after the one being swept (-1 = none), written by thread 0 of the group one leaf ahead
};
constexpr int META_CHUNKS = 1 + 4 + CRK_CCAP / 4;
static_assert(sizeof(Meta) == META_CHUNKS * 16 + 16, "Meta layout");

__device__ __forceinline__ void cp_async16(uint32_t dst_shared, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_shared), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }

// 128-bit shared-memory load from a 32-bit shared address (no generic-address window arithmetic in the inner loops)
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// MUFU approximations with flush-to-zero: one instruction each (the default rsqrtf / __fdividef / __expf wrap the MUFU in
// denormal rescaling, 3-4 extra instructions per call); relative error 2^-22, far below the 1e-4 parity bar
__device__ __forceinline__ float rsqrt_fast(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_fast(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_fast(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int WPL>
__device__ __forceinline__ void group_sync(int lg) {
    if (WPL == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(lg + 1), "r"(WPL * 32) : "memory");
}

// ---- persistent groups: work distribution and metadata prefetch --------------------------------------------------------
// A group (WPL warps) serves one leaf at a time and keeps taking leaves from a global counter until none is left; the
// kernels are launched with as many CTAs as are resident at once.  (One CTA per leaf cost the force sweep 19 % of its time
// in CTA turnover and 27 % in the dependent loads of the prologue -- measured with clock64 probes in round 2.)
// the counter's answer is only looked at (resolve_slot) when the leaf is needed, one leaf later: no thread waits for the atomic
__device__ __forceinline__ unsigned int grab_slot(const SweepArgs& a) { return atomicAdd(a.sched, 1u); }
__device__ __forceinline__ long long resolve_slot(const SweepArgs& a, unsigned int slot) {
    const long long total = a.ids ? a.n_ids : a.nl;
    if ((long long)slot >= total) return -1;
    return a.ids ? (long long)a.ids[slot] : (long long)slot;
}
__device__ __forceinline__ long long grab_leaf(const SweepArgs& a) { return resolve_slot(a, grab_slot(a)); }
// copies the metadata of a leaf's first segment (unit == 0) or of the arena segment `unit` into m; the caller commits
template <int NT>
__device__ __forceinline__ void issue_meta(Meta* m, const SweepArgs& a, long long leaf, uint32_t unit, int tg) {
    const uint32_t ms = (uint32_t)__cvta_generic_to_shared(m);
    for (int ch = tg; ch < META_CHUNKS; ch += NT) {
        const char* src;
        if (unit != 0u) src = (const char*)(a.arena + unit + ch);
        else if (ch == 0) src = (const char*)(a.seg_first + leaf);
        else if (ch < 5) src = (const char*)(a.leaf_cnt + leaf * 32) + (ch - 1) * 16;
        else src = (const char*)(a.cand_first + leaf * CRK_CAND_STRIDE) + (ch - 5) * 16;
        cp_async16(ms + (uint32_t)ch * 16u, src);
    }
}
// first work item of a group: returns the leaf (or -1) with the copy of its metadata in flight (committed)
template <int WPL>
__device__ __forceinline__ long long sweep_begin(const SweepArgs& a, Meta* m, int lg, int wl, int lane) {
    const int tg = wl * 32 + lane;
    if (tg == 0) {
        const long long l0 = grab_leaf(a);
        m->next_leaf = l0;
        m->next2 = (l0 >= 0) ? grab_leaf(a) : -1;
    }
    group_sync<WPL>(lg);
    const long long leaf = m->next_leaf;
    if (leaf >= 0) issue_meta<WPL * 32>(m, a, leaf, 0u, tg);
    cp_async_commit();
    return leaf;
}

// ---- the sweep over one leaf's segment chain -------------------------------------------------------------------------
// Rows [0, K) of a segment's entry block; lane l is active while k < cnt[l].  SYM = false (gather set, Eqs. 13-14): entries
// flagged CRK_ELL_SYM are skipped;  SYM = true (Eqs. 17-18): every entry is a pair.  Returns the lane's entry count (the
// number of its pairs of the symmetric set; a gather sweep that needs its own count takes it in `pair`).
// pair(slot_addr, crosses_boundary, plane0) evaluates one accepted pair (slot_addr = shared address of the candidate's
// plane-0 entry; plane p sits p * PSTRIDE bytes further); returns the number of pairs the lane owns.
// The tile's planes 0 .. ROWP-1 are the first ROWP float4 of the candidates' force-state rows (`rows_src`, FROW float4 per
// particle: consecutive lanes copy consecutive pieces of one row, so a warp-wide LDGSTS touches 32 / ROWP full lines or
// sectors instead of 32 scattered ones), planes ROWP .. ROWP+PLANES-1 come from the SoA arrays `planes`.
// On entry the copy of the leaf's metadata into m is in flight; on exit the group's next leaf is in `next_leaf` and the copy
// of ITS metadata is in flight.  Work items are taken two leaves ahead (thread 0 keeps the counter's answer in a register
// until the end of the leaf), so no barrier waits for the atomic.  Barriers per segment: B1 metadata landed and the previous
// rows are done (tile free); B2 everybody has read the metadata (m may be overwritten); B3 the state has landed.
// (Measured and not kept: prefetch.global.L2 of the next segment's candidate state a few rows into the current one -- the
// prefetches cost the load/store unit as much as the copies they were meant to speed up: forces 11.05 -> 11.9 ms.)
struct NoInit {
    __device__ __forceinline__ void operator()(uint32_t) const {}
};
struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};
// init(tile_s) runs once, after the first segment is staged: slots 0..31 of that tile are the leaf's own particles in lane
// order (lists.cu), so a sweep can take its i-state from there instead of loading it from global memory.
// (Measured in round 2 and not kept: a second, branch-free instantiation of the row loop for segments without
// boundary-crossing entries -- 172 instead of 190 instructions per pair of k_forces, but ptxas then sinks the shared loads
// next to their uses and the sweep loses 1.6 ms to short-scoreboard stalls.)
// staged() runs once per leaf between the issue of the first segment's copies and B2, i.e. while the copies are in flight and
// the group has nothing else to do: the place for work that does not need the tile (the previous leaf's epilogue).
template <int WPL, int ROWP, int PLANES, bool SYM, int NPRE = 1, typename Pair, typename Init = NoInit, typename Hook = NoHook>
__device__ __forceinline__ uint32_t leaf_sweep(const SweepArgs& a, const float4* __restrict__ rows_src, const float4* const* planes,
                                               long long leaf, long long& next_leaf, int lg, int wl, int lane, float4* tile, Meta* m,
                                               Pair pair, Init init = Init(), Hook staged = Hook()) {
    static_assert(ROWP == 0 || ROWP == 2 || ROWP == 8, "row pieces per candidate");
    constexpr int RSTRIDE = ROWP;   // float4 per source row: the compact (x,y,z,1/h)(v,V) array (2) or the full state rows (8 = FROW)
    constexpr int NT = WPL * 32;                                  // threads that serve the leaf
    uint32_t count = 0;
    bool first = true;
    const int tg = wl * 32 + lane;
    const uint32_t tile_s = (uint32_t)__cvta_generic_to_shared(tile);
    uint32_t unit = 0;                                            // arena unit of the segment being staged (0: not known yet)
    unsigned int pend = 0xffffffffu;                              // thread 0: the work item taken for the leaf after next (raw counter value)
    next_leaf = -1;
    for (;;) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        group_sync<WPL>(lg);                                   // B1
        const uint4 h0 = m->hdr;
        if (first) {
            unit = h0.w;
            next_leaf = m->next2;
        }
        if (unit == 0u) {                                      // a leaf without a segment (cannot happen for a built leaf)
            if (tg == 0 && next_leaf >= 0) pend = grab_slot(a);
            group_sync<WPL>(lg);
            if (next_leaf >= 0) issue_meta<NT>(m, a, next_leaf, 0u, tg);
            cp_async_commit();
            if (tg == 0) m->next2 = (next_leaf >= 0) ? resolve_slot(a, pend) : -1;
            break;
        }
        Seg s;
        s.next = h0.x;
        s.C = (int)(h0.y & 0x7fffu);
        s.K = (int)(h0.y >> 16);
        s.ct = (int)m->cnt[lane];
        s.ell = (const uint16_t*)(a.arena + unit + CRK_SEG_HDR_UNITS + (first ? 0 : ((s.C + 3) >> 2)));
        const int rows = s.K;
        const int mine = s.ct;
        const uint16_t* ep = s.ell + lane;
        CRK_CHECK(a.flag, s.C >= 0 && s.C <= CRK_CCAP && rows >= 0 && rows <= CRK_QCAP && mine <= rows, 8);   // segment header
        // stage: 16-byte asynchronous copies global -> shared (LDGSTS), no register round trip
        if (ROWP > 0) {
            constexpr int RS = (ROWP == 8) ? 3 : 1;                // log2(ROWP)
            const int total = s.C << RS;
            const uint32_t pc = (uint32_t)(tg & (ROWP - 1));       // NT is a multiple of ROWP: a thread always copies the same piece
            const uint32_t dst0 = tile_s + pc * PSTRIDE;
            const float4* src0 = rows_src + pc;
#pragma unroll 4
            for (int f = tg; f < total; f += NT) {
                const int c = f >> RS;
                const uint32_t j = m->cand[c];
                CRK_CHECK(a.flag, (int64_t)j < a.np, 9);                                    // candidate index
                cp_async16(dst0 + (uint32_t)c * 16u, src0 + (int64_t)j * RSTRIDE);
            }
        }
        if (PLANES > 0) {
            for (int c0 = 0; c0 < s.C; c0 += NT * 2) {
                const int ca = c0 + tg, cb = ca + NT;
                const uint32_t ja = (ca < s.C) ? m->cand[ca] : 0u;
                const uint32_t jb = (cb < s.C) ? m->cand[cb] : 0u;
                CRK_CHECK(a.flag, (int64_t)ja < a.np && (int64_t)jb < a.np, 9);             // candidate index
                if (ca < s.C) {
#pragma unroll
                    for (int p = 0; p < PLANES; ++p) cp_async16(tile_s + (uint32_t)(ROWP + p) * PSTRIDE + (uint32_t)ca * 16u, planes[p] + ja);
                }
                if (cb < s.C) {
#pragma unroll
                    for (int p = 0; p < PLANES; ++p) cp_async16(tile_s + (uint32_t)(ROWP + p) * PSTRIDE + (uint32_t)cb * 16u, planes[p] + jb);
                }
            }
        }
        cp_async_commit();
        // the first rows of the entry block travel together with the state
        uint32_t e[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int k = wl + q * WPL;
            e[q] = (k < rows) ? (uint32_t)__ldg(ep + k * 32) : CRK_ELL_SYM;
        }
        const bool last = (s.next == 0u);
        if (first) staged();
        if (last && tg == 0 && next_leaf >= 0) pend = grab_slot(a);          // looked at when the leaf ends
        group_sync<WPL>(lg);                                   // B2
        if (!last) issue_meta<NT>(m, a, 0, s.next, tg);
        else if (next_leaf >= 0) issue_meta<NT>(m, a, next_leaf, 0u, tg);
        cp_async_commit();
        asm volatile("cp.async.wait_group 1;" ::: "memory");   // the state copies (the metadata copy may still be in flight)
        group_sync<WPL>(lg);                                   // B3
        if (first) {
            init(tile_s);
            first = false;
        }
        // plane 0 of the next pair's candidate is fetched one pair ahead: the pair math starts without waiting for shared
        // memory, and the loads of the remaining planes are covered by the arithmetic that needs plane 0 only
        // Padding entries (rows beyond a lane's count) are CRK_ELL_SYM | slot 0: a gather sweep skips them with the test it makes
        // anyway, a symmetric sweep compares the row with the lane's count.
        auto slot_addr = [&](uint32_t ent) {
            uint32_t ad;
            asm("mad.lo.u32 %0, %1, 16, %2;" : "=r"(ad) : "r"(ent & CRK_ELL_MASK), "r"(tile_s));
            return ad;
        };
        float4 cur[NPRE];
        uint32_t sa = slot_addr(e[0]);
#pragma unroll
        for (int p = 0; p < NPRE; ++p) cur[p] = lds128(sa + (uint32_t)p * PSTRIDE);
        for (int k0 = wl; k0 < rows; k0 += 4 * WPL) {
            uint32_t nx[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = k0 + (4 + q) * WPL;
                nx[q] = (k < rows) ? (uint32_t)__ldg(ep + k * 32) : CRK_ELL_SYM;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = k0 + q * WPL;
                const uint32_t en = (q < 3) ? e[(q + 1) & 3] : nx[0];
                const uint32_t san = slot_addr(en);
                float4 nxt[NPRE];
#pragma unroll
                for (int p = 0; p < NPRE; ++p) nxt[p] = lds128(san + (uint32_t)p * PSTRIDE);
                CRK_CHECK(a.flag, k >= mine || (int)(e[q] & CRK_ELL_MASK) < s.C, 10);       // entry -> staged slot
                CRK_CHECK(a.flag, SYM || k < mine || (e[q] & CRK_ELL_SYM) != 0u, 11);       // padding carries the skip flag
                if (SYM ? (k < mine) : !(e[q] & CRK_ELL_SYM)) pair(sa, (e[q] & CRK_ELL_WRAP) != 0u, cur);
                sa = san;
#pragma unroll
                for (int p = 0; p < NPRE; ++p) cur[p] = nxt[p];
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) e[q] = nx[q];
        }
        count += (uint32_t)s.ct;
        if (last) {
            if (tg == 0) m->next2 = (next_leaf >= 0) ? resolve_slot(a, pend) : -1;
            break;
        }
        unit = s.next;
    }
    return count;
}

// add the WPL partial sums of each lane in warp order; the result lands in warp 0 of the group
template <int WPL, int NACC, bool MAX = false>
__device__ __forceinline__ void group_reduce(float (&acc)[NACC], int lg, int wl, int lane, float* red) {
    if (WPL == 1) return;
    group_sync<WPL>(lg);                                       // the tile is no longer read: reuse it
    if (wl > 0) {
#pragma unroll
        for (int q = 0; q < NACC; ++q) red[((wl - 1) * NACC + q) * 32 + lane] = acc[q];
    }
    group_sync<WPL>(lg);
    if (wl == 0) {
        for (int w2 = 1; w2 < WPL; ++w2)
#pragma unroll
            for (int q = 0; q < NACC; ++q) {
                const float v = red[((w2 - 1) * NACC + q) * 32 + lane];
                acc[q] = MAX ? fmaxf(acc[q], v) : acc[q] + v;
            }
    }
}

// Wendland C4 (Eq. 12) without its sigma/h^3 prefactor, and D~ with W'/r = sigma h^-5 D~:
//   W~ = (1-eta)^6 (1 + 6 eta + 35/3 eta^2),   D~ = -(56/3) (1-eta)^5 (1 + 5 eta)
__device__ __forceinline__ void wendland(float eta, float& Wt, float& Dt) {
    const float t = fmaxf(__fsub_rn(1.0f, eta), 0.0f);
    const float t2 = __fmul_rn(t, t);
    const float t5 = __fmul_rn(__fmul_rn(t2, t2), t);
    Wt = __fmul_rn(__fmul_rn(t5, t), __fmaf_rn(eta, __fmaf_rn(eta, C35_3, 6.0f), 1.0f));
    Dt = __fmul_rn(__fmul_rn(-C56_3, t5), __fmaf_rn(5.0f, eta, 1.0f));
}
__device__ __forceinline__ float wendland_w(float eta) {
    const float t = fmaxf(1.0f - eta, 0.0f);
    const float t2 = t * t;
    return t2 * t2 * t2 * fmaf(eta, fmaf(eta, C35_3, 6.0f), 1.0f);
}

// Separation of an accepted pair for the VALUES (the set membership was decided by the prescribed predicate).
// Plain pairs: d = x_i - x_j.  Pairs that cross the periodic boundary (entry bit 15): shift the coordinate that lies in
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

// =================================================================================================== a1: volumes
// Eq. 14: V_i^-1 = n_i = sum_j W(|x_i - x_j|, h_i), self term included (S4); rho_i = m_i / V_i (S2).
constexpr int W1_WPC = 2;
constexpr int W1_SMEM = (int)PSTRIDE + (int)sizeof(Meta);     // per warp
__global__ void __launch_bounds__(W1_WPC * 32) k_volumes(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    float4* tile = (float4*)(smem_raw + (size_t)w * W1_SMEM);
    Meta* meta = (Meta*)((unsigned char*)tile + PSTRIDE);
    const float4* const planes[1] = {a.posh};
    long long leaf = sweep_begin<1>(a, meta, w, 0, lane);
    while (leaf >= 0) {
        const int64_t i = leaf * CRK_LEAF + lane;
        const bool valid = i < a.n;
        const float4 pi = a.posh[i];
        const float xi = pi.x, yi = pi.y, zi = pi.z, hi = pi.w;
        const float inv_h = valid ? 1.0f / hi : 0.0f;
        float acc = 0.0f;
        uint32_t count = 0;                                  // neighbours of the gather set (Eqs. 13-14), self excluded
        long long next;
        leaf_sweep<1, 0, 1, false>(a, nullptr, planes, leaf, next, w, 0, lane, tile, meta, [&](uint32_t, bool wrapped, const float4* pre) {
            const float4 pj = pre[0];
            float dx, dy, dz, r2;
            sep3(a, wrapped, xi, yi, zi, pj, dx, dy, dz, r2);
            const float r = r2 * rsqrt_fast(fmaxf(r2, R2_TINY));
            acc += wendland_w(r * inv_h);
            ++count;
        });
        if (valid) {
            const float k3 = SIGMA_C4 * inv_h * inv_h * inv_h;
            const float ni = k3 * (acc + 1.0f);              // self term W~(0) = 1
            const float V = 1.0f / ni;
            const int32_t p = a.perm[i];
            const float mi = a.m_in[p];
            a.m_s[i] = mi;
            const float rho = mi * ni;
            a.posV[i] = make_float4(xi, yi, zi, V);
            a.rho_s[i] = rho;
            if (a.o0) a.o0[p] = V;
            if (a.o1) a.o1[p] = rho;
            if (a.ocnt) a.ocnt[p] = count;
        } else {
            a.posV[i] = make_float4(pi.x, pi.y, pi.z, 0.0f);
            a.rho_s[i] = 0.0f;
            a.m_s[i] = 1.0f;
        }
        leaf = next;
    }
}

// ---- hydro preparation: sorted (vx,vy,vz,V), and force-sweep plane 0 = (x,y,z,1/h) -----------------------------------
__global__ void __launch_bounds__(256) k_pack_vel(const float* __restrict__ vx, const float* __restrict__ vy,
                                                  const float* __restrict__ vz, const float* __restrict__ u, int64_t n,
                                                  float4* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_float4(vx[i], vy[i], vz[i], u[i]);
}
__global__ void __launch_bounds__(256) k_hydro_prep(SweepArgs a, const float4* __restrict__ vel_orig, float* __restrict__ u_s) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.np) return;
    const float4 ph = a.posh[k];
    if (k < a.n) {
        const float4 v = vel_orig[a.perm[k]];
        a.xv[k * 2] = make_float4(ph.x, ph.y, ph.z, 1.0f / ph.w);
        a.xv[k * 2 + 1] = make_float4(v.x, v.y, v.z, a.posV[k].w);
        u_s[k] = v.w;
    } else {
        a.xv[k * 2] = make_float4(ph.x, ph.y, ph.z, 0.0f);
        a.xv[k * 2 + 1] = make_float4(0, 0, 0, 0);
        u_s[k] = 0.0f;
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
// W~ = (1-eta)^6 (1 + 6 eta + 35/3 eta^2) and D~ = (1-eta)^5 (1 + 5 eta): Eq. 12 and W'/r without sigma/h^3 and
// -(56/3) sigma/h^5, which the force sweep keeps folded into c', M' and A' (explicit intrinsics: identical bits on both lanes)
__device__ __forceinline__ void wendland_folded(float eta, float& Wt, float& Dt) {
    const float t = fmaxf(__fsub_rn(1.0f, eta), 0.0f);
    const float t2 = __fmul_rn(t, t);
    const float t5 = __fmul_rn(__fmul_rn(t2, t2), t);
    Wt = __fmul_rn(__fmul_rn(t5, t), __fmaf_rn(eta, __fmaf_rn(eta, C35_3, 6.0f), 1.0f));
    Dt = __fmul_rn(t5, __fmaf_rn(5.0f, eta, 1.0f));
}

// ================================================================== a2 + a3 + a4: RK coefficients and velocity gradient
// A, B from  sum_j V_j WR_ij = 1,  sum_j V_j x_ij WR_ij = 0.  With moments over the gather set
//   m0 = sum w, m1 = sum w x, m2 = sum w x x  (w = V_j W_ij, self term in m0 only) and their gradients
//   d_c m0 = sum g x_c, d_c m1_a = sum g x_a x_c + delta_ac m0, d_c m2_ab = sum g x_a x_b x_c + delta_ac m1_b + delta_bc m1_a
//   (g = V_j W'_ij / r):   B = -m2^-1 m1,  A = 1/(m0 + B.m1),
//   d_c A = -A^2 (d_c m0 + 2 B.d_c m1 + B^T d_c m2 B),  d_c B = -m2^-1 (d_c m1 + d_c m2 B).
// 29 FP32 sums per particle in eta-normalised units, then an FP64 3x3 solve per particle (a3).
//
// Eq. 26: grad v_i = - sum_j V_j (v_i - v_j) (x) grad WR_ij over the same gather set; index [3a+b] = d_b v^a.
// grad WR_ij = W (cvec + M x) + A (1 + B.x) D x is linear in the coefficients of particle i, so the sweep accumulates 39
// velocity-weighted sums that do not need them (u = v_i - v_j, w = V_j W, g = V_j D):
//   S0^a = sum u^a w (3),  S1^ac = sum u^a w x^c (9),  T1^ab = sum u^a g x^b (9),  T2^a(cb) = sum u^a g x^c x^b (3 x 6)
// and the epilogue contracts  (grad v)^ab = -(cvec_b S0^a + M_bc S1^ac + A T1^ab + A B_c T2^acb)  with the stored FP32
// coefficients.  MOM && GV (crk_step_derivs): one sweep does both, so the lists and the tile are read once.  The
// accumulation code of each sum is the same in all three instantiations (explicit round-to-nearest intrinsics, nothing for
// the compiler to contract differently), so the staged calls and crk_step_derivs produce identical bits.
// The epilogue with GV also forms P = (gamma-1) rho u (Eq. 4, unclamped) and c_s = sqrt(gamma (gamma-1) max(u,0)) (S12) and
// writes the packed force-sweep state of the particle.
constexpr int W2_WPC = 2;
constexpr int RK_MINB = 8;        // resident CTAs per SM the merged moments + grad v sweep is compiled for
template <bool MOM, bool GV>
__global__ void __launch_bounds__(W2_WPC * 32, (MOM && GV) ? RK_MINB : (GV ? 8 : 10))
k_rk(SweepArgs a, const float* __restrict__ u_s, float* __restrict__ gv_full) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // tile: GV -> the candidates' entries of the compact array xv, (x,y,z,1/h) and (vx,vy,vz,V): one 32-byte sector each;
    // moments only (crk_rk_coefficients, before the hydro preparation) -> the SoA plane (x,y,z,V)
    constexpr int PL = GV ? 2 : 1;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    constexpr int WSMEM = PL * (int)PSTRIDE + (int)sizeof(Meta);     // per warp
    float4* tile = (float4*)(smem_raw + (size_t)w * WSMEM);
    Meta* meta = (Meta*)((unsigned char*)tile + PL * PSTRIDE);
    const float4* planes[1] = {a.posV};
    long long leaf = sweep_begin<1>(a, meta, w, 0, lane);
    while (leaf >= 0) {
        long long next;
        const int64_t i = leaf * CRK_LEAF + lane;
        const bool valid = i < a.n;
        const float4 ph = a.posh[i];
        const float xi = ph.x, yi = ph.y, zi = ph.z, hi = ph.w;
        const float inv_h = valid ? 1.0f / hi : 0.0f;
        float4 vi = make_float4(0.f, 0.f, 0.f, 0.f);
        if (GV) vi = a.xv[i * 2 + 1];
        // moment accumulators: s0; s1[3]; s2[6] (xx,xy,xz,yy,yz,zz); t0[3]; t1[6]; t2[10] (xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz)
        float s0 = 0.f, s1[3] = {0.f, 0.f, 0.f}, s2[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float t0[3] = {0.f, 0.f, 0.f}, t1[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, t2[10] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        // velocity sums, [a][..]
        float S0[3], S1[3][3], T1[3][3], T2[3][6];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            S0[q] = 0.f;
#pragma unroll
            for (int r = 0; r < 3; ++r) { S1[q][r] = 0.f; T1[q][r] = 0.f; }
#pragma unroll
            for (int r = 0; r < 6; ++r) T2[q][r] = 0.f;
        }
        leaf_sweep<1, GV ? 2 : 0, GV ? 0 : 1, false>(a, a.xv, planes, leaf, next, w, 0, lane, tile, meta, [&](uint32_t sa, bool wrapped, const float4* pre) {
            const float4 pj = pre[0];
            float4 vj = make_float4(0.f, 0.f, 0.f, 0.f);
            if (GV) vj = lds128(sa + PSTRIDE);
            const float Vj = GV ? vj.w : pj.w;
            float dx, dy, dz, r2;
            sep3(a, wrapped, xi, yi, zi, pj, dx, dy, dz, r2);
            const float r = __fmul_rn(r2, rsqrt_fast(fmaxf(r2, R2_TINY)));
            float Wt, Dt;
            wendland(__fmul_rn(r, inv_h), Wt, Dt);
            const float wv = __fmul_rn(Vj, Wt), gv = __fmul_rn(Vj, Dt);
            const float x[3] = {__fmul_rn(dx, inv_h), __fmul_rn(dy, inv_h), __fmul_rn(dz, inv_h)};
            const float m2[6] = {__fmul_rn(x[0], x[0]), __fmul_rn(x[0], x[1]), __fmul_rn(x[0], x[2]),
                                 __fmul_rn(x[1], x[1]), __fmul_rn(x[1], x[2]), __fmul_rn(x[2], x[2])};
            if (MOM) {
                s0 = __fadd_rn(s0, wv);
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    s1[q] = __fmaf_rn(wv, x[q], s1[q]);
                    t0[q] = __fmaf_rn(gv, x[q], t0[q]);
                }
                float g2[6];
#pragma unroll
                for (int q = 0; q < 6; ++q) {
                    s2[q] = __fmaf_rn(wv, m2[q], s2[q]);
                    g2[q] = __fmul_rn(gv, m2[q]);
                    t1[q] = __fadd_rn(t1[q], g2[q]);
                }
                t2[0] = __fmaf_rn(g2[0], x[0], t2[0]); t2[1] = __fmaf_rn(g2[0], x[1], t2[1]); t2[2] = __fmaf_rn(g2[0], x[2], t2[2]);
                t2[3] = __fmaf_rn(g2[1], x[1], t2[3]); t2[4] = __fmaf_rn(g2[1], x[2], t2[4]); t2[5] = __fmaf_rn(g2[2], x[2], t2[5]);
                t2[6] = __fmaf_rn(g2[3], x[1], t2[6]); t2[7] = __fmaf_rn(g2[3], x[2], t2[7]); t2[8] = __fmaf_rn(g2[4], x[2], t2[8]);
                t2[9] = __fmaf_rn(g2[5], x[2], t2[9]);
            }
            if (GV) {
                const float u[3] = {__fsub_rn(vi.x, vj.x), __fsub_rn(vi.y, vj.y), __fsub_rn(vi.z, vj.z)};
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const float uw = __fmul_rn(u[q], wv), ug = __fmul_rn(u[q], gv);
                    S0[q] = __fadd_rn(S0[q], uw);
#pragma unroll
                    for (int r = 0; r < 3; ++r) {
                        S1[q][r] = __fmaf_rn(uw, x[r], S1[q][r]);
                        T1[q][r] = __fmaf_rn(ug, x[r], T1[q][r]);
                    }
#pragma unroll
                    for (int r = 0; r < 6; ++r) T2[q][r] = __fmaf_rn(ug, m2[r], T2[q][r]);
                }
            }
        });
        float4 o0 = make_float4(0, 0, 0, 0), o1 = o0, o2 = o0, o3 = o0;
        const double h = (double)hi, ih = valid ? 1.0 / h : 0.0;
        const double k3 = (double)SIGMA_C4 * ih * ih * ih;
        if (MOM) {
            if (valid) {
                // ---- a3: FP64 solve (dimensional quantities; k3 = sigma/h^3)
                const double Vi = (double)a.posV[i].w;
                const double m0 = k3 * ((double)s0 + Vi);
                const double m1[3] = {k3 * h * s1[0], k3 * h * s1[1], k3 * h * s1[2]};
                const double k3h2 = k3 * h * h;
                const double mm[3][3] = {{k3h2 * s2[0], k3h2 * s2[1], k3h2 * s2[2]},
                                         {k3h2 * s2[1], k3h2 * s2[3], k3h2 * s2[4]},
                                         {k3h2 * s2[2], k3h2 * s2[4], k3h2 * s2[5]}};
                const double dm0[3] = {k3 * ih * t0[0], k3 * ih * t0[1], k3 * ih * t0[2]};
                // sum g x_a x_c (symmetric)
                const double q1[3][3] = {{k3 * t1[0], k3 * t1[1], k3 * t1[2]}, {k3 * t1[1], k3 * t1[3], k3 * t1[4]}, {k3 * t1[2], k3 * t1[4], k3 * t1[5]}};
                const double k3h = k3 * h;
                double cc[10];
#pragma unroll
                for (int q = 0; q < 10; ++q) cc[q] = k3h * t2[q];
                // inverse of m2 (adjugate)
                const double a00 = mm[1][1] * mm[2][2] - mm[1][2] * mm[1][2];
                const double a01 = mm[0][2] * mm[1][2] - mm[0][1] * mm[2][2];
                const double a02 = mm[0][1] * mm[1][2] - mm[0][2] * mm[1][1];
                const double a11 = mm[0][0] * mm[2][2] - mm[0][2] * mm[0][2];
                const double a12 = mm[0][1] * mm[0][2] - mm[0][0] * mm[1][2];
                const double a22 = mm[0][0] * mm[1][1] - mm[0][1] * mm[0][1];
                const double det = mm[0][0] * a00 + mm[0][1] * a01 + mm[0][2] * a02;
                double A, B[3], dA[3], dB[3][3];   // dB[c][a] = d_c B^a
                // S14: m2 counts as singular when det m2 <= 1e-4 (tr m2 / 3)^3 (neighbours span less than three dimensions)
                const double tr3 = (mm[0][0] + mm[1][1] + mm[2][2]) * (1.0 / 3.0);
                if (det > 1.0e-4 * tr3 * tr3 * tr3 && isfinite(det)) {
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
                    atomicAdd((unsigned int*)a.flag + FW_FALLBACK, 1u);   // reported by crk_get_stats (rare: none on the BASELINE configs)
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
        } else {
            o0 = a.coef[i]; o1 = a.coef[a.np + i]; o2 = a.coef[2 * a.np + i]; o3 = a.coef[3 * a.np + i];
        }
        if (!GV) {
            leaf = next;
            continue;
        }
        // ---- a4: contraction of the velocity sums with the stored FP32 coefficients (FP64 arithmetic)
        float g[9];
        {
            const Coef k = load_coef(o0, o1, o2, o3);
            const double cv[3] = {(double)k.cx, (double)k.cy, (double)k.cz};
            const double Bv[3] = {(double)k.Bx, (double)k.By, (double)k.Bz};
            const double A = (double)k.A;
            const double k3h = k3 * h, k3ih = k3 * ih;
            const int sym[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
#pragma unroll
            for (int al = 0; al < 3; ++al)
#pragma unroll
                for (int be = 0; be < 3; ++be) {
                    double t = cv[be] * (k3 * (double)S0[al]) + A * (k3ih * (double)T1[al][be]);
#pragma unroll
                    for (int c = 0; c < 3; ++c)
                        t += (double)k.M[3 * be + c] * (k3h * (double)S1[al][c]) + A * Bv[c] * (k3 * (double)T2[al][sym[c][be]]);
                    g[3 * al + be] = (float)(-t);
                }
        }
        // force-sweep state row (FROW float4 = one 128-byte line per particle; pieces 0 and 1 repeat the compact array xv):
        //   (x,y,z,1/h) (vx,vy,vz,V) | (A',B) (c',M'0) (M'1..M'4) (M'5..M'8) (gxx,gyy,gzz,P) (gxy+gyx, gxz+gzx, gyz+gzy, rho)
        // with the kernel normalisation folded into the coefficients, A' = -(56/3) sigma/h^5 A, c' = sigma/h^3 c,
        // M' = sigma/h^3 M, so that grad WR_ij = W~ (c' + M' x) + A' s D~ x with the dimensionless W~ = (1-eta)^6 (1+6 eta+35/3 eta^2),
        // D~ = (1-eta)^5 (1+5 eta).  Only x.(grad v x) enters Eqs. 27-30 and Eq. 25 (uhat_ij.x_ij), so the symmetric part of
        // grad v is all the force sweep needs; c_s = sqrt(gamma P / rho) is re-derived there (S12: P <= 0 -> c_s = 0).
        const float ihf = valid ? 1.0f / hi : 0.0f;
        const float k3f = SIGMA_C4 * ihf * ihf * ihf;
        const float k5f = -C56_3 * (k3f * ihf * ihf);
        const float u = u_s[i], rho = a.rho_s[i], gm = a.gamma;
        const float P = (gm - 1.0f) * rho * u;
        float4* f = a.fst + i * FROW;                        // the whole 128-byte line is written here
        f[0] = make_float4(xi, yi, zi, ihf);
        f[1] = vi;
        f[2] = make_float4(k5f * o0.x, o0.y, o0.z, o0.w);
        f[3] = make_float4(k3f * o1.x, k3f * o1.y, k3f * o1.z, k3f * o1.w);
        f[4] = make_float4(k3f * o2.x, k3f * o2.y, k3f * o2.z, k3f * o2.w);
        f[5] = make_float4(k3f * o3.x, k3f * o3.y, k3f * o3.z, k3f * o3.w);
        f[6] = make_float4(g[0], g[4], g[8], P);
        f[7] = make_float4(g[1] + g[3], g[2] + g[6], g[5] + g[7], rho);
        if (gv_full && valid) {                              // diagnostics (crk_get_gradv): all nine components, caller order
            const int32_t p = a.perm[i];
#pragma unroll
            for (int q = 0; q < 9; ++q) gv_full[q * a.n + p] = g[q];
        }
        leaf = next;
    }
}

// ============================================================================================ a5: momentum and energy
// Eq. 17:  m_i dv_i/dt = sum_j (1/2) V_i V_j (P_i+Q_i+P_j+Q_j) (grad WR_ji - grad WR_ij)
// Eq. 18:  m_i du_i/dt = sum_j (1/2) V_i V_j (P_j+Q_j) (v_j - v_i).(grad WR_ji - grad WR_ij)       (S6)
// Q from Eqs. 24-25 with the limited midpoint projection of Eqs. 27-32 (S7: division-free van Leer form).
// Sums over all j != i with r2 < max(h_i^2, h_j^2); each ordered pair is evaluated on a lane that holds i in registers.
// One CTA = one leaf: W5_WPL warps share the tile of the leaf's candidates and split each lane's entries by rows.
struct ForceConst {
    float L, half, eta_crit, inv_fold, eps2, Cl, Cq, gamma, n_h;
};
struct PState {           // one particle's force-sweep state in registers
    float x, y, z, ih, vx, vy, vz, V, P, rho, cs, qh;
    Coef c;                                              // A', B, c', M' (kernel normalisation folded in, see k_rk)
    float gxx, gyy, gzz, gxy, gxz, gyz;                  // symmetric part of grad v, off-diagonals summed
};
constexpr int FPRE = 1;   // planes of the next pair's j-state fetched one pair ahead (3, 5, 9 measured slower: 11.3, 11.5, 13.5 vs 11.1 ms)
// the row of candidate slot `sa` from the tile.  c_s = sqrt(gamma max(P,0) / rho) (Eq. 4 + PAPER.md:149, S12) and q = n_h / h are
// re-derived here with a fixed instruction sequence, so both lanes of a pair hold identical bits for either particle.
__device__ __forceinline__ PState load_pstate_shared(const ForceConst& k, uint32_t sa, const float4* pre) {
    float4 q[FROW];
#pragma unroll
    for (int p = 0; p < FROW; ++p) q[p] = (p < FPRE) ? pre[p] : lds128(sa + (uint32_t)p * PSTRIDE);
    PState s;
    s.x = q[0].x; s.y = q[0].y; s.z = q[0].z; s.ih = q[0].w;
    s.vx = q[1].x; s.vy = q[1].y; s.vz = q[1].z; s.V = q[1].w;
    s.c = load_coef(q[2], q[3], q[4], q[5]);
    s.gxx = q[6].x; s.gyy = q[6].y; s.gzz = q[6].z; s.P = q[6].w;
    s.gxy = q[7].x; s.gxz = q[7].y; s.gyz = q[7].z; s.rho = q[7].w;
    s.qh = __fmul_rn(k.n_h, s.ih);
    const float gp = __fmul_rn(k.gamma, fmaxf(s.P, 0.0f));
    s.cs = __fmul_rn(gp, rsqrt_fast(fmaxf(__fmul_rn(gp, s.rho), R2_TINY)));
    return s;
}
// x.(grad v x) with the symmetric part (Eq. 30 numerator / denominator)
__device__ __forceinline__ float quad_form(const PState& s, float dxx, float dyy, float dzz, float dxy, float dxz, float dyz) {
    return __fmaf_rn(s.gyz, dyz, __fmaf_rn(s.gxz, dxz, __fmaf_rn(s.gxy, dxy,
           __fmaf_rn(s.gzz, dzz, __fmaf_rn(s.gyy, dyy, __fmul_rn(s.gxx, dxx))))));
}
// Eq. 25 with hhat = h/n_h, q = 1/hhat:  mu = min(0, hhat (uhat.x) / (r^2 + hhat^2 eps^2)) = min(0, q (uhat.x) / (q^2 r^2 + eps^2))
__device__ __forceinline__ float visc_mu(float qh, float udx, float r2, float eps2) {
    return fminf(0.0f, __fmul_rn(__fmul_rn(qh, udx), rcp_fast(__fmaf_rn(__fmul_rn(qh, qh), r2, eps2))));
}
// one ordered pair (i, j): F = m_i a_ij (Eq. 17 with P -> P + Q) and e = its term of m_i du_i/dt (Eq. 18);
// vji = v_j - v_i
struct PairF { float Fx, Fy, Fz, e, vjix, vjiy, vjiz, app, Qi; };   // app = approach speed (Eq. 50), Qi (Eq. 24)
__device__ __forceinline__ PairF force_pair(const ForceConst& k, const PState& I, const PState& J, bool wrapped) {
    float dx, dy, dz;
    if (!wrapped) {
        dx = __fsub_rn(I.x, J.x);
        dy = __fsub_rn(I.y, J.y);
        dz = __fsub_rn(I.z, J.z);
    } else {
        dx = sep1_wrapped(I.x, J.x, k.L, k.half);
        dy = sep1_wrapped(I.y, J.y, k.L, k.half);
        dz = sep1_wrapped(I.z, J.z, k.L, k.half);
    }
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    const float rinv = rsqrt_fast(fmaxf(r2, R2_TINY));
    const float r = __fmul_rn(r2, rinv);
    float Wi, Di, Wj, Dj;                                       // W~, D~ (the normalisation sits in A', c', M')
    wendland_folded(__fmul_rn(r, I.ih), Wi, Di);
    wendland_folded(__fmul_rn(r, J.ih), Wj, Dj);
    float aix, aiy, aiz, ajx, ajy, ajz;
    rk_grad(I.c, dx, dy, dz, Wi, Di, aix, aiy, aiz);            // grad WR_ij
    rk_grad(J.c, -dx, -dy, -dz, Wj, Dj, ajx, ajy, ajz);         // grad WR_ji  (x_ji = -x_ij)
    const float Gx = __fsub_rn(ajx, aix), Gy = __fsub_rn(ajy, aiy), Gz = __fsub_rn(ajz, aiz);
    // Eq. 30: N = x.(grad v_i x), Dn = x.(grad v_j x); every product is even in x, so the mirrored lane forms the same bits
    const float dxx = __fmul_rn(dx, dx), dyy = __fmul_rn(dy, dy), dzz = __fmul_rn(dz, dz);
    const float dxy = __fmul_rn(dx, dy), dxz = __fmul_rn(dx, dz), dyz = __fmul_rn(dy, dz);
    const float Nn = quad_form(I, dxx, dyy, dzz, dxy, dxz, dyz);
    const float Dn = quad_form(J, dxx, dyy, dzz, dxy, dxz, dyz);
    // Eq. 29 with r_ij = N/Dn:  phi_VL = 4 N Dn / (N + Dn)^2 if N Dn > 0 else 0  (S7)
    const float nd = __fmul_rn(Nn, Dn);
    const float sm = __fadd_rn(Nn, Dn);
    float phi = (nd > 0.0f) ? fminf(__fmul_rn(4.0f * nd, rcp_fast(__fmul_rn(sm, sm))), 1.0f) : 0.0f;
    // Eqs. 31-32
    const float eta = __fmul_rn(r, fminf(I.ih, J.ih));
    if (eta < k.eta_crit) {
        const float q = (eta - k.eta_crit) * k.inv_fold;
        phi *= ex2_fast(-1.4426950408889634f * q * q);
    }
    // Eq. 27 (adot = 0): uhat_ij.x_ij = v_ij.x_ij - (1/2) phi x_ij.(grad v_i + grad v_j).x_ij = v_ij.x_ij - (1/2) phi (N + Dn)
    const float vx = __fsub_rn(I.vx, J.vx), vy = __fsub_rn(I.vy, J.vy), vz = __fsub_rn(I.vz, J.vz);
    const float vdx = __fmaf_rn(vz, dz, __fmaf_rn(vy, dy, __fmul_rn(vx, dx)));
    const float udx = __fmaf_rn(__fmul_rn(-0.5f, phi), sm, vdx);
    // Eqs. 24-25
    const float Qi = visc_Q(I.rho, I.cs, visc_mu(I.qh, udx, r2, k.eps2), k.Cl, k.Cq);
    const float Qj = visc_Q(J.rho, J.cs, visc_mu(J.qh, udx, r2, k.eps2), k.Cl, k.Cq);
    const float PQi = __fadd_rn(I.P, Qi), PQj = __fadd_rn(J.P, Qj);
    const float hvv = 0.5f * __fmul_rn(I.V, J.V);
    const float pf = __fmul_rn(hvv, __fadd_rn(PQi, PQj));
    const float vG = fmaf(vz, Gz, fmaf(vy, Gy, vx * Gx));       // (v_i - v_j).G = -(v_j - v_i).G
    PairF o;
    o.Fx = __fmul_rn(pf, Gx); o.Fy = __fmul_rn(pf, Gy); o.Fz = __fmul_rn(pf, Gz);
    o.e = -hvv * PQj * vG;
    o.vjix = -vx; o.vjiy = -vy; o.vjiz = -vz;
    o.app = fmaxf(-vdx * rinv, 0.0f);
    o.Qi = Qi;
    return o;
}

// One group = one CTA of W5_WPL warps: they share the tile of the leaf's candidates and split each lane's entries by rows;
// four persistent CTAs are resident per SM, so one group's staging overlaps the other three's pair math (with the copies
// switched off the sweep is 8 % faster, no more).  2 .. 6 warps per leaf were measured in round 2.
constexpr int W5_WPL = 4;
// The epilogue of a leaf (sum of the W5_WPL partial results in warp order, division by the mass, stores through the
// permutation) is deferred into the staging window of the group's NEXT leaf, where the warps only wait for their copies: the
// partial sums and what the stores need travel through this record.  One record is enough: nobody reaches the rows of leaf
// n + 1 (and so the next write of the record) before the warp that runs epilogue(n) has passed B2 of leaf n + 1.
template <bool TS>
struct ForceEpi {
    float part[W5_WPL][TS ? 6 : 4][32];      // Fx, Fy, Fz, dE (, max approach speed, max Q_i) of warp w
    float s[32], invm[32];                   // s = P / rho^gamma, 1 / m
    int32_t pidx[32];                        // caller index of the particle, -1: outputs not wanted (passive or padding)
    uint32_t cnt[32];
    long long leaf;                          // -1: nothing pending
    long long pad;
};
template <bool TS>
__device__ __forceinline__ void force_epilogue(const SweepArgs& a, const ForceEpi<TS>* ep, int lane) {
    const long long leaf = ep->leaf;
    if (leaf < 0) return;
    const int64_t i = leaf * CRK_LEAF + lane;
    float acc[TS ? 6 : 4];
#pragma unroll
    for (int q = 0; q < (TS ? 6 : 4); ++q) acc[q] = ep->part[0][q][lane];
    for (int w2 = 1; w2 < W5_WPL; ++w2) {
#pragma unroll
        for (int q = 0; q < 4; ++q) acc[q] += ep->part[w2][q][lane];
        if (TS) {
            acc[4] = fmaxf(acc[4], ep->part[w2][4][lane]);
            acc[5] = fmaxf(acc[5], ep->part[w2][5][lane]);
        }
    }
    if (TS) a.ts[i] = make_float2(acc[4], acc[5]);
    const float im = ep->invm[lane];
    const float4 as = make_float4(acc[0] * im, acc[1] * im, acc[2] * im, ep->s[lane]);
    const int32_t p = ep->pidx[lane];
    if (p >= 0) {
        a.o0[p] = as.x;
        a.o1[p] = as.y;
        a.o2[p] = as.z;
        a.o3[p] = acc[3] * im;
        if (a.ocnt) a.ocnt[p] = ep->cnt[lane];
    }
    a.facc[i] = as;                                      // (dv/dt, s = P / rho^gamma) for crk_compatible_energy, crk_timestep
}

template <bool TS>   // TS: also reduce the per-particle maxima the time-step criteria need (Eqs. 46, 50)
__global__ void __launch_bounds__(W5_WPL * 32, 4) k_forces(SweepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    float4* tile = (float4*)smem_raw;
    Meta* meta = (Meta*)(smem_raw + FROW * PSTRIDE);
    ForceEpi<TS>* epi = (ForceEpi<TS>*)(smem_raw + FROW * PSTRIDE + sizeof(Meta));
    const ForceConst fc = {a.L, a.half, 1.0f / a.n_h, a.n_h / 0.2f, a.eps2, a.C_l, a.C_q, a.gamma, a.n_h};
    if (threadIdx.x == 0) epi->leaf = -1;
    long long leaf = sweep_begin<W5_WPL>(a, meta, 0, wl, lane);
    while (leaf >= 0) {
        const int64_t i = leaf * CRK_LEAF + lane;
        const bool valid = i < a.n;
        PState I;                                            // taken from the tile (slots 0..31 = the leaf's own particles)
        // what the epilogue needs from global memory is requested now, not after the last row
        const float mi = (wl == 0) ? a.m_s[i] : 1.0f;
        const int32_t pidx = (wl == 0 && valid) ? a.perm[i] : 0;
        const bool write_out = (wl == 0 && valid) && (!a.active || a.active[pidx]);
        float acc[4] = {0.f, 0.f, 0.f, 0.f};                 // Fx, Fy, Fz, dE
        float mx[2] = {0.f, 0.f};                            // max approach speed, max Q_i
        long long next;
        const uint32_t count = leaf_sweep<W5_WPL, FROW, 0, true, FPRE>(a, a.fst, nullptr, leaf, next, 0, wl, lane, tile, meta, [&](uint32_t sa, bool wrapped, const float4* pre) {
            const PState J = load_pstate_shared(fc, sa, pre);
            const PairF f = force_pair(fc, I, J, wrapped);
            acc[0] += f.Fx; acc[1] += f.Fy; acc[2] += f.Fz; acc[3] += f.e;
            if (TS) {
                mx[0] = fmaxf(mx[0], f.app);
                mx[1] = fmaxf(mx[1], f.Qi);
            }
        }, [&](uint32_t ts) {
            float4 pre[FPRE];
#pragma unroll
            for (int p = 0; p < FPRE; ++p) pre[p] = lds128(ts + (uint32_t)p * PSTRIDE + (uint32_t)lane * 16u);
            I = load_pstate_shared(fc, ts + (uint32_t)lane * 16u, pre);
        }, [&]() {
            if (wl == W5_WPL - 1) force_epilogue<TS>(a, epi, lane);      // of the previous leaf (its record was complete at B1)
        });
#pragma unroll
        for (int q = 0; q < 4; ++q) epi->part[wl][q][lane] = acc[q];
        if (TS) {
            epi->part[wl][4][lane] = mx[0];
            epi->part[wl][5][lane] = mx[1];
        }
        if (wl == 0) {
            epi->s[lane] = valid ? I.P * __powf(I.rho, -a.gamma) : 0.0f;
            epi->invm[lane] = valid ? 1.0f / mi : 0.0f;
            epi->pidx[lane] = write_out ? pidx : -1;
            epi->cnt[lane] = count;
            if (lane == 0) epi->leaf = leaf;
        }
        leaf = next;
    }
    group_sync<W5_WPL>(0);
    if (wl == W5_WPL - 1) force_epilogue<TS>(a, epi, lane);
}

// ================================================================================ NEXT row 1: compatible energy update
// Eqs. 19-23 with a = 1, adot = 0, p = v:  Delta u_i = dt sum_j (f_ij / 2) (v_j + v'_j - v_i - v'_i) . a_ij,
// v' = v + (dv/dt) dt (Eq. 22), a_ij the pairwise acceleration of Eq. 17 (recomputed: storing it per pair would cost 12 GB).
// sign(dE_ij) = sign(m_i a_ij . (v_j + v'_j - v_i - v'_i)) (Eq. 21, independent of f); Eq. 23 per DESIGN.md reading G1;
// f = 1/2 if an entropy is not positive (S16).  Both lanes of a pair form bit-identical F and velocity sums, so they take
// the same branch of Eq. 23 and f_ij + f_ji = 1 up to the rounding of the reciprocal.
// kick plane: (v' - v, s) per particle, sorted order.  Eq. 22 as printed: v' - v = (dv/dt) dt (c1 = dt, no b).  The Verlet step's
// second half kick starts from v^1/2 while the sweep state holds the predicted velocities v_p = v^1/2 + a^0 dt/2, so there
// v^1/2 + v^1 = 2 v_p + (a^1 dt/2 - a^0 dt): c1 = dt/2 on the resident dv/dt, c0 = -dt on b = a^0 (caller order).
__global__ void __launch_bounds__(256) k_compat_prep(const float4* __restrict__ acc_s, const int32_t* __restrict__ perm, int64_t n,
                                                     int64_t np, float c1, float c0, const float* __restrict__ bx,
                                                     const float* __restrict__ by, const float* __restrict__ bz,
                                                     float4* __restrict__ kick) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= np) return;
    const float4 q = acc_s[k];
    float4 w = make_float4(c1 * q.x, c1 * q.y, c1 * q.z, q.w);
    if (bx && k < n) {
        const int32_t p = perm[k];
        w.x = fmaf(c0, bx[p], w.x); w.y = fmaf(c0, by[p], w.y); w.z = fmaf(c0, bz[p], w.z);
    }
    kick[k] = w;
}

__global__ void __launch_bounds__(W5_WPL * 32, 4) k_compat(SweepArgs a, float dt, const float4* __restrict__ kick) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    float4* tile = (float4*)smem_raw;
    Meta* meta = (Meta*)(smem_raw + CPL * PSTRIDE);
    const ForceConst fc = {a.L, a.half, 1.0f / a.n_h, a.n_h / 0.2f, a.eps2, a.C_l, a.C_q, a.gamma, a.n_h};
    const float4* planes[1] = {kick};                       // tile plane FROW
    long long leaf = sweep_begin<W5_WPL>(a, meta, 0, wl, lane);
    while (leaf >= 0) {
        const int64_t i = leaf * CRK_LEAF + lane;
        const bool valid = i < a.n;
        PState I;                                            // from the tile, as in k_forces
        const float4 qi = kick[i];
        float acc[1] = {0.f};
        long long next;
        leaf_sweep<W5_WPL, FROW, 1, true, FPRE>(a, a.fst, planes, leaf, next, 0, wl, lane, tile, meta, [&](uint32_t sa, bool wrapped, const float4* pre) {
            const PState J = load_pstate_shared(fc, sa, pre);
            const float4 qj = lds128(sa + (uint32_t)FROW * PSTRIDE);
            const PairF f = force_pair(fc, I, J, wrapped);
            // (v_j + v'_j - v_i - v'_i) = 2 (v_j - v_i) + (kick_j - kick_i)
            const float wx = __fmaf_rn(2.0f, f.vjix, __fsub_rn(qj.x, qi.x));
            const float wy = __fmaf_rn(2.0f, f.vjiy, __fsub_rn(qj.y, qi.y));
            const float wz = __fmaf_rn(2.0f, f.vjiz, __fsub_rn(qj.z, qi.z));
            const float w = __fmaf_rn(f.Fz, wz, __fmaf_rn(f.Fy, wy, __fmul_rn(f.Fx, wx)));       // = 2 dE_ij
            const float si = qi.w, sj = qj.w;
            float part = 0.5f;
            if (si > 0.0f && sj > 0.0f) {
                const bool small = (w >= 0.0f) ? (si >= sj) : (si < sj);
                part = (small ? fminf(si, sj) : fmaxf(si, sj)) * rcp_fast(__fadd_rn(si, sj));
            }
            acc[0] = fmaf(0.5f * part, w, acc[0]);
        }, [&](uint32_t ts) {
            float4 pre[FPRE];
#pragma unroll
            for (int p = 0; p < FPRE; ++p) pre[p] = lds128(ts + (uint32_t)p * PSTRIDE + (uint32_t)lane * 16u);
            I = load_pstate_shared(fc, ts + (uint32_t)lane * 16u, pre);
        });
        group_reduce<W5_WPL, 1>(acc, 0, wl, lane, (float*)tile);
        if (wl == 0 && valid) a.o0[a.perm[i]] = acc[0] * dt / a.m_s[i];
        leaf = next;
    }
}

SweepArgs make_args(crk_ctx* c) {
    SweepArgs a;
    memset(&a, 0, sizeof(a));
    a.n = c->n; a.nl = c->nl; a.np = c->nl * CRK_LEAF;
    a.L = c->prm.box; a.half = 0.5f * c->prm.box;
    a.arena = (const uint4*)c->arena.p; a.seg_first = (const uint4*)c->seg_first.p; a.leaf_cnt = (const uint16_t*)c->leaf_cnt.p;
    a.cand_first = (const uint32_t*)c->cand_first.p;
    a.perm = c->perm;
    a.posh = (const float4*)c->posh.p; a.posV = (float4*)c->posV.p;
    a.coef = (float4*)c->coef.p; a.fst = (float4*)c->fst.p; a.facc = (float4*)c->facc.p; a.xv = (float4*)c->xv.p;
    a.rho_s = (float*)c->rho_s.p; a.m_s = (float*)c->m_s.p;
    a.gamma = c->prm.gamma; a.n_h = c->prm.n_h; a.C_l = c->prm.C_l; a.C_q = c->prm.C_q;
    a.eps2 = c->prm.eps * c->prm.eps;
    a.flag = (int*)c->flag.p;
    a.sched = (unsigned int*)c->sched.p;
    return a;
}

// Launch geometry of a persistent sweep: as many CTAs as are resident at once (occupancy x SMs), never more than there are
// work items; the work counter is zeroed on the stream first.  groups_per_cta = leaves a CTA serves concurrently.
template <typename K>
int persistent_grid(crk_ctx* c, K kernel, int threads, int smem, int groups_per_cta, int64_t items, unsigned* grid) {
    // occupancy and SM count of a (kernel, shared-memory size, device) are asked for once per context, not once per launch.
    // The key is the kernel's ADDRESS: the template parameter K is only its function-pointer type, which k_volumes and both
    // k_forces instantiations share, as do the three k_rk instantiations.
    int dev = 0;
    CRK_CUDA(c, cudaGetDevice(&dev));
    const void* key = (const void*)kernel;
    crk_ctx::GridGeo* g = nullptr;
    for (int q = 0; q < c->n_geo; ++q)
        if (c->geo[q].kernel == key && c->geo[q].smem == smem && c->geo[q].threads == threads && c->geo[q].dev == dev) g = &c->geo[q];
    if (!g) {
        if (smem > 48 * 1024) CRK_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        int per_sm = 0, sms = 0;
        CRK_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, (size_t)smem));
        CRK_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (per_sm < 1) {
            snprintf(c->err, sizeof(c->err), "a sweep kernel does not fit on an SM (%d bytes of shared memory)", smem);
            return CRK_ECUDA;
        }
        g = &c->geo[c->n_geo < crk_ctx::GEO_CAP ? c->n_geo++ : crk_ctx::GEO_CAP - 1];   // a full table reuses its last entry
        g->kernel = key; g->smem = smem; g->threads = threads; g->dev = dev; g->per_sm = per_sm; g->sms = sms;
    }
    const int per_sm = g->per_sm, sms = g->sms;
    const int64_t need = (items + groups_per_cta - 1) / groups_per_cta;
    const int64_t res = (int64_t)per_sm * sms;
    *grid = (unsigned)(need < res ? need : res);
    CRK_TRY(crk_ensure(c, c->sched, 64));
    CRK_CUDA(c, cudaMemsetAsync(c->sched.p, 0, sizeof(unsigned int), c->stream));
    return CRK_OK;
}

}  // namespace

int crk_launch_volumes(crk_ctx* c, const float* m, float* V, float* rho, uint32_t* nbr_count) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->posV, (size_t)np * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->rho_s, (size_t)np * sizeof(float)));
    CRK_TRY(crk_ensure(c, c->m_s, (size_t)np * sizeof(float)));
    SweepArgs a = make_args(c);
    a.m_in = m;
    a.o0 = V; a.o1 = rho; a.ocnt = nbr_count;
    const int smem = W1_WPC * W1_SMEM;
    unsigned grid = 0;
    CRK_TRY(persistent_grid(c, k_volumes, W1_WPC * 32, smem, W1_WPC, c->nl, &grid));
    a.sched = (unsigned int*)c->sched.p;
    k_volumes<<<grid, W1_WPC * 32, smem, c->stream>>>(a);
    return crk_check_launch(c, "k_volumes");
}

// hydro preparation: velocities / energies in sorted order (force-sweep state planes 0 and 1); needs the volumes
int crk_launch_hydro_prep(crk_ctx* c, const float* vx, const float* vy, const float* vz, const float* u) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->vel_orig, (size_t)c->n * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->u_s, (size_t)np * sizeof(float)));
    CRK_TRY(crk_ensure(c, c->fst, (size_t)np * FROW * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->facc, (size_t)np * sizeof(float4)));
    CRK_TRY(crk_ensure(c, c->xv, (size_t)np * 2 * sizeof(float4)));
    k_pack_vel<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>(vx, vy, vz, u, c->n, (float4*)c->vel_orig.p);
    CRK_TRY(crk_check_launch(c, "k_pack_vel"));
    SweepArgs a = make_args(c);
    k_hydro_prep<<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>(a, (const float4*)c->vel_orig.p, (float*)c->u_s.p);
    return crk_check_launch(c, "k_hydro_prep");
}

// a2 + a3 (mom), a4 (gv) or both in one sweep; gv needs crk_launch_hydro_prep first; gradv_full: diagnostics (all 9 components)
int crk_launch_rk(crk_ctx* c, bool mom, bool gv, float* A, float* B, float* gradA, float* gradB, float* gradv_full,
                  const int32_t* ids, int64_t n_ids) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->coef, (size_t)np * 4 * sizeof(float4)));
    SweepArgs a = make_args(c);
    a.o0 = A; a.o1 = B; a.o2 = gradA; a.o3 = gradB;
    a.ids = ids; a.n_ids = n_ids;
    const int64_t items = ids ? n_ids : c->nl;
    if (items == 0) return CRK_OK;
    const int smem = W2_WPC * ((gv ? 2 : 1) * (int)PSTRIDE + (int)sizeof(Meta));
    const float* us = (const float*)c->u_s.p;
    unsigned grid = 0;
    if (mom && !ids) CRK_CUDA(c, cudaMemsetAsync((int*)c->flag.p + FW_FALLBACK, 0, sizeof(int), c->stream));   // counts this sweep only
    if (mom && gv) {
        CRK_TRY(persistent_grid(c, k_rk<true, true>, W2_WPC * 32, smem, W2_WPC, items, &grid));
        a.sched = (unsigned int*)c->sched.p;
        k_rk<true, true><<<grid, W2_WPC * 32, smem, c->stream>>>(a, us, gradv_full);
    } else if (mom) {
        CRK_TRY(persistent_grid(c, k_rk<true, false>, W2_WPC * 32, smem, W2_WPC, items, &grid));
        a.sched = (unsigned int*)c->sched.p;
        k_rk<true, false><<<grid, W2_WPC * 32, smem, c->stream>>>(a, nullptr, nullptr);
    } else {
        CRK_TRY(persistent_grid(c, k_rk<false, true>, W2_WPC * 32, smem, W2_WPC, items, &grid));
        a.sched = (unsigned int*)c->sched.p;
        k_rk<false, true><<<grid, W2_WPC * 32, smem, c->stream>>>(a, us, gradv_full);
    }
    return crk_check_launch(c, "k_rk");
}

// a5 on the state written by crk_launch_hydro_prep and the grad v sweep
int crk_launch_forces(crk_ctx* c, float* ax, float* ay, float* az, float* dudt, uint32_t* pair_count, const int32_t* ids,
                      int64_t n_ids, const uint8_t* active) {
    const int64_t np = c->nl * CRK_LEAF;
    SweepArgs a = make_args(c);
    a.ids = ids; a.n_ids = n_ids; a.active = active;
    const int64_t items = ids ? n_ids : c->nl;
    if (items == 0) return CRK_OK;
    a.o0 = ax; a.o1 = ay; a.o2 = az; a.o3 = dudt; a.ocnt = pair_count;
    const bool ts_on = (c->prm.flags & CRK_FLAG_TIMESTEP) != 0;
    const int smem = FROW * (int)PSTRIDE + (int)sizeof(Meta) + (int)(ts_on ? sizeof(ForceEpi<true>) : sizeof(ForceEpi<false>));
    unsigned grid = 0;
    if (ts_on) {
        CRK_TRY(crk_ensure(c, c->ts_s, (size_t)np * sizeof(float2)));
        a.ts = (float2*)c->ts_s.p;
        CRK_TRY(persistent_grid(c, k_forces<true>, W5_WPL * 32, smem, 1, items, &grid));
        a.sched = (unsigned int*)c->sched.p;
        k_forces<true><<<grid, W5_WPL * 32, smem, c->stream>>>(a);
    } else {
        CRK_TRY(persistent_grid(c, k_forces<false>, W5_WPL * 32, smem, 1, items, &grid));
        a.sched = (unsigned int*)c->sched.p;
        k_forces<false><<<grid, W5_WPL * 32, smem, c->stream>>>(a);
    }
    return crk_check_launch(c, "k_forces");
}

// NEXT row 4b: active / passive leaves.  A leaf is active when one of its particles is; the force sweep runs
// over the active leaves only, the grad v sweep over their "halo" (every leaf of an active leaf's interaction list, itself
// included: a passive neighbour's grad v_j enters Eqs. 27-30 of an active particle).  flags: [0, nl) active, [nl, 2 nl) halo.
namespace {
__global__ void __launch_bounds__(256) k_mark_active(const uint8_t* __restrict__ active, const int32_t* __restrict__ perm, int64_t n,
                                                     int64_t nl, const uint32_t* __restrict__ cnt, const uint32_t* __restrict__ list,
                                                     uint32_t cap, uint32_t* __restrict__ flags) {
    const int lane = threadIdx.x & 31;
    const int64_t leaf = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (leaf >= nl) return;
    const int64_t i = leaf * CRK_LEAF + lane;
    const bool on = (i < n) && active[perm[i]] != 0;
    if (!__any_sync(0xffffffffu, on)) return;
    if (lane == 0) flags[leaf] = 1u;
    const uint32_t m = cnt[leaf];
    for (uint32_t e = lane; e < m; e += 32) flags[nl + (list[(uint64_t)leaf * cap + e] & CRK_LEAF_MASK)] = 1u;
}
// ids[offs[q]] = q - base for every set flag (offs = exclusive scan of flags)
__global__ void __launch_bounds__(256) k_compact_ids(const uint32_t* __restrict__ flags, const uint32_t* __restrict__ offs, int64_t m,
                                                     int64_t nl, int32_t* __restrict__ ids) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < m && flags[q]) ids[offs[q]] = (int32_t)(q < nl ? q : q - nl);
}
}  // namespace

// fills c->act_ids with the active leaves followed by the halo leaves; counts on the host (one synchronisation)
int crk_select_active(crk_ctx* c, const uint8_t* active, int64_t* n_active, int64_t* n_halo) {
    const int64_t nl = c->nl;
    CRK_TRY(crk_ensure(c, c->act_flags, (size_t)2 * nl * sizeof(uint32_t)));
    CRK_TRY(crk_ensure(c, c->act_offs, ((size_t)2 * nl + 1) * sizeof(uint32_t)));
    CRK_TRY(crk_ensure(c, c->act_ids, (size_t)2 * nl * sizeof(int32_t)));
    uint32_t* flags = (uint32_t*)c->act_flags.p;
    uint32_t* offs = (uint32_t*)c->act_offs.p;
    CRK_CUDA(c, cudaMemsetAsync(flags, 0, (size_t)2 * nl * sizeof(uint32_t), c->stream));
    k_mark_active<<<(unsigned)((nl + 7) / 8), 256, 0, c->stream>>>(active, c->perm, c->n, nl, (const uint32_t*)c->nbr_cnt.p,
                                                                   (const uint32_t*)c->nbr_list.p, (uint32_t)c->leaf_list_cap, flags);
    CRK_TRY(crk_check_launch(c, "k_mark_active"));
    CRK_TRY(crk_exclusive_scan_u32(c, flags, offs, 2 * nl, c->scan_tmp));
    k_compact_ids<<<(unsigned)((2 * nl + 255) / 256), 256, 0, c->stream>>>(flags, offs, 2 * nl, nl, (int32_t*)c->act_ids.p);
    CRK_TRY(crk_check_launch(c, "k_compact_ids"));
    uint32_t* h = (uint32_t*)((char*)c->h_flag + 48);
    CRK_CUDA(c, cudaMemcpyAsync(h, offs + nl, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    CRK_CUDA(c, cudaMemcpyAsync(h + 1, offs + 2 * nl, sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    CRK_CUDA(c, cudaStreamSynchronize(c->stream));
    *n_active = (int64_t)h[0];
    *n_halo = (int64_t)h[1] - (int64_t)h[0];
    return CRK_OK;
}

// NEXT row 1: Eqs. 19-23 on the state left by crk_hydro_derivs
int crk_launch_compat(crk_ctx* c, float dt, float c1, float c0, const float* bx, const float* by, const float* bz,
                      float* delta_u) {
    const int64_t np = c->nl * CRK_LEAF;
    CRK_TRY(crk_ensure(c, c->kick, (size_t)np * sizeof(float4)));
    SweepArgs a = make_args(c);
    k_compat_prep<<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>((const float4*)c->facc.p, c->perm, c->n,
                                                                       np, c1, c0, bx, by, bz, (float4*)c->kick.p);
    CRK_TRY(crk_check_launch(c, "k_compat_prep"));
    a.o0 = delta_u;
    const int smem = CPL * (int)PSTRIDE + (int)sizeof(Meta);
    unsigned grid = 0;
    CRK_TRY(persistent_grid(c, k_compat, W5_WPL * 32, smem, 1, c->nl, &grid));
    a.sched = (unsigned int*)c->sched.p;
    k_compat<<<grid, W5_WPL * 32, smem, c->stream>>>(a, dt, (const float4*)c->kick.p);
    return crk_check_launch(c, "k_compat");
}

// NEXT row 3: evolved smoothing length, Eqs. 51-53, a stream pass over (h, V) of the last crk_volumes:
// N_i = (4/3) pi h^3 / V (Eq. 51), N_res = (4/3) pi n_h^3, Delta_N = (N_res/N_i)^(1/3) = n_h V^(1/3) / h,
// lambda = 0.2 (1 + Delta_N^2) if Delta_N < 1 else 0.2 (1 + 1/Delta_N^3) (Eq. 53), h~ = h (1 - lambda + lambda Delta_N) (Eq. 52)
namespace {
__global__ void __launch_bounds__(256) k_evolve_h(const float4* __restrict__ posh, const float4* __restrict__ posV,
                                                  const int32_t* __restrict__ perm, int64_t n, float n_h,
                                                  float* __restrict__ h_new) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float h = posh[k].w, V = posV[k].w;
    const float dN = n_h * cbrtf(V) / h;
    const float lambda = dN < 1.0f ? 0.2f * (1.0f + dN * dN) : 0.2f * (1.0f + 1.0f / (dN * dN * dN));
    h_new[perm[k]] = h * (1.0f - lambda + lambda * dN);
}
}  // namespace

int crk_launch_evolve_h(crk_ctx* c, float* h_new) {
    k_evolve_h<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>((const float4*)c->posh.p, (const float4*)c->posV.p,
                                                                      c->perm, c->n, c->prm.n_h, h_new);
    return crk_check_launch(c, "k_evolve_h");
}

// NEXT row 2a: time-step criteria, Eqs. 46-50 with a = 1, adot = 0, no gravity: a stream pass over the
// force-sweep state and the two per-particle maxima reduced by k_forces<true>
namespace {
__global__ void __launch_bounds__(256) k_timestep(const float4* __restrict__ fst, const float4* __restrict__ facc,
                                                  const float2* __restrict__ ts, const int32_t* __restrict__ perm, int64_t n,
                                                  float gamma, float n_h, float C_cfl, float* __restrict__ dt_min) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float4 g = fst[k * FROW + 6];                  // g_xx, g_yy, g_zz, P
    const float rho = fst[k * FROW + 7].w;
    const float cs = sqrtf(gamma * fmaxf(g.w, 0.0f) / rho);
    const float hhat = 1.0f / (n_h * fst[k * FROW].w);   // h / n_h
    const float4 acc = facc[k];                          // dv/dt
    const float2 mx = ts[k];
    const float csq = sqrtf(4.0f * mx.y / rho);                                              // sqrt(zeta Q / rho)
    const float vmax = fmaxf(fmaxf(mx.x, cs), fmaxf(csq, hhat * fabsf(g.x + g.y + g.z)));    // Eq. 46
    const float dth = C_cfl * hhat / vmax;                                                   // Eq. 47
    const float dta = sqrtf(hhat / sqrtf(acc.x * acc.x + acc.y * acc.y + acc.z * acc.z));    // Eq. 48, r_soft = inf
    dt_min[perm[k]] = fminf(dth, dta);                                                       // Eq. 49
}
}  // namespace

int crk_launch_timestep(crk_ctx* c, float C_cfl, float* dt_min) {
    k_timestep<<<(unsigned)((c->n + 255) / 256), 256, 0, c->stream>>>((const float4*)c->fst.p, (const float4*)c->facc.p,
                                                                      (const float2*)c->ts_s.p, c->perm, c->n, c->prm.gamma,
                                                                      c->prm.n_h, C_cfl, dt_min);
    return crk_check_launch(c, "k_timestep");
}
